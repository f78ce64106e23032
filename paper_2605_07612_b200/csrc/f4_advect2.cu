// Scalar advection stage kernel, 3D, TWO x-adjacent cells per thread (sm_100a): the same sub-step, data path and
// arithmetic as advect_kernel (f4_advect.cu; eq. (13), eq. (5)) with 16-byte
// shared-memory and global accesses, the face between the two cells inside the thread, and half the address
// arithmetic per cell: advect_kernel is bound by instruction issue (175 instructions per cell update,
// profiles/advect_kernel_r2.md), not by the 8 bytes per cell it moves.  At ~100 registers per thread the register
// file has room for it -- unlike in the Euler kernel (profiles/stage_kernel_r2_experiments.md).
#include <type_traits>

#include "../../include/f4.h"
#include "f4_dev.hpp"
#include "f4_stage_dev.cuh"

namespace f4 {
namespace {

__device__ __forceinline__ double2 ld2(const double* p) { return *reinterpret_cast<const double2*>(p); }
__device__ __forceinline__ void st2(double* p, double a, double b) { *reinterpret_cast<double2*>(p) = make_double2(a, b); }

template <int N, int TY, int G>
struct CfgA2 {
  static constexpr int P = N + 2 * NG, PP = P * P;
  static constexpr size_t VS = (size_t)P * P * P;
  static constexpr bool WHOLE = (TY == N);
  static constexpr int ROWS = TY + 4, PLANE = ROWS * P;
  static constexpr int NSLOT = 8;                       // ring depth (the march is unrolled by 8)
  static constexpr int HX = N / 2, TG = HX * TY, NT = TG * G, YT = N / TY;
  // half slopes: hx [TY][N] own cells | hxlo [TY], hxhi [TY] cells -1 / N of a row | hy [TY+2][N] rows -1 .. TY
  static constexpr int OXLO = TY * N, OXHI = OXLO + TY, OY = OXHI + TY, EXD = OY + (TY + 2) * N;
  static constexpr int GROUP_DOUBLES = NSLOT * PLANE + 2 * EXD;
  static constexpr size_t SMEM = (size_t)G * GROUP_DOUBLES * 8 + (size_t)G * NSLOT * 8;
  static constexpr int NHALO = 2 * TY + 2 * HX;         // x: cells -1 / N of a row; y: a pair of row -1 / TY
  static_assert(TG % 32 == 0 && N % TY == 0 && TY % 2 == 0 && GROUP_DOUBLES % 2 == 0 && PLANE % 2 == 0 && EXD % 2 == 0 &&
                    NHALO <= TG, "tile shape");
};

template <int N, int TY, int G, bool FAST, bool BF>
__global__ void __launch_bounds__(CfgA2<N, TY, G>::NT, 512 / CfgA2<N, TY, G>::NT) advect2_kernel(const __grid_constant__ StageParams p) {
  using C = CfgA2<N, TY, G>;
  constexpr int P = C::P, PP = C::PP, PLANE = C::PLANE, TG = C::TG, HX = C::HX;
  constexpr bool WHOLE = C::WHOLE;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int grp = (G == 1) ? 0 : (int)threadIdx.x / TG;
  const int t = (G == 1) ? (int)threadIdx.x : (int)threadIdx.x % TG;
  const int item = blockIdx.x * G + grp;
  if (item >= p.nblocks * C::YT) return;
  const int blk = WHOLE ? item : item / C::YT;
  const int j0 = WHOLE ? 0 : (item % C::YT) * TY;
  const int pi = t % HX, j = t / HX;       // cells (2 pi, 2 pi + 1) of tile row j

  double* ring = reinterpret_cast<double*>(smem_raw) + (size_t)grp * C::GROUP_DOUBLES;
  double* ex0 = ring + C::NSLOT * PLANE;
  uint64_t* bars = reinterpret_cast<uint64_t*>(reinterpret_cast<double*>(smem_raw) + (size_t)G * C::GROUP_DOUBLES) +
                   grp * C::NSLOT;
  const uint32_t ring_u32 = smem_u32(ring), bars_u32 = smem_u32(bars);
  auto gsync = [&]() {
    if (TG == 32) __syncwarp();
    else group_sync(1 + grp, TG);
  };
  const int limiter = p.limiter;
  const int lvl = p.level[blk];
  const size_t boff = (size_t)blk * C::VS;
  const double* dbase = p.deriv + boff;
  const double vpx = fmax(p.vel[0], 0.0), vmx = fmin(p.vel[0], 0.0);   // wave speeds max(v,0), min(v,0)
  const double vpy = fmax(p.vel[1], 0.0), vmy = fmin(p.vel[1], 0.0);
  const double vpz = fmax(p.vel[2], 0.0), vmz = fmin(p.vel[2], 0.0);
  auto rown = [&](int y) { return WHOLE ? (y < 0 ? y + P : y) : y - j0 + 2; };

  if (t == 0) {
    for (int s = 0; s < C::NSLOT; ++s) mbar_init(&bars[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  gsync();

  int gz0 = -1, gz1 = -1, gy0 = -1, gy1 = -1;
  if (p.nbr) {
    const int* nb = p.nbr + (size_t)blk * 6;
    gy0 = nb[2]; gy1 = nb[3]; gz0 = nb[4]; gz1 = nb[5];
  }
  const double* ylo_base = (gy0 >= 0) ? p.deriv + (size_t)gy0 * C::VS + (size_t)(N - 2) * P : dbase + (size_t)(P - 2) * P;
  const double* yhi_base = (gy1 >= 0) ? p.deriv + (size_t)gy1 * C::VS : dbase + (size_t)N * P;
  auto issue_plane = [&](int c, int s) {   // bulk copies of z plane c (c in [-2, N+2)) into ring slot s
    const bool interior = (c >= 0 && c < N);
    const int kslot = c < 0 ? c + P : c;
    const uint32_t dst = ring_u32 + (uint32_t)(s * PLANE) * 8u, bar = bars_u32 + 8u * s;
    const double* src = dbase + (size_t)kslot * PP;
    if (c < 0 && gz0 >= 0) src = p.deriv + (size_t)gz0 * C::VS + (size_t)(c + N) * PP;   // its planes N-2, N-1
    if (c >= N && gz1 >= 0) src = p.deriv + (size_t)gz1 * C::VS + (size_t)(c - N) * PP;  // its planes 0, 1
    const size_t ko = (size_t)kslot * PP;
    if (WHOLE) {
      constexpr uint32_t bytes = (uint32_t)N * P * 8, gbytes = (uint32_t)2 * P * 8;
      mbar_expect_tx(bar, bytes + (interior ? 2 * gbytes : 0u));
      bulk_g2s(dst, src, bytes, bar);
      if (interior) {
        bulk_g2s(dst + (uint32_t)(N * P) * 8u, yhi_base + ko, gbytes, bar);
        bulk_g2s(dst + (uint32_t)((P - 2) * P) * 8u, ylo_base + ko, gbytes, bar);
      }
    } else {
      const int ylo = interior ? j0 - 2 : j0, yhi = interior ? j0 + TY + 2 : j0 + TY;
      const int nlow = ylo < 0 ? -ylo : 0, nhigh = yhi > N ? yhi - N : 0;
      const uint32_t bytes_low = (uint32_t)nlow * P * 8, bytes_high = (uint32_t)nhigh * P * 8;
      const uint32_t bytes_mid = (uint32_t)(yhi - ylo - nlow - nhigh) * P * 8;
      mbar_expect_tx(bar, bytes_low + bytes_mid + bytes_high);
      if (nlow) bulk_g2s(dst + (uint32_t)((ylo - (j0 - 2)) * P) * 8u, ylo_base + ko, bytes_low, bar);
      bulk_g2s(dst + (uint32_t)((ylo + nlow - (j0 - 2)) * P) * 8u, src + (size_t)(ylo + nlow) * P, bytes_mid, bar);
      if (nhigh) bulk_g2s(dst + (uint32_t)((N - (j0 - 2)) * P) * 8u, yhi_base + ko, bytes_high, bar);
    }
  };

  // ---- per-thread constants of the x / y sweep (x ghosts are pair-transposed, f4_ghost.cu cell_off)
  const int rr = rown(j0 + j);
  const int own = rr * P + 2 * pi;
  const int own_ym = rown(j0 + j - 1) * P + 2 * pi, own_yp = rown(j0 + j + 1) * P + 2 * pi;
  const int gcol = N + 2 * (rr & 1);
  const int own_xm = (pi == 0) ? (rr | 1) * P + gcol + 1 : own - 1;        // cell 2 pi - 1
  const int own_xp = (pi == HX - 1) ? (rr & ~1) * P + gcol : own + 2;      // cell 2 pi + 2
  const int hxo = j * N + 2 * pi, hyo = C::OY + (j + 1) * N + 2 * pi;      // own entries of the half-slope arrays
  const int hxm = (pi == 0) ? C::OXLO + j : hxo - 1;                       // half slope of cell 2 pi - 1 / 2 pi + 2
  const int hxp = (pi == HX - 1) ? C::OXHI + j : hxo + 2;
  // halo role of the first NHALO threads: the half slope of one halo cell of a row (x) or of a halo cell pair (y)
  const bool is_h = t < C::NHALO, h_pair = t >= 2 * TY;
  int h0 = 0, hm = 0, hp = 0, hdst = 0;
  if (is_h) {
    if (!h_pair) {
      const int r = t >> 1, hi = t & 1, sr = rown(j0 + r), gc = N + 2 * (sr & 1);
      const int olo = (sr | 1) * P + gc, ohi = (sr & ~1) * P + gc;   // ghost pairs (-2,-1) and (N,N+1) of the row
      h0 = hi ? ohi : olo + 1;
      hm = hi ? sr * P + N - 1 : olo;
      hp = hi ? ohi + 1 : sr * P;
      hdst = (hi ? C::OXHI : C::OXLO) + r;
    } else {
      const int q = t - 2 * TY, hi = q / HX, col = 2 * (q % HX), y = hi ? j0 + TY : j0 - 1;
      h0 = rown(y) * P + col;
      hm = rown(y - 1) * P + col;
      hp = rown(y + 1) * P + col;
      hdst = C::OY + (hi ? TY + 1 : 0) * N + col;
    }
  }

  int bfs[6] = {-1, -1, -1, -1, -1, -1};
  if (BF && p.bfslot) {
#pragma unroll
    for (int f = 0; f < 6; ++f) bfs[f] = p.bfslot[(size_t)blk * 6 + f];
  }
  constexpr int BFS = N * N;
  auto bf_store = [&](int slot, double F, int t1, int t2) { p.bflux[(size_t)slot * BFS + t2 * N + t1] = F; };

  // x / y sweep of plane W (z index kk) around the own values wa: sum over the x, y faces of (F_in - F_out) per cell
  auto sweep_xy = [&](const double* W, const double (&wa)[2], double* ex, int kk, auto&& after_barrier, double (&acc)[2]) {
    const double wxm = W[own_xm], wxp = W[own_xp];
    const double2 ym = ld2(W + own_ym), yp = ld2(W + own_yp);
    const double d01 = wa[1] - wa[0];
    const double hx0 = half_slope<FAST>(wa[0] - wxm, d01, limiter), hx1 = half_slope<FAST>(d01, wxp - wa[1], limiter);
    const double hy0 = half_slope<FAST>(wa[0] - ym.x, yp.x - wa[0], limiter);
    const double hy1 = half_slope<FAST>(wa[1] - ym.y, yp.y - wa[1], limiter);
    st2(ex + hxo, hx0, hx1);
    st2(ex + hyo, hy0, hy1);
    if (is_h) {
      if (!h_pair) {
        const double w0 = W[h0];
        ex[hdst] = half_slope<FAST>(w0 - W[hm], W[hp] - w0, limiter);
      } else {
        const double2 w0 = ld2(W + h0), wm = ld2(W + hm), wp = ld2(W + hp);
        st2(ex + hdst, half_slope<FAST>(w0.x - wm.x, wp.x - w0.x, limiter), half_slope<FAST>(w0.y - wm.y, wp.y - w0.y, limiter));
      }
    }
    gsync();
    after_barrier();
    // upwind fluxes F = v+ rho_L + v- rho_R: three x faces of the pair, two y faces per cell
    const double2 hym = ld2(ex + hyo - N), hyp = ld2(ex + hyo + N);
    const double fxl = fma(vpx, wxm + ex[hxm], vmx * (wa[0] - hx0));
    const double fxc = fma(vpx, wa[0] + hx0, vmx * (wa[1] - hx1));
    const double fxh = fma(vpx, wa[1] + hx1, vmx * (wxp - ex[hxp]));
    const double fyl0 = fma(vpy, ym.x + hym.x, vmy * (wa[0] - hy0)), fyh0 = fma(vpy, wa[0] + hy0, vmy * (yp.x - hyp.x));
    const double fyl1 = fma(vpy, ym.y + hym.y, vmy * (wa[1] - hy1)), fyh1 = fma(vpy, wa[1] + hy1, vmy * (yp.y - hyp.y));
    if (BF) {
      if (pi == 0 && bfs[0] >= 0) bf_store(bfs[0], fxl, j0 + j, kk);
      if (pi == HX - 1 && bfs[1] >= 0) bf_store(bfs[1], fxh, j0 + j, kk);
      if (j0 + j == 0 && bfs[2] >= 0) { bf_store(bfs[2], fyl0, 2 * pi, kk); bf_store(bfs[2], fyl1, 2 * pi + 1, kk); }
      if (j0 + j == N - 1 && bfs[3] >= 0) { bf_store(bfs[3], fyh0, 2 * pi, kk); bf_store(bfs[3], fyh1, 2 * pi + 1, kk); }
    }
    acc[0] = (fxl - fxc) + (fyl0 - fyh0);
    acc[1] = (fxc - fxh) + (fyl1 - fyh1);
  };

  // ---- Runge-Kutta combine eq. (5), store, x push
  const double sdt = p.dt_dev ? (p.dtf * *p.dt_dev) * p.inv_dx_l[lvl] : p.sdt_l[lvl];   // dt_sub / dx of this block's level
  const int co = (j0 + j) * P + 2 * pi;
  const double* pa = p.prev0 + boff + co;
  const double* pb = p.prev1 ? p.prev1 + boff + co : nullptr;
  double* po = p.out + boff + co;
  double* ppx = nullptr;   // the first / last pair of a row is the x face layer of the neighbour's ghost cells
  if (p.nbr && p.push_x) {
    const int* nb = p.nbr + (size_t)blk * 6;
    const int jg = j0 + j;
    if (pi == 0 && nb[0] >= 0) ppx = p.out + (size_t)nb[0] * C::VS + ((jg & ~1) * P + N + 2 * (jg & 1));
    if (pi == HX - 1 && nb[1] >= 0) ppx = p.out + (size_t)nb[1] * C::VS + ((jg | 1) * P + N + 2 * (jg & 1));
  }
  auto finish = [&](int k, double t0, double t1, double2 a, double2 b) {
    const int ko = k * PP;
    const double u0 = fma(sdt, t0, fma(p.w1, b.x, p.w0 * a.x)), u1 = fma(sdt, t1, fma(p.w1, b.y, p.w0 * a.y));
    st2(po + ko, u0, u1);
    if (ppx) st2(ppx + ko, u0, u1);
  };

  constexpr int ISSUER = (TG >= 128) ? 96 : 0;
  constexpr int NS = C::NSLOT;
  if (t == ISSUER) {
    for (int q = 0; q < NS && q - 2 <= N + 1; ++q) issue_plane(q - 2, q);
  }
  double dA[2] = {0.0, 0.0}, Lz[2] = {0.0, 0.0}, accp[2] = {0.0, 0.0}, wa[2] = {0.0, 0.0};
  const double2 zero2 = make_double2(0.0, 0.0);
  double2 aq0 = zero2, aq1 = zero2, bq0 = zero2, bq1 = zero2;   // previous states: requested in iteration c, used in c + 2
  uint32_t ph = 0;
  auto march = [&](int c, auto sc_t, auto zflux_t, auto fin_t, auto sweep_t) {
    constexpr bool ZFLUX = decltype(zflux_t)::value, FIN = decltype(fin_t)::value, SWEEP = decltype(sweep_t)::value;
    constexpr int sc = decltype(sc_t)::value;
    constexpr int sk = (sc + NS - 1) & (NS - 1);          // slot of plane c-1
    double2 a_new = zero2, b_new = zero2;
    if (c >= 0 && c < N) { a_new = ld2(pa + c * PP); if (pb) b_new = ld2(pb + c * PP); }
    // stage 2: u_t comes from DRAM; pull the plane four iterations ahead into L2 (one 32-byte sector per two threads)
    if (pb && (pi & 1) == 0 && c + 4 >= 0 && c + 4 < N) asm volatile("prefetch.global.L2 [%0];" ::"l"(pa + (c + 4) * PP));
    mbar_wait(bars_u32 + 8u * sc, (ph >> sc) & 1u);
    ph ^= 1u << sc;
    const double2 wB2 = ld2(ring + sc * PLANE + own);
    const double wB[2] = {wB2.x, wB2.y};
    double Fz[2];
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      // z: slope of cell c-1 from rho(c-2), rho(c-1), rho(c); upwind flux at the face between cells c-2 and c-1
      const double dB = wB[e] - wa[e];
      const double hs = half_slope<FAST>(dA[e], dB, limiter);
      Fz[e] = ZFLUX ? fma(vpz, Lz[e], vmz * (wa[e] - hs)) : 0.0;
      Lz[e] = wa[e] + hs;
      dA[e] = dB;
    }
    if (BF && ZFLUX) {
      if (c == 1 && bfs[4] >= 0) { bf_store(bfs[4], Fz[0], 2 * pi, j0 + j); bf_store(bfs[4], Fz[1], 2 * pi + 1, j0 + j); }
      if (c == N + 1 && bfs[5] >= 0) { bf_store(bfs[5], Fz[0], 2 * pi, j0 + j); bf_store(bfs[5], Fz[1], 2 * pi + 1, j0 + j); }
    }
    if (FIN) finish(c - 2, accp[0] - Fz[0], accp[1] - Fz[1], aq1, bq1);
    aq1 = aq0; aq0 = a_new;
    bq1 = bq0; bq0 = b_new;
    auto refill = [&]() {   // every thread is past its reads of plane c-2: its slot takes the next plane of the ring
      if (t == ISSUER && c >= 0 && c - 2 + NS <= N + 1) issue_plane(c - 2 + NS, (sc + NS - 2) & (NS - 1));
    };
    if (SWEEP) {
      double acc[2];
      sweep_xy(ring + sk * PLANE, wa, ex0 + (c & 1) * C::EXD, c - 1, refill, acc);
      accp[0] = acc[0] + Fz[0];
      accp[1] = acc[1] + Fz[1];
    } else {
      gsync();
      refill();
    }
    wa[0] = wB[0];
    wa[1] = wB[1];
  };
  using T = std::true_type;
  using F_ = std::false_type;
  auto slot = [](auto c_t) { return std::integral_constant<int, (decltype(c_t)::value + 2) & (NS - 1)>{}; };
  march(-2, slot(std::integral_constant<int, -2>{}), F_{}, F_{}, F_{});
  march(-1, slot(std::integral_constant<int, -1>{}), F_{}, F_{}, F_{});
  march(0, slot(std::integral_constant<int, 0>{}), F_{}, F_{}, F_{});
  march(1, slot(std::integral_constant<int, 1>{}), T{}, F_{}, T{});
#pragma unroll 1
  for (int c0 = 2; c0 <= N; c0 += NS) {   // steady state, unrolled by the ring depth: plane c0 + u sits in slot (4 + u) & (NS - 1)
    auto body = [&](auto u_t) {
      constexpr int u = decltype(u_t)::value;
      if (c0 + u <= N) march(c0 + u, std::integral_constant<int, (4 + u) & (NS - 1)>{}, T{}, T{}, T{});
    };
    body(std::integral_constant<int, 0>{}); body(std::integral_constant<int, 1>{});
    body(std::integral_constant<int, 2>{}); body(std::integral_constant<int, 3>{});
    body(std::integral_constant<int, 4>{}); body(std::integral_constant<int, 5>{});
    body(std::integral_constant<int, 6>{}); body(std::integral_constant<int, 7>{});
  }
  march(N + 1, slot(std::integral_constant<int, N + 1>{}), T{}, T{}, F_{});
}

template <int N, int TY, int G>
cudaError_t launch_cfgA2(const StageParams& p, cudaStream_t s) {
  using C = CfgA2<N, TY, G>;
  const bool fast = p.limiter == F4_LIM_VANLEER, bf = p.bfslot != nullptr;
  void (*k)(StageParams) = bf ? (fast ? advect2_kernel<N, TY, G, true, true> : advect2_kernel<N, TY, G, false, true>)
                              : (fast ? advect2_kernel<N, TY, G, true, false> : advect2_kernel<N, TY, G, false, false>);
  cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
  if (e != cudaSuccess) return e;
  const int nitems = p.nblocks * C::YT;
  k<<<(nitems + G - 1) / G, C::NT, C::SMEM, s>>>(p);
  return cudaGetLastError();
}

}  // namespace

// 3D instances with two cells per thread; launch_advect (f4_advect.cu) dispatches to them
cudaError_t launch_advect2(int n, const StageParams& p, cudaStream_t s) {
  if (n == 8) return launch_cfgA2<8, 8, 4>(p, s);
  if (n == 16) return launch_cfgA2<16, 16, 1>(p, s);
  if (n == 32) return launch_cfgA2<32, 8, 1>(p, s);
  return cudaErrorInvalidValue;
}

}  // namespace f4
