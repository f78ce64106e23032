// Fused stage kernel of the scalar advection equation (13), PAPER.md:364-370 (sm_100a): one Runge-Kutta sub-step
//   rho(s_out) = dt_sub * F(rho(s_deriv)) + w0 rho(s_prev0) + w1 rho(s_prev1)        (eq. (5))
// over every block, F = -div(rho v) with limited reconstruction and the upwind flux that the wave speeds
// min(v,0), max(v,0) give: F_face = max(v,0) rho_L + min(v,0) rho_R.
//
// One variable, 8 bytes per cell: the kernel is bound by HBM bandwidth.  Same data path as the Euler stage kernel
// (f4_stage.cu): a thread group of N x TY threads owns a (block, y-tile) and marches through the z planes; padded
// planes arrive by bulk async copies (TMA engine, completion on an mbarrier) in an 8-slot shared-memory ring six
// planes ahead of use; z ghost planes / y ghost rows of same-level neighbours are fetched straight from their interior
// cells and the x face layers of the new state are pushed into the neighbours' ghost cells (a1 of the pattern,
// PAPER.md:195, 235-238).  Primitive and conservative variables are identical: nothing is converted,
// the ring is read-only for the threads, and the only exchange is one half slope per cell and direction (x, y)
// through shared memory, ONE group barrier per plane; the z direction lives in registers along the march.
#include <type_traits>

#include "../../include/f4.h"
#include "f4_dev.hpp"
#include "f4_stage_dev.cuh"

namespace f4 {
namespace {

template <int DIM, int N, int TY, int G>
struct CfgA {
  static constexpr int P = N + 2 * NG, PP = P * P;
  static constexpr int PZ = (DIM == 3) ? P : 1;
  static constexpr size_t VS = (size_t)P * P * PZ;   // one variable: VS doubles per block
  static constexpr bool WHOLE = (TY == N);
  static constexpr int ROWS = TY + 4, PLANE = ROWS * P;
  static constexpr int NSLOT = (DIM == 3) ? 8 : 1;     // ring depth (the march is unrolled by 8): planes c-1, c and six in flight
  static constexpr int TG = N * TY, NT = TG * G, YT = N / TY;
  // half slopes of the cells (-1 .. N) x rows (x direction) and columns x rows (-1 .. TY) (y direction), two buffers
  static constexpr int HX = TY * (N + 2), HY = (TY + 2) * N, EXD = HX + HY;
  static constexpr int NEX = (DIM == 3) ? 2 : 1;
  static constexpr int GROUP_DOUBLES = NSLOT * PLANE + NEX * EXD;
  static constexpr size_t SMEM = (size_t)G * GROUP_DOUBLES * 8 + (size_t)G * NSLOT * 8;
  static_assert(TG % 32 == 0 && N % TY == 0 && GROUP_DOUBLES % 2 == 0 && PLANE % 2 == 0, "tile shape");
};

// FAST: van Leer fixed at compile time; BF: store the face fluxes at refinement boundaries (flux fixing)
template <int DIM, int N, int TY, int G, bool FAST, bool BF>
__global__ void __launch_bounds__(CfgA<DIM, N, TY, G>::NT, 1024 / CfgA<DIM, N, TY, G>::NT) advect_kernel(const __grid_constant__ StageParams p) {
  using C = CfgA<DIM, N, TY, G>;
  constexpr int P = C::P, PP = C::PP, PLANE = C::PLANE, TG = C::TG;
  constexpr bool WHOLE = C::WHOLE;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int grp = (G == 1) ? 0 : (int)threadIdx.x / TG;
  const int t = (G == 1) ? (int)threadIdx.x : (int)threadIdx.x % TG;
  const int item = blockIdx.x * G + grp;
  if (item >= p.nblocks * C::YT) return;   // a whole group leaves together: its barriers are private to the group
  const int blk = WHOLE ? item : item / C::YT;
  const int j0 = WHOLE ? 0 : (item % C::YT) * TY;
  const int i = t % N, j = t / N;

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
  // wave speeds min(v,0), max(v,0) per direction
  const double vpx = fmax(p.vel[0], 0.0), vmx = fmin(p.vel[0], 0.0);
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
    gy0 = nb[2]; gy1 = nb[3];
    if (DIM == 3) { gz0 = nb[4]; gz1 = nb[5]; }
  }
  const double* ylo_base = (gy0 >= 0) ? p.deriv + (size_t)gy0 * C::VS + (size_t)(N - 2) * P : dbase + (size_t)(P - 2) * P;
  const double* yhi_base = (gy1 >= 0) ? p.deriv + (size_t)gy1 * C::VS : dbase + (size_t)N * P;
  // bulk copies of z plane c (c in [-2, N+2); 2D: c = 0) into ring slot s
  auto issue_plane = [&](int c, int s) {
    const bool interior = (DIM == 2) || (c >= 0 && c < N);
    const int kslot = (DIM == 3) ? (c < 0 ? c + P : c) : 0;
    const uint32_t dst = ring_u32 + (uint32_t)(s * PLANE) * 8u, bar = bars_u32 + 8u * s;
    const double* src = dbase + (size_t)kslot * PP;
    if (DIM == 3 && c < 0 && gz0 >= 0) src = p.deriv + (size_t)gz0 * C::VS + (size_t)(c + N) * PP;   // its planes N-2, N-1
    if (DIM == 3 && c >= N && gz1 >= 0) src = p.deriv + (size_t)gz1 * C::VS + (size_t)(c - N) * PP;  // its planes 0, 1
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

  // ---- per-thread constants of the x / y sweep
  const int rr = rown(j0 + j);
  const int own = rr * P + i;
  const int own_ym = rown(j0 + j - 1) * P + i, own_yp = rown(j0 + j + 1) * P + i;
  // x ghosts are pair-transposed (f4_ghost.cu cell_off): ghost (N+g, row r) sits in row r&~1, (g-2, row r) in row r|1,
  // both at column N + 2*(r&1) + g
  const int gcol = N + 2 * (rr & 1);
  const int own_xm = (i == 0) ? (rr | 1) * P + gcol + 1 : own - 1;
  const int own_xp = (i == N - 1) ? (rr & ~1) * P + gcol : own + 1;
  // halo role of the first 2*TY + 2*N threads: the half slope of one halo cell (cell -1 / N of a row, row -1 / TY of a
  // column): offsets of that cell (h0), its low (hm) and high (hp) neighbour, and where its half slope goes (hdst)
  constexpr int NHALO = 2 * TY + 2 * N;
  static_assert(NHALO <= TG, "halo roles need one pass");
  const bool is_h = t < NHALO;
  int h0 = 0, hm = 0, hp = 0, hdst = 0;
  if (is_h) {
    if (t < 2 * TY) {
      const int r = t >> 1, hi = t & 1, sr = rown(j0 + r), gc = N + 2 * (sr & 1);
      const int olo = (sr | 1) * P + gc, ohi = (sr & ~1) * P + gc;   // ghost pairs (-2,-1) and (N,N+1) of the row
      h0 = hi ? ohi : olo + 1;
      hm = hi ? sr * P + N - 1 : olo;
      hp = hi ? ohi + 1 : sr * P;
      hdst = r * (N + 2) + (hi ? N + 1 : 0);
    } else {
      const int q = t - 2 * TY, col = q >> 1, hi = q & 1, y = hi ? j0 + TY : j0 - 1;
      h0 = rown(y) * P + col;
      hm = rown(y - 1) * P + col;
      hp = rown(y + 1) * P + col;
      hdst = C::HX + (hi ? TY + 1 : 0) * N + col;
    }
  }
  const int hxo = j * (N + 2) + i + 1, hyo = C::HX + (j + 1) * N + i;   // own entries of the half-slope arrays

  int bfs[6] = {-1, -1, -1, -1, -1, -1};
  if (BF && p.bfslot) {
#pragma unroll
    for (int f = 0; f < 2 * DIM; ++f) bfs[f] = p.bfslot[(size_t)blk * 6 + f];
  }
  constexpr int BFS = N * ((DIM == 3) ? N : 1);   // cell faces of one block face
  auto bf_store = [&](int slot, double F, int t1, int t2) { p.bflux[(size_t)slot * BFS + t2 * N + t1] = F; };

  // x / y sweep of plane W (z index kk) around the own value wa: sum over the x, y faces of (F_in - F_out).
  // `after_barrier` runs once per group between the exchange barrier and the reads (the ring refill)
  auto sweep_xy = [&](const double* W, double wa, double* ex, int kk, auto&& after_barrier) -> double {
    const double wxm = W[own_xm], wxp = W[own_xp], wym = W[own_ym], wyp = W[own_yp];
    const double hsx = half_slope<FAST>(wa - wxm, wxp - wa, limiter);
    const double hsy = half_slope<FAST>(wa - wym, wyp - wa, limiter);
    ex[hxo] = hsx;
    ex[hyo] = hsy;
    if (is_h) {
      const double w0 = W[h0];
      ex[hdst] = half_slope<FAST>(w0 - W[hm], W[hp] - w0, limiter);
    }
    gsync();
    after_barrier();
    // upwind fluxes (wave speeds min(v,0), max(v,0)): F = v+ rho_L + v- rho_R at the four faces of the cell
    const double fxl = fma(vpx, wxm + ex[hxo - 1], vmx * (wa - hsx));
    const double fxh = fma(vpx, wa + hsx, vmx * (wxp - ex[hxo + 1]));
    const double fyl = fma(vpy, wym + ex[hyo - N], vmy * (wa - hsy));
    const double fyh = fma(vpy, wa + hsy, vmy * (wyp - ex[hyo + N]));
    if (BF) {
      if (i == 0 && bfs[0] >= 0) bf_store(bfs[0], fxl, j0 + j, kk);
      if (i == N - 1 && bfs[1] >= 0) bf_store(bfs[1], fxh, j0 + j, kk);
      if (j0 + j == 0 && bfs[2] >= 0) bf_store(bfs[2], fyl, i, kk);
      if (j0 + j == N - 1 && bfs[3] >= 0) bf_store(bfs[3], fyh, i, kk);
    }
    return (fxl - fxh) + (fyl - fyh);
  };

  // ---- Runge-Kutta combine eq. (5), store, x push
  const double sdt = p.dt_dev ? (p.dtf * *p.dt_dev) * p.inv_dx_l[lvl] : p.sdt_l[lvl];   // dt_sub / dx of this block's level
  const int co = (j0 + j) * P + i;
  const double* pa = p.prev0 + boff + co;
  const double* pb = p.prev1 ? p.prev1 + boff + co : nullptr;
  double* po = p.out + boff + co;
  double* ppx = nullptr;
  if (p.nbr && p.push_x) {
    const int* nb = p.nbr + (size_t)blk * 6;
    const int jg = j0 + j;
    if (i < NG && nb[0] >= 0) ppx = p.out + (size_t)nb[0] * C::VS + ((jg & ~1) * P + N + 2 * (jg & 1) + i);
    if (i >= N - NG && nb[1] >= 0) ppx = p.out + (size_t)nb[1] * C::VS + ((jg | 1) * P + N + 2 * (jg & 1) + (i - (N - NG)));
  }
  auto finish = [&](int k, double tot, double a, double b) {
    const int ko = (DIM == 3 ? k : 0) * PP;
    const double u = fma(sdt, tot, fma(p.w1, b, p.w0 * a));
    po[ko] = u;
    if (ppx) ppx[ko] = u;
  };

  constexpr int ISSUER = (TG >= 128) ? 96 : 0;
  if (DIM == 2) {
    if (t == ISSUER) issue_plane(0, 0);
    const double a = pa[0], b = pb ? pb[0] : 0.0;
    mbar_wait(bars_u32, 0);
    const double acc = sweep_xy(ring, ring[own], ex0, 0, []() {});
    finish(0, acc, a, b);
  } else {
    constexpr int NS = C::NSLOT;
    if (t == ISSUER) {
      for (int q = 0; q < NS && q - 2 <= N + 1; ++q) issue_plane(q - 2, q);
    }
    double dA = 0.0, Lz = 0.0, accp = 0.0, wa = 0.0;
    // previous states of plane c are requested in iteration c and consumed two iterations later (finish of cell c)
    double aq0 = 0.0, aq1 = 0.0, bq0 = 0.0, bq1 = 0.0;
    uint32_t ph = 0;       // phase parity of each slot's mbarrier
    // sc_t: ring slot of plane c, (c + 2) & (NS - 1), as a compile-time constant (shared-memory addresses become
    // register + immediate)
    auto march = [&](int c, auto sc_t, auto zflux_t, auto fin_t, auto sweep_t) {
      constexpr bool ZFLUX = decltype(zflux_t)::value, FIN = decltype(fin_t)::value, SWEEP = decltype(sweep_t)::value;
      constexpr int sc = decltype(sc_t)::value;
      constexpr int sk = (sc + NS - 1) & (NS - 1);          // slot of plane c-1
      double a_new = 0.0, b_new = 0.0;
      if (c >= 0 && c < N) { a_new = pa[c * PP]; b_new = pb ? pb[c * PP] : 0.0; }
      mbar_wait(bars_u32 + 8u * sc, (ph >> sc) & 1u);
      ph ^= 1u << sc;
      const double wB = ring[sc * PLANE + own];
      // z: slope of cell c-1 from rho(c-2), rho(c-1), rho(c); upwind flux at the face between cells c-2 and c-1
      const double dB = wB - wa;
      const double hs = half_slope<FAST>(dA, dB, limiter);  // c <= -1: values unused
      const double Fz = ZFLUX ? fma(vpz, Lz, vmz * (wa - hs)) : 0.0;
      Lz = wa + hs;
      dA = dB;
      if (BF && ZFLUX) {
        if (c == 1 && bfs[4] >= 0) bf_store(bfs[4], Fz, i, j0 + j);
        if (c == N + 1 && bfs[5] >= 0) bf_store(bfs[5], Fz, i, j0 + j);
      }
      if (FIN) finish(c - 2, accp - Fz, aq1, bq1);
      aq1 = aq0; aq0 = a_new;
      bq1 = bq0; bq0 = b_new;
      // after this iteration's barrier every thread is past its reads of plane c-2: its slot takes the next plane of the ring
      auto refill = [&]() {
        if (t == ISSUER && c >= 0 && c - 2 + NS <= N + 1) issue_plane(c - 2 + NS, (sc + NS - 2) & (NS - 1));   // plane c-2's slot
      };
      if (SWEEP) accp = sweep_xy(ring + sk * PLANE, wa, ex0 + (c & 1) * C::EXD, c - 1, refill) + Fz;
      else { gsync(); refill(); }
      wa = wB;
    };
    using T = std::true_type;
    using F_ = std::false_type;
    auto slot = [](auto c_t) { return std::integral_constant<int, (decltype(c_t)::value + 2) & (NS - 1)>{}; };
    march(-2, slot(std::integral_constant<int, -2>{}), F_{}, F_{}, F_{});
    march(-1, slot(std::integral_constant<int, -1>{}), F_{}, F_{}, F_{});
    march(0, slot(std::integral_constant<int, 0>{}), F_{}, F_{}, F_{});
    march(1, slot(std::integral_constant<int, 1>{}), T{}, F_{}, T{});
    // steady state c = 2 .. N, unrolled by the ring depth: plane c0 + u sits in slot (4 + u) & (NS - 1)
#pragma unroll 1
    for (int c0 = 2; c0 <= N; c0 += NS) {
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
}

template <int DIM, int N, int TY, int G>
cudaError_t launch_cfgA(const StageParams& p, cudaStream_t s) {
  using C = CfgA<DIM, N, TY, G>;
  const bool fast = p.limiter == F4_LIM_VANLEER, bf = p.bfslot != nullptr;
  void (*k)(StageParams) = bf ? (fast ? advect_kernel<DIM, N, TY, G, true, true> : advect_kernel<DIM, N, TY, G, false, true>)
                              : (fast ? advect_kernel<DIM, N, TY, G, true, false> : advect_kernel<DIM, N, TY, G, false, false>);
  cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
  if (e != cudaSuccess) return e;
  const int nitems = p.nblocks * C::YT;
  k<<<(nitems + G - 1) / G, C::NT, C::SMEM, s>>>(p);
  return cudaGetLastError();
}

}  // namespace

bool advect_supported(const StageParams& p) {
  return (p.limiter == F4_LIM_VANLEER || p.limiter == F4_LIM_MINMOD || p.limiter == F4_LIM_MC) && !p.prev2;
}

cudaError_t launch_advect(int dim, int n, const StageParams& p, cudaStream_t s) {
  if (p.nblocks <= 0) return cudaSuccess;
  if (dim == 2 && n == 8) return launch_cfgA<2, 8, 8, 4>(p, s);
  if (dim == 2 && n == 16) return launch_cfgA<2, 16, 16, 1>(p, s);
  if (dim == 2 && n == 32) return launch_cfgA<2, 32, 8, 1>(p, s);
  if (dim == 3) return launch_advect2(n, p, s);   // two cells per thread (f4_advect2.cu)
  return cudaErrorInvalidValue;
}

}  // namespace f4
