// Fused finite-volume stage kernel (sm_100a): one Runge-Kutta sub-step eq. (5)
//   u(s_out) = dt_sub * F(u(s_deriv)) + w0 u(s_prev0) + w1 u(s_prev1)
// over every block, F = -div of HLL fluxes of
// limited primitive reconstructions, optional
// fused CFL max of the NEW state.
//
// Design (differs from the paper's gang-per-block / collapse(3) OpenACC loop,
// PAPER.md:162-189, which converts the whole block to uu_prim in global
// memory and evaluates every face flux twice):
//  * a thread group of N x TY threads owns a (block, y-tile) and marches
//    through the z planes; every face flux is evaluated once;
//  * padded planes of the conservative state are fetched by bulk async copies
//    (cp.async.bulk, the TMA engine, completion on an mbarrier) into a 3-slot
//    shared-memory ring one plane ahead of use, and converted to primitives in
//    place (to_primitive once per cell);
//  * x/y fluxes exchange reconstructed states and fluxes through shared
//    memory; the z direction lives in registers along the march;
//  * fp64 division / sqrt are replaced by MUFU seeds + cubic Newton steps
//    (the kernel is co-limited by the fp64 pipe).
#include "../../include/f4.h"
#include "f4_dev.hpp"

namespace f4 {
namespace {

// ---- fast fp64 reciprocal / rsqrt: MUFU seed (~2^-22) + one cubic step -> < 2 ulp
__device__ __forceinline__ double rcp_fast(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  double e = fma(-x, r, 1.0);
  double e2 = fma(e, e, e);
  return fma(r, e2, r);
}
__device__ __forceinline__ double rsqrt_fast(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double t = x * y;
  double e = fma(-t, y, 1.0);
  double h = fma(0.375, e, 0.5);
  double he = h * e;
  return fma(y, he, y);
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
// 1-D bulk async copy global -> shared (TMA engine; SASS UBLKCP), completion counted on the mbarrier
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void group_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// limited HALF slope 1/2*phi(a,b) for the reconstruction w +- 1/2 phi (reading A1)
__device__ __forceinline__ double half_slope(double a, double b, int limiter) {
  double ab = a * b;
  double r;
  if (limiter == F4_LIM_VANLEER) {
    r = ab * rcp_fast(a + b);                         // 1/2 * 2ab/(a+b)
  } else {
    double th = (limiter == F4_LIM_MC) ? 2.0 : 1.0;   // eq. (1)
    double m = fmin(fmin(fabs(th * a), fabs(th * b)), fabs(a + b) * 0.5);
    r = 0.5 * ((a > 0.0) ? m : -m);
  }
  return (ab > 0.0) ? r : 0.0;
}

// HLL / Rusanov flux in the face-normal frame (readings A2-A3).
// q = (rho, un, ut1, ut2, p); F = (mass, normal momentum, tangential momenta, energy).
template <int DIM>
__device__ __forceinline__ void riemann_flux(const double (&L)[5], const double (&R)[5], double gamma, double ig1,
                                             int flux, double (&F)[5]) {
  const double yL = rsqrt_fast(L[0]), yR = rsqrt_fast(R[0]);  // 1/sqrt(rho)
  const double rL = L[0] * yL, rR = R[0] * yR;                // sqrt(rho)
  const double w = rcp_fast(rL + rR);
  const double uhat = (rL * L[1] + rR * R[1]) * w;
  const double du = R[1] - L[1];
  // d^2 = (rL cL^2 + rR cR^2)/(rL+rR) + 1/2 rL rR/(rL+rR)^2 du^2,  r c^2 = gamma p / sqrt(rho)
  const double d2 = fma(gamma * (L[4] * yL + R[4] * yR), w, 0.5 * (rL * w) * (rR * w) * du * du);
  const double dhat = d2 * rsqrt_fast(d2);
  double sm = uhat - dhat, sp = uhat + dhat;
  if (flux == F4_FLUX_RUSANOV) {
    double s = fmax(fabs(sm), fabs(sp));
    sm = -s;
    sp = s;
  } else {
    sm = fmin(sm, 0.0);
    sp = fmax(sp, 0.0);
  }
  const double inv = rcp_fast(sp - sm);
  const double a = sp * inv, b = -sm * inv, c = sp * sm * inv;  // F = a FL + b FR + c (UR - UL)
  double keL = L[1] * L[1] + L[2] * L[2], keR = R[1] * R[1] + R[2] * R[2];
  if (DIM == 3) { keL = fma(L[3], L[3], keL); keR = fma(R[3], R[3], keR); }
  const double EL = fma(L[4], ig1, 0.5 * L[0] * keL), ER = fma(R[4], ig1, 0.5 * R[0] * keR);  // eq. (15)
  const double mL = L[0] * L[1], mR = R[0] * R[1];
  F[0] = fma(a, mL, fma(b, mR, c * (R[0] - L[0])));
  F[1] = fma(a, fma(mL, L[1], L[4]), fma(b, fma(mR, R[1], R[4]), c * (mR - mL)));
  F[2] = fma(a, mL * L[2], fma(b, mR * R[2], c * (R[0] * R[2] - L[0] * L[2])));
  if (DIM == 3) F[3] = fma(a, mL * L[3], fma(b, mR * R[3], c * (R[0] * R[3] - L[0] * L[3])));
  else F[3] = 0.0;
  F[4] = fma(a, (EL + L[4]) * L[1], fma(b, (ER + R[4]) * R[1], c * (ER - EL)));
}

template <int DIM, int N, int TY, int G>
struct Cfg {
  static constexpr int P = N + 2 * NG;
  static constexpr int PZ = (DIM == 3) ? P : 1;
  static constexpr int NVAR = DIM + 2;
  static constexpr size_t VS = (size_t)P * P * PZ;
  static constexpr size_t BS = VS * NVAR;
  static constexpr int ROWS = TY + 4;
  static constexpr int PLANE = ROWS * P;      // doubles per variable in one ring slot
  static constexpr int SLOT = NVAR * PLANE;
  static constexpr int NSLOT = (DIM == 3) ? 3 : 1;
  static constexpr int EXV = (N + 1) * (TY + 1);  // exchange entries per variable
  static constexpr int EX = NVAR * EXV;
  static constexpr int TG = N * TY;           // threads per group
  static constexpr int NT = TG * G;
  static constexpr int YT = N / TY;           // y tiles per block
  static constexpr int GROUP_DOUBLES = NSLOT * SLOT + 2 * EX;
  static constexpr size_t SMEM = (size_t)G * GROUP_DOUBLES * 8 + (size_t)G * NSLOT * 8;
  static constexpr int HALO = 4 * TY + 4 * N;  // halo cells of an interior plane
  static_assert(HALO <= TG, "halo conversion needs one pass");
  static_assert(TG % 32 == 0 && N % TY == 0, "tile shape");
};

template <int DIM, int N, int TY, int G>
__global__ void __launch_bounds__(Cfg<DIM, N, TY, G>::NT, (Cfg<DIM, N, TY, G>::SMEM <= 100 * 1024) ? 2 : 1)
    stage_kernel(StageParams p) {
  using C = Cfg<DIM, N, TY, G>;
  constexpr int P = C::P, NV = C::NVAR, PLANE = C::PLANE, TG = C::TG, EXV = C::EXV;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int grp = threadIdx.x / TG, t = threadIdx.x % TG;
  double* ring = reinterpret_cast<double*>(smem_raw) + (size_t)grp * C::GROUP_DOUBLES;
  double* exb = ring + C::NSLOT * C::SLOT;  // [2][NV][EXV]
  uint64_t* bars = reinterpret_cast<uint64_t*>(reinterpret_cast<double*>(smem_raw) + (size_t)G * C::GROUP_DOUBLES) +
                   grp * C::NSLOT;
  const int bar_id = 1 + grp;

  const int item = blockIdx.x * G + grp;
  const int nitems = p.nblocks * C::YT;
  const bool active = item < nitems;
  const int blk = active ? item / C::YT : 0;
  const int j0 = active ? (item % C::YT) * TY : 0;
  const int i = t % N, j = t / N;

  const double gamma = p.gamma, gm1 = gamma - 1.0, ig1 = 1.0 / gm1;
  const int limiter = p.limiter, fluxs = p.flux;
  const double inv_dx = p.inv_dx0 * (double)(1u << p.level[blk]);
  const double* dbase = p.deriv + (size_t)blk * C::BS;

  if (t == 0) {
    for (int s = 0; s < C::NSLOT; ++s) mbar_init(&bars[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  group_sync(bar_id, TG);

  // issue the bulk copies of z plane c (c in [-2, N+2); 2D: c = 0) into its ring slot
  auto issue_plane = [&](int c) {
    const int idx = (DIM == 3) ? c + 2 : 0;
    const int s = idx % C::NSLOT;
    const bool interior = (DIM == 2) || (c >= 0 && c < N);
    const int kslot = (DIM == 3) ? (c < 0 ? c + P : c) : 0;
    double* dst = ring + s * C::SLOT;
    const double* src = dbase + (size_t)kslot * P * P;
    // rows y in [ylo, yhi) -> smem rows y - (j0-2); low part wraps to slots y + P
    const int ylo = interior ? j0 - 2 : j0, yhi = interior ? j0 + TY + 2 : j0 + TY;
    const int nlow = ylo < 0 ? -ylo : 0;  // rows with y < 0
    const uint32_t bytes_low = (uint32_t)nlow * P * 8, bytes_hi = (uint32_t)(yhi - ylo - nlow) * P * 8;
    mbar_expect_tx(&bars[s], (bytes_low + bytes_hi) * NV);
    for (int v = 0; v < NV; ++v) {
      const double* sv = src + (size_t)v * C::VS;
      double* dv = dst + v * PLANE;
      if (nlow) bulk_g2s(dv + (ylo - (j0 - 2)) * P, sv + (size_t)(ylo + P) * P, bytes_low, &bars[s]);
      bulk_g2s(dv + (ylo + nlow - (j0 - 2)) * P, sv + (size_t)(ylo + nlow) * P, bytes_hi, &bars[s]);
    }
  };

  // in-place conversion conservative -> primitive of one smem cell (to_primitive)
  auto convert = [&](double* W, int o, double (&w)[5]) {
    double rho = W[o];
    double ir = rcp_fast(rho);
    double ke = 0.0;
    w[0] = rho;
#pragma unroll
    for (int d = 0; d < DIM; ++d) {
      w[1 + d] = W[(1 + d) * PLANE + o] * ir;
      ke = fma(w[1 + d], w[1 + d], ke);
    }
    if (DIM == 2) w[3] = 0.0;
    w[4] = gm1 * fma(-0.5 * rho, ke, W[(NV - 1) * PLANE + o]);
#pragma unroll
    for (int d = 0; d < DIM; ++d) W[(1 + d) * PLANE + o] = w[1 + d];
    W[(NV - 1) * PLANE + o] = w[4];
  };

  // x/y sweep on the converted plane in slot W: returns sum over x,y faces of (F_in - F_out) for the own cell
  auto sweep_xy = [&](const double* W, int rot, double (&acc)[5]) {
#pragma unroll
    for (int v = 0; v < 5; ++v) acc[v] = 0.0;
#pragma unroll 1
    for (int dir = 0; dir < 2; ++dir) {
      double* ex = exb + dir * C::EX;
      const int cn = 1 + dir, ct = 2 - dir;                  // normal / tangential velocity planes
      const int cnt = dir ? N : TY;                          // halo cells per side in this direction
      // special roles, rotated over the warps from plane to plane
      const int q = (t + 32 * ((rot + 2 * dir) % (TG / 32))) % TG;
      const bool is_hi = q < cnt, is_lo = (q >= cnt) && (q < 2 * cnt);
      const int qq = is_hi ? q : q - cnt;
      double Rown[5], Rhi[5];
      // ---- phase 1: slopes -> left/right states
#pragma unroll 1
      for (int pass = 0; pass < 2; ++pass) {
        if (pass == 1 && !(is_hi || is_lo)) break;
        // cell whose slope is taken: own cell, or halo cell -1 (lo) / N or TY (hi) of row/column qq
        int ci = i, cj = j;
        if (pass == 1) {
          if (dir == 0) { cj = qq; ci = is_hi ? N : -1; } else { ci = qq; cj = is_hi ? TY : -1; }
        }
        int o0, om, op;
        if (dir == 0) {
          const int row = (cj + 2) * P;
          o0 = row + (ci < 0 ? ci + P : ci);
          om = row + (ci - 1 < 0 ? ci - 1 + P : ci - 1);
          op = row + ci + 1;   // ci+1 <= N+1: natural slot
        } else {
          o0 = (cj + 2) * P + ci;
          om = o0 - P;
          op = o0 + P;
        }
        double Lst[5], Rst[5];
        const int vmap[5] = {0, cn, ct, 3, NV - 1};
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          if (DIM == 2 && v == 3) { Lst[v] = 0.0; Rst[v] = 0.0; continue; }
          const double* Wv = W + vmap[v] * PLANE;
          double w0 = Wv[o0], wm = Wv[om], wp = Wv[op];
          double hs = half_slope(w0 - wm, wp - w0, limiter);
          Lst[v] = w0 + hs;
          Rst[v] = w0 - hs;
        }
        // left state of face f is stored at ex[f]: x: f = ci+1 in row cj; y: f = cj+1 in column ci
        const int fo = dir == 0 ? cj * (N + 1) + ci + 1 : (cj + 1) * N + ci;
        if (pass == 0) {
#pragma unroll
          for (int v = 0; v < 5; ++v) { Rown[v] = Rst[v]; if (!(DIM == 2 && v == 3)) ex[(v < 4 ? v : NV - 1) * EXV + fo] = Lst[v]; }
        } else if (is_lo) {
#pragma unroll
          for (int v = 0; v < 5; ++v) if (!(DIM == 2 && v == 3)) ex[(v < 4 ? v : NV - 1) * EXV + fo] = Lst[v];
        } else {
#pragma unroll
          for (int v = 0; v < 5; ++v) Rhi[v] = Rst[v];
        }
      }
      group_sync(bar_id, TG);
      // ---- phase 2: fluxes at the low face of the own cell (+ the last face of the row/column)
      double Fown[5];
#pragma unroll 1
      for (int pass = 0; pass < 2; ++pass) {
        if (pass == 1 && !is_hi) break;
        const int fo = pass == 0 ? (dir == 0 ? j * (N + 1) + i : j * N + i)
                                 : (dir == 0 ? qq * (N + 1) + N : TY * N + qq);
        double Lst[5], Rst[5], F[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          Lst[v] = (DIM == 2 && v == 3) ? 0.0 : ex[(v < 4 ? v : NV - 1) * EXV + fo];
          Rst[v] = pass == 0 ? Rown[v] : Rhi[v];
        }
        riemann_flux<DIM>(Lst, Rst, gamma, ig1, fluxs, F);
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          if (!(DIM == 2 && v == 3)) ex[(v < 4 ? v : NV - 1) * EXV + fo] = F[v];
          if (pass == 0) Fown[v] = F[v];
        }
      }
      group_sync(bar_id, TG);
      // ---- phase 3: difference with the next face
      {
        const int fn = dir == 0 ? j * (N + 1) + i + 1 : (j + 1) * N + i;
        const double d0 = Fown[0] - ex[0 * EXV + fn];
        const double dn = Fown[1] - ex[1 * EXV + fn];
        const double dt = Fown[2] - ex[2 * EXV + fn];
        const double de = Fown[4] - ex[(NV - 1) * EXV + fn];
        acc[0] += d0;
        acc[1] += dir == 0 ? dn : dt;
        acc[2] += dir == 0 ? dt : dn;
        if (DIM == 3) acc[3] += Fown[3] - ex[3 * EXV + fn];
        acc[4] += de;
      }
    }
  };

  // Runge-Kutta combine eq. (5) + store + optional CFL rate of the new state
  double rate_max = 0.0;
  auto finish = [&](int k, const double (&tot)[5]) {
    if (!active) return;
    const size_t o = (size_t)blk * C::BS + (size_t)(DIM == 3 ? k : 0) * P * P + (size_t)(j0 + j) * P + i;
    double u[5];
    const double s = p.dt_sub * inv_dx;
#pragma unroll
    for (int v = 0; v < NV; ++v) {
      const int tv = (v == NV - 1) ? 4 : v;
      double base = p.w0 * p.prev0[o + v * C::VS];
      if (p.prev1) base = fma(p.w1, p.prev1[o + v * C::VS], base);
      u[tv] = fma(s, tot[tv], base);
      p.out[o + v * C::VS] = u[tv];
    }
    if (p.maxrate) {
      double ir = rcp_fast(u[0]);
      double ke = 0.0, su = 0.0;
#pragma unroll
      for (int d = 0; d < DIM; ++d) {
        double vel = u[1 + d] * ir;
        ke = fma(vel, vel, ke);
        su += fabs(vel);
      }
      double pr = gm1 * fma(-0.5 * u[0], ke, u[4]);
      double c2 = gamma * pr * ir;
      double c = c2 * rsqrt_fast(c2);
      rate_max = fmax(rate_max, (su + DIM * c) * inv_dx);
    }
  };

  if (DIM == 2) {
    if (t == 0 && active) issue_plane(0);
    if (active) mbar_wait(&bars[0], 0);
    double w[5];
    if (active) {
      convert(ring, (j + 2) * P + i, w);
      if (t < C::HALO) {
        int row, col;
        if (t < 4 * TY) { row = 2 + t / 4; col = N + (t % 4); }
        else { int tq = t - 4 * TY, r4 = tq / N; row = r4 < 2 ? r4 : TY + r4; col = tq % N; }
        convert(ring, row * P + col, w);
      }
    }
    group_sync(bar_id, TG);
    double acc[5];
    sweep_xy(ring, 0, acc);
    finish(0, acc);
  } else {
    double dA[5], Lz[5], accp[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) { dA[v] = 0.0; Lz[v] = 0.0; accp[v] = 0.0; }
    if (t == 0 && active) issue_plane(-2);
#pragma unroll 1
    for (int c = -2; c <= N + 1; ++c) {
      const int idx = c + 2, s = idx % 3;
      double* Wc = ring + s * C::SLOT;                    // plane c
      const double* Wk = ring + ((idx + 2) % 3) * C::SLOT;  // plane c-1
      if (t == 0 && active && c + 1 <= N + 1) issue_plane(c + 1);
      double wB[5];
      if (active) {
        mbar_wait(&bars[s], (idx / 3) & 1);
        convert(Wc, (j + 2) * P + i, wB);
        if (c >= 0 && c < N && t < C::HALO) {
          int row, col;
          if (t < 4 * TY) { row = 2 + t / 4; col = N + (t % 4); }
          else { int tq = t - 4 * TY, r4 = tq / N; row = r4 < 2 ? r4 : TY + r4; col = tq % N; }
          double tmp[5];
          convert(Wc, row * P + col, tmp);
        }
      } else {
#pragma unroll
        for (int v = 0; v < 5; ++v) wB[v] = 1.0;
      }
      // ---- z direction along the march (frame: normal = w, tangentials u, v):
      //      slope of cell c-1 from w(c-2), w(c-1), w(c); flux at the face between cells c-2 and c-1
      double Fz[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
      if (c >= -1) {
        const int own = (j + 2) * P + i;
        double Rz[5], Ln[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
          const int pv = (v == 1) ? 3 : (v == 2 ? 1 : (v == 3 ? 2 : v));
          const double wa = Wk[pv * PLANE + own];   // w(c-1), resident in its ring slot
          const double dB = wB[pv] - wa;
          const double hs = half_slope(dA[v], dB, limiter);  // c == -1: dA = 0 -> hs = 0, result unused
          Rz[v] = wa - hs;
          Ln[v] = wa + hs;
          dA[v] = dB;
        }
        if (c >= 1) riemann_flux<3>(Lz, Rz, gamma, ig1, fluxs, Fz);
#pragma unroll
        for (int v = 0; v < 5; ++v) Lz[v] = Ln[v];
      }
      if (c >= 2) {
        double tot[5];
        tot[0] = accp[0] - Fz[0];
        tot[1] = accp[1] - Fz[2];   // Fz frame (mass, w, u, v, E) -> (rho, u, v, w, E)
        tot[2] = accp[2] - Fz[3];
        tot[3] = accp[3] - Fz[1];
        tot[4] = accp[4] - Fz[4];
        finish(c - 2, tot);
      }
      if (c >= 1 && c <= N) {
        double acc[5];
        sweep_xy(Wk, c, acc);
        accp[0] = acc[0] + Fz[0];
        accp[1] = acc[1] + Fz[2];
        accp[2] = acc[2] + Fz[3];
        accp[3] = acc[3] + Fz[1];
        accp[4] = acc[4] + Fz[4];
      }
      fence_proxy_async();
      group_sync(bar_id, TG);
    }
  }

  if (p.maxrate) {
    for (int sft = 16; sft > 0; sft >>= 1) rate_max = fmax(rate_max, __shfl_xor_sync(0xffffffffu, rate_max, sft));
    if ((threadIdx.x & 31) == 0 && rate_max > 0.0)
      atomicMax(p.maxrate, (unsigned long long)__double_as_longlong(rate_max));
  }
}

template <int DIM, int N, int TY, int G>
cudaError_t launch_cfg(const StageParams& p, cudaStream_t s) {
  using C = Cfg<DIM, N, TY, G>;
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(stage_kernel<DIM, N, TY, G>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)C::SMEM);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  const int nitems = p.nblocks * C::YT;
  const int grid = (nitems + G - 1) / G;
  stage_kernel<DIM, N, TY, G><<<grid, C::NT, C::SMEM, s>>>(p);
  return cudaGetLastError();
}

}  // namespace

bool stage_supported(int dim, int n) {
  return (dim == 2 && (n == 8 || n == 16)) || (dim == 3 && (n == 8 || n == 16 || n == 32));
}

cudaError_t launch_stage(int dim, int n, const StageParams& p, cudaStream_t s) {
  if (p.nblocks <= 0) return cudaSuccess;
  if (dim == 2 && n == 8) return launch_cfg<2, 8, 8, 4>(p, s);
  if (dim == 2 && n == 16) return launch_cfg<2, 16, 16, 1>(p, s);
  if (dim == 3 && n == 8) return launch_cfg<3, 8, 8, 4>(p, s);
  if (dim == 3 && n == 16) return launch_cfg<3, 16, 16, 1>(p, s);
  if (dim == 3 && n == 32) return launch_cfg<3, 32, 8, 1>(p, s);
  return cudaErrorInvalidValue;
}

}  // namespace f4
