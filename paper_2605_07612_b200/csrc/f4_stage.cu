// Fused finite-volume stage kernel (sm_100a): one Runge-Kutta sub-step eq. (5)
//   u(s_out) = dt_sub * F(u(s_deriv)) + w0 u(s_prev0) + w1 u(s_prev1)
// over every block, F = -div of HLL fluxes of
// limited primitive reconstructions, optional
// fused CFL max of the NEW state, fused same-level ghost copy
// (PAPER.md:195, 235-238): y ghost rows and z ghost planes of s_deriv are fetched
// from the same-level neighbours' interior cells, the x face layers of the new
// state are pushed into the neighbours' x ghost cells.
//
// Design (differs from the paper's gang-per-block / collapse(3) OpenACC loop,
// PAPER.md:162-189, which converts the whole block to uu_prim in global
// memory and evaluates every face flux twice):
//  * a thread group of N x TY threads owns a (block, y-tile) and marches
//    through the z planes; every face flux is evaluated once;
//  * padded planes of the conservative state are fetched by bulk async copies
//    (cp.async.bulk, the TMA engine, completion on an mbarrier) into a 4-slot (3 where two CTAs per SM would not fit otherwise)
//    shared-memory ring two planes ahead of use, and converted to primitives in
//    place (to_primitive once per cell); when the tile is the
//    whole block the smem plane keeps the store's wrapped row order, so one
//    bulk copy per variable moves the interior rows of a plane and two more
//    bring the ghost rows (from the +-y neighbours when they are same-level);
//  * x/y fluxes exchange reconstructed states and fluxes through shared
//    memory; the z direction lives in registers along the march;
//  * fp64 division / sqrt are replaced by MUFU seeds + cubic Newton steps, and
//    1/(S+ - S-) of the HLL flux by 1/(2 d^) = rsqrt(d^2)/2 (already at hand)
//    with the supersonic cases selected by sign bits: the kernel is co-limited
//    by the fp64 pipe and by dependent-issue latency.
#include <type_traits>

#include "../../include/f4.h"
#include "f4_dev.hpp"
#include "f4_stage_dev.cuh"

namespace f4 {
namespace {

__device__ __forceinline__ void sweep_sync(int id, int nthreads) { group_sync(id, nthreads); }

// HLL / Rusanov flux in the face-normal frame (readings A2-A3).
// q = (rho, un, ut1, ut2, p); F = (mass, normal momentum, tangential momenta, energy).
template <int DIM, bool FAST>
__device__ __forceinline__ void riemann_flux(const double (&L)[5], const double (&R)[5], double gamma, double ig1,
                                             int flux, double (&F)[5]) {
  // Roe weights from ONE rsqrt: z = 1/sqrt(rho_L rho_R), s = sqrt(rho_R/rho_L) = rho_R z, w_L = 1/(1+s), w_R = s w_L
  const double z = rsqrt_fast(L[0] * R[0]);
  const double sr = R[0] * z;
  const double wl = rcp_fast(1.0 + sr), wr = sr * wl;
  const double uhat = fma(wl, L[1], wr * R[1]);
  const double du = R[1] - L[1];
  // d^2 = (rL cL^2 + rR cR^2)/(rL+rR) + 1/2 wL wR du^2,  r c^2 = gamma p / sqrt(rho):
  //   (pL/rL + pR/rR)/(rL+rR) = wL z (pL s + pR)   (1/rho_L = z s, 1/(rL rR) = z)
  const double d2 = fma((0.5 * wl) * wr, du * du, fma(L[4], sr, R[4]) * ((wl * z) * gamma));
  const double y2 = rsqrt_fast(d2);
  // F = a FL + b FR + c (UR - UL) with a = S+/(S+ - S-), b = -S-/(S+ - S-), c = S+ S-/(S+ - S-)
  double a, b, c;
  if (FAST) {
    // HLL: S- = min(u^ - d^, 0), S+ = max(u^ + d^, 0).  Subsonic: S+ - S- = 2 d^ and 1/(2 d^) = y2/2 (no second
    // reciprocal), so a = 1/2 + u^/(2 d^); supersonic: (a,b,c) = (1,0,0) or (0,1,0).  Both cases:
    //   a = clamp(1/2 + u^ y2/2, 0, 1), b = 1 - a, c = -a b (2 d^);  the clamp is taken on the high word (no fp64 compare)
    const double a0 = fma(uhat, 0.5 * y2, 0.5);
    const int ah = __double2hiint(a0);
    const bool neg = ah < 0, big = ah >= 0x3FF00000;
    a = __hiloint2double(neg ? 0 : (big ? 0x3FF00000 : ah), (neg || big) ? 0 : __double2loint(a0));
    b = 1.0 - a;
    c = (a * b) * (d2 * (-2.0 * y2));
  } else {
    const double dhat = d2 * y2;
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
    a = sp * inv;
    b = -sm * inv;
    c = a * sm;
  }
  // regrouped per side: beta_L = a uL - c, beta_R = b uR + c, alpha = rho beta;  mass = alpha_L + alpha_R,
  //   momentum = alpha u (+ a pL + b pR for the normal component), energy = alpha h + p (beta/(gamma-1) + a u)
  //   with h = |u|^2/2  (eq. 14-15)
  const double auL = a * L[1], buR = b * R[1];
  const double bL = auL - c, bR = buR + c;
  const double aL = L[0] * bL, aR = R[0] * bR;
  double hL = fma(L[1], L[1], L[2] * L[2]), hR = fma(R[1], R[1], R[2] * R[2]);
  if (DIM == 3) { hL = fma(L[3], L[3], hL); hR = fma(R[3], R[3], hR); }
  F[0] = aL + aR;
  F[1] = fma(aL, L[1], fma(aR, R[1], fma(a, L[4], b * R[4])));
  F[2] = fma(aL, L[2], aR * R[2]);
  F[3] = (DIM == 3) ? fma(aL, L[3], aR * R[3]) : 0.0;
  F[4] = fma(0.5, fma(aL, hL, aR * hR), fma(L[4], fma(bL, ig1, auL), R[4] * fma(bR, ig1, buR)));
}

// Two independent HLL fluxes (van Leer/HLL fast path) written step by step across both faces, so that the
// rsqrt -> rcp -> rsqrt dependency chains of the two Riemann problems overlap (the kernel is bound by
// dependent-issue latency, not by instruction count).  Same arithmetic as riemann_flux<DIM, true>.
template <int DIM, int NF>
__device__ __forceinline__ void riemann_fluxN(const double (&L)[NF][5], const double (&R)[NF][5], double gamma,
                                              double ig1, double (&F)[NF][5]) {
  double qq[NF], z[NF], sr[NF], x[NF], wl[NF];
#pragma unroll
  for (int f = 0; f < NF; ++f) qq[f] = L[f][0] * R[f][0];
#pragma unroll
  for (int f = 0; f < NF; ++f) z[f] = rsqrt_seed(qq[f]);
#pragma unroll
  for (int f = 0; f < NF; ++f) z[f] = rsqrt_refine(qq[f], z[f]);   // 1/sqrt(rho_L rho_R)
#pragma unroll
  for (int f = 0; f < NF; ++f) { sr[f] = R[f][0] * z[f]; x[f] = 1.0 + sr[f]; }
#pragma unroll
  for (int f = 0; f < NF; ++f) wl[f] = rcp_seed(x[f]);
#pragma unroll
  for (int f = 0; f < NF; ++f) wl[f] = rcp_refine(x[f], wl[f]);
  double uhat[NF], d2[NF], y2[NF];
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    const double wr = sr[f] * wl[f];
    uhat[f] = fma(wl[f], L[f][1], wr * R[f][1]);
    const double du = R[f][1] - L[f][1];
    d2[f] = fma((0.5 * wl[f]) * wr, du * du, fma(L[f][4], sr[f], R[f][4]) * ((wl[f] * z[f]) * gamma));
  }
#pragma unroll
  for (int f = 0; f < NF; ++f) y2[f] = rsqrt_seed(d2[f]);
#pragma unroll
  for (int f = 0; f < NF; ++f) y2[f] = rsqrt_refine(d2[f], y2[f]);
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    const double a0 = fma(uhat[f], 0.5 * y2[f], 0.5);
    const int ah = __double2hiint(a0);
    const bool neg = ah < 0, big = ah >= 0x3FF00000;
    const double a = __hiloint2double(neg ? 0 : (big ? 0x3FF00000 : ah), (neg || big) ? 0 : __double2loint(a0));
    const double b = 1.0 - a;
    const double c = (a * b) * (d2[f] * (-2.0 * y2[f]));
    const double auL = a * L[f][1], buR = b * R[f][1];
    const double bL = auL - c, bR = buR + c;
    const double aL = L[f][0] * bL, aR = R[f][0] * bR;
    double hL = fma(L[f][1], L[f][1], L[f][2] * L[f][2]), hR = fma(R[f][1], R[f][1], R[f][2] * R[f][2]);
    if (DIM == 3) { hL = fma(L[f][3], L[f][3], hL); hR = fma(R[f][3], R[f][3], hR); }
    F[f][0] = aL + aR;
    F[f][1] = fma(aL, L[f][1], fma(aR, R[f][1], fma(a, L[f][4], b * R[f][4])));
    F[f][2] = fma(aL, L[f][2], aR * R[f][2]);
    F[f][3] = (DIM == 3) ? fma(aL, L[f][3], aR * R[f][3]) : 0.0;
    F[f][4] = fma(0.5, fma(aL, hL, aR * hR), fma(L[f][4], fma(bL, ig1, auL), R[f][4] * fma(bR, ig1, buR)));
  }
}

template <int DIM, int N, int TY, int G, int EXBUF>
struct Cfg {  // FAST (van Leer + HLL fixed at compile time) does not change the geometry
  static constexpr int P = N + 2 * NG;
  static constexpr int PZ = (DIM == 3) ? P : 1;
  static constexpr int NVAR = DIM + 2;
  static constexpr size_t VS = (size_t)P * P * PZ;
  static constexpr size_t BS = VS * NVAR;
  static constexpr bool WHOLE = (TY == N);    // the tile is the whole block plane: smem rows keep the wrapped slot order
  static constexpr int ROWS = TY + 4;
  static constexpr int PLANE = ROWS * P;      // doubles per variable in one ring slot
  static constexpr int SLOT = NVAR * PLANE;
  // ring depth: planes c-1 (swept), c (converted) and two in flight; all four are requested when the block starts, so
  // the DRAM latency of the first planes is paid once (with three slots every short prologue iteration waited for it)
  static constexpr size_t smem_for(int nslot) {
    return (size_t)G * (nslot * (NVAR * (TY + 4) * P) + 2 * EXBUF * (NVAR * (N + 1) * (TY + 1)) + EXBUF * NVAR * (TY + N)) * 8 +
           (size_t)G * (nslot + 2) * 8;
  }
  static constexpr size_t TWO_CTAS = 113 * 1024;   // two CTAs per SM: 2 x (SMEM + 1 KB reserved) <= 228 KB
  static constexpr int NSLOT = (DIM == 3) ? (smem_for(4) <= TWO_CTAS ? 4 : 3) : 1;
  static constexpr int EXV = (N + 1) * (TY + 1);  // exchange entries per variable
  static constexpr int EX = NVAR * EXV;
  static constexpr int NH = TY + N;           // halo cells per side (x rows + y columns)
  static constexpr int TG = N * TY;           // cell threads per group
  static constexpr int NT = TG * G;
  static constexpr int YT = N / TY;           // y tiles per block
  // ring | exX[EXBUF] | exY[EXBUF] | right states of the high halo cells [NVAR][NH]
  static constexpr int GROUP_DOUBLES = NSLOT * SLOT + 2 * EXBUF * EX + EXBUF * NVAR * NH;
  static constexpr int NBAR = NSLOT + 2;     // ring slots + "left states written" + "fluxes written"
  static constexpr size_t SMEM = (size_t)G * GROUP_DOUBLES * 8 + (size_t)G * NBAR * 8;
  static constexpr int HALO = 4 * TY + 4 * N;  // halo cells of an interior plane
  static_assert(HALO <= TG && 3 * NH <= TG, "halo work needs one pass");
  static_assert(TG % 32 == 0 && N % TY == 0 && GROUP_DOUBLES % 2 == 0, "tile shape");
};

// GEN: 0 = the path every BASELINE config takes; 1 = + gravity source term; 2 = + boundary-flux store (flux fixing)
// and a third / fourth previous state.
template <int DIM, int N, int TY, int G, int EXBUF, bool FAST, int GEN>
__global__ void __launch_bounds__(Cfg<DIM, N, TY, G, EXBUF>::NT, (Cfg<DIM, N, TY, G, EXBUF>::SMEM <= Cfg<DIM, N, TY, G, EXBUF>::TWO_CTAS) ? 2 : 1)
    stage_kernel(const __grid_constant__ StageParams p) {
  using C = Cfg<DIM, N, TY, G, EXBUF>;
  constexpr bool BF = (GEN == 2), GRAV = (GEN >= 1);
  constexpr int P = C::P, PP = C::P * C::P, NV = C::NVAR, PLANE = C::PLANE, TG = C::TG, EXV = C::EXV, NH = C::NH;
  constexpr bool WHOLE = C::WHOLE;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int grp = (G == 1) ? 0 : (int)threadIdx.x / TG;
  const int t = (G == 1) ? (int)threadIdx.x : (int)threadIdx.x % TG;
  const int item = blockIdx.x * G + grp;
  // a whole group leaves together: its named barrier and mbarriers are private to the group
  if (item >= p.nblocks * C::YT) return;
  const int blk = WHOLE ? item : item / C::YT;
  const int j0 = WHOLE ? 0 : (item % C::YT) * TY;
  const int i = t % N, j = t / N;

  double* ring = reinterpret_cast<double*>(smem_raw) + (size_t)grp * C::GROUP_DOUBLES;
  double* exX = ring + C::NSLOT * C::SLOT;   // [EXBUF][NV][EXV]
  double* exY = exX + EXBUF * C::EX;
  double* sRh0 = exY + EXBUF * C::EX;        // [EXBUF][NV][NH]
  uint64_t* bars = reinterpret_cast<uint64_t*>(reinterpret_cast<double*>(smem_raw) + (size_t)G * C::GROUP_DOUBLES) +
                   grp * C::NBAR;
  const uint32_t ring_u32 = smem_u32(ring), bars_u32 = smem_u32(bars);
  const int bar_id = 1 + grp;

  const double gamma = p.gamma, gm1 = gamma - 1.0, ig1 = 1.0 / gm1;
  const int limiter = p.limiter, fluxs = p.flux;
  const int lvl = p.level[blk];
  const size_t boff = (size_t)blk * C::BS;
  const double* dbase = p.deriv + boff;

  // register arrays are in "phys5" order (rho, u, v, w, p); smem plane of component q:
  auto pl = [](int q) { return q < 4 ? q : NV - 1; };
  // smem row of block row y (y in [j0-2, j0+TY+2)): the store's wrapped slot when the tile is the whole plane
  auto rown = [&](int y) { return WHOLE ? (y < 0 ? y + P : y) : y - j0 + 2; };

  if (t == 0) {
    for (int s = 0; s < C::NSLOT; ++s) mbar_init(&bars[s], 1);
    mbar_init(&bars[C::NSLOT], TG);       // every cell thread arrives once per plane
    mbar_init(&bars[C::NSLOT + 1], TG);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  group_sync(bar_id, TG);

  // Same-level z neighbours (fused ghost handling, a1 of the pattern): their interior planes ARE this block's z
  // ghost planes, so the march fetches planes -2,-1 / N,N+1 straight from the neighbour
  // block instead of from ghost cells somebody would have to write first.  -1: no same-level neighbour (physical
  // boundary, coarser or finer block): the block's own ghost planes, filled by the pattern executor, are read.
  // The same holds for the y ghost rows of an interior plane: rows N, N+1 are rows 0, 1 of the +y neighbour's
  // plane, rows -2, -1 are rows N-2, N-1 of the -y neighbour's (two more bulk copies per variable and plane).
  int gz0 = -1, gz1 = -1, gy0 = -1, gy1 = -1;
  if (DIM == 3 && p.nbr) { gz0 = p.nbr[(size_t)blk * 6 + 4]; gz1 = p.nbr[(size_t)blk * 6 + 5]; }
  if (p.nbr) { gy0 = p.nbr[(size_t)blk * 6 + 2]; gy1 = p.nbr[(size_t)blk * 6 + 3]; }
  // rows -2,-1 (slots P-2, P-1) and N, N+1 (slots N, N+1) of interior plane kslot: own ghost rows or the neighbours' rows
  const double* ylo_base = (gy0 >= 0) ? p.deriv + (size_t)gy0 * C::BS + (size_t)(N - 2) * P : dbase + (size_t)(P - 2) * P;
  const double* yhi_base = (gy1 >= 0) ? p.deriv + (size_t)gy1 * C::BS : dbase + (size_t)N * P;
  // issue the bulk copies of z plane c (c in [-2, N+2); 2D: c = 0) into ring slot s
  auto issue_plane = [&](int c, int s) {
    const bool interior = (DIM == 2) || (c >= 0 && c < N);
    const int kslot = (DIM == 3) ? (c < 0 ? c + P : c) : 0;
    const uint32_t dst = ring_u32 + (uint32_t)(s * C::SLOT) * 8u, bar = bars_u32 + 8u * s;
    const double* src = dbase + (size_t)kslot * PP;
    if (DIM == 3 && c < 0 && gz0 >= 0) src = p.deriv + (size_t)gz0 * C::BS + (size_t)(c + N) * PP;   // its planes N-2, N-1
    if (DIM == 3 && c >= N && gz1 >= 0) src = p.deriv + (size_t)gz1 * C::BS + (size_t)(c - N) * PP;  // its planes 0, 1
    if (WHOLE) {
      // interior plane: all P slot rows (N interior, 2 high, 2 low ghost rows); z-ghost plane: the N interior rows
      constexpr uint32_t bytes = (uint32_t)N * P * 8, gbytes = (uint32_t)2 * P * 8;
      mbar_expect_tx(bar, (bytes + (interior ? 2 * gbytes : 0u)) * NV);
#pragma unroll
      for (int v = 0; v < NV; ++v) bulk_g2s(dst + (uint32_t)(v * PLANE) * 8u, src + (size_t)v * C::VS, bytes, bar);
      if (interior) {
        const size_t ko = (size_t)kslot * PP;
#pragma unroll
        for (int v = 0; v < NV; ++v) {
          bulk_g2s(dst + (uint32_t)(v * PLANE + N * P) * 8u, yhi_base + ko + (size_t)v * C::VS, gbytes, bar);
          bulk_g2s(dst + (uint32_t)(v * PLANE + (P - 2) * P) * 8u, ylo_base + ko + (size_t)v * C::VS, gbytes, bar);
        }
      }
    } else {
      // rows y in [ylo, yhi) -> smem rows y - (j0-2); rows with y < 0 live in slots y + P
      const int ylo = interior ? j0 - 2 : j0, yhi = interior ? j0 + TY + 2 : j0 + TY;
      const int nlow = ylo < 0 ? -ylo : 0, nhigh = yhi > N ? yhi - N : 0;
      const uint32_t bytes_low = (uint32_t)nlow * P * 8, bytes_high = (uint32_t)nhigh * P * 8;
      const uint32_t bytes_mid = (uint32_t)(yhi - ylo - nlow - nhigh) * P * 8;
      mbar_expect_tx(bar, (bytes_low + bytes_mid + bytes_high) * NV);
      const size_t ko = (size_t)kslot * PP;
      for (int v = 0; v < NV; ++v) {
        const double* sv = src + (size_t)v * C::VS;
        const uint32_t dv = dst + (uint32_t)(v * PLANE) * 8u;
        // rows y < 0 and y >= N exist only in interior planes of the first / last tile (ghost rows, see above)
        if (nlow) bulk_g2s(dv + (uint32_t)((ylo - (j0 - 2)) * P) * 8u, ylo_base + ko + (size_t)v * C::VS, bytes_low, bar);
        bulk_g2s(dv + (uint32_t)((ylo + nlow - (j0 - 2)) * P) * 8u, sv + (size_t)(ylo + nlow) * P, bytes_mid, bar);
        if (nhigh) bulk_g2s(dv + (uint32_t)((N - (j0 - 2)) * P) * 8u, yhi_base + ko + (size_t)v * C::VS, bytes_high, bar);
      }
    }
  };

  // in-place conversion conservative -> primitive of one smem cell (to_primitive)
  auto convert = [&](double* W, int o, double (&w)[5]) {
    const double rho = W[o];
    const double ir = rcp_fast(rho);
    double ke = 0.0;
    w[0] = rho;
    w[3] = 0.0;
#pragma unroll
    for (int d = 0; d < DIM; ++d) {
      w[1 + d] = W[(1 + d) * PLANE + o] * ir;
      ke = fma(w[1 + d], w[1 + d], ke);
    }
    w[4] = gm1 * fma(-0.5 * rho, ke, W[(NV - 1) * PLANE + o]);
#pragma unroll
    for (int d = 0; d < DIM; ++d) W[(1 + d) * PLANE + o] = w[1 + d];
    W[(NV - 1) * PLANE + o] = w[4];
  };

  // limited reconstruction of one cell from its two neighbours along a line (offsets o0, om, op)
  // w0v: the cell's own primitives when the caller already holds them in registers (else read at offset o0)
  auto slope_states = [&](const double* W, int o0, int om, int op, double (&L)[5], double (&R)[5],
                          const double* w0v = nullptr) {
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      if (DIM == 2 && q == 3) { L[q] = 0.0; R[q] = 0.0; continue; }
      const double* Wv = W + pl(q) * PLANE;
      const double w0 = w0v ? w0v[q] : Wv[o0];
      const double da = w0 - Wv[om], db = Wv[op] - w0;
      const double hs = half_slope<FAST>(da, db, limiter);
      L[q] = w0 + hs;
      // Koren / WENO3 are not symmetric in (a, b): the slope towards the low face takes the arguments exchanged
      R[q] = w0 - ((!FAST && limiter >= F4_LIM_KOREN) ? half_slope<FAST>(db, da, limiter) : hs);
    }
  };

  // per-thread constants of the x/y sweep
  const int rr = rown(j0 + j);
  const int own = rr * P + i;
  const int own_ym = rown(j0 + j - 1) * P + i, own_yp = rown(j0 + j + 1) * P + i;
  // x ghosts are pair-transposed (f4_ghost.cu cell_off): ghost (N+g, row r) sits in row r&~1, (g-2, row r) in row r|1,
  // both at column N + 2*(r&1) + g  (smem rows have the parity of the store's slot rows)
  const int own_xm = (i == 0) ? (rr | 1) * P + N + 2 * (rr & 1) + 1 : own - 1;
  const int own_xp = (i == N - 1) ? (rr & ~1) * P + N + 2 * (rr & 1) : own + 1;
  const int fx = j * (N + 1) + i, fy = j * N + i;      // own low faces in the exchange arrays
  // ---- halo tasks (cells and faces outside the tile's own N x TY cells) are roles of the cell threads:
  //      [0,NH) high halo slopes, [NH,2NH) low halo slopes, [2NH,3NH) last-face fluxes, the last HALO threads
  //      convert the halo cells.  (A ninth helper warp looping over all of them was tried and removed, see Cfg.)
  // slope task h in [0, 2NH): high halo cell of row/column h (right state -> sRh), low halo cell h-NH (left state -> e)
  auto halo_slope_task = [&](const double* W, double* eX, double* eY, double* sRh, int h) {
    const bool hi = h < NH;
    const int hq = hi ? h : h - NH;
    const bool isx = hq < TY;                          // x halo of row hq, else y halo of column hq-TY
    int o0, om, op, f;
    if (isx) {
      const int r = rown(j0 + hq), gcol = N + 2 * (r & 1);
      o0 = hi ? (r & ~1) * P + gcol : (r | 1) * P + gcol + 1;   // cell N / cell -1
      om = hi ? r * P + N - 1 : o0 - 1;                         // cell N-1 / cell -2
      op = hi ? o0 + 1 : r * P;                                 // cell N+1 / cell 0
      f = hq * (N + 1);
    } else {
      const int col = hq - TY;
      const int y = hi ? j0 + TY : j0 - 1;                      // row TY / row -1 of the tile
      o0 = rown(y) * P + col;
      om = rown(y - 1) * P + col;
      op = rown(y + 1) * P + col;
      f = col;
    }
    double L[5], R[5];
    slope_states(W, o0, om, op, L, R);
    double* e = isx ? eX : eY;
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      if (DIM == 2 && q == 3) continue;
      if (!hi) e[pl(q) * EXV + f] = L[q];
      else sRh[pl(q) * NH + hq] = R[q];
    }
  };
  // flux task fq in [0, NH): the last face of row fq (x) or of column fq-TY (y)
  auto halo_flux_task = [&](double* eX, double* eY, const double* sRh, int fq) {
    const bool f_isx = fq < TY;
    const int f_f = f_isx ? fq * (N + 1) + N : TY * N + (fq - TY);
    double* e = f_isx ? eX : eY;
    double L[5], Rr[5], F[5];
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      L[q] = (DIM == 2 && q == 3) ? 0.0 : e[pl(q) * EXV + f_f];
      Rr[q] = (DIM == 2 && q == 3) ? 0.0 : sRh[pl(q) * NH + fq];
    }
    const double Ln[5] = {L[0], f_isx ? L[1] : L[2], f_isx ? L[2] : L[1], L[3], L[4]};
    const double Rn[5] = {Rr[0], f_isx ? Rr[1] : Rr[2], f_isx ? Rr[2] : Rr[1], Rr[3], Rr[4]};
    riemann_flux<DIM, FAST>(Ln, Rn, gamma, ig1, fluxs, F);
    const double Fp[5] = {F[0], f_isx ? F[1] : F[2], f_isx ? F[2] : F[1], F[3], F[4]};
#pragma unroll
    for (int q = 0; q < 5; ++q) if (!(DIM == 2 && q == 3)) e[pl(q) * EXV + f_f] = Fp[q];
  };
  // conversion task th in [0, HALO): x halo cells (4 per row), then the two rows below and above the tile
  auto halo_convert_task = [&](double* W, int th) {
    int o;
    if (th < 4 * TY) o = rown(j0 + th / 4) * P + N + (th % 4);
    else {
      const int tq = th - 4 * TY, r4 = tq / N;
      o = rown(r4 < 2 ? j0 - 2 + r4 : j0 + TY + r4 - 2) * P + tq % N;
    }
    double tmp[5];
    convert(W, o, tmp);
  };
  const bool is_hs = t < 2 * NH;
  const bool is_hf = (t >= 2 * NH) && (t < 3 * NH);
  const int th = t - (TG - C::HALO);
  constexpr bool HF3 = (NH % 32 == 0);   // the last-face flux warp is a whole warp
  const bool is_hc = th >= 0 && th < C::HALO;

  // flux fixing: slots of this block's faces at refinement boundaries (BF instances only)
  int bfs[6] = {-1, -1, -1, -1, -1, -1};
  if (BF && p.bfslot) {
#pragma unroll
    for (int f = 0; f < 2 * DIM; ++f) bfs[f] = p.bfslot[(size_t)blk * 6 + f];
  }
  constexpr int BFS = N * ((DIM == 3) ? N : 1);   // cell faces of one block face
  auto bf_store = [&](int slot, const double (&F)[5], int t1, int t2) {
    double* d = p.bflux + (size_t)slot * NV * BFS + t2 * N + t1;
#pragma unroll
    for (int q = 0; q < 5; ++q) if (!(DIM == 2 && q == 3)) d[pl(q) * BFS] = F[q];
  };
  // x/y sweep on the converted plane W (z index kk): sum over the x,y faces of (F_in - F_out) of the own cell
  // SPLIT (3D march, double-buffered exchange): both barriers of the x/y exchange are split into an arrive and a
  // wait on an mbarrier with exchange-independent work in between, so that a warp that is late delays the others only
  // by what exceeds that work: the z slope / z flux / Runge-Kutta combine and store of the finished plane between
  // arrive and wait of "left states written", phase 1 of the NEXT plane between arrive and wait of "fluxes written".
  constexpr bool SPLIT = DIM == 3 && EXBUF == 2;
  uint32_t xph = 0;   // phase parity of the two exchange mbarriers
  const uint32_t barL = bars_u32 + 8u * C::NSLOT, barF = barL + 8u;
  // The x/y sweep of one converted plane W (z index kk, exchange buffers of parity par) in three phases:
  //   1: slopes -> left states to shared memory, right states stay in registers
  //   2: flux at the low x and y face of the own cell, and at the last face of each row / column
  //   3: difference with the next faces: acc = sum over the x,y faces of (F_in - F_out) of the own cell
  auto phase1 = [&](const double* W, int par, double (&Rx)[5], double (&Ry)[5], const double* w0v = nullptr) {
    double* eX = exX + (EXBUF == 2 ? par : 0) * C::EX;
    double* eY = exY + (EXBUF == 2 ? par : 0) * C::EX;
    double* sRh = sRh0 + (EXBUF == 2 ? par : 0) * NV * NH;
    {  // ---- phase 1: slopes -> left states to smem, right states stay in registers
      double L[5], w0[5];
#pragma unroll
      for (int q = 0; q < 5; ++q) w0[q] = (DIM == 2 && q == 3) ? 0.0 : (w0v ? w0v[q] : W[pl(q) * PLANE + own]);   // read once
      slope_states(W, own, own_xm, own_xp, L, Rx, w0);
#pragma unroll
      for (int q = 0; q < 5; ++q) if (!(DIM == 2 && q == 3)) eX[pl(q) * EXV + fx + 1] = L[q];
      slope_states(W, own, own_ym, own_yp, L, Ry, w0);
#pragma unroll
      for (int q = 0; q < 5; ++q) if (!(DIM == 2 && q == 3)) eY[pl(q) * EXV + fy + N] = L[q];
      if (is_hs) halo_slope_task(W, eX, eY, sRh, t);
    }
  };
  auto phase2 = [&](int par, int kk, const double (&Rx)[5], const double (&Ry)[5], double (&Fx)[5], double (&Fy)[5]) {
    double* eX = exX + (EXBUF == 2 ? par : 0) * C::EX;
    double* eY = exY + (EXBUF == 2 ? par : 0) * C::EX;
    double* sRh = sRh0 + (EXBUF == 2 ? par : 0) * NV * NH;
    {  // ---- phase 2: flux at the low x and y face of the own cell, and at the last face of each row/column
      double L[5], F[5];
      if (FAST) {
        // x and y faces together (riemann_flux2); y in its normal frame (rho, v, u, w, p)
        double L2[2][5], R2[2][5], F2[2][5];
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          L2[0][q] = (DIM == 2 && q == 3) ? 0.0 : eX[pl(q) * EXV + fx];
          L[q] = (DIM == 2 && q == 3) ? 0.0 : eY[pl(q) * EXV + fy];
          R2[0][q] = Rx[q];
        }
        L2[1][0] = L[0]; L2[1][1] = L[2]; L2[1][2] = L[1]; L2[1][3] = L[3]; L2[1][4] = L[4];
        R2[1][0] = Ry[0]; R2[1][1] = Ry[2]; R2[1][2] = Ry[1]; R2[1][3] = Ry[3]; R2[1][4] = Ry[4];
        if (HF3 && is_hf) {
          // the warp that also owns the last-face fluxes of this plane solves its three Riemann problems together:
          // the extra dependency chain overlaps with the other two instead of following them (the other warps wait
          // for this one at the barrier below)
          const int fq = t - 2 * NH;
          const bool f_isx = fq < TY;
          const int f_f = f_isx ? fq * (N + 1) + N : TY * N + (fq - TY);
          double* e = f_isx ? eX : eY;
          double L3[3][5], R3[3][5], F3[3][5], Lh[5], Rh[5];
#pragma unroll
          for (int q = 0; q < 5; ++q) {
            L3[0][q] = L2[0][q]; L3[1][q] = L2[1][q]; R3[0][q] = R2[0][q]; R3[1][q] = R2[1][q];
            Lh[q] = (DIM == 2 && q == 3) ? 0.0 : e[pl(q) * EXV + f_f];
            Rh[q] = (DIM == 2 && q == 3) ? 0.0 : sRh[pl(q) * NH + fq];
          }
          L3[2][0] = Lh[0]; L3[2][1] = f_isx ? Lh[1] : Lh[2]; L3[2][2] = f_isx ? Lh[2] : Lh[1]; L3[2][3] = Lh[3]; L3[2][4] = Lh[4];
          R3[2][0] = Rh[0]; R3[2][1] = f_isx ? Rh[1] : Rh[2]; R3[2][2] = f_isx ? Rh[2] : Rh[1]; R3[2][3] = Rh[3]; R3[2][4] = Rh[4];
          riemann_fluxN<DIM, 3>(L3, R3, gamma, ig1, F3);
#pragma unroll
          for (int q = 0; q < 5; ++q) { F2[0][q] = F3[0][q]; F2[1][q] = F3[1][q]; }
          const double Fp[5] = {F3[2][0], f_isx ? F3[2][1] : F3[2][2], f_isx ? F3[2][2] : F3[2][1], F3[2][3], F3[2][4]};
#pragma unroll
          for (int q = 0; q < 5; ++q) if (!(DIM == 2 && q == 3)) e[pl(q) * EXV + f_f] = Fp[q];
        } else {
          riemann_fluxN<DIM, 2>(L2, R2, gamma, ig1, F2);
        }
#pragma unroll
        for (int q = 0; q < 5; ++q) Fx[q] = F2[0][q];
        Fy[0] = F2[1][0]; Fy[1] = F2[1][2]; Fy[2] = F2[1][1]; Fy[3] = F2[1][3]; Fy[4] = F2[1][4];
      } else {
#pragma unroll
        for (int q = 0; q < 5; ++q) L[q] = (DIM == 2 && q == 3) ? 0.0 : eX[pl(q) * EXV + fx];
        riemann_flux<DIM, FAST>(L, Rx, gamma, ig1, fluxs, Fx);
        // y: normal frame (rho, v, u, w, p)
#pragma unroll
        for (int q = 0; q < 5; ++q) L[q] = (DIM == 2 && q == 3) ? 0.0 : eY[pl(q) * EXV + fy];
        {
          const double Ln[5] = {L[0], L[2], L[1], L[3], L[4]}, Rn[5] = {Ry[0], Ry[2], Ry[1], Ry[3], Ry[4]};
          riemann_flux<DIM, FAST>(Ln, Rn, gamma, ig1, fluxs, F);
        }
        Fy[0] = F[0]; Fy[1] = F[2]; Fy[2] = F[1]; Fy[3] = F[3]; Fy[4] = F[4];
      }
#pragma unroll
      for (int q = 0; q < 5; ++q) if (!(DIM == 2 && q == 3)) eX[pl(q) * EXV + fx] = Fx[q];
#pragma unroll
      for (int q = 0; q < 5; ++q) if (!(DIM == 2 && q == 3)) eY[pl(q) * EXV + fy] = Fy[q];
      if (is_hf && !(FAST && HF3)) halo_flux_task(eX, eY, sRh, t - 2 * NH);
      if (BF) {
        if (i == 0 && bfs[0] >= 0) bf_store(bfs[0], Fx, j0 + j, kk);
        if (j0 + j == 0 && bfs[2] >= 0) bf_store(bfs[2], Fy, i, kk);
      }
    }
  };
  auto phase3 = [&](int par, int kk, const double (&Fx)[5], const double (&Fy)[5], double (&acc)[5]) {
    double* eX = exX + (EXBUF == 2 ? par : 0) * C::EX;
    double* eY = exY + (EXBUF == 2 ? par : 0) * C::EX;
    // ---- phase 3: difference with the next faces
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      if (DIM == 2 && q == 3) { acc[q] = 0.0; continue; }
      acc[q] = (Fx[q] - eX[pl(q) * EXV + fx + 1]) + (Fy[q] - eY[pl(q) * EXV + fy + N]);
    }
    if (BF) {
      if (i == N - 1 && bfs[1] >= 0) {
        double Fh[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) Fh[q] = (DIM == 2 && q == 3) ? 0.0 : eX[pl(q) * EXV + fx + 1];
        bf_store(bfs[1], Fh, j0 + j, kk);
      }
      if (j0 + j == N - 1 && bfs[3] >= 0) {
        double Fh[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) Fh[q] = (DIM == 2 && q == 3) ? 0.0 : eY[pl(q) * EXV + fy + N];
        bf_store(bfs[3], Fh, i, kk);
      }
    }
  };
  // the three phases with a group barrier in between (2D, single exchange buffer)
  auto sweep_xy = [&](const double* W, int par, int kk, double (&acc)[5]) {
    double Rx[5], Ry[5], Fx[5], Fy[5];
    phase1(W, par, Rx, Ry);
    sweep_sync(bar_id, TG);
    phase2(par, kk, Rx, Ry, Fx, Fy);
    sweep_sync(bar_id, TG);
    phase3(par, kk, Fx, Fy, acc);
    if (EXBUF == 1) sweep_sync(bar_id, TG);
  };

  // Runge-Kutta combine eq. (5) + store + optional CFL rate of the new state
  double rate_max = 0.0;
  // dt_sub and dt_sub / dx of this block's level: from the host, or from the time step resident on the device
  const double dt_sub = p.dt_dev ? p.dtf * *p.dt_dev : p.dt_sub;
  const double sdt = p.dt_dev ? dt_sub * p.inv_dx_l[lvl] : p.sdt_l[lvl];
  const int co = (j0 + j) * P + i;                          // own cell inside a (block, var) box, + k*PP + v*VS
  const double* pa = p.prev0 + boff + co;
  const double* pb = p.prev1 ? p.prev1 + boff + co : nullptr;
  double* po = p.out + boff + co;
  // fused same-level ghost fill: boundary layers are pushed from registers into the neighbours' ghost cells
  // (a1 of the pattern).  nbr[f] = same-level neighbour across face f, or -1.
  double* ppx = nullptr;   // x push target of this thread (k = 0, var 0); y and z ghosts are gathered by the reader
  if (p.nbr && p.push_x) {
    const int* nb = p.nbr + (size_t)blk * 6;
    const int jg = j0 + j;
    if (i < NG && nb[0] >= 0) ppx = p.out + (size_t)nb[0] * C::BS + ((jg & ~1) * P + N + 2 * (jg & 1) + i);
    if (i >= N - NG && nb[1] >= 0) ppx = p.out + (size_t)nb[1] * C::BS + ((jg | 1) * P + N + 2 * (jg & 1) + (i - (N - NG)));
  }
  // general instances (BF): up to four previous states in eq. (5) (classical RK4, eq. (11));
  // the third and fourth are folded into b: b <- b + (w2 c + w3 d) / w1 is avoided by carrying w1 b + w2 c + w3 d
  const double* pc = (BF && p.prev2) ? p.prev2 + boff + co : nullptr;
  const double* pd = (BF && p.prev3) ? p.prev3 + boff + co : nullptr;
  const double w1eff = (BF && pc) ? 1.0 : p.w1;
  auto load_prev = [&](int k, double (&a)[5], double (&b)[5]) {
    const int ko = (DIM == 3 ? k : 0) * PP;
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      if (DIM == 2 && q == 3) { a[q] = 0.0; b[q] = 0.0; continue; }
      a[q] = pa[ko + pl(q) * (int)C::VS];
      b[q] = pb ? pb[ko + pl(q) * (int)C::VS] : 0.0;
      if (BF && pc) {
        double e = p.w1 * b[q];
        e = fma(p.w2, pc[ko + pl(q) * (int)C::VS], e);
        if (pd) e = fma(p.w3, pd[ko + pl(q) * (int)C::VS], e);
        b[q] = e;
      }
    }
  };
  auto finish = [&](int k, const double (&tot)[5], const double (&a)[5], const double (&b)[5]) {
    const int ko = (DIM == 3 ? k : 0) * PP;
    double u[5];
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      if (DIM == 2 && q == 3) { u[q] = 0.0; continue; }
      u[q] = fma(sdt, tot[q], fma(w1eff, b[q], p.w0 * a[q]));
    }
    if (GRAV && p.has_grav) {
      // source term of eq. (20), S = (0, rho g, rho g.u) = (0, rho g, g.m) of s_deriv in this cell
      // (PAPER.md:334 step i): its conservative values are one of the previous states already in registers
      // (grav_from 0 / 1) or are loaded (2: s_deriv is not among the first two previous states)
      double r0, mm[3] = {0.0, 0.0, 0.0};
      if (p.grav_from == 0) { r0 = a[0]; mm[0] = a[1]; mm[1] = a[2]; mm[2] = a[3]; }
      else if (p.grav_from == 1 && !(BF && pc)) { r0 = b[0]; mm[0] = b[1]; mm[1] = b[2]; mm[2] = b[3]; }
      else {
        const double* pg = p.deriv + boff + co + ko;
        r0 = pg[0];
#pragma unroll
        for (int d = 0; d < DIM; ++d) mm[d] = pg[(1 + d) * (int)C::VS];
      }
      double gm = 0.0;
#pragma unroll
      for (int d = 0; d < DIM; ++d) {
        u[1 + d] = fma(dt_sub * p.grav[d], r0, u[1 + d]);
        gm = fma(p.grav[d], mm[d], gm);
      }
      u[4] = fma(dt_sub, gm, u[4]);
    }
#pragma unroll
    for (int q = 0; q < 5; ++q) {
      if (DIM == 2 && q == 3) continue;
      po[ko + pl(q) * (int)C::VS] = u[q];
    }
    if (ppx) {
#pragma unroll
      for (int q = 0; q < 5; ++q) if (!(DIM == 2 && q == 3)) ppx[ko + pl(q) * (int)C::VS] = u[q];
    }
    if (p.maxrate) {
      const double ir = rcp_fast(u[0]);
      double ke = 0.0, su = 0.0;
#pragma unroll
      for (int d = 0; d < DIM; ++d) {
        const double vel = u[1 + d] * ir;
        ke = fma(vel, vel, ke);
        su += fabs(vel);
      }
      const double pr = gm1 * fma(-0.5 * u[0], ke, u[4]);
      const double c2 = gamma * pr * ir;
      // a cell that is not a valid gas state (NaN, rho <= 0, p <= 0) makes the maximum +inf: compute_dt reports it
      const double rate = fma((double)DIM, c2 * rsqrt_fast(c2), su);
      rate_max = fmax(rate_max, (u[0] > 0.0 && pr > 0.0 && rate == rate) ? rate : __longlong_as_double(0x7ff0000000000000LL));
    }
  };
  auto convert_halo = [&](double* W) {
    if (is_hc) halo_convert_task(W, th);
  };

  constexpr int ISSUER = (TG >= 128) ? 96 : 0;   // lane 0 of a warp without halo roles when the group has one
  if (DIM == 3 && t == ISSUER) {
    for (int q = 0; q < C::NSLOT; ++q) issue_plane(q - 2, q);
  }
  if (DIM == 2) {
    double a[5], b[5], w[5], acc[5];
    if (t == ISSUER) issue_plane(0, 0);
    load_prev(0, a, b);
    mbar_wait(bars_u32, 0);
    convert(ring, own, w);
    convert_halo(ring);
    group_sync(bar_id, TG);
    sweep_xy(ring, 0, 0, acc);
    finish(0, acc, a, b);
  } else {
    double dA[5], Lz[5], accp[5];
    double Rxp[5], Ryp[5];           // SPLIT: right states of the plane whose phase 1 ran ahead
#pragma unroll
    for (int q = 0; q < 5; ++q) { dA[q] = 0.0; Lz[q] = 1.0; accp[q] = 0.0; Rxp[q] = 1.0; Ryp[q] = 1.0; }
    constexpr int NS = C::NSLOT;
    int sc = 0;            // ring slot of plane c: (c + 2) % NS
    uint32_t ph = 0;       // phase parity of each slot's mbarrier
    // one march iteration; the steady state (c in [2, N]) is the instance with every flag true
    auto march = [&](int c, auto zslope_t, auto zflux_t, auto fin_t, auto sweep_t) {
      constexpr bool ZSLOPE = decltype(zslope_t)::value, ZFLUX = decltype(zflux_t)::value;
      constexpr bool FIN = decltype(fin_t)::value, SWEEP = decltype(sweep_t)::value;
      const int sk = (sc == 0) ? NS - 1 : sc - 1;           // slot of plane c-1
      double* Wc = ring + sc * C::SLOT;
      const double* Wk = ring + sk * C::SLOT;
      double Fz[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
      // the part of the iteration that does not depend on the x/y exchange of plane c-1 (see sweep_xy)
      double Rz[5], Lf[5];
      double pa5[5], pb5[5], wB[5];
      auto midA = [&]() {
      mbar_wait(bars_u32 + 8u * sc, (ph >> sc) & 1u);
      ph ^= 1u << sc;
      convert(Wc, own, wB);
      if (c >= 0 && c < N) convert_halo(Wc);
      fence_proxy_async();   // generic-proxy writes before the async-proxy refill of this slot
      // after the fence (it compiles to MEMBAR.ALL.CTA, which would wait for these loads): previous states of the
      // finished plane, consumed after the z flux
      if (FIN) load_prev(c - 2, pa5, pb5);
      if (FIN && pb && c - 1 < N && (i & 3) == 0) {         // stage 2: u_t of the next plane comes from DRAM: pull it into L2 now
#pragma unroll
        for (int q = 0; q < 5; ++q)
          asm volatile("prefetch.global.L2 [%0];" ::"l"(pa + (c - 1) * PP + pl(q) * (int)C::VS));
      }
      };   // midA
      auto midB = [&]() {
      // ---- z direction along the march: slope of cell c-1 from w(c-2), w(c-1), w(c);
      //      flux at the face between cells c-2 and c-1 (normal frame (rho, w, u, v, p))
      if (ZSLOPE) {
#pragma unroll
        for (int q = 0; q < 5; ++q) {
          const double wa = Wk[pl(q) * PLANE + own];   // w(c-1), resident in its ring slot
          const double dB = wB[q] - wa;
          const double hs = half_slope<FAST>(dA[q], dB, limiter);  // c == -1: dA = 0 -> hs = 0, result unused
          Rz[q] = wa - ((!FAST && limiter >= F4_LIM_KOREN) ? half_slope<FAST>(dB, dA[q], limiter) : hs);
          Lf[q] = Lz[q];                               // left state of the face between cells c-2 and c-1
          Lz[q] = wa + hs;
          dA[q] = dB;
        }
      }
      };   // midB
      auto mid2 = [&]() {
      if (ZSLOPE) {
        if (ZFLUX) {
          const double Lfn[5] = {Lf[0], Lf[3], Lf[1], Lf[2], Lf[4]}, Rf[5] = {Rz[0], Rz[3], Rz[1], Rz[2], Rz[4]};
          double F[5];
          riemann_flux<3, FAST>(Lfn, Rf, gamma, ig1, fluxs, F);
          Fz[0] = F[0]; Fz[3] = F[1]; Fz[1] = F[2]; Fz[2] = F[3]; Fz[4] = F[4];
          if (BF) {   // the face between cells c-2 and c-1 is the block's low (c = 1) / high (c = N+1) z face
            if (c == 1 && bfs[4] >= 0) bf_store(bfs[4], Fz, i, j0 + j);
            if (c == N + 1 && bfs[5] >= 0) bf_store(bfs[5], Fz, i, j0 + j);
          }
        }
      }
      if (FIN) {
        double tot[5];
#pragma unroll
        for (int q = 0; q < 5; ++q) tot[q] = accp[q] - Fz[q];
        finish(c - 2, tot, pa5, pb5);
      }
      };   // mid2
      if (SWEEP && SPLIT) {
        // Split barriers, software-pipelined by one plane: the left states of plane c-1 were written in the previous
        // iteration (phase 1 runs one plane ahead, between arrive and wait of the flux barrier); the z work sits
        // between arrive and wait of the left-state barrier.  A wait on barL also guarantees that every thread has
        // converted plane c, which is what phase 1 of plane c reads.
        if (c == 1) phase1(Wk, c & 1, Rxp, Ryp);
        midA();
        mbar_arrive(barL);
        midB();
        mid2();
        mbar_wait(barL, xph);
        double Fx[5], Fy[5], acc[5];
        phase2(c & 1, c - 1, Rxp, Ryp, Fx, Fy);
        mbar_arrive(barF);
        if (c < N) phase1(Wc, (c + 1) & 1, Rxp, Ryp, wB);   // own cell of plane c: still in registers
        mbar_wait(barF, xph);
        xph ^= 1u;
        phase3(c & 1, c - 1, Fx, Fy, acc);
#pragma unroll
        for (int q = 0; q < 5; ++q) accp[q] = acc[q] + Fz[q];
      } else if (SWEEP) {
        double acc[5];
        midA();
        midB();
        mid2();
        sweep_xy(Wk, c & 1, c - 1, acc);
#pragma unroll
        for (int q = 0; q < 5; ++q) accp[q] = acc[q] + Fz[q];
      } else {
        midA();
        midB();
        mid2();
        group_sync(bar_id, TG);
      }
      // every thread is past its last read of plane c-1: refill that slot with the next plane of the ring
      if (t == ISSUER && c >= -1 && c + NS - 1 <= N + 1) issue_plane(c + NS - 1, sk);
      sc = (sc == NS - 1) ? 0 : sc + 1;
    };
    using T = std::true_type;
    using F_ = std::false_type;
    march(-2, F_{}, F_{}, F_{}, F_{});
    march(-1, T{}, F_{}, F_{}, F_{});
    march(0, T{}, F_{}, F_{}, F_{});
    march(1, T{}, T{}, F_{}, T{});
#pragma unroll 1
    for (int c = 2; c <= N; ++c) march(c, T{}, T{}, T{}, T{});
    march(N + 1, T{}, T{}, T{}, F_{});
  }

  if (p.maxrate) {
    rate_max *= p.inv_dx_l[lvl];   // max over cells of sum_d (|u_d| + c), scaled by 1/dx (> 0) once
    for (int sft = 16; sft > 0; sft >>= 1) rate_max = fmax(rate_max, __shfl_xor_sync(0xffffffffu, rate_max, sft));
    if ((threadIdx.x & 31) == 0 && rate_max > 0.0)
      atomicMax(p.maxrate, (unsigned long long)__double_as_longlong(rate_max));
  }
}

template <int DIM, int N, int TY, int G, int EXBUF>
cudaError_t launch_cfg(const StageParams& p, cudaStream_t s) {
  using C = Cfg<DIM, N, TY, G, EXBUF>;
  const int nitems = p.nblocks * C::YT;
  const int grid = (nitems + G - 1) / G;
  const bool fast = p.limiter == F4_LIM_VANLEER && p.flux == F4_FLUX_HLL;
  // general instances (2): boundary-flux store (flux fixing) and / or > 2 previous states; (1): the configs' path +
  // gravity source term; (0): the configs' path
  const int gen = (p.bfslot || p.prev2) ? 2 : (p.has_grav ? 1 : 0);
  void (*k)(StageParams) =
      gen == 2 ? (fast ? stage_kernel<DIM, N, TY, G, EXBUF, true, 2> : stage_kernel<DIM, N, TY, G, EXBUF, false, 2>)
      : gen == 1 ? (fast ? stage_kernel<DIM, N, TY, G, EXBUF, true, 1> : stage_kernel<DIM, N, TY, G, EXBUF, false, 1>)
                 : (fast ? stage_kernel<DIM, N, TY, G, EXBUF, true, 0> : stage_kernel<DIM, N, TY, G, EXBUF, false, 0>);
  // the opt-in dynamic shared-memory size is an attribute of the function ON THE CURRENT DEVICE: set it before every
  // launch (a host-side call without synchronisation) instead of caching "done" per process
  cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
  if (e != cudaSuccess) return e;
  k<<<grid, C::NT, C::SMEM, s>>>(p);
  return cudaGetLastError();
}

}  // namespace

bool stage_supported(int dim, int n) {
  return (dim == 2 && (n == 8 || n == 16 || n == 32)) || (dim == 3 && (n == 8 || n == 16 || n == 32));
}

cudaError_t launch_stage(int dim, int n, const StageParams& p, cudaStream_t s) {
  if (p.nblocks <= 0) return cudaSuccess;
  if (dim == 2 && n == 8) return launch_cfg<2, 8, 8, 4, 1>(p, s);
  if (dim == 2 && n == 16) return launch_cfg<2, 16, 16, 1, 1>(p, s);
  if (dim == 2 && n == 32) return launch_cfg<2, 32, 8, 1, 1>(p, s);
  if (dim == 3 && n == 8) return launch_cfg<3, 8, 8, 4, 1>(p, s);      // four blocks per CTA
  if (dim == 3 && n == 16) return launch_cfg<3, 16, 16, 1, 2>(p, s);   // one block per CTA, double-buffered exchange
  if (dim == 3 && n == 32) return launch_cfg<3, 32, 8, 1, 2>(p, s);    // 32 x 8 tiles
  return cudaErrorInvalidValue;
}

}  // namespace f4
