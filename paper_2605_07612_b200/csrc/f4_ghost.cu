// Ghost-pattern executor, regrid transfer and layout kernels (sm_100a).
//
// Ghost pattern (section 2.6): ONE batched kernel per round,
// driven by a device-resident list of records (dst block, src block, face, op)
// sorted by destination block, instead of one OpenACC loop per boundary type
// and face direction.  A CTA takes 2*DIM consecutive
// records (= all faces of one block on a uniform mesh).  HBM-bound: 16-byte
// vector accesses, all loads of a thread issued before its stores; with the
// pair-transposed x-ghost layout (cell_off) two adjacent lanes write one full
// 32-byte ghost sector.  Inside f4_advance the SRL records are not executed
// here: the stage kernel pushes those layers itself (f4_stage.cu).
#include <mutex>

#include "../../include/f4.h"
#include "f4_dev.hpp"
#include "f4_stage_dev.cuh"

namespace f4 {
namespace {

// NV: variables per cell (Euler: DIM + 2; scalar advection eq. (13): 1)
template <int DIM, int N, int NV = DIM + 2>
struct Geo {
  static constexpr int P = N + 2 * NG;
  static constexpr int PZ = (DIM == 3) ? P : 1;
  static constexpr int NZ = (DIM == 3) ? N : 1;
  static constexpr int NVAR = NV;
  static constexpr int H = N / 2;
  static constexpr size_t VS = (size_t)P * P * PZ;   // doubles per (block, var)
  static constexpr size_t BS = VS * NVAR;            // doubles per block
  __host__ __device__ static constexpr int slot(int i) { return i < 0 ? i + P : i; }
};

__device__ __forceinline__ double2 ld2(const double* p) { return *reinterpret_cast<const double2*>(p); }
__device__ __forceinline__ void st2(double* p, double2 v) { *reinterpret_cast<double2*>(p) = v; }

// slot offset of cell (i,j,k) inside one (block,var) box
template <int DIM, int N>
__device__ __forceinline__ int cell_off(int i, int j, int k) {
  using G = Geo<DIM, N>;
  // x ghosts are pair-transposed: the 4 ghost slots of rows (2m, 2m+1) hold [hi(2m) hi(2m+1)] in row 2m and
  // [lo(2m) lo(2m+1)] in row 2m+1, so that each 32-byte ghost sector has a single source block
  const int sj = G::slot(j);
  int row = sj, col = i;
  if (i >= N) { row = sj & ~1; col = N + 2 * (sj & 1) + (i - N); }
  else if (i < 0) { row = sj | 1; col = N + 2 * (sj & 1) + (i + NG); }
  int o = row * G::P + col;
  if (DIM == 3) o += G::slot(k) * G::P * G::P;
  return o;
}

// generalised minmod, eq. (1)
__device__ __forceinline__ double minmod_g(double a, double b, double theta) {
  double m = fmin(fmin(fabs(theta * a), fabs(theta * b)), fabs(a + b) * 0.5);
  double r = (a > 0.0) ? m : -m;
  return (a * b <= 0.0) ? 0.0 : r;
}

// mean of the 2^d fine cells with lowest member (i0,j0,k0); pairwise x -> y -> z, adds only
// (reading A8): bit-exact by construction.  i0 is even, so each x pair is one 16-byte load.
template <int DIM, int N>
__device__ __forceinline__ double restrict_mean(const double* fv, int i0, int j0, int k0) {
  using G = Geo<DIM, N>;
  const double* p = fv + cell_off<DIM, N>(i0, j0, k0);
  double2 a = ld2(p), b = ld2(p + G::P);
  double s0 = __dadd_rn(__dadd_rn(a.x, a.y), __dadd_rn(b.x, b.y));
  if (DIM == 2) return __dmul_rn(s0, 0.25);
  double2 c = ld2(p + G::P * G::P), d = ld2(p + G::P * G::P + G::P);
  double s1 = __dadd_rn(__dadd_rn(c.x, c.y), __dadd_rn(d.x, d.y));
  return __dmul_rn(__dadd_rn(s0, s1), 0.125);
}

// limited slopes of coarse cell (ic,jc,kc): one-sided differences -> eq. (1)
template <int DIM, int N>
__device__ __forceinline__ void coarse_slopes(const double* cv, int ic, int jc, int kc, double theta, double& uc,
                                              double& sx, double& sy, double& sz) {
  uc = cv[cell_off<DIM, N>(ic, jc, kc)];
  sx = minmod_g(uc - cv[cell_off<DIM, N>(ic - 1, jc, kc)], cv[cell_off<DIM, N>(ic + 1, jc, kc)] - uc, theta);
  sy = minmod_g(uc - cv[cell_off<DIM, N>(ic, jc - 1, kc)], cv[cell_off<DIM, N>(ic, jc + 1, kc)] - uc, theta);
  sz = 0.0;
  if (DIM == 3)
    sz = minmod_g(uc - cv[cell_off<DIM, N>(ic, jc, kc - 1)], cv[cell_off<DIM, N>(ic, jc, kc + 1)] - uc, theta);
}
// child value u_c + (+-1/4 dx +- 1/4 dy) +- 1/4 dz, evaluated in that order (reading A9)
template <int DIM>
__device__ __forceinline__ double child_value(double uc, double sx, double sy, double sz, int px, int py, int pz) {
  double r = __dadd_rn(px ? 0.25 * sx : -0.25 * sx, py ? 0.25 * sy : -0.25 * sy);
  if (DIM == 3) r = __dadd_rn(r, pz ? 0.25 * sz : -0.25 * sz);
  return __dadd_rn(uc, r);
}

// ---------------------------------------------------------------------------
// ghost executor
// ---------------------------------------------------------------------------
// Offsets, inside one (block, var) box, of the r-th 16-byte unit of a same-level / outflow face copy:
// so = source doubles (a pair, or one double replicated for an outflow x face), d_o = destination pair.
template <int DIM, int N>
__device__ __forceinline__ void copy_unit(int face, bool outflow, int r, int& so, int& d_o) {
  using G = Geo<DIM, N>;
  constexpr int P = G::P;
  const int a = face >> 1, side = face & 1;
  // destination ghost slots along the normal: low ghosts P-2,P-1 (cells -2,-1); high ghosts N,N+1
  const int dn = side ? N : P - 2;
  // source slots: SRL -x: neighbour's cells N-2,N-1; +x: cells 0,1.  Outflow: nearest own interior layer.
  const int sn = outflow ? (side ? N - 1 : 0) : (side ? 0 : N - 2);
  if (a == 0) {  // one row = one 16-byte ghost pair
    const int j = r % N, k = (DIM == 3) ? r / N : 0;
    const int pl0 = (DIM == 3 ? k * P * P : 0);
    d_o = pl0 + (side ? (j & ~1) : (j | 1)) * P + N + 2 * (j & 1);   // pair-transposed x ghosts (cell_off)
    so = pl0 + j * P + sn;
    return;
  }
  int h, q, t;
  if (DIM == 3) {
    if (a == 1) { t = r / N; q = (r % N) / G::H; h = r % G::H; }               // t = k
    else        { q = r / (N * G::H); t = (r / G::H) % N; h = r % G::H; }      // t = j
  } else { q = r / G::H; h = r % G::H; t = 0; }
  const int dl = dn + q, sl = outflow ? sn : sn + q;   // the source advances with the layer only for SRL
  if (DIM == 3) {
    if (a == 1) { d_o = t * P * P + dl * P + 2 * h; so = t * P * P + sl * P + 2 * h; }
    else        { d_o = dl * P * P + t * P + 2 * h; so = sl * P * P + t * P + 2 * h; }
  } else { d_o = dl * P + 2 * h; so = sl * P + 2 * h; }
}

// one coarse ghost cell of an F2C record: e in [0, NVAR * NG * H^(d-1)); returns the destination, the value in val
template <int DIM, int N, int NV>
__device__ __forceinline__ double* f2c_item(double* __restrict__ st, const DevRecord& rec, int e, double& val) {
  using G = Geo<DIM, N, NV>;
  constexpr int H = G::H;
  const int face = (rec.meta >> 2) & 7, o1 = (rec.meta >> 5) & 1, o2 = (rec.meta >> 6) & 1;
  const int a = face >> 1, side = face & 1;
  constexpr int PER_VAR = NG * ((DIM == 3) ? H * H : H);
  double* db = st + (size_t)rec.dst * G::BS;
  const double* sb = st + (size_t)rec.src * G::BS;
  const int v = e / PER_VAR, r = e % PER_VAR;
  const int tt1 = r % H, tt2 = (DIM == 3) ? (r / H) % H : 0, q = r / ((DIM == 3) ? H * H : H);
  // coarse ghost cell: normal index N+q (high) or -2+q (low); its fine children along the normal
  const int nc = side ? N + q : -2 + q;
  const int nf = side ? 2 * q : N - 4 + 2 * q;
  const int t1c = o1 * H + tt1, t2c = o2 * H + tt2;
  int ci, cj, ck, fi, fj, fk;
  if (a == 0) { ci = nc; cj = t1c; ck = t2c; fi = nf; fj = 2 * tt1; fk = 2 * tt2; }
  else if (a == 1) { cj = nc; ci = t1c; ck = t2c; fj = nf; fi = 2 * tt1; fk = 2 * tt2; }
  else { ck = nc; ci = t1c; cj = t2c; fk = nf; fi = 2 * tt1; fj = 2 * tt2; }
  if (DIM == 2) { ck = 0; fk = 0; }
  val = restrict_mean<DIM, N>(sb + (size_t)v * G::VS, fi, fj, fk);
  return db + (size_t)v * G::VS + cell_off<DIM, N>(ci, cj, ck);
}

// one coarse cell of a C2F record (its 2^d... the NG x 2^(d-1) fine ghost cells it covers): e in [0, NVAR * H^(d-1))
template <int DIM, int N, int NV>
__device__ __forceinline__ void c2f_item(double* __restrict__ st, const DevRecord& rec, int e, double theta) {
  using G = Geo<DIM, N, NV>;
  constexpr int H = G::H;
  const int face = (rec.meta >> 2) & 7, o1 = (rec.meta >> 5) & 1, o2 = (rec.meta >> 6) & 1;
  const int a = face >> 1, side = face & 1;
  constexpr int PER_VAR = (DIM == 3) ? H * H : H;  // coarse cells of the one coarse layer (NG/2 = 1)
  double* db = st + (size_t)rec.dst * G::BS;
  const double* sb = st + (size_t)rec.src * G::BS;
  const int ncoarse = side ? 0 : N - 1;   // F's high ghosts are covered by C's first cell, low ghosts by its last
  const int nfine = side ? N : -2;        // lower of the two fine ghost cells (lower half of the coarse cell)
  const int v = e / PER_VAR, r = e % PER_VAR;
  const int tt1 = r % H, tt2 = (DIM == 3) ? r / H : 0;
  const int t1c = o1 * H + tt1, t2c = o2 * H + tt2;
  int ic, jc, kc, fi, fj, fk;
  if (a == 0) { ic = ncoarse; jc = t1c; kc = t2c; fi = nfine; fj = 2 * tt1; fk = 2 * tt2; }
  else if (a == 1) { jc = ncoarse; ic = t1c; kc = t2c; fj = nfine; fi = 2 * tt1; fk = 2 * tt2; }
  else { kc = ncoarse; ic = t1c; jc = t2c; fk = nfine; fi = 2 * tt1; fj = 2 * tt2; }
  if (DIM == 2) { kc = 0; fk = 0; }
  double uc, sx, sy, sz;
  coarse_slopes<DIM, N>(sb + (size_t)v * G::VS, ic, jc, kc, theta, uc, sx, sy, sz);
  double* dv = db + (size_t)v * G::VS;
#pragma unroll
  for (int pz = 0; pz < (DIM == 3 ? 2 : 1); ++pz)
#pragma unroll
    for (int py = 0; py < 2; ++py) {
      double2 w;
      w.x = child_value<DIM>(uc, sx, sy, sz, 0, py, pz);
      w.y = child_value<DIM>(uc, sx, sy, sz, 1, py, pz);
      st2(dv + cell_off<DIM, N>(fi, fj + py, fk + pz), w);   // fi even or -2: the x pair is 16-byte aligned
    }
}

// Uniform Dirichlet / Neumann boundary face (readings A10, A10b), one record = one block face:
//   Dirichlet: ghost layer g mirrors interior layer g through the face, u_ghost = 2 u_b - u_interior;
//   Neumann:   ghost layer g = first interior layer + (g dx) u_b'  (u_b' = outward normal derivative).
// Individually rounded operations in the order the formulas are written: bit-exact against the oracle.
template <int DIM, int N, int NV>
__device__ __forceinline__ void do_bc_values(double* __restrict__ st, int blk, int face, bool neumann,
                                             const double* __restrict__ bcv, double dx,
                                             const double* __restrict__ data /* this face's bc_data, or nullptr */) {
  using G = Geo<DIM, N, NV>;
  constexpr int FS = (DIM == 3) ? N * N : N;
  const int a = face >> 1, side = face & 1;
  double* db = st + (size_t)blk * G::BS;
  for (int e = threadIdx.x; e < NV * NG * FS; e += blockDim.x) {
    const int v = e / (NG * FS), r = e % (NG * FS), g = r / FS + 1, t = r % FS, t1 = t % N, t2 = t / N;
    const int nd = side ? N - 1 + g : -g;                              // ghost cell along the normal
    const int ns = neumann ? (side ? N - 1 : 0) : (side ? N - g : g - 1);
    int di, dj, dk, si, sj, sk;
    if (a == 0) { di = nd; si = ns; dj = sj = t1; dk = sk = t2; }
    else if (a == 1) { dj = nd; sj = ns; di = si = t1; dk = sk = t2; }
    else { dk = nd; sk = ns; di = si = t1; dj = sj = t2; }
    double* dv = db + (size_t)v * G::VS;
    const double src = dv[cell_off<DIM, N>(si, sj, sk)], ub = data ? data[v * FS + t] : bcv[face * NV + v];
    dv[cell_off<DIM, N>(di, dj, dk)] =
        neumann ? __dadd_rn(src, __dmul_rn(__dmul_rn((double)g, dx), ub)) : __dsub_rn(__dmul_rn(2.0, ub), src);
  }
}

// CH: records per CTA.  2*DIM (= all faces of one block on a uniform mesh: one destination block per CTA) for long
// lists; 1 for the short lists inside a time step of an adaptive run (F2C / C2F / BC records only: a few hundred to
// a few thousand), where CTAs of 2*DIM records would leave most SMs idle and each thread with a long serial chain
// of dependent loads.
template <int DIM, int N, int NV, int CH>
__global__ void __launch_bounds__(256, 4) ghost_exec_kernel(GhostParams p) {
  using G = Geo<DIM, N, NV>;
  constexpr int PER_VAR = (DIM == 3) ? N * N : N;   // 16-byte units per variable of one face copy
  __shared__ DevRecord recs[CH];
  const int r0 = blockIdx.x * CH;
  const int n = (p.nrec - r0 < CH) ? p.nrec - r0 : CH;
  if ((int)threadIdx.x < n) recs[threadIdx.x] = p.rec[r0 + threadIdx.x];
  __syncthreads();
  // ---- same-level and outflow copies of all records of this CTA, flattened over (record, unit); every thread
  //      has the loads of two units (2 x NV x 16 bytes) in flight before it stores
  constexpr int UNR = 2;
  for (int e0 = threadIdx.x; e0 < n * PER_VAR; e0 += UNR * blockDim.x) {
    double2 val[UNR][NV];
    double* dptr[UNR];
#pragma unroll
    for (int u = 0; u < UNR; ++u) {
      const int e = e0 + u * blockDim.x;
      dptr[u] = nullptr;
      if (e >= n * PER_VAR) continue;
      const DevRecord rec = recs[e / PER_VAR];
      const int op = rec.meta & 3, face = (rec.meta >> 2) & 7;
      if (op > F4_OP_BC || (op == F4_OP_BC && (rec.meta >> 5) & 3)) continue;   // Dirichlet / Neumann faces: below
      const bool outflow = (op == F4_OP_BC);
      int so, d_o;
      copy_unit<DIM, N>(face, outflow, e % PER_VAR, so, d_o);
      const double* sp = p.state + (size_t)rec.src * G::BS + so;
      dptr[u] = p.state + (size_t)rec.dst * G::BS + d_o;
      if (outflow && face < 2) {
#pragma unroll
        for (int v = 0; v < NV; ++v) { const double x = sp[(size_t)v * G::VS]; val[u][v] = make_double2(x, x); }
      } else {
#pragma unroll
        for (int v = 0; v < NV; ++v) val[u][v] = ld2(sp + (size_t)v * G::VS);
      }
    }
#pragma unroll
    for (int u = 0; u < UNR; ++u)
      if (dptr[u]) {
#pragma unroll
        for (int v = 0; v < NV; ++v) st2(dptr[u] + (size_t)v * G::VS, val[u][v]);
      }
  }
  // ---- restriction / prolongation records of this CTA, flattened over (record, cell) like the copies above, so that
  //      a CTA with several such records (refinement boundaries) keeps all its threads and loads busy
  __shared__ int lst_f2c[CH], lst_c2f[CH], cnt[2];
  if (threadIdx.x == 0) {
    int nf = 0, nc = 0;
    for (int q = 0; q < n; ++q) {
      const int op = recs[q].meta & 3;
      if (op == F4_OP_F2C) lst_f2c[nf++] = q;
      else if (op == F4_OP_C2F) lst_c2f[nc++] = q;
    }
    cnt[0] = nf;
    cnt[1] = nc;
  }
  __syncthreads();
  {
    constexpr int ITEMS = NV * NG * ((DIM == 3) ? G::H * G::H : G::H);
    const int tot = cnt[0] * ITEMS;
    for (int e0 = threadIdx.x; e0 < tot; e0 += 2 * blockDim.x) {   // two cells (2 x 2^d loads) in flight per thread
      const int e1 = e0 + blockDim.x;
      double v0, v1 = 0.0;
      double* d0 = f2c_item<DIM, N, NV>(p.state, recs[lst_f2c[e0 / ITEMS]], e0 % ITEMS, v0);
      double* d1 = (e1 < tot) ? f2c_item<DIM, N, NV>(p.state, recs[lst_f2c[e1 / ITEMS]], e1 % ITEMS, v1) : nullptr;
      *d0 = v0;
      if (d1) *d1 = v1;
    }
  }
  {
    constexpr int ITEMS = NV * ((DIM == 3) ? G::H * G::H : G::H);
    const int tot = cnt[1] * ITEMS;
    for (int e = threadIdx.x; e < tot; e += blockDim.x)
      c2f_item<DIM, N, NV>(p.state, recs[lst_c2f[e / ITEMS]], e % ITEMS, p.theta);
  }
  // ---- uniform Dirichlet / Neumann / bc_data faces
#pragma unroll 1
  for (int q = 0; q < n; ++q) {
    const DevRecord rec = recs[q];
    const int op = rec.meta & 3, face = (rec.meta >> 2) & 7, o1 = (rec.meta >> 5) & 1, o2 = (rec.meta >> 6) & 1;
    if (op == F4_OP_BC && (o1 | o2))   // (1,0) Dirichlet, (0,1) Neumann, (1,1) bc_data of face rec.src (mirror rule)
      do_bc_values<DIM, N, NV>(p.state, rec.dst, face, o2 != 0 && o1 == 0, p.bcv,
                           p.dx0 * (1.0 / (double)(1u << p.level[rec.dst])),
                           (o1 & o2) ? p.bcdata + (size_t)rec.src * G::NVAR * ((DIM == 3) ? N * N : N) : nullptr);
  }
}

// ---------------------------------------------------------------------------
// Same-level copies of a WHOLE fill, by source block (the SRL part of round 1).
// The record list is sorted by destination: a CTA of ghost_exec_kernel gathers the six faces of one block from six
// neighbours, and the x-face sources -- the first / last 16 bytes of 160-byte rows -- cost a 64-byte DRAM atom each,
// in rows that the y / z copies of OTHER destinations fetch again (DRAM reads 2.4 x the algorithmic bytes,
// profiles/ghost_exec_r2.md).  Turned round, one CTA per (source block, variable) reads the block's interior rows
// ONCE and stores every 16-byte unit into the ghost region of each same-level neighbour it belongs to (up to three:
// an x, a y and a z face).
// nbr[b][f] = same-level neighbour across face f or -1 (then a BC / F2C / C2F record fills that face); same-level
// adjacency is symmetric, so b's cells next to its face f are the ghosts of nbr[b][f] at face f^1.
// ---------------------------------------------------------------------------
// The rows come in by the TMA engine: one bulk copy per z plane (its N interior rows with the ghost slots between
// them are contiguous: N*P doubles) into shared memory, all planes of the CTA's z chunk requested at once by the
// lanes of one warp -- tens of KB in flight per CTA without a register -- then every thread stores the 16-byte units of the
// chunk that belong to a face layer.
template <int DIM, int N, int NV>
struct PushCfg {
  static constexpr int P = N + 2 * NG;
  static constexpr int NZ = (DIM == 3) ? N : 1;
  static constexpr int PLANE = N * P;                                   // doubles per bulk copy
  static constexpr int BUDGET = 40 * 1024;                              // bytes of bulk copies per CTA
  static constexpr int ZC_MAX = BUDGET / (PLANE * 8);
  static constexpr int ZC = (NZ <= ZC_MAX) ? NZ : (ZC_MAX >= 16 ? 16 : (ZC_MAX >= 8 ? 8 : (ZC_MAX >= 4 ? 4 : (ZC_MAX >= 2 ? 2 : 1))));
  static constexpr int NCHUNK = NZ / ZC;
  static constexpr int VC = (NV * ZC * PLANE * 8 <= BUDGET) ? NV : 1;   // small blocks: all variables in one CTA
  static constexpr size_t SMEM = (size_t)VC * ZC * PLANE * 8 + 16;
  static_assert(NZ % ZC == 0 && (PLANE * 8) % 16 == 0 && NV % VC == 0, "chunking");
};

template <int DIM, int N, int NV>
__global__ void __launch_bounds__(256) srl_push_kernel(double* __restrict__ st, const int* __restrict__ nbr) {
  using G = Geo<DIM, N, NV>;
  using C = PushCfg<DIM, N, NV>;
  constexpr int H = G::H, P = G::P, PP = P * P, ZC = C::ZC, PLANE = C::PLANE, VC = C::VC;
  constexpr int UNITS = H * N * ZC;                     // 16-byte units of one variable's chunk interior
  extern __shared__ __align__(128) unsigned char push_smem[];
  double* sm = reinterpret_cast<double*>(push_smem);    // [VC][ZC][PLANE]
  uint64_t* bar = reinterpret_cast<uint64_t*>(sm + VC * ZC * PLANE);
  __shared__ int nb[6];
  // consecutive CTAs take the variables of one block: they read one contiguous stretch of the store
  constexpr int NVQ = NV / VC;
  const int b = blockIdx.x / NVQ, v0 = (blockIdx.x % NVQ) * VC, k0 = blockIdx.y * ZC;
  const double* sb = st + (size_t)b * G::BS;
  if (threadIdx.x < 32) {                               // warp 0 requests the copies, a share per lane
    const uint32_t bar32 = smem_u32(bar);
    if (threadIdx.x == 0) {
      mbar_init(bar, 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
      mbar_expect_tx(bar32, (uint32_t)(VC * ZC * PLANE * 8));
    }
    __syncwarp();
    for (int c = threadIdx.x; c < VC * ZC; c += 32) {
      const int vv = c / ZC, kk = c % ZC;
      bulk_g2s(smem_u32(sm + c * PLANE), sb + (size_t)(v0 + vv) * G::VS + (size_t)(k0 + kk) * PP, (uint32_t)(PLANE * 8), bar32);
    }
  } else if (threadIdx.x < 38) {
    const int f = threadIdx.x - 32;
    nb[f] = (f < 2 * DIM) ? nbr[(size_t)b * 6 + f] : -1;
  }
  __syncthreads();                                      // the barrier is initialised, nb[] is there
  mbar_wait(smem_u32(bar), 0);
  const bool zlo = DIM == 3 && k0 < NG && nb[4] >= 0, zhi = DIM == 3 && k0 + ZC > N - NG && nb[5] >= 0;
  for (int e = threadIdx.x; e < VC * UNITS; e += 256) {
    const int vv = e / UNITS, r = e % UNITS;
    const int h = r % H, j = (r / H) % N, kk = r / (H * N), k = k0 + kk;
    const bool x0 = h == 0 && nb[0] >= 0, x1 = h == H - 1 && nb[1] >= 0;
    const bool y0 = j < NG && nb[2] >= 0, y1 = j >= N - NG && nb[3] >= 0;
    const bool z0 = zlo && k < NG, z1 = zhi && k >= N - NG;
    if (!(x0 | x1 | y0 | y1 | z0 | z1)) continue;       // a unit of the core: nobody's ghost
    const double2 val = *reinterpret_cast<const double2*>(sm + (vv * ZC + kk) * PLANE + j * P + 2 * h);
    const size_t vo = (size_t)(v0 + vv) * G::VS;
    const int kp = (DIM == 3) ? k * PP : 0;
    // x: pair-transposed ghost slots (cell_off): cells N, N+1 of row j in row j&~1, cells -2, -1 in row j|1
    if (x0) st2(st + (size_t)nb[0] * G::BS + vo + kp + (j & ~1) * P + N + 2 * (j & 1), val);
    if (x1) st2(st + (size_t)nb[1] * G::BS + vo + kp + (j | 1) * P + N + 2 * (j & 1), val);
    // y: rows 0, 1 are the low neighbour's ghost rows N, N+1; rows N-2, N-1 the high neighbour's slots P-2, P-1
    if (y0) st2(st + (size_t)nb[2] * G::BS + vo + kp + (N + j) * P + 2 * h, val);
    if (y1) st2(st + (size_t)nb[3] * G::BS + vo + kp + (j - N + P) * P + 2 * h, val);
    if (z0) st2(st + (size_t)nb[4] * G::BS + vo + (N + k) * PP + j * P + 2 * h, val);
    if (z1) st2(st + (size_t)nb[5] * G::BS + vo + (k - N + P) * PP + j * P + 2 * h, val);
  }
}

// ---------------------------------------------------------------------------
// regrid transfer: one CTA per new block
// ---------------------------------------------------------------------------
template <int DIM, int N, int NV>
__global__ void __launch_bounds__(256) transfer_kernel(const double* __restrict__ old_st, double* __restrict__ new_st,
                                                       const DevTransfer* __restrict__ plan, double theta) {
  using G = Geo<DIM, N, NV>;
  constexpr int H = G::H, NZ = G::NZ;
  const DevTransfer t = plan[blockIdx.x];
  double* db = new_st + (size_t)t.dst * G::BS;
  if (t.kind == 0) {  // unaltered: copy the interior
    const double* sb = old_st + (size_t)t.src[0] * G::BS;
    for (int e = threadIdx.x; e < NV * NZ * N * H; e += blockDim.x) {
      int h = e % H, j = (e / H) % N, k = (e / (H * N)) % NZ, v = e / (H * N * NZ);
      size_t o = (size_t)v * G::VS + cell_off<DIM, N>(2 * h, j, k);
      st2(db + o, ld2(sb + o));
    }
  } else if (t.kind == 1) {  // refined: limited prolongation of the parent's octant (needs the parent's face ghosts)
    const double* sb = old_st + (size_t)t.src[0] * G::BS;
    const int ox = t.oct & 1, oy = (t.oct >> 1) & 1, oz = (t.oct >> 2) & 1;
    constexpr int HZ = (DIM == 3) ? H : 1;
    for (int e = threadIdx.x; e < NV * HZ * H * H; e += blockDim.x) {
      int i = e % H, j = (e / H) % H, k = (e / (H * H)) % HZ, v = e / (H * H * HZ);
      double uc, sx, sy, sz;
      coarse_slopes<DIM, N>(sb + (size_t)v * G::VS, ox * H + i, oy * H + j, (DIM == 3) ? oz * H + k : 0, theta, uc, sx,
                            sy, sz);
      double* dv = db + (size_t)v * G::VS;
#pragma unroll
      for (int pz = 0; pz < (DIM == 3 ? 2 : 1); ++pz)
#pragma unroll
        for (int py = 0; py < 2; ++py) {
          double2 w;
          w.x = child_value<DIM>(uc, sx, sy, sz, 0, py, pz);
          w.y = child_value<DIM>(uc, sx, sy, sz, 1, py, pz);
          st2(dv + cell_off<DIM, N>(2 * i, 2 * j + py, 2 * k + pz), w);
        }
    }
  } else {  // coarsened: restriction of the 2^d children
    constexpr int HZ = (DIM == 3) ? H : 1;
    constexpr int NCH = 1 << DIM;
    for (int e = threadIdx.x; e < NCH * NV * HZ * H * H; e += blockDim.x) {
      int i = e % H, j = (e / H) % H, k = (e / (H * H)) % HZ, v = (e / (H * H * HZ)) % NV, c = e / (H * H * HZ * NV);
      const double* sb = old_st + (size_t)t.src[c] * G::BS + (size_t)v * G::VS;
      int ox = c & 1, oy = (c >> 1) & 1, oz = (c >> 2) & 1;
      db[(size_t)v * G::VS + cell_off<DIM, N>(ox * H + i, oy * H + j, (DIM == 3) ? oz * H + k : 0)] =
          restrict_mean<DIM, N>(sb, 2 * i, 2 * j, 2 * k);
    }
  }
}

// ---------------------------------------------------------------------------
// layout kernels (not on the per-step path)
// ---------------------------------------------------------------------------
template <int DIM, int N, int NV, bool PACK>
__global__ void __launch_bounds__(256) layout_kernel(double* __restrict__ store, double* __restrict__ user, int b0,
                                                     int with_ghosts) {
  using G = Geo<DIM, N, NV>;
  const int E = with_ghosts ? G::P : N, EZ = (DIM == 3) ? E : 1, lo = with_ghosts ? -NG : 0;
  const int b = blockIdx.x, v = blockIdx.y;
  const size_t ubase = ((size_t)b * G::NVAR + v) * (size_t)(E * E * EZ);
  double* sv = store + ((size_t)(b0 + b) * G::NVAR + v) * G::VS;
  for (int e = threadIdx.x; e < E * E * EZ; e += blockDim.x) {
    int i = e % E + lo, j = (e / E) % E + lo, k = (DIM == 3) ? e / (E * E) + lo : 0;
    int o = cell_off<DIM, N>(i, j, k);
    if (PACK) sv[o] = user[ubase + e];
    else user[ubase + e] = sv[o];
  }
}

template <int DIM, int N, int NV>
__global__ void __launch_bounds__(256) init_benign_kernel(double* __restrict__ store, double gamma) {
  using G = Geo<DIM, N, NV>;
  const int b = blockIdx.x, v = blockIdx.y;
  double val = (v == 0) ? 1.0 : (v == G::NVAR - 1 ? 1.0 / (gamma - 1.0) : 0.0);  // rho=1, u=0, p=1
  double* sv = store + ((size_t)b * G::NVAR + v) * G::VS;
  for (int e = threadIdx.x; e < (int)G::VS; e += blockDim.x) sv[e] = val;
}

// per-(block,var) interior sums, fixed order inside the CTA (for f4_conserved_totals)
template <int DIM, int N, int NV>
__global__ void __launch_bounds__(256) block_sums_kernel(const double* __restrict__ st, double* __restrict__ sums) {
  using G = Geo<DIM, N, NV>;
  __shared__ double sh[256];
  const int b = blockIdx.x, v = blockIdx.y;
  const double* sv = st + ((size_t)b * G::NVAR + v) * G::VS;
  double acc = 0.0;
  for (int e = threadIdx.x; e < N * N * G::NZ; e += blockDim.x) {
    int i = e % N, j = (e / N) % N, k = e / (N * N);
    acc += sv[cell_off<DIM, N>(i, j, k)];
  }
  sh[threadIdx.x] = acc;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) sums[(size_t)b * G::NVAR + v] = sh[0];
}

// Refinement criteria (section 3.3 eq. (12); BASELINE config 5's pressure-jump rule, reading A15):
// one CTA per block reduces the per-cell indicator to its maximum over the block's interior cells and writes the
// flag (+1 if max > params[0]; -1 if max < params[1], i.e. ALL cells below; else 0).  Face ghosts of the first layer
// are read, so the state must be ghost-filled.  The flag is a discrete decision taken from floating point: every
// operation is an explicitly rounded IEEE add / mul / div / sqrt in the order the paper writes the formula, no
// contraction, so that the indicator does not depend on compiler choices.
template <int DIM, int N, int NV>
__global__ void __launch_bounds__(256) flags_kernel(const double* __restrict__ st, int criterion, int var, double gamma,
                                                    double p0, double p1, double p2, double p3,
                                                    int* __restrict__ flags, double* __restrict__ indicator) {
  using G = Geo<DIM, N, NV>;
  __shared__ double sh[8];
  const int b = blockIdx.x;
  const double* sb = st + (size_t)b * G::BS;
  auto pressure = [&](int i, int j, int k) {   // eq. (15) inverted: p = (gamma-1)(E - 1/2 |m|^2 / rho)
    const int o = cell_off<DIM, N>(i, j, k);
    const double rho = sb[o];
    double ke = 0.0;
#pragma unroll
    for (int a = 0; a < DIM; ++a) { const double mom = sb[(size_t)(1 + a) * G::VS + o]; ke = __dadd_rn(ke, __dmul_rn(mom, mom)); }
    return __dmul_rn(gamma - 1.0, __dsub_rn(sb[(size_t)(G::NVAR - 1) * G::VS + o], __ddiv_rn(__dmul_rn(0.5, ke), rho)));
  };
  double mx = 0.0;
  for (int e = threadIdx.x; e < N * N * G::NZ; e += blockDim.x) {
    const int i = e % N, j = (e / N) % N, k = e / (N * N);
    double cell = 0.0;
    if (criterion == F4_CRIT_LOHNER) {
      const double* sv = sb + (size_t)var * G::VS;
      const double u0 = sv[cell_off<DIM, N>(i, j, k)];
      double sumsq = 0.0;
#pragma unroll
      for (int a = 0; a < DIM; ++a) {
        const int di = (a == 0), dj = (a == 1), dk = (a == 2);
        const double um = sv[cell_off<DIM, N>(i - di, j - dj, k - dk)];
        const double up = sv[cell_off<DIM, N>(i + di, j + dj, k + dk)];
        const double num = fabs(__dadd_rn(__dsub_rn(um, __dmul_rn(2.0, u0)), up));
        const double ustar = __dadd_rn(__dadd_rn(fabs(um), __dmul_rn(2.0, fabs(u0))), fabs(up));
        const double den = __dadd_rn(__dadd_rn(__dadd_rn(p3, fabs(__dsub_rn(u0, um))), fabs(__dsub_rn(up, u0))),
                                     __dmul_rn(p2, ustar));
        const double En = __ddiv_rn(num, den);
        sumsq = __dadd_rn(sumsq, __dmul_rn(En, En));
      }
      cell = sumsq;   // the square root is taken once, of the block maximum (monotone and correctly rounded: same bits)
    } else {
      const double pc = pressure(i, j, k);
#pragma unroll
      for (int a = 0; a < DIM; ++a) {
        const int di = (a == 0), dj = (a == 1), dk = (a == 2);
#pragma unroll
        for (int sg = -1; sg <= 1; sg += 2) {
          const double pn = pressure(i + sg * di, j + sg * dj, k + sg * dk);
          const double jump = __ddiv_rn(fabs(__dsub_rn(pc, pn)), fmin(pc, pn));
          if (jump > cell) cell = jump;
        }
      }
    }
    if (cell > mx) mx = cell;
  }
  for (int sft = 16; sft > 0; sft >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, sft));
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = mx;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; ++w) mx = fmax(mx, sh[w]);
    if (criterion == F4_CRIT_LOHNER) mx = __dsqrt_rn(mx);
    if (indicator) indicator[b] = mx;
    flags[b] = (mx > p0) ? 1 : ((mx < p1) ? -1 : 0);
  }
}

// The pressure-jump rule alone (BASELINE config 5, reading A15), the regrid's device cost on adaptive runs: the same
// indicator as flags_kernel's, max over face-adjacent cell pairs (at least one of them interior) of
// |p_a - p_b| / min(p_a, p_b), with every pressure computed ONCE (a two-plane ring in shared memory) and every pair
// visited ONCE (the quotient is symmetric) instead of seven pressures and six quotients per cell: 4.6 IEEE divisions
// per cell instead of 13.  Same explicitly rounded operations, and a maximum does not depend on the order: the
// indicator is bit-identical to flags_kernel's.
template <int DIM, int N, int NV>
__global__ void __launch_bounds__(256) pjump_flags_kernel(const double* __restrict__ st, double gamma, double p0, double p1,
                                                          int* __restrict__ flags, double* __restrict__ indicator) {
  using G = Geo<DIM, N, NV>;
  constexpr int E = N + 2;                     // plane edge with one ghost layer
  constexpr int K0 = (DIM == 3) ? -1 : 0, K1 = (DIM == 3) ? N : 0;
  __shared__ double pp[2][E * E];
  __shared__ double sh[8];
  const int b = blockIdx.x, tid = threadIdx.x;
  const double* sb = st + (size_t)b * G::BS;
  auto pressure = [&](int i, int j, int k) {   // eq. (15) inverted: p = (gamma-1)(E - 1/2 |m|^2 / rho)
    const int o = cell_off<DIM, N>(i, j, k);
    const double rho = sb[o];
    double ke = 0.0;
#pragma unroll
    for (int a = 0; a < DIM; ++a) { const double mom = sb[(size_t)(1 + a) * G::VS + o]; ke = __dadd_rn(ke, __dmul_rn(mom, mom)); }
    return __dmul_rn(gamma - 1.0, __dsub_rn(sb[(size_t)(G::NVAR - 1) * G::VS + o], __ddiv_rn(__dmul_rn(0.5, ke), rho)));
  };
  double mx = 0.0;
  auto jump = [&](double pa, double pb) {
    const double q = __ddiv_rn(fabs(__dsub_rn(pa, pb)), fmin(pa, pb));
    if (q > mx) mx = q;
  };
  for (int k = K0; k <= K1; ++k) {
    double* cur = pp[(k - K0) & 1];
    const double* prev = pp[(k - K0 + 1) & 1];
    const bool kin = (k >= 0 && k < N);
    // pressures of plane k: the interior columns always, the x / y face ghosts where the plane is an interior one
    for (int e = tid; e < E * E; e += 256) {
      const int i = e % E - 1, j = e / E - 1;
      const bool iin = (i >= 0 && i < N), jin = (j >= 0 && j < N);
      if ((iin && jin) || (kin && (iin || jin))) cur[e] = pressure(i, j, k);
    }
    __syncthreads();
    if (kin) {
      for (int e = tid; e < (N + 1) * N; e += 256) {        // x pairs (i, i+1), i = -1 .. N-1
        const int i = e % (N + 1) - 1, j = e / (N + 1);
        jump(cur[(j + 1) * E + i + 1], cur[(j + 1) * E + i + 2]);
      }
      for (int e = tid; e < (N + 1) * N; e += 256) {        // y pairs (j, j+1), j = -1 .. N-1
        const int i = e % N, j = e / N - 1;
        jump(cur[(j + 1) * E + i + 1], cur[(j + 2) * E + i + 1]);
      }
    }
    if (DIM == 3 && k >= 0) {                               // z pairs (k-1, k), k = 0 .. N
      for (int e = tid; e < N * N; e += 256) {
        const int i = e % N, j = e / N;
        jump(prev[(j + 1) * E + i + 1], cur[(j + 1) * E + i + 1]);
      }
    }
    __syncthreads();
  }
  for (int sft = 16; sft > 0; sft >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, sft));
  if ((tid & 31) == 0) sh[tid >> 5] = mx;
  __syncthreads();
  if (tid == 0) {
    for (int w = 1; w < 8; ++w) mx = fmax(mx, sh[w]);
    if (indicator) indicator[b] = mx;
    flags[b] = (mx > p0) ? 1 : ((mx < p1) ? -1 : 0);
  }
}

// CFL: max over interior cells of sum_dim (|u_d| + c)/dx (readings A4-A5).
// Warp shuffle max, then one atomicMax per warp on the bit pattern (non-negative doubles order as integers).
template <int DIM, int N>
__global__ void __launch_bounds__(256) maxrate_kernel(const double* __restrict__ st, const int* __restrict__ level,
                                                      double gamma, double inv_dx0, unsigned long long* maxrate) {
  using G = Geo<DIM, N>;
  const int b = blockIdx.x;
  const double* sb = st + (size_t)b * G::BS;
  const double inv_dx = inv_dx0 * (double)(1u << level[b]);
  double mx = 0.0;
  for (int e = threadIdx.x; e < N * N * G::NZ; e += blockDim.x) {
    int i = e % N, j = (e / N) % N, k = e / (N * N);
    int o = cell_off<DIM, N>(i, j, k);
    double rho = sb[o], ir = 1.0 / rho, ke = 0.0, su = 0.0;
#pragma unroll
    for (int d = 0; d < DIM; ++d) {
      double u = sb[(size_t)(1 + d) * G::VS + o] * ir;
      ke += u * u;
      su += fabs(u);
    }
    double p = (gamma - 1.0) * (sb[(size_t)(DIM + 1) * G::VS + o] - 0.5 * rho * ke);
    double c = sqrt(gamma * p * ir);
    // a cell that is not a valid gas state (NaN, rho <= 0, p <= 0) makes the maximum +inf: compute_dt reports it
    const double rate = (su + DIM * c) * inv_dx;
    mx = fmax(mx, (rho > 0.0 && p > 0.0 && rate == rate) ? rate : __longlong_as_double(0x7ff0000000000000LL));
  }
  for (int s = 16; s > 0; s >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, s));
  if ((threadIdx.x & 31) == 0) atomicMax(maxrate, (unsigned long long)__double_as_longlong(mx));
}

__global__ void dt_from_rate_kernel(const unsigned long long* __restrict__ maxrate, double cfl, double* __restrict__ dt) {
  const double rate = __longlong_as_double((long long)*maxrate);
  const bool ok = rate > 0.0 && rate <= 1.7976931348623157e308;
  dt[0] = ok ? cfl / rate : 0.0;      // dt = 0: the stages leave the state as it is; f4_last_dt reports the failure
  dt[1] = ok ? 0.0 : 1.0;
}

template <typename F>
cudaError_t dispatch(int dim, int n, int nvar, F&& f) {
#define F4_CASE(D, NN)                                                   \
  if (dim == D && n == NN) {                                             \
    if (nvar == D + 2) return f(Geo<D, NN, D + 2>{});                    \
    if (nvar == 1) return f(Geo<D, NN, 1>{});                            \
  }
  F4_CASE(2, 8) F4_CASE(2, 16) F4_CASE(2, 32) F4_CASE(3, 8) F4_CASE(3, 16) F4_CASE(3, 32)
#undef F4_CASE
  return cudaErrorInvalidValue;
}
template <int D, int N, int V>
constexpr int dim_of(Geo<D, N, V>) { return D; }
template <int D, int N, int V>
constexpr int n_of(Geo<D, N, V>) { return N; }
template <int D, int N, int V>
constexpr int nv_of(Geo<D, N, V>) { return V; }

}  // namespace

#define F4_DISPATCH(body)                                        \
  return dispatch(dim, n, nvar, [&](auto g) -> cudaError_t {     \
    constexpr int D = dim_of(decltype(g){});                     \
    constexpr int NN = n_of(decltype(g){});                      \
    constexpr int NVV = nv_of(decltype(g){});                    \
    body;                                                        \
    return cudaGetLastError();                                   \
  })

cudaError_t launch_dt_from_rate(const unsigned long long* maxrate, double cfl, double* dt, cudaStream_t s) {
  dt_from_rate_kernel<<<1, 1, 0, s>>>(maxrate, cfl, dt);
  return cudaGetLastError();
}
cudaError_t launch_ghost(int dim, int n, int nvar, const GhostParams& p, cudaStream_t s) {
  if (p.nrec <= 0) return cudaSuccess;
  F4_DISPATCH(({
    const int grouped = (p.nrec + 2 * D - 1) / (2 * D);
    if (grouped < 2 * 4 * 148)   // fewer than two waves of grouped CTAs (4 resident per SM): one record per CTA
      ghost_exec_kernel<D, NN, NVV, 1><<<p.nrec, 256, 0, s>>>(p);
    else
      ghost_exec_kernel<D, NN, NVV, 2 * D><<<grouped, 256, 0, s>>>(p);
  }));
}
cudaError_t launch_srl_push(int dim, int n, int nvar, double* state, const int* nbr, int nblocks, cudaStream_t s) {
  if (nblocks <= 0) return cudaSuccess;
  F4_DISPATCH(({
    using C = PushCfg<D, NN, NVV>;
    auto k = srl_push_kernel<D, NN, NVV>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM);
    if (e != cudaSuccess) return e;
    k<<<dim3((unsigned)nblocks * (NVV / C::VC), C::NCHUNK), 256, C::SMEM, s>>>(state, nbr);
  }));
}
cudaError_t launch_transfer(int dim, int n, int nvar, const double* old_state, double* new_state, const DevTransfer* plan,
                            int nplan, double theta, cudaStream_t s) {
  if (nplan <= 0) return cudaSuccess;
  F4_DISPATCH((transfer_kernel<D, NN, NVV><<<nplan, 256, 0, s>>>(old_state, new_state, plan, theta)));
}
cudaError_t launch_pack(int dim, int n, int nvar, double* store_state, const double* src, int b0, int nb, int with_ghosts,
                        cudaStream_t s) {
  if (nb <= 0) return cudaSuccess;
  F4_DISPATCH((layout_kernel<D, NN, NVV, true><<<dim3(nb, NVV), 256, 0, s>>>(store_state, const_cast<double*>(src), b0,
                                                                           with_ghosts)));
}
cudaError_t launch_unpack(int dim, int n, int nvar, const double* store_state, double* dst, int b0, int nb, int with_ghosts,
                          cudaStream_t s) {
  if (nb <= 0) return cudaSuccess;
  F4_DISPATCH((layout_kernel<D, NN, NVV, false><<<dim3(nb, NVV), 256, 0, s>>>(const_cast<double*>(store_state), dst, b0,
                                                                            with_ghosts)));
}
cudaError_t launch_init_benign(int dim, int n, int nvar, double* store_state, int nb, double gamma, cudaStream_t s) {
  if (nb <= 0) return cudaSuccess;
  F4_DISPATCH((init_benign_kernel<D, NN, NVV><<<dim3(nb, NVV), 256, 0, s>>>(store_state, gamma)));
}
cudaError_t launch_block_sums(int dim, int n, int nvar, const double* state, int nb, double* sums, cudaStream_t s) {
  if (nb <= 0) return cudaSuccess;
  F4_DISPATCH((block_sums_kernel<D, NN, NVV><<<dim3(nb, NVV), 256, 0, s>>>(state, sums)));
}
cudaError_t launch_flags(int dim, int n, int nvar, const double* state, int nblocks, int criterion, int var, double gamma,
                         const double params[4], int* flags, double* indicator, cudaStream_t s) {
  if (nblocks <= 0) return cudaSuccess;
  F4_DISPATCH(({
    if constexpr (NVV == D + 2) {
      if (criterion == F4_CRIT_PJUMP) {
        pjump_flags_kernel<D, NN, NVV><<<nblocks, 256, 0, s>>>(state, gamma, params[0], params[1], flags, indicator);
        return cudaGetLastError();
      }
    }
    flags_kernel<D, NN, NVV><<<nblocks, 256, 0, s>>>(state, criterion, var, gamma, params[0], params[1], params[2],
                                                       params[3], flags, indicator);
  }));
}
cudaError_t launch_maxrate(int dim, int n, const double* state, const int* level, int nblocks, double gamma,
                           double inv_dx0, unsigned long long* maxrate, cudaStream_t s) {
  if (nblocks <= 0) return cudaSuccess;
  const int nvar = dim + 2;   // Euler only: scalar advection has the constant wave speed v (f4_compute_dt)
  F4_DISPATCH((maxrate_kernel<D, NN><<<nblocks, 256, 0, s>>>(state, level, gamma, inv_dx0, maxrate)));
}

// ---- f4_conserved_totals_noalloc: the block-sum reduction with its scratch in a static device array ------------
// For callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).
// g_noalloc_sums takes the place of the mesh's cudaMalloc'ed per-(block,var) sums; it is part of the loaded module, so
// every GPU that loads the library holds F4_NOALLOC_MAX_BLOCKS * 5 * 8 bytes (1.25 MiB) until the process exits.
// In host code the NAME g_noalloc_sums is a host-side stand-in, not a device address: the launcher below asks the
// runtime for the device address once per device (cudaGetSymbolAddress, with that device current) and hands THAT to
// the kernels.  Every call on a device shares the array: block_sums_kernel overwrites each entry the finishing
// kernel reads, so nothing has to be cleared between calls, but two calls that overlap on the GPU (different
// streams) race on it.
namespace {

constexpr int NOALLOC_MAX_VARS = 5;
static __device__ __align__(256) double g_noalloc_sums[(size_t)F4_NOALLOC_MAX_BLOCKS * NOALLOC_MAX_VARS];

constexpr int NOALLOC_MAX_DEVICES = 64;
double* g_noalloc_ptr[NOALLOC_MAX_DEVICES];   // device address of g_noalloc_sums on device d, 0 = not yet asked
std::mutex g_noalloc_mutex;

// error-free transformations: (s, e) with s + e = a + b exactly; the partial totals are carried as such pairs
__device__ __forceinline__ void two_sum(double a, double b, double& s, double& e) {
  s = __dadd_rn(a, b);
  const double bb = __dsub_rn(s, a);
  e = __dadd_rn(__dsub_rn(a, __dsub_rn(s, bb)), __dsub_rn(b, bb));
}
__device__ __forceinline__ void dd_add(double& hi, double& lo, double xh, double xl) {
  double s, e;
  two_sum(hi, xh, s, e);
  e = __dadd_rn(e, __dadd_rn(lo, xl));
  hi = __dadd_rn(s, e);
  lo = __dsub_rn(e, __dsub_rn(hi, s));
}

// totals[v] = sum_b sums[b][v] * dx(level_b)^dim: one CTA per variable, fixed order, double-double accumulation
// (the host path of f4_conserved_totals accumulates in long double; both are far inside the 1e-12 the tests ask)
__global__ void __launch_bounds__(256) totals_finish_kernel(const double* __restrict__ sums, const int* __restrict__ level,
                                                            int nb, int nvar, int dim, double dx0,
                                                            double* __restrict__ totals) {
  __shared__ double sh[256], sl[256];
  const int v = blockIdx.x;
  double hi = 0.0, lo = 0.0;
  for (int b = threadIdx.x; b < nb; b += blockDim.x) {
    const double h = dx0 / (double)(1u << level[b]);            // exact: a power of two
    const double vol = (dim == 3) ? __dmul_rn(__dmul_rn(h, h), h) : __dmul_rn(h, h);
    const double x = sums[(size_t)b * nvar + v];
    const double p = __dmul_rn(x, vol);
    dd_add(hi, lo, p, fma(x, vol, -p));
  }
  sh[threadIdx.x] = hi;
  sl[threadIdx.x] = lo;
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) {
      dd_add(hi, lo, sh[threadIdx.x + s], sl[threadIdx.x + s]);
      sh[threadIdx.x] = hi;
      sl[threadIdx.x] = lo;
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) totals[v] = __dadd_rn(hi, lo);
}

// device address of the static scratch on the CURRENT device; asks the runtime once per device
cudaError_t noalloc_scratch(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_ptr[dev]) {
    double* ptr = nullptr;
    e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_sums);
    if (e != cudaSuccess) return e;
    if (!ptr) return cudaErrorInvalidSymbol;
    g_noalloc_ptr[dev] = ptr;
  }
  *out = g_noalloc_ptr[dev];
  return cudaSuccess;
}

}  // namespace

cudaError_t launch_totals_noalloc(int dim, int n, int nvar, const double* state, const int* level, int nb, double dx0,
                                  double* totals_dev, cudaStream_t s) {
  if (nb <= 0 || nb > F4_NOALLOC_MAX_BLOCKS || nvar < 1 || nvar > NOALLOC_MAX_VARS) return cudaErrorInvalidValue;
  double* scratch = nullptr;
  cudaError_t e = noalloc_scratch(&scratch);
  if (e != cudaSuccess) return e;
  e = launch_block_sums(dim, n, nvar, state, nb, scratch, s);   // the kernel of f4_conserved_totals, static scratch
  if (e != cudaSuccess) return e;
  totals_finish_kernel<<<nvar, 256, 0, s>>>(scratch, level, nb, nvar, dim, dx0, totals_dev);
  return cudaGetLastError();
}

}  // namespace f4
