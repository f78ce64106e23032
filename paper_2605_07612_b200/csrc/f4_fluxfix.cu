// Flux fixing at refinement boundaries (section 2.7), coarse-side correction.
//
// The stage kernel stores the face-normal flux of every block face whose neighbour is coarser or finer
// ("during the flux computation, fluxes at refinement boundaries are stored in a pre-allocated array bflux",
// PAPER.md:257).  This kernel is the paper's "loop over all coarse sides of refinement boundaries": the cell next
// to the boundary was updated with the coarse flux Fc through that face; with the mean Ff of the 2^(d-1) fine
// fluxes instead, u changes by +dt_sub/dx_c (Ff - Fc) on a low face (the flux enters the cell) and by
// -dt_sub/dx_c (Ff - Fc) on a high face.
//
// One CTA per coarse block that has a finer face neighbour; its faces are taken one after the other with a
// barrier in between, because an edge / corner cell belongs to two / three faces (read-modify-write).
#include "f4_dev.hpp"

namespace f4 {
namespace {

template <int DIM, int N, int NV>
__global__ void __launch_bounds__(256) fluxfix_kernel(const __grid_constant__ FixParams p) {
  constexpr int P = N + 2 * NG, H = N / 2;
  constexpr int KM = (DIM == 3) ? N : 1;       // cells along t2
  constexpr int FS = N * KM;                   // cells of one block face
  constexpr size_t VS = (size_t)P * P * ((DIM == 3) ? P : 1);
  const DevFixBlock fb = p.fix[blockIdx.x];
  const double sdt = p.dt_dev ? (p.dtf * *p.dt_dev) * p.inv_dx_l[fb.level] : p.sdt_l[fb.level];
  const double* bflux = p.bflux;
  double* blk = p.out + (size_t)fb.blk * VS * NV;
  for (int f = 0; f < 2 * DIM; ++f) {
    if (fb.slot_c[f] >= 0) {
      const int a = f >> 1, side = f & 1;
      const double* bc = bflux + (size_t)fb.slot_c[f] * NV * FS;
      for (int idx = threadIdx.x; idx < NV * FS; idx += blockDim.x) {
        const int v = idx / FS, r = idx % FS, t2 = r / N, t1 = r % N;
        const int o1 = t1 / H, tt1 = t1 % H;
        const int o2 = (DIM == 3) ? t2 / H : 0, tt2 = (DIM == 3) ? t2 % H : 0;
        const double* bf = bflux + ((size_t)fb.slot_f[f][o1 + 2 * o2] * NV + v) * FS;
        // mean of the 2^(d-1) fine fluxes covering this coarse cell face, summed t1 first
        double sum = bf[(2 * tt2) * N + 2 * tt1] + bf[(2 * tt2) * N + 2 * tt1 + 1];
        if (DIM == 3) {
          sum += bf[(2 * tt2 + 1) * N + 2 * tt1];
          sum += bf[(2 * tt2 + 1) * N + 2 * tt1 + 1];
        }
        const double Ff = sum * ((DIM == 3) ? 0.25 : 0.5);
        const double corr = sdt * (Ff - bc[idx]);
        const int n = side ? N - 1 : 0;        // interior cell next to the face (0-based = its slot)
        int i, j, k;
        if (a == 0) { i = n; j = t1; k = t2; }
        else if (a == 1) { j = n; i = t1; k = t2; }
        else { k = n; i = t1; j = t2; }
        double* c = blk + (size_t)v * VS + ((size_t)k * P + j) * P + i;
        *c += side ? -corr : corr;
      }
    }
    __syncthreads();
  }
}

}  // namespace

cudaError_t launch_fluxfix(int dim, int n, int nvar, const FixParams& p, cudaStream_t s) {
  if (p.nfix <= 0) return cudaSuccess;
#define F4_FIX(D, NN)                                                                     \
  if (dim == D && n == NN) {                                                              \
    if (nvar == 1) fluxfix_kernel<D, NN, 1><<<p.nfix, 256, 0, s>>>(p);                    \
    else fluxfix_kernel<D, NN, D + 2><<<p.nfix, 256, 0, s>>>(p);                          \
    return cudaGetLastError();                                                            \
  }
  F4_FIX(2, 8) F4_FIX(2, 16) F4_FIX(2, 32) F4_FIX(3, 8) F4_FIX(3, 16) F4_FIX(3, 32)
#undef F4_FIX
  return cudaErrorInvalidValue;
}

}  // namespace f4
