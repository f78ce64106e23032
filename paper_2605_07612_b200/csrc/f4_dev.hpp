// Device-side interface between the C-ABI (f4_api.cu) and the kernels.
// Store layout: [state][block][var][kslot][jslot][islot],
// P = N + 2*NG slots per axis, slot(i) = i for i >= 0, i + P for i < 0.
#pragma once
#include <cuda_runtime.h>

#include <cstddef>
#include <cstdint>

namespace f4 {

constexpr int NG = 2;  // ghost layers compiled into the kernels
constexpr int MAXL = 20;  // refinement levels (f4_mesh_create checks max_level <= 18)

// meta = op | face << 2 | o1 << 5 | o2 << 6
struct DevRecord {
  int dst, src, meta, pad;
};

struct DevTransfer {
  int kind, dst, oct, pad;
  int src[8];
};

struct StageParams {
  const double* deriv;  // state whose time derivative is taken (ghosts filled)
  const double* prev0;  // eq. (5): out = dt_sub*F(deriv) + w0*prev0 + w1*prev1
  const double* prev1;  // may be nullptr (w1 ignored)
  const double* prev2;  // third / fourth previous state (classical RK4 eq. (11)); nullptr = none; prev3 needs prev2
  const double* prev3;
  double* out;
  double w0, w1, w2, w3, dt_sub;
  // time step resident on the device (f4_advance_cfl): when dt_dev != nullptr the kernels take dt_sub = dtf * *dt_dev and
  // dt_sub / dx = dt_sub * inv_dx_l[level] themselves (same operations, same order as the host path) and ignore
  // dt_sub / sdt_l
  const double* dt_dev;
  double dtf;
  double gamma;
  double inv_dx_l[MAXL];  // 1/dx per refinement level (1/dx_0 * 2^l, exact)
  double sdt_l[MAXL];     // dt_sub/dx per level: the factor of the flux difference in eq. (5)
  const int* level;     // per block
  int nblocks;
  int limiter, flux;
  unsigned long long* maxrate;  // bits of a non-negative double, atomicMax; nullptr = no CFL reduction
  const int* nbr;               // [nblocks][6] same-level neighbour per face or -1: fused same-level ghosts; nullptr = off
  int push_x;                   // with nbr: also push the x face layers of s_out into the neighbours' ghost cells
  // flux fixing: face-normal fluxes at refinement boundaries are stored "during the flux
  // computation" into bflux[slot][var][t2][t1]; bfslot[blk][6] = slot of that block face or -1; nullptr = off
  const int* bfslot;
  double* bflux;
  // gravity source term S = (0, rho g, rho g.u), eq. (20) PAPER.md:429-431 (general instances)
  double grav[3];
  double vel[3];   // scalar advection eq. (13): the uniform velocity field (f4_advect.cu)
  int has_grav;
  int grav_from;   // where the kernel finds s_deriv's own-cell conservative values: 0 prev0, 1 prev1, 2 load from deriv
};

// one coarse block with at least one finer face neighbour (flux fixing)
struct DevFixBlock {
  int blk, level;
  int slot_c[6];     // bflux slot of the coarse side of face f, or -1 when the neighbour across f is not finer
  int slot_f[6][4];  // bflux slots of the fine sides, index o1 + 2*o2 (hanging-face offsets)
};

struct GhostParams {
  double* state;
  const DevRecord* rec;
  int nrec;
  double theta;
  const double* bcv;   // [6][Nvar] uniform Dirichlet values / Neumann normal derivatives
  const double* bcdata;  // [n_bc_faces][Nvar][N^(d-1)] spatially varying boundary values, eq. (4)
  const int* level;    // per block (Neumann: dx of the block)
  double dx0;          // cell size of level 0
};

// every launcher returns the cudaError_t of the launch
// all same-level copies of a whole fill, by source block (one CTA per block and variable); nbr: [nblocks][6]
cudaError_t launch_srl_push(int dim, int n, int nvar, double* state, const int* nbr, int nblocks, cudaStream_t s);
cudaError_t launch_ghost(int dim, int n, int nvar, const GhostParams& p, cudaStream_t s);
cudaError_t launch_stage(int dim, int n, const StageParams& p, cudaStream_t s);
// dt[0] = cfl / rate with rate = the CFL maximum as bits of a double (0 and dt[1] = 1 if the rate is not a positive finite
// number); one thread
cudaError_t launch_dt_from_rate(const unsigned long long* maxrate, double cfl, double* dt, cudaStream_t s);
cudaError_t launch_maxrate(int dim, int n, const double* state, const int* level, int nblocks, double gamma,
                           double inv_dx0, unsigned long long* maxrate, cudaStream_t s);
cudaError_t launch_transfer(int dim, int n, int nvar, const double* old_state, double* new_state, const DevTransfer* plan,
                            int nplan, double theta, cudaStream_t s);
// layout kernels: natural (interior or padded) <-> wrapped padded store
cudaError_t launch_pack(int dim, int n, int nvar, double* store_state, const double* src, int b0, int nb, int with_ghosts,
                        cudaStream_t s);
cudaError_t launch_unpack(int dim, int n, int nvar, const double* store_state, double* dst, int b0, int nb, int with_ghosts,
                          cudaStream_t s);
cudaError_t launch_init_benign(int dim, int n, int nvar, double* store_state, int nb, double gamma, cudaStream_t s);
cudaError_t launch_block_sums(int dim, int n, int nvar, const double* state, int nb, double* sums /*[nb][nvar]*/, cudaStream_t s);
// the same reduction with its scratch in a static device array, finished on the device (f4_conserved_totals_noalloc):
// no allocation; nb <= F4_NOALLOC_MAX_BLOCKS, else cudaErrorInvalidValue; totals_dev: device, [nvar]
cudaError_t launch_totals_noalloc(int dim, int n, int nvar, const double* state, const int* level, int nb, double dx0,
                                  double* totals_dev, cudaStream_t s);
// coarse-side correction u -= -+ dt_sub/dx_c (mean fine flux - coarse flux) in the cells next to refinement boundaries
struct FixParams {
  double* out;              // the state the stage kernel just wrote
  const DevFixBlock* fix;
  int nfix;
  const double* bflux;
  double sdt_l[MAXL];       // dt_sub/dx per level
  const double* dt_dev;     // see StageParams: dt_sub / dx = (dtf * *dt_dev) * inv_dx_l[level]
  double dtf;
  double inv_dx_l[MAXL];
};
cudaError_t launch_fluxfix(int dim, int n, int nvar, const FixParams& p, cudaStream_t s);
// per-block refinement flags and indicator (device arrays) from a ghost-filled state
cudaError_t launch_flags(int dim, int n, int nvar, const double* state, int nblocks, int criterion, int var, double gamma,
                         const double params[4], int* flags, double* indicator, cudaStream_t s);
bool stage_supported(int dim, int n);
// scalar advection eq. (13), PAPER.md:364-370 (f4_advect.cu): symmetric limiters, at most two previous states
bool advect_supported(const StageParams& p);
cudaError_t launch_advect(int dim, int n, const StageParams& p, cudaStream_t s);
cudaError_t launch_advect2(int n, const StageParams& p, cudaStream_t s);   // 3D, two cells per thread (f4_advect2.cu)


}  // namespace f4
