/* f4.h -- C-ABI of the B200-native hot path of foap4 (arxiv/paper_2605_07612).
 *
 * One explicit Heun step of Euler's equations over every block of a
 * quadtree/octree AMR mesh: execution of a precomputed ghost-cell pattern
 * (section 2.6) + the per-block finite-volume update
 * (section 3.2), with mesh adapt / regrid transfer
 * (section 2.2).  Citations are /root/reference/PAPER.md:<line>;
 * "reading Ax" refers to DESIGN.md "Readings of the paper".
 *
 * General conventions
 *  - Every function returns F4_OK (0) or a negative F4_E* code; nothing throws
 *    across the ABI.  f4_last_error() gives the message of the last failure.
 *  - Pointers are HOST pointers unless the argument says "device".  The block
 *    store is DEVICE memory owned by the caller (e.g. a torch tensor) and lent
 *    to the mesh with f4_bind_storage(); the library owns only small metadata
 *    (block table, pattern records, staging buffers).
 *  - All device work is enqueued on the stream given to f4_bind_storage().
 *    Only f4_compute_dt, f4_get_state / f4_set_state with a host buffer,
 *    f4_adapt, f4_conserved_totals and f4_profile_get synchronise that stream.
 *  - There is no CPU fallback: a call that needs the device fails with
 *    F4_EUNBOUND / F4_ECUDA when no storage is bound or CUDA reports an error.
 *    Host-only calls (mesh_create, num_blocks, get_blocks, build_ghost_pattern,
 *    pattern_size, get_pattern and adapt on an UNBOUND mesh = topology only)
 *    work without a GPU.
 *  - Variables per cell: Nvar = dim+2 = (rho, rho*u_1..dim, E)
 *    eq. (14)-(15).  State arrays passed through this ABI are
 *    [block][var][k][j][i], i fastest (eq. 3), block order =
 *    the library's (Morton order over the brick; discover it with
 *    f4_get_blocks).  "interior" arrays have N cells per axis, "padded" arrays
 *    N+2*Ng per axis in natural order (index p = i+Ng for i in [-Ng, N+Ng)).
 *    In 2D the k extent is 1.
 *  - Device layout of the bound store: state-major,
 *    then block, var, and a ghost-WRAPPED padded box: along every axis slot
 *    s(i) = i for i >= 0 (interior, then high ghosts) and i + P for i < 0 (low
 *    ghosts last), so that interior rows start on 32-byte sectors; the four
 *    x-ghost slots of each row pair (2m, 2m+1) are regrouped by side
 *    ([hi(2m) hi(2m+1)] in row 2m, [lo(2m) lo(2m+1)] in row 2m+1) so that every
 *    32-byte ghost sector has exactly one source block.
 */
#ifndef F4_H
#define F4_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct f4_mesh f4_mesh; /* opaque: host mesh + pattern + device metadata */

enum {
  F4_OK = 0,
  F4_EINVAL = -1,    /* bad argument (N odd, N < Ng, 2*Ng > N, dim not 2/3, ...) */
  F4_ENOBLOCKS = -2, /* mesh would exceed max_blocks (store is statically sized) */
  F4_ECUDA = -3,     /* a CUDA call failed; message in f4_last_error */
  F4_EUNBOUND = -4,  /* device work requested but no storage bound */
  F4_EUNBALANCED = -5, /* face connectivity found a >1 level jump */
  F4_EUNSUPPORTED = -6 /* configuration outside the compiled kernel set (see f4_bind_storage) */
};

/* physical boundary kinds per face direction */
enum {
  F4_BC_PERIODIC = 0, /* via connectivity */
  F4_BC_OUTFLOW = 1,  /* uniform Neumann, zero normal derivative: ghost = nearest interior layer (reading A10) */
  F4_BC_KEEP = 2,     /* no record: ghosts on that face stay as the caller wrote them (the "boundary values set
                         analytically" of the linear-field test).  Contract: the library never writes
                         these ghost cells, so the caller must set them (f4_set_state with_ghosts = 1) in EVERY temporal
                         state that f4_advance differentiates (intermediate Runge-Kutta states start from a benign
                         constant, rho = 1, u = 0, p = 1), and again after f4_adapt (the regrid transfer carries
                         interior cells only). */
  F4_BC_DIRICHLET = 3, /* uniform value u_b per face direction and variable (f4_set_bc_values): ghost layer g mirrors
                          interior layer g through the face, u_ghost = 2 u_b - u_interior (reading A10) */
  F4_BC_NEUMANN = 4,   /* uniform outward normal derivative u_b': ghost layer g = first interior layer + g dx u_b'
                          (reading A10b; u_b' = 0 is F4_BC_OUTFLOW) */
  F4_BC_DATA = 5       /* spatially varying boundary values bc_data (eq. 4), one value per face cell
                          and variable, supplied by a callback (f4_set_bc_callback); same mirror rule as Dirichlet */
};

enum { F4_LIM_VANLEER = 0, F4_LIM_MINMOD = 1, F4_LIM_MC = 2, /* PAPER.md:322-326; reading A1 */
       F4_LIM_KOREN = 3, F4_LIM_WENO3 = 4 };                 /* 2-ghost schemes of PAPER.md:325-326; reading A1b */
enum { F4_FLUX_HLL = 0, F4_FLUX_RUSANOV = 1 };                 /* PAPER.md:328; reading A2 */
/* Runge-Kutta schemes of the restricted class eq. (5): Heun = SSPRK(2,2) eq. (6)-(7) (default),
 * forward Euler, SSPRK(3,3), SSPRK(4,3) ("optimal SSP schemes with two, three and four stages"),
 * classical RK4 eq. (8)-(11).  Temporal states needed (n_states of f4_mesh_create): 2, 2, 3, 3, 4. */
enum { F4_RK_HEUN = 0, F4_RK_EULER = 1, F4_RK_SSP33 = 2, F4_RK_SSP43 = 3, F4_RK_RK4 = 4, F4_RK_N = 5 };
enum { F4_CRIT_LOHNER = 0, F4_CRIT_PJUMP = 1 };                 /* PAPER.md:349-362 eq. (12); reading A15 */

/* pattern record ops (data-flow naming) */
enum {
  F4_OP_SRL = 0, /* same-level copy, round R1 */
  F4_OP_BC = 1,  /* physical boundary (outflow), round R1 */
  F4_OP_F2C = 2, /* restriction of one fine neighbour into a quarter (3D) / half (2D) of a coarse ghost face, R1 */
  F4_OP_C2F = 3  /* limited prolongation from the coarse neighbour into a fine ghost face, round R2 */
};

/* ---- mesh_create(dim, block_n, n_ghost, levels) ----------------------------
 * Brick of brick[0] x brick[1] (x brick[2]) trees refined
 * uniformly to base_level; leaves are blocks of block_n^dim cells with n_ghost
 * ghost layers.  Domain: [0, brick[a]/max(brick)] along
 * axis a, cubic cells of size dx_l = 1/(max(brick) * 2^l * block_n) (reading
 * A13).  bc_kind[6]: per face direction -x,+x,-y,+y,-z,+z; an
 * axis is periodic only if both its faces say so.  n_states >= 2 (Heun needs
 * two); max_blocks sizes the store.  Host only.
 * Errors: F4_EINVAL, F4_ENOBLOCKS (base mesh larger than max_blocks). */
int f4_mesh_create(int dim, int block_n, int n_ghost, const int brick[3], int base_level, int max_level,
                   const int bc_kind[6], double gamma, int n_states, int max_blocks, f4_mesh **out);
int f4_mesh_destroy(f4_mesh *m);

/* limiter / flux scheme / prolongation theta of eq. (1) (default van Leer, HLL, theta=1). */
int f4_set_options(f4_mesh *m, int limiter, int flux_scheme, double theta);

/* Flux fixing at refinement boundaries (section 2.7; the paper's f4_fix_c2f_flux), default off.
 * When on, every stage of f4_advance stores the face-normal fluxes of block faces whose neighbour is coarser or
 * finer ("bflux"; device memory owned by the library, sized by f4_build_ghost_pattern / f4_adapt) and
 * then corrects the coarse cells next to such a face by -+ dt_sub/dx_c * (mean of the 2^(dim-1) fine fluxes - coarse
 * flux), which makes the update conservative across levels.  A mesh without refinement boundaries
 * takes exactly the same path as with the switch off.  Host only; takes effect at the next f4_advance. */
int f4_set_flux_fix(f4_mesh *m, int on);

/* Physics (default Euler gas dynamics, Nvar = dim + 2).  F4_PHYS_ADVECTION: the scalar advection
 * equation (13) of PAPER.md:364-370, d(rho)/dt + div(rho v) = 0 with the uniform velocity field `velocity` (host,
 * [3], the first dim entries are used): ONE variable per cell, primitive = conservative, wave speeds min(v_i, 0) and
 * max(v_i, 0), i.e. the upwind flux; f4_compute_dt = CFL dx_finest / sum_i |v_i| without a device pass.  Limiters:
 * van Leer, minmod, MC; Runge-Kutta schemes with at most two previous states; no gravity; the pressure-jump
 * criterion is not defined.  Must be called before f4_bind_storage (the storage size changes with Nvar).
 * Errors: F4_EINVAL (unknown physics, NaN velocity, already bound). */
enum { F4_PHYS_EULER = 0, F4_PHYS_ADVECTION = 1 };
int f4_set_physics(f4_mesh *m, int physics, const double velocity[3]);
/* variables per cell of the mesh's physics */
int f4_num_vars(const f4_mesh *m);

/* bytes of the block store: n_states*max_blocks*Nvar*P^dim*8. */
size_t f4_storage_bytes(const f4_mesh *m);

/* Lend the DEVICE store (>= f4_storage_bytes, 256-byte aligned) and a CUDA
 * stream (cudaStream_t as void*, NULL = default stream).  Ownership stays with
 * the caller, who must keep it alive until destroy/rebind.  Initialises every
 * padded cell (unused edge/corner ghosts included) to a benign state
 * (rho=1, u=0, p=1) and uploads the block table.  The CUDA kernels are
 * compiled for n_ghost == 2 and (dim, block_n) in {(2,8), (2,16), (3,8), (3,16),
 * (3,32)}: anything else gives F4_EUNSUPPORTED.  Errors: F4_EINVAL, F4_ECUDA. */
int f4_bind_storage(f4_mesh *m, void *dev_ptr, size_t bytes, void *cuda_stream);

int f4_num_blocks(const f4_mesh *m);
/* Block metadata: refinement level, integer block coordinates
 * on the level's grid [nb][3], spatial origin (low corner) [nb][3], cell size
 * [nb].  Any output pointer may be NULL. */
int f4_get_blocks(const f4_mesh *m, int *level, int *coords, double *origin, double *dx);

/* ---- set_state / get_state -------------------------------------------------
 * Copy a state between caller memory and the store.  with_ghosts = 0: interior
 * array [nb][Nvar][N..]; 1: natural padded array [nb][Nvar][P..] (ghosts
 * included).  *_is_device says where the caller's buffer lives; a host buffer
 * is staged through pinned memory in chunks and the call returns after the
 * last chunk (synchronises).  State s in [0, n_states). */
int f4_set_state(f4_mesh *m, int state, const double *src, int src_is_device, int with_ghosts);
int f4_get_state(f4_mesh *m, int state, double *dst, int dst_is_device, int with_ghosts);

/* ---- build_ghost_pattern ---------------------------------------------------
 * Host: face connectivity -> device-resident record lists for round R1
 * {SRL, BC, F2C} and round R2 {C2F}, sorted by
 * (destination block, face direction).  Uploaded when storage is bound.
 * Called automatically by mesh_create, adapt.  Errors: F4_EUNBALANCED. */
int f4_build_ghost_pattern(f4_mesh *m);
int f4_pattern_size(const f4_mesh *m, int *n_r1, int *n_r2);
/* records[n][6] = {op, face, dst_block, src_block, off_t1, off_t2}, R1 first.
 * face: 0..5 = -x,+x,-y,+y,-z,+z of the DESTINATION block; off_*: hanging-face
 * offset of the fine block within its group.  F4_OP_BC records
 * carry the boundary kind in (off_t1, off_t2): (0,0) outflow, (1,0) Dirichlet,
 * (0,1) Neumann, (1,1) bc_data, whose src_block field is the face index ibf. */
int f4_get_pattern(const f4_mesh *m, int *records);

/* ---- fill_ghosts -----------------------------------------------------------
 * Execute the whole pattern on one state: R1 = one kernel for all same-level
 * copies (by source block) and one batched kernel over the BC / F2C records,
 * then one batched kernel for R2 iff the mesh has refinement boundaries
 * (PAPER.md:202-212).  Asynchronous.  (Inside f4_advance the same-level copies of the state a
 * stage kernel produces are pushed by that kernel itself, and only the
 * BC / F2C / C2F records are executed by the batched kernel.) */
int f4_fill_ghosts(f4_mesh *m, int state);

/* ---- compute_dt ------------------------------------------------------------
 * dt = cfl / max over interior cells of sum_dim (|u_dim| + c)/dx_l (PAPER.md:336,
 * 339, eq. 16; readings A4-A6).  After f4_advance the maximum of the new
 * state 0 is already on the device (fused into the last stage); otherwise a
 * reduction kernel runs.  Synchronises to read one double back. */
int f4_compute_dt(f4_mesh *m, int state, double cfl, double *dt_out);

/* Uniform boundary data of the F4_BC_DIRICHLET / F4_BC_NEUMANN faces ("a Dirichlet boundary condition
 * with a uniform value u = u_b ... stored per face direction and per variable ... and the same ... for a Neumann
 * boundary condition with a uniform normal derivative"): values[6][Nvar], face directions -x,+x,-y,+y,-z,+z, stored
 * (conservative) variables; entries of other faces are ignored.  Default: zeros.  Copied to the device when storage
 * is bound (host call otherwise); takes effect at the next ghost fill.  Spatially varying values (eq. 4) are the
 * F4_BC_DATA kind below. */
int f4_set_bc_values(f4_mesh *m, const double *values);

/* Spatially varying boundary values, eq. (4): bc_data(i, j, ivar, ibf), ibf = 0 .. n_faces-1 over the
 * block faces on a physical boundary whose direction has kind F4_BC_DATA, in (block, face) order.  "A callback function
 * has to be stored so that boundary data is automatically updated when the mesh changes": fn is called by
 * f4_build_ghost_pattern, f4_bind_storage, f4_adapt (when the mesh changed) and f4_update_bc_data ("for temporally
 * varying boundary conditions this callback function can be called by the application code whenever necessary") with
 * the face list block[n_faces], face[n_faces] (block geometry: f4_get_blocks) and must fill the HOST array
 * bc_data[n_faces][Nvar][N^(dim-1)] (t1 fastest; t1 < t2 the transverse axes in x,y,z order) with stored
 * (conservative) variables at the face-cell centres; the library copies it to the device.  Ghost layer g then mirrors
 * interior layer g: u_ghost = 2 bc_data - u_interior.  Without a callback the values are zero. */
typedef void (*f4_bc_data_fn)(void *user, int n_faces, const int *block, const int *face, double *bc_data);
int f4_set_bc_callback(f4_mesh *m, f4_bc_data_fn fn, void *user);
int f4_update_bc_data(f4_mesh *m);
int f4_num_bc_faces(const f4_mesh *m);

/* Gravitational acceleration g[3] of the source term S = (0, rho g, rho g.u), eq. (20), evaluated
 * from the primitives of s_deriv in each cell and added to the flux divergence in every sub-step (PAPER.md:334 step i).
 * Default (0,0,0): no source term, the path every BASELINE config times.  Components beyond `dim` are ignored. */
int f4_set_gravity(f4_mesh *m, const double g[3]);

/* Select the time integrator used by f4_advance (F4_RK_*).  Every sub-step is one launch of the fused stage kernel
 * in the form of eq. (5), u(s_out) = dt_sub F(u(s_deriv)) + sum_i w_i u(s_prev,i), n_prev <= 4, preceded by the ghost
 * fill of s_deriv; the CFL maximum of the new state is fused into the last sub-step.  GCUPS counts one
 * cell update per sub-step.  Errors: F4_EINVAL (unknown scheme, or n_states too small). */
int f4_set_rk_scheme(f4_mesh *m, int scheme);

/* ---- advance(dt) -----------------------------------------------------------
 * One step of the selected Runge-Kutta scheme (f4_set_rk_scheme); default:
 * one step of Heun's method, eq. (6)-(7), as two sub-steps of
 * eq. (5): fill_ghosts(0); u1 = dt F(ut) + ut -> state 1; fill_ghosts(1);
 * u = dt/2 F(u1) + (ut + u1)/2 -> state 0 (in place).  F = limited primitive
 * reconstruction + HLL/Einfeldt flux divergence.
 * Asynchronous; result in state 0, whose ghosts are then stale. */
int f4_advance(f4_mesh *m, double dt);

/* compute_dt + advance in one call without a host round trip: dt = cfl / (CFL maximum of state 0) stays on the device.
 * The maximum is the one the previous f4_advance / f4_advance_cfl fused into its last stage (forward
 * Euler "provide[s] a limit for the next time step"), else one reduction pass runs first; a one-thread kernel turns
 * it into dt, and the stage kernels read dt from device memory (same operations and order as with a host dt: the
 * results are those of f4_compute_dt followed by f4_advance).  Nothing synchronises: a step loop of f4_advance_cfl
 * calls is enqueued as fast as the host can launch.  f4_last_dt reads the last step's dt back (synchronises);
 * it returns F4_EINVAL if the wave speed was zero or not finite -- that step then ran with dt = 0.
 * Scalar advection: dt is known on the host (constant wave speed); same call, no device scalar. */
int f4_advance_cfl(f4_mesh *m, double cfl);
int f4_last_dt(f4_mesh *m, double *dt_out);

/* ---- refinement flags on the device ----------------------------------------
 * Per-block flags for f4_adapt from state `state` (its ghosts are filled first: the criteria read the first layer
 * of face ghosts, never edge / corner ghosts).
 *   F4_CRIT_LOHNER  PAPER.md:349-362 eq. (12) on stored variable `var` (0 = density, the paper's choice,
 *                   PAPER.md:560): per cell and direction E_n = |u_{n-1} - 2u_n + u_{n+1}| /
 *                   (eps_abs + |u_n - u_{n-1}| + |u_{n+1} - u_n| + eps (|u_{n-1}| + 2|u_n| + |u_{n+1}|)),
 *                   |E| = sqrt(sum_n E_n^2); params = {c_refine, c_derefine, eps, eps_abs}.
 *   F4_CRIT_PJUMP   BASELINE config 5 (reading A15): J = max over face-adjacent cell pairs (interior-interior,
 *                   interior-first ghost layer) of |p_a - p_b| / min(p_a, p_b); params = {hi, lo, -, -}.
 * flag = +1 if the block maximum exceeds params[0] ("in one cell"), -1 if it is below params[1] ("in all cells"),
 * else 0; strict comparisons.  flags_out[nb] (host, required) and indicator_out[nb] (host, may be NULL: the block
 * maxima) are filled; synchronises.  Errors: F4_EINVAL, F4_EUNBOUND, F4_ECUDA. */
int f4_refine_flags(f4_mesh *m, int state, int criterion, int var, const double params[4], int *flags_out,
                    double *indicator_out);

/* ---- adapt(refine_flags) ---------------------------------------------------
 * flags[nb]: >0 refine, <0 may coarsen, 0 keep.  refine, then
 * coarsen complete families (one level per call, never below base_level or
 * above max_level), then 2:1 balance with corner connectivity (
 * reading A11).  If the mesh changed: state 0 is transferred (copy /
 * prolongation / restriction; ghosts of state 0 are filled
 * first), the pattern is rebuilt, *changed_out = 1.  On an unbound mesh only
 * the topology changes.  Other states become undefined.  Synchronises.
 * Errors: F4_ENOBLOCKS (nothing modified), F4_ECUDA. */
int f4_adapt(f4_mesh *m, const int *refine_flags, int *changed_out);

/* The same regrid split in two, so that the host part (refine / coarsen / balance and the pattern records of the new
 * mesh) overlaps device work: f4_adapt_begin copies the flags and starts that part on a
 * worker thread, on a copy of the mesh; the mesh in use stays valid, so f4_compute_dt / f4_advance (and nothing that
 * changes the mesh or its state layout) may be called in between.  f4_adapt_end waits for the worker and, if the mesh
 * changes, does what f4_adapt does on the device (ghost fill, transfer of state 0 AS IT IS NOW, record upload).  The
 * new mesh is the one f4_adapt would have built from the same flags; only the moment of the switch differs.
 * Errors: F4_EINVAL (begin while pending, end without begin, f4_adapt while pending), else as f4_adapt. */
int f4_adapt_begin(f4_mesh *m, const int *refine_flags);
int f4_adapt_end(f4_mesh *m, int *changed_out);

/* sum over interior cells of u * dx^dim, per variable [Nvar] (for conservation tests). */
int f4_conserved_totals(f4_mesh *m, int state, double *totals);

/* The same totals for callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that
 * forbid cudaMalloc): the per-block sums go to a STATIC device array inside the library instead of the mesh's
 * cudaMalloc'ed scratch, and a second kernel finishes the sum on the device.  The call allocates nothing on the
 * device or the host (no cudaMalloc / cudaFree, no allocating library routine), enqueues two kernels on the mesh's
 * stream and does not synchronise.
 *   totals_dev  DEVICE pointer, [Nvar] doubles, owned by the caller; valid once the stream reaches this point.
 * Limit: at most F4_NOALLOC_MAX_BLOCKS blocks (the array holds F4_NOALLOC_MAX_BLOCKS * 5 doubles = 1.25 MiB on every
 * GPU that loads the library, until the process exits); a larger mesh gives F4_EINVAL and a message that says so.
 * The array is shared by every mesh and every call on a device and keeps the last call's contents (each call
 * overwrites the entries it reads, nothing has to be cleared): calls that OVERLAP on the GPU -- two meshes on two
 * streams -- race on it; calls on one stream do not.  The first call on a device also asks the CUDA runtime for the
 * array's device address (cudaGetSymbolAddress): make that call outside a graph capture.
 * Result: equal to f4_conserved_totals to ~1e-15 relative (same per-block sums; the sum over blocks is carried in
 * double-double here, in long double there).  Errors: F4_EINVAL (null / host pointer, too many blocks),
 * F4_EUNBOUND, F4_ECUDA. */
#define F4_NOALLOC_MAX_BLOCKS 32768
int f4_conserved_totals_noalloc(f4_mesh *m, int state, double *totals_dev);

/* ---- measurement helpers ---------------------------------------------------
 * f4_profile_enable(1): bracket every kernel class with CUDA events on the
 * bound stream.  f4_profile_get: accumulated milliseconds and launch counts
 * since the last reset, classes: 0 ghost R1, 1 ghost R2, 2 stage, 3 dt reduce,
 * 4 regrid transfer, 5 layout (set/get/init).  f4_launch_count: kernels
 * launched by this mesh since creation (always counted). */
enum { F4_PROF_R1 = 0, F4_PROF_R2 = 1, F4_PROF_STAGE = 2, F4_PROF_DT = 3, F4_PROF_REGRID = 4, F4_PROF_LAYOUT = 5, F4_PROF_N = 6 };
int f4_profile_enable(f4_mesh *m, int on);
int f4_profile_get(f4_mesh *m, double ms[F4_PROF_N], long long launches[F4_PROF_N], int reset);
long long f4_launch_count(const f4_mesh *m);
/* host wall time (ms) of the last f4_adapt that changed the mesh, by part: [0] refine / coarsen / balance + pattern
 * records on the host, [1] regrid transfer kernel + wait, [2] record upload. */
int f4_last_adapt_ms(const f4_mesh *m, double ms[3]);

const char *f4_last_error(const f4_mesh *m);
const char *f4_version(void);

#ifdef __cplusplus
}
#endif
#endif /* F4_H */
