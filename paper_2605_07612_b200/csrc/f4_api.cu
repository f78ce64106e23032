// C-ABI of the f4 library (include/f4.h): argument checking, device metadata,
// launch sequencing.  All arithmetic of the path lives in f4_ghost.cu / f4_stage.cu.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <chrono>
#include <string>
#include <thread>
#include <vector>

#include "../../include/f4.h"
#include "f4_dev.hpp"
#include "f4_mesh.hpp"

using namespace f4;

struct f4_mesh {
  HostMesh hm;
  double gamma = 1.4, theta = 1.0;
  int limiter = F4_LIM_VANLEER, flux = F4_FLUX_HLL;
  int rk = F4_RK_HEUN;
  double grav[3] = {0.0, 0.0, 0.0};
  int physics = F4_PHYS_EULER;           // F4_PHYS_ADVECTION: scalar advection eq. (13) with the uniform velocity vel
  double vel[3] = {0.0, 0.0, 0.0};
  double bcv[6 * 5] = {0.0};     // uniform Dirichlet values / Neumann derivatives [6][nvar]
  double* d_bcv = nullptr;
  // spatially varying boundary data (eq. 4): faces in record order, host copy, device copy
  f4_bc_data_fn bc_fn = nullptr;
  void* bc_user = nullptr;
  std::vector<int> bc_block, bc_face;
  std::vector<double> bc_host;
  double* d_bcdata = nullptr;
  size_t cap_bcdata = 0;
  int n_states = 2;
  int nvar = 5;
  size_t vs = 0, bs = 0, state_doubles = 0;  // doubles per (block,var), per block, per state
  // device
  bool bound = false;
  int device = -1;            // the device dev_ptr of f4_bind_storage lives on: every device call runs there
  double* store = nullptr;
  cudaStream_t stream = nullptr;
  std::vector<int> phys;  // logical state -> physical state slab
  int* d_level = nullptr;
  DevRecord* d_r1 = nullptr;
  DevRecord* d_r2 = nullptr;
  DevRecord* d_r1n = nullptr;  // R1 without the same-level copies (the stage kernel pushes / gathers those itself)
  DevRecord* d_r1z = nullptr;  // R1 without the x same-level copies: d_r1n plus the y- and z-face same-level copies
  DevRecord* d_r1c = nullptr;  // d_r1n plus the y- / z-face same-level copies into blocks that are C2F sources
  DevRecord* d_r1f = nullptr;  // d_r1c plus all x-face same-level copies (flux-fixing mode: the stage does not push x)
  int* d_nbr = nullptr;        // [max_blocks][6] same-level neighbour per face or -1
  int nb_dev = 0;              // blocks of the mesh whose tables and records are on the device (during a regrid the
                               // host mesh is already the new one while the device still holds the old pattern)
  // all of the above (and d_bfslot, d_fix) point into one device blob, uploaded from one pinned host buffer
  char* d_meta = nullptr;
  char* h_meta = nullptr;
  size_t cap_meta = 0;
  cudaEvent_t meta_ev = nullptr;
  int n_r1 = 0, n_r2 = 0, n_r1n = 0, n_r1z = 0, n_r1c = 0, n_r1f = 0;
  // per logical state, same-level face ghosts: 0 = stale, 1 = x faces up to date (pushed by the stage kernel that
  // produced the state; its y ghost rows and z ghost planes were never written because stage kernels fetch them
  // from the neighbours' interiors), 2 = all faces up to date
  std::vector<char> srl_valid;
  DevTransfer* d_plan = nullptr;
  size_t cap_plan = 0;
  // flux fixing at refinement boundaries
  bool flux_fix = false;
  int* d_bfslot = nullptr;       // [max_blocks][6] bflux slot of a block face at a refinement boundary, or -1
  DevFixBlock* d_fix = nullptr;  // coarse blocks with a finer face neighbour
  double* d_bflux = nullptr;     // [n_bfslots][nvar][N^(d-1)]
  size_t cap_bflux = 0;
  int n_fix = 0, n_bfslots = 0;
  unsigned long long* d_maxrate = nullptr;
  double* d_dt = nullptr;        // [2]: time step of f4_advance_cfl, error flag
  bool dt_on_device = false;
  double host_dt = 0.0;
  double* d_sums = nullptr;
  int* d_flags = nullptr;        // [max_blocks] refinement flags
  double* d_indicator = nullptr; // [max_blocks] block maxima of the refinement indicator
  double* d_stage = nullptr;  // staging for host set/get
  size_t stage_bytes = 0;
  bool rate_valid = false;
  // measurement
  bool prof = false;
  // a fixed pool of event pairs created by f4_profile_enable (no cudaEventCreate inside a timed loop); when the pool
  // is used up the recorded pairs are folded into prof_ms (one stream synchronisation) and the pool starts again
  struct Ev { int cls; cudaEvent_t a, b; };
  static constexpr size_t EV_POOL = 2048;
  std::vector<Ev> evs;
  size_t evs_used = 0;
  void fold_events() {
    if (evs_used == 0) return;
    cudaEventSynchronize(evs[evs_used - 1].b);
    for (size_t q = 0; q < evs_used; ++q) {
      float t = 0.f;
      if (cudaEventElapsedTime(&t, evs[q].a, evs[q].b) == cudaSuccess) prof_ms[evs[q].cls] += t;
    }
    evs_used = 0;
  }
  double prof_ms[F4_PROF_N] = {0, 0, 0, 0, 0, 0};
  long long prof_n[F4_PROF_N] = {0, 0, 0, 0, 0, 0};
  long long launches = 0;
  // asynchronous regrid (f4_adapt_begin / f4_adapt_end): the host part runs on a worker thread on a copy of the mesh
  std::thread worker;
  bool pending = false;
  HostMesh hm_next;
  std::vector<int> flags_next;
  std::vector<Transfer> plan_next;
  bool changed_next = false;
  int rc_next = 0;
  std::string err_next;
  double adapt_ms[3] = {0.0, 0.0, 0.0};   // last f4_adapt: host mesh + pattern, transfer kernel + wait, record upload
  std::string err;

  double* state_ptr(int s) { return store + (size_t)phys[s] * state_doubles; }
};

namespace {

int fail(f4_mesh* m, int code, const std::string& msg) {
  if (m) m->err = msg;
  return code;
}
int cuda_fail(f4_mesh* m, cudaError_t e, const char* what) {
  return fail(m, F4_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define CU(call)                                          \
  do {                                                    \
    cudaError_t e_ = (call);                              \
    if (e_ != cudaSuccess) return cuda_fail(m, e_, #call); \
  } while (0)

// Makes the mesh's device current for the duration of a call and restores the caller's (a C-ABI that takes any
// pointer / stream must not depend on which device happens to be current)
struct DeviceScope {
  int prev = -1;
  bool switched = false;
  explicit DeviceScope(const f4_mesh* m) {
    if (m && m->device >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != m->device)
      switched = cudaSetDevice(m->device) == cudaSuccess;
  }
  ~DeviceScope() {
    if (switched) cudaSetDevice(prev);
  }
};

struct Scope {  // event bracket around one kernel launch
  f4_mesh* m;
  f4_mesh::Ev* ev = nullptr;
  Scope(f4_mesh* m_, int cls) : m(m_) {
    m->launches++;
    m->prof_n[cls]++;
    if (m->prof && !m->evs.empty()) {
      if (m->evs_used == m->evs.size()) m->fold_events();
      ev = &m->evs[m->evs_used++];
      ev->cls = cls;
      cudaEventRecord(ev->a, m->stream);
    }
  }
  ~Scope() {
    if (ev) cudaEventRecord(ev->b, m->stream);
  }
};

template <typename T>
int ensure(f4_mesh* m, T*& ptr, size_t& cap, size_t need) {
  if (need <= cap) return F4_OK;
  if (ptr) cudaFree(ptr);
  ptr = nullptr;
  size_t ncap = need + need / 2 + 64;
  CU(cudaMalloc((void**)&ptr, ncap * sizeof(T)));
  cap = ncap;
  return F4_OK;
}

// (re)evaluate the boundary-data callback for the current face list and copy the values to the device
int refresh_bc_data(f4_mesh* m) {
  m->bc_block.clear();
  m->bc_face.clear();
  for (const Record& r : m->hm.r1)
    if (r.op == F4_OP_BC && r.o1 && r.o2) { m->bc_block.push_back(r.dst); m->bc_face.push_back(r.face); }
  const size_t nf = m->bc_block.size();
  const size_t per_face = (size_t)m->nvar * m->hm.N * (m->hm.dim == 3 ? m->hm.N : 1);
  m->bc_host.assign(nf * per_face, 0.0);
  if (nf && m->bc_fn) m->bc_fn(m->bc_user, (int)nf, m->bc_block.data(), m->bc_face.data(), m->bc_host.data());
  if (!m->bound || !nf) return F4_OK;
  int rc;
  if ((rc = ensure(m, m->d_bcdata, m->cap_bcdata, nf * per_face))) return rc;
  CU(cudaMemcpyAsync(m->d_bcdata, m->bc_host.data(), nf * per_face * sizeof(double), cudaMemcpyHostToDevice, m->stream));
  CU(cudaStreamSynchronize(m->stream));
  std::fill(m->srl_valid.begin(), m->srl_valid.end(), 0);   // boundary ghosts of every state are stale now
  return F4_OK;
}

// Pattern records, block levels, neighbour table and flux-fixing tables of the current mesh go to the device as ONE
// blob: packed into a pinned host buffer and sent by a single asynchronous copy on the bound stream (kernels enqueued
// afterwards are ordered behind it; the host buffer is guarded by an event until the copy has finished).
int upload_meta(f4_mesh* m) {
  {
    int rc0 = refresh_bc_data(m);
    if (rc0) return rc0;
  }
  if (!m->bound) return F4_OK;
  const int nb = (int)m->hm.leaves.size();
  auto dev = [](const Record& r) { return DevRecord{r.dst, r.src, r.op | r.face << 2 | r.o1 << 5 | r.o2 << 6, 0}; };
  std::vector<char> c2f_src(nb, 0);   // coarse blocks whose cells (face ghosts included) a prolongation stencil reads
  for (const Record& r : m->hm.r2) c2f_src[r.src] = 1;
  // sizes of the record lists (see the d_r1* members)
  size_t n_a = m->hm.r1.size(), n_b2 = m->hm.r2.size(), n_an = 0, n_az = 0, n_ac = 0, n_af = 0;
  for (const Record& r : m->hm.r1) {
    const bool srl = r.op == F4_OP_SRL;
    n_an += !srl;
    n_az += (!srl || r.face >= 2);
    n_ac += (!srl || (r.face >= 2 && c2f_src[r.dst]));
    n_af += (!srl || r.face < 2 || c2f_src[r.dst]);
  }
  // flux fixing: a bflux slot for every block face whose neighbour is finer (F2C records end there) or coarser
  // (a C2F record ends there); one DevFixBlock per coarse block with a finer face neighbour
  std::vector<int> fix_of(nb, -1);
  size_t n_fix = 0;
  for (const Record& r : m->hm.r1)
    if (r.op == F4_OP_F2C && fix_of[r.dst] < 0) fix_of[r.dst] = (int)n_fix++;
  // blob layout (every section 256-byte aligned)
  size_t off = 0;
  auto section = [&](size_t bytes) { size_t o = off; off += (bytes + 255) & ~(size_t)255; return o; };
  const size_t o_level = section((size_t)nb * sizeof(int)), o_nbr = section((size_t)nb * 6 * sizeof(int)),
               o_bfs = section((size_t)nb * 6 * sizeof(int)), o_a = section(n_a * sizeof(DevRecord)),
               o_b2 = section(n_b2 * sizeof(DevRecord)), o_an = section(n_an * sizeof(DevRecord)),
               o_az = section(n_az * sizeof(DevRecord)), o_ac = section(n_ac * sizeof(DevRecord)),
               o_af = section(n_af * sizeof(DevRecord)), o_fix = section(n_fix * sizeof(DevFixBlock));
  const size_t total = off;
  if (m->meta_ev) CU(cudaEventSynchronize(m->meta_ev));   // the previous upload has left the host buffer
  if (total > m->cap_meta) {
    CU(cudaStreamSynchronize(m->stream));   // kernels in flight still read the old blob
    if (m->d_meta) cudaFree(m->d_meta);
    if (m->h_meta) cudaFreeHost(m->h_meta);
    m->d_meta = m->h_meta = nullptr;
    m->cap_meta = 0;
    const size_t ncap = total + total / 2 + 4096;
    CU(cudaMalloc((void**)&m->d_meta, ncap));
    CU(cudaHostAlloc((void**)&m->h_meta, ncap, cudaHostAllocDefault));
    m->cap_meta = ncap;
  }
  if (!m->meta_ev) CU(cudaEventCreateWithFlags(&m->meta_ev, cudaEventDisableTiming));
  char* h = m->h_meta;
  int* lev = (int*)(h + o_level);
  int* nbr = (int*)(h + o_nbr);
  int* bfslot = (int*)(h + o_bfs);
  DevRecord *a = (DevRecord*)(h + o_a), *b2 = (DevRecord*)(h + o_b2), *an = (DevRecord*)(h + o_an),
            *az = (DevRecord*)(h + o_az), *ac = (DevRecord*)(h + o_ac), *af = (DevRecord*)(h + o_af);
  DevFixBlock* fix = (DevFixBlock*)(h + o_fix);
  for (int b = 0; b < nb; ++b) lev[b] = m->hm.leaves[b].level;
  for (int q = 0; q < nb * 6; ++q) { nbr[q] = -1; bfslot[q] = -1; }
  {
    size_t qa = 0, qn = 0, qz = 0, qc = 0, qf = 0;
    for (const Record& r : m->hm.r1) {
      const DevRecord dr = dev(r);
      const bool srl = r.op == F4_OP_SRL;
      a[qa++] = dr;
      if (srl) nbr[(size_t)r.dst * 6 + r.face] = r.src;
      else an[qn++] = dr;
      if (!srl || r.face >= 2) az[qz++] = dr;
      if (!srl || (r.face >= 2 && c2f_src[r.dst])) ac[qc++] = dr;
      if (!srl || r.face < 2 || c2f_src[r.dst]) af[qf++] = dr;
    }
    size_t qb = 0;
    for (const Record& r : m->hm.r2) b2[qb++] = dev(r);
  }
  int nslots = 0;
  for (const Record& r : m->hm.r1)
    if (r.op == F4_OP_F2C && bfslot[(size_t)r.dst * 6 + r.face] < 0) bfslot[(size_t)r.dst * 6 + r.face] = nslots++;
  for (const Record& r : m->hm.r2)
    if (r.op == F4_OP_C2F) bfslot[(size_t)r.dst * 6 + r.face] = nslots++;
  for (int b = 0; b < nb; ++b)
    if (fix_of[b] >= 0) {
      DevFixBlock& fb = fix[fix_of[b]];
      fb.blk = b;
      fb.level = m->hm.leaves[b].level;
      for (int f = 0; f < 6; ++f) {
        fb.slot_c[f] = -1;
        for (int o = 0; o < 4; ++o) fb.slot_f[f][o] = -1;
      }
    }
  for (const Record& r : m->hm.r1) {
    if (r.op != F4_OP_F2C) continue;
    DevFixBlock& fb = fix[fix_of[r.dst]];
    fb.slot_c[r.face] = bfslot[(size_t)r.dst * 6 + r.face];
    fb.slot_f[r.face][r.o1 + 2 * r.o2] = bfslot[(size_t)r.src * 6 + (r.face ^ 1)];   // the fine block's face towards us
  }
  for (size_t q = 0; q < n_fix; ++q)
    for (int f = 0; f < 2 * m->hm.dim; ++f)
      if (fix[q].slot_c[f] >= 0)
        for (int o = 0; o < (m->hm.dim == 3 ? 4 : 2); ++o)
          if (fix[q].slot_f[f][o] < 0) return fail(m, F4_EUNBALANCED, "flux fixing: a fine face has no coarse-to-fine record");
  m->n_bfslots = nslots;
  m->n_fix = (int)n_fix;
  {
    int rc;
    const size_t face_doubles = (size_t)m->nvar * m->hm.N * (m->hm.dim == 3 ? m->hm.N : 1);
    if ((rc = ensure(m, m->d_bflux, m->cap_bflux, (size_t)nslots * face_doubles))) return rc;
  }
  CU(cudaMemcpyAsync(m->d_meta, m->h_meta, total, cudaMemcpyHostToDevice, m->stream));
  CU(cudaEventRecord(m->meta_ev, m->stream));
  char* d = m->d_meta;
  m->d_level = (int*)(d + o_level);
  m->d_nbr = (int*)(d + o_nbr);
  m->nb_dev = nb;
  m->d_bfslot = (int*)(d + o_bfs);
  m->d_r1 = (DevRecord*)(d + o_a);
  m->d_r2 = (DevRecord*)(d + o_b2);
  m->d_r1n = (DevRecord*)(d + o_an);
  m->d_r1z = (DevRecord*)(d + o_az);
  m->d_r1c = (DevRecord*)(d + o_ac);
  m->d_r1f = (DevRecord*)(d + o_af);
  m->d_fix = (DevFixBlock*)(d + o_fix);
  m->n_r1 = (int)n_a; m->n_r2 = (int)n_b2; m->n_r1n = (int)n_an; m->n_r1z = (int)n_az; m->n_r1c = (int)n_ac;
  m->n_r1f = (int)n_af;
  std::fill(m->srl_valid.begin(), m->srl_valid.end(), 0);
  return F4_OK;
}

// have = srl_valid[state]: which same-level ghosts are already up to date (those records are skipped).
// need_z: the reader uses same-level y / z ghost cells (prolongation stencils, refinement criteria, regrid transfer,
// the caller of f4_fill_ghosts); a stage kernel does not (it fetches those rows / planes from the neighbours' interiors).
// for_stage: the reader is a stage kernel preceded by this fill's R2 round: of the same-level y / z ghosts only
// those of C2F source blocks have to be in memory.  no_push (flux-fixing mode): the stage that produced the state
// did not push its x layers either (they were corrected afterwards), so the x-face copies run here.
int fill_ghosts_impl(f4_mesh* m, int state, int have, bool need_z, bool for_stage = false, bool no_push = false) {
  double* st = m->state_ptr(state);
  const DevRecord* r1 = m->d_r1;
  int n1 = m->n_r1, after = 2;
  if (have == 2 || (have == 1 && !need_z)) { r1 = m->d_r1n; n1 = m->n_r1n; after = have; }
  else if (have == 1 && for_stage) { r1 = m->d_r1c; n1 = m->n_r1c; after = 1; }
  else if (have == 1) { r1 = m->d_r1z; n1 = m->n_r1z; }
  // nothing valid and the reader is a stage kernel: of the same-level copies it needs the x faces only (and the y / z
  // ones into C2F source blocks); its y / z halos come from the neighbours' interiors
  else if (for_stage) { r1 = m->d_r1f; n1 = m->n_r1f; after = no_push ? 0 : 1; }
  if (r1 == m->d_r1 && n1 > m->n_r1n) {
    // the whole pattern: the same-level copies go by SOURCE block (every interior row read once, f4_ghost.cu), the
    // executor runs the rest of round 1 (physical boundaries, restrictions); the two write disjoint ghost regions
    Scope sc(m, F4_PROF_R1);
    CU(launch_srl_push(m->hm.dim, m->hm.N, m->nvar, st, m->d_nbr, m->nb_dev, m->stream));
    r1 = m->d_r1n;
    n1 = m->n_r1n;
  }
  if (n1) {
    Scope sc(m, F4_PROF_R1);
    CU(launch_ghost(m->hm.dim, m->hm.N, m->nvar,
                    GhostParams{st, r1, n1, m->theta, m->d_bcv, m->d_bcdata, m->d_level, m->hm.dx_of_level(0)}, m->stream));
  }
  m->srl_valid[state] = (char)after;
  if (m->n_r2) {
    Scope sc(m, F4_PROF_R2);
    CU(launch_ghost(m->hm.dim, m->hm.N, m->nvar,
                    GhostParams{st, m->d_r2, m->n_r2, m->theta, m->d_bcv, m->d_bcdata, m->d_level, m->hm.dx_of_level(0)},
                    m->stream));
  }
  return F4_OK;
}

int check_state(f4_mesh* m, int state) {
  if (!m) return F4_EINVAL;
  if (!m->bound) return fail(m, F4_EUNBOUND, "no device storage bound (f4_bind_storage); there is no CPU fallback");
  if (state < 0 || state >= m->n_states) return fail(m, F4_EINVAL, "state index out of range");
  return F4_OK;
}

}  // namespace

extern "C" {

const char* f4_version(void) { return "f4 0.1 (sm_100a)"; }

int f4_mesh_create(int dim, int block_n, int n_ghost, const int brick[3], int base_level, int max_level,
                   const int bc_kind[6], double gamma, int n_states, int max_blocks, f4_mesh** out) {
  if (!out || !brick || !bc_kind) return F4_EINVAL;
  *out = nullptr;
  if (n_states < 2 || max_blocks < 1 || !(gamma > 1.0)) return F4_EINVAL;
  f4_mesh* m = new (std::nothrow) f4_mesh();
  if (!m) return F4_EINVAL;
  m->hm.dim = dim;
  m->hm.N = block_n;
  m->hm.Ng = n_ghost;
  for (int a = 0; a < 3; ++a) m->hm.brick[a] = (a < dim) ? brick[a] : 1;
  m->hm.base_level = base_level;
  m->hm.max_level = max_level;
  for (int f = 0; f < 6; ++f) m->hm.bc[f] = (f < 2 * dim) ? bc_kind[f] : F4_BC_PERIODIC;
  m->hm.max_blocks = max_blocks;
  m->gamma = gamma;
  m->n_states = n_states;
  std::string err;
  int rc = m->hm.init(err);
  if (rc != F4_OK) {
    delete m;
    return rc;
  }
  m->nvar = dim + 2;
  const size_t P = block_n + 2 * n_ghost;
  m->vs = P * P * (dim == 3 ? P : 1);
  m->bs = m->vs * m->nvar;
  m->state_doubles = m->bs * (size_t)max_blocks;
  m->phys.resize(n_states);
  m->srl_valid.assign(n_states, 0);
  for (int s = 0; s < n_states; ++s) m->phys[s] = s;
  *out = m;
  return F4_OK;
}

int f4_mesh_destroy(f4_mesh* m) {
  DeviceScope dev_scope(m);
  if (!m) return F4_EINVAL;
  if (m->pending) m->worker.join();
  if (m->bound) cudaStreamSynchronize(m->stream);
  for (auto& e : m->evs) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
  if (m->d_meta) cudaFree(m->d_meta);
  if (m->h_meta) cudaFreeHost(m->h_meta);
  if (m->meta_ev) cudaEventDestroy(m->meta_ev);
  if (m->d_bflux) cudaFree(m->d_bflux);
  if (m->d_plan) cudaFree(m->d_plan);
  if (m->d_maxrate) cudaFree(m->d_maxrate);
  if (m->d_dt) cudaFree(m->d_dt);
  if (m->d_sums) cudaFree(m->d_sums);
  if (m->d_flags) cudaFree(m->d_flags);
  if (m->d_bcv) cudaFree(m->d_bcv);
  if (m->d_bcdata) cudaFree(m->d_bcdata);
  if (m->d_indicator) cudaFree(m->d_indicator);
  if (m->d_stage) cudaFree(m->d_stage);
  delete m;
  return F4_OK;
}

int f4_set_options(f4_mesh* m, int limiter, int flux_scheme, double theta) {
  if (!m) return F4_EINVAL;
  if (limiter < 0 || limiter > F4_LIM_WENO3 || flux_scheme < 0 || flux_scheme > F4_FLUX_RUSANOV || !(theta >= 1.0))
    return fail(m, F4_EINVAL, "bad option");
  m->limiter = limiter;
  m->flux = flux_scheme;
  m->theta = theta;
  return F4_OK;
}

int f4_set_flux_fix(f4_mesh* m, int on) {
  if (!m) return F4_EINVAL;
  m->flux_fix = on != 0;
  return F4_OK;
}

int f4_set_physics(f4_mesh* m, int physics, const double velocity[3]) {
  if (!m) return F4_EINVAL;
  if (physics != F4_PHYS_EULER && physics != F4_PHYS_ADVECTION) return fail(m, F4_EINVAL, "unknown physics");
  if (m->bound) return fail(m, F4_EINVAL, "f4_set_physics must precede f4_bind_storage (it changes the storage size)");
  if (physics == F4_PHYS_ADVECTION) {
    if (!velocity) return fail(m, F4_EINVAL, "scalar advection needs a velocity");
    for (int a = 0; a < 3; ++a) {
      if (velocity[a] != velocity[a]) return fail(m, F4_EINVAL, "velocity is not a number");
      m->vel[a] = (a < m->hm.dim) ? velocity[a] : 0.0;
    }
  }
  m->physics = physics;
  m->nvar = (physics == F4_PHYS_ADVECTION) ? 1 : m->hm.dim + 2;
  m->bs = m->vs * m->nvar;
  m->state_doubles = m->bs * (size_t)m->hm.max_blocks;
  return F4_OK;
}

int f4_num_vars(const f4_mesh* m) { return m ? m->nvar : F4_EINVAL; }

size_t f4_storage_bytes(const f4_mesh* m) { return m ? m->state_doubles * (size_t)m->n_states * sizeof(double) : 0; }

int f4_bind_storage(f4_mesh* m, void* dev_ptr, size_t bytes, void* cuda_stream) {
  if (!m) return F4_EINVAL;
  if (!dev_ptr || bytes < f4_storage_bytes(m) || ((uintptr_t)dev_ptr & 255)) return fail(m, F4_EINVAL, "bad storage");
  if (m->hm.Ng != NG || !stage_supported(m->hm.dim, m->hm.N))
    return fail(m, F4_EUNSUPPORTED, "CUDA kernels exist for n_ghost=2 and (dim,N) in {(2,8),(2,16),(2,32),(3,8),(3,16),(3,32)}");
  int ndev = 0;
  CU(cudaGetDeviceCount(&ndev));
  if (ndev < 1) return fail(m, F4_ECUDA, "no CUDA device");
  {
    cudaPointerAttributes pa{};
    CU(cudaPointerGetAttributes(&pa, dev_ptr));
    if (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged)
      return fail(m, F4_EINVAL, "storage is not device memory");
    if (m->d_maxrate && m->device != pa.device)
      return fail(m, F4_EINVAL, "storage was bound on another device before");
    m->device = pa.device;
  }
  DeviceScope dev_scope(m);
  m->store = (double*)dev_ptr;
  m->stream = (cudaStream_t)cuda_stream;
  if (!m->d_maxrate) {
    CU(cudaMalloc((void**)&m->d_maxrate, sizeof(unsigned long long)));
    CU(cudaMalloc((void**)&m->d_dt, 2 * sizeof(double)));
    CU(cudaMalloc((void**)&m->d_sums, (size_t)m->hm.max_blocks * m->nvar * sizeof(double)));
    CU(cudaMalloc((void**)&m->d_flags, (size_t)m->hm.max_blocks * sizeof(int)));
    CU(cudaMalloc((void**)&m->d_bcv, sizeof(m->bcv)));
    CU(cudaMalloc((void**)&m->d_indicator, (size_t)m->hm.max_blocks * sizeof(double)));
    // staging: whole blocks of the natural padded layout, at most 128 MiB
    size_t per_block = m->bs * sizeof(double);
    size_t nblk = (128u << 20) / per_block;
    if (nblk < 1) nblk = 1;
    if (nblk > (size_t)m->hm.max_blocks) nblk = m->hm.max_blocks;
    m->stage_bytes = nblk * per_block;
    CU(cudaMalloc((void**)&m->d_stage, m->stage_bytes));
  }
  m->bound = true;
  CU(cudaMemcpyAsync(m->d_bcv, m->bcv, sizeof(m->bcv), cudaMemcpyHostToDevice, m->stream));
  for (int s = 0; s < m->n_states; ++s) {
    Scope sc(m, F4_PROF_LAYOUT);
    CU(launch_init_benign(m->hm.dim, m->hm.N, m->nvar, m->state_ptr(s), m->hm.max_blocks, m->gamma, m->stream));
  }
  m->rate_valid = false;
  return upload_meta(m);
}

int f4_num_blocks(const f4_mesh* m) { return m ? (int)m->hm.leaves.size() : F4_EINVAL; }

int f4_get_blocks(const f4_mesh* m, int* level, int* coords, double* origin, double* dx) {
  if (!m) return F4_EINVAL;
  const int nb = (int)m->hm.leaves.size();
  for (int b = 0; b < nb; ++b) {
    const Leaf& l = m->hm.leaves[b];
    const double h = m->hm.dx_of_level(l.level);
    if (level) level[b] = l.level;
    if (dx) dx[b] = h;
    for (int a = 0; a < 3; ++a) {
      if (coords) coords[3 * b + a] = l.c[a];
      if (origin) origin[3 * b + a] = (a < m->hm.dim) ? (double)l.c[a] * m->hm.N * h : 0.0;
    }
  }
  return F4_OK;
}

int f4_set_state(f4_mesh* m, int state, const double* src, int src_is_device, int with_ghosts) {
  DeviceScope dev_scope(m);
  int rc = check_state(m, state);
  if (rc) return rc;
  if (!src) return fail(m, F4_EINVAL, "null source");
  const int nb = (int)m->hm.leaves.size(), dim = m->hm.dim, N = m->hm.N;
  const size_t E = with_ghosts ? N + 2 * m->hm.Ng : N;
  const size_t per_block = (size_t)m->nvar * E * E * (dim == 3 ? E : 1);
  if (state == 0) m->rate_valid = false;
  m->srl_valid[state] = 0;
  if (src_is_device) {
    Scope sc(m, F4_PROF_LAYOUT);
    CU(launch_pack(dim, N, m->nvar, m->state_ptr(state), src, 0, nb, with_ghosts, m->stream));
    return F4_OK;
  }
  const int chunk = (int)(m->stage_bytes / (per_block * sizeof(double)));
  for (int b0 = 0; b0 < nb; b0 += chunk) {
    const int n = (nb - b0 < chunk) ? nb - b0 : chunk;
    CU(cudaMemcpyAsync(m->d_stage, src + (size_t)b0 * per_block, (size_t)n * per_block * sizeof(double),
                       cudaMemcpyHostToDevice, m->stream));
    Scope sc(m, F4_PROF_LAYOUT);
    CU(launch_pack(dim, N, m->nvar, m->state_ptr(state), m->d_stage, b0, n, with_ghosts, m->stream));
  }
  CU(cudaStreamSynchronize(m->stream));
  return F4_OK;
}

int f4_get_state(f4_mesh* m, int state, double* dst, int dst_is_device, int with_ghosts) {
  DeviceScope dev_scope(m);
  int rc = check_state(m, state);
  if (rc) return rc;
  if (!dst) return fail(m, F4_EINVAL, "null destination");
  const int nb = (int)m->hm.leaves.size(), dim = m->hm.dim, N = m->hm.N;
  const size_t E = with_ghosts ? N + 2 * m->hm.Ng : N;
  const size_t per_block = (size_t)m->nvar * E * E * (dim == 3 ? E : 1);
  if (dst_is_device) {
    Scope sc(m, F4_PROF_LAYOUT);
    CU(launch_unpack(dim, N, m->nvar, m->state_ptr(state), dst, 0, nb, with_ghosts, m->stream));
    return F4_OK;
  }
  const int chunk = (int)(m->stage_bytes / (per_block * sizeof(double)));
  for (int b0 = 0; b0 < nb; b0 += chunk) {
    const int n = (nb - b0 < chunk) ? nb - b0 : chunk;
    {
      Scope sc(m, F4_PROF_LAYOUT);
      CU(launch_unpack(dim, N, m->nvar, m->state_ptr(state), m->d_stage, b0, n, with_ghosts, m->stream));
    }
    CU(cudaMemcpyAsync(dst + (size_t)b0 * per_block, m->d_stage, (size_t)n * per_block * sizeof(double),
                       cudaMemcpyDeviceToHost, m->stream));
  }
  CU(cudaStreamSynchronize(m->stream));
  return F4_OK;
}

int f4_build_ghost_pattern(f4_mesh* m) {
  DeviceScope dev_scope(m);
  if (!m) return F4_EINVAL;
  std::string err;
  int rc = m->hm.build_pattern(err);
  if (rc) return fail(m, rc, err);
  return upload_meta(m);
}

int f4_pattern_size(const f4_mesh* m, int* n_r1, int* n_r2) {
  if (!m) return F4_EINVAL;
  if (n_r1) *n_r1 = (int)m->hm.r1.size();
  if (n_r2) *n_r2 = (int)m->hm.r2.size();
  return F4_OK;
}

int f4_get_pattern(const f4_mesh* m, int* records) {
  if (!m || !records) return F4_EINVAL;
  size_t q = 0;
  for (const std::vector<Record>* r : {&m->hm.r1, &m->hm.r2})
    for (const Record& x : *r) {
      int* o = records + 6 * q++;
      o[0] = x.op; o[1] = x.face; o[2] = x.dst; o[3] = x.src; o[4] = x.o1; o[5] = x.o2;
    }
  return F4_OK;
}

int f4_fill_ghosts(f4_mesh* m, int state) {
  DeviceScope dev_scope(m);
  int rc = check_state(m, state);
  if (rc) return rc;
  return fill_ghosts_impl(m, state, 0, true);
}

int f4_compute_dt(f4_mesh* m, int state, double cfl, double* dt_out) {
  DeviceScope dev_scope(m);
  int rc = check_state(m, state);
  if (rc) return rc;
  if (!dt_out || !(cfl > 0.0)) return fail(m, F4_EINVAL, "bad cfl / null output");
  if (m->physics == F4_PHYS_ADVECTION) {
    // the only wave speed is v: max over cells of sum_d |v_d| / dx is taken on the finest level present
    int lmax = 0;
    for (const Leaf& l : m->hm.leaves) lmax = l.level > lmax ? l.level : lmax;
    double sv = 0.0;
    for (int a = 0; a < m->hm.dim; ++a) sv += std::fabs(m->vel[a]);
    const double rate = sv / m->hm.dx_of_level(lmax);
    if (!(rate > 0.0)) return fail(m, F4_EINVAL, "compute_dt: the advection velocity is zero");
    *dt_out = cfl / rate;
    return F4_OK;
  }
  if (!(state == 0 && m->rate_valid)) {
    CU(cudaMemsetAsync(m->d_maxrate, 0, sizeof(unsigned long long), m->stream));
    Scope sc(m, F4_PROF_DT);
    CU(launch_maxrate(m->hm.dim, m->hm.N, m->state_ptr(state), m->d_level, (int)m->hm.leaves.size(), m->gamma,
                      1.0 / m->hm.dx_of_level(0), m->d_maxrate, m->stream));
  }
  double rate = 0.0;
  CU(cudaMemcpyAsync(&rate, m->d_maxrate, sizeof(double), cudaMemcpyDeviceToHost, m->stream));
  CU(cudaStreamSynchronize(m->stream));
  m->rate_valid = (state == 0);  // d_maxrate now describes this state
  if (!(rate > 0.0) || !(rate <= 1.7976931348623157e308))
    return fail(m, F4_EINVAL, "compute_dt: wave speed is zero or not finite (a cell with NaN, rho <= 0 or p <= 0?)");
  *dt_out = cfl / rate;
  return F4_OK;
}

namespace {

// One sub-step of eq. (5): u(out) = dtf*dt F(u(deriv)) + sum_i w[i] u(prev[i]); logical states.
struct SubStep {
  int out, deriv;
  double dtf;
  int np;
  double w[4];
  int prev[4];
};
struct Scheme {
  int n_sub, n_states, result;   // result: logical state that holds u(t+dt) after the last sub-step
  SubStep sub[4];
};

// The schemes foap4 includes ("optimal SSP schemes with two, three and four stages", eq. (6)-(11)).
// out != deriv always (the stage kernel pushes ghost layers of `out` into neighbour blocks that may still be
// reading `deriv`); out == prev[i] is allowed (a cell of prev is read only by the thread that writes it).
const Scheme& scheme_table(int rk) {
  static const Scheme tab[F4_RK_N] = {
      // Heun = SSPRK(2,2), eq. (6)-(7)
      {2, 2, 0, {{1, 0, 1.0, 1, {1.0}, {0}}, {0, 1, 0.5, 2, {0.5, 0.5}, {0, 1}}}},
      // forward Euler: one sub-step of eq. (5) with n_prev = 1
      {1, 2, 1, {{1, 0, 1.0, 1, {1.0}, {0}}}},
      // SSPRK(3,3) (Shu-Osher): u1 = ut + dt F(ut); u2 = 3/4 ut + 1/4 (u1 + dt F(u1)); u = 1/3 ut + 2/3 (u2 + dt F(u2))
      {3, 3, 0, {{1, 0, 1.0, 1, {1.0}, {0}},
                 {2, 1, 0.25, 2, {0.75, 0.25}, {0, 1}},
                 {0, 2, 2.0 / 3.0, 2, {1.0 / 3.0, 2.0 / 3.0}, {0, 2}}}},
      // SSPRK(4,3): u1 = ut + dt/2 F(ut); u2 = u1 + dt/2 F(u1); u3 = 2/3 ut + 1/3 (u2 + dt/2 F(u2)); u = u3 + dt/2 F(u3)
      {4, 3, 0, {{1, 0, 0.5, 1, {1.0}, {0}},
                 {2, 1, 0.5, 1, {1.0}, {1}},
                 {1, 2, 1.0 / 6.0, 2, {2.0 / 3.0, 1.0 / 3.0}, {0, 2}},
                 {0, 1, 0.5, 1, {1.0}, {1}}}},
      // classical RK4, eq. (8)-(11)
      {4, 4, 0, {{1, 0, 0.5, 1, {1.0}, {0}},
                 {2, 1, 0.5, 1, {1.0}, {0}},
                 {3, 2, 1.0, 1, {1.0}, {0}},
                 {0, 3, 1.0 / 6.0, 4, {-1.0 / 3.0, 1.0 / 3.0, 2.0 / 3.0, 1.0 / 3.0}, {0, 1, 2, 3}}}},
  };
  return tab[rk];
}

}  // namespace

int f4_set_bc_values(f4_mesh* m, const double* values) {
  DeviceScope dev_scope(m);
  if (!m || !values) return F4_EINVAL;
  for (int q = 0; q < 6 * m->nvar; ++q) m->bcv[q] = values[q];
  if (m->bound) {
    CU(cudaMemcpyAsync(m->d_bcv, m->bcv, sizeof(m->bcv), cudaMemcpyHostToDevice, m->stream));
    CU(cudaStreamSynchronize(m->stream));
    for (auto& v : m->srl_valid) v = 0;   // boundary ghosts of every state are stale now
  }
  return F4_OK;
}

int f4_set_bc_callback(f4_mesh* m, f4_bc_data_fn fn, void* user) {
  DeviceScope dev_scope(m);
  if (!m) return F4_EINVAL;
  m->bc_fn = fn;
  m->bc_user = user;
  return refresh_bc_data(m);
}

int f4_update_bc_data(f4_mesh* m) {
  DeviceScope dev_scope(m);
  return m ? refresh_bc_data(m) : F4_EINVAL;
}

int f4_num_bc_faces(const f4_mesh* m) { return m ? (int)m->bc_block.size() : F4_EINVAL; }

int f4_set_gravity(f4_mesh* m, const double g[3]) {
  if (!m || !g) return F4_EINVAL;
  for (int a = 0; a < 3; ++a) {
    if (g[a] != g[a]) return fail(m, F4_EINVAL, "gravity is not a number");
    m->grav[a] = (a < m->hm.dim) ? g[a] : 0.0;
  }
  return F4_OK;
}

int f4_set_rk_scheme(f4_mesh* m, int scheme) {
  if (!m) return F4_EINVAL;
  if (scheme < 0 || scheme >= F4_RK_N) return fail(m, F4_EINVAL, "unknown Runge-Kutta scheme");
  if (scheme_table(scheme).n_states > m->n_states)
    return fail(m, F4_EINVAL, "this scheme needs more temporal states than f4_mesh_create allocated (PAPER.md:318)");
  m->rk = scheme;
  return F4_OK;
}

namespace {
// one step of the chosen Runge-Kutta scheme; dev_dt: the time step is the device-resident m->d_dt[0] (f4_advance_cfl)
int advance_impl(f4_mesh* m, double dt, bool dev_dt);
}

int f4_advance(f4_mesh* m, double dt) {
  DeviceScope dev_scope(m);
  int rc = check_state(m, 0);
  if (rc) return rc;
  if (!(dt > 0.0)) return fail(m, F4_EINVAL, "dt must be positive");
  return advance_impl(m, dt, false);
}

int f4_advance_cfl(f4_mesh* m, double cfl) {
  DeviceScope dev_scope(m);
  int rc = check_state(m, 0);
  if (rc) return rc;
  if (!(cfl > 0.0)) return fail(m, F4_EINVAL, "cfl must be positive");
  if (m->physics == F4_PHYS_ADVECTION) {   // constant wave speed: dt is known on the host without a device pass
    double dt = 0.0;
    if ((rc = f4_compute_dt(m, 0, cfl, &dt))) return rc;
    m->dt_on_device = false;
    m->host_dt = dt;
    return advance_impl(m, dt, false);
  }
  if (!m->rate_valid) {   // no fused CFL maximum of state 0 at hand (first step, after set_state / adapt / flux fixing)
    CU(cudaMemsetAsync(m->d_maxrate, 0, sizeof(unsigned long long), m->stream));
    Scope sc(m, F4_PROF_DT);
    CU(launch_maxrate(m->hm.dim, m->hm.N, m->state_ptr(0), m->d_level, (int)m->hm.leaves.size(), m->gamma,
                      1.0 / m->hm.dx_of_level(0), m->d_maxrate, m->stream));
  }
  {
    Scope sc(m, F4_PROF_DT);
    CU(launch_dt_from_rate(m->d_maxrate, cfl, m->d_dt, m->stream));
  }
  m->dt_on_device = true;
  return advance_impl(m, 0.0, true);
}

int f4_last_dt(f4_mesh* m, double* dt_out) {
  DeviceScope dev_scope(m);
  if (!m || !dt_out) return F4_EINVAL;
  if (!m->dt_on_device) { *dt_out = m->host_dt; return F4_OK; }
  double h[2] = {0.0, 0.0};
  CU(cudaMemcpyAsync(h, m->d_dt, sizeof(h), cudaMemcpyDeviceToHost, m->stream));
  CU(cudaStreamSynchronize(m->stream));
  *dt_out = h[0];
  if (h[1] != 0.0) return fail(m, F4_EINVAL, "advance_cfl: wave speed is zero or not finite (a cell with NaN, rho <= 0 or p <= 0?)");
  return F4_OK;
}

namespace {
int advance_impl(f4_mesh* m, double dt, bool dev_dt) {
  int rc;
  const int dim = m->hm.dim, N = m->hm.N, nb = (int)m->hm.leaves.size();
  const Scheme& sch = scheme_table(m->rk);
  StageParams p{};
  p.gamma = m->gamma;
  const double inv_dx0 = 1.0 / m->hm.dx_of_level(0);
  p.level = m->d_level;
  p.nblocks = nb;
  p.limiter = m->limiter;
  p.flux = m->flux;
  const bool adv = m->physics == F4_PHYS_ADVECTION;
  for (int a = 0; a < 3; ++a) p.vel[a] = m->vel[a];
  for (int a = 0; a < 3; ++a) p.grav[a] = m->grav[a];
  p.has_grav = (m->grav[0] != 0.0 || m->grav[1] != 0.0 || m->grav[2] != 0.0) ? 1 : 0;
  // flux fixing acts only where the mesh has refinement boundaries.  The corrected cells must be
  // what the neighbours see: the stage kernel then does not push its x layers (the executor copies them after the
  // correction; y / z ghosts are gathered by the next stage from interiors that are corrected by then) and the CFL
  // maximum is left to the standalone reduction (the stage kernel would take it before the correction).
  const bool ff = m->flux_fix && m->n_fix > 0;
  FixParams fp{};
  fp.fix = m->d_fix;
  fp.nfix = m->n_fix;
  fp.bflux = m->d_bflux;
  p.bfslot = ff ? m->d_bfslot : nullptr;
  p.bflux = m->d_bflux;
  p.nbr = m->d_nbr;        // y / z ghosts are always gathered from the (already corrected) neighbour interiors
  p.push_x = ff ? 0 : 1;
  for (int q = 0; q < sch.n_sub; ++q) {
    const SubStep& ss = sch.sub[q];
    const bool last = (q == sch.n_sub - 1);
    // ghost fill precedes each F evaluation; same-level ghosts of a state a stage produced were pushed
    // (C2F prolongation stencils read the coarse blocks' same-level y / z ghosts: with such records those are filled too)
    if ((rc = fill_ghosts_impl(m, ss.deriv, m->srl_valid[ss.deriv], m->n_r2 > 0, true, ff))) return rc;
    p.deriv = m->state_ptr(ss.deriv);
    p.out = m->state_ptr(ss.out);
    const double* pv[4] = {nullptr, nullptr, nullptr, nullptr};
    double w[4] = {0.0, 0.0, 0.0, 0.0};
    for (int r = 0; r < ss.np; ++r) { pv[r] = m->state_ptr(ss.prev[r]); w[r] = ss.w[r]; }
    p.prev0 = pv[0]; p.prev1 = pv[1]; p.prev2 = pv[2]; p.prev3 = pv[3];
    p.w0 = w[0]; p.w1 = w[1]; p.w2 = w[2]; p.w3 = w[3];
    p.grav_from = (ss.prev[0] == ss.deriv) ? 0 : ((ss.np > 1 && ss.prev[1] == ss.deriv) ? 1 : 2);
    p.dt_sub = ss.dtf * dt;
    p.dt_dev = dev_dt ? m->d_dt : nullptr;
    p.dtf = ss.dtf;
    for (int l = 0; l < MAXL; ++l) {
      p.inv_dx_l[l] = inv_dx0 * (double)(1u << l);
      p.sdt_l[l] = p.dt_sub * p.inv_dx_l[l];
    }
    // CFL max of the new state fused into the last sub-step ("a limit for the next time step")
    p.maxrate = (last && !ff && !adv) ? m->d_maxrate : nullptr;
    if (p.maxrate) CU(cudaMemsetAsync(m->d_maxrate, 0, sizeof(unsigned long long), m->stream));
    {
      Scope sc(m, F4_PROF_STAGE);
      if (adv) {
        if (!advect_supported(p))
          return fail(m, F4_EUNSUPPORTED, "scalar advection: van Leer / minmod / MC limiters and at most two previous states");
        CU(launch_advect(dim, N, p, m->stream));
      } else {
        CU(launch_stage(dim, N, p, m->stream));
      }
    }
    if (ff) {
      fp.out = p.out;
      for (int l = 0; l < MAXL; ++l) { fp.sdt_l[l] = p.sdt_l[l]; fp.inv_dx_l[l] = p.inv_dx_l[l]; }
      fp.dt_dev = p.dt_dev;
      fp.dtf = p.dtf;
      Scope sc(m, F4_PROF_STAGE);
      CU(launch_fluxfix(dim, N, m->nvar, fp, m->stream));
    }
    // x same-level ghosts of `out` were pushed by the stage (its y ghost rows / z ghost planes were not written);
    // BC / F2C / C2F ghosts of `out` are stale until the next fill
    m->srl_valid[ss.out] = ff ? 0 : 1;
  }
  if (sch.result != 0) std::swap(m->phys[0], m->phys[sch.result]), std::swap(m->srl_valid[0], m->srl_valid[sch.result]);
  m->rate_valid = !ff && !adv;
  return F4_OK;
}
}  // namespace

int f4_refine_flags(f4_mesh* m, int state, int criterion, int var, const double params[4], int* flags_out,
                    double* indicator_out) {
  DeviceScope dev_scope(m);
  int rc = check_state(m, state);
  if (rc) return rc;
  if (!params || !flags_out) return fail(m, F4_EINVAL, "null params / flags");
  if (criterion != F4_CRIT_LOHNER && criterion != F4_CRIT_PJUMP) return fail(m, F4_EINVAL, "unknown criterion");
  if (criterion == F4_CRIT_LOHNER && (var < 0 || var >= m->nvar)) return fail(m, F4_EINVAL, "variable out of range");
  if (criterion == F4_CRIT_PJUMP && m->physics != F4_PHYS_EULER) return fail(m, F4_EINVAL, "the pressure-jump rule needs Euler");
  const int nb = (int)m->hm.leaves.size();
  if ((rc = fill_ghosts_impl(m, state, m->srl_valid[state], true))) return rc;
  {
    Scope sc(m, F4_PROF_REGRID);
    CU(launch_flags(m->hm.dim, m->hm.N, m->nvar, m->state_ptr(state), nb, criterion, var, m->gamma, params, m->d_flags,
                    m->d_indicator, m->stream));
  }
  CU(cudaMemcpyAsync(flags_out, m->d_flags, (size_t)nb * sizeof(int), cudaMemcpyDeviceToHost, m->stream));
  if (indicator_out)
    CU(cudaMemcpyAsync(indicator_out, m->d_indicator, (size_t)nb * sizeof(double), cudaMemcpyDeviceToHost, m->stream));
  CU(cudaStreamSynchronize(m->stream));
  return F4_OK;
}

namespace {

// device side of a regrid whose host part (m->hm already is the new mesh) produced `plan`: ghost fill of state 0
// with the records of the OLD mesh (still the ones on the device; prolongation reads the parents' face ghosts),
// transfer into the other slab, record upload
int commit_adapt(f4_mesh* m, const std::vector<Transfer>& plan) {
  int rc;
  const auto t1 = std::chrono::steady_clock::now();
  if ((rc = fill_ghosts_impl(m, 0, m->srl_valid[0], true))) return rc;
  std::vector<DevTransfer> dp(plan.size());
  for (size_t q = 0; q < plan.size(); ++q) {
    dp[q].kind = plan[q].kind;
    dp[q].dst = plan[q].dst;
    dp[q].oct = plan[q].oct;
    dp[q].pad = 0;
    for (int c = 0; c < 8; ++c) dp[q].src[c] = plan[q].src[c];
  }
  if ((rc = ensure(m, m->d_plan, m->cap_plan, dp.size()))) return rc;
  CU(cudaMemcpyAsync(m->d_plan, dp.data(), dp.size() * sizeof(DevTransfer), cudaMemcpyHostToDevice, m->stream));
  {
    Scope sc(m, F4_PROF_REGRID);
    CU(launch_transfer(m->hm.dim, m->hm.N, m->nvar, m->state_ptr(0), m->state_ptr(1), m->d_plan, (int)dp.size(), m->theta,
                       m->stream));
  }
  CU(cudaStreamSynchronize(m->stream));
  const auto t2 = std::chrono::steady_clock::now();
  m->adapt_ms[1] = std::chrono::duration<double, std::milli>(t2 - t1).count();
  std::swap(m->phys[0], m->phys[1]);  // the new numbering lives in the slab that was state 1
  std::fill(m->srl_valid.begin(), m->srl_valid.end(), 0);
  m->rate_valid = false;
  rc = upload_meta(m);
  m->adapt_ms[2] = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t2).count();
  return rc;
}

}  // namespace

int f4_adapt(f4_mesh* m, const int* refine_flags, int* changed_out) {
  DeviceScope dev_scope(m);
  if (!m || !refine_flags || !changed_out) return F4_EINVAL;
  *changed_out = 0;
  if (m->pending) return fail(m, F4_EINVAL, "f4_adapt: an asynchronous regrid is pending (f4_adapt_end)");
  std::vector<Transfer> plan;
  bool changed = false;
  std::string err;
  const auto t0 = std::chrono::steady_clock::now();
  int rc = m->hm.adapt(refine_flags, plan, changed, err);
  m->adapt_ms[0] = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
  m->adapt_ms[1] = m->adapt_ms[2] = 0.0;
  if (rc) return fail(m, rc, err);
  if (!changed) return F4_OK;
  *changed_out = 1;
  if (!m->bound) return refresh_bc_data(m);
  return commit_adapt(m, plan);
}

int f4_adapt_begin(f4_mesh* m, const int* refine_flags) {
  if (!m || !refine_flags) return F4_EINVAL;
  if (m->pending) return fail(m, F4_EINVAL, "f4_adapt_begin: a regrid is already pending");
  m->flags_next.assign(refine_flags, refine_flags + m->hm.leaves.size());
  m->hm_next = m->hm;   // the worker edits a copy: the mesh in use stays valid for compute_dt / advance
  m->plan_next.clear();
  m->changed_next = false;
  m->rc_next = F4_OK;
  m->err_next.clear();
  m->pending = true;
  m->worker = std::thread([m]() {
    const auto t0 = std::chrono::steady_clock::now();
    m->rc_next = m->hm_next.adapt(m->flags_next.data(), m->plan_next, m->changed_next, m->err_next);
    m->adapt_ms[0] = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
  });
  return F4_OK;
}

int f4_adapt_end(f4_mesh* m, int* changed_out) {
  DeviceScope dev_scope(m);
  if (!m || !changed_out) return F4_EINVAL;
  *changed_out = 0;
  if (!m->pending) return fail(m, F4_EINVAL, "f4_adapt_end: no regrid pending");
  m->worker.join();
  m->pending = false;
  m->adapt_ms[1] = m->adapt_ms[2] = 0.0;
  if (m->rc_next) return fail(m, m->rc_next, m->err_next);
  if (!m->changed_next) return F4_OK;
  *changed_out = 1;
  m->hm = std::move(m->hm_next);
  if (!m->bound) return refresh_bc_data(m);
  return commit_adapt(m, m->plan_next);
}

int f4_last_adapt_ms(const f4_mesh* m, double ms[3]) {
  if (!m || !ms) return F4_EINVAL;
  for (int q = 0; q < 3; ++q) ms[q] = m->adapt_ms[q];
  return F4_OK;
}

int f4_conserved_totals(f4_mesh* m, int state, double* totals) {
  DeviceScope dev_scope(m);
  int rc = check_state(m, state);
  if (rc) return rc;
  if (!totals) return fail(m, F4_EINVAL, "null output");
  const int nb = (int)m->hm.leaves.size();
  {
    Scope sc(m, F4_PROF_LAYOUT);
    CU(launch_block_sums(m->hm.dim, m->hm.N, m->nvar, m->state_ptr(state), nb, m->d_sums, m->stream));
  }
  std::vector<double> sums((size_t)nb * m->nvar);
  CU(cudaMemcpyAsync(sums.data(), m->d_sums, sums.size() * sizeof(double), cudaMemcpyDeviceToHost, m->stream));
  CU(cudaStreamSynchronize(m->stream));
  for (int v = 0; v < m->nvar; ++v) {
    long double acc = 0.0L;
    for (int b = 0; b < nb; ++b) {
      long double h = m->hm.dx_of_level(m->hm.leaves[b].level);
      acc += (long double)sums[(size_t)b * m->nvar + v] * (h * h * (m->hm.dim == 3 ? h : 1.0L));
    }
    totals[v] = (double)acc;
  }
  return F4_OK;
}

int f4_conserved_totals_noalloc(f4_mesh* m, int state, double* totals_dev) {
  DeviceScope dev_scope(m);
  int rc = check_state(m, state);
  if (rc) return rc;
  if (!totals_dev) return fail(m, F4_EINVAL, "f4_conserved_totals_noalloc: null output");
  cudaPointerAttributes attr;
  if (cudaPointerGetAttributes(&attr, totals_dev) != cudaSuccess ||
      (attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged)) {
    cudaGetLastError();
    return fail(m, F4_EINVAL, "f4_conserved_totals_noalloc: totals_dev must be a device pointer");
  }
  const int nb = (int)m->hm.leaves.size();
  if (nb > F4_NOALLOC_MAX_BLOCKS) {
    char msg[160];
    snprintf(msg, sizeof msg, "f4_conserved_totals_noalloc: %d blocks exceed the static scratch's maximum of %d "
             "(F4_NOALLOC_MAX_BLOCKS); use f4_conserved_totals", nb, F4_NOALLOC_MAX_BLOCKS);
    return fail(m, F4_EINVAL, msg);
  }
  m->launches++;   // two kernels: the Scope counts the first
  Scope sc(m, F4_PROF_LAYOUT);
  CU(launch_totals_noalloc(m->hm.dim, m->hm.N, m->nvar, m->state_ptr(state), m->d_level, nb, m->hm.dx_of_level(0),
                           totals_dev, m->stream));
  return F4_OK;
}

int f4_profile_enable(f4_mesh* m, int on) {
  DeviceScope dev_scope(m);
  if (!m) return F4_EINVAL;
  if (on && m->evs.empty()) {
    m->evs.resize(f4_mesh::EV_POOL);
    for (auto& e : m->evs) {
      CU(cudaEventCreate(&e.a));
      CU(cudaEventCreate(&e.b));
    }
  }
  m->prof = on != 0;
  return F4_OK;
}

int f4_profile_get(f4_mesh* m, double ms[F4_PROF_N], long long launches[F4_PROF_N], int reset) {
  DeviceScope dev_scope(m);
  if (!m) return F4_EINVAL;
  if (m->bound) CU(cudaStreamSynchronize(m->stream));
  m->fold_events();
  for (int c = 0; c < F4_PROF_N; ++c) {
    if (ms) ms[c] = m->prof_ms[c];
    if (launches) launches[c] = m->prof_n[c];
    if (reset) { m->prof_ms[c] = 0.0; m->prof_n[c] = 0; }
  }
  return F4_OK;
}

long long f4_launch_count(const f4_mesh* m) { return m ? m->launches : 0; }

const char* f4_last_error(const f4_mesh* m) { return m ? m->err.c_str() : "null mesh"; }

}  // extern "C"
