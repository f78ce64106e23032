// =============================================================================
// ORACLE -- TEST INFRASTRUCTURE ONLY.
//
// Plain, slow, single-threaded CPU statement of the hot path of foap4
// (arxiv/paper_2605_07612; citations are /root/reference/PAPER.md:<line>):
// one explicit Heun step of Euler's equations over every block of a
// quadtree/octree AMR mesh = ghost-cell fill (SRL copy, physical BC, F2C
// restriction, C2F prolongation in two rounds) + per-block finite-volume
// update (primitive reconstruction, HLL flux with Einfeldt speeds,
// conservative update, Runge-Kutta combine, CFL reduction) + mesh adapt with
// regrid data transfer; also flux fixing at refinement boundaries,
// the refinement criteria (eq. (12); config 5's pressure jump), the
// other Runge-Kutta schemes of eq. (5), the gravity source term
// eq. (20) and uniform Dirichlet / Neumann boundaries.
// Second physics: scalar advection eq. (13) with a uniform velocity field, one variable per cell,
// wave speeds min(v,0) / max(v,0); pinned (tests/test_oracle_advection.py) by upwind hand values, the dt closed form,
// the paper's Gaussian convergence test (L1 order ~ 2) and its flux-fixing conservation test in the
// original scalar form.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may build, load or call this file.  It shares no code
// with paper_2605_07612_b200/csrc (the CUDA product path) and imports nothing
// from it.  It follows the paper step by step, in the paper's 1-based index
// notation uu(i,j,k,ivar,iblock), i in [1-Ng, N+Ng]; there
// is no blocking, fusion or reordering.  Where the paper is silent the
// readings A1..A19 of DESIGN.md ("Readings of the paper") are taken and named
// at the place they are used.
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): uniform state bit-exact (P1),
// conservation (P2), Sod vs exact Riemann solution (P3), 2nd-order density
// wave (P4), linear-field ghost/prolong/restrict exactness PAPER.md:433-447
// (P5), restriction = block average (P6), Appendix-A closed form eq. (24)
// (P7), block permutation (P8), RK closed form (P9), 1D-in-3D (P10), mirror
// symmetry (P11), brute-force mesh validity; flux fixing by the paper's conservation
// test; eq. (12) by hand-worked values (tests/golden/lohner_eq12.txt);
// RK schemes by their stability polynomials and temporal order; gravity by the free-fall
// closed form and hydrostatic convergence; Dirichlet / Neumann ghosts by exact
// continuation of linear profiles.
// PARITY UNPINNED: the *choice* among readings A1 (van Leer harmonic form),
// A2 (HLL), A3 (Einfeldt speeds = Roe-average u^ +- d^), A5 (CFL sum over
// dimensions), A10 / A10b (outflow = zero-order extrapolation; Dirichlet mirror,
// Neumann first-order extrapolation) and the SSPRK(3,3) / SSPRK(4,3) tableaux (taken
// from the literature the paper cites, [20]) cannot be pinned against foap4 itself:
// the paper prints no formula or worked value for them.
// =============================================================================
#include <algorithm>
#include <array>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <map>
#include <set>
#include <string>
#include <thread>
#include <vector>

namespace {

enum { BC_PERIODIC = 0, BC_OUTFLOW = 1, BC_KEEP = 2, BC_DIRICHLET = 3, BC_NEUMANN = 4, BC_DATA = 5 };
enum { LIM_VANLEER = 0, LIM_MINMOD = 1, LIM_MC = 2, LIM_KOREN = 3, LIM_WENO3 = 4 };
enum { FLUX_HLL = 0, FLUX_RUSANOV = 1 };
enum { NB_BOUNDARY = 0, NB_SAME = 1, NB_COARSE = 2, NB_FINE = 3 };
enum { PHYS_EULER = 0, PHYS_ADVECTION = 1 };

struct Key {
  int level;
  std::array<int, 3> c;
  bool operator<(const Key& o) const {
    if (level != o.level) return level < o.level;
    return c < o.c;
  }
  bool operator==(const Key& o) const { return level == o.level && c == o.c; }
};

struct Neighbor {
  int kind;
  int blk[4];  // NB_SAME/NB_COARSE: blk[0]; NB_FINE: 2^(d-1) fine blocks indexed o_t1 + 2*o_t2
  int off[2];  // NB_COARSE: hanging-face offset of *this* fine block
};

struct Mesh {
  int dim, N, Ng, P, Pz, nvar;
  int brick[3], base_level, max_level, bc[6];
  double gamma, theta;
  double bcv[6][5] = {};  // uniform boundary value u_b (Dirichlet) or normal derivative u_b' (Neumann) per face direction and variable
  // spatially varying boundary values bc_data(i, j, ivar, ibf), eq. (4); here keyed by (block, face),
  // layout [var][t2][t1] over the cells of the block face
  std::map<std::pair<int, int>, std::vector<double>> bcdata;
  double grav[3] = {0.0, 0.0, 0.0};  // gravitational acceleration g of the source term eq. (20)
  // physics: 0 = Euler gas dynamics (nvar = dim + 2), 1 = scalar advection eq. (13) with the uniform
  // velocity field vel (nvar = 1: the scalar sits in Prim::rho)
  int physics = 0;
  double vel[3] = {0.0, 0.0, 0.0};
  int limiter, flux_scheme;
  int nstates;
  bool test_rhs = false;  // P9 pin: F(u) = lambda*u
  double test_lambda = 0.0;
  bool flux_fix = false;  // PAPER.md:253-261 section 2.7: conservative correction at refinement boundaries
  std::map<std::pair<int, int>, std::vector<double>> bflux;  // (block, face) -> fluxes [var][t2][t1] at that face
  std::vector<Key> blocks;
  std::map<Key, int> index;
  std::vector<std::vector<double>> uu;  // [state][block][var][k][j][i] padded, i fastest (eq. 3)
  std::string err;

  size_t block_stride() const { return (size_t)nvar * Pz * P * P; }
  size_t var_stride() const { return (size_t)Pz * P * P; }
  // paper's 1-based cell index -> storage offset inside one (block,var)
  size_t off(int i, int j, int k) const {
    int pi = i + Ng - 1, pj = j + Ng - 1, pk = (dim == 3) ? k + Ng - 1 : 0;
    return ((size_t)pk * P + pj) * P + pi;
  }
  double& at(int s, int b, int v, int i, int j, int k) {
    return uu[s][(size_t)b * block_stride() + (size_t)v * var_stride() + off(i, j, k)];
  }
  double dx_of_level(int l) const {
    int mb = std::max(brick[0], std::max(brick[1], dim == 3 ? brick[2] : 1));
    return 1.0 / ((double)mb * std::ldexp(1.0, l) * N);  // PAPER.md:31 factor 2^-l; reading A13
  }
  int extent(int l, int a) const { return brick[a] << l; }
};

// index triple from (normal, t1, t2) for a face on axis a
inline void compose(int a, int n, int t1, int t2, int& i, int& j, int& k) {
  if (a == 0) { i = n; j = t1; k = t2; }
  else if (a == 1) { j = n; i = t1; k = t2; }
  else { k = n; i = t1; j = t2; }
}
inline void transverse_axes(int a, int& ta, int& tb) {
  if (a == 0) { ta = 1; tb = 2; } else if (a == 1) { ta = 0; tb = 2; } else { ta = 0; tb = 1; }
}

// ----------------------------------------------------------------------------
// Limiters
// ----------------------------------------------------------------------------
// Generalised minmod, eq. (1): 0 if signs differ, else
// sign(a) min(|theta a|, |theta b|, |a+b|/2).
double minmod_G(double a, double b, double theta) {
  if (a * b <= 0.0) return 0.0;
  double m = std::min(std::fabs(theta * a), std::min(std::fabs(theta * b), std::fabs(a + b) / 2.0));
  return (a > 0.0) ? m : -m;
}
// van Leer limited (undivided) slope, reading A1: harmonic mean 2ab/(a+b) if ab>0 else 0
// (limiter named PAPER.md:325, 461; the paper prints no formula).
double vanleer(double a, double b) {
  if (a * b > 0.0) return 2.0 * a * b / (a + b);
  return 0.0;
}
// Koren's limiter (reading A1b): the kappa = 1/3 (third-order) slope (a + 2b)/3 towards the face on the
// b side, limited to [0, 2a] and [0, 2b]: phi(r) = max(0, min(2r, (2 + r)/3, 2)), r = a/b.  Not symmetric in (a, b).
double koren(double a, double b) {
  if (a * b <= 0.0) return 0.0;
  double m = std::min(std::min(2.0 * std::fabs(a), (std::fabs(a) + 2.0 * std::fabs(b)) / 3.0), 2.0 * std::fabs(b));
  return (a > 0.0) ? m : -m;
}
// Third-order WENO (reading A1b: the classical Jiang-Shu weights, eps = 1e-6): two linear candidates
// w + a/2 (from the far side) and w + b/2 (from the face side), ideal weights 1/3 and 2/3, smoothness a^2 and b^2.
// Returned as the equivalent slope s with w_face = w + s/2.
double weno3(double a, double b) {
  const double eps = 1e-6;
  double a0 = (1.0 / 3.0) / ((eps + a * a) * (eps + a * a));
  double a1 = (2.0 / 3.0) / ((eps + b * b) * (eps + b * b));
  return (a0 * a + a1 * b) / (a0 + a1);
}
// slope of a cell towards the face on the side of difference b (a = the difference on the other side): the left state
// of the cell's high face is w + s(a,b)/2 with a = w_i - w_{i-1}, b = w_{i+1} - w_i; the right state of its low face
// is w - s(b,a)/2.  van Leer, minmod and MC are symmetric in (a, b).
double limited_slope(const Mesh& m, double a, double b) {
  switch (m.limiter) {
    case LIM_VANLEER: return vanleer(a, b);
    case LIM_MINMOD: return minmod_G(a, b, 1.0);
    case LIM_MC: return minmod_G(a, b, 2.0);      // MC
    case LIM_KOREN: return koren(a, b);
    default: return weno3(a, b);
  }
}

// ----------------------------------------------------------------------------
// Mesh topology
// ----------------------------------------------------------------------------
void rebuild_index(Mesh& m) {
  m.index.clear();
  for (size_t b = 0; b < m.blocks.size(); ++b) m.index[m.blocks[b]] = (int)b;
}

// neighbour coordinates on the same level across face f; false if physical boundary
bool face_coords(const Mesh& m, const Key& kq, int f, std::array<int, 3>& n) {
  int a = f / 2, side = f % 2;
  n = kq.c;
  n[a] += side ? 1 : -1;
  int ext = m.extent(kq.level, a);
  if (n[a] < 0 || n[a] >= ext) {
    if (m.bc[f] != BC_PERIODIC) return false;
    n[a] = (n[a] + ext) % ext;
  }
  return true;
}

Neighbor find_neighbor(const Mesh& m, int b, int f) {
  Neighbor nb{};
  const Key& kq = m.blocks[b];
  int a = f / 2, side = f % 2;
  std::array<int, 3> n;
  if (!face_coords(m, kq, f, n)) { nb.kind = NB_BOUNDARY; return nb; }
  auto it = m.index.find(Key{kq.level, n});
  if (it != m.index.end()) { nb.kind = NB_SAME; nb.blk[0] = it->second; return nb; }
  if (kq.level > 0) {
    Key kc{kq.level - 1, {n[0] >> 1, n[1] >> 1, n[2] >> 1}};
    it = m.index.find(kc);
    if (it != m.index.end()) {
      int ta, tb; transverse_axes(a, ta, tb);
      nb.kind = NB_COARSE; nb.blk[0] = it->second;
      nb.off[0] = kq.c[ta] & 1;                       // relative position within the group
      nb.off[1] = (m.dim == 3) ? (kq.c[tb] & 1) : 0;
      return nb;
    }
  }
  // finer neighbours: children of (level, n) touching the shared face
  int ta, tb; transverse_axes(a, ta, tb);
  int n2 = (m.dim == 3) ? 2 : 1;
  nb.kind = NB_FINE;
  for (int o2 = 0; o2 < n2; ++o2)
    for (int o1 = 0; o1 < 2; ++o1) {
      std::array<int, 3> cc = {2 * n[0], 2 * n[1], 2 * n[2]};
      if (m.dim == 2) cc[2] = 0;
      cc[a] += side ? 0 : 1;  // neighbour on my + side: its low children touch me
      cc[ta] += o1;
      if (m.dim == 3) cc[tb] += o2;
      auto jt = m.index.find(Key{kq.level + 1, cc});
      nb.blk[o1 + 2 * o2] = (jt == m.index.end()) ? -1 : jt->second;
    }
  return nb;
}

// ----------------------------------------------------------------------------
// Ghost cells, PAPER.md:191-220 (two rounds R1 {SRL, BC, F2C} then R2 {C2F})
// ----------------------------------------------------------------------------
void fill_srl(Mesh& m, int s, int A, int f, int B) {
  // uu(bx+i,j,.,iq) = uu(i,j,.,jq); uu(-n_gc+i,j,.,jq) = uu(bx-n_gc+i,j,.,iq)
  int a = f / 2, side = f % 2, N = m.N, kmax = (m.dim == 3) ? N : 1;
  for (int v = 0; v < m.nvar; ++v)
    for (int g = 1; g <= m.Ng; ++g)
      for (int t2 = 1; t2 <= kmax; ++t2)
        for (int t1 = 1; t1 <= N; ++t1) {
          int di, dj, dk, si, sj, sk;
          if (side) { compose(a, N + g, t1, t2, di, dj, dk); compose(a, g, t1, t2, si, sj, sk); }
          else      { compose(a, 1 - g, t1, t2, di, dj, dk); compose(a, N + 1 - g, t1, t2, si, sj, sk); }
          m.at(s, A, v, di, dj, dk) = m.at(s, B, v, si, sj, sk);
        }
}

void fill_bc(Mesh& m, int s, int A, int f) {
  if (m.bc[f] == BC_KEEP) return;  // ghost values preset by the caller (linear-field test)
  // Outflow = uniform Neumann with zero normal derivative; reading A10:
  // every ghost layer = nearest interior layer.  Uniform Dirichlet / Neumann values: m.bcv.
  int a = f / 2, side = f % 2, N = m.N, kmax = (m.dim == 3) ? N : 1;
  for (int v = 0; v < m.nvar; ++v)
    for (int g = 1; g <= m.Ng; ++g)
      for (int t2 = 1; t2 <= kmax; ++t2)
        for (int t1 = 1; t1 <= N; ++t1) {
          int di, dj, dk, si, sj, sk;
          if (side) { compose(a, N + g, t1, t2, di, dj, dk); compose(a, N, t1, t2, si, sj, sk); }
          else      { compose(a, 1 - g, t1, t2, di, dj, dk); compose(a, 1, t1, t2, si, sj, sk); }
          if (m.bc[f] == BC_OUTFLOW) {
            m.at(s, A, v, di, dj, dk) = m.at(s, A, v, si, sj, sk);
          } else if (m.bc[f] == BC_NEUMANN) {
            // uniform normal derivative u_b' along the outward normal: the centre of ghost layer g is
            // g dx outside the centre of the first interior cell -> first-order extrapolation with that derivative
            // (reading A10b; u_b' = 0 is the outflow rule)
            const double dx = m.dx_of_level(m.blocks[A].level);
            m.at(s, A, v, di, dj, dk) = m.at(s, A, v, si, sj, sk) + ((double)g * dx) * m.bcv[f][v];
          } else if (m.bc[f] == BC_DATA) {
            // spatially varying Dirichlet data, eq. (4): the same mirror rule with the value of this face cell
            auto it = m.bcdata.find({A, f});
            double ub = (it == m.bcdata.end()) ? 0.0 : it->second[((size_t)v * kmax + (t2 - 1)) * N + (t1 - 1)];
            int mi, mj, mk;
            if (side) compose(a, N + 1 - g, t1, t2, mi, mj, mk); else compose(a, g, t1, t2, mi, mj, mk);
            m.at(s, A, v, di, dj, dk) = 2.0 * ub - m.at(s, A, v, mi, mj, mk);
          } else {  // BC_DIRICHLET
            // uniform value u_b on the boundary face: ghost layer g mirrors interior layer g through
            // the face, u_ghost = 2 u_b - u_interior, so that the linear interpolant takes u_b on the face (reading A10)
            int mi, mj, mk;
            if (side) compose(a, N + 1 - g, t1, t2, mi, mj, mk); else compose(a, g, t1, t2, mi, mj, mk);
            m.at(s, A, v, di, dj, dk) = 2.0 * m.bcv[f][v] - m.at(s, A, v, mi, mj, mk);
          }
        }
}

// mean of the 2^d fine cells whose lowest-index member is (i0,j0,k0) in block F.
// Reading A8: pairwise x -> y -> z, adds only, exact scaling by 2^-d.
double restrict_mean(Mesh& m, int s, int F, int v, int i0, int j0, int k0) {
  if (m.dim == 2) {
    double a0 = m.at(s, F, v, i0, j0, 1) + m.at(s, F, v, i0 + 1, j0, 1);
    double a1 = m.at(s, F, v, i0, j0 + 1, 1) + m.at(s, F, v, i0 + 1, j0 + 1, 1);
    return (a0 + a1) * 0.25;
  }
  double a00 = m.at(s, F, v, i0, j0, k0) + m.at(s, F, v, i0 + 1, j0, k0);
  double a10 = m.at(s, F, v, i0, j0 + 1, k0) + m.at(s, F, v, i0 + 1, j0 + 1, k0);
  double a01 = m.at(s, F, v, i0, j0, k0 + 1) + m.at(s, F, v, i0 + 1, j0, k0 + 1);
  double a11 = m.at(s, F, v, i0, j0 + 1, k0 + 1) + m.at(s, F, v, i0 + 1, j0 + 1, k0 + 1);
  return ((a00 + a10) + (a01 + a11)) * 0.125;
}

void fill_f2c(Mesh& m, int s, int C, int f, const Neighbor& nb) {
  // coarse ghost = average of its 2^d fine children taken from the 2Ng fine interior layers
  // next to the face.
  int a = f / 2, side = f % 2, N = m.N, h = N / 2, kmax = (m.dim == 3) ? N : 1;
  for (int v = 0; v < m.nvar; ++v)
    for (int g = 1; g <= m.Ng; ++g)
      for (int t2 = 1; t2 <= kmax; ++t2)
        for (int t1 = 1; t1 <= N; ++t1) {
          int o1 = (t1 - 1) / h, tt1 = (t1 - 1) % h;
          int o2 = (m.dim == 3) ? (t2 - 1) / h : 0, tt2 = (m.dim == 3) ? (t2 - 1) % h : 0;
          int F = nb.blk[o1 + 2 * o2];
          int nf = side ? (2 * g - 1) : (N - 2 * g + 1);  // lower of the two fine normal indices
          int fi, fj, fk, di, dj, dk;
          compose(a, nf, 2 * tt1 + 1, (m.dim == 3) ? 2 * tt2 + 1 : 1, fi, fj, fk);
          compose(a, side ? N + g : 1 - g, t1, t2, di, dj, dk);
          m.at(s, C, v, di, dj, dk) = restrict_mean(m, s, F, v, fi, fj, fk);
        }
}

// Limited prolongation of coarse cell (ic,jc,kc) of block C to the child in the
// (sx,sy,sz) half (each +-1): u_c + sum_dim s*1/4*delta_dim, delta from the
// generalised minmod of one-sided differences (eq. 1; reading A9 for 3D).
double prolong_value(Mesh& m, int s, int C, int v, int ic, int jc, int kc, int sx, int sy, int sz) {
  double uc = m.at(s, C, v, ic, jc, kc);
  double dxs = minmod_G(uc - m.at(s, C, v, ic - 1, jc, kc), m.at(s, C, v, ic + 1, jc, kc) - uc, m.theta);
  double dys = minmod_G(uc - m.at(s, C, v, ic, jc - 1, kc), m.at(s, C, v, ic, jc + 1, kc) - uc, m.theta);
  double r = sx * 0.25 * dxs + sy * 0.25 * dys;
  if (m.dim == 3) {
    double dzs = minmod_G(uc - m.at(s, C, v, ic, jc, kc - 1), m.at(s, C, v, ic, jc, kc + 1) - uc, m.theta);
    r = r + sz * 0.25 * dzs;
  }
  return uc + r;
}

void fill_c2f(Mesh& m, int s, int F, int f, const Neighbor& nb) {
  int a = f / 2, side = f % 2, N = m.N, h = N / 2, kmax = (m.dim == 3) ? N : 1;
  int C = nb.blk[0];
  for (int v = 0; v < m.nvar; ++v)
    for (int g = 1; g <= m.Ng; ++g)
      for (int t2 = 1; t2 <= kmax; ++t2)
        for (int t1 = 1; t1 <= N; ++t1) {
          int gc = (g + 1) / 2;  // ceil(g/2)
          int nc, sn;
          if (side) { nc = gc; sn = (g % 2) ? -1 : +1; }            // F's +side ghost: lower half first
          else      { nc = N + 1 - gc; sn = (g % 2) ? +1 : -1; }    // F's -side ghost: upper half first
          int c1 = nb.off[0] * h + (t1 + 1) / 2, s1 = (t1 % 2 == 0) ? +1 : -1;
          int c2 = 1, s2 = 0;
          if (m.dim == 3) { c2 = nb.off[1] * h + (t2 + 1) / 2; s2 = (t2 % 2 == 0) ? +1 : -1; }
          int ic, jc, kc, di, dj, dk, sx, sy, sz;
          compose(a, nc, c1, c2, ic, jc, kc);
          compose(a, sn, s1, s2, sx, sy, sz);
          compose(a, side ? N + g : 1 - g, t1, t2, di, dj, dk);
          m.at(s, F, v, di, dj, dk) = prolong_value(m, s, C, v, ic, jc, kc, sx, sy, sz);
        }
}

// One round of the ghost fill over the blocks [b0, b1) (every block of the range is a DESTINATION: a round writes
// ghost cells of its own blocks only and reads interiors -- round 2 also the round-1 ghosts -- of others).
int fill_ghosts_round(Mesh& m, int s, int round, int b0, int b1) {
  if (round == 1) {
    // R1: SRL, BC and F2C
    for (int b = b0; b < b1; ++b)
      for (int f = 0; f < 2 * m.dim; ++f) {
        Neighbor nb = find_neighbor(m, b, f);
        if (nb.kind == NB_SAME) fill_srl(m, s, b, f, nb.blk[0]);
        else if (nb.kind == NB_BOUNDARY) fill_bc(m, s, b, f);
        else if (nb.kind == NB_FINE) {
          for (int q = 0; q < (m.dim == 3 ? 4 : 2); ++q)
            if (nb.blk[q] < 0) { m.err = "mesh not 2:1 balanced (missing fine neighbour)"; return -1; }
          fill_f2c(m, s, b, f, nb);
        }
      }
  } else {
    // R2: C2F by interpolation, after R1
    for (int b = b0; b < b1; ++b)
      for (int f = 0; f < 2 * m.dim; ++f) {
        Neighbor nb = find_neighbor(m, b, f);
        if (nb.kind == NB_COARSE) fill_c2f(m, s, b, f, nb);
      }
  }
  return 0;
}

int fill_ghosts(Mesh& m, int s) {
  const int nb_ = (int)m.blocks.size();
  int rc;
  if ((rc = fill_ghosts_round(m, s, 1, 0, nb_))) return rc;
  return fill_ghosts_round(m, s, 2, 0, nb_);
}

// ----------------------------------------------------------------------------
// Euler physics
// ----------------------------------------------------------------------------
struct Prim { double rho, u[3], p; };

// to_primitive: rho, u = m/rho, p = (gamma-1)(E - 1/2 rho |u|^2) (eq. 15 inverted)
Prim to_primitive(const Mesh& m, const double* U) {
  Prim w{};
  w.rho = U[0];
  if (m.physics == PHYS_ADVECTION) return w;   // "primitive and conservative variables are identical"
  double ke = 0.0;
  for (int d = 0; d < m.dim; ++d) { w.u[d] = U[1 + d] / w.rho; ke += w.u[d] * w.u[d]; }
  w.p = (m.gamma - 1.0) * (U[m.nvar - 1] - 0.5 * w.rho * ke);
  return w;
}
// to_conservative, eq. (15)
void to_conservative(const Mesh& m, const Prim& w, double* U) {
  double ke = 0.0;
  U[0] = w.rho;
  if (m.physics == PHYS_ADVECTION) return;
  for (int d = 0; d < m.dim; ++d) { U[1 + d] = w.rho * w.u[d]; ke += w.u[d] * w.u[d]; }
  U[m.nvar - 1] = w.p / (m.gamma - 1.0) + 0.5 * w.rho * ke;
}
// get_flux: flux of eq. (14) along direction dir from primitive variables
void get_flux(const Mesh& m, const Prim& w, int dir, double* F) {
  if (m.physics == PHYS_ADVECTION) { F[0] = w.rho * m.vel[dir]; return; }   // eq. (13): flux rho v
  double U[5];
  to_conservative(m, w, U);
  double un = w.u[dir];
  F[0] = w.rho * un;
  for (int d = 0; d < m.dim; ++d) F[1 + d] = w.rho * w.u[d] * un + (d == dir ? w.p : 0.0);
  F[m.nvar - 1] = (U[m.nvar - 1] + w.p) * un;
}
// get_min_max_wavespeed: Einfeldt, reading A3: Roe averages u^ -+ d^
void get_min_max_wavespeed(const Mesh& m, const Prim& L, const Prim& R, int dir, double& smin, double& smax) {
  if (m.physics == PHYS_ADVECTION) {   // "the minimum and maximum wave speeds in direction i are min(v_i, 0) and max(v_i, 0)"
    smin = std::min(m.vel[dir], 0.0);
    smax = std::max(m.vel[dir], 0.0);
    return;
  }
  double rL = std::sqrt(L.rho), rR = std::sqrt(R.rho);
  double cL2 = m.gamma * L.p / L.rho, cR2 = m.gamma * R.p / R.rho;  // eq. (16)
  double uL = L.u[dir], uR = R.u[dir];
  double uhat = (rL * uL + rR * uR) / (rL + rR);
  double dhat2 = (rL * cL2 + rR * cR2) / (rL + rR) +
                 0.5 * rL * rR / ((rL + rR) * (rL + rR)) * (uR - uL) * (uR - uL);
  double dhat = std::sqrt(dhat2);
  smin = uhat - dhat;
  smax = uhat + dhat;
}
// HLL (reading A2) or Rusanov flux at one face
void riemann_flux(const Mesh& m, const Prim& L, const Prim& R, int dir, double* F) {
  double smin, smax;
  get_min_max_wavespeed(m, L, R, dir, smin, smax);
  double Sm, Sp;
  if (m.flux_scheme == FLUX_RUSANOV) {
    double S = std::max(std::fabs(smin), std::fabs(smax));
    Sm = -S; Sp = S;
  } else {
    Sm = std::min(smin, 0.0); Sp = std::max(smax, 0.0);
  }
  double FL[5], FR[5], UL[5], UR[5];
  get_flux(m, L, dir, FL); get_flux(m, R, dir, FR);
  to_conservative(m, L, UL); to_conservative(m, R, UR);
  if (Sp - Sm == 0.0) {   // scalar advection with v_dir = 0: no wave crosses the face, F_L = F_R = 0
    for (int v = 0; v < m.nvar; ++v) F[v] = 0.0;
    return;
  }
  for (int v = 0; v < m.nvar; ++v)
    F[v] = (Sp * FL[v] - Sm * FR[v] + Sp * Sm * (UR[v] - UL[v])) / (Sp - Sm);
}

// ----------------------------------------------------------------------------
// Finite-volume forward-Euler sub-step, eq. (5)
//   u(s_out) = dt_sub * F(u(s_deriv)) + sum_i w_i u(s_prev_i)
// Ghosts of s_deriv must be filled.  Returns 0, or a negative code with Mesh::err set (positivity lost, reading A18).
// ----------------------------------------------------------------------------
// steps (a), (b) and flux-fixing step 0 for the blocks [b0, b1): a block's update reads and writes that block only
int forward_euler_blocks(Mesh& m, int b0, int b1, int s_out, int s_deriv, double dt_sub, int n_prev, const double* w,
                         const int* s_prev) {
  const int N = m.N, Ng = m.Ng, P = m.P, nvar = m.nvar, dim = m.dim;
  const int kmax = (dim == 3) ? N : 1;
  const size_t vs = m.var_stride();
  std::vector<Prim> prim(vs);        // uu_prim
  std::vector<char> valid(vs);
  std::vector<double> result((size_t)nvar * vs);
  for (int b = b0; b < b1; ++b) {
    const double dx = m.dx_of_level(m.blocks[b].level);
    // (a) to_primitive over the padded block; corner/edge ghosts are never used -> skipped
    for (int k = (dim == 3 ? 1 - Ng : 1); k <= (dim == 3 ? N + Ng : 1); ++k)
      for (int j = 1 - Ng; j <= N + Ng; ++j)
        for (int i = 1 - Ng; i <= N + Ng; ++i) {
          int outside = (i < 1 || i > N) + (j < 1 || j > N) + ((dim == 3) && (k < 1 || k > N));
          size_t o = m.off(i, j, k);
          valid[o] = outside <= 1;
          if (!valid[o]) continue;
          double U[5];
          for (int v = 0; v < nvar; ++v) U[v] = m.at(s_deriv, b, v, i, j, k);
          prim[o] = to_primitive(m, U);
        }
    auto W = [&](int i, int j, int k) -> const Prim& { return prim[m.off(i, j, k)]; };
    auto comp = [&](const Prim& q, int v) -> double { return v == 0 ? q.rho : (v == nvar - 1 ? q.p : q.u[v - 1]); };
    auto setc = [&](Prim& q, int v, double x) { if (v == 0) q.rho = x; else if (v == nvar - 1) q.p = x; else q.u[v - 1] = x; };
    // face flux between cell c and c+e_dir: limited primitive reconstruction
    auto face_flux = [&](int i, int j, int k, int dir, double* F) {
      int e[3] = {0, 0, 0}; e[dir] = 1;
      const Prim &wm1 = W(i - e[0], j - e[1], k - e[2]), &w0 = W(i, j, k);
      const Prim &w1 = W(i + e[0], j + e[1], k + e[2]), &w2 = W(i + 2 * e[0], j + 2 * e[1], k + 2 * e[2]);
      Prim L{}, R{};
      for (int v = 0; v < nvar; ++v) {
        double sl = limited_slope(m, comp(w0, v) - comp(wm1, v), comp(w1, v) - comp(w0, v));
        double sr = limited_slope(m, comp(w2, v) - comp(w1, v), comp(w1, v) - comp(w0, v));  // towards its low face
        setc(L, v, comp(w0, v) + 0.5 * sl);  // w_{i+1/2,L}
        setc(R, v, comp(w1, v) - 0.5 * sr);  // w_{i+1/2,R}
      }
      riemann_flux(m, L, R, dir, F);
    };
    // (b) loop over the cells of the block
    for (int k = 1; k <= kmax; ++k)
      for (int j = 1; j <= N; ++j)
        for (int i = 1; i <= N; ++i) {
          // i. source term ("get_source: compute the source term from primitive variables in one
          //    cell"): gravity, eq. (20): S = (0, rho g, rho g.u); zero for the BASELINE configs
          double Lu[5] = {0, 0, 0, 0, 0};
          if (!m.test_rhs && m.physics == PHYS_EULER) {
            const Prim& w0 = W(i, j, k);
            double gu = 0.0;
            for (int a = 0; a < dim; ++a) {
              Lu[1 + a] = w0.rho * m.grav[a];
              gu = gu + m.grav[a] * w0.u[a];
            }
            Lu[nvar - 1] = w0.rho * gu;
          }
          if (m.test_rhs) {
            for (int v = 0; v < nvar; ++v) Lu[v] = m.test_lambda * m.at(s_deriv, b, v, i, j, k);
          } else {
            // ii. fluxes at the cell's faces; subtract their divergence
            for (int dir = 0; dir < dim; ++dir) {
              int e[3] = {0, 0, 0}; e[dir] = 1;
              double Fp[5], Fm[5];
              face_flux(i, j, k, dir, Fp);
              face_flux(i - e[0], j - e[1], k - e[2], dir, Fm);
              for (int v = 0; v < nvar; ++v) Lu[v] -= (Fp[v] - Fm[v]) / dx;
            }
          }
          // iv. Runge-Kutta update, eq. (5)
          for (int v = 0; v < nvar; ++v) {
            double acc = 0.0;
            for (int q = 0; q < n_prev; ++q) {
              double term = w[q] * m.at(s_prev[q], b, v, i, j, k);
              acc = (q == 0) ? term : acc + term;
            }
            result[(size_t)v * vs + m.off(i, j, k)] = dt_sub * Lu[v] + acc;
          }
        }
    // flux fixing, step 0: "during the flux computation, fluxes at refinement boundaries are
    // stored in a pre-allocated array bflux" -- the face-normal flux at every cell face of a block face whose
    // neighbour is coarser or finer, from the same face_flux as the update.
    if (m.flux_fix && !m.test_rhs) {
      for (int f = 0; f < 2 * dim; ++f) {
        Neighbor nb = find_neighbor(m, b, f);
        if (nb.kind != NB_FINE && nb.kind != NB_COARSE) continue;
        const int a = f / 2, side = f % 2;
        std::vector<double>& bf = m.bflux[{b, f}];
        bf.assign((size_t)nvar * N * kmax, 0.0);
        for (int t2 = 1; t2 <= kmax; ++t2)
          for (int t1 = 1; t1 <= N; ++t1) {
            int i, j, k;
            compose(a, side ? N : 0, t1, (dim == 3) ? t2 : 1, i, j, k);   // face between cells n and n+1 along a
            if (dim == 2) k = 1;
            double F[5];
            face_flux(i, j, k, a, F);
            for (int v = 0; v < nvar; ++v) bf[((size_t)v * kmax + (t2 - 1)) * N + (t1 - 1)] = F[v];
          }
      }
    }
    for (int k = 1; k <= kmax; ++k)
      for (int j = 1; j <= N; ++j)
        for (int i = 1; i <= N; ++i)
          for (int v = 0; v < nvar; ++v) {
            double r = result[(size_t)v * vs + m.off(i, j, k)];
            m.at(s_out, b, v, i, j, k) = r;
          }
    // reading A18: positivity is asserted, not repaired
    for (int k = 1; k <= kmax; ++k)
      for (int j = 1; j <= N; ++j)
        for (int i = 1; i <= N; ++i) {
          if (m.test_rhs || m.physics != PHYS_EULER) continue;
          double U[5];
          for (int v = 0; v < nvar; ++v) U[v] = m.at(s_out, b, v, i, j, k);
          Prim q = to_primitive(m, U);
          if (!(q.rho > 0.0) || !(q.p > 0.0)) {
            char buf[200];
            std::snprintf(buf, sizeof buf, "positivity lost: block %d cell (%d,%d,%d) rho=%g p=%g", b, i, j, k, q.rho, q.p);
            m.err = buf;
            return -2;
          }
        }
    (void)P;
  }
  return 0;
}

int forward_euler(Mesh& m, int s_out, int s_deriv, double dt_sub, int n_prev, const double* w, const int* s_prev) {
  const int N = m.N, nvar = m.nvar, dim = m.dim;
  const int kmax = (dim == 3) ? N : 1;
  {
    int rc = forward_euler_blocks(m, 0, (int)m.blocks.size(), s_out, s_deriv, dt_sub, n_prev, w, s_prev);
    if (rc) return rc;
  }
  // flux fixing, step 3: "a loop over all coarse sides of refinement boundaries is performed, and
  // the solution in the cells adjacent to the boundary is corrected based on the difference in the coarse-side
  // flux and the average fine-side flux".  The update above used the coarse flux Fc through that face; with the
  // mean Ff of the 2^(d-1) fine fluxes instead, u changes by -+ dt_sub/dx_c (Ff - Fc) (+ on the low side, where
  // the face flux enters the cell; - on the high side, where it leaves).
  if (m.flux_fix && !m.test_rhs) {
    const int h = N / 2;
    for (int C = 0; C < (int)m.blocks.size(); ++C) {
      const double dxc = m.dx_of_level(m.blocks[C].level);
      for (int f = 0; f < 2 * dim; ++f) {
        Neighbor nb = find_neighbor(m, C, f);
        if (nb.kind != NB_FINE) continue;
        const int a = f / 2, side = f % 2;
        const std::vector<double>& bc = m.bflux[{C, f}];
        for (int v = 0; v < nvar; ++v)
          for (int t2 = 1; t2 <= kmax; ++t2)
            for (int t1 = 1; t1 <= N; ++t1) {
              int o1 = (t1 - 1) / h, tt1 = (t1 - 1) % h;
              int o2 = (dim == 3) ? (t2 - 1) / h : 0, tt2 = (dim == 3) ? (t2 - 1) % h : 0;
              const std::vector<double>& bf = m.bflux[{nb.blk[o1 + 2 * o2], f ^ 1}];
              double sum = 0.0;
              int cnt = 0;
              for (int q2 = 0; q2 < (dim == 3 ? 2 : 1); ++q2)
                for (int q1 = 0; q1 < 2; ++q1) {
                  sum += bf[((size_t)v * kmax + (2 * tt2 + q2)) * N + (2 * tt1 + q1)];
                  ++cnt;
                }
              double Ff = sum / cnt;
              double Fc = bc[((size_t)v * kmax + (t2 - 1)) * N + (t1 - 1)];
              int i, j, k;
              compose(a, side ? N : 1, t1, (dim == 3) ? t2 : 1, i, j, k);
              if (dim == 2) k = 1;
              double corr = dt_sub / dxc * (Ff - Fc);
              m.at(s_out, C, v, i, j, k) += side ? -corr : corr;
            }
      }
    }
  }
  return 0;
}

// iii. CFL: reading A5 (sum over dimensions) on interior cells, one global dt
double max_wave_rate_blocks(Mesh& m, int s, int b0, int b1) {
  const int N = m.N, kmax = (m.dim == 3) ? N : 1;
  double mx = 0.0;
  for (int b = b0; b < b1; ++b) {
    const double dx = m.dx_of_level(m.blocks[b].level);
    for (int k = 1; k <= kmax; ++k)
      for (int j = 1; j <= N; ++j)
        for (int i = 1; i <= N; ++i) {
          double U[5];
          for (int v = 0; v < m.nvar; ++v) U[v] = m.at(s, b, v, i, j, k);
          Prim q = to_primitive(m, U);
          double r = 0.0;
          if (m.physics == PHYS_ADVECTION) {   // the only wave speed is v; reading A5: sum over dimensions
            for (int d = 0; d < m.dim; ++d) r += std::fabs(m.vel[d]) / dx;
          } else {
            double c = std::sqrt(m.gamma * q.p / q.rho);  // eq. (16)
            for (int d = 0; d < m.dim; ++d) r += (std::fabs(q.u[d]) + c) / dx;
          }
          if (r > mx) mx = r;
        }
  }
  return mx;
}
double max_wave_rate(Mesh& m, int s) { return max_wave_rate_blocks(m, s, 0, (int)m.blocks.size()); }

// Heun's method, eq. (6)-(7); ghost fill precedes each F
int advance_heun(Mesh& m, double dt) {
  int rc;
  if ((rc = fill_ghosts(m, 0))) return rc;
  { double w[1] = {1.0}; int sp[1] = {0};
    if ((rc = forward_euler(m, 1, 0, dt, 1, w, sp))) return rc; }          // u1 = dt F(ut) + ut
  if ((rc = fill_ghosts(m, 1))) return rc;
  { double w[2] = {0.5, 0.5}; int sp[2] = {0, 1};
    if ((rc = forward_euler(m, 0, 1, 0.5 * dt, 2, w, sp))) return rc; }    // u = 1/2 dt F(u1) + 1/2 (ut + u1)
  return 0;
}

// The other members of the restricted Runge-Kutta class eq. (5) that foap4 includes: every
// sub-step is one forward_euler call preceded by the ghost fill of the state it differentiates.
// States: 0 = u_t (and the result), 1.. = intermediate u_1, u_2, u_3.
enum { RK_HEUN = 0, RK_EULER = 1, RK_SSP33 = 2, RK_SSP43 = 3, RK_RK4 = 4 };

int advance_rk(Mesh& m, int scheme, double dt) {
  int rc;
  auto sub = [&](int s_out, int s_deriv, double dt_sub, std::vector<double> w, std::vector<int> sp) -> int {
    if ((rc = fill_ghosts(m, s_deriv))) return rc;
    return forward_euler(m, s_out, s_deriv, dt_sub, (int)w.size(), w.data(), sp.data());
  };
  switch (scheme) {
    case RK_HEUN:
      return advance_heun(m, dt);
    case RK_EULER:   // u_{t+1} = dt F(u_t) + u_t
      if ((rc = sub(1, 0, dt, {1.0}, {0}))) return rc;
      m.uu[0] = m.uu[1];
      return 0;
    case RK_SSP33:   // optimal 3-stage SSP scheme [20]: Shu-Osher form with one F per sub-step
      if ((rc = sub(1, 0, dt, {1.0}, {0}))) return rc;                                  // u1 = ut + dt F(ut)
      if ((rc = sub(2, 1, 0.25 * dt, {0.75, 0.25}, {0, 1}))) return rc;                 // u2 = 3/4 ut + 1/4 (u1 + dt F(u1))
      return sub(0, 2, 2.0 / 3.0 * dt, {1.0 / 3.0, 2.0 / 3.0}, {0, 2});                 // u  = 1/3 ut + 2/3 (u2 + dt F(u2))
    case RK_SSP43:   // optimal 4-stage, third-order SSP scheme [20]
      if ((rc = sub(1, 0, 0.5 * dt, {1.0}, {0}))) return rc;                            // u1 = ut + dt/2 F(ut)
      if ((rc = sub(2, 1, 0.5 * dt, {1.0}, {1}))) return rc;                            // u2 = u1 + dt/2 F(u1)
      if ((rc = sub(1, 2, dt / 6.0, {2.0 / 3.0, 1.0 / 3.0}, {0, 2}))) return rc;        // u3 = 2/3 ut + 1/3 (u2 + dt/2 F(u2))
      return sub(0, 1, 0.5 * dt, {1.0}, {1});                                           // u  = u3 + dt/2 F(u3)
    case RK_RK4:     // eq. (8)-(11)
      if ((rc = sub(1, 0, 0.5 * dt, {1.0}, {0}))) return rc;                            // (8)
      if ((rc = sub(2, 1, 0.5 * dt, {1.0}, {0}))) return rc;                            // (9)
      if ((rc = sub(3, 2, dt, {1.0}, {0}))) return rc;                                  // (10)
      return sub(0, 3, dt / 6.0, {-1.0 / 3.0, 1.0 / 3.0, 2.0 / 3.0, 1.0 / 3.0}, {0, 1, 2, 3});   // (11)
  }
  m.err = "unknown Runge-Kutta scheme";
  return -1;
}

// ----------------------------------------------------------------------------
// Mesh adapt + regrid transfer, PAPER.md:111-117 (readings A11, A12)
// ----------------------------------------------------------------------------
std::vector<Key> children_of(const Mesh& m, const Key& k) {
  std::vector<Key> ch;
  int nz = (m.dim == 3) ? 2 : 1;
  for (int dz = 0; dz < nz; ++dz)
    for (int dy = 0; dy < 2; ++dy)
      for (int dx = 0; dx < 2; ++dx)
        ch.push_back(Key{k.level + 1, {2 * k.c[0] + dx, 2 * k.c[1] + dy, (m.dim == 3) ? 2 * k.c[2] + dz : 0}});
  return ch;
}

// 2:1 balance with corner connectivity (P4EST_CONNECT_FULL)
void balance_full(const Mesh& m, std::set<Key>& S) {
  bool changed = true;
  while (changed) {
    changed = false;
    std::vector<Key> leaves(S.begin(), S.end());
    for (const Key& A : leaves) {
      if (!S.count(A)) continue;
      int zlo = (m.dim == 3) ? -1 : 0, zhi = (m.dim == 3) ? 1 : 0;
      for (int dz = zlo; dz <= zhi; ++dz)
        for (int dy = -1; dy <= 1; ++dy)
          for (int dx = -1; dx <= 1; ++dx) {
            if (!dx && !dy && !dz) continue;
            std::array<int, 3> n = {A.c[0] + dx, A.c[1] + dy, A.c[2] + dz};
            bool outside = false;
            for (int a = 0; a < m.dim; ++a) {
              int ext = m.extent(A.level, a);
              if (n[a] < 0 || n[a] >= ext) {
                if (m.bc[2 * a] == BC_PERIODIC) n[a] = (n[a] + ext) % ext; else outside = true;
              }
            }
            if (outside) continue;
            // find the leaf covering region (A.level, n), walking towards the root
            for (int l = A.level; l >= 0; --l) {
              int sh = A.level - l;
              Key q{l, {n[0] >> sh, n[1] >> sh, n[2] >> sh}};
              if (S.count(q)) {
                if (l < A.level - 1) {
                  S.erase(q);
                  for (const Key& c : children_of(m, q)) S.insert(c);
                  changed = true;
                }
                break;
              }
            }
          }
    }
  }
}

int adapt(Mesh& m, const int* flags, int* changed_out) {
  int rc;
  if ((rc = fill_ghosts(m, 0))) return rc;  // prolongation reads the parents' face ghosts
  const int nb_old = (int)m.blocks.size();
  const std::set<Key> old_set(m.blocks.begin(), m.blocks.end());
  std::set<Key> S = old_set;
  // refine (flag > 0)
  for (int b = 0; b < nb_old; ++b)
    if (flags[b] > 0 && m.blocks[b].level < m.max_level) {
      S.erase(m.blocks[b]);
      for (const Key& c : children_of(m, m.blocks[b])) S.insert(c);
    }
  // coarsen (whole family flagged < 0, one level per call, never below base_level), reading A11
  std::map<Key, int> fam;
  for (int b = 0; b < nb_old; ++b) {
    const Key& k = m.blocks[b];
    if (flags[b] < 0 && k.level > m.base_level && S.count(k))
      fam[Key{k.level - 1, {k.c[0] >> 1, k.c[1] >> 1, k.c[2] >> 1}}]++;
  }
  for (auto& pr : fam)
    if (pr.second == (1 << m.dim)) {
      for (const Key& c : children_of(m, pr.first)) S.erase(c);
      S.insert(pr.first);
    }
  balance_full(m, S);

  if (S == old_set) {  // mesh revision unchanged
    *changed_out = 0;
    return 0;
  }
  std::vector<Key> nblocks(S.begin(), S.end());
  // regrid transfer of state 0: copy / prolong / restrict by comparing levels
  Mesh old = m;  // temporary copy of the old blocks
  m.blocks = nblocks;
  rebuild_index(m);
  for (int s = 0; s < m.nstates; ++s) m.uu[s].assign(m.blocks.size() * m.block_stride(), 0.0);
  const int N = m.N, h = N / 2, kmax = (m.dim == 3) ? N : 1;
  for (int b = 0; b < (int)m.blocks.size(); ++b) {
    const Key& k = m.blocks[b];
    auto it = old.index.find(k);
    if (it != old.index.end()) {  // unaltered: copy
      for (int v = 0; v < m.nvar; ++v)
        for (int kk = 1; kk <= kmax; ++kk) for (int j = 1; j <= N; ++j) for (int i = 1; i <= N; ++i)
          m.at(0, b, v, i, j, kk) = old.at(0, it->second, v, i, j, kk);
      continue;
    }
    Key par{k.level - 1, {k.c[0] >> 1, k.c[1] >> 1, k.c[2] >> 1}};
    it = (k.level > 0) ? old.index.find(par) : old.index.end();
    if (it != old.index.end()) {  // refined: prolongation of the parent's interior
      int ox = k.c[0] & 1, oy = k.c[1] & 1, oz = k.c[2] & 1;
      for (int v = 0; v < m.nvar; ++v)
        for (int kk = 1; kk <= kmax; ++kk) for (int j = 1; j <= N; ++j) for (int i = 1; i <= N; ++i) {
          int ic = ox * h + (i + 1) / 2, jc = oy * h + (j + 1) / 2;
          int kc = (m.dim == 3) ? oz * h + (kk + 1) / 2 : 1;
          int sx = (i % 2 == 0) ? 1 : -1, sy = (j % 2 == 0) ? 1 : -1, sz = (kk % 2 == 0) ? 1 : -1;
          m.at(0, b, v, i, j, kk) = prolong_value(old, 0, it->second, v, ic, jc, kc, sx, sy, sz);
        }
      continue;
    }
    // coarsened: restriction of the 2^d children
    for (const Key& c : children_of(m, k)) {
      auto jt = old.index.find(c);
      if (jt == old.index.end()) { m.err = "adapt: block changed by more than one level"; return -3; }
      int ox = c.c[0] & 1, oy = c.c[1] & 1, oz = c.c[2] & 1;
      for (int v = 0; v < m.nvar; ++v)
        for (int kk = 1; kk <= (m.dim == 3 ? h : 1); ++kk) for (int j = 1; j <= h; ++j) for (int i = 1; i <= h; ++i)
          m.at(0, b, v, ox * h + i, oy * h + j, (m.dim == 3) ? oz * h + kk : 1) =
              restrict_mean(old, 0, jt->second, v, 2 * i - 1, 2 * j - 1, (m.dim == 3) ? 2 * kk - 1 : 1);
    }
  }
  *changed_out = 1;
  return 0;
}

// ----------------------------------------------------------------------------
// Refinement criteria: per-block flags {+1 refine, 0 keep, -1 derefine} from a ghost-filled state.
// ----------------------------------------------------------------------------
// CRIT_LOHNER -- PAPER.md:349-362 section 3.3 eq. (12), on stored variable `var` (the paper uses the gas density,
//   PAPER.md:560).  Per interior cell and per direction n = i, j, k:
//     E_n = |u_{n-1} - 2 u_n + u_{n+1}| / (eps_abs + |u_n - u_{n-1}| + |u_{n+1} - u_n| + eps u*),
//     u* = |u_{n-1}| + 2 |u_n| + |u_{n+1}|,   |E| = sqrt(E_i^2 + E_j^2 + E_k^2);
//   "If in one cell in a block |E| > c_refine, mark the block for refinement; if in all cells in a block
//   |E| < c_derefine, mark the block for derefinement; otherwise keep".  No cross-derivative terms, so only face
//   ghosts are read.  params = {c_refine, c_derefine, eps, eps_abs}.
// CRIT_PJUMP -- BASELINE.json config 5 / DESIGN.md reading A15: J = max over face-adjacent cell pairs
//   (interior-interior and interior-first ghost layer) of |p_a - p_b| / min(p_a, p_b), p from eq. (15);
//   +1 if J > hi, -1 if J < lo, else 0.  params = {hi, lo}.
// indicator[b] = max over the block's cells of |E| (or J).  Strict comparisons: ties keep (reading A19).
enum { CRIT_LOHNER = 0, CRIT_PJUMP = 1 };

int refine_flags(Mesh& m, int s, int criterion, int var, const double* params, int* flags, double* indicator) {
  const int N = m.N, dim = m.dim, kmax = (dim == 3) ? N : 1;
  if (criterion == CRIT_LOHNER && (var < 0 || var >= m.nvar)) { m.err = "refine_flags: bad variable"; return -1; }
  if (criterion == CRIT_PJUMP && m.physics != PHYS_EULER) { m.err = "refine_flags: the pressure-jump rule needs Euler"; return -1; }
  auto pressure = [&](int b, int i, int j, int k) {
    double rho = m.at(s, b, 0, i, j, k), ke = 0.0;
    for (int a = 0; a < dim; ++a) { double mom = m.at(s, b, 1 + a, i, j, k); ke = ke + mom * mom; }
    return (m.gamma - 1.0) * (m.at(s, b, m.nvar - 1, i, j, k) - 0.5 * ke / rho);   // eq. (15) inverted
  };
  for (int b = 0; b < (int)m.blocks.size(); ++b) {
    double ind = 0.0;
    for (int k = 1; k <= kmax; ++k)
      for (int j = 1; j <= N; ++j)
        for (int i = 1; i <= N; ++i) {
          double cell = 0.0;
          if (criterion == CRIT_LOHNER) {
            const double c_eps = params[2], c_abs = params[3];
            double sumsq = 0.0;
            for (int a = 0; a < dim; ++a) {
              int e[3] = {0, 0, 0}; e[a] = 1;
              double um = m.at(s, b, var, i - e[0], j - e[1], k - e[2]);
              double u0 = m.at(s, b, var, i, j, k);
              double up = m.at(s, b, var, i + e[0], j + e[1], k + e[2]);
              double num = std::fabs((um - 2.0 * u0) + up);
              double ustar = (std::fabs(um) + 2.0 * std::fabs(u0)) + std::fabs(up);
              double den = ((c_abs + std::fabs(u0 - um)) + std::fabs(up - u0)) + c_eps * ustar;
              double En = num / den;
              sumsq = sumsq + En * En;
            }
            cell = std::sqrt(sumsq);
          } else {
            double p0 = pressure(b, i, j, k);
            for (int a = 0; a < dim; ++a) {
              int e[3] = {0, 0, 0}; e[a] = 1;
              for (int sgn = -1; sgn <= 1; sgn += 2) {
                double p1 = pressure(b, i + sgn * e[0], j + sgn * e[1], k + sgn * e[2]);
                double jump = std::fabs(p0 - p1) / std::min(p0, p1);
                if (jump > cell) cell = jump;
              }
            }
          }
          if (cell > ind) ind = cell;
        }
    if (indicator) indicator[b] = ind;
    flags[b] = (ind > params[0]) ? 1 : ((ind < params[1]) ? -1 : 0);
  }
  return 0;
}

// ----------------------------------------------------------------------------
// Block-parallel DRIVER of the same routines (timing only: bench.py's all-cores cpu_baseline leg; SURVEY 8(d)
// "Timing the oracle beside it").  The routines above are unchanged: every thread calls them on its own contiguous
// range of blocks.  A block's update reads and writes that block only and the CFL maximum does not depend on the
// order, so the results are bit-identical to one thread (tests/test_oracle_pins.py asserts it).  No flux fixing
// here (its bflux map is filled during the update).
// ----------------------------------------------------------------------------
template <typename F>
int over_block_ranges(Mesh& m, int nthreads, F&& body) {
  const int nb = (int)m.blocks.size();
  if (nthreads < 1) nthreads = 1;
  if (nthreads > nb) nthreads = nb;
  std::vector<int> rcs(nthreads, 0);
  std::vector<std::thread> th;
  for (int t = 0; t < nthreads; ++t) {
    const int b0 = (int)((long long)nb * t / nthreads), b1 = (int)((long long)nb * (t + 1) / nthreads);
    th.emplace_back([&, t, b0, b1]() { rcs[t] = body(t, b0, b1); });
  }
  for (auto& x : th) x.join();
  for (int rc : rcs) if (rc) return rc;
  return 0;
}

int fill_ghosts_mt(Mesh& m, int s, int nthreads) {
  int rc;
  if ((rc = over_block_ranges(m, nthreads, [&](int, int b0, int b1) { return fill_ghosts_round(m, s, 1, b0, b1); }))) return rc;
  return over_block_ranges(m, nthreads, [&](int, int b0, int b1) { return fill_ghosts_round(m, s, 2, b0, b1); });
}

int advance_heun_mt(Mesh& m, double dt, int nthreads) {
  if (m.flux_fix) { m.err = "the block-parallel driver does not do flux fixing"; return -3; }
  int rc;
  if ((rc = fill_ghosts_mt(m, 0, nthreads))) return rc;
  { double w[1] = {1.0}; int sp[1] = {0};
    if ((rc = over_block_ranges(m, nthreads, [&](int, int b0, int b1) {
          return forward_euler_blocks(m, b0, b1, 1, 0, dt, 1, w, sp); }))) return rc; }
  if ((rc = fill_ghosts_mt(m, 1, nthreads))) return rc;
  { double w[2] = {0.5, 0.5}; int sp[2] = {0, 1};
    if ((rc = over_block_ranges(m, nthreads, [&](int, int b0, int b1) {
          return forward_euler_blocks(m, b0, b1, 0, 1, 0.5 * dt, 2, w, sp); }))) return rc; }
  return 0;
}

double max_wave_rate_mt(Mesh& m, int s, int nthreads) {
  std::vector<double> mx(std::max(nthreads, 1), 0.0);
  over_block_ranges(m, nthreads, [&](int t, int b0, int b1) { mx[t] = max_wave_rate_blocks(m, s, b0, b1); return 0; });
  double r = 0.0;
  for (double x : mx) if (x > r) r = x;
  return r;
}

}  // namespace

// =============================================================================
// C interface (ctypes) -- used by oracle/oracle.py
// =============================================================================
extern "C" {

void* ora_create(int dim, int block_n, int n_ghost, const int* brick, int base_level, int max_level,
                 const int* bc_kind, double gamma, int n_states) {
  if ((dim != 2 && dim != 3) || block_n % 2 || block_n < n_ghost || 2 * n_ghost > block_n) return nullptr;
  Mesh* m = new Mesh();
  m->dim = dim; m->N = block_n; m->Ng = n_ghost; m->P = block_n + 2 * n_ghost;
  m->Pz = (dim == 3) ? m->P : 1; m->nvar = dim + 2;
  for (int a = 0; a < 3; ++a) m->brick[a] = (a < dim) ? brick[a] : 1;
  m->base_level = base_level; m->max_level = max_level;
  for (int f = 0; f < 6; ++f) m->bc[f] = (f < 2 * dim) ? bc_kind[f] : BC_PERIODIC;
  m->gamma = gamma; m->theta = 1.0; m->limiter = LIM_VANLEER; m->flux_scheme = FLUX_HLL;
  m->nstates = n_states;
  int ez = (dim == 3) ? m->extent(base_level, 2) : 1;
  for (int k = 0; k < ez; ++k)
    for (int j = 0; j < m->extent(base_level, 1); ++j)
      for (int i = 0; i < m->extent(base_level, 0); ++i)
        m->blocks.push_back(Key{base_level, {i, j, k}});
  rebuild_index(*m);
  m->uu.resize(n_states);
  for (auto& u : m->uu) u.assign(m->blocks.size() * m->block_stride(), 0.0);
  return m;
}
void ora_destroy(void* h) { delete (Mesh*)h; }
void ora_set_options(void* h, int limiter, int flux_scheme, double theta) {
  Mesh* m = (Mesh*)h; m->limiter = limiter; m->flux_scheme = flux_scheme; m->theta = theta;
}
void ora_set_flux_fix(void* h, int on) { ((Mesh*)h)->flux_fix = on != 0; }
void ora_set_bc_values(void* h, const double* v) {   // [6][nvar]
  Mesh* m = (Mesh*)h;
  for (int f = 0; f < 6; ++f) for (int q = 0; q < m->nvar; ++q) m->bcv[f][q] = v[f * m->nvar + q];
}
// boundary values of one block face of kind BC_DATA: data[nvar][kmax][N]; all entries are dropped by ora_clear_bc_data
void ora_set_bc_face_data(void* h, int block, int face, const double* data) {
  Mesh* m = (Mesh*)h;
  size_t n = (size_t)m->nvar * m->N * (m->dim == 3 ? m->N : 1);
  m->bcdata[{block, face}] = std::vector<double>(data, data + n);
}
void ora_clear_bc_data(void* h) { ((Mesh*)h)->bcdata.clear(); }
// physics 1 = scalar advection eq. (13) with uniform velocity vel: one variable per cell.  Call
// right after ora_create (the block store is re-allocated for the new number of variables).
int ora_set_physics(void* h, int physics, const double* vel) {
  Mesh* m = (Mesh*)h;
  if (physics != PHYS_EULER && physics != PHYS_ADVECTION) return -1;
  m->physics = physics;
  m->nvar = (physics == PHYS_ADVECTION) ? 1 : m->dim + 2;
  for (int a = 0; a < 3; ++a) m->vel[a] = (vel && a < m->dim) ? vel[a] : 0.0;
  for (auto& u : m->uu) u.assign(m->blocks.size() * m->block_stride(), 0.0);
  return 0;
}
void ora_set_gravity(void* h, const double* g) { for (int a = 0; a < 3; ++a) ((Mesh*)h)->grav[a] = g[a]; }
void ora_set_test_rhs(void* h, int on, double lambda) { Mesh* m = (Mesh*)h; m->test_rhs = on; m->test_lambda = lambda; }
int ora_num_blocks(void* h) { return (int)((Mesh*)h)->blocks.size(); }
void ora_get_blocks(void* h, int* level, int* coords) {
  Mesh* m = (Mesh*)h;
  for (size_t b = 0; b < m->blocks.size(); ++b) {
    level[b] = m->blocks[b].level;
    for (int a = 0; a < 3; ++a) coords[3 * b + a] = m->blocks[b].c[a];
  }
}
double ora_dx(void* h, int level) { return ((Mesh*)h)->dx_of_level(level); }
const char* ora_last_error(void* h) { return ((Mesh*)h)->err.c_str(); }

// interior [block][var][k][j][i] unpadded, or natural padded layout if with_ghosts
void ora_set_state(void* h, int s, const double* src, int with_ghosts) {
  Mesh* m = (Mesh*)h;
  const int N = m->N, Ng = m->Ng, kdim = (m->dim == 3);
  if (with_ghosts) { std::memcpy(m->uu[s].data(), src, m->uu[s].size() * sizeof(double)); return; }
  size_t q = 0;
  for (int b = 0; b < (int)m->blocks.size(); ++b)
    for (int v = 0; v < m->nvar; ++v)
      for (int k = 1; k <= (kdim ? N : 1); ++k) for (int j = 1; j <= N; ++j) for (int i = 1; i <= N; ++i)
        m->at(s, b, v, i, j, k) = src[q++];
  (void)Ng;
}
void ora_get_state(void* h, int s, double* dst, int with_ghosts) {
  Mesh* m = (Mesh*)h;
  const int N = m->N, kdim = (m->dim == 3);
  if (with_ghosts) { std::memcpy(dst, m->uu[s].data(), m->uu[s].size() * sizeof(double)); return; }
  size_t q = 0;
  for (int b = 0; b < (int)m->blocks.size(); ++b)
    for (int v = 0; v < m->nvar; ++v)
      for (int k = 1; k <= (kdim ? N : 1); ++k) for (int j = 1; j <= N; ++j) for (int i = 1; i <= N; ++i)
        dst[q++] = m->at(s, b, v, i, j, k);
}
int ora_fill_ghosts(void* h, int s) { return fill_ghosts(*(Mesh*)h, s); }
double ora_max_wave_rate(void* h, int s) { return max_wave_rate(*(Mesh*)h, s); }
double ora_compute_dt(void* h, int s, double cfl) { return cfl / max_wave_rate(*(Mesh*)h, s); }
int ora_advance(void* h, double dt) { return advance_heun(*(Mesh*)h, dt); }
// block-parallel driver (timing only; bit-identical results)
int ora_advance_mt(void* h, double dt, int nthreads) { return advance_heun_mt(*(Mesh*)h, dt, nthreads); }
double ora_compute_dt_mt(void* h, int s, double cfl, int nthreads) { return cfl / max_wave_rate_mt(*(Mesh*)h, s, nthreads); }
int ora_advance_rk(void* h, int scheme, double dt) { return advance_rk(*(Mesh*)h, scheme, dt); }
int ora_forward_euler(void* h, int s_out, int s_deriv, double dt_sub, int n_prev, const double* w, const int* s_prev) {
  return forward_euler(*(Mesh*)h, s_out, s_deriv, dt_sub, n_prev, w, s_prev);
}
int ora_adapt(void* h, const int* flags, int* changed) { return adapt(*(Mesh*)h, flags, changed); }
// ghosts of state s must be filled (ora_fill_ghosts); criterion 0 = eq. (12), 1 = pressure jump (see refine_flags)
int ora_refine_flags(void* h, int s, int criterion, int var, const double* params, int* flags, double* indicator) {
  return refine_flags(*(Mesh*)h, s, criterion, var, params, flags, indicator);
}

// sum u * dx^d per variable, fixed block order, long double accumulation (P2)
void ora_totals(void* h, int s, double* out) {
  Mesh* m = (Mesh*)h;
  const int N = m->N, kdim = (m->dim == 3);
  for (int v = 0; v < m->nvar; ++v) {
    long double acc = 0.0L;
    for (int b = 0; b < (int)m->blocks.size(); ++b) {
      long double dx = m->dx_of_level(m->blocks[b].level), vol = dx * dx * (kdim ? dx : 1.0L), sb = 0.0L;
      for (int k = 1; k <= (kdim ? N : 1); ++k) for (int j = 1; j <= N; ++j) for (int i = 1; i <= N; ++i)
        sb += (long double)m->at(s, b, v, i, j, k);
      acc += sb * vol;
    }
    out[v] = (double)acc;
  }
}

// reorder block storage: new block q = old block perm[q] (P8)
void ora_permute(void* h, const int* perm) {
  Mesh* m = (Mesh*)h;
  size_t bs = m->block_stride();
  std::vector<Key> nb(m->blocks.size());
  for (size_t q = 0; q < nb.size(); ++q) nb[q] = m->blocks[perm[q]];
  for (auto& u : m->uu) {
    std::vector<double> t(u.size());
    for (size_t q = 0; q < nb.size(); ++q) std::memcpy(&t[q * bs], &u[(size_t)perm[q] * bs], bs * sizeof(double));
    u.swap(t);
  }
  m->blocks = nb;
  rebuild_index(*m);
}

// face classification for cross-checking the library's pattern on the CPU:
// kind[b*2d+f] in {0 boundary,1 same,2 coarse,3 fine}; nbr[(b*2d+f)*4+q] block ids; off[(b*2d+f)*2+t]
void ora_face_table(void* h, int* kind, int* nbr, int* off) {
  Mesh* m = (Mesh*)h;
  int nf = 2 * m->dim;
  for (int b = 0; b < (int)m->blocks.size(); ++b)
    for (int f = 0; f < nf; ++f) {
      Neighbor nb = find_neighbor(*m, b, f);
      size_t q = (size_t)b * nf + f;
      kind[q] = nb.kind;
      for (int r = 0; r < 4; ++r) nbr[q * 4 + r] = -1;
      if (nb.kind == NB_SAME || nb.kind == NB_COARSE) nbr[q * 4] = nb.blk[0];
      if (nb.kind == NB_FINE) for (int r = 0; r < (m->dim == 3 ? 4 : 2); ++r) nbr[q * 4 + r] = nb.blk[r];
      off[q * 2] = (nb.kind == NB_COARSE) ? nb.off[0] : 0;
      off[q * 2 + 1] = (nb.kind == NB_COARSE) ? nb.off[1] : 0;
    }
}

// elementary functions exposed for the pins
double ora_minmod_G(double a, double b, double theta) { return minmod_G(a, b, theta); }
double ora_vanleer(double a, double b) { return vanleer(a, b); }
double ora_koren(double a, double b) { return koren(a, b); }
double ora_weno3(double a, double b) { return weno3(a, b); }
// HLL/Rusanov flux for primitive states wL, wR = (rho, u[dim], p) along dir
void ora_riemann_flux(int dim, double gamma, int flux_scheme, const double* wL, const double* wR, int dir, double* F) {
  Mesh m{}; m.dim = dim; m.nvar = dim + 2; m.gamma = gamma; m.flux_scheme = flux_scheme;
  Prim L{}, R{};
  L.rho = wL[0]; R.rho = wR[0]; L.p = wL[dim + 1]; R.p = wR[dim + 1];
  for (int d = 0; d < dim; ++d) { L.u[d] = wL[1 + d]; R.u[d] = wR[1 + d]; }
  riemann_flux(m, L, R, dir, F);
}
void ora_to_primitive(int dim, double gamma, const double* U, double* w) {
  Mesh m{}; m.dim = dim; m.nvar = dim + 2; m.gamma = gamma;
  Prim q = to_primitive(m, U);
  w[0] = q.rho;
  for (int a = 0; a < dim; ++a) w[1 + a] = q.u[a];
  w[dim + 1] = q.p;
}
void ora_to_conservative(int dim, double gamma, const double* w, double* U) {
  Mesh m{}; m.dim = dim; m.nvar = dim + 2; m.gamma = gamma;
  Prim q{};
  q.rho = w[0];
  for (int a = 0; a < dim; ++a) q.u[a] = w[1 + a];
  q.p = w[dim + 1];
  to_conservative(m, q, U);
}
// face flux of scalar advection eq. (13) with velocity vel between the states rhoL, rhoR (test hook)
double ora_advection_flux(int dim, const double* vel, int flux_scheme, double rhoL, double rhoR, int dir) {
  Mesh m{}; m.dim = dim; m.nvar = 1; m.physics = PHYS_ADVECTION; m.flux_scheme = flux_scheme;
  for (int a = 0; a < 3; ++a) m.vel[a] = (a < dim) ? vel[a] : 0.0;
  Prim L{}, R{};
  L.rho = rhoL; R.rho = rhoR;
  double F[5];
  riemann_flux(m, L, R, dir, F);
  return F[0];
}
void ora_wavespeeds(int dim, double gamma, const double* wL, const double* wR, int dir, double* smin, double* smax) {
  Mesh m{}; m.dim = dim; m.nvar = dim + 2; m.gamma = gamma;
  Prim L{}, R{};
  L.rho = wL[0]; R.rho = wR[0]; L.p = wL[dim + 1]; R.p = wR[dim + 1];
  for (int d = 0; d < dim; ++d) { L.u[d] = wL[1 + d]; R.u[d] = wR[1 + d]; }
  get_min_max_wavespeed(m, L, R, dir, *smin, *smax);
}

}  // extern "C"
