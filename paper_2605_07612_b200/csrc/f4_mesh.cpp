// Host-side mesh of the f4 library (see f4_mesh.hpp).  Written from the
// paper's statement of what p4est provides: refine, coarsen,
// balance with P4EST_CONNECT_FULL semantics, face connectivity with hanging
// face offsets.  Linear octree: leaves sorted by the Morton key of their low
// corner at max_level resolution; lookups are binary searches.
#include "f4_mesh.hpp"

#include <algorithm>
#include <deque>
#include <string>
#include <vector>

#include "../../include/f4.h"

namespace f4 {

static inline uint64_t spread3(uint64_t v) {  // 21 bits -> every third bit
  v &= 0x1fffffULL;
  v = (v | v << 32) & 0x1f00000000ffffULL;
  v = (v | v << 16) & 0x1f0000ff0000ffULL;
  v = (v | v << 8) & 0x100f00f00f00f00fULL;
  v = (v | v << 4) & 0x10c30c30c30c30c3ULL;
  v = (v | v << 2) & 0x1249249249249249ULL;
  return v;
}
uint64_t morton3(uint32_t x, uint32_t y, uint32_t z) { return spread3(x) | spread3(y) << 1 | spread3(z) << 2; }

// (level, c) packed into one word for hashing: 5 + 3*19 bits
static inline uint64_t pack(int level, int cx, int cy, int cz) {
  return (uint64_t)level | (uint64_t)cx << 5 | (uint64_t)cy << 24 | (uint64_t)cz << 43;
}
// Open-addressing hash map for packed keys (linear probing, tombstones; keys never reach the two sentinels): the
// mesh adapt is a few thousand inserts / lookups per call, where std::unordered_* spends its time allocating nodes.
class KeyMap {
 public:
  explicit KeyMap(size_t expected) {
    size_t cap = 64;
    while (cap < 2 * expected + 64) cap <<= 1;
    k_.assign(cap, EMPTY);
    v_.assign(cap, 0);
    mask_ = cap - 1;
  }
  int* find(uint64_t key) {
    for (size_t i = hash(key) & mask_;; i = (i + 1) & mask_) {
      if (k_[i] == key) return &v_[i];
      if (k_[i] == EMPTY) return nullptr;
    }
  }
  bool count(uint64_t key) { return find(key) != nullptr; }
  void set(uint64_t key, int val) {
    if (int* p = find(key)) { *p = val; return; }
    if (2 * (used_ + 1) > k_.size()) grow();
    size_t i = hash(key) & mask_;
    while (k_[i] != EMPTY && k_[i] != TOMB) i = (i + 1) & mask_;
    if (k_[i] == EMPTY) ++used_;
    k_[i] = key;
    v_[i] = val;
    ++n_;
  }
  int& ref(uint64_t key) {   // value of key, inserted as 0 if absent
    if (!find(key)) set(key, 0);
    return *find(key);
  }
  void erase(uint64_t key) {
    for (size_t i = hash(key) & mask_;; i = (i + 1) & mask_) {
      if (k_[i] == key) { k_[i] = TOMB; --n_; return; }
      if (k_[i] == EMPTY) return;
    }
  }
  size_t size() const { return n_; }
  template <class F>
  void for_each(F f) const {
    for (size_t i = 0; i < k_.size(); ++i)
      if (k_[i] < TOMB) f(k_[i], v_[i]);
  }

 private:
  static constexpr uint64_t EMPTY = ~0ULL, TOMB = ~0ULL - 1;
  static uint64_t hash(uint64_t x) {
    x ^= x >> 31;
    x *= 0x9E3779B97F4A7C15ULL;
    return x ^ (x >> 29);
  }
  void grow() {
    std::vector<uint64_t> ok;
    std::vector<int> ov;
    ok.swap(k_);
    ov.swap(v_);
    k_.assign(ok.size() * 2, EMPTY);
    v_.assign(ok.size() * 2, 0);
    mask_ = k_.size() - 1;
    n_ = used_ = 0;
    for (size_t i = 0; i < ok.size(); ++i)
      if (ok[i] < TOMB) set(ok[i], ov[i]);
  }
  std::vector<uint64_t> k_;
  std::vector<int> v_;
  size_t mask_ = 0, n_ = 0, used_ = 0;
};

static inline Leaf unpack(uint64_t k) {
  Leaf l;
  l.level = (int)(k & 31);
  l.c[0] = (int)(k >> 5 & 0x7ffff);
  l.c[1] = (int)(k >> 24 & 0x7ffff);
  l.c[2] = (int)(k >> 43 & 0x7ffff);
  return l;
}

double HostMesh::dx_of_level(int level) const {
  int mb = std::max(brick[0], std::max(brick[1], dim == 3 ? brick[2] : 1));
  return 1.0 / ((double)mb * (double)(1u << level) * (double)N);
}

int HostMesh::init(std::string& err) {
  if (dim != 2 && dim != 3) { err = "dim must be 2 or 3"; return F4_EINVAL; }
  if (N < 2 || N % 2 || N < Ng || 2 * Ng > N || Ng < 1) {  // PAPER.md:141; 2Ng <= N for restriction into ghosts
    err = "block_n must be even, >= n_ghost and >= 2*n_ghost";
    return F4_EINVAL;
  }
  if (base_level < 0 || max_level < base_level || max_level > 18) { err = "bad levels"; return F4_EINVAL; }
  for (int a = 0; a < dim; ++a) {
    if (brick[a] < 1 || ((int64_t)brick[a] << max_level) > (1 << 19)) { err = "bad brick"; return F4_EINVAL; }
    if ((bc[2 * a] == F4_BC_PERIODIC) != (bc[2 * a + 1] == F4_BC_PERIODIC)) {
      err = "an axis is periodic only if both of its faces are";
      return F4_EINVAL;
    }
  }
  for (int f = 0; f < 2 * dim; ++f)
    if (bc[f] < 0 || bc[f] > F4_BC_DATA) { err = "bad bc_kind"; return F4_EINVAL; }
  if (dim == 2) brick[2] = 1;
  int64_t nb = 1;
  for (int a = 0; a < dim; ++a) nb *= extent(base_level, a);
  if (nb > max_blocks) { err = "base mesh exceeds max_blocks"; return F4_ENOBLOCKS; }
  leaves.clear();
  int ez = (dim == 3) ? extent(base_level, 2) : 1;
  for (int k = 0; k < ez; ++k)
    for (int j = 0; j < extent(base_level, 1); ++j)
      for (int i = 0; i < extent(base_level, 0); ++i) leaves.push_back(Leaf{base_level, {i, j, k}});
  sort_leaves();
  return build_pattern(err);
}

void HostMesh::sort_leaves() {
  std::vector<std::pair<uint64_t, Leaf>> t(leaves.size());
  for (size_t q = 0; q < leaves.size(); ++q) {
    const Leaf& l = leaves[q];
    int sh = max_level - l.level;
    t[q] = {morton3((uint32_t)l.c[0] << sh, (uint32_t)l.c[1] << sh, (uint32_t)l.c[2] << sh), l};
  }
  std::sort(t.begin(), t.end(), [](const auto& a, const auto& b) { return a.first < b.first; });
  mkeys.resize(t.size());
  for (size_t q = 0; q < t.size(); ++q) { mkeys[q] = t[q].first; leaves[q] = t[q].second; }
}

int HostMesh::find_leaf(int level, const int c[3]) const {
  int sh = max_level - level;
  uint32_t ax = (uint32_t)c[0] << sh, ay = (uint32_t)c[1] << sh, az = (uint32_t)c[2] << sh;
  uint64_t m = morton3(ax, ay, az);
  auto it = std::upper_bound(mkeys.begin(), mkeys.end(), m);
  if (it == mkeys.begin()) return -1;
  int q = (int)(it - mkeys.begin()) - 1;
  const Leaf& l = leaves[q];
  int s2 = max_level - l.level;
  if ((int)(ax >> s2) != l.c[0] || (int)(ay >> s2) != l.c[1] || (int)(az >> s2) != l.c[2]) return -1;
  return q;
}

static inline void transverse(int a, int& ta, int& tb) {
  if (a == 0) { ta = 1; tb = 2; } else if (a == 1) { ta = 0; tb = 2; } else { ta = 0; tb = 1; }
}

int HostMesh::build_pattern(std::string& err) {
  r1.clear();
  r2.clear();
  n_bc_faces = 0;
  const int nb = (int)leaves.size();
  r1.reserve((size_t)nb * 2 * dim);
  // (level, coordinates) -> leaf index: on a balanced mesh the neighbour across a face is the same-level region, its
  // parent, or its children, so one or two hash lookups decide the case
  KeyMap idx(nb);
  for (int b = 0; b < nb; ++b) idx.set(pack(leaves[b].level, leaves[b].c[0], leaves[b].c[1], leaves[b].c[2]), b);
  for (int b = 0; b < nb; ++b) {
    const Leaf& L = leaves[b];
    for (int f = 0; f < 2 * dim; ++f) {
      const int a = f / 2, side = f % 2;
      int n[3] = {L.c[0], L.c[1], L.c[2]};
      n[a] += side ? 1 : -1;
      const int ext = extent(L.level, a);
      if (n[a] < 0 || n[a] >= ext) {
        if (bc[f] == F4_BC_PERIODIC) n[a] = (n[a] + ext) % ext;
        else {
          // o1 / o2 of a boundary record carry its kind: (0,0) outflow, (1,0) Dirichlet, (0,1) Neumann
          if (bc[f] == F4_BC_OUTFLOW) r1.push_back(Record{F4_OP_BC, f, b, b, 0, 0});
          else if (bc[f] == F4_BC_DIRICHLET) r1.push_back(Record{F4_OP_BC, f, b, b, 1, 0});
          else if (bc[f] == F4_BC_NEUMANN) r1.push_back(Record{F4_OP_BC, f, b, b, 0, 1});
          // (1,1): spatially varying data; src is the face's index ibf into bc_data
          else if (bc[f] == F4_BC_DATA) r1.push_back(Record{F4_OP_BC, f, b, n_bc_faces++, 1, 1});
          continue;  // F4_BC_KEEP: no record
        }
      }
      int q = -1, ql = L.level + 1;   // neither the region nor its parent is a leaf: refined (or not balanced)
      if (int* ps = idx.find(pack(L.level, n[0], n[1], n[2]))) { q = *ps; ql = L.level; }
      else if (L.level > 0) {
        if (int* pp = idx.find(pack(L.level - 1, n[0] >> 1, n[1] >> 1, n[2] >> 1))) { q = *pp; ql = L.level - 1; }
      }
      int ta, tb;
      transverse(a, ta, tb);
      if (ql == L.level) {
        r1.push_back(Record{F4_OP_SRL, f, b, q, 0, 0});
      } else if (ql == L.level - 1) {
        // this block is fine, neighbour coarse: prolongation in R2; offset = position in the group
        r2.push_back(Record{F4_OP_C2F, f, b, q, L.c[ta] & 1, dim == 3 ? (L.c[tb] & 1) : 0});
      } else if (ql > L.level) {
        // neighbour region is refined: the 2^(d-1) children touching the face restrict into my ghosts (R1)
        for (int o2 = 0; o2 < (dim == 3 ? 2 : 1); ++o2)
          for (int o1 = 0; o1 < 2; ++o1) {
            int cc[3] = {2 * n[0], 2 * n[1], dim == 3 ? 2 * n[2] : 0};
            cc[a] += side ? 0 : 1;
            cc[ta] += o1;
            if (dim == 3) cc[tb] += o2;
            int* pf = idx.find(pack(L.level + 1, cc[0], cc[1], cc[2]));
            if (!pf) {
              err = "face connectivity: neighbour differs by more than one level (mesh not 2:1 balanced)";
              return F4_EUNBALANCED;
            }
            r1.push_back(Record{F4_OP_F2C, f, b, *pf, o1, o2});
          }
      }
    }
  }
  return F4_OK;
}

int HostMesh::adapt(const int* flags, std::vector<Transfer>& plan, bool& changed, std::string& err) {
  changed = false;
  plan.clear();
  const int nb_old = (int)leaves.size();
  const int nch = 1 << dim;
  {  // no flag that can take effect: the mesh (already balanced) stays as it is
    bool any = false;
    for (int b = 0; b < nb_old && !any; ++b)
      any = (flags[b] > 0 && leaves[b].level < max_level) || (flags[b] < 0 && leaves[b].level > base_level);
    if (!any) return F4_OK;
  }
  KeyMap old_index(nb_old), S(2 * nb_old);   // old leaves -> index; the leaf set being edited
  for (int b = 0; b < nb_old; ++b) {
    uint64_t k = pack(leaves[b].level, leaves[b].c[0], leaves[b].c[1], leaves[b].c[2]);
    old_index.set(k, b);
    S.set(k, 1);
  }
  auto children = [&](const Leaf& l, uint64_t* out) {
    int q = 0;
    for (int dz = 0; dz < (dim == 3 ? 2 : 1); ++dz)
      for (int dy = 0; dy < 2; ++dy)
        for (int dx = 0; dx < 2; ++dx)
          out[q++] = pack(l.level + 1, 2 * l.c[0] + dx, 2 * l.c[1] + dy, dim == 3 ? 2 * l.c[2] + dz : 0);
  };
  uint64_t ch[8];
  // 1. refine
  for (int b = 0; b < nb_old; ++b)
    if (flags[b] > 0 && leaves[b].level < max_level) {
      S.erase(pack(leaves[b].level, leaves[b].c[0], leaves[b].c[1], leaves[b].c[2]));
      children(leaves[b], ch);
      for (int q = 0; q < nch; ++q) S.set(ch[q], 1);
    }
  // 2. coarsen complete families of old leaves, one level, never below base_level
  {
    KeyMap fam(nb_old / 4 + 16);
    for (int b = 0; b < nb_old; ++b) {
      const Leaf& l = leaves[b];
      if (flags[b] < 0 && l.level > base_level) fam.ref(pack(l.level - 1, l.c[0] >> 1, l.c[1] >> 1, l.c[2] >> 1))++;
    }
    // A family whose parent would touch a leaf two levels finer is not coarsened: balance (which only refines)
    // would split the parent again at once.  Checking here keeps the balance work list below to the NEW leaves.
    auto can_coarsen = [&](const Leaf& par) {
      for (int dz = (dim == 3 ? -1 : 0); dz <= (dim == 3 ? 1 : 0); ++dz)
        for (int dy = -1; dy <= 1; ++dy)
          for (int dx = -1; dx <= 1; ++dx) {
            if (!dx && !dy && !dz) continue;
            const int d[3] = {dx, dy, dz};
            int n[3] = {par.c[0] + dx, par.c[1] + dy, par.c[2] + dz};
            bool outside = false;
            for (int a = 0; a < dim; ++a) {
              int ext = extent(par.level, a);
              if (n[a] < 0 || n[a] >= ext) {
                if (bc[2 * a] == F4_BC_PERIODIC) n[a] = (n[a] + ext) % ext; else outside = true;
              }
            }
            if (outside) continue;
            bool covered = false;   // the neighbour region is a leaf or inside a coarser leaf
            for (int l = par.level; l >= 0 && !covered; --l) {
              int sh = par.level - l;
              covered = S.count(pack(l, n[0] >> sh, n[1] >> sh, n[2] >> sh));
            }
            if (covered) continue;
            // subdivided: its children that touch the parent must be leaves (level par.level + 1), not finer
            for (int cz = 0; cz < (dim == 3 ? 2 : 1); ++cz)
              for (int cy = 0; cy < 2; ++cy)
                for (int cx = 0; cx < 2; ++cx) {
                  const int cc[3] = {cx, cy, cz};
                  bool touches = true;
                  for (int a = 0; a < dim; ++a)
                    if ((d[a] == 1 && cc[a] != 0) || (d[a] == -1 && cc[a] != 1)) touches = false;
                  if (!touches) continue;
                  if (!S.count(pack(par.level + 1, 2 * n[0] + cx, 2 * n[1] + cy, dim == 3 ? 2 * n[2] + cz : 0))) return false;
                }
          }
      return true;
    };
    fam.for_each([&](uint64_t kp, int members) {
      if (members == nch && can_coarsen(unpack(kp))) {
        Leaf par = unpack(kp);
        children(par, ch);
        for (int q = 0; q < nch; ++q) S.erase(ch[q]);
        S.set(kp, 1);
      }
    });
  }
  // 3. balance, corner connectivity: ripple from a work queue
  {
    // the old mesh was balanced, so only a leaf created by this call can be the finer side of a violation
    std::deque<uint64_t> Q;
    S.for_each([&](uint64_t k, int) {
      if (!old_index.count(k)) Q.push_back(k);
    });
    while (!Q.empty()) {
      uint64_t ka = Q.front();
      Q.pop_front();
      if (!S.count(ka)) continue;
      Leaf A = unpack(ka);
      if (A.level < 2) continue;   // nothing can be two levels coarser
      // A leaf Q that touches A (face, edge or corner) and is more than one level coarser contains the parent region
      // R' (level A.level-1) of one of A's 26 neighbour regions.  Those parents are A's own parent P shifted by 0 or
      // by one step TOWARDS the corner of P in which A sits: at most 7 regions.  R' violates iff one of its
      // ancestors (levels A.level-2 .. 0) is a leaf.
      const int lp = A.level - 1;
      const int pc[3] = {A.c[0] >> 1, A.c[1] >> 1, A.c[2] >> 1};
      const int st[3] = {(A.c[0] & 1) ? 1 : -1, (A.c[1] & 1) ? 1 : -1, (A.c[2] & 1) ? 1 : -1};
      bool again = false;
      for (int mz = 0; mz <= (dim == 3 ? 1 : 0) && !again; ++mz)
        for (int my = 0; my <= 1 && !again; ++my)
          for (int mx = 0; mx <= 1 && !again; ++mx) {
            if (!mx && !my && !mz) continue;
            int n[3] = {pc[0] + mx * st[0], pc[1] + my * st[1], pc[2] + mz * st[2]};
            bool outside = false;
            for (int a = 0; a < dim; ++a) {
              int ext = extent(lp, a);
              if (n[a] < 0 || n[a] >= ext) {
                if (bc[2 * a] == F4_BC_PERIODIC) n[a] = (n[a] + ext) % ext; else outside = true;
              }
            }
            if (outside) continue;
            for (int l = lp - 1; l >= 0; --l) {
              int sh = lp - l;
              uint64_t kq = pack(l, n[0] >> sh, n[1] >> sh, n[2] >> sh);
              if (S.count(kq)) {
                S.erase(kq);
                children(unpack(kq), ch);
                for (int q = 0; q < nch; ++q) { S.set(ch[q], 1); Q.push_back(ch[q]); }
                Q.push_back(ka);  // look again: the new children may still be too coarse
                again = true;
                break;
              }
            }
          }
    }
  }
  // 4. unchanged? (mesh revision)
  if ((int)S.size() == nb_old) {
    bool same = true;
    old_index.for_each([&](uint64_t k, int) { if (!S.count(k)) same = false; });
    if (same) return F4_OK;
  }
  if ((int)S.size() > max_blocks) {
    err = "adapt: mesh would need " + std::to_string(S.size()) + " blocks > max_blocks";
    return F4_ENOBLOCKS;
  }
  // 5. new leaf array + transfer plan by comparing with the old leaves
  std::vector<Leaf> old_leaves;
  old_leaves.swap(leaves);
  leaves.reserve(S.size());
  S.for_each([&](uint64_t k, int) { leaves.push_back(unpack(k)); });
  sort_leaves();
  plan.resize(leaves.size());
  for (int b = 0; b < (int)leaves.size(); ++b) {
    const Leaf& l = leaves[b];
    Transfer t{};
    t.dst = b;
    int* it = old_index.find(pack(l.level, l.c[0], l.c[1], l.c[2]));
    if (it) {
      t.kind = 0;
      t.src[0] = *it;
    } else if (l.level > 0 && (it = old_index.find(pack(l.level - 1, l.c[0] >> 1, l.c[1] >> 1, l.c[2] >> 1)))) {
      t.kind = 1;
      t.src[0] = *it;
      t.oct = (l.c[0] & 1) | (l.c[1] & 1) << 1 | (l.c[2] & 1) << 2;
    } else {
      t.kind = 2;
      children(l, ch);
      for (int q = 0; q < nch; ++q) {
        int* jt = old_index.find(ch[q]);
        if (!jt) { err = "adapt: block changed by more than one level"; leaves.swap(old_leaves); sort_leaves(); return F4_EINVAL; }
        t.src[q] = *jt;
      }
    }
    plan[b] = t;
  }
  changed = true;
  return build_pattern(err);
}

}  // namespace f4
