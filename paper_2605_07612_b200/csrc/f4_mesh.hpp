// Host-side mesh of the f4 library: brick of quad/octrees stored as a linear
// (Morton-ordered) leaf array, 2:1 balance with corner connectivity, face
// connectivity -> ghost pattern records, regrid transfer plan.
// Replaces p4est (section 2.2) for one GPU.  Plain C++, no CUDA.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace f4 {

struct Leaf {
  int level;
  int c[3];  // block coordinates on the level's grid
};

// One ghost-pattern record: the face `face` of block `dst`
// is filled from block `src` with operation `op` (include/f4.h F4_OP_*).
struct Record {
  int op, face, dst, src, o1, o2;
};

// regrid transfer: how new block `dst` gets its data from the old mesh
struct Transfer {
  int kind;    // 0 copy, 1 prolong from old parent src[0] (octant `oct`), 2 restrict from 2^d old children src[]
  int dst;
  int oct;
  int src[8];
};

class HostMesh {
 public:
  int dim = 3, N = 16, Ng = 2;
  int brick[3] = {1, 1, 1};
  int base_level = 0, max_level = 0;
  int bc[6] = {0, 0, 0, 0, 0, 0};
  int max_blocks = 0;
  std::vector<Leaf> leaves;       // Morton order of the anchors at max_level resolution
  std::vector<uint64_t> mkeys;    // sorted Morton keys, parallel to leaves
  std::vector<Record> r1, r2;     // rounds R1 {SRL, BC, F2C} and R2 {C2F}
  int n_bc_faces = 0;             // block faces with spatially varying boundary data (their records' src = ibf)

  int init(std::string& err);
  int extent(int level, int a) const { return brick[a] << level; }
  double dx_of_level(int level) const;
  // index of the leaf containing the low corner of region (level, c), or -1
  int find_leaf(int level, const int c[3]) const;
  int build_pattern(std::string& err);
  // refine / coarsen / balance.  On change fills `plan`
  // (indices into the OLD leaf array) and replaces leaves.
  int adapt(const int* flags, std::vector<Transfer>& plan, bool& changed, std::string& err);

 private:
  void sort_leaves();
};

uint64_t morton3(uint32_t x, uint32_t y, uint32_t z);

}  // namespace f4
