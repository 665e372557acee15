// sc_internal.h — internal types of libsubcycle (not part of the ABI).
//
// Data layout in HBM: every box owns NSLOT = 7 slots; a slot holds the
// V = 2F component arrays of the box back to back; a component array is the box padded by g ghost
// cells, stored [z][y][x] with x contiguous:
//     offset(i,j,k) = (XOFF + i) + px * ((j + g) + py * (k + g)),   i in [-g, n0+g) etc.
// XOFF = 4 doubles puts interior cell i = 0 on a 32-byte sector boundary; px is a multiple of 16
// doubles so every row starts on a 128-byte line. Slots 0..2 rotate between the roles y / Y_even /
// y_old (PAPER.md:54-75 needs y_n, one stage vector being read and one being written); slots 3..6
// hold k_1..k_4, which the child level reads for its dense-output ghost fill ("Store k").
#ifndef SC_INTERNAL_H_
#define SC_INTERNAL_H_

#include <cstddef>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/subcycle.h"

#ifdef __CUDACC__
#define SC_HD __host__ __device__
#else
#define SC_HD
#endif

namespace sc {

constexpr int XOFF = 4;        // doubles of left padding in x (>= max ghost width)
constexpr int MAX_GHOST = 4;
constexpr int MIN_GHOST = 2;   // stencil radius of the 4th-order Laplacian; restriction reads 2 layers
constexpr int NSLOT = 7;       // 3 rotating state buffers + k1..k4
constexpr int SLOT_K1 = 3;
constexpr int MAX_FIELDS = 32;

// Geometry of one box's arrays; passed by value to kernels.
struct BoxView {
  int n[3];        // interior cells (x, y, z)
  int lo[3];       // level-global index of interior cell 0
  int g;           // ghost width
  int px;          // x pitch in doubles
  int py;          // rows per plane  = n[1] + 2g
  int pz;          // planes          = n[2] + 2g
  long long plane; // px * py
  long long vol;   // doubles per component array = px * py * pz (multiple of 32)
};

SC_HD inline long long cell_offset(const BoxView& b, int i, int j, int k) {
  return (long long)(XOFF + i) + (long long)b.px * ((long long)(j + b.g) + (long long)b.py * (k + b.g));
}

struct BoxInfo {
  BoxView v;
  int level;
  int index_in_level;
  int parent;            // global box index on level-1, or -1
  unsigned long long arena_offset;  // bytes, start of slot 0
  unsigned long long slot_bytes;    // bytes of one slot (V arrays)
};

struct Layout {
  int nlevels = 0, g = 3, F = 1, V = 2;
  int domain[3] = {0, 0, 0};
  double xlo[3] = {0, 0, 0}, xhi[3] = {0, 0, 0};
  std::vector<BoxInfo> boxes;
  std::vector<std::vector<int>> level_boxes;
  unsigned long long coupling_offset = 0;   // bytes into the arena (F*F doubles) if has_coupling
  unsigned long long scratch_offset = 0;
  unsigned long long arena_bytes = 0;
  bool has_coupling = false;
  double dx(int level, int a) const { return (xhi[a] - xlo[a]) / ((double)domain[a] * (double)(1u << level)); }
};

// Validate a description and compute the layout. Host only, no CUDA calls.
// Returns SC_OK or an SC_ERR_* code; err receives a message.
int build_layout(const sc_hierarchy_desc* d, Layout* out, std::string* err);

void set_error(const std::string& msg);

}  // namespace sc

#endif  // SC_INTERNAL_H_
