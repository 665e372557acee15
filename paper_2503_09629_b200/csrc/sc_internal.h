// sc_internal.h — internal types of libsubcycle (not part of the ABI).
//
// Data layout in HBM. A box owns a run of equally sized ARRAYS; an array is one
// scalar grid function on the box padded by g ghost cells, stored [z][y][x] with x contiguous:
//     offset(i,j,k) = (XOFF + i) + px * ((j + g) + py * (k + g)),   i in [-g, n0+g) etc.
// XOFF = 8 doubles puts interior cell i = 0 on a 64-byte boundary; px is a multiple of 16 doubles so
// every row starts on a 128-byte line (and every TMA global stride is a multiple of 16 bytes).
// Arrays of a box, in order (F = number of fields, V = 2F):
//     [0, V)            state slot 0:  u_0..u_{F-1}, rho_0..rho_{F-1}
//     [V, 2V)           state slot 1   (slots 0/1 alternate between y_n and y_{n+1})
//     [2V, 2V+F)        Y2r = rho-part of the stage vector Y_2 (eq 7)
//     [2V+F, 2V+2F)     Y3r = rho-part of Y_3 (eq 8)
//     [2V+2F, 2V+3F)    Y4r = rho-part of Y_4 (eq 9)
//     [2V+3F, 2V+5F)    only if a coupling matrix is set: scratch for A*u_n and A*R of the current stage
//     then, only with Kreiss-Oliger dissipation (ko_sigma > 0): U2, U3, U4 (F each: u-parts of the stage
//                       vectors) and K4 (V: the slope k_4), see stage_ko.cu
// The u-parts of the stage vectors and the slopes k_1..k_4 are never materialised (S26): for
// d_t u = rho the slope k_{s,u} IS Y_{s,rho}, so Y_{s+1,u} = u_n + a_s dt Y_{s,rho} is rebuilt where it is
// needed, and k_{s,rho} = (Y_{s+1,rho} - rho_n)/(a_s dt). After a level-step the child level reads
// (u_n, rho_n, Y2r, Y3r, Y4r) of its parent for the dense-output ghost fill ("Store k").
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

constexpr int XOFF = 8;        // doubles of left padding in x (>= max ghost width; a multiple of 4: 32-byte sectors)
constexpr int MAX_GHOST = 5;
constexpr int MIN_GHOST = 2;   // stencil radius of the 4th-order Laplacian; restriction reads 2 layers
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
  long long vol;   // doubles per array = px * py * pz (multiple of 32)
};

SC_HD inline long long cell_offset(const BoxView& b, int i, int j, int k) {
  return (long long)(XOFF + i) + (long long)b.px * ((long long)(j + b.g) + (long long)b.py * (k + b.g));
}

// Prolongation / restriction stencils (S3, S4 and their NEXT-3 variants S30, S31), built on the host by
// make_interp_ops() from the Lagrange formula. Prolongation: parent offsets pmin .. pmin + np - 1 around the parent
// index I >> 1, weights w[parity of I][.]; restriction: fine offsets rmin .. rmin + nr - 1 around 2J.
struct InterpOps {
  int np = 5, pmin = -2, nr = 6, rmin = -2;
  double w[2][10];
  double r[10];
  int reach() const { return -pmin > pmin + np - 1 ? -pmin : pmin + np - 1; }
  bool is_default() const { return np == 5 && nr == 6; }
};
InterpOps make_interp_ops(int interp, int vertex);

struct BoxInfo {
  BoxView v;
  int level;
  int index_in_level;
  int parent;                       // global box index on level-1, or -1
  unsigned long long arena_offset;  // bytes, start of array 0
  int narrays;                      // arrays this box owns
};

struct Layout {
  int nlevels = 0, g = 3, F = 1, V = 2;
  int domain[3] = {0, 0, 0};
  double xlo[3] = {0, 0, 0}, xhi[3] = {0, 0, 0};
  std::vector<BoxInfo> boxes;
  std::vector<std::vector<int>> level_boxes;
  unsigned long long coupling_offset = 0;   // bytes into the arena (F*F doubles) if has_coupling
  unsigned long long arena_bytes = 0;
  bool has_coupling = false;
  double ko_sigma = 0.0;                    // > 0: Kreiss-Oliger dissipation, general stage-by-stage path
  int fd_order = 4;                         // 4 (S2) or 8: centred differences of the RHS
  int ko_order = 5;                         // 5: delta^6, 9: delta^10 (eq 36)
  int integrator = 4;                       // 4 | 3 | 2 (S28)
  int outer_bc = 0;                         // 0 periodic | 1 radiative (S29)
  int interp = 0, vertex = 0;               // S30, S31
  InterpOps ops;                            // prolongation / restriction stencils and weights in use
  // the general stage-by-stage path (stage_gen.cu): whole stage vectors stored, one launch per stage
  bool general() const { return ko_sigma > 0.0 || integrator != 4 || outer_bc != 0; }
  double dx(int level, int a) const { return (xhi[a] - xlo[a]) / ((double)domain[a] * (double)(1u << level)); }
  // first array index of each role
  int a_state(int slot) const { return slot * V; }
  int a_Y2r() const { return 2 * V; }
  int a_Y3r() const { return 2 * V + F; }
  int a_Y4r() const { return 2 * V + 2 * F; }
  int a_scratch() const { return 2 * V + 3 * F; }
  // dissipation path only: u-parts of Y_2..Y_4 (the rho-parts are Y2r..Y4r) and the slope k_4 (u, then rho)
  int a_extra() const { return 2 * V + 3 * F + (has_coupling ? 2 * F : 0); }
  int a_U(int s) const { return a_extra() + (s - 2) * F; }   // s = 2, 3, 4
  int a_R(int s) const { return 2 * V + (s - 2) * F; }       // = Y2r, Y3r, Y4r
  int a_K4() const { return a_extra() + 3 * F; }             // V arrays
};

// Validate a description and compute the layout. Host only, no CUDA calls.
// Returns SC_OK or an SC_ERR_* code; err receives a message.
int build_layout(const sc_hierarchy_desc* d, Layout* out, std::string* err);

void set_error(const std::string& msg);

}  // namespace sc

#endif  // SC_INTERNAL_H_
