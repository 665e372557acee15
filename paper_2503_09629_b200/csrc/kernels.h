// kernels.h — launch interface between the level scheduler and the CUDA kernels.
#ifndef SC_KERNELS_H_
#define SC_KERNELS_H_

#include <cuda_runtime.h>

#include "sc_internal.h"

namespace sc {

// a1 / a2: k_s = f(Y_s) on the interior fused with the RK4 stage combine.
//   stage 1..3:  k_s = f(Yin);  Yout = yn + cdt * k_s          (cdt = a_s * dt; eqs 1-3, 7-9)
//   stage 4:     k_4 = f(Yin);  Yout = yn + cdt * (k1 + 2 k2 + 2 k3 + k4)   (cdt = dt/6; eqs 4-5)
// f: k_u = rho, k_rho = Lap_h u + A u. All pointers are slot bases (V arrays).
struct RhsArgs {
  BoxView b;
  int F;
  int stage;
  const double* Yin;
  const double* yn;
  double* kout;       // k_s (may be null at stage 4 when no child level needs k_4)
  double* Yout;       // Y_{s+1} or y_{n+1}
  const double* k1;
  const double* k2;
  const double* k3;
  double cdt;
  double inv12dx2[3];
  const double* A;    // device F*F or null
};
void launch_rhs_stage(const RhsArgs& a, cudaStream_t st);

// a3: dense-output + prolongation ghost fill of a level >= 1 box:
//   ghost(dst) = P[ base + sum_j coef[j] * k[j] ]  over the parent's cells, P = 5x5x5 tensor Lagrange.
// coef[j] already contains the parent step h_p (coef = h_p * c_j(stage, theta)); nk = number of leading
// k arrays with a non-zero coefficient pattern (0 = pure prolongation of base).
struct GhostTile {   // a piece of one ghost slab, box-local fine indices
  int lo[3];
  int n[3];
  int axis;          // the slab's thin axis: 0 = x-slab, 1 = y-slab, 2 = z-slab
  int pad;
};

struct GhostArgs {
  BoxView child, parent;
  int V;
  double* dst;          // child slot base
  const double* base;   // parent y_old (subcycled) or the parent's same-stage buffer (uniform)
  const double* k[4];   // parent k_1..k_4 slot bases
  double coef[4];
  int use_k;            // bit j set -> k[j] is read
  const GhostTile* tiles;  // device; tile list of the child box (built once per box)
  int ntiles;
  int s0_doubles, s1_doubles;  // shared-memory staging sizes the tile list needs
};
void build_ghost_tiles(const BoxView& child, std::vector<GhostTile>& tiles, size_t* s0_doubles, size_t* s1_doubles);
void launch_ghost_fill(const GhostArgs& a, cudaStream_t st);

// a4: periodic ghost fill of the level-0 box (reading S9).
void launch_periodic_fill(const BoxView& b, int V, double* y, cudaStream_t st);

// a5: restriction child -> parent (reading S4).
void launch_restrict(const BoxView& child, const BoxView& parent, int V, const double* ychild,
                     double* yparent, cudaStream_t st);

// interior-only <-> padded copies for sc_set_state / sc_read_level (device src/dst, dense [k][j][i])
void launch_pack(const BoxView& b, const double* padded, double* dense, int with_ghosts, cudaStream_t st);
void launch_unpack(const BoxView& b, const double* dense, double* padded, cudaStream_t st);

// debug: ghost index map with the same device index arithmetic as the ghost kernel
void launch_ghost_map(const BoxView& child, const BoxView& parent, int* out, cudaStream_t st);
long long ghost_cell_count(const BoxView& b);

}  // namespace sc
#endif
