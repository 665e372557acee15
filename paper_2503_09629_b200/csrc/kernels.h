// kernels.h — launch interface between the level scheduler (capi.cu) and the CUDA kernels.
#ifndef SC_KERNELS_H_
#define SC_KERNELS_H_

#include <cuda_runtime.h>

#include "sc_internal.h"

namespace sc {

// ------------------------------------------------------------------------------------------------
// a1 / a2: the four RHS evaluations of one RK4 level-step (eqs 1-9) fused with
// the stage combines, for  d_t u = rho,  d_t rho = Lap_h u + A u =: L u. Written on
// the stored quantities (u_n, rho_n, Y2r, Y3r, Y4r) — see sc_internal.h and DESIGN.md S26. Because
// k_{s,u} = Y_{s,rho}, the stage vectors Y_3 and Y_4 depend on Y_2 only through arrays the FIRST kernel
// already produced, so one level-step is TWO launches:
//   STAGE_12  (k_1, k_2):  Y2r = rho_n + dt/2 L u_n                       (k_{1,rho} = L u_n, eq 7)
//                          Y3r = rho_n + dt/2 L (u_n + dt/2 rho_n)        (k_{2,rho} = L Y_{2,u}, eq 8)
//   STAGE_34  (k_3, k_4):  Y4r = rho_n + dt   L (u_n + dt/2 Y2r)          (k_{3,rho} = L Y_{3,u}, eq 9)
//                          k4r   = L (u_n + dt Y3r)                       (k_{4,rho} = L Y_{4,u})
//                          u_new   = u_n + dt/6 (rho_n + 2 Y2r + 2 Y3r + Y4r)                       (eq 5)
//                          rho_new = rho_n + (Y2r-rho_n)/3 + 2 (Y3r-rho_n)/3 + (Y4r-rho_n)/3 + dt/6 k4r
// Inputs marked (h) are read with 2 ghost layers; everything is written on the interior only. Y4r is
// stored only when a child level needs it for its dense-output ghost fill (write_Y4r).
// ------------------------------------------------------------------------------------------------
enum { STAGE_12 = 0, STAGE_34 = 1 };

struct StageArgs {
  BoxView b;
  int F;
  int mode;
  int fd_order;        // 4: 13-point Laplacian (S2); 8: 25-point, direct-load kernel only
  int write_Y4r;
  const double* yn;    // (h) state slot of y_n: u_f at f*vol (h), rho_f at (F+f)*vol ((h) in STAGE_12)
  double* Y2r;         // F arrays: written by STAGE_12, read (h) by STAGE_34
  double* Y3r;         // F arrays: written by STAGE_12, read (h) by STAGE_34
  double* Y4r;         // F arrays: written by STAGE_34 if write_Y4r
  double* ynew;        // state slot of y_{n+1} (STAGE_34)
  double dt;
  double inv12dx2[3];  // 1 / (12 dx_a^2)
  const double* A;     // device F*F row-major coupling, or null
  const double* A_host; // the same matrix in host memory (kernel-parameter copy for couple_matvec)
  double* S;           // coupled systems: 2F scratch arrays for the coupling terms (A W) of the two operands
  // TMA path: tensor map of the box (all arrays as the 4th dimension) and the array indices of the roles
  const void* tmap;    // host pointer to the box's CUtensorMap, or null -> direct-load kernel
  int tile_variant;    // halo tile the map was built for (0: 32 x 16, 1: 64 x 7), decided ONCE at sc_create_hierarchy on the
                       // device the hierarchy lives on: the launch must use this, never re-derive it from the current device
  int a_yn, a_Y2r, a_Y3r;
};
int launch_stage(const StageArgs& a, cudaStream_t st);  // returns the number of kernels launched
int stage_tile_variant(const BoxView& b, int F);          // which halo tile the tuned stage kernels use on this box (tensor map kind 0 / 8)
// 128-byte CUtensorMaps of a box: dims (px, py, pz, narrays), fp64, no swizzle; kind 0: box = the stage
// kernels' halo tile, kind 1: box = the restriction kernel's pair of fine planes, kinds 2..4: the ghost
// fill's parent footprint of a tile of an x- / y- / z-slab, kind 5: the dissipative stage kernel's halo-3 tile, kinds 6, 7: the
// wide-stencil stage kernel's halo-4 / halo-5 tiles, kind 8: the stage kernels' 64 x 7 tile. Returns false (and leaves
// the direct-load kernels in charge) when the driver entry point is unavailable or a TMA limit is violated.
bool make_box_tensor_map(const BoxView& b, int narrays, void* base, int kind, void* out_map128);

// ------------------------------------------------------------------------------------------------
// The GENERAL stage-by-stage formulation: one launch per RK stage, the stage
// vectors stored whole. Used with Kreiss-Oliger dissipation (any order), with the RK3 / RK2 integrators and with the
// radiative outer boundary — everything the two-launch formulation above does not cover (stage_gen.cu; the tuned
// stage_ko_tma.cu takes the RK4 / 4th-order / delta^6 / periodic case). All pointers are field-0 arrays of one box;
// field f is f arrays further.
//   k = M Y_s,   M (U, R) = (R + Q U,  Lap_h U + A U + Q R)      (on level-0 boundary points: the radiative operator)
//   RK4 (eqs 1-9):   s = 1..3: Y_{s+1} = y_n + a_s dt k;   s = 4: y_{n+1} = y_n + dt/6 (k_1 + 2 k_2 + 2 k_3 + k), K <- k
//   RK3 (S28):       s = 1: Y_2 = y_n + dt/2 k;  s = 2: Y_3 = y_n - dt k_1 + 2 dt k;  s = 3: y_{n+1} = y_n + dt/6 (k_1 + 4 k_2 + k),
//                    K3 <- k;  s = 4 (levels with a child): K <- k = M y_{n+1}, nothing else is written
//   RK2 (S28):       s = 1: Y_2 = y_n + dt/2 k;  s = 2: y_{n+1} = y_n + dt k, K <- k
// Earlier slopes are not stored: they are recovered from the stage vectors at the cell (k_1 = (Y_2 - y_n) / (dt/2), ...).
// ------------------------------------------------------------------------------------------------
struct StageKOArgs {
  BoxView b;
  int F;
  int stage;             // 1..S (RK3 on a level with a child: also 4)
  int integrator;        // 4 | 3 | 2
  int fd_order;          // 4 | 8
  int ko_order;          // 0: no dissipation (ko_sigma = 0); 5: delta^6; 9: delta^10
  int tile_variant;      // as StageArgs::tile_variant (tensor map kind 5 / 9), fixed at creation
  const double* Yu;      // u- and rho-part of the stage vector Y_s (stage 1: the state y_n), read with ghost layers
  const double* Yr;
  const double* yn_u;    // y_n, centre only
  const double* yn_r;
  double* outU;          // stage < S: Y_{s+1};  stage S: y_{n+1}
  double* outR;
  const double* U2;      // final stage, centre only: Y_2, Y_3 (the last stage vector is Yu, Yr)
  const double* U3;
  const double* R2;
  const double* R3;
  double* K4u;           // slope kept for the child's dense output (see above), or null where no child reads it
  double* K4r;
  double* K3u;           // RK3, stage 3: k_3, or null
  double* K3r;
  double dt;
  double inv12dx2[3];    // 1 / (12 dx_a^2)
  double ko[3];          // sigma / (64 dx_a)  (ko_order 9: sigma / (1024 dx_a))
  const double* A;       // device F*F coupling, or null
  const void* tmap;      // host pointer to the box's stage_ko CUtensorMap (kind 5), or null -> direct-load kernel
  int a_Yu, a_Yr;        // array indices of Yu, Yr (field 0) in the tensor map
  // radiative outer boundary (S29), level 0 only: cells within `rad_nb` of a face are boundary points
  int rad_nb;            // 0: none
  int zone_only;         // 1: redo the boundary points only (after the tuned kernel took the whole box)
  double x0[3], dx[3];   // position of cell 0 (centre or grid point) and spacing
};
void launch_stage_ko(const StageKOArgs& a, cudaStream_t st);

// ------------------------------------------------------------------------------------------------
// a3: refinement-boundary ghost fill. One launch fills, for every ghost cell of a level >= 1 box, the shells
// of up to GF_MAX_PROB independent PROBLEMS; problem p writes, for every output o,
//     child array dst_arr[o] (ghost cell) = P[ sum_s coef[o][s] * parent array src_arr[s] ]
// with P = 5x5x5 tensor quartic Lagrange (S3). The dense-output time polynomial (eqs 10-18) is folded into
// coef by the scheduler, which asks for all ghost shells one child level-step needs in ONE launch: the
// (5 sources -> 4 outputs) dense-output problem and, when the step ends at the parent's t_{n+1}, the
// (2 -> 2) same-time prolongation of the parent's new state. Arrays are named by their index inside the
// box (sc_internal.h); field f of every source / output is f arrays further.
// ------------------------------------------------------------------------------------------------
constexpr int GF_MAX_SRC = 5, GF_MAX_OUT = 4, GF_MAX_PROB = 3;

struct GhostTile {   // one work tile of a ghost slab; everything the kernel needs is precomputed on the host
  int axis;                // the slab's thin axis: 0 = x-slab, 1 = y-slab, 2 = z-slab
  int nt;                  // thin cells (= ghost width)
  int par;                 // ghost width 3: parity of the first thin cell's level-global index; else -1
  int vA0, vA1, vB0, vB1;  // valid tile-local fine range along the transverse axes A (more contiguous), B
  int cx, cy, cz;          // start of the parent footprint in the parent's tensor map (cx even)
  int xoff;                // x-slabs: position of footprint cell 0 inside the loaded 8-wide row
  int sector;              // x-slabs: 0 = scalar stores, 1 / 2 = whole-sector stores on the low / high side
  int IT0;                 // level-global index of the first thin cell (weight table for widths != 3)
  int pad;
  long long cell0;         // offset inside a child array of tile-local (a = 0, b = 0, thin cell 0)
};
static_assert(sizeof(GhostTile) == 64, "the kernel fetches descriptors as four 16-byte copies");

struct GhostProblem {
  int nsrc, nout;
  int src_arr[GF_MAX_SRC];
  int dst_arr[GF_MAX_OUT];
  double coef[GF_MAX_OUT][GF_MAX_SRC];
};

struct GhostArgs {
  BoxView child, parent;
  int F;
  int nprob;
  int np, pmin;               // prolongation stencil: parent offsets pmin .. pmin + np - 1 (default 5, -2: S3)
  double w[2][10];            // weights by parity of the fine index (direct kernel; the tuned kernel has S3's built in)
  const double* parent_base;  // array 0 of the parent box
  double* child_base;         // array 0 of the child box
  GhostProblem prob[GF_MAX_PROB];
  const GhostTile* tiles;     // device; tile list of the child box (built once per box)
  int ntiles;
  const void* tmaps;          // host pointer to the parent's three footprint CUtensorMaps (thin axis x, y, z;
                              // 128 bytes each, contiguous), or null -> direct-load kernel
};
// `siblings`: the other boxes of the child's level; a tile whose cells ALL lie in the interior of one sibling is
// left out (the same-level exchange a7 overwrites every one of them right after the fill).
void build_ghost_tiles(const BoxView& child, const BoxView& parent, std::vector<GhostTile>& tiles,
                       const std::vector<BoxView>* siblings = nullptr);
bool ghost_tma_geometry_ok(const BoxView& child);  // ghost widths the tuned kernel's tiles cover
void launch_ghost_fill(const GhostArgs& a, cudaStream_t st);

// a4: periodic ghost fill of `narrays` consecutive arrays of the level-0 box (reading S9).
void launch_periodic_fill(const BoxView& b, int narrays, double* y, cudaStream_t st);

// a5: restriction child -> parent of V consecutive arrays (reading S4).
struct RestrictArgs {
  BoxView child, parent;
  int V;
  int nr, rmin;          // restriction stencil: fine offsets rmin .. rmin + nr - 1 around 2J (default 6, -2: S4; 1, 0: injection)
  double r[10];
  const double* ychild;  // child state, component 0 (read with 2 ghost layers)
  double* yparent;       // parent state, component 0
  const void* tmap;      // host pointer to the child's kind-1 CUtensorMap, or null -> direct-load kernel
  int a_child;           // array index of ychild in the child's tensor map
};
void launch_restrict(const RestrictArgs& a, cudaStream_t st);

// a7: same-level ghost exchange. Boxes of one level may abut or sit closer
// than a ghost width; every ghost cell of a box that lies in the INTERIOR of a sibling takes the sibling's value
// of the same array, after the refinement-boundary fill wrote its (prolonged) value there. One record per
// ordered pair (dst, src) whose  padded(dst) n interior(src)  is not empty; the region is a box.
struct SiblingPair {
  BoxView dst, src;
  long long dst_off, src_off;  // doubles from the arena base to array 0 of the two boxes
  int lo[3], n[3];             // the region: first cell (level-global index) and extent
};
// copies arrays [first_array, first_array + narrays) of every pair; `maxcells` = largest region
void launch_sibling_copy(const SiblingPair* pairs_dev, int npairs, long long maxcells, double* arena, int first_array,
                         int narrays, cudaStream_t st);

// interior-only <-> padded copies for sc_set_state / sc_read_level (device src/dst, dense [k][j][i])
void launch_pack(const BoxView& b, const double* padded, double* dense, int with_ghosts, cudaStream_t st);
void launch_unpack(const BoxView& b, const double* dense, double* padded, cudaStream_t st);

// measurement: plain streaming kernel, nread arrays in (n doubles apart) summed into nwrite arrays out
void launch_stream_mix(const double* in, double* out, unsigned long long n, int nread, int nwrite, cudaStream_t st);

// debug: max |x| over the interior (NaN if any value is NaN); *out_bits (device) must be zeroed by the caller and
// receives the bit pattern of the result (non-negative doubles order like their bit patterns)
void launch_max_abs(const BoxView& b, const double* padded, unsigned long long* out_bits, cudaStream_t st);

// debug: ghost index map with the same device index arithmetic as the ghost kernels
void launch_ghost_map(const BoxView& child, const BoxView& parent, int* out, cudaStream_t st);
long long ghost_cell_count(const BoxView& b);

}  // namespace sc
#endif
