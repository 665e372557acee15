/* subcycle.h — C ABI of libsubcycle: one Berger–Oliger subcycled RK4 step over a nested-box AMR
 * hierarchy with dense-output ghost fill, hand-written fp64 CUDA for sm_100a (B200).
 *
 * What the calls compute is fixed by the paper (arXiv 2503.09629, "PAPER.md"):
 *   - RK4 stages and update ............................ PAPER.md:54-75   (Sec. II, eqs 1-9)
 *   - dense output b_i(theta) and its derivatives ...... PAPER.md:79-96   (eqs 10-14)
 *   - stage reconstruction at refinement ghosts ........ PAPER.md:98-109  (eqs 15-18)
 *   - the subcycling recursion, steps 1-7 .............. PAPER.md:111-119
 *   - the evolved system  d_t u = rho, d_t rho = Lap u . PAPER.md:222-226 (Sec. IV.A, eqs 39-40)
 * and, where the paper is silent, by the readings S1..S24 listed in DESIGN.md.
 *
 * Conventions (all calls):
 *   - return 0 (SC_OK) on success, a negative SC_ERR_* otherwise; nothing aborts or throws across the
 *     ABI; sc_last_error() returns a thread-local message for the last failing call.
 *   - every pointer says whether it is a HOST or a DEVICE pointer; the library never frees caller memory.
 *   - all index quantities are int32; all field data are IEEE fp64.
 */
#ifndef SUBCYCLE_H_
#define SUBCYCLE_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  SC_OK = 0,
  SC_ERR_INVALID_ARG = -1, /* null pointer, index out of range, non-finite dt, capacity too small */
  SC_ERR_NESTING = -2,     /* box list violates the nesting rules below                           */
  SC_ERR_UNSUPPORTED = -3, /* ref_ratio != 2, ghost outside [2,5], nlevels > SC_MAX_LEVELS, F > 32, bad option */
  SC_ERR_OOM = -4,         /* arena too small / device allocation failed                          */
  SC_ERR_CUDA = -5         /* a CUDA runtime/driver call failed (message has the CUDA error string) */
};

#define SC_MAX_LEVELS 16

/* One box of one refinement level (nested levels, h^(l)/h^(l+1) = 2).
 * lo[] is the index of the box's first interior cell in that level's GLOBAL cell index space
 * [0, domain_cells[a]*2^level) per axis a = (x,y,z); n[] is the number of interior cells.
 * Grids are cell-centred (reading S1): cell i of level l has centre xlo + (i+1/2)*dx_l. */
typedef struct {
  int32_t level;
  int32_t lo[3];
  int32_t n[3];
} sc_box;

/* Hierarchy description (HOST memory, read only during the call).
 * Rules checked by sc_create_hierarchy (violations -> SC_ERR_NESTING unless noted):
 *   - boxes sorted by level; level 0 is exactly one box with lo = 0 and n = domain_cells
 *     (the periodic domain, reading S9); every level 0..nlevels-1 has at least one box;
 *   - every level >= 1 box: lo and n even on every axis (it covers whole parent cells), n >= 8;
 *     it lies inside ONE box of level-1 with at least ceil(ghost/2) + 2 (= 4 at ghost 3; more with the interp_order /
 *     centering options below) parent cells of margin to that box's
 *     interior edge (reading S13: the 5-point prolongation footprint never touches parent ghosts);
 *   - the interiors of the boxes of one level are disjoint. Boxes may abut or sit at any distance: every ghost
 *     cell of a box that lies in the interior of a box of the same level takes that box's value of the same
 *     stage vector (same-level ghost exchange after every fill and stage; a refinement
 *     boundary uses the same ghost zones as an inter-process boundary), so a level cut into abutting boxes
 *     computes what the uncut level computes. A child box must still nest in ONE parent box.
 * The state has nfields second-order fields u_f with first-order partners rho_f = d_t u_f:
 *   component index comp = f        -> u_f
 *                   comp = nfields+f -> rho_f            (V = 2*nfields arrays per box)
 * coupling: HOST pointer to nfields*nfields doubles, row-major A[f][j], or NULL for A = 0:
 *   d_t u_f = rho_f,   d_t rho_f = Lap_h u_f + sum_j A[f][j] u_j       (BASELINE cfg 4)
 * ko_sigma: strength of the Kreiss-Oliger dissipation added to the time derivative of EVERY evolved variable,
 *   d_t y -> RHS + Q y,  Q y = sigma/64 sum_i delta_i^6 y / h_i  (eqs 35-36 with r = 4);
 *   needs ghost >= 3 (ko_order 9: sigma/1024 sum_i delta_i^10 y / h_i, ghost >= 5). With sigma > 0 the step runs the general stage-by-stage kernels (the stage vectors' u parts
 *   are stored: 5 more arrays per field), with sigma = 0 the two-launch formulation of DESIGN.md section 6.
 * fd_order: 8 selects the paper's BBH discretisation, the 9-point second difference
 *   (-1/560, 8/315, -1/5, 8/5, -205/72, ...)/h^2 per axis; needs ghost >= 4 -> SC_ERR_UNSUPPORTED otherwise.
 * ko_order: order of the dissipation operator: 5 -> delta^6 (eq 36 with r = 4; 3 ghost layers), 9 -> delta^10 (eq 36 with
 *   r = 8, "ninth-order"; 5 ghost layers), 0 -> eq 36's rule r = fd_order. (The paper's production runs
 *   pair 8th-order differences with FIFTH-order dissipation: fd_order = 8, ko_order = 5, ghost = 4.)
 * integrator: 0 or 4 -> classical RK4 (eqs 1-9); 3 -> Kutta's RK3 with the slope at the new state completing a third-
 *   order dense output; 2 -> midpoint RK2 (reading S28 gives tableaux, b_i(theta) and the ghost
 *   stage formulas).
 * outer_bc: 0 -> periodic level 0 (S9); 1 -> radiative (Sommerfeld) boundary (reading S29): the
 *   cells of level 0 within `ghost` cells of a domain face are boundary points, every evolved variable obeys
 *   d_t y = -[(x^i/r) d_i y + y/r] there (second-order centred / one-sided differences), at every stage; the ghost
 *   cells of level 0 are then unused. The origin must lie inside the domain, more than ghost * dx_0 from every face
 *   (the boundary zone evaluates 1/r; SC_ERR_INVALID_ARG otherwise).
 * interp_order: 0 -> quartic prolongation, quintic restriction (S3, S4); 1 -> 9-point prolongation and 10-point
 *   restriction, the orders that follow 8th-order differences (reading S30; needs ghost >= 4; nesting margin
 *   ceil(g/2) + 4 parent cells).
 * centering: 0 -> cell-centred grids (S1); 1 -> vertex-centred: grid point i of level l sits at xlo + i dx_l, fine
 *   point 2J coincides with parent point J: restriction is injection, even ghost points copy, odd ghost points take the
 *   6-point (interp_order 1: 10-point) midpoint interpolant (reading S31; nesting margin ceil(g/2) + 3 (5)).
 * Any of ko_sigma > 0, integrator != RK4, outer_bc != 0 selects the general stage-by-stage kernels.
 * arena: optional DEVICE memory of at least sc_arena_bytes() bytes, 256-byte aligned, owned by the
 *   caller, who keeps it alive and does not touch it until sc_destroy; NULL -> the library allocates.
 * cuda_stream: a cudaStream_t (as void*) on which all work of this hierarchy is enqueued (must not be
 *   the legacy default stream: steps are captured into CUDA graphs); NULL -> the library creates and
 *   owns a private non-blocking stream. */
typedef struct {
  int32_t nlevels;
  int32_t nboxes;
  const sc_box* boxes;
  int32_t ref_ratio;       /* must be 2                                      */
  int32_t ghost;           /* ghost width g; 3 in all configurations (stencil radius is 2)  */
  int32_t nfields;         /* F >= 1                                                        */
  int32_t domain_cells[3]; /* level-0 cells per axis                                        */
  double xlo[3], xhi[3];   /* physical extent of the level-0 domain                         */
  const double* coupling;  /* HOST, F*F, or NULL                                            */
  void* arena;             /* DEVICE or NULL                                                */
  uint64_t arena_bytes;
  void* cuda_stream;
  double ko_sigma;         /* Kreiss-Oliger strength sigma >= 0; 0 = none */
  int32_t fd_order;        /* centred differences of the RHS: 0 or 4 -> 4th order (S2); 8 -> 8th order           */
  int32_t ko_order;        /* 0 (follow fd_order), 5 or 9                                                          */
  int32_t integrator;      /* 0 / 4: RK4; 3: RK3; 2: RK2                                                           */
  int32_t outer_bc;        /* 0: periodic; 1: radiative                                                            */
  int32_t interp_order;    /* 0: quartic / quintic; 1: 9-point / 10-point                                          */
  int32_t centering;       /* 0: cell-centred; 1: vertex-centred with injection                                    */
} sc_hierarchy_desc;

typedef struct sc_hierarchy sc_hierarchy; /* opaque; created by sc_create_hierarchy, freed by sc_destroy */

/* Bytes of device memory a hierarchy with this description needs (0 on an invalid description;
 * sc_last_error says why). Host-only computation: works without a GPU. */
uint64_t sc_arena_bytes(const sc_hierarchy_desc* desc);

/* Validate the description, lay the boxes out in device memory, zero all
 * state, build the TMA tensor maps. The time is set to 0. On failure *out is NULL.
 * Fails with SC_ERR_CUDA when no CUDA device is usable: there is no CPU fallback. */
int32_t sc_create_hierarchy(const sc_hierarchy_desc* desc, sc_hierarchy** out);

/* Copy one component of one box into the current state y of that box.
 * src: dense INTERIOR-ONLY array [k][j][i], i (x) fastest, n[0]*n[1]*n[2] doubles; HOST if
 * src_on_device == 0, DEVICE otherwise. box is the box's index within its level (0-based, in the
 * order given at creation). Ghost cells are never supplied: the first stage of every level-step
 * refills them (reading S8). Enqueued on the hierarchy's stream; a host source is consumed before the
 * call returns. A DEVICE source is read by a kernel enqueued on the hierarchy's stream and the call returns
 * without waiting for it: the caller must (i) have made that stream wait for whatever produces src (an event
 * or stream wait; the library knows nothing about the caller's streams) and (ii) keep src alive and unchanged
 * until the hierarchy's stream has passed this point. The Python binding does both for torch tensors. */
int32_t sc_set_state(sc_hierarchy* h, int32_t level, int32_t box, int32_t comp, const double* src,
                     int32_t src_on_device);

/* Advance the whole hierarchy by dt_coarse (steps 1-7).
 * subcycling = 1: level l takes 2^l steps of dt_coarse/2^l; refinement-boundary ghosts of Y_1..Y_4 and
 *   of y_{n+1} come from the parent's dense output (eqs 10-18) prolonged in space (reading S3);
 *   fine-to-coarse restriction (reading S4) after each pair of child steps.
 * subcycling = 0: 2^(nlevels-1) uniform steps of dt_coarse/2^(nlevels-1) on all levels, same-time
 *   spatial prolongation after every stage, restriction once per uniform step (reading S11).
 * Asynchronous: returns once the work is enqueued on the stream. */
int32_t sc_step(sc_hierarchy* h, double dt_coarse, int32_t subcycling);

/* Copy one component of one box's current state y (interior only, same layout as sc_set_state) to dst
 * (HOST if dst_on_device == 0, else DEVICE). Synchronises the hierarchy's stream before returning. */
int32_t sc_read_level(sc_hierarchy* h, int32_t level, int32_t box, int32_t comp, double* dst,
                      int32_t dst_on_device);

/* Simulation time: the sum of dt_coarse over all sc_step calls. */
double sc_time(const sc_hierarchy* h);

/* Number of kernels the library has launched (or replayed inside CUDA graphs) for this hierarchy. */
uint64_t sc_launch_count(const sc_hierarchy* h);

/* Debug: the refinement-boundary ghost index map of a level >= 1 box, computed on the device with the index
 * arithmetic of the direct-load ghost kernel (parent = I >> 1, parity = I & 1 on level-global indices). The tuned
 * ghost kernel works from tile descriptors built on the host with the same arithmetic; it is held to this map
 * through the element-wise parity of every ghost value. For every ghost cell of the padded box, in canonical order (k, then j, then
 * i over [-g, n+g), skipping the interior), 7 int32: (i, j, k) box-local fine index, (pi, pj, pk)
 * parent-box-local index of the containing parent cell, and parity bits (px | py<<1 | pz<<2) where
 * p = 1 means the fine centre sits at +dx_parent/4 from the parent centre. out: HOST, cap = capacity in
 * int32. Returns the number of ghost cells (>= 0) or an error. */
int64_t sc_debug_ghost_map(sc_hierarchy* h, int32_t level, int32_t box, int32_t* out, uint64_t cap);

/* Debug: copy one component of the current state INCLUDING ghosts, dense [n2+2g][n1+2g][n0+2g], to HOST
 * memory. Synchronises the stream. Ghost values are those of the last stage-5 fill. */
int32_t sc_debug_read_padded(sc_hierarchy* h, int32_t level, int32_t box, int32_t comp, double* dst);

/* Debug: what the library keeps of the last level-step of a box (S26), interior only, HOST dst:
 * slot 1 = y_n (the state before that level-step), any comp; slot 2, 3, 4 = the stage vectors Y_2, Y_3, Y_4
 * (eqs 7-9), rho components only (nfields <= comp < 2*nfields): for d_t u = rho the slope
 * k_{s,u} is Y_{s,rho}, so the u-parts of the stage vectors and the slopes k_1..k_4 are never stored
 * (Y_{s+1,u} = u_n + a_s dt Y_{s,rho};  k_{s,rho} = (Y_{s+1,rho} - rho_n) / (a_s dt)). */
int32_t sc_debug_read_slot(sc_hierarchy* h, int32_t level, int32_t box, int32_t slot, int32_t comp,
                           double* dst);

/* Debug: max |value| over the INTERIOR of one component of the current state of a box, reduced on the device
 * (one 8-byte read-back). *out (HOST) is NaN as soon as one value is NaN, +inf if one is infinite: the check
 * for a run that blew up, without copying the state. Synchronises the stream. */
int32_t sc_debug_max_abs(sc_hierarchy* h, int32_t level, int32_t box, int32_t comp, double* out);

/* Debug: the scheduler's CUDA-graph bookkeeping since creation. A coarse step is captured once per (mode, state-slot
 * phase) and replayed; a step with a different dt_coarse re-records the launch sequence on the host and updates the
 * parameters of the existing executable graph in place, so `instantiations` and `cached` stay bounded by the number of
 * phases however many distinct step sizes a run uses. Out pointers: HOST, may be NULL. */
int32_t sc_debug_graph_stats(const sc_hierarchy* h, uint64_t* captures, uint64_t* instantiations, uint64_t* updates,
                             uint64_t* cached);

/* Measurement: the practical HBM ceiling of this device for a PLAIN streaming kernel with a stage kernel's read / write
 * mix — nread arrays read and nwrite arrays written, `ndoubles` doubles each (grid-stride, 16-byte accesses, no
 * stencil, no shared memory), allocated and freed inside the call. *gbps (HOST) receives the best of 5 timed launches,
 * (nread + nwrite) * 8 * ndoubles bytes / time. Context for the roofline fractions (which stay against the copy peak):
 * what a kernel that only moves the same bytes reaches. Synchronises the stream. 1 <= nread, nwrite <= 8. */
int32_t sc_debug_stream(sc_hierarchy* h, int32_t nread, int32_t nwrite, uint64_t ndoubles, double* gbps);

/* Debug, host only (no GPU needed): the one-dimensional interpolation operators the library uses between levels for
 * the given options (readings S3, S4, S30, S31; 3-D operators are their tensor products). Prolongation: the fine point
 * of parity p (0: at -1/4 parent spacing from parent point 0 on cell-centred grids, ON it on vertex-centred grids;
 * 1: at +1/4, resp. +1/2) is sum_m w_p[m] * parent[pmin + m], m < np. Restriction: parent point I is
 * sum_m r[m] * fine[2 I + rmin + m], m < nr. The library derives them in exact integer arithmetic and rounds once,
 * so each is the correctly rounded value of its rational (tests/golden/interp_weights*.txt). All out pointers HOST;
 * w0, w1, r hold 10 doubles each (entries beyond np / nr are 0). */
int32_t sc_debug_interp_weights(int32_t interp_order, int32_t centering, int32_t* np, int32_t* pmin, double* w0,
                                double* w1, int32_t* nr, int32_t* rmin, double* r);

/* Per-kernel timing for the roofline report. sc_profile(h, 1): from now on sc_step launches its kernels
 * one by one (no graph replay) with a CUDA-event pair around each on the hierarchy's stream;
 * sc_profile(h, 0) stops and discards the records. sc_profile_read sums, over the records since
 * enabling, for kernel kind 0 = rk_stage, 1 = ghost_dense_prolong, 2 = periodic_fill, 3 = restrict:
 * the number of launches, their total device time (ms) and their total ALGORITHMIC bytes (DESIGN.md
 * "Rooflines": what the method must move, not what the kernel happened to move). Out pointers: HOST,
 * may be NULL. Both calls synchronise the stream. */
int32_t sc_profile(sc_hierarchy* h, int32_t enable);
int32_t sc_profile_read(sc_hierarchy* h, int32_t kind, uint64_t* launches, double* ms, double* bytes);

/* The blow-up check of sc_debug_max_abs for callers that must not allocate device memory: max |x[i]| over a dense
 * array, with the same NaN / inf rule (*out is NaN as soon as one value is NaN, else +inf if one is infinite).
 *
 * Why it exists: sc_debug_max_abs works on a hierarchy, and creating one calls cudaMalloc. That is no use to an
 * application that gave all device memory to its own pool at start-up (any further cudaMalloc fails), nor to a time
 * loop that must not take the device-wide synchronisation cudaMalloc / cudaFree imply just to look for a NaN. This
 * call allocates nothing and frees nothing: its working memory (one partial maximum per 8192 inputs and a counter)
 * is a fixed array compiled into the library, about 64 KB, present on every GPU that loads libsubcycle.so until the
 * process exits.
 *
 *   x            DEVICE, n contiguous doubles, read only (any 8-byte aligned address; may be NULL if n == 0)
 *   n            number of doubles, at most SC_NOALLOC_MAX_DOUBLES (2^26, 512 MB of input; a padded 256^3 box is
 *                1.8e7). A larger n is refused with SC_ERR_INVALID_ARG and a message naming the limit: split the
 *                input and take the maximum of the pieces. n == 0 gives 0.0.
 *   out          DEVICE, one double, written by the kernel. The call is asynchronous and does not synchronise:
 *                read *out after the stream has passed this point.
 *   cuda_stream  a cudaStream_t (as void*) of the CURRENT device; NULL is the default stream. x and out must belong
 *                to the current device.
 *
 * Set-up: the first call on each GPU looks up where that GPU keeps the built-in array (cudaGetSymbolAddress, with
 * that GPU current) and remembers it. Make that first call during start-up, outside any stream capture.
 * Shared state: all calls on one GPU use the same array, which still holds the last call's partials; each call clears
 * what it needs at zero itself. Calls that can run on the GPU at the same time (different streams without an event
 * between them) race on the array and return garbage: keep them on one stream or order them.
 * Returns SC_OK, SC_ERR_INVALID_ARG (null pointer, n over the limit) or SC_ERR_CUDA. */
#define SC_NOALLOC_MAX_DOUBLES (1ull << 26)
int32_t sc_max_abs_noalloc(const double* x, uint64_t n, double* out, void* cuda_stream);

/* Free everything the library owns (never the caller's arena). Synchronises the stream. */
int32_t sc_destroy(sc_hierarchy* h);

/* Message of the last failing call on this thread; valid until the next sc_ call on this thread. */
const char* sc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SUBCYCLE_H_ */
