// capi.cu — the C ABI of libsubcycle (include/subcycle.h) and the level scheduler:
// the Berger–Oliger recursion of PAPER.md:111-119 (steps 1-7) unrolled on the host into a fixed sequence
// of kernel launches on one CUDA stream, captured once per (mode, buffer phase) into a CUDA graph and replayed
// (another dt_coarse re-records the sequence and updates the executable graph's parameters in place). No host
// synchronisation inside a step.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <algorithm>
#include <cstring>
#include <map>
#include <string>
#include <vector>

#include "kernels.h"
#include "sc_internal.h"

namespace sc {
const std::string& last_error();
void select_kernels(int mode);
}  // namespace sc

using namespace sc;

// One executable graph per (mode, state-slot phase). The step size is NOT part of the key: a step with another
// dt_coarse re-records the same launch sequence (host work only) and updates the executable graph's kernel
// parameters in place (cudaGraphExecUpdate), so an adaptive-dt caller neither instantiates nor leaks a graph per step.
struct GraphKey {
  int sub;
  uint32_t phase;
  bool operator<(const GraphKey& o) const {
    if (sub != o.sub) return sub < o.sub;
    return phase < o.phase;
  }
};
struct GraphEntry {
  cudaGraphExec_t exec = nullptr;
  uint64_t dt_bits = 0;  // the step size the executable graph's parameters currently hold
  uint64_t launches = 0;
  std::vector<int> cur_after;
};
constexpr size_t kMaxGraphs = 64;  // far above the phases a run visits (2 per mode); beyond it the cache is flushed

struct sc_hierarchy {
  Layout L;
  char* arena = nullptr;
  bool own_arena = false;
  cudaStream_t stream = nullptr;
  bool own_stream = false;
  // second stream of the level scheduler: a level's theta = 1/2 ghost fill runs beside its children's sub-steps
  cudaStream_t side = nullptr;
  std::vector<cudaEvent_t> ev_fork, ev_join;  // per level
  int overlap_mode = -1;                      // SC_OVERLAP: 0 / 1 force the side stream off / on, default by level size
  double* staging = nullptr;      // device, largest padded dense box
  size_t staging_bytes = 0;
  std::vector<double> coupling_host;  // F*F, host copy of the coupling matrix
  std::vector<int> cur;           // per level: state slot (0 or 1) that holds the current state y
  bool l0_ghosts_valid = false;   // level 0: ghosts of y hold the periodic copies (no set_state since)
  double time = 0.0;
  uint64_t launches = 0;
  bool use_graph = true;
  bool debug_sync = false;
  uint64_t debug_seq = 0;
  int debug_kind = 0;
  std::string debug_fail;
  std::map<GraphKey, GraphEntry> graphs;
  uint64_t n_captures = 0, n_instantiations = 0, n_updates = 0;  // sc_debug_graph_stats
  struct BoxTiles { GhostTile* dev = nullptr; int n = 0; };
  std::vector<BoxTiles> tiles;    // per box (levels >= 1): ghost-shell tile list on the device
  struct alignas(64) TMap { unsigned char bytes[128]; };
  std::vector<TMap> tmaps;        // per box: CUtensorMap over all arrays of the box (stage-kernel tile)
  std::vector<TMap> rmaps;        // per box: same tensor, box = the restriction kernel's fine-plane pair
  std::vector<char> tmap_ok;
  std::vector<char> tile_variant; // per box: stage tile (stage_tile_variant) chosen at creation; maps and launches both use it
  struct GMaps { TMap m[3]; };
  std::vector<GMaps> gmaps;       // per box: ghost-fill footprint maps of the box as PARENT (thin axis x, y, z)
  std::vector<char> gmap_ok;
  std::vector<TMap> kmaps;        // per box: halo-3 tile of the dissipative stage kernel (ko_sigma > 0)
  std::vector<char> kmap_ok;
  struct LevelSiblings { SiblingPair* dev = nullptr; int n = 0; long long maxcells = 0; double cells = 0.0; };
  std::vector<LevelSiblings> sib; // per level: ordered pairs of boxes that exchange ghosts (kernels.h a7)
  // per-launch CUDA-event timing (sc_profile): eager launches, one event pair per kernel
  bool profiling = false;
  struct ProfRec { int kind; double bytes; cudaEvent_t e0, e1; };
  std::vector<ProfRec> prof;

  double* arr(int box, int array) const {
    const BoxInfo& b = L.boxes[box];
    return reinterpret_cast<double*>(arena + b.arena_offset) + (long long)array * b.v.vol;
  }
  const double* coupling() const {
    return L.has_coupling ? reinterpret_cast<const double*>(arena + L.coupling_offset) : nullptr;
  }
};

namespace {

#define SC_CUDA(call)                                                                    \
  do {                                                                                   \
    cudaError_t e_ = (call);                                                             \
    if (e_ != cudaSuccess) {                                                             \
      set_error(std::string(#call) + ": " + cudaGetErrorString(e_));                     \
      return SC_ERR_CUDA;                                                                \
    }                                                                                    \
  } while (0)

// Folded dense-output coefficients: the value of RK stage `stage` of a child step that starts at parent
// progress theta is  y_old^p + h_p * sum_j c_j k_j^p  with, from eqs (10)-(18) and child
// step h = r h_p, r = 1/2:
//   stage 1, 5:  c = b(theta)                               (eq 15 / eq 10; stage 5 gets theta + 1/2)
//   stage 2:     c = b + (r/2) b'                           (eq 16)
//   stage 3:     c = b + (r/2) b' + (r^2/4) b'' + (r^3/16)(b''' - phi)   (eq 17)
//   stage 4:     c = b + r b' + (r^2/2) b'' + (r^3/8)(b''' + phi)        (eq 18)
// where b', b'', b''' are theta-derivatives of eqs (11)-(13) (eq 14 supplies the powers of h_p) and
// phi = (0, -4, 4, 0) encodes f_y y'' = 4 (k_3 - k_2) / h_p^2 (parent step, reading S5).
void dense_coeffs(int stage, double th, double c[4]) {
  const double r = 0.5;
  const double b0[4] = {th - 1.5 * th * th + (2.0 / 3.0) * th * th * th, th * th - (2.0 / 3.0) * th * th * th,
                        th * th - (2.0 / 3.0) * th * th * th, -0.5 * th * th + (2.0 / 3.0) * th * th * th};
  const double b1[4] = {1.0 - 3.0 * th + 2.0 * th * th, 2.0 * th - 2.0 * th * th, 2.0 * th - 2.0 * th * th,
                        -th + 2.0 * th * th};
  const double b2[4] = {-3.0 + 4.0 * th, 2.0 - 4.0 * th, 2.0 - 4.0 * th, -1.0 + 4.0 * th};
  const double b3[4] = {4.0, -4.0, -4.0, 4.0};
  const double phi[4] = {0.0, -4.0, 4.0, 0.0};
  for (int j = 0; j < 4; ++j) {
    switch (stage) {
      case 2: c[j] = b0[j] + 0.5 * r * b1[j]; break;
      case 3: c[j] = b0[j] + 0.5 * r * b1[j] + 0.25 * r * r * b2[j] + (r * r * r / 16.0) * (b3[j] - phi[j]); break;
      case 4: c[j] = b0[j] + r * b1[j] + 0.5 * r * r * b2[j] + (r * r * r / 8.0) * (b3[j] + phi[j]); break;
      default: c[j] = b0[j]; break;
    }
  }
}

// The same for the RK3 / RK2 integrators (reading S28); value = y_old^p + h_p * sum_j c_j k_j^p.
//   RK3 (k_4 = f(y_{n+1}) is the fourth slope): b = (th - 3/2 th^2 + 2/3 th^3, 2 th^2 - 4/3 th^3, 1/2 th^2 - 1/3 th^3, th^3 - th^2)
//     stage 2: c = b + (r/2) b';   stage 3: c = b + r b' + r^2 b'' + (r^3/4)(b(3) - phi), b(3) = third theta-derivative,  phi = (0, 0, 2, -2)
//     (Y_3 = y + h y' + h^2 y'' + h^3/4 (y(3) - f_y y''),  f_y y'' = 2 (k_3 - k_4) / h_p^2)
//   RK2: b = (th - th^2, th^2);  stage 2: c = b + (r/2) b'
void dense_coeffs_rk(int integrator, int stage, double th, double c[4]) {
  if (integrator == 4) { dense_coeffs(stage, th, c); return; }
  const double r = 0.5;
  if (integrator == 3) {
    const double b0[4] = {th - 1.5 * th * th + (2.0 / 3.0) * th * th * th, 2.0 * th * th - (4.0 / 3.0) * th * th * th,
                          0.5 * th * th - (1.0 / 3.0) * th * th * th, th * th * th - th * th};
    const double b1[4] = {1.0 - 3.0 * th + 2.0 * th * th, 4.0 * th - 4.0 * th * th, th - th * th, 3.0 * th * th - 2.0 * th};
    const double b2[4] = {-3.0 + 4.0 * th, 4.0 - 8.0 * th, 1.0 - 2.0 * th, 6.0 * th - 2.0};
    const double b3[4] = {4.0, -8.0, -2.0, 6.0};
    const double phi[4] = {0.0, 0.0, 2.0, -2.0};
    for (int j = 0; j < 4; ++j) {
      if (stage == 2) c[j] = b0[j] + 0.5 * r * b1[j];
      else if (stage == 3) c[j] = b0[j] + r * b1[j] + r * r * b2[j] + (r * r * r / 4.0) * (b3[j] - phi[j]);
      else c[j] = b0[j];
    }
    return;
  }
  const double b0[2] = {th - th * th, th * th}, b1[2] = {1.0 - 2.0 * th, 2.0 * th};
  c[2] = c[3] = 0.0;
  for (int j = 0; j < 2; ++j) c[j] = stage == 2 ? b0[j] + 0.5 * r * b1[j] : b0[j];
}

// ---- launch recording -----------------------------------------------------------------------
struct Seq {
  sc_hierarchy* h;
  std::vector<int> cur;  // working copy of the state-slot phases
  bool l0_valid;         // working copy of l0_ghosts_valid
  uint64_t n = 0;
  bool sub = true;       // subcycled mode (parents keep k_4 for their children)
  bool capturing = false;       // the launches are being captured into a CUDA graph (fork / join allowed)
  cudaError_t err = cudaSuccess;  // first failing fork / join call of the recording (reported by sc_step)
  std::vector<char> prefilled;  // per level: the next level-step's refinement ghosts are already written
};

enum { KIND_STAGE = 0, KIND_GHOST = 1, KIND_PERIODIC = 2, KIND_RESTRICT = 3, NKIND = 4 };

// Algorithmic bytes per launch: every array a kernel must read once and every
// array it must write once, in the formulation of sc_internal.h.
double cells(const BoxView& v) { return (double)v.n[0] * v.n[1] * v.n[2]; }
double shell_cells(const BoxView& v) {
  return (double)(v.n[0] + 2 * v.g) * (v.n[1] + 2 * v.g) * (v.n[2] + 2 * v.g) - cells(v);
}
double footprint_cells(const BoxView& v, int reach = 2) {  // parent cells a ghost fill of this box reads
  // ghost cells sit in parent cells up to gc = ceil(g/2) beyond the child's coverage [0, nc); the interpolation
  // stencil adds `reach` more on every side (2 for S3) and reaches as far into the coverage
  const int gc = (v.g + 1) / 2;
  double outer = 1.0, inner = 1.0;
  for (int a = 0; a < 3; ++a) {
    const int nc = v.n[a] / 2;
    outer *= nc + 2 * gc + 2 * reach;
    inner *= nc > 2 * reach ? nc - 2 * reach : 0;
  }
  return outer - inner;
}
double stage_bytes(const BoxView& v, int F, int mode, int write_Y4r) {
  // STAGE_12: read u_n, rho_n; write Y2r, Y3r.  STAGE_34: read u_n, rho_n, Y2r, Y3r; write u_new, rho_new [, Y4r].
  const double per = mode == STAGE_12 ? 4.0 : (write_Y4r ? 7.0 : 6.0);
  return 8.0 * per * F * cells(v);
}

void prof_begin(sc_hierarchy* h, int kind, double bytes) {
  h->debug_kind = kind;
  if (!h->profiling) return;
  sc_hierarchy::ProfRec r{kind, bytes, nullptr, nullptr};
  cudaEventCreate(&r.e0);
  cudaEventCreate(&r.e1);
  cudaEventRecord(r.e0, h->stream);
  h->prof.push_back(r);
}
void prof_end(sc_hierarchy* h) {
  if (h->debug_sync) {  // SC_DEBUG_SYNC=1 (with SC_GRAPH=0): name the first failing launch
    const cudaError_t e = cudaStreamSynchronize(h->stream);
    if (e != cudaSuccess && h->debug_fail.empty()) {
      h->debug_fail = "launch #" + std::to_string(h->debug_seq) + " (kind " + std::to_string(h->debug_kind) + ") failed: " + cudaGetErrorString(e);
      fprintf(stderr, "libsubcycle: %s\n", h->debug_fail.c_str());
    }
    ++h->debug_seq;
  }
  if (!h->profiling) return;
  cudaEventRecord(h->prof.back().e1, h->stream);
}

// ---- per (level, kernel): a loop over the boxes of the level, ONE LAUNCH PER BOX ---------------------------
void stage_level(Seq& q, int level, int mode, double dt) {
  sc_hierarchy* h = q.h;
  const Layout& L = h->L;
  const int yn = q.cur[level], ynew = 1 - yn;
  for (int ib : L.level_boxes[level]) {
    StageArgs a{};
    a.b = L.boxes[ib].v;
    a.F = L.F;
    a.mode = mode;
    a.fd_order = L.fd_order;
    // the slope k_4 (= Y4r) is kept only where a child level reads it for its dense-output ghosts
    a.write_Y4r = (q.sub && level + 1 < L.nlevels) ? 1 : 0;
    a.a_yn = L.a_state(yn);
    a.a_Y2r = L.a_Y2r();
    a.a_Y3r = L.a_Y3r();
    a.yn = h->arr(ib, a.a_yn);
    a.Y2r = h->arr(ib, L.a_Y2r());
    a.Y3r = h->arr(ib, L.a_Y3r());
    a.Y4r = h->arr(ib, L.a_Y4r());
    a.ynew = h->arr(ib, L.a_state(ynew));
    a.dt = dt;
    for (int d = 0; d < 3; ++d) {
      const double dx = L.dx(level, d);
      a.inv12dx2[d] = 1.0 / (12.0 * dx * dx);
    }
    a.A = h->coupling();
    a.A_host = a.A ? h->coupling_host.data() : nullptr;
    a.S = a.A ? h->arr(ib, L.a_scratch()) : nullptr;
    a.tmap = h->tmap_ok[ib] ? h->tmaps[ib].bytes : nullptr;
    a.tile_variant = h->tile_variant[ib];
    prof_begin(h, KIND_STAGE, stage_bytes(a.b, L.F, mode, a.write_Y4r));
    q.n += launch_stage(a, h->stream);
    prof_end(h);
  }
}

void periodic_level0(Seq& q, int first_array, int narrays) {
  sc_hierarchy* h = q.h;
  const int ib = h->L.level_boxes[0][0];
  const BoxView& v = h->L.boxes[ib].v;
  prof_begin(h, KIND_PERIODIC, 16.0 * narrays * shell_cells(v));
  launch_periodic_fill(v, narrays, h->arr(ib, first_array), h->stream);
  prof_end(h);
  ++q.n;
}

// Same-level ghost exchange of arrays [first_array, first_array + narrays) between the boxes of `level`
// (kernels.h a7). Called after every refinement-boundary fill and after every kernel that produced a
// stage vector, for exactly the arrays written: a ghost cell inside a sibling's interior ends up with the
// sibling's value of the same stage vector, as on an uncut level. No launch when no two boxes are in reach.
void sibling_level(Seq& q, int level, int first_array, int narrays) {
  sc_hierarchy* h = q.h;
  const sc_hierarchy::LevelSiblings& s = h->sib[level];
  if (s.n == 0) return;
  prof_begin(h, KIND_PERIODIC, 16.0 * narrays * s.cells);
  launch_sibling_copy(s.dev, s.n, s.maxcells, reinterpret_cast<double*>(h->arena), first_array, narrays, h->stream);
  prof_end(h);
  ++q.n;
}

void ghost_launch(Seq& q, int ib, GhostArgs& a) {
  sc_hierarchy* h = q.h;
  const BoxInfo& b = h->L.boxes[ib];
  a.child = b.v;
  a.parent = h->L.boxes[b.parent].v;
  a.F = h->L.F;
  a.parent_base = h->arr(b.parent, 0);
  a.child_base = h->arr(ib, 0);
  a.tiles = h->tiles[ib].dev;
  a.ntiles = h->tiles[ib].n;
  a.tmaps = h->gmap_ok[b.parent] ? h->gmaps[b.parent].m[0].bytes : nullptr;
  const InterpOps& P = h->L.ops;
  a.np = P.np;
  a.pmin = P.pmin;
  for (int m = 0; m < 10; ++m) { a.w[0][m] = P.w[0][m]; a.w[1][m] = P.w[1][m]; }
  double bytes = 0.0;
  for (int p = 0; p < a.nprob; ++p) {
    int nreal = 0;  // sources padded for the tuned kernel's shape (coefficient column all zero) are not algorithmic traffic
    for (int sidx = 0; sidx < a.prob[p].nsrc; ++sidx) {
      bool used = false;
      for (int o = 0; o < a.prob[p].nout; ++o) used = used || a.prob[p].coef[o][sidx] != 0.0;
      nreal += used ? 1 : 0;
    }
    bytes += 8.0 * h->L.F * (nreal * footprint_cells(b.v, P.reach()) + a.prob[p].nout * shell_cells(b.v));
  }
  prof_begin(h, KIND_GHOST, bytes);
  launch_ghost_fill(a, h->stream);
  prof_end(h);
  ++q.n;
}

// Subcycled mode: ALL refinement-boundary ghosts one level-step of `level` (>= 1) needs, in one launch per
// box, from the parent's stored (u_n, rho_n, Y2r, Y3r, Y4r) =: (u^p, K_1..K_4), K_j = k_{j,u}^p
// (steps 2-6). With c^(s) = dense_coeffs(s, theta), parent step h_p, child step dt = h_p/2,
// a = (1/2, 1/2, 1):
//   shell of u_n    <- P[ u^p + h_p sum_j c^(1)_j K_j ]                               ghost of Y_1 (eq 15)
//   shell of rho_n  <- P[ sum_j (c^(2)_j - c^(1)_j) / (a_1/2) K_j ] =: D_1,   u_n + a_1 dt D_1 = ghost of Y_{2,u} (eq 16)
//   shell of Y2r    <- D_2 likewise from c^(3)                                        ghost of Y_{3,u} (eq 17)
//   shell of Y3r    <- D_3 likewise from c^(4)                                        ghost of Y_{4,u} (eq 18)
// (the stage kernels rebuild Y_{s+1,u} = u_n + a_s dt Y_{s,rho} on ghost cells exactly as on interior
// cells; only ghosts of u are ever read, S25). If theta = 1/2 the step ends at the parent's t_{n+1}: eq (10)
// at theta + 1/2 = 1 is the parent's own RK4 update, so the shells of y_{n+1} (all V components; the
// restriction reads them) are P[u_new^p], P[rho_new^p] taken BEFORE the restriction into the parent. At
// theta = 0 the y_{n+1} ghosts are the next step's Y_1 ghosts (S8) and are written by its launch.
void fill_level_dense(Seq& q, int level, double theta, double dt) {
  sc_hierarchy* h = q.h;
  const Layout& L = h->L;
  const double hp = 2.0 * dt;
  const int yn = q.cur[level];
  const int pnew = q.cur[level - 1], pold = 1 - pnew;  // the parent has already stepped
  double c1[4], cs[4];
  dense_coeffs(1, theta, c1);
  for (int ib : L.level_boxes[level]) {
    GhostArgs a{};
    a.nprob = 1;
    GhostProblem& d = a.prob[0];
    d.nsrc = 5;
    d.src_arr[0] = L.a_state(pold);
    d.src_arr[1] = L.a_state(pold) + L.F;
    d.src_arr[2] = L.a_Y2r();
    d.src_arr[3] = L.a_Y3r();
    d.src_arr[4] = L.a_Y4r();
    d.nout = 4;
    d.dst_arr[0] = L.a_state(yn);
    d.dst_arr[1] = L.a_state(yn) + L.F;
    d.dst_arr[2] = L.a_Y2r();
    d.dst_arr[3] = L.a_Y3r();
    d.coef[0][0] = 1.0;
    for (int j = 0; j < 4; ++j) d.coef[0][1 + j] = hp * c1[j];
    const double as[3] = {0.5, 0.5, 1.0};
    for (int s = 0; s < 3; ++s) {
      dense_coeffs(s + 2, theta, cs);
      for (int j = 0; j < 4; ++j) d.coef[1 + s][1 + j] = 2.0 * (cs[j] - c1[j]) / as[s];  // h_p / (a_s dt) = 2 / a_s
    }
    if (theta != 0.0) {  // second problem: same-time prolongation of the parent's new state into y_{n+1}
      a.nprob = 2;
      GhostProblem& e = a.prob[1];
      e.nsrc = e.nout = 2;
      e.src_arr[0] = L.a_state(pnew);
      e.src_arr[1] = L.a_state(pnew) + L.F;
      e.dst_arr[0] = L.a_state(1 - yn);
      e.dst_arr[1] = L.a_state(1 - yn) + L.F;
      e.coef[0][0] = 1.0;
      e.coef[1][1] = 1.0;
    }
    ghost_launch(q, ib, a);
  }
}

// Uniform mode (S11): ghosts = plain prolongation of the parent's arrays at the same time / stage.
void fill_level_same_time(Seq& q, int level, int n, const int* child_arrays, const int* parent_arrays) {
  sc_hierarchy* h = q.h;
  for (int ib : h->L.level_boxes[level]) {
    GhostArgs a{};
    a.nprob = 1;
    GhostProblem& d = a.prob[0];
    d.nsrc = d.nout = n;
    for (int s = 0; s < n; ++s) {
      d.src_arr[s] = parent_arrays[s];
      d.dst_arr[s] = child_arrays[s];
      d.coef[s][s] = 1.0;
    }
    ghost_launch(q, ib, a);
  }
}

void restrict_level(Seq& q, int level) {  // level -> level-1, into the parents' current y
  sc_hierarchy* h = q.h;
  for (int ib : h->L.level_boxes[level]) {
    const BoxInfo& b = h->L.boxes[ib];
    prof_begin(h, KIND_RESTRICT, 8.0 * h->L.V * (cells(b.v) + cells(b.v) / 8.0));
    RestrictArgs a{};
    a.child = b.v;
    a.parent = h->L.boxes[b.parent].v;
    a.V = h->L.V;
    a.a_child = h->L.a_state(q.cur[level]);
    a.ychild = h->arr(ib, a.a_child);
    a.yparent = h->arr(b.parent, h->L.a_state(q.cur[level - 1]));
    a.tmap = h->tmap_ok[ib] ? h->rmaps[ib].bytes : nullptr;
    a.nr = h->L.ops.nr;
    a.rmin = h->L.ops.rmin;
    for (int m = 0; m < 10; ++m) a.r[m] = h->L.ops.r[m];
    launch_restrict(a, h->stream);
    prof_end(h);
    ++q.n;
  }
}

// ---- the general stage-by-stage path (stage_gen.cu / stage_ko_tma.cu): Kreiss-Oliger dissipation of either order,
// the RK3 / RK2 integrators, the radiative outer boundary ------------------------
// Arrays of stage s: U_s = a_U(s), R_s = a_R(s) for s = 2..4; Y_1 = y_n lives in the state slot. RK3 keeps k_3 in
// the (otherwise unused) arrays of stage 4 and k_4 = f(y_{n+1}) in K4; RK2 keeps k_2 in K4.
void stage_ko_level(Seq& q, int level, int s, double dt) {
  sc_hierarchy* h = q.h;
  const Layout& L = h->L;
  const int S = L.integrator;
  // s == S + 1 (RK3 only): the slope at the new state; q.cur[level] has already been flipped
  const bool extra = s > S;
  const int yn = extra ? 1 - q.cur[level] : q.cur[level], ynew = 1 - yn, F = L.F;
  const bool keep = q.sub && level + 1 < L.nlevels;
  for (int ib : L.level_boxes[level]) {
    StageKOArgs a{};
    a.b = L.boxes[ib].v;
    a.F = F;
    a.stage = s;
    a.integrator = S;
    a.fd_order = L.fd_order;
    a.ko_order = L.ko_sigma > 0.0 ? L.ko_order : 0;
    a.yn_u = h->arr(ib, L.a_state(yn));
    a.yn_r = h->arr(ib, L.a_state(yn) + F);
    const int in_u = s == 1 ? L.a_state(yn) : (extra ? L.a_state(ynew) : L.a_U(s));
    const int in_r = s == 1 ? L.a_state(yn) + F : (extra ? L.a_state(ynew) + F : L.a_R(s));
    a.Yu = h->arr(ib, in_u);
    a.Yr = h->arr(ib, in_r);
    a.outU = s < S ? h->arr(ib, L.a_U(s + 1)) : h->arr(ib, L.a_state(ynew));
    a.outR = s < S ? h->arr(ib, L.a_R(s + 1)) : h->arr(ib, L.a_state(ynew) + F);
    a.U2 = h->arr(ib, L.a_U(2)); a.U3 = h->arr(ib, L.a_U(3));
    a.R2 = h->arr(ib, L.a_R(2)); a.R3 = h->arr(ib, L.a_R(3));
    const bool write_k = extra || (keep && s == S && S != 3);
    a.K4u = write_k ? h->arr(ib, L.a_K4()) : nullptr;
    a.K4r = write_k ? h->arr(ib, L.a_K4() + F) : nullptr;
    const bool write_k3 = keep && S == 3 && s == 3;
    a.K3u = write_k3 ? h->arr(ib, L.a_U(4)) : nullptr;
    a.K3r = write_k3 ? h->arr(ib, L.a_R(4)) : nullptr;
    a.dt = dt;
    for (int d = 0; d < 3; ++d) {
      const double dx = L.dx(level, d);
      a.inv12dx2[d] = 1.0 / (12.0 * dx * dx);
      a.ko[d] = L.ko_sigma / ((L.ko_order == 9 ? 1024.0 : 64.0) * dx);
      a.dx[d] = dx;
      a.x0[d] = L.xlo[d] + ((double)a.b.lo[d] + (L.vertex ? 0.0 : 0.5)) * dx;
    }
    a.rad_nb = (level == 0 && L.outer_bc == 1) ? L.g : 0;
    a.A = h->coupling();
    a.tmap = h->kmap_ok[ib] ? h->kmaps[ib].bytes : nullptr;
    a.tile_variant = h->tile_variant[ib];
    a.a_Yu = in_u;
    a.a_Yr = in_r;
    // reads: Y_s (2 arrays); + y_n (2) for s >= 2; + the earlier stage vectors of the final combine.  writes: 2 (+ 2 per kept slope)
    double per = extra ? 4.0 : (s == 1 ? 4.0 : 6.0);
    if (!extra && s == S) per += 2.0 * (S - 2) + (write_k || write_k3 ? 2.0 : 0.0);
    prof_begin(h, KIND_STAGE, 8.0 * per * F * cells(a.b));
    launch_stage_ko(a, h->stream);
    prof_end(h);
    ++q.n;
  }
}

// ghosts of one stage's output arrays on level 0 (periodic boundary; the radiative boundary has no ghosts, S29)
void periodic_stage_ko(Seq& q, int s) {
  const Layout& L = q.h->L;
  if (L.outer_bc != 0) return;
  periodic_level0(q, L.a_U(s), L.F);
  periodic_level0(q, L.a_R(s), L.F);
}
void periodic_state_gen(Seq& q, int slot) {
  const Layout& L = q.h->L;
  if (L.outer_bc != 0) return;
  periodic_level0(q, L.a_state(slot), L.V);
}

// Dense-output ghosts of ALL stage vectors of one level-step of `level` >= 1, one launch
// per box. The parent stores, per variable, (y_n, Y_2, .., Y_S) and the slopes that cannot be recovered from them:
//   RK4: (y_n, Y_2, Y_3, Y_4, k_4),   k_j = (Y_{j+1} - y_n)/(a_j h_p), j = 1..3
//   RK3: (y_n, Y_2, Y_3, k_3, k_4),   k_1 = 2 (Y_2 - y_n)/h_p,  k_2 = (Y_3 - y_n)/(2 h_p) + (Y_2 - y_n)/h_p
//   RK2: (y_n, Y_2, k_2),             k_1 = 2 (Y_2 - y_n)/h_p
// so the value of the stage formulas,  y_n^p + h_p sum_j c^(s)_j k_j  (dense_coeffs_rk), is a fixed combination of
// the stored arrays — one (5 -> S) problem for the u variables and one for the rho variables (RK2's three sources
// are padded to five with zero coefficients: the tuned kernel's shape). At theta = 1/2 a third problem
// prolongs the parent's new state into the shells of y_{n+1} (eq (10) at theta + 1/2 = 1, S8).
void fill_level_dense_ko(Seq& q, int level, double theta, double dt) {
  sc_hierarchy* h = q.h;
  const Layout& L = h->L;
  const double hp = 2.0 * dt;
  const int yn = q.cur[level], F = L.F, S = L.integrator;
  const int pnew = q.cur[level - 1], pold = 1 - pnew;
  for (int ib : L.level_boxes[level]) {
    GhostArgs a{};
    a.nprob = 2;
    for (int v = 0; v < 2; ++v) {  // v = 0: u variables, v = 1: rho variables
      GhostProblem& d = a.prob[v];
      d.nsrc = 5;
      d.nout = S;
      const int st_p = L.a_state(pold) + v * F;
      d.src_arr[0] = st_p;
      d.dst_arr[0] = L.a_state(yn) + v * F;
      for (int s = 2; s <= S; ++s) d.dst_arr[s - 1] = v ? L.a_R(s) : L.a_U(s);
      auto stage_arr = [&](int s) { return v ? L.a_R(s) : L.a_U(s); };
      if (S == 4) {
        for (int s = 2; s <= 4; ++s) d.src_arr[s - 1] = stage_arr(s);
        d.src_arr[4] = L.a_K4() + v * F;
      } else if (S == 3) {
        d.src_arr[1] = stage_arr(2);
        d.src_arr[2] = stage_arr(3);
        d.src_arr[3] = stage_arr(4);           // k_3
        d.src_arr[4] = L.a_K4() + v * F;       // k_4 = f(y_{n+1})
      } else {
        d.src_arr[1] = stage_arr(2);
        d.src_arr[2] = L.a_K4() + v * F;       // k_2
        d.src_arr[3] = d.src_arr[4] = st_p;    // padding, coefficients 0
      }
      for (int s = 1; s <= S; ++s) {
        double c[4];
        dense_coeffs_rk(S, s, theta, c);
        double* co = d.coef[s - 1];
        if (S == 4) {
          const double as[3] = {0.5, 0.5, 1.0};
          double c0 = 1.0;
          for (int j = 0; j < 3; ++j) { co[1 + j] = c[j] / as[j]; c0 -= c[j] / as[j]; }
          co[0] = c0;
          co[4] = hp * c[3];
        } else if (S == 3) {
          co[1] = 2.0 * c[0] + c[1];
          co[2] = 0.5 * c[1];
          co[0] = 1.0 - co[1] - co[2];
          co[3] = hp * c[2];
          co[4] = hp * c[3];
        } else {
          co[1] = 2.0 * c[0];
          co[0] = 1.0 - co[1];
          co[2] = hp * c[1];
        }
      }
    }
    if (theta != 0.0) {
      a.nprob = 3;
      GhostProblem& e = a.prob[2];
      e.nsrc = e.nout = 2;
      e.src_arr[0] = L.a_state(pnew);
      e.src_arr[1] = L.a_state(pnew) + F;
      e.dst_arr[0] = L.a_state(1 - yn);
      e.dst_arr[1] = L.a_state(1 - yn) + F;
      e.coef[0][0] = 1.0;
      e.coef[1][1] = 1.0;
    }
    ghost_launch(q, ib, a);
  }
}

// Fork / join of the level scheduler. The refinement ghosts of a level's SECOND sub-step (theta = 1/2) depend only on
// the parent's stored step, which is complete once the parent has stepped: they can be written as soon as the
// first sub-step's kernels have read the shells they replace — while the children of this level take their two
// sub-steps and restrict (those read and write this level's INTERIOR only: footprints lie 4 cells inside, S13).
// In a captured step the fill is recorded on a second stream (a parallel branch of the graph) and joined before
// the second sub-step's first stage kernel; eager / profiled steps issue it in place on the one stream.
void prefill_second_substep(Seq& q, int level, double dt, bool in_line = false) {
  sc_hierarchy* h = q.h;
  const Layout& L = h->L;
  cudaStream_t main = h->stream;
  const bool fork = q.capturing && !in_line;
  auto chk = [&](cudaError_t e) { if (e != cudaSuccess && q.err == cudaSuccess) q.err = e; };
  if (fork) {
    chk(cudaEventRecord(h->ev_fork[level], main));
    chk(cudaStreamWaitEvent(h->side, h->ev_fork[level], 0));
    h->stream = h->side;
  }
  if (L.general()) fill_level_dense_ko(q, level, 0.5, dt);
  else fill_level_dense(q, level, 0.5, dt);
  sibling_level(q, level, L.a_state(q.cur[level]), L.V);
  if (fork) {
    chk(cudaEventRecord(h->ev_join[level], h->side));
    h->stream = main;
  }
  q.prefilled[level] = fork ? 1 : 2;  // 2: written in line on the main stream, nothing to join
}
// Measured (profiles/r01_v4.md): beside the children's kernels the fill costs nothing on 128^3 levels (cfg 3 0.806 ->
// 0.798 ms per coarse step, cfg 4 184.4 -> 183.6 ms) but its CTAs disturb the bandwidth-bound stage kernels of 256^3
// levels (cfg 5 21.68 -> 21.9 ms): the branch is taken for levels of at most 6 M cells. SC_OVERLAP=0 / 1 forces it.
bool overlap_wanted(const sc_hierarchy* h, int level) {
  if (h->overlap_mode >= 0) return h->overlap_mode != 0;
  double n = 0.0;
  for (int ib : h->L.level_boxes[level]) n += cells(h->L.boxes[ib].v);
  return n <= 6.0e6;
}
// true if the ghosts of the level-step about to start were prefilled (and, in a captured step, joins the branch)
bool join_prefill(Seq& q, int level) {
  if (!q.prefilled[level]) return false;
  if (q.prefilled[level] == 1 && q.capturing) {
    const cudaError_t e = cudaStreamWaitEvent(q.h->stream, q.h->ev_join[level], 0);
    if (e != cudaSuccess && q.err == cudaSuccess) q.err = e;
  }
  q.prefilled[level] = 0;
  return true;
}

void level_step_ko(Seq& q, int level, double dt, double theta) {
  const Layout& L = q.h->L;
  const int yn = q.cur[level], S = L.integrator;
  if (level == 0) {
    if (!q.l0_valid) periodic_state_gen(q, yn);
  } else if (!join_prefill(q, level)) {
    fill_level_dense_ko(q, level, theta, dt);
    sibling_level(q, level, L.a_state(yn), L.V);
  }
  for (int s = 1; s <= S; ++s) {
    stage_ko_level(q, level, s, dt);
    if (level == 0) {
      if (s < S) periodic_stage_ko(q, s + 1);
      else periodic_state_gen(q, 1 - yn);
    } else if (s < S) {  // the stage vector just produced: ghosts inside a sibling take the sibling's Y_{s+1}
      sibling_level(q, level, L.a_U(s + 1), L.F);
      sibling_level(q, level, L.a_R(s + 1), L.F);
    } else if (theta != 0.0) {
      sibling_level(q, level, L.a_state(1 - yn), L.V);
    }
  }
  if (level == 0) q.l0_valid = true;
  q.cur[level] = 1 - yn;
}

// non-subcycled step of the general path (S11/S15): same-time prolongation of the parent's same stage vector
void uniform_step_ko(Seq& q, double dt) {
  const Layout& L = q.h->L;
  const int Lv = L.nlevels, F = L.F, S = L.integrator;
  if (!q.l0_valid) periodic_state_gen(q, q.cur[0]);
  for (int l = 1; l < Lv; ++l) {
    const int ca[2] = {L.a_state(q.cur[l]), L.a_state(q.cur[l]) + F};
    const int pa[2] = {L.a_state(q.cur[l - 1]), L.a_state(q.cur[l - 1]) + F};
    fill_level_same_time(q, l, 2, ca, pa);
    sibling_level(q, l, ca[0], L.V);
  }
  for (int s = 1; s <= S; ++s) {
    for (int l = 0; l < Lv; ++l) stage_ko_level(q, l, s, dt);
    if (s < S) {
      periodic_stage_ko(q, s + 1);
      const int ca[2] = {L.a_U(s + 1), L.a_R(s + 1)};
      for (int l = 1; l < Lv; ++l) {
        fill_level_same_time(q, l, 2, ca, ca);
        sibling_level(q, l, ca[0], F);
        sibling_level(q, l, ca[1], F);
      }
    }
  }
  periodic_state_gen(q, 1 - q.cur[0]);
  q.l0_valid = true;
  for (int l = 1; l < Lv; ++l) {
    const int ca[2] = {L.a_state(1 - q.cur[l]), L.a_state(1 - q.cur[l]) + F};
    const int pa[2] = {L.a_state(1 - q.cur[l - 1]), L.a_state(1 - q.cur[l - 1]) + F};
    fill_level_same_time(q, l, 2, ca, pa);
    sibling_level(q, l, ca[0], L.V);
  }
  for (int l = 0; l < Lv; ++l) q.cur[l] = 1 - q.cur[l];
  for (int l = Lv - 1; l >= 1; --l) restrict_level(q, l);
}

// One RK4 step of one level (eqs 1-9) with its ghost fills. theta: start of this step inside the parent's.
void level_step(Seq& q, int level, double dt, double theta) {
  const Layout& L = q.h->L;
  if (L.general()) { level_step_ko(q, level, dt, theta); return; }
  const int yn = q.cur[level];
  if (level == 0) {
    if (!q.l0_valid) periodic_level0(q, L.a_state(yn), L.V);
  } else if (!join_prefill(q, level)) {
    fill_level_dense(q, level, theta, dt);
    sibling_level(q, level, L.a_state(yn), L.V);  // u_n, rho_n: on a sibling's interior u_n + a_1 dt rho_n IS Y_{2,u}
  }
  stage_level(q, level, STAGE_12, dt);
  if (level == 0) periodic_level0(q, L.a_Y2r(), 2 * L.F);  // Y2r and Y3r are adjacent
  else sibling_level(q, level, L.a_Y2r(), 2 * L.F);
  stage_level(q, level, STAGE_34, dt);
  if (level == 0) {
    periodic_level0(q, L.a_state(1 - yn), L.V);
    q.l0_valid = true;
  } else if (theta != 0.0) {
    // y_{n+1} of the step that ends at the parent's t_{n+1}: read by the restriction and sc_debug_read_padded. After
    // a first sub-step (theta = 0) nothing reads these ghosts before the next launch refills and re-exchanges them.
    sibling_level(q, level, L.a_state(1 - yn), L.V);
  }
  q.cur[level] = 1 - yn;
}

// steps 1-7 of PAPER.md:113-119
void advance(Seq& q, int level, double dt, double theta) {
  level_step(q, level, dt, theta);
  if (level + 1 < q.h->L.nlevels) {
    // RK3 (S28): the child's dense output reads k_4 = f(y_{n+1}) of this level, whose ghosts are the NEXT sub-step's
    // Y_1 ghosts (S8): after a first sub-step they are written now, in line, by that sub-step's fill
    const bool rk3 = q.h->L.integrator == 3;
    if (level >= 1 && theta == 0.0 && (rk3 || overlap_wanted(q.h, level))) prefill_second_substep(q, level, dt, rk3);
    if (rk3) stage_ko_level(q, level, 4, dt);
    advance(q, level + 1, 0.5 * dt, 0.0);
    advance(q, level + 1, 0.5 * dt, 0.5);
    restrict_level(q, level + 1);
  }
}

// non-subcycled step of all levels (reading S11/S15)
void uniform_step(Seq& q, double dt) {
  const Layout& L = q.h->L;
  if (L.general()) { uniform_step_ko(q, dt); return; }
  const int Lv = L.nlevels, F = L.F;
  // ghosts of y_n = (u_n, rho_n): from the parent's y_n after the last restriction
  if (!q.l0_valid) periodic_level0(q, L.a_state(q.cur[0]), L.V);
  for (int l = 1; l < Lv; ++l) {
    const int ca[2] = {L.a_state(q.cur[l]), L.a_state(q.cur[l]) + F};
    const int pa[2] = {L.a_state(q.cur[l - 1]), L.a_state(q.cur[l - 1]) + F};
    fill_level_same_time(q, l, 2, ca, pa);
    sibling_level(q, l, ca[0], L.V);
  }
  for (int l = 0; l < Lv; ++l) stage_level(q, l, STAGE_12, dt);
  // ghosts of Y_{3,u}, Y_{4,u} = P[parent's Y_{3,u}, Y_{4,u}]  <=>  shells of Y2r, Y3r = P[parent's Y2r, Y3r]
  periodic_level0(q, L.a_Y2r(), 2 * F);
  for (int l = 1; l < Lv; ++l) {
    const int ca[2] = {L.a_Y2r(), L.a_Y3r()};
    fill_level_same_time(q, l, 2, ca, ca);
    sibling_level(q, l, ca[0], 2 * F);
  }
  for (int l = 0; l < Lv; ++l) stage_level(q, l, STAGE_34, dt);
  // ghosts of y_{n+1} from the parent's y_{n+1} before the restriction
  periodic_level0(q, L.a_state(1 - q.cur[0]), L.V);
  q.l0_valid = true;
  for (int l = 1; l < Lv; ++l) {
    const int ca[2] = {L.a_state(1 - q.cur[l]), L.a_state(1 - q.cur[l]) + F};
    const int pa[2] = {L.a_state(1 - q.cur[l - 1]), L.a_state(1 - q.cur[l - 1]) + F};
    fill_level_same_time(q, l, 2, ca, pa);
    sibling_level(q, l, ca[0], L.V);
  }
  for (int l = 0; l < Lv; ++l) q.cur[l] = 1 - q.cur[l];
  for (int l = Lv - 1; l >= 1; --l) restrict_level(q, l);
}

void record_step(Seq& q, double dt_coarse, int subcycling) {
  q.sub = subcycling != 0;
  if (subcycling) {
    advance(q, 0, dt_coarse, 0.0);
  } else {
    const int nsub = 1 << (q.h->L.nlevels - 1);
    for (int i = 0; i < nsub; ++i) uniform_step(q, dt_coarse / (double)nsub);
  }
}

int check_box(sc_hierarchy* h, int level, int box, int comp, int* gbox) {
  if (!h) { set_error("null hierarchy"); return SC_ERR_INVALID_ARG; }
  if (level < 0 || level >= h->L.nlevels) { set_error("level out of range"); return SC_ERR_INVALID_ARG; }
  if (box < 0 || box >= (int)h->L.level_boxes[level].size()) { set_error("box out of range"); return SC_ERR_INVALID_ARG; }
  if (comp < 0 || comp >= h->L.V) { set_error("component out of range"); return SC_ERR_INVALID_ARG; }
  *gbox = h->L.level_boxes[level][box];
  return SC_OK;
}

int read_array(sc_hierarchy* h, int gbox, const double* padded, double* dst, int with_ghosts, int dst_on_device) {
  const BoxView& v = h->L.boxes[gbox].v;
  const int e = with_ghosts ? v.g : 0;
  const size_t bytes = sizeof(double) * (size_t)(v.n[0] + 2 * e) * (v.n[1] + 2 * e) * (v.n[2] + 2 * e);
  if (dst_on_device) {
    launch_pack(v, padded, dst, with_ghosts, h->stream);
    ++h->launches;
    SC_CUDA(cudaGetLastError());
    SC_CUDA(cudaStreamSynchronize(h->stream));
    return SC_OK;
  }
  launch_pack(v, padded, h->staging, with_ghosts, h->stream);
  ++h->launches;
  SC_CUDA(cudaGetLastError());
  SC_CUDA(cudaMemcpyAsync(dst, h->staging, bytes, cudaMemcpyDeviceToHost, h->stream));
  SC_CUDA(cudaStreamSynchronize(h->stream));
  return SC_OK;
}

}  // namespace

// =================================================================================================
extern "C" {

const char* sc_last_error(void) { return sc::last_error().c_str(); }

uint64_t sc_arena_bytes(const sc_hierarchy_desc* desc) {
  Layout L;
  std::string err;
  if (build_layout(desc, &L, &err) != SC_OK) { set_error(err); return 0; }
  return L.arena_bytes;
}

int32_t sc_create_hierarchy(const sc_hierarchy_desc* desc, sc_hierarchy** out) {
  if (!out) { set_error("null out pointer"); return SC_ERR_INVALID_ARG; }
  *out = nullptr;
  sc_hierarchy* h = new sc_hierarchy;
  std::string err;
  int rc = build_layout(desc, &h->L, &err);
  if (rc != SC_OK) { set_error(err); delete h; return rc; }
  int ndev = 0;
  cudaError_t ce = cudaGetDeviceCount(&ndev);
  if (ce != cudaSuccess || ndev < 1) {
    set_error(std::string("no usable CUDA device (there is no CPU fallback): ") + cudaGetErrorString(ce));
    delete h;
    return SC_ERR_CUDA;
  }
  h->stream = static_cast<cudaStream_t>(desc->cuda_stream);
  if (!h->stream) {  // stream capture is illegal on the legacy default stream: use a private one
    if ((ce = cudaStreamCreateWithFlags(&h->stream, cudaStreamNonBlocking)) != cudaSuccess) {
      set_error(std::string("cudaStreamCreate: ") + cudaGetErrorString(ce));
      delete h;
      return SC_ERR_CUDA;
    }
    h->own_stream = true;
  }
  if (desc->arena) {
    if (desc->arena_bytes < h->L.arena_bytes || (reinterpret_cast<uintptr_t>(desc->arena) & 255)) {
      set_error("arena too small or not 256-byte aligned");
      if (h->own_stream) cudaStreamDestroy(h->stream);
      delete h;
      return SC_ERR_OOM;
    }
    h->arena = static_cast<char*>(desc->arena);
  } else {
    if (cudaMalloc(&h->arena, h->L.arena_bytes) != cudaSuccess) {
      cudaGetLastError();
      set_error("cudaMalloc of the arena failed");
      if (h->own_stream) cudaStreamDestroy(h->stream);
      delete h;
      return SC_ERR_OOM;
    }
    h->own_arena = true;
  }
  size_t smax = 0;
  for (const BoxInfo& b : h->L.boxes) {
    const size_t s = sizeof(double) * (size_t)(b.v.n[0] + 2 * b.v.g) * (b.v.n[1] + 2 * b.v.g) * (b.v.n[2] + 2 * b.v.g);
    if (s > smax) smax = s;
  }
  h->staging_bytes = smax;
  h->tiles.resize(h->L.boxes.size());
  auto bail = [&](const char* what, cudaError_t e) {
    set_error(std::string(what) + ": " + cudaGetErrorString(e));
    if (h->staging) cudaFree(h->staging);
    for (auto& bt : h->tiles) if (bt.dev) cudaFree(bt.dev);
    for (auto& s : h->sib) if (s.dev) cudaFree(s.dev);
    if (h->own_arena) cudaFree(h->arena);
    if (h->own_stream) cudaStreamDestroy(h->stream);
    delete h;
    return SC_ERR_CUDA;
  };
  if ((ce = cudaMalloc(&h->staging, smax)) != cudaSuccess) return bail("cudaMalloc(staging)", ce);
  if ((ce = cudaMemsetAsync(h->arena, 0, h->L.arena_bytes, h->stream)) != cudaSuccess) return bail("memset", ce);
  if (h->L.has_coupling) {
    h->coupling_host.assign(desc->coupling, desc->coupling + (size_t)h->L.F * h->L.F);
    ce = cudaMemcpyAsync(h->arena + h->L.coupling_offset, desc->coupling, sizeof(double) * h->L.F * h->L.F,
                         cudaMemcpyHostToDevice, h->stream);
    if (ce != cudaSuccess) return bail("copy coupling", ce);
  }
  for (size_t ib = 0; ib < h->L.boxes.size(); ++ib) {
    if (h->L.boxes[ib].level == 0) continue;
    std::vector<GhostTile> tl;
    std::vector<BoxView> sibs;
    for (int jb : h->L.level_boxes[h->L.boxes[ib].level])
      if (jb != (int)ib) sibs.push_back(h->L.boxes[jb].v);
    if (!h->L.ops.is_default() || !ghost_tma_geometry_ok(h->L.boxes[ib].v)) continue;  // the direct-load kernel fills these
    build_ghost_tiles(h->L.boxes[ib].v, h->L.boxes[h->L.boxes[ib].parent].v, tl, &sibs);
    sc_hierarchy::BoxTiles& bt = h->tiles[ib];
    bt.n = (int)tl.size();
    if (tl.empty()) continue;
    if ((ce = cudaMalloc(&bt.dev, sizeof(GhostTile) * tl.size())) != cudaSuccess) return bail("cudaMalloc(tiles)", ce);
    if ((ce = cudaMemcpy(bt.dev, tl.data(), sizeof(GhostTile) * tl.size(), cudaMemcpyHostToDevice)) != cudaSuccess)
      return bail("copy tiles", ce);
  }
  h->sib.assign(h->L.nlevels, {});
  for (int l = 1; l < h->L.nlevels; ++l) {
    std::vector<SiblingPair> pr;
    sc_hierarchy::LevelSiblings& s = h->sib[l];
    for (int ia : h->L.level_boxes[l])
      for (int ib : h->L.level_boxes[l]) {
        if (ia == ib) continue;
        const BoxInfo &A = h->L.boxes[ia], &B = h->L.boxes[ib];
        SiblingPair p{};
        long long nc = 1;
        for (int a = 0; a < 3; ++a) {  // padded(A) n interior(B), level-global indices
          const int lo = std::max(A.v.lo[a] - A.v.g, B.v.lo[a]);
          const int hi = std::min(A.v.lo[a] + A.v.n[a] + A.v.g, B.v.lo[a] + B.v.n[a]);
          p.lo[a] = lo;
          p.n[a] = hi - lo;
          nc *= hi > lo ? hi - lo : 0;
        }
        if (nc == 0) continue;
        p.dst = A.v;
        p.src = B.v;
        p.dst_off = (long long)(A.arena_offset / sizeof(double));
        p.src_off = (long long)(B.arena_offset / sizeof(double));
        pr.push_back(p);
        s.maxcells = std::max(s.maxcells, nc);
        s.cells += (double)nc;
      }
    s.n = (int)pr.size();
    if (pr.empty()) continue;
    if ((ce = cudaMalloc(&s.dev, sizeof(SiblingPair) * pr.size())) != cudaSuccess) return bail("cudaMalloc(sibling pairs)", ce);
    if ((ce = cudaMemcpy(s.dev, pr.data(), sizeof(SiblingPair) * pr.size(), cudaMemcpyHostToDevice)) != cudaSuccess)
      return bail("copy sibling pairs", ce);
  }
  h->tmaps.resize(h->L.boxes.size());
  h->tmap_ok.assign(h->L.boxes.size(), 0);
  h->tile_variant.assign(h->L.boxes.size(), 0);
  h->rmaps.resize(h->L.boxes.size());
  h->gmaps.resize(h->L.boxes.size());
  h->kmaps.resize(h->L.boxes.size());
  h->kmap_ok.assign(h->L.boxes.size(), 0);
  h->gmap_ok.assign(h->L.boxes.size(), 0);
  for (size_t ib = 0; ib < h->L.boxes.size(); ++ib) {
    const BoxInfo& b = h->L.boxes[ib];
    // decided here, once, with the hierarchy's device current (the choice reads its SM count); ADVICE r2
    h->tile_variant[ib] = (char)stage_tile_variant(b.v, h->L.F);
    h->tmap_ok[ib] = make_box_tensor_map(b.v, b.narrays, h->arr((int)ib, 0), h->tile_variant[ib] ? 8 : 0, h->tmaps[ib].bytes) &&
                     make_box_tensor_map(b.v, b.narrays, h->arr((int)ib, 0), 1, h->rmaps[ib].bytes);
    {  // the general path's stage tile: halo 3 (4th-order differences), 4 (8th order) or 5 (with delta^10)
      const Layout& L = h->L;
      const bool ko9 = L.ko_sigma > 0.0 && L.ko_order == 9;
      const int kind = L.fd_order == 8 ? (ko9 ? 7 : 6) : (h->tile_variant[ib] ? 9 : 5);
      const int need = kind == 7 ? 5 : (kind == 6 ? 4 : 3);  // kinds 5, 9: halo 3
      h->kmap_ok[ib] = L.general() && (L.fd_order == 8 || !ko9) && L.g >= need &&
                       make_box_tensor_map(b.v, b.narrays, h->arr((int)ib, 0), kind, h->kmaps[ib].bytes);
    }
    h->gmap_ok[ib] = 1;
    for (int ax = 0; ax < 3; ++ax)
      if (!make_box_tensor_map(b.v, b.narrays, h->arr((int)ib, 0), 2 + ax, h->gmaps[ib].m[ax].bytes)) h->gmap_ok[ib] = 0;
  }
  if ((ce = cudaStreamSynchronize(h->stream)) != cudaSuccess) return bail("sync", ce);
  h->cur.assign(h->L.nlevels, 0);
  h->l0_ghosts_valid = false;
  const char* env = getenv("SC_KERNELS");
  select_kernels(env && !strcmp(env, "ref") ? 0 : 1);
  {
    const char* eo = getenv("SC_OVERLAP");
    h->overlap_mode = eo ? (strcmp(eo, "0") ? 1 : 0) : -1;
    if ((ce = cudaStreamCreateWithFlags(&h->side, cudaStreamNonBlocking)) != cudaSuccess) return bail("cudaStreamCreate(side)", ce);
    h->ev_fork.assign(h->L.nlevels, nullptr);
    h->ev_join.assign(h->L.nlevels, nullptr);
    for (int l = 0; l < h->L.nlevels; ++l) {
      if ((ce = cudaEventCreateWithFlags(&h->ev_fork[l], cudaEventDisableTiming)) != cudaSuccess) return bail("cudaEventCreate", ce);
      if ((ce = cudaEventCreateWithFlags(&h->ev_join[l], cudaEventDisableTiming)) != cudaSuccess) return bail("cudaEventCreate", ce);
    }
  }
  const char* eg = getenv("SC_GRAPH");
  h->use_graph = !(eg && !strcmp(eg, "0"));
  const char* ed = getenv("SC_DEBUG_SYNC");
  h->debug_sync = ed && !strcmp(ed, "1") && !h->use_graph;
  *out = h;
  return SC_OK;
}

int32_t sc_set_state(sc_hierarchy* h, int32_t level, int32_t box, int32_t comp, const double* src,
                     int32_t src_on_device) {
  int gb;
  int rc = check_box(h, level, box, comp, &gb);
  if (rc != SC_OK) return rc;
  if (!src) { set_error("null src"); return SC_ERR_INVALID_ARG; }
  const BoxView& v = h->L.boxes[gb].v;
  double* dstarr = h->arr(gb, h->L.a_state(h->cur[level]) + comp);
  const size_t bytes = sizeof(double) * (size_t)v.n[0] * v.n[1] * v.n[2];
  if (src_on_device) {
    launch_unpack(v, src, dstarr, h->stream);
    ++h->launches;
    SC_CUDA(cudaGetLastError());
  } else {
    SC_CUDA(cudaMemcpyAsync(h->staging, src, bytes, cudaMemcpyHostToDevice, h->stream));
    launch_unpack(v, h->staging, dstarr, h->stream);
    ++h->launches;
    SC_CUDA(cudaGetLastError());
    SC_CUDA(cudaStreamSynchronize(h->stream));
  }
  if (level == 0) h->l0_ghosts_valid = false;
  return SC_OK;
}

int32_t sc_step(sc_hierarchy* h, double dt_coarse, int32_t subcycling) {
  if (!h) { set_error("null hierarchy"); return SC_ERR_INVALID_ARG; }
  if (!std::isfinite(dt_coarse) || dt_coarse <= 0.0) { set_error("dt_coarse must be finite and > 0"); return SC_ERR_INVALID_ARG; }
  subcycling = subcycling ? 1 : 0;
  Seq q{};
  q.h = h;
  q.cur = h->cur;
  q.l0_valid = h->l0_ghosts_valid;
  q.prefilled.assign(h->L.nlevels, 0);
  if (!h->use_graph || h->profiling) {
    record_step(q, dt_coarse, subcycling);
    SC_CUDA(cudaGetLastError());
    SC_CUDA(q.err);
    h->launches += q.n;
  } else {
    GraphKey key{subcycling, 0};
    uint64_t dt_bits = 0;
    memcpy(&dt_bits, &dt_coarse, sizeof(double));
    for (int l = 0; l < h->L.nlevels; ++l) key.phase |= (uint32_t)(h->cur[l] ? 1 : 0) << l;
    if (h->l0_ghosts_valid) key.phase |= 1u << 31;
    auto it = h->graphs.find(key);
    if (it == h->graphs.end() || it->second.dt_bits != dt_bits) {
      cudaGraph_t g = nullptr;
      SC_CUDA(cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal));
      q.capturing = true;
      record_step(q, dt_coarse, subcycling);
      cudaError_t le = cudaGetLastError();
      if (le == cudaSuccess) le = q.err;
      cudaError_t ee = cudaStreamEndCapture(h->stream, &g);
      ++h->n_captures;
      if (le != cudaSuccess || ee != cudaSuccess) {
        set_error(std::string("graph capture failed: ") + cudaGetErrorString(le != cudaSuccess ? le : ee));
        if (g) cudaGraphDestroy(g);
        return SC_ERR_CUDA;
      }
      bool updated = false;
      if (it != h->graphs.end()) {  // same launch sequence, other step size: new parameters into the existing executable
        cudaGraphExecUpdateResultInfo info;
        if (cudaGraphExecUpdate(it->second.exec, g, &info) == cudaSuccess) {
          updated = true;
          ++h->n_updates;
        } else {
          cudaGetLastError();
          cudaGraphExecDestroy(it->second.exec);
          h->graphs.erase(it);
          it = h->graphs.end();
        }
      }
      if (!updated) {
        if (h->graphs.size() >= kMaxGraphs) {
          for (auto& kv : h->graphs)
            if (kv.second.exec) cudaGraphExecDestroy(kv.second.exec);
          h->graphs.clear();
        }
        GraphEntry e;
        cudaError_t ie = cudaGraphInstantiate(&e.exec, g, 0);
        ++h->n_instantiations;
        if (ie != cudaSuccess) {
          cudaGraphDestroy(g);
          set_error(std::string("cudaGraphInstantiate: ") + cudaGetErrorString(ie));
          return SC_ERR_CUDA;
        }
        it = h->graphs.emplace(key, e).first;
      }
      cudaGraphDestroy(g);
      it->second.dt_bits = dt_bits;
      it->second.launches = q.n;
      it->second.cur_after = q.cur;
    }
    SC_CUDA(cudaGraphLaunch(it->second.exec, h->stream));
    h->launches += it->second.launches;
    q.cur = it->second.cur_after;
  }
  h->cur = q.cur;
  h->l0_ghosts_valid = true;
  h->time += dt_coarse;
  return SC_OK;
}

int32_t sc_read_level(sc_hierarchy* h, int32_t level, int32_t box, int32_t comp, double* dst,
                      int32_t dst_on_device) {
  int gb;
  int rc = check_box(h, level, box, comp, &gb);
  if (rc != SC_OK) return rc;
  if (!dst) { set_error("null dst"); return SC_ERR_INVALID_ARG; }
  return read_array(h, gb, h->arr(gb, h->L.a_state(h->cur[level]) + comp), dst, 0, dst_on_device);
}

int32_t sc_debug_graph_stats(const sc_hierarchy* h, uint64_t* captures, uint64_t* instantiations, uint64_t* updates,
                             uint64_t* cached) {
  if (!h) { set_error("null hierarchy"); return SC_ERR_INVALID_ARG; }
  if (captures) *captures = h->n_captures;
  if (instantiations) *instantiations = h->n_instantiations;
  if (updates) *updates = h->n_updates;
  if (cached) *cached = h->graphs.size();
  return SC_OK;
}

double sc_time(const sc_hierarchy* h) { return h ? h->time : 0.0; }
uint64_t sc_launch_count(const sc_hierarchy* h) { return h ? h->launches : 0; }

int64_t sc_debug_ghost_map(sc_hierarchy* h, int32_t level, int32_t box, int32_t* out, uint64_t cap) {
  int gb;
  int rc = check_box(h, level, box, 0, &gb);
  if (rc != SC_OK) return rc;
  if (level < 1) { set_error("level 0 has no refinement-boundary ghosts"); return SC_ERR_INVALID_ARG; }
  const BoxInfo& b = h->L.boxes[gb];
  const long long ns = ghost_cell_count(b.v);
  if (!out) return ns;
  if (cap < (uint64_t)(7 * ns)) { set_error("ghost map capacity too small"); return SC_ERR_INVALID_ARG; }
  int* dev = nullptr;
  SC_CUDA(cudaMalloc(&dev, sizeof(int) * 7 * ns));
  launch_ghost_map(b.v, h->L.boxes[b.parent].v, dev, h->stream);
  ++h->launches;
  cudaError_t e = cudaMemcpyAsync(out, dev, sizeof(int) * 7 * ns, cudaMemcpyDeviceToHost, h->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(h->stream);
  cudaFree(dev);
  if (e != cudaSuccess) { set_error(std::string("ghost map: ") + cudaGetErrorString(e)); return SC_ERR_CUDA; }
  return ns;
}

int32_t sc_debug_read_padded(sc_hierarchy* h, int32_t level, int32_t box, int32_t comp, double* dst) {
  int gb;
  int rc = check_box(h, level, box, comp, &gb);
  if (rc != SC_OK) return rc;
  if (!dst) { set_error("null dst"); return SC_ERR_INVALID_ARG; }
  return read_array(h, gb, h->arr(gb, h->L.a_state(h->cur[level]) + comp), dst, 1, 0);
}

int32_t sc_debug_max_abs(sc_hierarchy* h, int32_t level, int32_t box, int32_t comp, double* out) {
  int gb;
  int rc = check_box(h, level, box, comp, &gb);
  if (rc != SC_OK) return rc;
  if (!out) { set_error("null out"); return SC_ERR_INVALID_ARG; }
  unsigned long long* bits = reinterpret_cast<unsigned long long*>(h->staging);
  SC_CUDA(cudaMemsetAsync(bits, 0, sizeof(unsigned long long), h->stream));
  launch_max_abs(h->L.boxes[gb].v, h->arr(gb, h->L.a_state(h->cur[level]) + comp), bits, h->stream);
  ++h->launches;
  SC_CUDA(cudaGetLastError());
  unsigned long long r = 0;
  SC_CUDA(cudaMemcpyAsync(&r, bits, sizeof r, cudaMemcpyDeviceToHost, h->stream));
  SC_CUDA(cudaStreamSynchronize(h->stream));
  memcpy(out, &r, sizeof r);
  return SC_OK;
}

int32_t sc_debug_read_slot(sc_hierarchy* h, int32_t level, int32_t box, int32_t slot, int32_t comp, double* dst) {
  int gb;
  int rc = check_box(h, level, box, comp, &gb);
  if (rc != SC_OK) return rc;
  if (!dst) { set_error("null dst"); return SC_ERR_INVALID_ARG; }
  const Layout& L = h->L;
  int a;
  if (slot == 1) a = L.a_state(1 - h->cur[level]) + comp;
  else if (slot >= 2 && slot <= 4) {
    if (comp < L.F) { set_error("stage vectors store the rho components only (comp >= nfields)"); return SC_ERR_INVALID_ARG; }
    a = (slot == 2 ? L.a_Y2r() : (slot == 3 ? L.a_Y3r() : L.a_Y4r())) + comp - L.F;
  } else { set_error("slot must be 1 (y_n) or 2..4 (Y_2..Y_4)"); return SC_ERR_INVALID_ARG; }
  return read_array(h, gb, h->arr(gb, a), dst, 0, 0);
}

int32_t sc_debug_stream(sc_hierarchy* h, int32_t nread, int32_t nwrite, uint64_t ndoubles, double* gbps) {
  if (!h || !gbps || nread < 1 || nread > 8 || nwrite < 1 || nwrite > 8 || ndoubles < 2 || (ndoubles & 1)) {
    set_error("sc_debug_stream: bad argument");
    return SC_ERR_INVALID_ARG;
  }
  double *in = nullptr, *out = nullptr;
  if (cudaMalloc(&in, sizeof(double) * ndoubles * nread) != cudaSuccess ||
      cudaMalloc(&out, sizeof(double) * ndoubles * nwrite) != cudaSuccess) {
    cudaGetLastError();
    if (in) cudaFree(in);
    set_error("sc_debug_stream: allocation failed");
    return SC_ERR_OOM;
  }
  cudaMemsetAsync(in, 0, sizeof(double) * ndoubles * nread, h->stream);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  float best = 1e30f;
  for (int rep = 0; rep < 7; ++rep) {  // two warm-up launches, five timed
    cudaEventRecord(e0, h->stream);
    launch_stream_mix(in, out, ndoubles, nread, nwrite, h->stream);
    cudaEventRecord(e1, h->stream);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep >= 2 && ms < best) best = ms;
  }
  h->launches += 7;
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(in);
  cudaFree(out);
  SC_CUDA(cudaGetLastError());
  *gbps = (double)(nread + nwrite) * 8.0 * (double)ndoubles / ((double)best * 1e-3) / 1e9;
  return SC_OK;
}

int32_t sc_debug_interp_weights(int32_t interp_order, int32_t centering, int32_t* np, int32_t* pmin, double* w0,
                                double* w1, int32_t* nr, int32_t* rmin, double* r) {
  if ((interp_order != 0 && interp_order != 1) || (centering != 0 && centering != 1)) {
    set_error("interp_order and centering must be 0 or 1");
    return SC_ERR_UNSUPPORTED;
  }
  if (!np || !pmin || !w0 || !w1 || !nr || !rmin || !r) { set_error("null out pointer"); return SC_ERR_INVALID_ARG; }
  const InterpOps P = make_interp_ops(interp_order, centering);
  *np = P.np; *pmin = P.pmin; *nr = P.nr; *rmin = P.rmin;
  for (int m = 0; m < 10; ++m) { w0[m] = P.w[0][m]; w1[m] = P.w[1][m]; r[m] = P.r[m]; }
  return SC_OK;
}

int32_t sc_profile(sc_hierarchy* h, int32_t enable) {
  if (!h) { set_error("null hierarchy"); return SC_ERR_INVALID_ARG; }
  SC_CUDA(cudaStreamSynchronize(h->stream));
  for (auto& r : h->prof) { cudaEventDestroy(r.e0); cudaEventDestroy(r.e1); }
  h->prof.clear();
  h->profiling = enable != 0;
  return SC_OK;
}

int32_t sc_profile_read(sc_hierarchy* h, int32_t kind, uint64_t* launches, double* ms, double* bytes) {
  if (!h || kind < 0 || kind >= NKIND) { set_error("bad hierarchy or kind"); return SC_ERR_INVALID_ARG; }
  SC_CUDA(cudaStreamSynchronize(h->stream));
  uint64_t n = 0;
  double t = 0.0, b = 0.0;
  for (auto& r : h->prof) {
    if (r.kind != kind) continue;
    float e = 0.f;
    SC_CUDA(cudaEventElapsedTime(&e, r.e0, r.e1));
    t += e;
    b += r.bytes;
    ++n;
  }
  if (launches) *launches = n;
  if (ms) *ms = t;
  if (bytes) *bytes = b;
  return SC_OK;
}

int32_t sc_destroy(sc_hierarchy* h) {
  if (!h) return SC_OK;
  cudaStreamSynchronize(h->stream);
  for (auto& r : h->prof) { cudaEventDestroy(r.e0); cudaEventDestroy(r.e1); }
  for (auto& kv : h->graphs)
    if (kv.second.exec) cudaGraphExecDestroy(kv.second.exec);
  if (h->staging) cudaFree(h->staging);
  for (auto& bt : h->tiles) if (bt.dev) cudaFree(bt.dev);
  for (auto& s : h->sib) if (s.dev) cudaFree(s.dev);
  if (h->own_arena && h->arena) cudaFree(h->arena);
  for (auto e : h->ev_fork) if (e) cudaEventDestroy(e);
  for (auto e : h->ev_join) if (e) cudaEventDestroy(e);
  if (h->side) cudaStreamDestroy(h->side);
  if (h->own_stream) cudaStreamDestroy(h->stream);
  delete h;
  return SC_OK;
}

}  // extern "C"
