// capi.cu — the C ABI of libsubcycle (include/subcycle.h) and the level scheduler:
// the Berger–Oliger recursion of PAPER.md:111-119 (steps 1-7) unrolled on the host into a fixed sequence
// of kernel launches on one CUDA stream, captured once per (mode, dt, buffer phase) into a CUDA graph
// and replayed. No host synchronisation inside a step.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
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

struct GraphKey {
  int sub;
  uint64_t dt_bits;
  uint32_t phase;
  bool operator<(const GraphKey& o) const {
    if (sub != o.sub) return sub < o.sub;
    if (dt_bits != o.dt_bits) return dt_bits < o.dt_bits;
    return phase < o.phase;
  }
};
struct GraphEntry {
  cudaGraphExec_t exec = nullptr;
  uint64_t launches = 0;
  std::vector<int> cur_after;
};

struct sc_hierarchy {
  Layout L;
  char* arena = nullptr;
  bool own_arena = false;
  cudaStream_t stream = nullptr;
  bool own_stream = false;
  double* staging = nullptr;      // device, largest padded dense box
  size_t staging_bytes = 0;
  std::vector<int> cur;           // per level: slot (0 or 2) that holds the current state y
  std::vector<char> ghosts_valid; // per level: ghosts of y hold the last stage-5 fill (no set_state since)
  double time = 0.0;
  uint64_t launches = 0;
  uint64_t counting = 0;          // launches of the sequence being recorded
  bool use_graph = true;
  std::map<GraphKey, GraphEntry> graphs;
  // per-launch CUDA-event timing (sc_profile): eager launches, one event pair per kernel
  struct BoxTiles { GhostTile* dev = nullptr; int n = 0; int s0 = 0, s1 = 0; };
  std::vector<BoxTiles> tiles;    // per box (levels >= 1): ghost-shell tile list on the device
  bool profiling = false;
  struct ProfRec { int kind; double bytes; cudaEvent_t e0, e1; };
  std::vector<ProfRec> prof;

  double* slot(int box, int s) const {
    const BoxInfo& b = L.boxes[box];
    return reinterpret_cast<double*>(arena + b.arena_offset + (unsigned long long)s * b.slot_bytes);
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

// Folded dense-output coefficients: ghost value of RK stage `stage` of a child step that starts at
// parent progress theta is  P[ y_old^p + h_p * sum_j c_j k_j^p ]  with, from eqs (10)-(18)
// and child step h = r h_p, r = 1/2:
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

// ---- launch recording -----------------------------------------------------------------------
struct Seq {
  sc_hierarchy* h;
  std::vector<int> cur;  // working copy of the slot phases
  uint64_t n = 0;
};

enum { KIND_RHS = 0, KIND_GHOST = 1, KIND_PERIODIC = 2, KIND_RESTRICT = 3, NKIND = 4 };

// Algorithmic bytes per launch: what the method must move.
double cells(const BoxView& v) { return (double)v.n[0] * v.n[1] * v.n[2]; }
double shell_cells(const BoxView& v) {
  return (double)(v.n[0] + 2 * v.g) * (v.n[1] + 2 * v.g) * (v.n[2] + 2 * v.g) - cells(v);
}
double footprint_cells(const BoxView& v) {  // parent cells a ghost fill of this box reads
  // ghost cells sit in parent cells up to gc = ceil(g/2) beyond the child's coverage [0, nc); the 5-point
  // interpolation adds 2 more on every side and reaches 2 cells into the coverage
  const int gc = (v.g + 1) / 2;
  double outer = 1.0, inner = 1.0;
  for (int a = 0; a < 3; ++a) {
    const int nc = v.n[a] / 2;
    outer *= nc + 2 * gc + 4;
    inner *= nc > 4 ? nc - 4 : 0;
  }
  return outer - inner;
}
double rhs_bytes(const BoxView& v, int V, int stage, bool keep_k) {
  const double per = stage == 1 ? 3.0 : (stage == 4 ? (keep_k ? 7.0 : 6.0) : 4.0);
  return 8.0 * per * V * cells(v);
}

void prof_begin(sc_hierarchy* h, int kind, double bytes) {
  if (!h->profiling) return;
  sc_hierarchy::ProfRec r{kind, bytes, nullptr, nullptr};
  cudaEventCreate(&r.e0);
  cudaEventCreate(&r.e1);
  cudaEventRecord(r.e0, h->stream);
  h->prof.push_back(r);
}
void prof_end(sc_hierarchy* h) {
  if (!h->profiling) return;
  cudaEventRecord(h->prof.back().e1, h->stream);
}

void rhs_level(Seq& q, int level, int stage, int sYin, int sYn, int sYout, double cdt, bool keep_k) {
  sc_hierarchy* h = q.h;
  for (int ib : h->L.level_boxes[level]) {
    RhsArgs a{};
    a.b = h->L.boxes[ib].v;
    a.F = h->L.F;
    a.stage = stage;
    a.Yin = h->slot(ib, sYin);
    a.yn = h->slot(ib, sYn);
    a.kout = keep_k ? h->slot(ib, SLOT_K1 + stage - 1) : nullptr;
    a.Yout = h->slot(ib, sYout);
    a.k1 = h->slot(ib, SLOT_K1);
    a.k2 = h->slot(ib, SLOT_K1 + 1);
    a.k3 = h->slot(ib, SLOT_K1 + 2);
    a.cdt = cdt;
    for (int d = 0; d < 3; ++d) {
      const double dx = h->L.dx(level, d);
      a.inv12dx2[d] = 1.0 / (12.0 * dx * dx);
    }
    a.A = h->coupling();
    prof_begin(h, KIND_RHS, rhs_bytes(a.b, h->L.V, stage, keep_k));
    launch_rhs_stage(a, h->stream);
    prof_end(h);
    ++q.n;
  }
}

// ghosts of slot `sdst` of every box of `level`: periodic (level 0) or dense output of the parent
// (subcycled: base = parent's y_old slot, coefficients of (stage, theta) times the parent step hp).
void fill_level_dense(Seq& q, int level, int sdst, int stage, double theta, double hp, int parent_yold) {
  sc_hierarchy* h = q.h;
  for (int ib : h->L.level_boxes[level]) {
    const BoxInfo& b = h->L.boxes[ib];
    if (level == 0) {
      prof_begin(h, KIND_PERIODIC, 16.0 * h->L.V * shell_cells(b.v));
      launch_periodic_fill(b.v, h->L.V, h->slot(ib, sdst), h->stream);
      prof_end(h);
      ++q.n;
      continue;
    }
    GhostArgs a{};
    a.child = b.v;
    a.parent = h->L.boxes[b.parent].v;
    a.V = h->L.V;
    a.dst = h->slot(ib, sdst);
    a.base = h->slot(b.parent, parent_yold);
    a.tiles = h->tiles[ib].dev; a.ntiles = h->tiles[ib].n;
    a.s0_doubles = h->tiles[ib].s0; a.s1_doubles = h->tiles[ib].s1;
    double c[4];
    dense_coeffs(stage, theta, c);
    a.use_k = 0;
    for (int j = 0; j < 4; ++j) {
      a.k[j] = h->slot(b.parent, SLOT_K1 + j);
      a.coef[j] = hp * c[j];
      if (c[j] != 0.0) a.use_k |= 1 << j;
    }
    prof_begin(h, KIND_GHOST, 8.0 * h->L.V * ((1 + __builtin_popcount(a.use_k)) * footprint_cells(b.v) + shell_cells(b.v)));
    launch_ghost_fill(a, h->stream);
    prof_end(h);
    ++q.n;
  }
}

// uniform mode: ghosts = plain prolongation of the parent's slot `sparent` (same RK stage, same time)
void fill_level_same_time(Seq& q, int level, int sdst, int sparent) {
  sc_hierarchy* h = q.h;
  for (int ib : h->L.level_boxes[level]) {
    const BoxInfo& b = h->L.boxes[ib];
    if (level == 0) {
      prof_begin(h, KIND_PERIODIC, 16.0 * h->L.V * shell_cells(b.v));
      launch_periodic_fill(b.v, h->L.V, h->slot(ib, sdst), h->stream);
      prof_end(h);
      ++q.n;
      continue;
    }
    GhostArgs a{};
    a.child = b.v;
    a.parent = h->L.boxes[b.parent].v;
    a.V = h->L.V;
    a.dst = h->slot(ib, sdst);
    a.base = h->slot(b.parent, sparent);
    a.use_k = 0;
    a.tiles = h->tiles[ib].dev; a.ntiles = h->tiles[ib].n;
    a.s0_doubles = h->tiles[ib].s0; a.s1_doubles = h->tiles[ib].s1;
    for (int j = 0; j < 4; ++j) { a.k[j] = a.base; a.coef[j] = 0.0; }
    prof_begin(h, KIND_GHOST, 8.0 * h->L.V * (footprint_cells(b.v) + shell_cells(b.v)));
    launch_ghost_fill(a, h->stream);
    prof_end(h);
    ++q.n;
  }
}

void restrict_level(Seq& q, int level) {  // level -> level-1, into the parents' current y
  sc_hierarchy* h = q.h;
  for (int ib : h->L.level_boxes[level]) {
    const BoxInfo& b = h->L.boxes[ib];
    prof_begin(h, KIND_RESTRICT, 8.0 * h->L.V * (cells(b.v) + cells(b.v) / 8.0));
    launch_restrict(b.v, h->L.boxes[b.parent].v, h->L.V, h->slot(ib, q.cur[level]),
                    h->slot(b.parent, q.cur[level - 1]), h->stream);
    prof_end(h);
    ++q.n;
  }
}

// One RK4 step of one level (eqs 1-9) with its five ghost fills. theta: start of this step inside the
// parent's step. Slot roles: y_n = cur, Y_2 -> slot 1, Y_3 -> other, Y_4 -> slot 1, y_{n+1} -> other.
void level_step(Seq& q, int level, double dt, double theta, bool first_fill) {
  sc_hierarchy* h = q.h;
  const int yn = q.cur[level], A = 1, B = 2 - yn;
  const int pyold = level > 0 ? 2 - q.cur[level - 1] : 0;  // the parent already stepped: its y_n is "other"
  const double hp = 2.0 * dt;
  const bool has_child = level + 1 < h->L.nlevels;
  if (first_fill) fill_level_dense(q, level, yn, 1, theta, hp, pyold);
  rhs_level(q, level, 1, yn, yn, A, 0.5 * dt, true);
  fill_level_dense(q, level, A, 2, theta, hp, pyold);
  rhs_level(q, level, 2, A, yn, B, 0.5 * dt, true);
  fill_level_dense(q, level, B, 3, theta, hp, pyold);
  rhs_level(q, level, 3, B, yn, A, dt, true);
  fill_level_dense(q, level, A, 4, theta, hp, pyold);
  rhs_level(q, level, 4, A, yn, B, dt / 6.0, has_child);
  fill_level_dense(q, level, B, 5, theta + 0.5, hp, pyold);
  q.cur[level] = B;
}

// steps 1-7 of PAPER.md:113-119
void advance(Seq& q, int level, double dt, double theta, bool first_fill) {
  level_step(q, level, dt, theta, first_fill);
  if (level + 1 < q.h->L.nlevels) {
    advance(q, level + 1, 0.5 * dt, 0.0, true);
    // the stage-1 fill at theta = 1/2 would rewrite the values the stage-5 fill at 0 + 1/2 just wrote
    // (same coefficients b(1/2), same parent data): skipped (reading S8)
    advance(q, level + 1, 0.5 * dt, 0.5, false);
    restrict_level(q, level + 1);
  }
}

// non-subcycled step of all levels (reading S11/S15)
void uniform_step(Seq& q, double dt) {
  sc_hierarchy* h = q.h;
  const int Lv = h->L.nlevels;
  auto role = [&](int level, int which) {  // 0: y_n, 1: A, 2: B
    return which == 0 ? q.cur[level] : (which == 1 ? 1 : 2 - q.cur[level]);
  };
  const double cdt[4] = {0.5 * dt, 0.5 * dt, dt, dt / 6.0};
  const int yin_role[4] = {0, 1, 2, 1}, yout_role[4] = {1, 2, 1, 2};
  for (int l = 0; l < Lv; ++l) fill_level_same_time(q, l, role(l, 0), l ? role(l - 1, 0) : 0);
  for (int s = 1; s <= 4; ++s) {
    for (int l = 0; l < Lv; ++l)
      rhs_level(q, l, s, role(l, yin_role[s - 1]), role(l, 0), role(l, yout_role[s - 1]), cdt[s - 1], s < 4);
    for (int l = 0; l < Lv; ++l)
      fill_level_same_time(q, l, role(l, yout_role[s - 1]), l ? role(l - 1, yout_role[s - 1]) : 0);
  }
  for (int l = 0; l < Lv; ++l) q.cur[l] = 2 - q.cur[l];
  for (int l = Lv - 1; l >= 1; --l) restrict_level(q, l);
}

void record_step(Seq& q, double dt_coarse, int subcycling) {
  if (subcycling) {
    advance(q, 0, dt_coarse, 0.0, true);
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
  auto bail = [&](const char* what, cudaError_t e) {
    set_error(std::string(what) + ": " + cudaGetErrorString(e));
    if (h->staging) cudaFree(h->staging);
    for (auto& bt : h->tiles) if (bt.dev) cudaFree(bt.dev);
    if (h->own_arena) cudaFree(h->arena);
    if (h->own_stream) cudaStreamDestroy(h->stream);
    delete h;
    return SC_ERR_CUDA;
  };
  if ((ce = cudaMalloc(&h->staging, smax)) != cudaSuccess) return bail("cudaMalloc(staging)", ce);
  if ((ce = cudaMemsetAsync(h->arena, 0, h->L.arena_bytes, h->stream)) != cudaSuccess) return bail("memset", ce);
  if (h->L.has_coupling) {
    ce = cudaMemcpyAsync(h->arena + h->L.coupling_offset, desc->coupling, sizeof(double) * h->L.F * h->L.F,
                         cudaMemcpyHostToDevice, h->stream);
    if (ce != cudaSuccess) return bail("copy coupling", ce);
  }
  h->tiles.resize(h->L.boxes.size());
  for (size_t ib = 0; ib < h->L.boxes.size(); ++ib) {
    if (h->L.boxes[ib].level == 0) continue;
    std::vector<GhostTile> tl;
    size_t s0 = 0, s1 = 0;
    build_ghost_tiles(h->L.boxes[ib].v, tl, &s0, &s1);
    sc_hierarchy::BoxTiles& bt = h->tiles[ib];
    bt.n = (int)tl.size(); bt.s0 = (int)s0; bt.s1 = (int)s1;
    if ((ce = cudaMalloc(&bt.dev, sizeof(GhostTile) * tl.size())) != cudaSuccess) return bail("cudaMalloc(tiles)", ce);
    if ((ce = cudaMemcpy(bt.dev, tl.data(), sizeof(GhostTile) * tl.size(), cudaMemcpyHostToDevice)) != cudaSuccess)
      return bail("copy tiles", ce);
  }
  if ((ce = cudaStreamSynchronize(h->stream)) != cudaSuccess) return bail("sync", ce);
  h->cur.assign(h->L.nlevels, 0);
  h->ghosts_valid.assign(h->L.nlevels, 0);
  const char* env = getenv("SC_KERNELS");
  select_kernels(env && !strcmp(env, "ref") ? 0 : 1);
  const char* eg = getenv("SC_GRAPH");
  h->use_graph = !(eg && !strcmp(eg, "0"));
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
  double* dstarr = h->slot(gb, h->cur[level]) + (long long)comp * v.vol;
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
  h->ghosts_valid[level] = 0;
  return SC_OK;
}

int32_t sc_step(sc_hierarchy* h, double dt_coarse, int32_t subcycling) {
  if (!h) { set_error("null hierarchy"); return SC_ERR_INVALID_ARG; }
  if (!std::isfinite(dt_coarse) || dt_coarse <= 0.0) { set_error("dt_coarse must be finite and > 0"); return SC_ERR_INVALID_ARG; }
  subcycling = subcycling ? 1 : 0;
  Seq q{h, h->cur, 0};
  if (!h->use_graph || h->profiling) {
    record_step(q, dt_coarse, subcycling);
    SC_CUDA(cudaGetLastError());
    h->launches += q.n;
  } else {
    GraphKey key{subcycling, 0, 0};
    memcpy(&key.dt_bits, &dt_coarse, sizeof(double));
    for (int l = 0; l < h->L.nlevels; ++l) key.phase |= (uint32_t)(h->cur[l] ? 1 : 0) << l;
    auto it = h->graphs.find(key);
    if (it == h->graphs.end()) {
      cudaGraph_t g = nullptr;
      SC_CUDA(cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal));
      record_step(q, dt_coarse, subcycling);
      cudaError_t le = cudaGetLastError();
      cudaError_t ee = cudaStreamEndCapture(h->stream, &g);
      if (le != cudaSuccess || ee != cudaSuccess) {
        set_error(std::string("graph capture failed: ") + cudaGetErrorString(le != cudaSuccess ? le : ee));
        if (g) cudaGraphDestroy(g);
        return SC_ERR_CUDA;
      }
      GraphEntry e;
      cudaError_t ie = cudaGraphInstantiate(&e.exec, g, 0);
      cudaGraphDestroy(g);
      if (ie != cudaSuccess) { set_error(std::string("cudaGraphInstantiate: ") + cudaGetErrorString(ie)); return SC_ERR_CUDA; }
      e.launches = q.n;
      e.cur_after = q.cur;
      it = h->graphs.emplace(key, e).first;
    }
    SC_CUDA(cudaGraphLaunch(it->second.exec, h->stream));
    h->launches += it->second.launches;
    q.cur = it->second.cur_after;
  }
  h->cur = q.cur;
  for (auto& gv : h->ghosts_valid) gv = 1;
  h->time += dt_coarse;
  return SC_OK;
}

int32_t sc_read_level(sc_hierarchy* h, int32_t level, int32_t box, int32_t comp, double* dst,
                      int32_t dst_on_device) {
  int gb;
  int rc = check_box(h, level, box, comp, &gb);
  if (rc != SC_OK) return rc;
  if (!dst) { set_error("null dst"); return SC_ERR_INVALID_ARG; }
  const BoxView& v = h->L.boxes[gb].v;
  return read_array(h, gb, h->slot(gb, h->cur[level]) + (long long)comp * v.vol, dst, 0, dst_on_device);
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
  const BoxView& v = h->L.boxes[gb].v;
  return read_array(h, gb, h->slot(gb, h->cur[level]) + (long long)comp * v.vol, dst, 1, 0);
}

int32_t sc_debug_read_slot(sc_hierarchy* h, int32_t level, int32_t box, int32_t slot, int32_t comp, double* dst) {
  int gb;
  int rc = check_box(h, level, box, comp, &gb);
  if (rc != SC_OK) return rc;
  if (!dst || slot < 0 || slot > 4) { set_error("bad slot or null dst"); return SC_ERR_INVALID_ARG; }
  const BoxView& v = h->L.boxes[gb].v;
  const int s = slot == 0 ? 2 - h->cur[level] : SLOT_K1 + slot - 1;
  return read_array(h, gb, h->slot(gb, s) + (long long)comp * v.vol, dst, 0, 0);
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
  if (h->own_arena && h->arena) cudaFree(h->arena);
  if (h->own_stream) cudaStreamDestroy(h->stream);
  delete h;
  return SC_OK;
}

}  // extern "C"
