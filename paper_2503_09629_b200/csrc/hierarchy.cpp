// hierarchy.cpp — host-only: validation of a hierarchy description (nesting rules, S13) and
// the arena layout. No CUDA calls here, so sc_arena_bytes() works on a machine without a GPU.
#include <cmath>
#include <cstdio>

#include "sc_internal.h"

namespace sc {

namespace {
thread_local std::string g_last_error;
inline unsigned long long round_up(unsigned long long x, unsigned long long a) { return (x + a - 1) / a * a; }
}  // namespace

void set_error(const std::string& msg) { g_last_error = msg; }
const std::string& last_error() { return g_last_error; }

static int fail(std::string* err, int code, const char* fmt, int a = 0, int b = 0, int c = 0) {
  char buf[256];
  snprintf(buf, sizeof buf, fmt, a, b, c);
  if (err) *err = buf;
  return code;
}

// ------------------------------------------------------------------------------------------------
// Interpolation operators (readings S3, S4, S30, S31) as EXACT rationals.
// Every operator here interpolates through equally spaced nodes to a target that is a whole number of QUARTER node
// spacings away from them, so in quarter-spacing units all positions are integers and each Lagrange weight
//     w_q = prod_{j != q} (T - X_j) / prod_{j != q} (X_q - X_j)
// is a ratio of two integers below 2^53 (at most ten nodes: |numerator| <= 9.1e8, |denominator| <= 4^9 9!). One IEEE
// division of the two then gives the correctly rounded value of the rational; no floating-point product is formed.
// ------------------------------------------------------------------------------------------------
struct Stencil {
  int count;  // number of nodes
  int first;  // offset of node 0 in cells / grid points
  int shift;  // node q sits at quarter-position 4 * (first + q) + shift  (shift -2: nodes at half-integer offsets)
};

static void exact_weights(const Stencil& st, int target, double* w) {
  for (int q = 0; q < st.count; ++q) {
    const long long xq = 4ll * (st.first + q) + st.shift;
    long long num = 1, den = 1;
    for (int j = 0; j < st.count; ++j) {
      if (j == q) continue;
      const long long xj = 4ll * (st.first + j) + st.shift;
      num *= target - xj;
      den *= xq - xj;
    }
    w[q] = num == 0 ? 0.0 : (double)num / (double)den;  // (no -0.0 where the target sits on another node)
  }
}

InterpOps make_interp_ops(int interp, int vertex) {
  // rows: [centering][interp_order];  prolongation stencil over parent points, restriction stencil over fine points
  static const Stencil PROLONG[2][2] = {{{5, -2, 0}, {9, -4, 0}}, {{6, -2, 0}, {10, -4, 0}}};
  static const Stencil RESTRICT[2][2] = {{{6, -2, -2}, {10, -4, -2}}, {{1, 0, 0}, {1, 0, 0}}};
  const Stencil& p = PROLONG[vertex ? 1 : 0][interp ? 1 : 0];
  const Stencil& r = RESTRICT[vertex ? 1 : 0][interp ? 1 : 0];
  InterpOps P;
  for (int m = 0; m < 10; ++m) P.w[0][m] = P.w[1][m] = P.r[m] = 0.0;
  P.np = p.count;
  P.pmin = p.first;
  P.nr = r.count;
  P.rmin = r.first;
  // fine point of parity 0 / 1 relative to parent point 0: cell-centred -1/4, +1/4 (S1); vertex-centred 0, +1/2 (S31)
  exact_weights(p, vertex ? 0 : -1, P.w[0]);
  exact_weights(p, vertex ? 2 : +1, P.w[1]);
  // the parent point lies midway between fine cells 2I and 2I + 1 (cell-centred: fine cell 2I + j at j - 1/2), or on
  // fine point 0 (vertex-centred: the one-node stencil is injection)
  exact_weights(r, 0, P.r);
  return P;
}

int build_layout(const sc_hierarchy_desc* d, Layout* L, std::string* err) {
  if (!d || !L) return fail(err, SC_ERR_INVALID_ARG, "null description");
  if (!d->boxes || d->nboxes < 1 || d->nlevels < 1) return fail(err, SC_ERR_INVALID_ARG, "no boxes / levels");
  if (d->ref_ratio != 2) return fail(err, SC_ERR_UNSUPPORTED, "ref_ratio must be 2 (got %d)", d->ref_ratio);
  if (d->ghost < MIN_GHOST || d->ghost > MAX_GHOST)
    return fail(err, SC_ERR_UNSUPPORTED, "ghost width %d outside [2, 5]", d->ghost);
  if (d->nlevels > SC_MAX_LEVELS) return fail(err, SC_ERR_UNSUPPORTED, "too many levels (%d)", d->nlevels);
  if (d->nfields < 1 || d->nfields > MAX_FIELDS)
    return fail(err, SC_ERR_UNSUPPORTED, "nfields %d outside [1, 32]", d->nfields);
  for (int a = 0; a < 3; ++a) {
    if (d->domain_cells[a] < 8 || d->domain_cells[a] > (1 << 20))
      return fail(err, SC_ERR_INVALID_ARG, "domain_cells[%d] = %d out of range", a, d->domain_cells[a]);
    if (!(d->xhi[a] > d->xlo[a]) || !std::isfinite(d->xhi[a]) || !std::isfinite(d->xlo[a]))
      return fail(err, SC_ERR_INVALID_ARG, "empty or non-finite physical extent on axis %d", a);
    // level-global indices must fit int32 with room for ghosts
    if ((long long)d->domain_cells[a] << (d->nlevels - 1) > (1ll << 30))
      return fail(err, SC_ERR_UNSUPPORTED, "finest index space exceeds 2^30 on axis %d", a);
  }
  if (d->coupling)
    for (int q = 0; q < d->nfields * d->nfields; ++q)
      if (!std::isfinite(d->coupling[q])) return fail(err, SC_ERR_INVALID_ARG, "non-finite coupling entry %d", q);

  if (!(d->ko_sigma >= 0.0) || !std::isfinite(d->ko_sigma))
    return fail(err, SC_ERR_INVALID_ARG, "ko_sigma must be finite and >= 0");
  if (d->fd_order != 0 && d->fd_order != 4 && d->fd_order != 8)
    return fail(err, SC_ERR_UNSUPPORTED, "fd_order must be 4 or 8 (got %d)", d->fd_order);
  const int fd = d->fd_order == 8 ? 8 : 4;
  if (fd == 8 && d->ghost < 4)
    return fail(err, SC_ERR_UNSUPPORTED, "8th-order differences read 4 ghost layers (ghost = %d)", d->ghost);
  if (d->ko_order != 0 && d->ko_order != 5 && d->ko_order != 9)
    return fail(err, SC_ERR_UNSUPPORTED, "ko_order must be 0, 5 or 9 (got %d)", d->ko_order);
  const int ko = d->ko_order ? d->ko_order : (fd == 8 ? 9 : 5);
  if (d->ko_sigma > 0.0 && d->ghost < (ko == 9 ? 5 : 3))
    return fail(err, SC_ERR_UNSUPPORTED, "Kreiss-Oliger dissipation of order %d reads %d ghost layers", ko, ko == 9 ? 5 : 3);
  if (d->integrator != 0 && d->integrator != 4 && d->integrator != 3 && d->integrator != 2)
    return fail(err, SC_ERR_UNSUPPORTED, "integrator must be 4 (RK4), 3 (RK3) or 2 (RK2) (got %d)", d->integrator);
  if (d->outer_bc != 0 && d->outer_bc != 1) return fail(err, SC_ERR_UNSUPPORTED, "outer_bc must be 0 or 1 (got %d)", d->outer_bc);
  if ((d->interp_order != 0 && d->interp_order != 1) || (d->centering != 0 && d->centering != 1))
    return fail(err, SC_ERR_UNSUPPORTED, "interp_order and centering must be 0 or 1");
  if (d->outer_bc == 1)
    for (int a = 0; a < 3; ++a) {
      if (!(d->xlo[a] < 0.0 && d->xhi[a] > 0.0))
        return fail(err, SC_ERR_INVALID_ARG, "radiative boundary: the origin must lie strictly inside the domain (axis %d)", a);
      // the boundary operator divides by r = |x| at every point within `ghost` level-0 points of a face (S29): keep the
      // origin out of that zone, so that no boundary point (cell- or vertex-centred) can sit at r = 0
      const double zone = d->ghost * (d->xhi[a] - d->xlo[a]) / d->domain_cells[a];
      if (!(-d->xlo[a] > zone && d->xhi[a] > zone))
        return fail(err, SC_ERR_INVALID_ARG,
                    "radiative boundary: the origin must lie more than ghost * dx0 = %g from both faces of axis %d "
                    "(the boundary zone evaluates 1/r)", zone, a);
    }

  L->nlevels = d->nlevels;
  L->fd_order = fd;
  L->ko_order = ko;
  L->integrator = d->integrator ? d->integrator : 4;
  L->outer_bc = d->outer_bc;
  L->interp = d->interp_order;
  L->vertex = d->centering;
  L->ops = make_interp_ops(L->interp, L->vertex);
  if (L->ops.nr > 1 && -L->ops.rmin > d->ghost)
    return fail(err, SC_ERR_UNSUPPORTED, "the restriction reads %d ghost layers (ghost = %d)", -L->ops.rmin, d->ghost);
  L->ko_sigma = d->ko_sigma;
  L->g = d->ghost;
  L->F = d->nfields;
  L->V = 2 * d->nfields;
  L->has_coupling = d->coupling != nullptr;
  for (int a = 0; a < 3; ++a) { L->domain[a] = d->domain_cells[a]; L->xlo[a] = d->xlo[a]; L->xhi[a] = d->xhi[a]; }
  L->boxes.clear();
  L->level_boxes.assign(d->nlevels, {});

  const int g = d->ghost;
  const int margin = (g + 1) / 2 + L->ops.reach();  // parent cells between a child's coverage and its parent's edge
  for (int ib = 0; ib < d->nboxes; ++ib) {
    const sc_box& s = d->boxes[ib];
    if (s.level < 0 || s.level >= d->nlevels) return fail(err, SC_ERR_INVALID_ARG, "box %d: level %d out of range", ib, s.level);
    if (ib > 0 && s.level < d->boxes[ib - 1].level) return fail(err, SC_ERR_NESTING, "boxes must be sorted by level (box %d)", ib);
    BoxInfo b{};
    b.level = s.level;
    b.index_in_level = (int)L->level_boxes[s.level].size();
    b.parent = -1;
    for (int a = 0; a < 3; ++a) {
      if (s.n[a] < 8) return fail(err, SC_ERR_NESTING, "box %d: n[%d] = %d < 8", ib, a, s.n[a]);
      const long long ext = (long long)d->domain_cells[a] << s.level;
      if (s.lo[a] < 0 || (long long)s.lo[a] + s.n[a] > ext)
        return fail(err, SC_ERR_NESTING, "box %d: outside the level's index space on axis %d", ib, a);
      b.v.n[a] = s.n[a];
      b.v.lo[a] = s.lo[a];
    }
    b.v.g = g;
    b.v.px = (int)round_up((unsigned long long)(XOFF + s.n[0] + g), 16);
    b.v.py = s.n[1] + 2 * g;
    b.v.pz = s.n[2] + 2 * g;
    b.v.plane = (long long)b.v.px * b.v.py;
    b.v.vol = (long long)round_up((unsigned long long)(b.v.plane * b.v.pz), 32);
    L->level_boxes[s.level].push_back(ib);
    L->boxes.push_back(b);
  }
  if (L->level_boxes[0].size() != 1) return fail(err, SC_ERR_NESTING, "level 0 must be exactly one box");
  {
    const BoxInfo& b0 = L->boxes[L->level_boxes[0][0]];
    for (int a = 0; a < 3; ++a)
      if (b0.v.lo[a] != 0 || b0.v.n[a] != d->domain_cells[a])
        return fail(err, SC_ERR_NESTING, "level 0 box must cover the whole periodic domain (axis %d)", a);
  }
  for (int l = 1; l < d->nlevels; ++l) {
    if (L->level_boxes[l].empty()) return fail(err, SC_ERR_NESTING, "level %d has no box", l);
    for (int ib : L->level_boxes[l]) {
      BoxInfo& b = L->boxes[ib];
      for (int a = 0; a < 3; ++a)
        if ((b.v.lo[a] & 1) || (b.v.n[a] & 1))
          return fail(err, SC_ERR_NESTING, "box %d: lo and n must be even on axis %d (whole parent cells)", ib, a);
      for (int ip : L->level_boxes[l - 1]) {
        const BoxInfo& p = L->boxes[ip];
        bool inside = true;
        for (int a = 0; a < 3; ++a) {
          const int plo = b.v.lo[a] / 2 - p.v.lo[a];
          const int phi = (b.v.lo[a] + b.v.n[a]) / 2 - p.v.lo[a];
          if (plo < margin || phi > p.v.n[a] - margin) inside = false;
        }
        if (inside) { b.parent = ip; break; }
      }
      if (b.parent < 0)
        return fail(err, SC_ERR_NESTING, "box %d (level %d): not inside a parent box with %d parent cells of margin", ib, l, margin);
      for (int jb : L->level_boxes[l]) {
        if (jb == ib) continue;
        const BoxInfo& o = L->boxes[jb];
        bool disjoint = false;  // any distance is fine (abutting boxes exchange ghosts, kernels.h a7)
        for (int a = 0; a < 3; ++a)
          if (b.v.lo[a] >= o.v.lo[a] + o.v.n[a] || o.v.lo[a] >= b.v.lo[a] + b.v.n[a]) disjoint = true;
        if (!disjoint) return fail(err, SC_ERR_NESTING, "boxes %d and %d overlap", ib, jb);
      }
    }
  }
  // arena: boxes in order, each a run of narrays arrays of vol doubles (sc_internal.h); vol is a multiple
  // of 32 doubles, so every array starts on a 256-byte boundary
  unsigned long long off = 0;
  for (BoxInfo& b : L->boxes) {
    b.narrays = 2 * L->V + 3 * L->F + (L->has_coupling ? 2 * L->F : 0) + (L->general() ? 3 * L->F + L->V : 0);
    b.arena_offset = off;
    off += (unsigned long long)b.narrays * (unsigned long long)b.v.vol * sizeof(double);
  }
  L->coupling_offset = off;
  off += round_up((unsigned long long)L->F * L->F * sizeof(double), 256);
  L->arena_bytes = off;
  return SC_OK;
}

}  // namespace sc
