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

int build_layout(const sc_hierarchy_desc* d, Layout* L, std::string* err) {
  if (!d || !L) return fail(err, SC_ERR_INVALID_ARG, "null description");
  if (!d->boxes || d->nboxes < 1 || d->nlevels < 1) return fail(err, SC_ERR_INVALID_ARG, "no boxes / levels");
  if (d->ref_ratio != 2) return fail(err, SC_ERR_UNSUPPORTED, "ref_ratio must be 2 (got %d)", d->ref_ratio);
  if (d->ghost < MIN_GHOST || d->ghost > MAX_GHOST)
    return fail(err, SC_ERR_UNSUPPORTED, "ghost width %d outside [2, 4]", d->ghost);
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
  if (d->ko_sigma > 0.0 && d->ghost < 3)
    return fail(err, SC_ERR_UNSUPPORTED, "Kreiss-Oliger dissipation reads 3 ghost layers (ghost = %d)", d->ghost);

  if (d->fd_order != 0 && d->fd_order != 4 && d->fd_order != 8)
    return fail(err, SC_ERR_UNSUPPORTED, "fd_order must be 4 or 8 (got %d)", d->fd_order);
  if (d->fd_order == 8 && (d->ghost < 4 || d->ko_sigma > 0.0))
    return fail(err, SC_ERR_UNSUPPORTED, "8th-order differences read 4 ghost layers (ghost = %d) and run without dissipation", d->ghost);

  L->nlevels = d->nlevels;
  L->fd_order = d->fd_order == 8 ? 8 : 4;
  L->ko_sigma = d->ko_sigma;
  L->g = d->ghost;
  L->F = d->nfields;
  L->V = 2 * d->nfields;
  L->has_coupling = d->coupling != nullptr;
  for (int a = 0; a < 3; ++a) { L->domain[a] = d->domain_cells[a]; L->xlo[a] = d->xlo[a]; L->xhi[a] = d->xhi[a]; }
  L->boxes.clear();
  L->level_boxes.assign(d->nlevels, {});

  const int g = d->ghost;
  const int margin = (g + 1) / 2 + 2;  // parent cells between a child's coverage and its parent's edge
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
    b.narrays = 2 * L->V + 3 * L->F + (L->has_coupling ? 2 * L->F : 0) + (L->ko_sigma > 0.0 ? 3 * L->F + L->V : 0);
    b.arena_offset = off;
    off += (unsigned long long)b.narrays * (unsigned long long)b.v.vol * sizeof(double);
  }
  L->coupling_offset = off;
  off += round_up((unsigned long long)L->F * L->F * sizeof(double), 256);
  L->arena_bytes = off;
  return SC_OK;
}

}  // namespace sc
