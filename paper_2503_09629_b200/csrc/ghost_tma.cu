// ghost_tma.cu — tuned refinement-boundary ghost fill (eqs 10-18 folded
// into the coefficient matrices by the scheduler; spatial operator = reading S3), sm_100a.
//
//   child array dst_arr[o](ghost cell) = P[ sum_s coef[o][s] * parent array src_arr[s] ],   P = 5x5x5 quartic Lagrange
//
// The ghost shell of a box is the union of six slabs (z-lo, z-hi, y-lo, y-hi, x-lo, x-hi); each slab is cut
// into tiles  g (thin axis) x TA x TB  fine cells whose origin is EVEN in every axis, so the parent footprint
// of a tile is exactly (TA/2+4) x (TB/2+4) x 6 parent cells. A work ITEM is (problem, field, tile).
// Persistent CTAs (two per SM) walk the item list; per item
//   0. the footprint of every source array arrives in shared memory through ONE TMA tiled load per source
//      (cp.async.bulk.tensor.4d on the parent's footprint tensor map, out-of-range cells zero-filled),
//      requested one item AHEAD: the loads of item i+1 fly while item i is interpolated, so no warp ever
//      waits on HBM (the v2 kernel spent 35 % of its samples on 7 dependent global round trips per tile);
//   1. one thread per parent column: thin-axis interpolation (6 parent cells -> g fine cells) of every
//      source, then the time combination into the outputs          -> T[plane = (o, thin cell)][b][a]
//   2. interpolation along b, register-blocked: one thread per (plane, a)  -> U[plane][fb][a]
//   3. interpolation along a and the store: thread (a-pair, fb) walks the planes; for z- and y-slabs a = x
//      and the pair is one 16-byte store, coalesced across the warp; for x-slabs (thin = x) the thread
//      writes whole 32-byte sectors (the g = 3 ghosts of a row plus one unused pad double), so no sector
//      is written partially.
// A ghost value costs 6 + 5 + 5 FMA instead of 125 and every parent value is fetched once per tile.
#include <cuda.h>

#include <cstdio>
#include <cstdlib>

#include "kernels.h"

namespace sc {

void launch_ghost_fill_direct(const GhostArgs& a, cudaStream_t st);

namespace {

// Tile geometry per thin axis AX. z- and y-slabs (A = x): 32 x 16 fine cells. x-slabs (A = y, thin = x):
// 16 x 16, and the footprint's x extent is loaded as 8 doubles from an EVEN x coordinate — a TMA tiled load
// whose innermost fp64 coordinate is odd (start not 16-byte aligned) faults on sm_100a (measured).
constexpr int TB = 16, PB = TB / 2 + 4;          // fine cells / parent footprint along B
constexpr int PT = 6;                            // parent cells along the thin axis (ghost width <= 4)
constexpr int PTX = 8;                           // ... as loaded for x-slabs (even start, 64-byte rows)
constexpr int PAMAX = 20;                        // pitch of T and U rows
template <int AX> struct Geo {
  static constexpr int TA = AX == 0 ? 16 : 32;   // fine cells along A
  static constexpr int PA = TA / 2 + 4;          // parent footprint along A (2-cell halo each side)
  static constexpr int FOOT = AX == 0 ? PTX * PA * PB : PA * PB * PT;  // doubles per source footprint
};
constexpr int FOOTMAX = Geo<2>::FOOT;            // 1440 doubles = 11520 B: stride between sources in smem
constexpr int NTHR = 256;
static_assert(Geo<0>::FOOT <= FOOTMAX && Geo<1>::FOOT == FOOTMAX, "source slots are FOOTMAX doubles");
static_assert(Geo<2>::PA * PB <= NTHR && Geo<2>::PA <= PAMAX, "phase 1: one thread per parent column");
static_assert(TB * (Geo<2>::TA / 2) == NTHR && TB * Geo<0>::TA == NTHR, "phase 3 thread maps");
static_assert((FOOTMAX * 8) % 128 == 0 && (Geo<0>::FOOT * 8) % 16 == 0, "TMA destination alignment");

__device__ __forceinline__ uint32_t smem_u32g(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_wait_g(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
  } while (!ok);
}

// quartic Lagrange weights at -1/4 (parity 0) and +1/4 (parity 1) of the parent spacing, offsets -2..2 (S3)
__device__ __forceinline__ double wprol(int parity, int c) {
  constexpr double w1[5] = {35.0 / 2048.0, -252.0 / 2048.0, 1890.0 / 2048.0, 420.0 / 2048.0, -45.0 / 2048.0};
  return parity ? w1[c] : w1[4 - c];
}
// 5-point interpolation to the two children of the parent cell at p[0] (unit stride)
__device__ __forceinline__ void children(const double* p, double& lo, double& hi) {
  const double a = p[-2], b = p[-1], c = p[0], d = p[1], e = p[2];
  constexpr double w0 = 35.0 / 2048.0, w1 = -252.0 / 2048.0, w2 = 1890.0 / 2048.0, w3 = 420.0 / 2048.0,
                   w4 = -45.0 / 2048.0;
  hi = w0 * a + w1 * b + w2 * c + w3 * d + w4 * e;  // parity 1: +1/4
  lo = w4 * a + w3 * b + w2 * c + w1 * d + w0 * e;  // parity 0: -1/4
}

// shared-memory index of footprint cell (ia, ib, c) of a tile whose thin axis is AX: the layout the TMA box
// of that axis produces (x fastest)
template <int AX>
__device__ __forceinline__ int raw_idx(int ia, int ib, int c) {
  constexpr int PA = Geo<AX>::PA;
  if (AX == 2) return (c * PB + ib) * PA + ia;   // box (PA x, PB y, PT z)
  if (AX == 1) return (ib * PT + c) * PA + ia;   // box (PA x, PT y, PB z)
  return (ib * PA + ia) * PTX + c;               // box (PTX x, PA y, PB z); c counts from the even start
}

// geometry of one tile (box-local fine indices, parent-local footprint origin)
struct TileGeo {
  int axT, axA, axB;
  int oA, oB;              // even tile origin along A, B
  int vA0, vA1, vB0, vB1;  // valid tile-local fine range
  int q[3];                // parent-local index of footprint cell 0 along x, y, z
  int IT0, PT0, nt;        // level-global first thin cell, parent-global first footprint cell, thin cells
};
__device__ __forceinline__ int sel3(int ax, int x, int y, int z) { return ax == 0 ? x : (ax == 1 ? y : z); }
__device__ __forceinline__ TileGeo tile_geo(const BoxView& ch, const BoxView& pa, const GhostTile& t) {
  TileGeo g;  // (no dynamically indexed local arrays: they would live in local memory)
  g.axT = t.axis;
  g.axA = g.axT == 0 ? 1 : 0;
  g.axB = g.axT == 2 ? 1 : 2;
  const int tloA = sel3(g.axA, t.lo[0], t.lo[1], t.lo[2]), tloB = sel3(g.axB, t.lo[0], t.lo[1], t.lo[2]);
  const int tloT = sel3(g.axT, t.lo[0], t.lo[1], t.lo[2]);
  const int chA = sel3(g.axA, ch.lo[0], ch.lo[1], ch.lo[2]), chB = sel3(g.axB, ch.lo[0], ch.lo[1], ch.lo[2]);
  const int paA = sel3(g.axA, pa.lo[0], pa.lo[1], pa.lo[2]), paB = sel3(g.axB, pa.lo[0], pa.lo[1], pa.lo[2]);
  g.oA = sel3(g.axA, t.org[0], t.org[1], t.org[2]);
  g.oB = sel3(g.axB, t.org[0], t.org[1], t.org[2]);
  g.vA0 = tloA - g.oA; g.vA1 = g.vA0 + sel3(g.axA, t.n[0], t.n[1], t.n[2]);
  g.vB0 = tloB - g.oB; g.vB1 = g.vB0 + sel3(g.axB, t.n[0], t.n[1], t.n[2]);
  g.IT0 = sel3(g.axT, ch.lo[0], ch.lo[1], ch.lo[2]) + tloT;
  g.PT0 = (g.IT0 >> 1) - 2;
  g.nt = sel3(g.axT, t.n[0], t.n[1], t.n[2]);
  const int qA = ((chA + g.oA) >> 1) - 2 - paA, qB = ((chB + g.oB) >> 1) - 2 - paB;
  const int qT = g.PT0 - sel3(g.axT, pa.lo[0], pa.lo[1], pa.lo[2]);
  // axT = 2: (A, B, T) = (x, y, z);  axT = 1: (x, z, y);  axT = 0: (y, z, x)
  g.q[0] = g.axT == 0 ? qT : qA;
  g.q[1] = g.axT == 0 ? qA : (g.axT == 1 ? qT : qB);
  g.q[2] = g.axT == 2 ? qT : qB;
  return g;
}

// ---- phase 1: thin-axis interpolation of every source, then the time combination ---------------------
template <int AX, int NS, int NO>
__device__ __forceinline__ void phase1(const GhostProblem& pr, int nt, int xoff, const double* __restrict__ raw,
                                       double* __restrict__ T, const double (*sWt)[PT], int tid) {
  constexpr int PA = Geo<AX>::PA;
  if (tid >= PA * PB) return;
  const int ia = tid % PA, ib = tid / PA;
  double acc[NO][4];
#pragma unroll
  for (int o = 0; o < NO; ++o)
#pragma unroll
    for (int k = 0; k < 4; ++k) acc[o][k] = 0.0;
#pragma unroll
  for (int s = 0; s < NS; ++s) {
    double L[PT];
#pragma unroll
    for (int c = 0; c < PT; ++c) L[c] = raw[s * FOOTMAX + raw_idx<AX>(ia, ib, c) + (AX == 0 ? xoff : 0)];
    double v[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      double r = 0.0;
      if (k < nt) {
#pragma unroll
        for (int c = 0; c < PT; ++c) r = fma(sWt[k][c], L[c], r);
      }
      v[k] = r;
    }
#pragma unroll
    for (int o = 0; o < NO; ++o) {
      const double cf = pr.coef[o][s];
      if (cf != 0.0) {
#pragma unroll
        for (int k = 0; k < 4; ++k) acc[o][k] = fma(cf, v[k], acc[o][k]);
      }
    }
  }
#pragma unroll
  for (int o = 0; o < NO; ++o)
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if (k < nt) T[((o * nt + k) * PB + ib) * PAMAX + ia] = acc[o][k];
}

// ---- phase 2: interpolation along B, register-blocked ------------------------------------------------
template <int AX>
__device__ __forceinline__ void phase2(int nplanes, const double* __restrict__ T, double* __restrict__ U, int tid) {
  constexpr int PA = Geo<AX>::PA;
  for (int w = tid; w < nplanes * PA; w += NTHR) {
    const int ia = w % PA, pl = w / PA;
    const double* __restrict__ in = T + pl * (PB * PAMAX) + ia;
    double* __restrict__ out = U + pl * (TB * PAMAX) + ia;
    double v[PB];
#pragma unroll
    for (int j = 0; j < PB; ++j) v[j] = in[j * PAMAX];
#pragma unroll
    for (int j = 0; j < TB / 2; ++j) {
      double lo, hi;
      children(&v[j + 2], lo, hi);
      out[(2 * j) * PAMAX] = lo;
      out[(2 * j + 1) * PAMAX] = hi;
    }
  }
}

// ---- phase 3: interpolation along A and the store ----------------------------------------------------
// z- and y-slabs (A = x): thread (a-pair ja, fb) walks the planes; the two children are one 16-byte store.
template <int AX>
__device__ __forceinline__ void phase3(const GhostArgs& a, const GhostProblem& pr, int NO, const GhostTile& t,
                                       const TileGeo& g, int f, const double* __restrict__ U, int tid) {
  static_assert(AX != 0, "x-slabs have their own phase 3");
  const BoxView& ch = a.child;
  const int ja = tid % 16, fb = tid / 16, fa = 2 * ja;
  const bool v0 = fa >= g.vA0 && fa < g.vA1, v1 = fa + 1 >= g.vA0 && fa + 1 < g.vA1;
  if (fb < g.vB0 || fb >= g.vB1 || !(v0 || v1)) return;
  const int nt = g.nt;
  const double* __restrict__ up = U + fb * PAMAX + ja + 2;
  const int cA = g.oA + fa, cB = g.oB + fb;
  const long long cell = AX == 2 ? cell_offset(ch, cA, cB, t.lo[2]) : cell_offset(ch, cA, t.lo[1], cB);
  const long long csT = AX == 1 ? ch.px : ch.plane;
  for (int o = 0; o < NO; ++o) {
    if (o >= pr.nout) break;
    double* __restrict__ d = a.child_base + (long long)(pr.dst_arr[o] + f) * ch.vol + cell;
    double lo[4], hi[4];
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if (k < nt) children(up + (o * nt + k) * (TB * PAMAX), lo[k], hi[k]);
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if (k < nt) {
        if (v0 && v1) *reinterpret_cast<double2*>(d + k * csT) = make_double2(lo[k], hi[k]);
        else if (v0) d[k * csT] = lo[k];
        else d[k * csT + 1] = hi[k];
      }
  }
}

// x-slabs (thin = x, A = y): thread (fine row fa, fb) owns the g ghosts of one row and writes them as ONE
// whole 32-byte sector when it can: with g = 3 the low ghosts sit at row positions 1..3 (position 0 is an
// unused pad double), the high ghosts at XOFF+n .. XOFF+n+2 followed by a pad double when XOFF+n is a
// multiple of 4 — no sector is written partially.
__device__ __forceinline__ void phase3x(const GhostArgs& a, const GhostProblem& pr, int NO, const GhostTile& t,
                                        const TileGeo& g, int f, const double* __restrict__ U, int tid) {
  const BoxView& ch = a.child;
  const int fa = tid % 16, fb = tid / 16;
  if (fb < g.vB0 || fb >= g.vB1 || fa < g.vA0 || fa >= g.vA1) return;
  const int nt = g.nt;
  const double* __restrict__ up = U + fb * PAMAX + (fa >> 1) + 2;
  const bool odd = fa & 1;
  const long long cell = cell_offset(ch, t.lo[0], g.oA + fa, g.oB + fb);
  const bool lowside = t.lo[0] < 0;
  const bool sector = ch.g == 3 && nt == 3 && (lowside || ((XOFF + ch.n[0]) & 3) == 0);
  for (int o = 0; o < NO; ++o) {
    if (o >= pr.nout) break;
    double* __restrict__ d = a.child_base + (long long)(pr.dst_arr[o] + f) * ch.vol + cell;
    double v[4];
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if (k < nt) {
        double lo, hi;
        children(up + (o * nt + k) * (TB * PAMAX), lo, hi);
        v[k] = odd ? hi : lo;
      }
    if (sector) {
      if (lowside) {
        *reinterpret_cast<double2*>(d - 1) = make_double2(0.0, v[0]);
        *reinterpret_cast<double2*>(d + 1) = make_double2(v[1], v[2]);
      } else {
        *reinterpret_cast<double2*>(d) = make_double2(v[0], v[1]);
        *reinterpret_cast<double2*>(d + 2) = make_double2(v[2], 0.0);
      }
    } else {
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (k < nt) d[k] = v[k];
    }
  }
}

}  // namespace

// ---- the kernel ----------------------------------------------------------------------------------------
// dynamic shared memory: raw[GF_MAX_SRC][FOOTMAX] | T[GF_MAX_OUT * g][PB][PAMAX] | U[GF_MAX_OUT * g][TB][PAMAX]
__global__ void __launch_bounds__(NTHR, 2)
    ghost_fill_tma(const __grid_constant__ CUtensorMap mapx, const __grid_constant__ CUtensorMap mapy,
                   const __grid_constant__ CUtensorMap mapz, const __grid_constant__ GhostArgs a) {
  extern __shared__ unsigned char gsm_raw[];
  __shared__ double sWt[4][PT];  // thin-axis weights: fine thin cell k <- footprint cell c
  __shared__ __align__(8) unsigned long long sbar;
  const uint32_t s0 = (smem_u32g(gsm_raw) + 127u) & ~127u;
  double* const raw = reinterpret_cast<double*>(gsm_raw + (s0 - smem_u32g(gsm_raw)));
  const int maxplanes = GF_MAX_OUT * a.child.g;
  double* const T = raw + GF_MAX_SRC * FOOTMAX;
  double* const U = T + maxplanes * PB * PAMAX;
  const uint32_t bar = smem_u32g(&sbar);
  const int tid = threadIdx.x;
  const int per_prob = a.ntiles * a.F;
  const int nitems = a.nprob * per_prob;

  // one thread: arm the barrier and request the source footprints of an item
  auto issue = [&](int item) {
    const int p = item / per_prob, rem = item - p * per_prob;
    const int f = rem / a.ntiles, ti = rem - f * a.ntiles;
    const GhostTile t = a.tiles[ti];
    const TileGeo g = tile_geo(a.child, a.parent, t);
    const GhostProblem& pr = a.prob[p];
    const CUtensorMap* map = g.axT == 0 ? &mapx : (g.axT == 1 ? &mapy : &mapz);
    const int foot = g.axT == 0 ? Geo<0>::FOOT : FOOTMAX;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(pr.nsrc * foot * 8)
                 : "memory");
    const int cx = g.axT == 0 ? (XOFF + g.q[0]) & ~1 : XOFF + g.q[0];  // x-slabs: even start (XOFF is even)
    for (int s = 0; s < pr.nsrc; ++s)
      asm volatile(
          "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, "
          "%4, %5}], [%6];" ::"r"(s0 + s * FOOTMAX * 8),
          "l"(map), "r"(cx), "r"(a.parent.g + g.q[1]), "r"(a.parent.g + g.q[2]), "r"(pr.src_arr[s] + f),
          "r"(bar)
          : "memory");
  };
  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(1));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if ((int)blockIdx.x < nitems) issue(blockIdx.x);
  }
  __syncthreads();

  int it = 0;
  for (int item = blockIdx.x; item < nitems; item += gridDim.x, ++it) {
    const int p = item / per_prob, rem = item - p * per_prob;
    const int f = rem / a.ntiles, ti = rem - f * a.ntiles;
    const GhostTile t = a.tiles[ti];
    const TileGeo g = tile_geo(a.child, a.parent, t);
    const GhostProblem& pr = a.prob[p];
    const bool small = pr.nsrc <= 2 && pr.nout <= 2;
    if (tid < 4 * PT) {
      const int kt = tid / PT, c = tid % PT;
      double w = 0.0;
      if (kt < g.nt) {
        const int Ig = g.IT0 + kt;
        const int d = c - ((Ig >> 1) - g.PT0 - 2);  // offset from the first stencil cell of thin cell kt
        if (d >= 0 && d < 5) w = wprol(Ig & 1, d);
      }
      sWt[kt][c] = w;
    }
    __syncthreads();
    mbar_wait_g(bar, it & 1);
    // phase 1 (the footprints have landed)
    const int xoff = g.q[0] & 1;  // x-slabs: footprint cell 0 sits at this offset of the loaded row
    if (small) {
      if (g.axT == 2) phase1<2, 2, 2>(pr, g.nt, 0, raw, T, sWt, tid);
      else if (g.axT == 1) phase1<1, 2, 2>(pr, g.nt, 0, raw, T, sWt, tid);
      else phase1<0, 2, 2>(pr, g.nt, xoff, raw, T, sWt, tid);
    } else {
      if (g.axT == 2) phase1<2, GF_MAX_SRC, GF_MAX_OUT>(pr, g.nt, 0, raw, T, sWt, tid);
      else if (g.axT == 1) phase1<1, GF_MAX_SRC, GF_MAX_OUT>(pr, g.nt, 0, raw, T, sWt, tid);
      else phase1<0, GF_MAX_SRC, GF_MAX_OUT>(pr, g.nt, xoff, raw, T, sWt, tid);
    }
    __syncthreads();  // raw is free again, T is complete
    if (tid == 0 && item + (int)gridDim.x < nitems) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      issue(item + gridDim.x);
    }
    const int NO = small ? 2 : GF_MAX_OUT;  // planes are laid out for NO outputs (unused ones hold zeros)
    if (g.axT == 0) phase2<0>(NO * g.nt, T, U, tid);
    else phase2<2>(NO * g.nt, T, U, tid);
    __syncthreads();
    if (g.axT == 0) phase3x(a, pr, NO, t, g, f, U, tid);
    else if (g.axT == 1) phase3<1>(a, pr, NO, t, g, f, U, tid);
    else phase3<2>(a, pr, NO, t, g, f, U, tid);
  }
}

// ---- host ---------------------------------------------------------------------------------------------
namespace {
struct Piece { int lo, n, org; };
// cut [r0, r1) into pieces of a grid of period T whose origin o <= r0 is the largest with (base + o) a
// multiple of `align` (base = level-global index of box-local 0)
void cut(int r0, int r1, int T, int base, int align, std::vector<Piece>& out) {
  out.clear();
  int o = r0;
  while (((base + o) % align + align) % align != 0) --o;
  for (int s = o; s < r1; s += T) {
    const int lo = s < r0 ? r0 : s, hi = s + T < r1 ? s + T : r1;
    if (hi > lo) out.push_back({lo, hi - lo, s});
  }
}
}  // namespace

// Tile origins are even in y and z (so a tile covers whole parent cells) and a multiple of 4 in x in
// LEVEL-GLOBAL index: the parent footprint of an x-extended tile then starts at an even parent x index,
// i.e. on a 16-byte boundary (XOFF and lo are even) — TMA loads of 160-byte box rows from an odd fp64
// coordinate fault on sm_100a ("illegal instruction", measured; 48-byte rows do not).
void build_ghost_tiles(const BoxView& ch, std::vector<GhostTile>& tiles) {
  tiles.clear();
  const int g = ch.g;
  std::vector<Piece> as, bs;
  // z-slabs: A = x over the padded extent, B = y over the padded extent
  cut(-g, ch.n[0] + g, Geo<2>::TA, ch.lo[0], 4, as);
  cut(-g, ch.n[1] + g, TB, ch.lo[1], 2, bs);
  for (int hi = 0; hi < 2; ++hi)
    for (auto& b : bs)
      for (auto& x : as) {
        const int z = hi ? ch.n[2] : -g;
        tiles.push_back(GhostTile{{x.lo, b.lo, z}, {x.n, b.n, g}, {x.org, b.org, z}, 2});
      }
  // y-slabs: A = x padded, B = z interior
  cut(0, ch.n[2], TB, ch.lo[2], 2, bs);
  for (int hi = 0; hi < 2; ++hi)
    for (auto& b : bs)
      for (auto& x : as) {
        const int y = hi ? ch.n[1] : -g;
        tiles.push_back(GhostTile{{x.lo, y, b.lo}, {x.n, g, b.n}, {x.org, y, b.org}, 1});
      }
  // x-slabs: A = y interior, B = z interior
  cut(0, ch.n[1], Geo<0>::TA, ch.lo[1], 2, as);
  for (int hi = 0; hi < 2; ++hi)
    for (auto& b : bs)
      for (auto& y : as) {
        const int x = hi ? ch.n[0] : -g;
        tiles.push_back(GhostTile{{x, y.lo, b.lo}, {g, y.n, b.n}, {x, y.org, b.org}, 0});
      }
  if (const char* e = getenv("SC_DBG_TILE")) {  // DEBUG
    int lo = 0, hi = 1 << 30;
    sscanf(e, "%d:%d", &lo, &hi);
    std::vector<GhostTile> keep;
    for (int i = 0; i < (int)tiles.size(); ++i) if (i >= lo && i < hi) keep.push_back(tiles[i]);
    tiles = keep;
  }
}

void ghost_box_dims(int axis, unsigned box[4]) {
  box[0] = axis == 0 ? PTX : Geo<2>::PA;
  box[1] = axis == 0 ? Geo<0>::PA : (axis == 1 ? PT : PB);
  box[2] = axis == 2 ? PT : PB;
  box[3] = 1;
}

// problems the tuned kernel takes: exactly the (5 -> 4) and (<= 2 -> <= 2) shapes the scheduler produces
bool ghost_tma_takes(const GhostArgs& a) {
  if (!a.tmaps || a.ntiles == 0 || a.child.g > 4) return false;
  for (int p = 0; p < a.nprob; ++p) {
    const GhostProblem& pr = a.prob[p];
    const bool small = pr.nsrc <= 2 && pr.nout <= 2;
    if (!small && pr.nsrc != GF_MAX_SRC) return false;  // the TMA transaction count is per real source
    if (pr.nsrc < 1 || pr.nout < 1) return false;
  }
  return true;
}

void launch_ghost_fill_tma(const GhostArgs& a, cudaStream_t st) {
  static const int nsm = [] {
    int dev = 0, n = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
    return n > 0 ? n : 148;
  }();
  const int maxplanes = GF_MAX_OUT * a.child.g;
  const size_t smem = 128 + sizeof(double) * ((size_t)GF_MAX_SRC * FOOTMAX + (size_t)maxplanes * (PB * PAMAX + TB * PAMAX));
  static size_t configured = 0;
  if (smem > configured) {
    cudaFuncSetAttribute(ghost_fill_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    configured = smem;
  }
  const long long nitems = (long long)a.nprob * a.ntiles * a.F;
  const int per_sm = smem <= 112 * 1024 ? 2 : 1;
  const unsigned grid = (unsigned)(nitems < (long long)nsm * per_sm ? nitems : (long long)nsm * per_sm);
  const CUtensorMap* m = static_cast<const CUtensorMap*>(a.tmaps);
  ghost_fill_tma<<<grid, NTHR, smem, st>>>(m[0], m[1], m[2], a);
}

}  // namespace sc
