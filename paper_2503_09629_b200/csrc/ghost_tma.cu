// ghost_tma.cu — tuned refinement-boundary ghost fill (eqs 10-18 folded
// into the coefficient matrices by the scheduler; spatial operator = reading S3), sm_100a.
//
//   child array dst_arr[o](ghost cell) = P[ sum_s coef[o][s] * parent array src_arr[s] ],   P = 5x5x5 quartic Lagrange
//
// The ghost shell of a box is the union of six slabs (z-lo, z-hi, y-lo, y-hi, x-lo, x-hi); each slab is cut
// into tiles  g (thin axis) x 32 (A) x 16 (B)  fine cells whose origin is even in every axis, so a tile covers
// whole parent cells and its parent footprint is exactly 20 x 12 x 6 cells (x-slabs: rows of 8, see below). The
// host precomputes one 64-byte descriptor per tile (index maps, TMA coordinates, ragged-edge ranges, store
// mode). A work ITEM is (problem, field, tile). Persistent CTAs (two per SM, equal item counts) walk the item
// list; per item
//   0. the footprint of every source array arrives in shared memory through ONE TMA tiled load per source
//      (cp.async.bulk.tensor.4d on the parent's footprint tensor map, out-of-range cells zero-filled),
//      requested one item AHEAD so it flies while the current item is interpolated; the descriptor of the
//      next item comes by cp.async, so no global load sits on a warp's path into a barrier;
//   1. one thread per parent column: thin-axis interpolation (6 parent cells -> g fine cells; for g = 3 the
//      weights are compile-time constants chosen by the parity of the first thin cell) of every source,
//      then the time combination into the outputs             -> T[plane = (o, thin cell)][b][a]
//   2. both transverse interpolations and the store in ONE pass that never returns to shared memory: thread
//      (plane, parent column) marches along b; each T row is interpolated along a to the column's two children
//      and pushed into a 5-row register window, from which every step produces two fine rows. z- and y-slabs
//      (a = x): a row pair is one 16-byte store, 512 contiguous bytes per warp. x-slabs (thin = x): the four
//      lanes (3 ghosts + 1 pad double) of a row are adjacent lanes and write ONE whole 32-byte sector.
// A ghost value costs 6 + 5 + 5 FMA instead of 125 and every parent value is fetched once per tile.
// Measured (r01, profiles/r01_v4.md): 256^3 child box, (5 -> 4) problem 25 us, with the (2 -> 2) problem 38 us
// (v3 with separate b- and a-passes through shared memory: 31 / 42 us). What the profiles showed on the way:
//   * an empty launch of this grid already costs 6 us between its two events;
//   * the kernel is sensitive to instruction fetch: with phase 2's 12-step march unrolled (12 KB of straight-
//     line code per variant) 35-50 % of the stall samples were stall_no_inst and the launch took 44 us; rolled
//     (20 register moves per step) 40 us; with phase 1's source loop rolled as well 35.6 us; a 5-way unrolled
//     rotating window without moves was slower again (43.7 us);
//   * the x-slab footprint rows (64 B each) are read by one thread per row: unswizzled that is a 16-way bank
//     conflict (2.7 M conflict wavefronts per launch), hence the SWIZZLE_64B tensor map;
//   * doubling the CTA to 512 threads (half the outputs per thread) and programmatic dependent launch of the
//     whole kernel chain both made the step slower (48.8 us per launch; 22.0 -> 22.8 ms per coarse step).
#include <cuda.h>

#include <cstdlib>

#include "kernels.h"
#include "launch_cfg.h"
#include "pdl.h"

namespace sc {

void launch_ghost_fill_direct(const GhostArgs& a, cudaStream_t st);

namespace {

// Tile geometry per thin axis AX: 32 x 16 fine cells along (A, B). x-slabs (A = y, thin = x): the footprint's
// x extent is loaded as 8 doubles from an EVEN x coordinate — a TMA tiled load whose innermost fp64
// coordinate is odd (start not 16-byte aligned) faults on sm_100a (measured) — through a SWIZZLE_64B tensor
// map: the 64-byte rows land with their 16-byte chunks XOR-ed by bits 1-2 of the row index, so that phase 1's
// one-thread-per-row 16-byte loads are bank-conflict free.
constexpr int TA = 32, PA = TA / 2 + 4;          // fine cells / parent footprint along A (2-cell halo each side)
constexpr int TB = 16, PB = TB / 2 + 4;          // ... along B
constexpr int PT = 6;                            // parent cells along the thin axis (ghost width <= 4)
constexpr int PTX = 8;                           // ... as loaded for x-slabs (even start, 64-byte rows)
constexpr int PAMAX = PA;                        // pitch of a T row
constexpr int TPLANE = PB * PAMAX + 4;           // pitch of a T plane: 8 banks past a multiple of 32 (x-slab lanes)
template <int AX> struct Geo {
  static constexpr int FOOT = AX == 0 ? PTX * PA * PB : PA * PB * PT;  // doubles per source footprint
};
constexpr int FOOTMAX = Geo<0>::FOOT;            // 1920 doubles = 15360 B: stride between sources in smem
constexpr int NTHR = 256;
static_assert(Geo<1>::FOOT <= FOOTMAX && Geo<2>::FOOT <= FOOTMAX, "source slots are FOOTMAX doubles");
static_assert(PA * PB <= NTHR, "phase 1: one thread per parent column");
static_assert((TA / 2) * GF_MAX_OUT * 4 == NTHR, "phase 2: thread = (output, thin cell, parent column)");
static_assert((FOOTMAX * 8) % 1024 == 0, "TMA destination alignment (swizzle atom)");
static_assert((TPLANE * 2) % 32 == 8, "x-slab phase 2: the four thin-cell lanes of a column hit distinct banks");

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

// shared-memory index of footprint cell (ia, ib, c) of a tile whose thin axis is AX (1 or 2): the layout the
// TMA box of that axis produces (x fastest)
template <int AX>
__device__ __forceinline__ int raw_idx(int ia, int ib, int c) {
  static_assert(AX != 0, "x-slab rows are read as swizzled 16-byte chunks");
  if (AX == 2) return (c * PB + ib) * PA + ia;   // box (PA x, PB y, PT z)
  return (ib * PT + c) * PA + ia;                // box (PA x, PT y, PB z)
}

// ---- phase 1: thin-axis interpolation of every source, then the time combination ---------------------
// 5-point thin-axis interpolation with immediate weights (P = parity of the fine cell), depth-3 tree
template <int P>
__device__ __forceinline__ double ip5(const double* L) {
  constexpr double w0 = 35.0 / 2048.0, w1 = -252.0 / 2048.0, w2 = 1890.0 / 2048.0, w3 = 420.0 / 2048.0,
                   w4 = -45.0 / 2048.0;
  if (P) return fma(w4, L[4], fma(w1, L[1], w0 * L[0])) + fma(w3, L[3], w2 * L[2]);
  return fma(w0, L[4], fma(w3, L[1], w4 * L[0])) + fma(w1, L[3], w2 * L[2]);
}
// PAR >= 0: ghost width 3 and PAR = parity of the first thin cell: the (parent cell, parity) pattern of the
// three thin cells is known at compile time (no weight table, no barrier). PAR < 0: any width, weights in sWt.
// XO (x-slabs): position of footprint cell 0 inside the loaded 8-wide row.
template <int AX, int NS, int NO, int PAR, int XO>
__device__ __forceinline__ void phase1(const GhostProblem& pr, int nt, const double* __restrict__ raw,
                                       double* __restrict__ T, const double (*sWt)[PT], int tid) {
  if (tid >= PA * PB) return;
  const int ia = tid % PA, ib = tid / PA;
  double acc[NO][4];
#pragma unroll
  for (int o = 0; o < NO; ++o)
#pragma unroll
    for (int k = 0; k < 4; ++k) acc[o][k] = 0.0;
#pragma unroll 1
  for (int s = 0; s < NS; ++s) {  // rolled: the kernel is sensitive to instruction fetch (see phase 2)
    double L[PT];
    if (AX == 0) {  // row tid of the (PTX x, PA y, PB z) box; chunk q sits at q ^ bits 1-2 of the row (SWIZZLE_64B)
      const double2* __restrict__ row = reinterpret_cast<const double2*>(raw + s * FOOTMAX) + tid * 4;
      const int sw = (tid >> 1) & 3;
      double d[PTX];
#pragma unroll
      for (int q = 0; q < (XO ? 4 : 3); ++q) {
        const double2 t2 = row[q ^ sw];
        d[2 * q] = t2.x;
        d[2 * q + 1] = t2.y;
      }
#pragma unroll
      for (int c = 0; c < PT; ++c) L[c] = d[c + XO];
    } else {
#pragma unroll
      for (int c = 0; c < PT; ++c) L[c] = raw[s * FOOTMAX + raw_idx<AX == 0 ? 1 : AX>(ia, ib, c)];
    }
    double v[4];
    if (PAR == 0) {         // first thin cell even: (j, parity) = (2,0), (2,1), (3,0)
      v[0] = ip5<0>(L); v[1] = ip5<1>(L); v[2] = ip5<0>(L + 1); v[3] = 0.0;
    } else if (PAR == 1) {  // odd: (2,1), (3,0), (3,1)
      v[0] = ip5<1>(L); v[1] = ip5<0>(L + 1); v[2] = ip5<1>(L + 1); v[3] = 0.0;
    } else {
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        double r = 0.0;
        if (k < nt) {
#pragma unroll
          for (int c = 0; c < PT; ++c) r = fma(sWt[k][c], L[c], r);
        }
        v[k] = r;
      }
    }
#pragma unroll
    for (int o = 0; o < NO; ++o) {
      const double cf = pr.coef[o][s];
      // small shape: a slot beyond nsrc holds stale data (possibly NaN) and has coefficient 0 -> skip it
      if (NS == GF_MAX_SRC || cf != 0.0) {
#pragma unroll
        for (int k = 0; k < (PAR >= 0 ? 3 : 4); ++k) acc[o][k] = fma(cf, v[k], acc[o][k]);
      }
    }
  }
#pragma unroll
  for (int o = 0; o < NO; ++o)
#pragma unroll
    for (int k = 0; k < (PAR >= 0 ? 3 : 4); ++k)
      if (k < nt) T[(o * (PAR >= 0 ? 3 : nt) + k) * TPLANE + ib * PAMAX + ia] = acc[o][k];
}
template <int AX, int NS, int NO, int XO>
__device__ __forceinline__ void phase1_par(int par, const GhostProblem& pr, int nt, const double* __restrict__ raw,
                                           double* __restrict__ T, const double (*sWt)[PT], int tid) {
  if (par == 0) phase1<AX, NS, NO, 0, XO>(pr, nt, raw, T, sWt, tid);
  else if (par == 1) phase1<AX, NS, NO, 1, XO>(pr, nt, raw, T, sWt, tid);
  else phase1<AX, NS, NO, -1, XO>(pr, nt, raw, T, sWt, tid);
}
template <int NS, int NO>
__device__ __forceinline__ void phase1_any(const GhostTile& t, const GhostProblem& pr, const double* __restrict__ raw,
                                           double* __restrict__ T, const double (*sWt)[PT], int tid) {
  if (t.axis == 2) phase1_par<2, NS, NO, 0>(t.par, pr, t.nt, raw, T, sWt, tid);
  else if (t.axis == 1) phase1_par<1, NS, NO, 0>(t.par, pr, t.nt, raw, T, sWt, tid);
  else if (t.xoff) phase1_par<0, NS, NO, 1>(t.par, pr, t.nt, raw, T, sWt, tid);
  else phase1_par<0, NS, NO, 0>(t.par, pr, t.nt, raw, T, sWt, tid);
}

// ---- phase 2: the two transverse interpolations and the store, marching along B in registers ----------
// children of the centre of a 5-value window held in registers
__device__ __forceinline__ void children5(const double (&w)[5], double& lo, double& hi) {
  constexpr double w0 = 35.0 / 2048.0, w1 = -252.0 / 2048.0, w2 = 1890.0 / 2048.0, w3 = 420.0 / 2048.0,
                   w4 = -45.0 / 2048.0;
  hi = fma(w4, w[4], fma(w1, w[1], w0 * w[0])) + fma(w3, w[3], w2 * w[2]);
  lo = fma(w0, w[4], fma(w3, w[1], w4 * w[0])) + fma(w1, w[3], w2 * w[2]);
}
// z- and y-slabs (A = x): thread = (plane = (output, thin cell), parent column ja). It walks the PB parent rows of
// its plane of T: each row is interpolated along A to the column's two children (5 shared loads, 10 FMA) and
// pushed into a 5-row register window; once the window is full every new row yields two fine rows (20 FMA), each
// stored as one 16-byte pair — 512 contiguous bytes per warp and store. Nothing goes back through shared memory.
// The march is a rolled loop on purpose: unrolled, the phase is 12 KB of straight-line code per variant and the
// kernel stalls on instruction fetch (measured: stall_no_inst 35-50 % of the samples).
__device__ __forceinline__ void push_row(const double* __restrict__ p, double (&wl)[5], double (&wh)[5]) {
#pragma unroll
  for (int i = 0; i < 4; ++i) { wl[i] = wl[i + 1]; wh[i] = wh[i + 1]; }
  children(p, wl[4], wh[4]);
}
__device__ __forceinline__ void phase2(const GhostArgs& a, const GhostProblem& pr, const GhostTile& t, int f,
                                       const double* __restrict__ T, int tid) {
  const BoxView& ch = a.child;
  const int ja = tid & 15, pl = tid >> 4, nt = t.nt;
  if (pl >= pr.nout * nt) return;
  const int o = pl / nt, k = pl - o * nt, fa = 2 * ja;
  const bool full = t.vA0 == 0 && t.vB0 == 0 && t.vB1 == TB && t.vA1 == TA;
  const bool v0 = fa >= t.vA0 && fa < t.vA1, v1 = fa + 1 >= t.vA0 && fa + 1 < t.vA1;
  if (!(v0 || v1)) return;
  const long long csT = t.axis == 1 ? ch.px : ch.plane, csB = t.axis == 1 ? ch.plane : ch.px;
  double* __restrict__ d = a.child_base + (long long)(pr.dst_arr[o] + f) * ch.vol + t.cell0 + fa + k * csT;
  const double* __restrict__ tp = T + pl * TPLANE + ja + 2;
  double wl[5], wh[5];
#pragma unroll
  for (int i = 0; i < 5; ++i) wl[i] = wh[i] = 0.0;
#pragma unroll 1
  for (int jb = 0; jb < 4; ++jb, tp += PAMAX) push_row(tp, wl, wh);
#pragma unroll 1
  for (int fb = 0; fb < TB; fb += 2, tp += PAMAX, d += 2 * csB) {
    push_row(tp, wl, wh);
    double l0, l1, h0, h1;
    children5(wl, l0, l1);  // fine rows fb (l0), fb + 1 (l1) of fine column fa
    children5(wh, h0, h1);  // ... of fine column fa + 1
    double* __restrict__ r1 = d + csB;
    if (full) {
      *reinterpret_cast<double2*>(d) = make_double2(l0, h0);
      *reinterpret_cast<double2*>(r1) = make_double2(l1, h1);
    } else {
      if (fb >= t.vB0 && fb < t.vB1) {
        if (v0 && v1) *reinterpret_cast<double2*>(d) = make_double2(l0, h0);
        else if (v0) d[0] = l0;
        else d[1] = h0;
      }
      if (fb + 1 >= t.vB0 && fb + 1 < t.vB1) {
        if (v0 && v1) *reinterpret_cast<double2*>(r1) = make_double2(l1, h1);
        else if (v0) r1[0] = l1;
        else r1[1] = h1;
      }
    }
  }
}

// x-slabs (thin = x, A = y, B = z): thread = (output, parent column ja, lane kk of four); the four kk lanes of a
// column are adjacent lanes of a warp and own the four doubles of the 32-byte sector that holds the g = 3
// ghosts of a row plus one unused pad double (low side: pad first; high side: pad last, when XOFF + n is a
// multiple of 4 — t.sector, decided on the host), so every store instruction writes whole sectors. The pad lane
// computes nothing and stores 0. Other widths (t.sector = 0): lane kk stores thin cell kk.
__device__ __forceinline__ void phase2x(const GhostArgs& a, const GhostProblem& pr, const GhostTile& t, int f,
                                        const double* __restrict__ T, int tid) {
  const BoxView& ch = a.child;
  const int kk = tid & 3, ja = (tid >> 2) & 15, o = tid >> 6, nt = t.nt, fa = 2 * ja;
  if (o >= pr.nout) return;
  const int kt = kk - (t.sector == 1);  // thin cell of this lane
  const bool comp = kt >= 0 && kt < nt;
  if (!comp && t.sector == 0) return;
  const bool v0 = fa >= t.vA0 && fa < t.vA1, v1 = fa + 1 >= t.vA0 && fa + 1 < t.vA1;
  if (!(v0 || v1)) return;
  double* __restrict__ d = a.child_base + (long long)(pr.dst_arr[o] + f) * ch.vol + t.cell0 + (long long)fa * ch.px + kt;
  const double* __restrict__ tp = T + (o * nt + (comp ? kt : 0)) * TPLANE + ja + 2;
  double wl[5], wh[5];
#pragma unroll
  for (int i = 0; i < 5; ++i) wl[i] = wh[i] = 0.0;
  if (comp) {
#pragma unroll 1
    for (int jb = 0; jb < 4; ++jb, tp += PAMAX) push_row(tp, wl, wh);
  }
#pragma unroll 1
  for (int fb = 0; fb < TB; fb += 2, tp += PAMAX, d += 2 * ch.plane) {
    double l0 = 0.0, l1 = 0.0, h0 = 0.0, h1 = 0.0;
    if (comp) {
      push_row(tp, wl, wh);
      children5(wl, l0, l1);  // fine z rows fb, fb + 1 of fine y row fa
      children5(wh, h0, h1);  // ... of fine y row fa + 1
    }
    double* __restrict__ r1 = d + ch.plane;
    if (fb >= t.vB0 && fb < t.vB1) {
      if (v0) d[0] = l0;
      if (v1) d[ch.px] = h0;
    }
    if (fb + 1 >= t.vB0 && fb + 1 < t.vB1) {
      if (v0) r1[0] = l1;
      if (v1) r1[ch.px] = h1;
    }
  }
}

}  // namespace

// ---- the kernel ----------------------------------------------------------------------------------------
// dynamic shared memory (1024-byte aligned): raw[GF_MAX_SRC][FOOTMAX] | T[GF_MAX_OUT * g][TPLANE]
__global__ void __launch_bounds__(NTHR, 2)
    ghost_fill_tma(const __grid_constant__ CUtensorMap mapx, const __grid_constant__ CUtensorMap mapy,
                   const __grid_constant__ CUtensorMap mapz, const __grid_constant__ GhostArgs a) {
  pdl_enter();
  extern __shared__ unsigned char gsm_raw[];
  __shared__ double sWt[4][PT];  // thin-axis weights (ghost widths other than 3): thin cell k <- footprint cell c
  __shared__ __align__(8) unsigned long long sbar;
  __shared__ __align__(16) GhostTile sTile[2];  // tile descriptors of the current and the next item
  const uint32_t s0 = (smem_u32g(gsm_raw) + 1023u) & ~1023u;
  double* const raw = reinterpret_cast<double*>(gsm_raw + (s0 - smem_u32g(gsm_raw)));
  double* const T = raw + GF_MAX_SRC * FOOTMAX;
  const uint32_t bar = smem_u32g(&sbar);
  const int tid = threadIdx.x;
  const int per_prob = a.ntiles * a.F;
  const int nitems = a.nprob * per_prob;

  auto tile_index = [&](int item) { return (item % per_prob) % a.ntiles; };
  // one thread: arm the barrier and request the source footprints of an item (descriptor already on chip)
  auto issue = [&](int item, const GhostTile& t) {
    const int p = item / per_prob, f = (item - p * per_prob) / a.ntiles;
    const GhostProblem& pr = a.prob[p];
    const CUtensorMap* map = t.axis == 0 ? &mapx : (t.axis == 1 ? &mapy : &mapz);
    const int foot = t.axis == 0 ? Geo<0>::FOOT : Geo<2>::FOOT;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(pr.nsrc * foot * 8)
                 : "memory");
    for (int s = 0; s < pr.nsrc; ++s)
      asm volatile(
          "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, "
          "%4, %5}], [%6];" ::"r"(s0 + s * FOOTMAX * 8),
          "l"(map), "r"(t.cx), "r"(t.cy), "r"(t.cz), "r"(pr.src_arr[s] + f), "r"(bar)
          : "memory");
  };
  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(1));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if ((int)blockIdx.x < nitems) {
      sTile[0] = a.tiles[tile_index(blockIdx.x)];
      issue(blockIdx.x, sTile[0]);
    }
  }
  __syncthreads();

  int it = 0;
  for (int item = blockIdx.x; item < nitems; item += gridDim.x, ++it) {
    const int p = item / per_prob, f = (item - p * per_prob) / a.ntiles;
    const GhostTile t = sTile[it & 1];
    const bool more = item + (int)gridDim.x < nitems;
    // next descriptor -> the other slot, asynchronously: no global load sits on any warp's path into a barrier
    if (tid >= 32 && tid < 36 && more) {
      const char* src = reinterpret_cast<const char*>(a.tiles + tile_index(item + gridDim.x)) + 16 * (tid - 32);
      const uint32_t dst = smem_u32g(&sTile[(it + 1) & 1]) + 16 * (tid - 32);
      asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
    }
    const GhostProblem& pr = a.prob[p];
    const bool small = pr.nsrc <= 2 && pr.nout <= 2;
    if (t.par < 0) {  // ghost width != 3: weight table (CTA-uniform branch)
      if (tid < 4 * PT) {
        const int kt = tid / PT, c = tid % PT;
        double w = 0.0;
        if (kt < t.nt) {
          const int Ig = t.IT0 + kt;
          const int d = c - ((Ig >> 1) - (t.IT0 >> 1));  // offset from the first stencil cell of thin cell kt
          if (d >= 0 && d < 5) w = wprol(Ig & 1, d);
        }
        sWt[kt][c] = w;
      }
      __syncthreads();
    }
    mbar_wait_g(bar, it & 1);
    // phase 1 (the footprints have landed); T planes are laid out per output (o * nt + k)
    if (small) phase1_any<2, 2>(t, pr, raw, T, sWt, tid);
    else phase1_any<GF_MAX_SRC, GF_MAX_OUT>(t, pr, raw, T, sWt, tid);
    if (tid >= 32 && tid < 36) asm volatile("cp.async.wait_all;" ::: "memory");
    __syncthreads();  // raw is free again, T is complete, the next descriptor is in sTile
    if (tid == 0 && more) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      issue(item + gridDim.x, sTile[(it + 1) & 1]);
    }
    if (t.axis == 0) phase2x(a, pr, t, f, T, tid);
    else phase2(a, pr, t, f, T, tid);
    __syncthreads();  // T may be overwritten by the next item's phase 1
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

namespace {
// Descriptor of the piece [lo, lo + n) of the tile-grid cell at `org` (box-local fine indices) of a slab with
// thin axis axT. Index maps: fine cell I (level-global) has parent I >> 1 (S1); the footprint starts 2 parent
// cells before the first covered parent cell along every axis.
GhostTile make_tile(const BoxView& ch, const BoxView& pa, int axT, const int lo[3], const int n[3], const int org[3]) {
  const int axA = axT == 0 ? 1 : 0, axB = axT == 2 ? 1 : 2;  // (A, B, T) = (x,y,z) | (x,z,y) | (y,z,x)
  GhostTile t{};
  t.axis = axT;
  t.nt = n[axT];
  t.IT0 = ch.lo[axT] + lo[axT];
  t.par = t.nt == 3 ? (t.IT0 & 1) : -1;
  t.vA0 = lo[axA] - org[axA]; t.vA1 = t.vA0 + n[axA];
  t.vB0 = lo[axB] - org[axB]; t.vB1 = t.vB0 + n[axB];
  int q[3];  // parent-local index of footprint cell 0
  q[axA] = ((ch.lo[axA] + org[axA]) >> 1) - 2 - pa.lo[axA];
  q[axB] = ((ch.lo[axB] + org[axB]) >> 1) - 2 - pa.lo[axB];
  q[axT] = (t.IT0 >> 1) - 2 - pa.lo[axT];
  t.cx = XOFF + q[0];
  t.xoff = 0;
  if (axT == 0) { t.xoff = t.cx & 1; t.cx &= ~1; }  // x-slabs: 8-wide rows from an even start
  t.cy = pa.g + q[1];
  t.cz = pa.g + q[2];
  const bool lowside = lo[0] < 0;
  t.sector = (axT == 0 && ch.g == 3 && t.nt == 3) ? (lowside ? 1 : (((XOFF + ch.n[0]) & 3) == 0 ? 2 : 0)) : 0;
  int c0[3];
  c0[axT] = lo[axT]; c0[axA] = org[axA]; c0[axB] = org[axB];
  t.cell0 = cell_offset(ch, c0[0], c0[1], c0[2]);
  return t;
}
}  // namespace

// Tile origins are even in y and z (so a tile covers whole parent cells) and a multiple of 4 in x in
// LEVEL-GLOBAL index: the parent footprint of an x-extended tile then starts at an even parent x index,
// i.e. on a 16-byte boundary (XOFF and lo are even) — a TMA tiled load whose innermost fp64 coordinate is
// odd faults on sm_100a ("illegal instruction", measured).
void build_ghost_tiles(const BoxView& ch, const BoxView& pa, std::vector<GhostTile>& tiles,
                       const std::vector<BoxView>* siblings) {
  tiles.clear();
  const int g = ch.g;
  std::vector<Piece> as, bs;
  auto push = [&](int ax, int l0, int l1, int l2, int n0, int n1, int n2, int o0, int o1, int o2) {
    const int lo[3] = {l0, l1, l2}, n[3] = {n0, n1, n2}, org[3] = {o0, o1, o2};
    if (siblings)
      for (const BoxView& s : *siblings) {
        bool inside = true;
        for (int a = 0; a < 3; ++a)
          if (ch.lo[a] + lo[a] < s.lo[a] || ch.lo[a] + lo[a] + n[a] > s.lo[a] + s.n[a]) inside = false;
        if (inside) return;  // the exchange supplies every cell of this tile
      }
    tiles.push_back(make_tile(ch, pa, ax, lo, n, org));
  };
  // z-slabs: A = x over the padded extent, B = y over the padded extent
  cut(-g, ch.n[0] + g, TA, ch.lo[0], 4, as);
  cut(-g, ch.n[1] + g, TB, ch.lo[1], 2, bs);
  for (int hi = 0; hi < 2; ++hi)
    for (auto& b : bs)
      for (auto& x : as) {
        const int z = hi ? ch.n[2] : -g;
        push(2, x.lo, b.lo, z, x.n, b.n, g, x.org, b.org, z);
      }
  // y-slabs: A = x padded, B = z interior
  cut(0, ch.n[2], TB, ch.lo[2], 2, bs);
  for (int hi = 0; hi < 2; ++hi)
    for (auto& b : bs)
      for (auto& x : as) {
        const int y = hi ? ch.n[1] : -g;
        push(1, x.lo, y, b.lo, x.n, g, b.n, x.org, y, b.org);
      }
  // x-slabs: A = y interior, B = z interior
  cut(0, ch.n[1], TA, ch.lo[1], 2, as);
  for (int hi = 0; hi < 2; ++hi)
    for (auto& b : bs)
      for (auto& y : as) {
        const int x = hi ? ch.n[0] : -g;
        push(0, x, y.lo, b.lo, g, y.n, b.n, x, y.org, b.org);
      }
}

void ghost_box_dims(int axis, unsigned box[4]) {
  box[0] = axis == 0 ? PTX : PA;
  box[1] = axis == 0 ? PA : (axis == 1 ? PT : PB);
  box[2] = axis == 2 ? PT : PB;
  box[3] = 1;
}

bool ghost_tma_geometry_ok(const BoxView& child) { return child.g <= 4; }

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
  const int nsm = device_sm_count();
  const int maxplanes = GF_MAX_OUT * a.child.g;
  const size_t smem = 1024 + sizeof(double) * ((size_t)GF_MAX_SRC * FOOTMAX + (size_t)maxplanes * TPLANE);
  ensure_dynamic_smem(ghost_fill_tma, smem);
  const long long nitems = (long long)a.nprob * a.ntiles * a.F;
  const int per_sm = smem <= 112 * 1024 ? 2 : 1;
  const long long want = (long long)nsm * per_sm;
  // equal item counts per CTA: with R = ceil(nitems / want) rounds, ceil(nitems / R) CTAs all do R items (+-1)
  const long long rounds = (nitems + want - 1) / want;
  const unsigned grid = (unsigned)(nitems <= want ? nitems : (nitems + rounds - 1) / rounds);
  const CUtensorMap* m = static_cast<const CUtensorMap*>(a.tmaps);
  launch_pdl(ghost_fill_tma, dim3(grid), dim3(NTHR), smem, st, m[0], m[1], m[2], a);
}

}  // namespace sc
