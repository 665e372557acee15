// ghost_tiled.cu — tuned refinement-boundary ghost fill (eqs 10-18 folded
// into the coefficient matrix by the scheduler; spatial operator = reading S3).
//
//   dst[o](ghost cell) = P[ sum_s coef[o][s] * src[s] ],   P = 5x5x5 tensor-product quartic Lagrange
//
// The ghost shell of a box is the union of six slabs (z-lo, z-hi, y-lo, y-hi, x-lo, x-hi); each slab is cut
// into tiles  g (thin axis) x TA x TB  fine cells whose origin is EVEN in every axis, so that the parent
// footprint of a tile is exactly (TA/2+4) x (TB/2+4) x (<= 6) parent cells and every index below is a
// compile-time function of the loop counters. One CTA per (tile, field), three phases:
//   1. one thread per parent column (a, b): for every source array read the <= 6 parent cells along the
//      thin axis ONCE, interpolate them to the g fine thin cells (weights from a per-tile table, so the
//      lo / hi side and any ghost width are the same code), and time-combine into the nout outputs
//      -> T[plane = (o, thin cell)][b][a] in shared memory. All global reads of the kernel happen here.
//   2. interpolation along b, register-blocked: one thread per (plane, a) loads the PB parent values once
//      and produces the TB fine values -> U[plane][fb][a].
//   3. interpolation along a and the store: one thread per (plane, fb, parent a) produces its two fine
//      children; for z- and y-slabs a = x and the pair is one 16-byte store, coalesced across the warp.
// Every parent value is read from HBM once per tile and a ghost value costs 6 + 5 + 5 FMA instead of 125.
#include "kernels.h"

namespace sc {

namespace {

constexpr int TA = 32, TB = 16;                  // fine cells per tile along the two transverse axes
constexpr int PA = TA / 2 + 4, PB = TB / 2 + 4;  // parent footprint of a tile (2-cell halo each side)
constexpr int PTMAX = 6;                         // parent cells along the thin axis (ghost width <= 4)
constexpr int NTHREADS = 256;

// quartic Lagrange weights at -1/4 (parity 0) and +1/4 (parity 1) of the parent spacing, offsets -2..2 (S3)
__device__ __forceinline__ double wprol(int parity, int c) {
  constexpr double w1[5] = {35.0 / 2048.0, -252.0 / 2048.0, 1890.0 / 2048.0, 420.0 / 2048.0, -45.0 / 2048.0};
  return parity ? w1[c] : w1[4 - c];
}
// 5-point interpolation to the two children of the parent cell at p[0] (values at stride s)
__device__ __forceinline__ void children(const double* p, int s, double& lo, double& hi) {
  const double a = p[-2 * s], b = p[-s], c = p[0], d = p[s], e = p[2 * s];
  constexpr double w0 = 35.0 / 2048.0, w1 = -252.0 / 2048.0, w2 = 1890.0 / 2048.0, w3 = 420.0 / 2048.0,
                   w4 = -45.0 / 2048.0;
  hi = w0 * a + w1 * b + w2 * c + w3 * d + w4 * e;  // parity 1: +1/4
  lo = w4 * a + w3 * b + w2 * c + w1 * d + w0 * e;  // parity 0: -1/4
}

}  // namespace

__global__ void __launch_bounds__(NTHREADS) ghost_fill_tiled(const __grid_constant__ GhostArgs a) {
  extern __shared__ __align__(16) double gsm[];
  __shared__ double sWt[4][PTMAX];  // thin-axis weights: fine thin cell kt <- parent cell c of the footprint
  const GhostTile t = a.tiles[blockIdx.x];
  const int f = blockIdx.y;
  const BoxView& ch = a.child;
  const BoxView& pa = a.parent;
  const int tid = threadIdx.x;
  // axes: thin = t.axis; transverse A = the more contiguous one
  const int axT = t.axis, axA = axT == 0 ? 1 : 0, axB = axT == 2 ? 1 : 2;
  // even tile origin (box-local fine index), valid fine range [lo, lo+n) from the tile descriptor
  const int oA = t.lo[axA] & ~1, oB = t.lo[axB] & ~1;
  const int vA0 = t.lo[axA] - oA, vA1 = vA0 + t.n[axA];  // valid tile-local fine range along A
  const int vB0 = t.lo[axB] - oB, vB1 = vB0 + t.n[axB];
  // parent-local index of footprint cell 0 along each axis
  const int qA = ((ch.lo[axA] + oA) >> 1) - 2 - pa.lo[axA];
  const int qB = ((ch.lo[axB] + oB) >> 1) - 2 - pa.lo[axB];
  const int IT0 = ch.lo[axT] + t.lo[axT];                       // level-global index of the first thin cell
  const int PT0 = (IT0 >> 1) - 2;                               // parent-global, first footprint cell
  const int ptn = ((IT0 + t.n[axT] - 1) >> 1) + 2 - PT0 + 1;    // parent cells along the thin axis (<= 6)
  const int qT = PT0 - pa.lo[axT];
  const int nA = ((vA1 - 1) >> 1) + 5, nB = ((vB1 - 1) >> 1) + 5;  // parent columns actually needed
  const int nt = t.n[axT];                                      // = g
  const int nplanes = a.nout * nt;
  double* T = gsm;                                 // [nplanes][PB][PA]
  double* U = gsm + (size_t)nplanes * PB * PA;     // [nplanes][TB][PA]
  if (tid < 4 * PTMAX) {
    const int kt = tid / PTMAX, c = tid % PTMAX;
    double w = 0.0;
    if (kt < nt) {
      const int Ig = IT0 + kt;
      const int j = (Ig >> 1) - PT0;  // footprint index of the containing parent cell (2 or 3)
      const int d = c - (j - 2);
      if (d >= 0 && d < 5) w = wprol(Ig & 1, d);
    }
    sWt[kt][c] = w;
  }
  __syncthreads();
  const long long psT = axT == 0 ? 1 : (axT == 1 ? pa.px : pa.plane);
  // ---- phase 1: gather, thin-axis interpolation, time combination ----------------------------------
  for (int col = tid; col < PA * PB; col += NTHREADS) {
    const int ia = col % PA, ib = col / PA;
    double acc[GF_MAX_OUT][4];
#pragma unroll
    for (int o = 0; o < GF_MAX_OUT; ++o)
#pragma unroll
      for (int k = 0; k < 4; ++k) acc[o][k] = 0.0;
    if (ia < nA && ib < nB) {
      int pc[3];
      pc[axT] = qT; pc[axA] = qA + ia; pc[axB] = qB + ib;
      const long long off = (long long)f * pa.vol + cell_offset(pa, pc[0], pc[1], pc[2]);
#pragma unroll
      for (int s = 0; s < GF_MAX_SRC; ++s) {
        if (s < a.nsrc) {
          const double* __restrict__ p = a.src[s] + off;
          double L[PTMAX];
#pragma unroll
          for (int c = 0; c < PTMAX; ++c) L[c] = c < ptn ? __ldg(p + c * psT) : 0.0;
          double v[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            double r = 0.0;
#pragma unroll
            for (int c = 0; c < PTMAX; ++c) r = fma(sWt[k][c], L[c], r);
            v[k] = r;
          }
#pragma unroll
          for (int o = 0; o < GF_MAX_OUT; ++o) {
            const double cf = a.coef[o][s];
            if (o < a.nout && cf != 0.0) {
#pragma unroll
              for (int k = 0; k < 4; ++k) acc[o][k] = fma(cf, v[k], acc[o][k]);
            }
          }
        }
      }
    }
#pragma unroll
    for (int o = 0; o < GF_MAX_OUT; ++o)
      if (o < a.nout) {
#pragma unroll
        for (int k = 0; k < 4; ++k)
          if (k < nt) T[((size_t)(o * nt + k) * PB + ib) * PA + ia] = acc[o][k];
      }
  }
  __syncthreads();
  // ---- phase 2: interpolation along B --------------------------------------------------------------
  for (int w = tid; w < nplanes * PA; w += NTHREADS) {
    const int ia = w % PA, pl = w / PA;
    const double* __restrict__ in = T + (size_t)pl * PB * PA + ia;
    double* __restrict__ out = U + (size_t)pl * TB * PA + ia;
    double v[PB];
#pragma unroll
    for (int j = 0; j < PB; ++j) v[j] = in[j * PA];
#pragma unroll
    for (int j = 0; j < TB / 2; ++j) {
      double lo, hi;
      children(&v[j + 2], 1, lo, hi);
      out[(2 * j) * PA] = lo;
      out[(2 * j + 1) * PA] = hi;
    }
  }
  __syncthreads();
  // ---- phase 3: interpolation along A, store -------------------------------------------------------
  const long long csT = axT == 0 ? 1 : (axT == 1 ? ch.px : ch.plane);
  const long long csA = axA == 0 ? 1 : ch.px;
  const long long csB = axB == 1 ? ch.px : ch.plane;
  int c0[3];
  c0[axT] = t.lo[axT]; c0[axA] = oA; c0[axB] = oB;
  const long long cbase = (long long)f * ch.vol + cell_offset(ch, c0[0], c0[1], c0[2]);
  const int nwork = nplanes * TB * (TA / 2);
  for (int w = tid; w < nwork; w += NTHREADS) {
    const int ja = w % (TA / 2);
    const int r = w / (TA / 2);
    const int fb = r % TB, pl = r / TB;
    if (fb < vB0 || fb >= vB1) continue;
    const int fa = 2 * ja;
    if (fa + 1 < vA0 || fa >= vA1) continue;
    double lo, hi;
    children(U + ((size_t)pl * TB + fb) * PA + ja + 2, 1, lo, hi);
    const int o = pl / nt, k = pl - o * nt;
    double* __restrict__ d = a.dst[o] + cbase + k * csT + fb * csB + fa * csA;
    const bool v0 = fa >= vA0, v1 = fa + 1 < vA1;
    if (axA == 0 && v0 && v1) {
      *reinterpret_cast<double2*>(d) = make_double2(lo, hi);
    } else {
      if (v0) d[0] = lo;
      if (v1) d[csA] = hi;
    }
  }
}

// ---- host: tile list ---------------------------------------------------------------------------------
namespace {
// cut [r0, r1) into pieces [max(r0, o + m T), min(r1, o + (m+1) T)) with o = r0 rounded down to even
void cut(int r0, int r1, int T, std::vector<std::pair<int, int>>& out) {
  out.clear();
  const int o = r0 & ~1;
  for (int s = o; s < r1; s += T) {
    const int lo = s < r0 ? r0 : s, hi = s + T < r1 ? s + T : r1;
    if (hi > lo) out.push_back({lo, hi - lo});
  }
}
}  // namespace

void build_ghost_tiles(const BoxView& ch, std::vector<GhostTile>& tiles) {
  tiles.clear();
  const int g = ch.g;
  std::vector<std::pair<int, int>> as, bs;
  // z-slabs: A = x over the padded extent, B = y over the padded extent
  cut(-g, ch.n[0] + g, TA, as);
  cut(-g, ch.n[1] + g, TB, bs);
  for (int hi = 0; hi < 2; ++hi)
    for (auto& b : bs)
      for (auto& x : as)
        tiles.push_back(GhostTile{{x.first, b.first, hi ? ch.n[2] : -g}, {x.second, b.second, g}, 2, 0});
  // y-slabs: A = x padded, B = z interior
  cut(0, ch.n[2], TB, bs);
  for (int hi = 0; hi < 2; ++hi)
    for (auto& b : bs)
      for (auto& x : as)
        tiles.push_back(GhostTile{{x.first, hi ? ch.n[1] : -g, b.first}, {x.second, g, b.second}, 1, 0});
  // x-slabs: A = y interior, B = z interior
  cut(0, ch.n[1], TA, as);
  for (int hi = 0; hi < 2; ++hi)
    for (auto& b : bs)
      for (auto& y : as)
        tiles.push_back(GhostTile{{hi ? ch.n[0] : -g, y.first, b.first}, {g, y.second, b.second}, 0, 0});
}

void launch_ghost_fill_tiled(const GhostArgs& a, cudaStream_t st) {
  const size_t smem = sizeof(double) * (size_t)a.nout * a.child.g * (PB * PA + TB * PA);
  static size_t configured = 0;
  if (smem > configured) {
    cudaFuncSetAttribute(ghost_fill_tiled, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    configured = smem;
  }
  dim3 grd(a.ntiles, a.F, 1);
  ghost_fill_tiled<<<grd, NTHREADS, smem, st>>>(a);
}

}  // namespace sc
