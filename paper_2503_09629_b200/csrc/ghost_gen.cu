// ghost_gen.cu — general refinement-boundary ghost fill (SURVEY 8a row a3 for the NEXT-3 variants): any ghost width
// up to MAX_GHOST, any prolongation stencil of up to 10 points per axis (quartic S3, 9-point S30, the vertex-centred
// 6- / 10-point midpoint operators S31), any problem shape (kernels.h: GhostProblem). The tuned kernel of ghost_tma.cu
// covers g <= 4 with the quartic cell-centred operator; everything else used to fall to the one-thread-per-cell
// np^3-point gather of kernels_basic.cu (4-10 ms per 256^3 launch). Here the tensor operator is applied SEPARABLY:
//
//   child array dst_arr[o](ghost cell) = P[ sum_s coef[o][s] * parent array src_arr[s] ],   P = Px Py Pz
//
// The shell is cut into the six slabs of ghost_tma.cu (z-lo, z-hi over the padded x-y extent; y-lo, y-hi over padded x
// and interior z; x-lo, x-hi over interior y-z) and every slab into tiles of 16 x 16 cells times the slab's thickness.
// One CTA per (tile, field, problem); it
//   1. reads every source's footprint ONCE and forms all combined fields C_o = sum_s coef[o][s] src_s in shared memory,
//   2. per output: interpolates along x, then y, then z through two more shared-memory buffers (np FMA per value and
//      pass),
//   3. stores the tile's cells.
// Index maps: fine cell I (level-global) has parent I >> 1 and parity I & 1 (S1; vertex grids: parity 0 = ON the
// parent point, S31); the footprint of fine cells [I0, I1) along an axis is parents (I0 >> 1) + pmin .. ((I1 - 1) >> 1)
// + pmin + np - 1, inside the parent's interior by the nesting rule.
#include "kernels.h"
#include "launch_cfg.h"

namespace sc {

namespace {

constexpr int GT = 16;                 // tile edge along the two long axes of a slab
constexpr int GNT = 256;

struct GenSlab {   // one of the six slabs: box-local fine ranges and its tiling
  int lo[3], hi[3];
  int nta, ntb;    // tiles along the two long axes (A = lower axis index, B = higher)
  int first;       // index of its first tile in the launch
};
struct GenArgs {
  GhostArgs g;
  GenSlab slab[6];
  int ntiles;
  int fpcap, bcap;  // doubles reserved per combined field (footprint) and for the x-pass buffer
};

}  // namespace

template <int NP>  // points of the prolongation stencil per axis: 5 (S3), 9 (S30), 6 / 10 (vertex-centred, S31)
__global__ void __launch_bounds__(GNT) ghost_fill_tiled(const __grid_constant__ GenArgs A) {
  extern __shared__ double gsm[];
  const GhostArgs& a = A.g;
  double* const bufC = gsm;                              // [nout][pz][py][px]: the combined fields on the footprint
  double* const bufB = gsm + GF_MAX_OUT * A.fpcap;       // [pz][py][tx]
  double* const bufA = bufB + A.bcap;                    // [pz][ty][tx]
  const int f = blockIdx.y;
  const GhostProblem& pr = a.prob[blockIdx.z];
  // which slab, which tile
  int s = 0;
  while (s < 5 && (int)blockIdx.x >= A.slab[s + 1].first) ++s;
  const GenSlab& sl = A.slab[s];
  const int thin = 2 - s / 2;                     // slabs 0,1: z; 2,3: y; 4,5: x
  const int axA = thin == 0 ? 1 : 0, axB = thin == 2 ? 1 : 2;
  const int t = blockIdx.x - sl.first, ta = t % sl.nta, tb = t / sl.nta;
  int f0[3], f1[3];                               // the tile's fine range, box-local, clipped to the slab
  f0[thin] = sl.lo[thin]; f1[thin] = sl.hi[thin];
  f0[axA] = sl.lo[axA] + ta * GT; f1[axA] = min(sl.hi[axA], f0[axA] + GT);
  f0[axB] = sl.lo[axB] + tb * GT; f1[axB] = min(sl.hi[axB], f0[axB] + GT);
  int tn[3], pn[3], p0[3], I0[3];                 // fine extent, parent extent, first parent cell (parent-box-local), first fine global index
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    I0[d] = a.child.lo[d] + f0[d];
    const int I1 = a.child.lo[d] + f1[d] - 1;
    tn[d] = f1[d] - f0[d];
    p0[d] = (I0[d] >> 1) + a.pmin - a.parent.lo[d];
    pn[d] = ((I1 >> 1) - (I0[d] >> 1)) + a.np;
  }
  // thread = (x index ix = tid & 15 [and ix + 16 on the footprint], row ir = tid >> 4 stepping by 16)
  const int tid = threadIdx.x, ix = tid & 15, ir = tid >> 4;
  const int prow = pn[1] * pn[2], npar = prow * pn[0];
  // 1. every source is read ONCE; all combined fields C_o = sum_s coef[o][s] src_s of the footprint go to shared memory
  {
    double cf[GF_MAX_OUT][GF_MAX_SRC];  // the problem's coefficients in registers (unused entries are zero)
    const double* sp[GF_MAX_SRC];
#pragma unroll
    for (int sidx = 0; sidx < GF_MAX_SRC; ++sidx) {
      sp[sidx] = a.parent_base + (long long)(pr.src_arr[sidx < pr.nsrc ? sidx : 0] + f) * a.parent.vol;
#pragma unroll
      for (int o = 0; o < GF_MAX_OUT; ++o) cf[o][sidx] = (sidx < pr.nsrc && o < pr.nout) ? pr.coef[o][sidx] : 0.0;
    }
    for (int r = ir; r < prow; r += 16) {
      const int j = r % pn[1], k = r / pn[1];
      const long long off = cell_offset(a.parent, p0[0], p0[1] + j, p0[2] + k);
      for (int i = ix; i < pn[0]; i += 16) {
        double v[GF_MAX_SRC];
#pragma unroll
        for (int sidx = 0; sidx < GF_MAX_SRC; ++sidx) v[sidx] = sidx < pr.nsrc ? sp[sidx][off + i] : 0.0;
#pragma unroll
        for (int o = 0; o < GF_MAX_OUT; ++o) {
          if (o < pr.nout) {
            double c = 0.0;
#pragma unroll
            for (int sidx = 0; sidx < GF_MAX_SRC; ++sidx) c = fma(cf[o][sidx], v[sidx], c);
            bufC[o * npar + r * pn[0] + i] = c;
          }
        }
      }
    }
  }
  __syncthreads();
  for (int o = 0; o < pr.nout; ++o) {
    const double* C = bufC + o * npar;
    // 2a. x: C [pz][py][px] -> bufB [pz][py][tx]
    if (ix < tn[0]) {
      const int I = I0[0] + ix, jp = (I >> 1) - (I0[0] >> 1);
      double w[NP];
#pragma unroll
      for (int m = 0; m < NP; ++m) w[m] = a.w[I & 1][m];
      for (int r = ir; r < prow; r += 16) {
        const double* src = C + r * pn[0] + jp;
        double v = 0.0;
#pragma unroll
        for (int m = 0; m < NP; ++m) v = fma(w[m], src[m], v);
        bufB[r * tn[0] + ix] = v;
      }
    }
    __syncthreads();
    // 2b. y: bufB [pz][py][tx] -> bufA [pz][ty][tx];  thread = (ix, j = ir), loop over planes
    if (ix < tn[0] && ir < tn[1]) {
      const int I = I0[1] + ir, jp = (I >> 1) - (I0[1] >> 1);
      double w[NP];
#pragma unroll
      for (int m = 0; m < NP; ++m) w[m] = a.w[I & 1][m];
      const int rowB = pn[1] * tn[0], rowA = tn[1] * tn[0];
      const double* src = bufB + jp * tn[0] + ix;
      double* out = bufA + ir * tn[0] + ix;
      for (int k = 0; k < pn[2]; ++k, src += rowB, out += rowA) {
        double v = 0.0;
#pragma unroll
        for (int m = 0; m < NP; ++m) v = fma(w[m], src[m * tn[0]], v);
        *out = v;
      }
    }
    __syncthreads();
    // 2c + 3. z: bufA [pz][ty][tx] -> the child's ghost cells
    if (ix < tn[0] && ir < tn[1]) {
      double* dst = a.child_base + (long long)(pr.dst_arr[o] + f) * a.child.vol + cell_offset(a.child, f0[0] + ix, f0[1] + ir, f0[2]);
      const int plane = tn[0] * tn[1];
      for (int k = 0; k < tn[2]; ++k) {
        const int I = I0[2] + k, jp = (I >> 1) - (I0[2] >> 1);
        const double* w = a.w[I & 1];
        const double* src = bufA + jp * plane + ir * tn[0] + ix;
        double v = 0.0;
#pragma unroll
        for (int m = 0; m < NP; ++m) v = fma(w[m], src[m * plane], v);
        dst[(long long)k * a.child.plane] = v;
      }
    }
    // (the next output's x pass overwrites bufB only after every thread has passed the barrier behind 2b; bufA is
    // rewritten behind the barrier of its 2a)
  }
}

void launch_ghost_fill_tiled(const GhostArgs& a, cudaStream_t st) {
  GenArgs A{};
  A.g = a;
  const BoxView& c = a.child;
  const int g = c.g;
  int first = 0;
  for (int s = 0; s < 6; ++s) {
    GenSlab& sl = A.slab[s];
    const int thin = 2 - s / 2, hi = s & 1;
    for (int d = 0; d < 3; ++d) {
      // z-slabs span the padded x-y extent, y-slabs padded x and interior z, x-slabs the interior y-z extent
      const bool padded = d < thin;
      sl.lo[d] = padded ? -g : 0;
      sl.hi[d] = padded ? c.n[d] + g : c.n[d];
    }
    sl.lo[thin] = hi ? c.n[thin] : -g;
    sl.hi[thin] = hi ? c.n[thin] + g : 0;
    const int axA = thin == 0 ? 1 : 0, axB = thin == 2 ? 1 : 2;
    sl.nta = (sl.hi[axA] - sl.lo[axA] + GT - 1) / GT;
    sl.ntb = (sl.hi[axB] - sl.lo[axB] + GT - 1) / GT;
    sl.first = first;
    first += sl.nta * sl.ntb;
  }
  A.ntiles = first;
  // footprint bounds: n fine cells touch at most n/2 + np parent cells (any parity)
  const int PL = GT / 2 + a.np, PT = g / 2 + a.np;
  A.fpcap = PL * PL * PT;
  A.bcap = PL * PL * GT;
  const size_t smem = sizeof(double) * ((size_t)GF_MAX_OUT * A.fpcap + A.bcap + (size_t)GT * GT * PL);
  dim3 grd(A.ntiles, a.F, a.nprob);
  auto go = [&](auto kernel) {
    ensure_dynamic_smem(kernel, smem);  // smem depends on g and np
    kernel<<<grd, GNT, smem, st>>>(A);
  };
  if (a.np == 5) go(ghost_fill_tiled<5>);
  else if (a.np == 6) go(ghost_fill_tiled<6>);
  else if (a.np == 9) go(ghost_fill_tiled<9>);
  else go(ghost_fill_tiled<10>);
}


// ------------------------------------------------------------------------------------------------
// General restriction (SURVEY 8a row a5 for the NEXT-3 variants): any stencil of up to 10 fine points per axis (quintic
// S4 is taken by restrict_zmarch.cu; here: the 10-point operator of S30 and injection on vertex-centred grids, S31),
// applied separably: parent cell J <- sum_{a,b,c} r[c] r[b] r[a] child[2J + rmin + (a, b, c)].
// One CTA per (tile of 8 x 8 x 4 parent cells, component): the x pass runs straight from global memory (the nr-fold
// re-reads hit L1), y and z through shared memory.
// ------------------------------------------------------------------------------------------------
namespace {
constexpr int RTX = 8, RTY = 8, RTZ = 4;
constexpr int RFY = 2 * (RTY - 1) + 10, RFZ = 2 * (RTZ - 1) + 10;  // fine rows / planes a tile reads at most
}  // namespace

template <int NR>
__global__ void __launch_bounds__(256) restrict_tiled(const __grid_constant__ RestrictArgs a) {
  __shared__ double sx[RFZ][RFY][RTX];
  __shared__ double sy[RFZ][RTY][RTX];
  const BoxView& ch = a.child;
  const BoxView& pa = a.parent;
  const int ncx = ch.n[0] / 2, ncy = ch.n[1] / 2, ncz = ch.n[2] / 2;
  const int tzn = (ncz + RTZ - 1) / RTZ;
  const int I0 = blockIdx.x * RTX, J0 = blockIdx.y * RTY, K0 = (blockIdx.z % tzn) * RTZ, c = blockIdx.z / tzn;
  const int nI = min(RTX, ncx - I0), nJ = min(RTY, ncy - J0), nK = min(RTZ, ncz - K0);
  const int fy = 2 * (nJ - 1) + a.nr, fz = 2 * (nK - 1) + a.nr;
  const double* s = a.ychild + (long long)c * ch.vol;
  // thread = (i = tid & 7, row = tid >> 3 stepping by 32): no division in the inner loops
  const int tid = threadIdx.x, i = tid & 7, ir = tid >> 3;
  double w[NR];
#pragma unroll
  for (int m = 0; m < NR; ++m) w[m] = a.r[m];
  if (i < nI) {
    for (int r = ir; r < fy * fz; r += 32) {
      const int j = r % fy, k = r / fy;
      const double* row = s + cell_offset(ch, 2 * (I0 + i) + a.rmin, 2 * J0 + a.rmin + j, 2 * K0 + a.rmin + k);
      double v = 0.0;
      _Pragma("unroll") for (int m = 0; m < NR; ++m) v = fma(w[m], row[m], v);
      sx[k][j][i] = v;
    }
  }
  __syncthreads();
  if (i < nI) {
    for (int r = ir; r < nJ * fz; r += 32) {
      const int j = r % nJ, k = r / nJ;
      double v = 0.0;
      _Pragma("unroll") for (int m = 0; m < NR; ++m) v = fma(w[m], sx[k][2 * j + m][i], v);
      sy[k][j][i] = v;
    }
  }
  __syncthreads();
  const int P0 = (ch.lo[0] >> 1) - pa.lo[0], P1 = (ch.lo[1] >> 1) - pa.lo[1], P2 = (ch.lo[2] >> 1) - pa.lo[2];
  if (i < nI) {
    for (int r = ir; r < nJ * nK; r += 32) {
      const int j = r % nJ, k = r / nJ;
      double v = 0.0;
      _Pragma("unroll") for (int m = 0; m < NR; ++m) v = fma(w[m], sy[2 * k + m][j][i], v);
      a.yparent[(long long)c * pa.vol + cell_offset(pa, P0 + I0 + i, P1 + J0 + j, P2 + K0 + k)] = v;
    }
  }
}

void launch_restrict_ref(const RestrictArgs& a, cudaStream_t st);

void launch_restrict_tiled(const RestrictArgs& a, cudaStream_t st) {
  const int ncx = a.child.n[0] / 2, ncy = a.child.n[1] / 2, ncz = a.child.n[2] / 2;
  dim3 grd((ncx + RTX - 1) / RTX, (ncy + RTY - 1) / RTY, ((ncz + RTZ - 1) / RTZ) * a.V);
  if (a.nr == 10) restrict_tiled<10><<<grd, 256, 0, st>>>(a);
  else if (a.nr == 6) restrict_tiled<6><<<grd, 256, 0, st>>>(a);
  else launch_restrict_ref(a, st);
}

}  // namespace sc
