// kernels_opt.cu — tuned sm_100a kernels for the ghost fill (a3) and the restriction (a5).
//
// ghost_fill_tiled: the ghost shell of a box is cut into tiles of the six slabs (z-lo, z-hi, y-lo, y-hi,
//   x-lo, x-hi). One CTA per (tile, component): it gathers the tile's parent footprint ONCE into shared
//   memory, folding the dense-output time polynomial into the load (value = y_old + sum_j coef_j k_j,
//   eqs 10-18), then applies the 5-point Lagrange prolongation separably — thin axis first — so a ghost
//   value costs ~11 FMA instead of 125 and every parent value is read once per tile.
// restrict_zmarch: one CTA owns PX x PY parent columns and marches through the child's z-planes; each
//   fine plane is staged in shared memory, reduced in x then y by the 6-point weights, and kept in a
//   6-deep register ring that is contracted in z every second plane. Each fine value is read once per CTA.
#include "kernels.h"

namespace sc {

namespace {

// prolongation weights for parity 1 (fine centre at +1/4 of the parent spacing), offsets -2..2;
// parity 0 uses the mirror image (reading S3)
__device__ __forceinline__ double lagr5(const double* p, int stride, int par) {
  const int s = par ? stride : -stride;
  return (35.0 / 2048.0) * p[-2 * s] + (-252.0 / 2048.0) * p[-s] + (1890.0 / 2048.0) * p[0] +
         (420.0 / 2048.0) * p[s] + (-45.0 / 2048.0) * p[2 * s];
}

struct Dims { int d0, d1, d2; };

// One separable pass along AXIS: in (coarse along AXIS, dims din) -> out (fine along AXIS, nf cells whose
// level-global indices start at I0; in[0] along AXIS is the parent cell with global index C0).
// TO_GLOBAL: out is the child array; (gx,gy,gz) = box-local fine index of the tile origin.
template <int AXIS, bool TO_GLOBAL>
__device__ __forceinline__ void prolong_pass(const double* __restrict__ in, Dims din, double* __restrict__ out,
                                             int nf, int I0, int C0, const BoxView& ch, int gx, int gy, int gz) {
  const int o0 = AXIS == 0 ? nf : din.d0, o1 = AXIS == 1 ? nf : din.d1, o2 = AXIS == 2 ? nf : din.d2;
  const int total = o0 * o1 * o2;
  const int stride = AXIS == 0 ? 1 : (AXIS == 1 ? din.d0 : din.d0 * din.d1);
  for (int idx = threadIdx.x; idx < total; idx += blockDim.x) {
    const int x = idx % o0;
    const int t = idx / o0;
    const int y = t % o1;
    const int z = t / o1;
    const int f = AXIS == 0 ? x : (AXIS == 1 ? y : z);
    const int I = I0 + f;
    const int pc = (I >> 1) - C0;
    const int base = (AXIS == 0 ? pc : x) + din.d0 * ((AXIS == 1 ? pc : y) + din.d1 * (AXIS == 2 ? pc : z));
    const double v = lagr5(in + base, stride, I & 1);
    if (TO_GLOBAL) out[cell_offset(ch, gx + x, gy + y, gz + z)] = v;
    else out[idx] = v;
  }
}

}  // namespace

__global__ void __launch_bounds__(256) ghost_fill_tiled(GhostArgs a) {
  extern __shared__ double smem[];
  const GhostTile t = a.tiles[blockIdx.x];
  const int comp = blockIdx.y;
  const BoxView& ch = a.child;
  const BoxView& pa = a.parent;
  // level-global fine index of the tile origin, and parent footprint [C0, C0 + nc) per axis (parent-global)
  int I0[3], C0[3], nc[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    I0[d] = ch.lo[d] + t.lo[d];
    C0[d] = (I0[d] >> 1) - 2;
    nc[d] = ((I0[d] + t.n[d] - 1) >> 1) + 2 - C0[d] + 1;
  }
  const int n0 = nc[0] * nc[1] * nc[2];
  double* S0 = smem;
  double* S1 = smem + a.s0_doubles;
  // ---- gather + time-combine the parent footprint -------------------------------------------------
  {
    const long long pv = (long long)comp * pa.vol;
    const double* __restrict__ base = a.base + pv;
    const double* __restrict__ k0 = a.k[0] + pv;
    const double* __restrict__ k1 = a.k[1] + pv;
    const double* __restrict__ k2 = a.k[2] + pv;
    const double* __restrict__ k3 = a.k[3] + pv;
    const double c0 = a.coef[0], c1 = a.coef[1], c2 = a.coef[2], c3 = a.coef[3];
    const int use = a.use_k;
    const int px0 = C0[0] - pa.lo[0], py0 = C0[1] - pa.lo[1], pz0 = C0[2] - pa.lo[2];
    for (int idx = threadIdx.x; idx < n0; idx += blockDim.x) {
      const int x = idx % nc[0];
      const int r = idx / nc[0];
      const int y = r % nc[1];
      const int z = r / nc[1];
      const long long off = cell_offset(pa, px0 + x, py0 + y, pz0 + z);
      double v = base[off];
      if (use & 1) v += c0 * k0[off];
      if (use & 2) v += c1 * k1[off];
      if (use & 4) v += c2 * k2[off];
      if (use & 8) v += c3 * k3[off];
      S0[idx] = v;
    }
  }
  __syncthreads();
  double* dst = a.dst + (long long)comp * ch.vol;
  Dims d0{nc[0], nc[1], nc[2]};
  if (t.axis == 2) {  // z-slab: z, y, x
    prolong_pass<2, false>(S0, d0, S1, t.n[2], I0[2], C0[2], ch, 0, 0, 0);
    __syncthreads();
    Dims d1{nc[0], nc[1], t.n[2]};
    prolong_pass<1, false>(S1, d1, S0, t.n[1], I0[1], C0[1], ch, 0, 0, 0);
    __syncthreads();
    Dims d2{nc[0], t.n[1], t.n[2]};
    prolong_pass<0, true>(S0, d2, dst, t.n[0], I0[0], C0[0], ch, t.lo[0], t.lo[1], t.lo[2]);
  } else if (t.axis == 1) {  // y-slab: y, z, x
    prolong_pass<1, false>(S0, d0, S1, t.n[1], I0[1], C0[1], ch, 0, 0, 0);
    __syncthreads();
    Dims d1{nc[0], t.n[1], nc[2]};
    prolong_pass<2, false>(S1, d1, S0, t.n[2], I0[2], C0[2], ch, 0, 0, 0);
    __syncthreads();
    Dims d2{nc[0], t.n[1], t.n[2]};
    prolong_pass<0, true>(S0, d2, dst, t.n[0], I0[0], C0[0], ch, t.lo[0], t.lo[1], t.lo[2]);
  } else {  // x-slab: x, z, y
    prolong_pass<0, false>(S0, d0, S1, t.n[0], I0[0], C0[0], ch, 0, 0, 0);
    __syncthreads();
    Dims d1{t.n[0], nc[1], nc[2]};
    prolong_pass<2, false>(S1, d1, S0, t.n[2], I0[2], C0[2], ch, 0, 0, 0);
    __syncthreads();
    Dims d2{t.n[0], nc[1], t.n[2]};
    prolong_pass<1, true>(S0, d2, dst, t.n[1], I0[1], C0[1], ch, t.lo[0], t.lo[1], t.lo[2]);
  }
}

// ---- host: tile list -------------------------------------------------------------------------------
static void split(int lo, int extent, int target, std::vector<std::pair<int, int>>& out) {
  out.clear();
  const int parts = (extent + target - 1) / target;
  const int base = extent / parts, rem = extent % parts;
  int p = lo;
  for (int q = 0; q < parts; ++q) {
    const int s = base + (q < rem ? 1 : 0);
    out.push_back({p, s});
    p += s;
  }
}

static void footprint_doubles(const BoxView& ch, const GhostTile& t, size_t* s0, size_t* s1) {
  long long nc[3];
  for (int d = 0; d < 3; ++d) {
    const int I0 = ch.lo[d] + t.lo[d];
    nc[d] = ((I0 + t.n[d] - 1) >> 1) + 2 - ((I0 >> 1) - 2) + 1;
  }
  const long long a = nc[0] * nc[1] * nc[2];
  long long b, c;
  if (t.axis == 2) { b = nc[0] * nc[1] * t.n[2]; c = nc[0] * (long long)t.n[1] * t.n[2]; }
  else if (t.axis == 1) { b = nc[0] * t.n[1] * nc[2]; c = nc[0] * (long long)t.n[1] * t.n[2]; }
  else { b = t.n[0] * nc[1] * nc[2]; c = (long long)t.n[0] * nc[1] * t.n[2]; }
  *s0 = (size_t)(a > c ? a : c);
  *s1 = (size_t)b;
}

void build_ghost_tiles(const BoxView& ch, std::vector<GhostTile>& tiles, size_t* s0_doubles, size_t* s1_doubles) {
  tiles.clear();
  const int g = ch.g;
  const int TX = 64, TY = 32, TZ = 32;
  std::vector<std::pair<int, int>> xs, ys, zs;
  // z slabs: full padded x and y extent
  split(-g, ch.n[0] + 2 * g, TX, xs);
  split(-g, ch.n[1] + 2 * g, TY, ys);
  for (int hi = 0; hi < 2; ++hi)
    for (auto& y : ys)
      for (auto& x : xs) tiles.push_back(GhostTile{{x.first, y.first, hi ? ch.n[2] : -g}, {x.second, y.second, g}, 2, 0});
  // y slabs: full padded x extent, interior z
  split(0, ch.n[2], TZ, zs);
  for (int hi = 0; hi < 2; ++hi)
    for (auto& z : zs)
      for (auto& x : xs) tiles.push_back(GhostTile{{x.first, hi ? ch.n[1] : -g, z.first}, {x.second, g, z.second}, 1, 0});
  // x slabs: interior y and z
  split(0, ch.n[1], TY, ys);
  for (int hi = 0; hi < 2; ++hi)
    for (auto& z : zs)
      for (auto& y : ys) tiles.push_back(GhostTile{{hi ? ch.n[0] : -g, y.first, z.first}, {g, y.second, z.second}, 0, 0});
  size_t m0 = 0, m1 = 0;
  for (const GhostTile& t : tiles) {
    size_t a, b;
    footprint_doubles(ch, t, &a, &b);
    if (a > m0) m0 = a;
    if (b > m1) m1 = b;
  }
  *s0_doubles = m0;
  *s1_doubles = m1;
}

void launch_ghost_fill_opt(const GhostArgs& a, cudaStream_t st) {
  const size_t smem = sizeof(double) * (size_t)(a.s0_doubles + a.s1_doubles);
  static size_t configured = 0;
  if (smem > configured) {
    cudaFuncSetAttribute(ghost_fill_tiled, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    configured = smem;
  }
  dim3 grd(a.ntiles, a.V, 1);
  ghost_fill_tiled<<<grd, 256, smem, st>>>(a);
}

// ====================================================================================================
// restriction: z-march
// ====================================================================================================
namespace {
constexpr int RPX = 32, RPY = 8;            // parent cells per CTA in x, y  (256 threads, one column each)
constexpr int RFX = 2 * RPX + 4, RFY = 2 * RPY + 4;  // fine plane tile incl. the 2-cell halo
__device__ __forceinline__ double lagr6(double a, double b, double c, double d, double e, double f) {
  return (3.0 / 256.0) * (a + f) + (-25.0 / 256.0) * (b + e) + (150.0 / 256.0) * (c + d);
}
}  // namespace

__global__ void __launch_bounds__(RPX* RPY) restrict_zmarch(BoxView ch, BoxView pa, const double* __restrict__ yc,
                                                            double* __restrict__ yp, int pz_per_cta) {
  __shared__ double sF[RFY][RFX];   // fine plane tile
  __shared__ double sX[RFY][RPX];   // after the x reduction
  const int tx = threadIdx.x % RPX, ty = threadIdx.x / RPX;
  const int X0 = blockIdx.x * RPX, Y0 = blockIdx.y * RPY;
  const int nzc = (ch.n[2] / 2 + pz_per_cta - 1) / pz_per_cta;
  const int comp = blockIdx.z / nzc;
  const int Z0 = (blockIdx.z % nzc) * pz_per_cta;
  const int Z1 = min(Z0 + pz_per_cta, ch.n[2] / 2);
  const int npx = ch.n[0] / 2, npy = ch.n[1] / 2;
  const double* __restrict__ src = yc + (long long)comp * ch.vol;
  double* __restrict__ dst = yp + (long long)comp * pa.vol;
  const int P0 = (ch.lo[0] >> 1) - pa.lo[0], P1 = (ch.lo[1] >> 1) - pa.lo[1], P2 = (ch.lo[2] >> 1) - pa.lo[2];
  // fine extent actually needed by this CTA (ragged tiles)
  const int fx = min(RFX, 2 * (npx - X0) + 4), fy = min(RFY, 2 * (npy - Y0) + 4);
  const int nload = fx * fy;
  const bool active = (X0 + tx < npx) && (Y0 + ty < npy);
  double ring[6];
#pragma unroll
  for (int q = 0; q < 6; ++q) ring[q] = 0.0;
  // fine planes 2*Z0-2 .. 2*Z1+1 ; parent plane Z is complete after fine plane 2Z+3
  constexpr int NPRE = (RFX * RFY + RPX * RPY - 1) / (RPX * RPY);
  double pre[NPRE];
  auto load_plane = [&](int kf) {
#pragma unroll
    for (int q = 0; q < NPRE; ++q) {
      const int idx = threadIdx.x + q * (RPX * RPY);
      if (idx < nload) {
        const int x = idx % fx, y = idx / fx;
        pre[q] = src[cell_offset(ch, 2 * X0 - 2 + x, 2 * Y0 - 2 + y, kf)];
      }
    }
  };
  const int kf0 = 2 * Z0 - 2, kf1 = 2 * Z1 + 1;
  load_plane(kf0);
  for (int kf = kf0; kf <= kf1; ++kf) {
#pragma unroll
    for (int q = 0; q < NPRE; ++q) {
      const int idx = threadIdx.x + q * (RPX * RPY);
      if (idx < nload) sF[idx / fx][idx % fx] = pre[q];
    }
    __syncthreads();
    if (kf < kf1) load_plane(kf + 1);  // prefetch the next plane while this one is reduced
    for (int idx = threadIdx.x; idx < RPX * fy; idx += RPX * RPY) {
      const int x = idx % RPX, y = idx / RPX;
      const double* r = &sF[y][2 * x];
      sX[y][x] = lagr6(r[0], r[1], r[2], r[3], r[4], r[5]);
    }
    __syncthreads();
    const double v = lagr6(sX[2 * ty][tx], sX[2 * ty + 1][tx], sX[2 * ty + 2][tx], sX[2 * ty + 3][tx],
                           sX[2 * ty + 4][tx], sX[2 * ty + 5][tx]);
#pragma unroll
    for (int q = 0; q < 5; ++q) ring[q] = ring[q + 1];
    ring[5] = v;
    const int rel = kf - kf0;  // 0-based plane counter; parent plane Z0 + m completes at rel = 2m + 5
    if (rel >= 5 && ((rel - 5) & 1) == 0 && active) {
      const int Z = Z0 + (rel - 5) / 2;
      dst[cell_offset(pa, P0 + X0 + tx, P1 + Y0 + ty, P2 + Z)] =
          lagr6(ring[0], ring[1], ring[2], ring[3], ring[4], ring[5]);
    }
  }
}

void launch_restrict_opt(const BoxView& ch, const BoxView& pa, int V, const double* yc, double* yp, cudaStream_t st) {
  const int npx = ch.n[0] / 2, npy = ch.n[1] / 2, npz = ch.n[2] / 2;
  const int gx = (npx + RPX - 1) / RPX, gy = (npy + RPY - 1) / RPY;
  // enough CTAs for ~4 per SM: split z into chunks of at least 8 parent planes
  int pz = npz;
  while (pz > 8 && (long long)gx * gy * V * ((npz + pz - 1) / pz) < 148 * 6) pz = (pz + 1) / 2;
  const int nzc = (npz + pz - 1) / pz;
  dim3 grd(gx, gy, nzc * V);
  restrict_zmarch<<<grd, RPX * RPY, 0, st>>>(ch, pa, yc, yp, pz);
}

}  // namespace sc
