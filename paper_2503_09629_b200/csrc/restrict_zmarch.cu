// restrict_zmarch.cu — tuned restriction kernel (a5, reading S4).
// One CTA owns RPX x RPY parent columns and marches through the child's z-planes; each fine plane is
// staged in shared memory, reduced in x then y by the 6-point weights, and kept in a 6-deep register ring
// that is contracted in z every second plane. Each fine value is read once per CTA.
#include "kernels.h"

namespace sc {

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
