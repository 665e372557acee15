// stage_fd8.cu — the two RK4 stage kernels (kernels.h: STAGE_12, STAGE_34) with 8th-order centred differences
// (the paper's BBH discretisation), sm_100a. First tiled version: it replaces the
// one-thread-per-cell kernel (stage_direct<8>, 2 x 25 global loads per cell: 660 us per 256^3 launch) at 331 us
// (0.33 of the HBM peak); it is not yet the radius-4 counterpart of the TMA z-march of stage_tma.cu (136 us for
// the 4th-order stencil). What the profile of its first version showed: half of all stall samples sat on the FMA
// that formed an operand right after its global load — the loads of the next plane must stay RAW in registers
// until they are stored to shared memory one iteration later (625 -> 516 us), and the 80-register cap of a third
// CTA per SM spilled the nine-slot accumulators (516 -> 343 us with two CTAs and 128 registers); interleaving the
// two operands in shared memory halves the shared loads (343 -> 331 us).
//
// A CTA owns a 32 x 8 (x, y) tile of one field and marches along a z-chunk. Per arriving plane k
//   * all threads build the two stage operands W1, W2 of the launch (kernels.h) on the tile plus a 4-cell halo
//     in shared memory (40 x 16 cells, double-buffered by plane parity: one barrier per plane); the global loads
//     of plane k+1 are issued before plane k is worked on and wait in registers;
//   * each thread forms the in-plane part of the 25-point Laplacian of its cell (17 16-byte shared loads: the two
//     operands are interleaved) and
//     SCATTERS the z part: plane k contributes c_|d| W(k) to the nine pending outputs k-4 .. k+4, held in
//     registers and shifted by one per plane, so the output of plane k-4 completes as plane k arrives;
//   * the completed plane is combined with the centre-only operands exactly as in stage_direct.
// Coupled systems add  sum_q A_fq W_q  at the centre cell from global memory, as stage_direct does.
#include "kernels.h"

namespace sc {

namespace {

constexpr int BX = 32, BY = 8, R8 = 4, HX8 = BX + 2 * R8, HY8 = BY + 2 * R8, NT8 = BX * BY;

// weights of the 8th-order second difference for |offset| = 0..4, in units of 1/dx^2
__device__ __forceinline__ double c8(int d) {
  constexpr double c[5] = {-205.0 / 72.0, 8.0 / 5.0, -1.0 / 5.0, 8.0 / 315.0, -1.0 / 560.0};
  return c[d];
}

template <int MODE>
__global__ void __launch_bounds__(NT8, 2) stage_fd8(StageArgs a, int chunk, int nchunks) {
  __shared__ double2 sW[2][HY8][HX8];  // [plane parity][y][x] -> (W1, W2): 20 KB, one 16-byte load serves both operands
  const BoxView& b = a.b;
  const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * BX + tx;
  const int X0 = blockIdx.x * BX, Y0 = blockIdx.y * BY;
  const int f = blockIdx.z / nchunks, c = blockIdx.z % nchunks;
  const int z0 = c * chunk, z1 = min(b.n[2], z0 + chunk);
  const int i = X0 + tx, j = Y0 + ty, F = a.F;
  const bool active = i < b.n[0] && j < b.n[1];
  const double dt = a.dt, hdt = 0.5 * a.dt;
  const double wx = 12.0 * a.inv12dx2[0], wy = 12.0 * a.inv12dx2[1], wz = 12.0 * a.inv12dx2[2];
  const double* __restrict__ u = a.yn + (long long)f * b.vol;
  // second array of each operand: W1 = u + s1 * r1, W2 = u + s2 * r2
  const double* __restrict__ r1 = MODE == STAGE_12 ? u : a.Y2r + (long long)f * b.vol;
  const double* __restrict__ r2 = MODE == STAGE_12 ? a.yn + (long long)(F + f) * b.vol : a.Y3r + (long long)f * b.vol;
  const double s1 = MODE == STAGE_12 ? 0.0 : hdt, s2 = MODE == STAGE_12 ? hdt : dt;

  auto couple = [&](double cf, const double* Rr, long long o) {  // sum_q A_fq (u_q + cf R_q) at one cell
    double s = 0.0;
    if (a.A)
      for (int q = 0; q < F; ++q) {
        const double uq = a.yn[(long long)q * b.vol + o];
        const double wq = Rr ? fma(cf, Rr[(long long)q * b.vol + o], uq) : uq;
        s = fma(a.A[f * F + q], wq, s);
      }
    return s;
  };

  double acc1[9], acc2[9];  // pending Laplacians of W1, W2 for the planes k-4 .. k+4
#pragma unroll
  for (int m = 0; m < 9; ++m) acc1[m] = acc2[m] = 0.0;

  // the operands of the NEXT plane travel in registers while the current plane is worked on (the loads are the
  // only long-latency step of the march)
  constexpr int NF = (HX8 * HY8 + NT8 - 1) / NT8;
  double pu[NF], pa[NF], pb[NF];  // raw values of the next plane: the operands are formed when they are stored
  long long fo_[NF];  // offset of this thread's halo cells in plane 0 (negative: none); a plane further is + b.plane
#pragma unroll
  for (int t = 0; t < NF; ++t) {
    const int q = tid + t * NT8, hx = q % HX8, hy = q / HX8, gi = X0 - R8 + hx, gj = Y0 - R8 + hy;
    fo_[t] = (q < HX8 * HY8 && gi < b.n[0] + R8 && gj < b.n[1] + R8) ? cell_offset(b, gi, gj, 0) : -1;
    pu[t] = pa[t] = pb[t] = 0.0;
  }
  auto fetch = [&](int k) {
    const long long zo = (long long)k * b.plane;
#pragma unroll
    for (int t = 0; t < NF; ++t)
      if (fo_[t] >= 0) {
        const long long o = fo_[t] + zo;
        pu[t] = u[o];
        if (MODE == STAGE_34) pa[t] = r1[o];
        pb[t] = r2[o];
      }
  };
  const long long oc0 = cell_offset(b, active ? i : 0, active ? j : 0, 0);  // this thread's cell in plane 0
  const double wzc[5] = {0.0, wz * c8(1), wz * c8(2), wz * c8(3), wz * c8(4)};
  const double ccen = c8(0) * (wx + wy + wz);
  fetch(z0 - R8);
  double cn[4] = {0.0, 0.0, 0.0, 0.0}, cx[4] = {0.0, 0.0, 0.0, 0.0};  // centre operands: this / next output plane
#pragma unroll 1
  for (int k = z0 - R8; k < z1 + R8; ++k) {
    const int p = (k - z0) & 1, kz1 = k + 1 - R8;
#pragma unroll
    for (int t = 0; t < NF; ++t) {
      const int q = tid + t * NT8;
      if (q < HX8 * HY8)
        (&sW[p][0][0])[q] = make_double2(MODE == STAGE_12 ? pu[t] : fma(s1, pa[t], pu[t]), fma(s2, pb[t], pu[t]));
    }
    __syncthreads();
    if (k + 1 < z1 + R8) fetch(k + 1);
    if (active && kz1 >= z0 && kz1 < z1) {  // centre-only operands of the NEXT output plane, one plane ahead
      const long long o = oc0 + (long long)kz1 * b.plane;
      cx[0] = a.yn[(long long)(F + f) * b.vol + o];
      if (MODE == STAGE_34) { cx[1] = r1[o]; cx[2] = r2[o]; cx[3] = u[o]; }
    }
    {
      const double2* __restrict__ s = &sW[p][ty + R8][tx + R8];
      const double2 wc = s[0];
      double2 dx = make_double2(0.0, 0.0), dy = dx;
#pragma unroll
      for (int d = 1; d <= R8; ++d) {
        const double2 xm = s[-d], xp = s[d], ym = s[-d * HX8], yp = s[d * HX8];
        dx.x = fma(c8(d), xm.x + xp.x, dx.x);
        dx.y = fma(c8(d), xm.y + xp.y, dx.y);
        dy.x = fma(c8(d), ym.x + yp.x, dy.x);
        dy.y = fma(c8(d), ym.y + yp.y, dy.y);
      }
      acc1[4] += fma(wx, dx.x, fma(wy, dy.x, ccen * wc.x));
      acc2[4] += fma(wx, dx.y, fma(wy, dy.y, ccen * wc.y));
#pragma unroll
      for (int d = 1; d <= R8; ++d) {
        const double t1 = wzc[d] * wc.x, t2 = wzc[d] * wc.y;
        acc1[4 - d] += t1;
        acc1[4 + d] += t1;
        acc2[4 - d] += t2;
        acc2[4 + d] += t2;
      }
    }
    const int kz = k - R8;  // the plane whose Laplacians are now complete
    if (active && kz >= z0 && kz < z1) {
      const long long o = oc0 + (long long)kz * b.plane, fo = (long long)f * b.vol + o;
      const double rho = cn[0];
      if (MODE == STAGE_12) {
        const double Lu = acc1[0] + couple(0.0, nullptr, o);
        const double L2 = acc2[0] + couple(hdt, a.yn + (long long)F * b.vol, o);
        a.Y2r[fo] = fma(hdt, Lu, rho);
        a.Y3r[fo] = fma(hdt, L2, rho);
      } else {
        const double L3 = acc1[0] + couple(hdt, a.Y2r, o);
        const double k4r = acc2[0] + couple(dt, a.Y3r, o);
        const double y2 = cn[1], y3 = cn[2], y4 = fma(dt, L3, rho), third = 1.0 / 3.0;
        a.ynew[fo] = fma(dt / 6.0, (rho + y4) + 2.0 * (y2 + y3), cn[3]);
        a.ynew[(long long)F * b.vol + fo] =
            rho + (third * ((y2 - rho) + (y4 - rho)) + (2.0 * third) * (y3 - rho)) + (dt / 6.0) * k4r;
        if (a.write_Y4r) a.Y4r[fo] = y4;
      }
    }
#pragma unroll
    for (int m = 0; m < 4; ++m) cn[m] = cx[m];
#pragma unroll
    for (int m = 0; m < 8; ++m) { acc1[m] = acc1[m + 1]; acc2[m] = acc2[m + 1]; }
    acc1[8] = acc2[8] = 0.0;
  }
}

}  // namespace

void launch_stage_fd8(const StageArgs& a, cudaStream_t st) {
  const int chunk = a.b.n[2] < 32 ? a.b.n[2] : 32;
  const int nchunks = (a.b.n[2] + chunk - 1) / chunk;
  dim3 blk(BX, BY, 1), grd((a.b.n[0] + BX - 1) / BX, (a.b.n[1] + BY - 1) / BY, nchunks * a.F);
  if (a.mode == STAGE_12) stage_fd8<STAGE_12><<<grd, blk, 0, st>>>(a, chunk, nchunks);
  else stage_fd8<STAGE_34><<<grd, blk, 0, st>>>(a, chunk, nchunks);
}

}  // namespace sc
