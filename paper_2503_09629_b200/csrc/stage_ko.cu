// stage_ko.cu — the RK4 stage kernel of the GENERAL formulation, used when Kreiss-Oliger dissipation is on
// (eqs 35-36: d_t y -> RHS + Q y for every evolved variable).
//
// With Q acting on u the slope k_{s,u} = Y_{s,rho} + Q Y_{s,u} is no longer Y_{s,rho}, so the two-launch
// formulation of DESIGN.md section 6 does not apply: the stage vectors are stored whole (U_s = u-part,
// R_s = rho-part, s = 2..4) and a level-step is four launches, eqs (1)-(9) stage by stage:
//   s = 1..3:  k_s = M Y_s,   Y_{s+1} = y_n + a_s dt k_s,        a = (1/2, 1/2, 1)          (eqs 6-9)
//   s = 4:     k_4 = M Y_4,   y_{n+1} = y_n + dt/6 (k_1 + 2 k_2 + 2 k_3 + k_4)               (eq 5)
// with M (U, R) = (R + Q U,  Lap_h U + A U + Q R). The slopes k_1..k_3 are not stored: k_j = (Y_{j+1} - y_n)/(a_j dt),
// so dt/6 (k_1 + 2 k_2 + 2 k_3) = [(Y_2 - y_n) + 2 (Y_3 - y_n) + (Y_4 - y_n)] / 3; k_4 is written only where a child
// level reads it for its dense-output ghost fill (eqs 10-18).
//   Q y = sigma/64 sum_i delta_i^6 y / h_i,  delta^6 y = y[-3] - 6 y[-2] + 15 y[-1] - 20 y[0] + 15 y[1] - 6 y[2] + y[3]
// One thread per cell and field, every operand straight from global memory (L1/L2 serve the stencil reuse).
#include "kernels.h"

namespace sc {

namespace {

__device__ __forceinline__ double d6(const double* y, long long s) {
  return (y[-3 * s] + y[3 * s]) - 6.0 * (y[-2 * s] + y[2 * s]) + 15.0 * (y[-s] + y[s]) - 20.0 * y[0];
}
__device__ __forceinline__ double d2(const double* y, long long s) {  // 12 h^2 x 4th-order second derivative (S2)
  return 16.0 * (y[-s] + y[s]) - (y[-2 * s] + y[2 * s]) - 30.0 * y[0];
}

}  // namespace

__global__ void __launch_bounds__(256) stage_ko(const __grid_constant__ StageKOArgs a) {
  const BoxView& b = a.b;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z % b.n[2];
  const int f = blockIdx.z / b.n[2];
  if (i >= b.n[0] || j >= b.n[1]) return;
  const long long o = (long long)f * b.vol + cell_offset(b, i, j, k);
  const long long sy = b.px, sz = b.plane;
  const double* U = a.Yu + o;
  const double* R = a.Yr + o;
  double LU = a.inv12dx2[0] * d2(U, 1) + a.inv12dx2[1] * d2(U, sy) + a.inv12dx2[2] * d2(U, sz);
  if (a.A) {
    const long long c0 = cell_offset(b, i, j, k);
    double s = 0.0;
    for (int q = 0; q < a.F; ++q) s = fma(a.A[f * a.F + q], a.Yu[(long long)q * b.vol + c0], s);
    LU += s;
  }
  const double QU = a.ko[0] * d6(U, 1) + a.ko[1] * d6(U, sy) + a.ko[2] * d6(U, sz);
  const double QR = a.ko[0] * d6(R, 1) + a.ko[1] * d6(R, sy) + a.ko[2] * d6(R, sz);
  const double ku = R[0] + QU, kr = LU + QR;
  const double un = a.yn_u[o], rn = a.yn_r[o];
  if (a.stage < 4) {
    const double adt = (a.stage == 3 ? 1.0 : 0.5) * a.dt;
    a.outU[o] = fma(adt, ku, un);
    a.outR[o] = fma(adt, kr, rn);
  } else {
    const double third = 1.0 / 3.0, dt6 = a.dt / 6.0;
    a.outU[o] = un + (third * ((a.U2[o] - un) + (U[0] - un)) + (2.0 * third) * (a.U3[o] - un)) + dt6 * ku;
    a.outR[o] = rn + (third * ((a.R2[o] - rn) + (R[0] - rn)) + (2.0 * third) * (a.R3[o] - rn)) + dt6 * kr;
    if (a.K4u) { a.K4u[o] = ku; a.K4r[o] = kr; }
  }
}

void launch_stage_ko_direct(const StageKOArgs& a, cudaStream_t st) {
  dim3 blk(64, 4, 1);
  dim3 grd((a.b.n[0] + 63) / 64, (a.b.n[1] + 3) / 4, a.b.n[2] * a.F);
  stage_ko<<<grd, blk, 0, st>>>(a);
}

}  // namespace sc
