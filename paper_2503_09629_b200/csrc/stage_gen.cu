// stage_gen.cu — the stage kernel of the GENERAL stage-by-stage formulation (kernels.h: StageKOArgs), direct loads.
//
// One launch = one RK stage of one box: k = M Y_s at every interior cell, then the integrator's stage combine. It
// covers what the two-launch formulation of DESIGN.md section 6 cannot:
//   * Kreiss-Oliger dissipation (eqs 35-36): with Q acting on u the slope k_{s,u} = Y_{s,rho} + Q Y_{s,u}
//     is no longer Y_{s,rho};  Q y = sigma/64 sum_i delta_i^6 y / h_i  (r = 4)  or  sigma/1024 sum_i delta_i^10 y / h_i
//     (r = 8, "ninth-order");
//   * 8th-order differences together with dissipation (the paper's production discretisation);
//   * the RK3 / RK2 integrators (reading S28);
//   * the radiative outer boundary (reading S29): level-0 cells within g of a domain face obey
//     d_t y = -[(x^i / r) d_i y + y / r] with second-order centred / one-sided differences, for u and rho alike.
// The slopes of earlier stages are not stored; they are recovered at the cell from the stage vectors
// (RK4: k_j = (Y_{j+1} - y_n)/(a_j dt);  RK3: k_1 = 2 (Y_2 - y_n)/dt, k_2 = (Y_3 - y_n)/(2 dt) + (Y_2 - y_n)/dt).
// One thread per cell and field, every operand straight from global memory (L1/L2 serve the stencil reuse); the tuned
// kernel for the RK4 / 4th-order / delta^6 / periodic case is stage_ko_tma.cu.
#include "kernels.h"

namespace sc {

namespace {

__device__ __forceinline__ double d6(const double* y, long long s) {
  return (y[-3 * s] + y[3 * s]) - 6.0 * (y[-2 * s] + y[2 * s]) + 15.0 * (y[-s] + y[s]) - 20.0 * y[0];
}
__device__ __forceinline__ double d10(const double* y, long long s) {
  return (y[-5 * s] + y[5 * s]) - 10.0 * (y[-4 * s] + y[4 * s]) + 45.0 * (y[-3 * s] + y[3 * s]) -
         120.0 * (y[-2 * s] + y[2 * s]) + 210.0 * (y[-s] + y[s]) - 252.0 * y[0];
}
// 12 h^2 x second difference: 4th order (S2) or 8th order
template <int FD>
__device__ __forceinline__ double d2(const double* y, long long s) {
  if (FD == 8)
    return 12.0 * ((-1.0 / 560.0) * (y[-4 * s] + y[4 * s]) + (8.0 / 315.0) * (y[-3 * s] + y[3 * s]) -
                   (1.0 / 5.0) * (y[-2 * s] + y[2 * s]) + (8.0 / 5.0) * (y[-s] + y[s]) - (205.0 / 72.0) * y[0]);
  return 16.0 * (y[-s] + y[s]) - (y[-2 * s] + y[2 * s]) - 30.0 * y[0];
}
template <int KO>
__device__ __forceinline__ double diss(const double* y, long long sy, long long sz, const double ko[3]) {
  if (KO == 9) return ko[0] * d10(y, 1) + ko[1] * d10(y, sy) + ko[2] * d10(y, sz);
  if (KO == 5) return ko[0] * d6(y, 1) + ko[1] * d6(y, sy) + ko[2] * d6(y, sz);
  return 0.0;
}
// radiative operator at a boundary point (S29): second-order centred differences where both neighbours are in the
// box, the one-sided three-point formula on the outermost layer
__device__ __forceinline__ double radiative(const double* y, const int idx[3], const int n[3], const long long st[3],
                                            const double x[3], const double dx[3], double rinv) {
  double s = 0.0;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    double d;
    if (idx[a] == 0) d = -3.0 * y[0] + 4.0 * y[st[a]] - y[2 * st[a]];
    else if (idx[a] == n[a] - 1) d = 3.0 * y[0] - 4.0 * y[-st[a]] + y[-2 * st[a]];
    else d = y[st[a]] - y[-st[a]];
    s += x[a] * (d / (2.0 * dx[a]));
  }
  return -(s * rinv + y[0] * rinv);
}

}  // namespace

template <int FD, int KO>
__global__ void __launch_bounds__(256) stage_gen(const __grid_constant__ StageKOArgs a) {
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
  double ku, kr;
  const int nb = a.rad_nb;
  const bool zone = nb > 0 && (i < nb || i >= b.n[0] - nb || j < nb || j >= b.n[1] - nb || k < nb || k >= b.n[2] - nb);
  if (a.zone_only && !zone) return;
  if (zone) {
    const int idx[3] = {i, j, k};
    const long long st[3] = {1, sy, sz};
    const double x[3] = {a.x0[0] + i * a.dx[0], a.x0[1] + j * a.dx[1], a.x0[2] + k * a.dx[2]};
    const double rinv = 1.0 / sqrt(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]);
    ku = radiative(U, idx, b.n, st, x, a.dx, rinv);
    kr = radiative(R, idx, b.n, st, x, a.dx, rinv);
  } else {
    double LU = a.inv12dx2[0] * d2<FD>(U, 1) + a.inv12dx2[1] * d2<FD>(U, sy) + a.inv12dx2[2] * d2<FD>(U, sz);
    if (a.A) {
      const long long c0 = cell_offset(b, i, j, k);
      double s = 0.0;
      for (int q = 0; q < a.F; ++q) s = fma(a.A[f * a.F + q], a.Yu[(long long)q * b.vol + c0], s);
      LU += s;
    }
    ku = R[0] + diss<KO>(U, sy, sz, a.ko);
    kr = LU + diss<KO>(R, sy, sz, a.ko);
  }
  const double un = a.yn_u[o], rn = a.yn_r[o], dt = a.dt;
  const int S = a.integrator, s = a.stage;
  if (s > S) {  // RK3: the slope at the new state (the child's dense output reads it)
    a.K4u[o] = ku; a.K4r[o] = kr;
    return;
  }
  if (s == 1 && S > 1) {  // Y_2 = y_n + dt/2 k_1 (all three integrators)
    a.outU[o] = fma(0.5 * dt, ku, un);
    a.outR[o] = fma(0.5 * dt, kr, rn);
    return;
  }
  if (S == 4) {
    if (s < 4) {
      const double adt = (s == 3 ? 1.0 : 0.5) * dt;
      a.outU[o] = fma(adt, ku, un);
      a.outR[o] = fma(adt, kr, rn);
    } else {
      const double third = 1.0 / 3.0, dt6 = dt / 6.0;
      a.outU[o] = un + (third * ((a.U2[o] - un) + (U[0] - un)) + (2.0 * third) * (a.U3[o] - un)) + dt6 * ku;
      a.outR[o] = rn + (third * ((a.R2[o] - rn) + (R[0] - rn)) + (2.0 * third) * (a.R3[o] - rn)) + dt6 * kr;
      if (a.K4u) { a.K4u[o] = ku; a.K4r[o] = kr; }
    }
  } else if (S == 3) {
    if (s == 2) {  // Y_3 = y_n - dt k_1 + 2 dt k_2,  dt k_1 = 2 (Y_2 - y_n);  Y_2 is this stage's input
      a.outU[o] = un - 2.0 * (U[0] - un) + 2.0 * dt * ku;
      a.outR[o] = rn - 2.0 * (R[0] - rn) + 2.0 * dt * kr;
    } else {       // y_{n+1} = y_n + dt/6 (k_1 + 4 k_2 + k_3) = y_n + (Y_2 - y_n) + (Y_3 - y_n)/3 + dt/6 k_3;  Y_3 is the input
      const double dt6 = dt / 6.0;
      a.outU[o] = un + ((a.U2[o] - un) + (U[0] - un) * (1.0 / 3.0)) + dt6 * ku;
      a.outR[o] = rn + ((a.R2[o] - rn) + (R[0] - rn) * (1.0 / 3.0)) + dt6 * kr;
      if (a.K3u) { a.K3u[o] = ku; a.K3r[o] = kr; }
    }
  } else {         // RK2, s = 2: y_{n+1} = y_n + dt k_2
    a.outU[o] = fma(dt, ku, un);
    a.outR[o] = fma(dt, kr, rn);
    if (a.K4u) { a.K4u[o] = ku; a.K4r[o] = kr; }
  }
}

void launch_stage_ko_direct(const StageKOArgs& a, cudaStream_t st) {
  dim3 blk(64, 4, 1);
  dim3 grd((a.b.n[0] + 63) / 64, (a.b.n[1] + 3) / 4, a.b.n[2] * a.F);
  if (a.fd_order == 8) {
    if (a.ko_order == 9) stage_gen<8, 9><<<grd, blk, 0, st>>>(a);
    else if (a.ko_order == 5) stage_gen<8, 5><<<grd, blk, 0, st>>>(a);
    else stage_gen<8, 0><<<grd, blk, 0, st>>>(a);
  } else {
    if (a.ko_order == 9) stage_gen<4, 9><<<grd, blk, 0, st>>>(a);
    else if (a.ko_order == 5) stage_gen<4, 5><<<grd, blk, 0, st>>>(a);
    else stage_gen<4, 0><<<grd, blk, 0, st>>>(a);
  }
}

}  // namespace sc
