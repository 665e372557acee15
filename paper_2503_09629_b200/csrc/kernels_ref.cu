// kernels_ref.cu — first, straightforward CUDA kernels of every step of the hot path (one thread per
// output cell, gathers straight from global memory). They define the arithmetic of the CUDA path; the
// tuned kernels in kernels_opt.cu must agree with them to rounding. Selected with SC_KERNELS=ref.
//
// Index conventions: box-local cell (i,j,k), i fastest; level-global index I = lo + i; the parent cell
// containing fine cell I is I >> 1 (arithmetic shift = floor), its parity I & 1 (1: fine centre at
// +dx_parent/4). Cell-centred grids (reading S1).
#include "kernels.h"

namespace sc {

// ------------------------------------------------------------------------------------------------
// weights (device constants; written out as exact binary fractions / rationals)
//   prolongation: quartic Lagrange at +-1/4 through offsets -2..2   (reading S3)
//   restriction:  quintic Lagrange at 0 through -5/2..5/2          (reading S4)
// ------------------------------------------------------------------------------------------------
__device__ __constant__ double c_wp[2][5] = {
    {-45.0 / 2048.0, 420.0 / 2048.0, 1890.0 / 2048.0, -252.0 / 2048.0, 35.0 / 2048.0},   // parity 0: x = -1/4
    {35.0 / 2048.0, -252.0 / 2048.0, 1890.0 / 2048.0, 420.0 / 2048.0, -45.0 / 2048.0}};  // parity 1: x = +1/4
__device__ __constant__ double c_wr[6] = {3.0 / 256.0,   -25.0 / 256.0, 150.0 / 256.0,
                                          150.0 / 256.0, -25.0 / 256.0, 3.0 / 256.0};

// ------------------------------------------------------------------------------------------------
// shell enumeration: q in [0, nshell) -> ghost cell (i,j,k); six slabs (z-lo, z-hi, y-lo, y-hi, x-lo, x-hi)
// ------------------------------------------------------------------------------------------------
long long ghost_cell_count(const BoxView& b) {
  const long long PX = b.n[0] + 2 * b.g, PY = b.n[1] + 2 * b.g, PZ = b.n[2] + 2 * b.g;
  return PX * PY * PZ - (long long)b.n[0] * b.n[1] * b.n[2];
}

__device__ inline bool shell_cell(const BoxView& b, long long q, int& i, int& j, int& k) {
  const int g = b.g;
  const long long PX = b.n[0] + 2 * g, PY = b.n[1] + 2 * g;
  const long long zs = (long long)g * PY * PX;      // one z slab
  const long long ys = (long long)b.n[2] * g * PX;  // one y slab
  const long long xs = (long long)b.n[2] * b.n[1] * g;
  if (q < 2 * zs) {
    const int hi = q >= zs;
    if (hi) q -= zs;
    k = (int)(q / (PY * PX));
    q -= (long long)k * PY * PX;
    j = (int)(q / PX) - g;
    i = (int)(q % PX) - g;
    k = hi ? b.n[2] + k : k - g;
    return true;
  }
  q -= 2 * zs;
  if (q < 2 * ys) {
    const int hi = q >= ys;
    if (hi) q -= ys;
    k = (int)(q / (g * PX));
    q -= (long long)k * g * PX;
    j = (int)(q / PX);
    i = (int)(q % PX) - g;
    j = hi ? b.n[1] + j : j - g;
    return true;
  }
  q -= 2 * ys;
  if (q < 2 * xs) {
    const int hi = q >= xs;
    if (hi) q -= xs;
    k = (int)(q / ((long long)b.n[1] * g));
    q -= (long long)k * b.n[1] * g;
    j = (int)(q / g);
    i = (int)(q % g);
    i = hi ? b.n[0] + i : i - g;
    return true;
  }
  return false;
}

// ------------------------------------------------------------------------------------------------
// a1/a2  rhs + stage combine
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) rhs_stage_ref(RhsArgs a) {
  const BoxView& b = a.b;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z % b.n[2];
  const int f = blockIdx.z / b.n[2];
  if (i >= b.n[0] || j >= b.n[1]) return;
  const long long o = cell_offset(b, i, j, k);
  const long long sx = 1, sy = b.px, sz = b.plane;
  const double* u = a.Yin + (long long)f * b.vol + o;
  const double* r = a.Yin + (long long)(a.F + f) * b.vol + o;
  const double uc = u[0];
  const double dxx = (-u[-2 * sx] + 16.0 * u[-sx] - 30.0 * uc + 16.0 * u[sx] - u[2 * sx]) * a.inv12dx2[0];
  const double dyy = (-u[-2 * sy] + 16.0 * u[-sy] - 30.0 * uc + 16.0 * u[sy] - u[2 * sy]) * a.inv12dx2[1];
  const double dzz = (-u[-2 * sz] + 16.0 * u[-sz] - 30.0 * uc + 16.0 * u[sz] - u[2 * sz]) * a.inv12dx2[2];
  double src = 0.0;
  if (a.A)
    for (int q = 0; q < a.F; ++q) src += a.A[f * a.F + q] * a.Yin[(long long)q * b.vol + o];
  const double ku = r[0];
  const double kr = dxx + dyy + dzz + src;
  const long long ou = (long long)f * b.vol + o, orr = (long long)(a.F + f) * b.vol + o;
  if (a.kout) {
    a.kout[ou] = ku;
    a.kout[orr] = kr;
  }
  if (a.stage < 4) {
    a.Yout[ou] = a.yn[ou] + a.cdt * ku;
    a.Yout[orr] = a.yn[orr] + a.cdt * kr;
  } else {
    a.Yout[ou] = a.yn[ou] + a.cdt * (a.k1[ou] + 2.0 * a.k2[ou] + 2.0 * a.k3[ou] + ku);
    a.Yout[orr] = a.yn[orr] + a.cdt * (a.k1[orr] + 2.0 * a.k2[orr] + 2.0 * a.k3[orr] + kr);
  }
}

void launch_rhs_stage_ref(const RhsArgs& a, cudaStream_t st) {
  dim3 blk(64, 4, 1);
  dim3 grd((a.b.n[0] + 63) / 64, (a.b.n[1] + 3) / 4, a.b.n[2] * a.F);
  rhs_stage_ref<<<grd, blk, 0, st>>>(a);
}

// ------------------------------------------------------------------------------------------------
// a3  dense output + prolongation, one thread per ghost cell, 125-point gather
// ------------------------------------------------------------------------------------------------
__device__ inline double combine_parent(const GhostArgs& a, long long off) {
  double v = a.base[off];
  if (a.use_k & 1) v += a.coef[0] * a.k[0][off];
  if (a.use_k & 2) v += a.coef[1] * a.k[1][off];
  if (a.use_k & 4) v += a.coef[2] * a.k[2][off];
  if (a.use_k & 8) v += a.coef[3] * a.k[3][off];
  return v;
}

__global__ void __launch_bounds__(128) ghost_fill_ref(GhostArgs a, long long nshell) {
  const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int c = blockIdx.y;
  if (q >= nshell) return;
  int i, j, k;
  if (!shell_cell(a.child, q, i, j, k)) return;
  const int I[3] = {a.child.lo[0] + i, a.child.lo[1] + j, a.child.lo[2] + k};
  int J[3], p[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    J[d] = (I[d] >> 1) - a.parent.lo[d];
    p[d] = I[d] & 1;
  }
  const long long pv = (long long)c * a.parent.vol;
  double sz = 0.0;
  for (int cc = -2; cc <= 2; ++cc) {
    double sy = 0.0;
    for (int bb = -2; bb <= 2; ++bb) {
      double sx = 0.0;
      const long long row = pv + cell_offset(a.parent, J[0], J[1] + bb, J[2] + cc);
#pragma unroll
      for (int aa = -2; aa <= 2; ++aa) sx += c_wp[p[0]][aa + 2] * combine_parent(a, row + aa);
      sy += c_wp[p[1]][bb + 2] * sx;
    }
    sz += c_wp[p[2]][cc + 2] * sy;
  }
  a.dst[(long long)c * a.child.vol + cell_offset(a.child, i, j, k)] = sz;
}

void launch_ghost_fill_ref(const GhostArgs& a, cudaStream_t st) {
  const long long ns = ghost_cell_count(a.child);
  dim3 grd((unsigned)((ns + 127) / 128), a.V, 1);
  ghost_fill_ref<<<grd, 128, 0, st>>>(a, ns);
}

// ------------------------------------------------------------------------------------------------
// a4  periodic fill
// ------------------------------------------------------------------------------------------------
__device__ inline int wrap(int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); }

__global__ void __launch_bounds__(128) periodic_fill_ref(BoxView b, double* y, long long nshell) {
  const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= nshell) return;
  int i, j, k;
  if (!shell_cell(b, q, i, j, k)) return;
  double* a = y + (long long)blockIdx.y * b.vol;
  a[cell_offset(b, i, j, k)] = a[cell_offset(b, wrap(i, b.n[0]), wrap(j, b.n[1]), wrap(k, b.n[2]))];
}

void launch_periodic_fill_ref(const BoxView& b, int V, double* y, cudaStream_t st) {
  const long long ns = ghost_cell_count(b);
  dim3 grd((unsigned)((ns + 127) / 128), V, 1);
  periodic_fill_ref<<<grd, 128, 0, st>>>(b, y, ns);
}

// ------------------------------------------------------------------------------------------------
// a5  restriction, one thread per parent cell, 216-point gather
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) restrict_ref(BoxView ch, BoxView pa, const double* yc, double* yp) {
  const int I = blockIdx.x * blockDim.x + threadIdx.x;
  const int J = blockIdx.y;
  const int nz = ch.n[2] / 2;
  const int K = blockIdx.z % nz;
  const int c = blockIdx.z / nz;
  if (I >= ch.n[0] / 2) return;
  const double* s = yc + (long long)c * ch.vol;
  double sz = 0.0;
  for (int cc = 0; cc < 6; ++cc) {
    double sy = 0.0;
    for (int bb = 0; bb < 6; ++bb) {
      double sx = 0.0;
      const long long row = cell_offset(ch, 2 * I - 2, 2 * J - 2 + bb, 2 * K - 2 + cc);
#pragma unroll
      for (int aa = 0; aa < 6; ++aa) sx += c_wr[aa] * s[row + aa];
      sy += c_wr[bb] * sx;
    }
    sz += c_wr[cc] * sy;
  }
  const int P0 = (ch.lo[0] >> 1) - pa.lo[0], P1 = (ch.lo[1] >> 1) - pa.lo[1], P2 = (ch.lo[2] >> 1) - pa.lo[2];
  yp[(long long)c * pa.vol + cell_offset(pa, P0 + I, P1 + J, P2 + K)] = sz;
}

void launch_restrict_ref(const BoxView& ch, const BoxView& pa, int V, const double* yc, double* yp,
                         cudaStream_t st) {
  dim3 grd((ch.n[0] / 2 + 127) / 128, ch.n[1] / 2, (ch.n[2] / 2) * V);
  restrict_ref<<<grd, 128, 0, st>>>(ch, pa, yc, yp);
}

// ------------------------------------------------------------------------------------------------
// pack / unpack / ghost map
// ------------------------------------------------------------------------------------------------
__global__ void pack_kernel(BoxView b, const double* padded, double* dense, int e) {
  const int nx = b.n[0] + 2 * e, ny = b.n[1] + 2 * e;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y, k = blockIdx.z;
  if (i >= nx) return;
  dense[(long long)i + (long long)nx * (j + (long long)ny * k)] = padded[cell_offset(b, i - e, j - e, k - e)];
}

__global__ void unpack_kernel(BoxView b, const double* dense, double* padded) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y, k = blockIdx.z;
  if (i >= b.n[0]) return;
  padded[cell_offset(b, i, j, k)] = dense[(long long)i + (long long)b.n[0] * (j + (long long)b.n[1] * k)];
}

void launch_pack(const BoxView& b, const double* padded, double* dense, int with_ghosts, cudaStream_t st) {
  const int e = with_ghosts ? b.g : 0;
  dim3 grd((b.n[0] + 2 * e + 127) / 128, b.n[1] + 2 * e, b.n[2] + 2 * e);
  pack_kernel<<<grd, 128, 0, st>>>(b, padded, dense, e);
}

void launch_unpack(const BoxView& b, const double* dense, double* padded, cudaStream_t st) {
  dim3 grd((b.n[0] + 127) / 128, b.n[1], b.n[2]);
  unpack_kernel<<<grd, 128, 0, st>>>(b, dense, padded);
}

__global__ void ghost_map_kernel(BoxView ch, BoxView pa, int* out, long long nshell) {
  const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= nshell) return;
  int i, j, k;
  if (!shell_cell(ch, q, i, j, k)) return;
  // rank of (k,j,i) in canonical order = padded cells before it minus interior cells before it
  const int g = ch.g;
  const long long PX = ch.n[0] + 2 * g, PY = ch.n[1] + 2 * g;
  const long long before = ((long long)(k + g) * PY + (j + g)) * PX + (i + g);
  long long inter;
  if (k < 0) inter = 0;
  else if (k >= ch.n[2]) inter = (long long)ch.n[0] * ch.n[1] * ch.n[2];
  else {
    long long inrow = j < 0 ? 0 : (j >= ch.n[1] ? (long long)ch.n[1] * ch.n[0]
                                                : (long long)j * ch.n[0] + (i < 0 ? 0 : (i >= ch.n[0] ? ch.n[0] : i)));
    inter = (long long)k * ch.n[1] * ch.n[0] + inrow;
  }
  int* o = out + 7 * (before - inter);
  const int I[3] = {ch.lo[0] + i, ch.lo[1] + j, ch.lo[2] + k};
  o[0] = i; o[1] = j; o[2] = k;
  o[3] = (I[0] >> 1) - pa.lo[0];
  o[4] = (I[1] >> 1) - pa.lo[1];
  o[5] = (I[2] >> 1) - pa.lo[2];
  o[6] = (I[0] & 1) | ((I[1] & 1) << 1) | ((I[2] & 1) << 2);
}

void launch_ghost_map(const BoxView& ch, const BoxView& pa, int* out, cudaStream_t st) {
  const long long ns = ghost_cell_count(ch);
  ghost_map_kernel<<<(unsigned)((ns + 127) / 128), 128, 0, st>>>(ch, pa, out, ns);
}

}  // namespace sc
