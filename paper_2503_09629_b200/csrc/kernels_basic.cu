// kernels_basic.cu — straightforward CUDA kernels of every step of the hot path (one thread per output
// cell, gathers straight from global memory). They define the arithmetic of the CUDA path; the tuned
// kernels (stage_tma.cu, ghost_tma.cu, restrict_zmarch.cu) must agree with them to rounding. Selected
// with SC_KERNELS=ref; also the home of the periodic fill, pack/unpack and the ghost-map debug kernel.
//
// Index conventions: box-local cell (i,j,k), i fastest; level-global index I = lo + i; the parent cell
// containing fine cell I is I >> 1 (arithmetic shift = floor), its parity I & 1 (1: fine centre at
// +dx_parent/4). Cell-centred grids (reading S1).
#include "kernels.h"
#include "pdl.h"

namespace sc {

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
// a1/a2  the RK4 stage kernels, direct-load version: one thread per interior cell, every operand read
// straight from global memory. Defines the arithmetic of the stage kernels (kernels.h); the TMA kernels
// in stage_tma.cu must agree with it to rounding. Used for SC_KERNELS=ref and for boxes the TMA path
// does not take.
// ------------------------------------------------------------------------------------------------
namespace {
// Laplacian of W = u + c r at one cell; c == 0 -> r is not read. ORDER 4: 13 points (S2), weights w = 1/(12 dx^2);
// ORDER 8: 25 points, (-1/560, 8/315, -1/5, 8/5, -205/72, ...)/dx^2 per axis.
template <bool WITH_R, int ORDER>
__device__ __forceinline__ double lap_w(const double* u, const double* r, double c, long long sy, long long sz,
                                        const double w[3], double* centre) {
  auto W = [&](long long d) { return WITH_R ? fma(c, r[d], u[d]) : u[d]; };
  const double wc = W(0);
  *centre = wc;
  if (ORDER == 8) {
    constexpr double c1 = 8.0 / 5.0, c2 = -1.0 / 5.0, c3 = 8.0 / 315.0, c4 = -1.0 / 560.0, c0 = -205.0 / 72.0;
    auto d2 = [&](long long s) {
      return c4 * (W(-4 * s) + W(4 * s)) + c3 * (W(-3 * s) + W(3 * s)) + c2 * (W(-2 * s) + W(2 * s)) +
             c1 * (W(-s) + W(s)) + c0 * wc;
    };
    return 12.0 * (w[0] * d2(1) + w[1] * d2(sy) + w[2] * d2(sz));
  }
  const double dxx = (-W(-2) + 16.0 * W(-1) - 30.0 * wc + 16.0 * W(1) - W(2)) * w[0];
  const double dyy = (-W(-2 * sy) + 16.0 * W(-sy) - 30.0 * wc + 16.0 * W(sy) - W(2 * sy)) * w[1];
  const double dzz = (-W(-2 * sz) + 16.0 * W(-sz) - 30.0 * wc + 16.0 * W(sz) - W(2 * sz)) * w[2];
  return dxx + dyy + dzz;
}
}  // namespace

template <int ORDER>
__global__ void __launch_bounds__(256) stage_direct(StageArgs a) {
  const BoxView& b = a.b;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z % b.n[2];
  const int f = blockIdx.z / b.n[2];
  if (i >= b.n[0] || j >= b.n[1]) return;
  const long long o = cell_offset(b, i, j, k);
  const long long sy = b.px, sz = b.plane;
  const int F = a.F;
  const long long fo = (long long)f * b.vol + o;
  const double* u = a.yn + fo;
  const double rho = a.yn[(long long)(F + f) * b.vol + o];
  const double dt = a.dt;
  // coupling  sum_q A_fq (u_q + c R_q)  at this cell
  auto couple = [&](double c, const double* R) {
    double s = 0.0;
    if (a.A)
      for (int q = 0; q < F; ++q) {
        const double uq = a.yn[(long long)q * b.vol + o];
        const double wq = R ? fma(c, R[(long long)q * b.vol + o], uq) : uq;
        s = fma(a.A[f * F + q], wq, s);
      }
    return s;
  };
  double wc;
  if (a.mode == STAGE_12) {
    const double* rhoarr = a.yn + (long long)F * b.vol;
    const double Lu = lap_w<false, ORDER>(u, u, 0.0, sy, sz, a.inv12dx2, &wc) + couple(0.0, nullptr);
    const double L2 = lap_w<true, ORDER>(u, rhoarr + fo, 0.5 * dt, sy, sz, a.inv12dx2, &wc) + couple(0.5 * dt, rhoarr);
    a.Y2r[fo] = fma(0.5 * dt, Lu, rho);
    a.Y3r[fo] = fma(0.5 * dt, L2, rho);
  } else {
    const double L3 = lap_w<true, ORDER>(u, a.Y2r + fo, 0.5 * dt, sy, sz, a.inv12dx2, &wc) + couple(0.5 * dt, a.Y2r);
    const double k4r = lap_w<true, ORDER>(u, a.Y3r + fo, dt, sy, sz, a.inv12dx2, &wc) + couple(dt, a.Y3r);
    const double y2 = a.Y2r[fo], y3 = a.Y3r[fo], y4 = fma(dt, L3, rho);
    const double third = 1.0 / 3.0;
    a.ynew[fo] = fma(dt / 6.0, (rho + y4) + 2.0 * (y2 + y3), u[0]);
    a.ynew[(long long)F * b.vol + fo] =
        rho + (third * ((y2 - rho) + (y4 - rho)) + (2.0 * third) * (y3 - rho)) + (dt / 6.0) * k4r;
    if (a.write_Y4r) a.Y4r[fo] = y4;
  }
}

void launch_stage_direct(const StageArgs& a, cudaStream_t st) {
  dim3 blk(64, 4, 1);
  dim3 grd((a.b.n[0] + 63) / 64, (a.b.n[1] + 3) / 4, a.b.n[2] * a.F);
  if (a.fd_order == 8) stage_direct<8><<<grd, blk, 0, st>>>(a);
  else stage_direct<4><<<grd, blk, 0, st>>>(a);
}

// ------------------------------------------------------------------------------------------------
// a3  ghost fill, direct version: one thread per (ghost cell, field), np^3-point gather per source (125 for S3)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) ghost_fill_direct(const __grid_constant__ GhostArgs a, int ip, long long nshell) {
  const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int f = blockIdx.y;
  if (q >= nshell) return;
  int i, j, k;
  if (!shell_cell(a.child, q, i, j, k)) return;
  const GhostProblem& pr = a.prob[ip];
  const int I[3] = {a.child.lo[0] + i, a.child.lo[1] + j, a.child.lo[2] + k};
  int J[3], p[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    J[d] = (I[d] >> 1) - a.parent.lo[d];
    p[d] = I[d] & 1;
  }
  double acc[GF_MAX_OUT];
#pragma unroll
  for (int o = 0; o < GF_MAX_OUT; ++o) acc[o] = 0.0;
  // tensor Lagrange stencil of a.np points per axis starting a.pmin parent cells from the containing one (S3; S30, S31)
  for (int cc = 0; cc < a.np; ++cc)
    for (int bb = 0; bb < a.np; ++bb) {
      const double wyz = a.w[p[1]][bb] * a.w[p[2]][cc];
      if (wyz == 0.0) continue;  // vertex-centred grids: a point ON a parent point has one non-zero weight per axis
      const long long row = cell_offset(a.parent, J[0] + a.pmin, J[1] + a.pmin + bb, J[2] + a.pmin + cc);
      for (int aa = 0; aa < a.np; ++aa) {
        const double w = wyz * a.w[p[0]][aa];
        if (w == 0.0) continue;
        double v[GF_MAX_SRC];
#pragma unroll
        for (int s = 0; s < GF_MAX_SRC; ++s)
          v[s] = s < pr.nsrc ? a.parent_base[(long long)(pr.src_arr[s] + f) * a.parent.vol + row + aa] : 0.0;
#pragma unroll
        for (int o = 0; o < GF_MAX_OUT; ++o) {
          if (o < pr.nout) {
            double t = 0.0;
#pragma unroll
            for (int s = 0; s < GF_MAX_SRC; ++s)
              if (s < pr.nsrc) t = fma(pr.coef[o][s], v[s], t);
            acc[o] = fma(w, t, acc[o]);
          }
        }
      }
    }
  const long long dofs = cell_offset(a.child, i, j, k);
#pragma unroll
  for (int o = 0; o < GF_MAX_OUT; ++o)
    if (o < pr.nout) a.child_base[(long long)(pr.dst_arr[o] + f) * a.child.vol + dofs] = acc[o];
}

void launch_ghost_fill_direct(const GhostArgs& a, cudaStream_t st) {
  const long long ns = ghost_cell_count(a.child);
  dim3 grd((unsigned)((ns + 127) / 128), a.F, 1);
  for (int ip = 0; ip < a.nprob; ++ip) ghost_fill_direct<<<grd, 128, 0, st>>>(a, ip, ns);
}

// ------------------------------------------------------------------------------------------------
// a4  periodic fill
// ------------------------------------------------------------------------------------------------
__device__ inline int wrap(int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); }

__global__ void __launch_bounds__(128) periodic_fill_ref(BoxView b, double* y, long long nshell) {
  pdl_enter();
  const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= nshell) return;
  int i, j, k;
  if (!shell_cell(b, q, i, j, k)) return;
  double* a = y + (long long)blockIdx.y * b.vol;
  a[cell_offset(b, i, j, k)] = a[cell_offset(b, wrap(i, b.n[0]), wrap(j, b.n[1]), wrap(k, b.n[2]))];
}

void launch_periodic_fill(const BoxView& b, int V, double* y, cudaStream_t st) {
  const long long ns = ghost_cell_count(b);
  dim3 grd((unsigned)((ns + 127) / 128), V, 1);
  launch_pdl(periodic_fill_ref, grd, dim3(128), 0, st, b, y, ns);
}

// ------------------------------------------------------------------------------------------------
// a7  same-level ghost exchange: one thread per cell of the region  padded(dst) n interior(src)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) sibling_copy(const SiblingPair* __restrict__ pairs, double* __restrict__ arena,
                                                    int first_array) {
  const SiblingPair& p = pairs[blockIdx.y];
  const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= (long long)p.n[0] * p.n[1] * p.n[2]) return;
  const int i = p.lo[0] + (int)(q % p.n[0]), j = p.lo[1] + (int)((q / p.n[0]) % p.n[1]),
            k = p.lo[2] + (int)(q / ((long long)p.n[0] * p.n[1]));
  const int arr = first_array + blockIdx.z;
  arena[p.dst_off + (long long)arr * p.dst.vol + cell_offset(p.dst, i - p.dst.lo[0], j - p.dst.lo[1], k - p.dst.lo[2])] =
      arena[p.src_off + (long long)arr * p.src.vol + cell_offset(p.src, i - p.src.lo[0], j - p.src.lo[1], k - p.src.lo[2])];
}

void launch_sibling_copy(const SiblingPair* pairs_dev, int npairs, long long maxcells, double* arena, int first_array,
                         int narrays, cudaStream_t st) {
  if (npairs <= 0 || narrays <= 0 || maxcells <= 0) return;
  dim3 grd((unsigned)((maxcells + 127) / 128), npairs, narrays);
  sibling_copy<<<grd, 128, 0, st>>>(pairs_dev, arena, first_array);
}

// ------------------------------------------------------------------------------------------------
// debug: max |x| over the interior. |x| of a NaN has a larger bit pattern than +inf, so the integer maximum of
// the bit patterns returns NaN if there is one, else +inf if there is one, else the largest magnitude.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) max_abs_kernel(BoxView b, const double* __restrict__ a,
                                                      unsigned long long* __restrict__ out) {
  const int j = blockIdx.x, k = blockIdx.y;
  unsigned long long m = 0ull;
  for (int i = threadIdx.x; i < b.n[0]; i += blockDim.x) {
    const unsigned long long bits = (unsigned long long)__double_as_longlong(fabs(a[cell_offset(b, i, j, k)]));
    m = bits > m ? bits : m;
  }
  for (int s = 16; s > 0; s >>= 1) {
    const unsigned long long o = __shfl_xor_sync(0xffffffffu, m, s);
    m = o > m ? o : m;
  }
  if ((threadIdx.x & 31) == 0 && m) atomicMax(out, m);
}
void launch_max_abs(const BoxView& b, const double* padded, unsigned long long* out_bits, cudaStream_t st) {
  dim3 grd(b.n[1], b.n[2], 1);
  max_abs_kernel<<<grd, 128, 0, st>>>(b, padded, out_bits);
}

// ------------------------------------------------------------------------------------------------
// measurement (sc_debug_stream): what a kernel that ONLY moves a stage kernel's bytes reaches on this device
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) stream_mix(const double2* __restrict__ in, double2* __restrict__ out,
                                                  unsigned long long n2, int nread, int nwrite) {
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < n2;
       i += (unsigned long long)gridDim.x * blockDim.x) {
    double2 s = make_double2(0.0, 0.0);
    for (int r = 0; r < nread; ++r) {
      const double2 v = in[r * n2 + i];
      s.x += v.x;
      s.y += v.y;
    }
    for (int w = 0; w < nwrite; ++w) out[w * n2 + i] = make_double2(s.x + w, s.y - w);
  }
}
void launch_stream_mix(const double* in, double* out, unsigned long long n, int nread, int nwrite, cudaStream_t st) {
  stream_mix<<<148 * 32, 256, 0, st>>>(reinterpret_cast<const double2*>(in), reinterpret_cast<double2*>(out), n / 2, nread,
                                       nwrite);
}

// ------------------------------------------------------------------------------------------------
// a5  restriction, one thread per parent cell, nr^3-point gather (216 for S4; 1 for injection on vertex-centred grids)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) restrict_ref(const __grid_constant__ RestrictArgs a) {
  const BoxView& ch = a.child;
  const BoxView& pa = a.parent;
  const int I = blockIdx.x * blockDim.x + threadIdx.x;
  const int J = blockIdx.y;
  const int nz = ch.n[2] / 2;
  const int K = blockIdx.z % nz;
  const int c = blockIdx.z / nz;
  if (I >= ch.n[0] / 2) return;
  const double* s = a.ychild + (long long)c * ch.vol;
  double sz = 0.0;
  for (int cc = 0; cc < a.nr; ++cc) {
    double sy = 0.0;
    for (int bb = 0; bb < a.nr; ++bb) {
      double sx = 0.0;
      const long long row = cell_offset(ch, 2 * I + a.rmin, 2 * J + a.rmin + bb, 2 * K + a.rmin + cc);
      for (int aa = 0; aa < a.nr; ++aa) sx += a.r[aa] * s[row + aa];
      sy += a.r[bb] * sx;
    }
    sz += a.r[cc] * sy;
  }
  const int P0 = (ch.lo[0] >> 1) - pa.lo[0], P1 = (ch.lo[1] >> 1) - pa.lo[1], P2 = (ch.lo[2] >> 1) - pa.lo[2];
  a.yparent[(long long)c * pa.vol + cell_offset(pa, P0 + I, P1 + J, P2 + K)] = sz;
}

void launch_restrict_ref(const RestrictArgs& a, cudaStream_t st) {
  dim3 grd((a.child.n[0] / 2 + 127) / 128, a.child.n[1] / 2, (a.child.n[2] / 2) * a.V);
  restrict_ref<<<grd, 128, 0, st>>>(a);
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
