// restrict_zmarch.cu — tuned restriction kernel (PAPER.md:119 step 7; operator = reading
// S4: tensor-product quintic Lagrange (3,-25,150,150,-25,3)/256 on fine cells 2J-2 .. 2J+3 per axis).
//
// One CTA owns RPX x RPY parent columns and marches through a chunk of parent planes. Fine planes arrive in
// PAIRS (2m, 2m+1) as one TMA tiled load each (box = fine tile x 2 planes) into a ring of NSTR stages, so
// several pairs are always in flight and DRAM latency (and its tail) never meets a warp.
//   x: a thread owns two x-adjacent parents of one fine row: it reads the 8 fine values under them (four
//      16-byte shared loads, conflict-free by the lane -> (column, row) mapping and the 70-double pitch)
//      and reduces them to two x-restricted values per plane;
//   z: scatter form in registers — the pair completes parent plane m-1 and feeds the pending accumulators
//      of m and m+1 (by the symmetry of the operator the same code marches down);
//   y: only the completed x,z-restricted plane goes through shared memory (double-buffered, one
//      __syncthreads per pair) for the 6-point y reduction and the coalesced store.
// Neighbouring z-chunks march in opposite directions (as in stage_tma.cu) so their shared planes hit L2.
#include <cuda.h>

#include <cstdlib>

#include "kernels.h"
#include "launch_cfg.h"
#include "pdl.h"

namespace sc {

void launch_restrict_ref(const RestrictArgs& a, cudaStream_t st);

namespace {
constexpr int RPX = 32, RPY = 6;              // parent cells per CTA in x, y
constexpr int RFY = 2 * RPY + 4;              // 16 fine rows incl. the 2-row halo
constexpr int RPITCH = 2 * RPX + 6;           // 70: fine row incl. halo (68) + 2 pad columns (bank spread)
constexpr int RNT = 256;                      // 16 parent pairs x 16 fine rows
constexpr int RSTAGE = 2 * RFY * RPITCH;      // doubles per stage (one pair of fine planes) = 2240
constexpr int NSTR = 3;                       // pairs in flight (3 CTAs/SM x 3 x 17.5 KB)
constexpr int SXP = 40;                       // pitch of the x,z-restricted plane (bank spread)
constexpr double R0 = 3.0 / 256.0, R1 = -25.0 / 256.0, R2 = 150.0 / 256.0;
static_assert((RSTAGE * 8) % 128 == 0, "TMA destination must stay 128-byte aligned");
static_assert(RNT == (RPX / 2) * RFY, "one thread per (parent pair, fine row)");

__device__ __forceinline__ double lagr6(double a, double b, double c, double d, double e, double f) {
  return R0 * (a + f) + R1 * (b + e) + R2 * (c + d);
}
__device__ __forceinline__ uint32_t smem_u32r(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_wait_r(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
  } while (!ok);
}

struct RestrictParams {
  BoxView ch, pa;
  int a_child;       // array index (in the child's tensor map) of component 0 of the child's state
  int pz_per_cta, nzc;
  double* yp;        // parent state, component 0
};
}  // namespace

__global__ void __launch_bounds__(RNT, 3)
    restrict_zmarch(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ RestrictParams p) {
  pdl_enter();
  extern __shared__ unsigned char rsm[];
  const uint32_t s0 = (smem_u32r(rsm) + 127u) & ~127u;
  const double* const tiles = reinterpret_cast<const double*>(rsm + (s0 - smem_u32r(rsm)));  // [NSTR][2][RFY][RPITCH]
  double* const sX = const_cast<double*>(tiles) + NSTR * RSTAGE;                              // [2][RFY][SXP]
  const uint32_t bar0 = s0 + (NSTR * RSTAGE + 2 * RFY * SXP) * 8;

  const BoxView& ch = p.ch;
  const BoxView& pa = p.pa;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int xp = (lane & 3) | ((lane >> 3) << 2);   // parent pair 0..15  -> parents 2xp, 2xp+1
  const int row = 2 * warp + ((lane >> 2) & 1);     // fine row 0..15 of the tile
  const int X0 = blockIdx.x * RPX, Y0 = blockIdx.y * RPY;
  const int comp = blockIdx.z / p.nzc, chunk = blockIdx.z % p.nzc;
  const int npx = ch.n[0] / 2, npy = ch.n[1] / 2, npz = ch.n[2] / 2;
  const int Z0 = chunk * p.pz_per_cta, Z1 = min(Z0 + p.pz_per_cta, npz);
  const int dir = (chunk & 1) ? 1 : -1;
  const int npairs = Z1 - Z0 + 2;  // fine-plane pairs m = Z0-1 .. Z1
  auto pair_m = [&](int i) { return dir > 0 ? Z0 - 1 + i : Z1 - i; };
  auto issue = [&](int i) {
    const int st = i % NSTR;
    const uint32_t bar = bar0 + 8 * st;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(RSTAGE * 8) : "memory");
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, "
        "%5}], [%6];" ::"r"(s0 + st * RSTAGE * 8),
        "l"(&tmap), "r"(XOFF + 2 * X0 - 2), "r"(ch.g + 2 * Y0 - 2), "r"(ch.g + 2 * pair_m(i)), "r"(p.a_child + comp),
        "r"(bar)
        : "memory");
  };
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NSTR; ++s)
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar0 + 8 * s), "r"(1));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    for (int i = 0; i < NSTR && i < npairs; ++i) issue(i);
  }
  __syncthreads();

  const int P0 = (ch.lo[0] >> 1) - pa.lo[0], P1 = (ch.lo[1] >> 1) - pa.lo[1], P2 = (ch.lo[2] >> 1) - pa.lo[2];
  const int tx = tid % RPX, ty = tid / RPX;  // y-pass: one thread per parent cell (ty < RPY)
  const bool active = ty < RPY && (X0 + tx < npx) && (Y0 + ty < npy);
  double* __restrict__ dst = p.yp + (long long)comp * pa.vol + cell_offset(pa, P0 + X0 + tx, P1 + Y0 + ty, P2);
  double2 a0 = make_double2(0.0, 0.0), a1 = a0;  // pending z-accumulators: planes m - dir (completes next), m
  for (int i = 0; i < npairs; ++i) {
    const int st = i % NSTR;
    mbar_wait_r(bar0 + 8 * st, (i / NSTR) & 1);
    const double* t = tiles + st * RSTAGE + row * RPITCH + 4 * xp;
    double2 xr[2];  // x-restricted values of the two planes (lower z first)
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      const double2* r = reinterpret_cast<const double2*>(t + q * (RFY * RPITCH));
      const double2 a = r[0], b = r[1], c = r[2], d = r[3];
      xr[q] = make_double2(lagr6(a.x, a.y, b.x, b.y, c.x, c.y), lagr6(b.x, b.y, c.x, c.y, d.x, d.y));
    }
    const double2 f = dir > 0 ? xr[0] : xr[1], s = dir > 0 ? xr[1] : xr[0];  // first / second in marching order
    const double2 done = make_double2(a0.x + (R1 * f.x + R0 * s.x), a0.y + (R1 * f.y + R0 * s.y));
    a0 = make_double2(a1.x + R2 * (f.x + s.x), a1.y + R2 * (f.y + s.y));
    a1 = make_double2(R0 * f.x + R1 * s.x, R0 * f.y + R1 * s.y);
    double* sx = sX + (i & 1) * (RFY * SXP);
    if (i >= 2) *reinterpret_cast<double2*>(sx + row * SXP + 2 * xp) = done;
    __syncthreads();  // the x,z-restricted plane is visible; every thread is done with stage st
    if (tid == 0 && i + NSTR < npairs) issue(i + NSTR);
    if (i >= 2 && active) {
      const double* c = sx + 2 * ty * SXP + tx;
      dst[(long long)(pair_m(i) - dir) * pa.plane] =
          lagr6(c[0], c[SXP], c[2 * SXP], c[3 * SXP], c[4 * SXP], c[5 * SXP]);
    }
  }
}

namespace {
size_t restrict_smem() { return (size_t)(NSTR * RSTAGE + 2 * RFY * SXP) * 8 + NSTR * 8 + 128; }
}  // namespace

void restrict_box_dims(unsigned box[4]) { box[0] = RPITCH; box[1] = RFY; box[2] = 2; box[3] = 1; }

void launch_restrict_opt(const RestrictArgs& a, cudaStream_t st) {
  if (!a.tmap) { launch_restrict_ref(a, st); return; }
  static const int forced = [] { const char* e = getenv("SC_RCHUNKS"); return e ? atoi(e) : 0; }();
  const int nsm = device_sm_count();
  ensure_dynamic_smem(restrict_zmarch, restrict_smem());
  const BoxView& ch = a.child;
  const int npx = ch.n[0] / 2, npy = ch.n[1] / 2, npz = ch.n[2] / 2;
  const int gx = (npx + RPX - 1) / RPX, gy = (npy + RPY - 1) / RPY;
  // z-chunks: whole waves of CTAs (3 per SM), few halo pairs
  const long long cols = (long long)gx * gy * a.V, slots = 3LL * nsm;
  int best = 1;
  double best_cost = 1e300;
  const int maxch = npz / 4 > 1 ? npz / 4 : 1;
  for (int nch = 1; nch <= maxch; ++nch) {
    const int pz = (npz + nch - 1) / nch;
    const long long ctas = cols * ((npz + pz - 1) / pz);
    const double cost = (double)((ctas + slots - 1) / slots) * (pz + 2 + 3);
    if (cost < best_cost - 1e-9) { best_cost = cost; best = nch; }
  }
  if (forced > 0) best = forced < npz ? forced : npz;
  RestrictParams p{};
  p.ch = ch;
  p.pa = a.parent;
  p.a_child = a.a_child;
  p.pz_per_cta = (npz + best - 1) / best;
  p.nzc = (npz + p.pz_per_cta - 1) / p.pz_per_cta;
  p.yp = a.yparent;
  dim3 grd(gx, gy, p.nzc * a.V);
  launch_pdl(restrict_zmarch, grd, dim3(RNT), restrict_smem(), st, *static_cast<const CUtensorMap*>(a.tmap), p);
}

}  // namespace sc
