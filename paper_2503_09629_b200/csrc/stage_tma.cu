// stage_tma.cu — tuned RK4 stage kernels (eqs 1-9 on the wave system
// PAPER.md:222-226), sm_100a: z-march with TMA-staged halo planes.
//
// One CTA owns a TX x TY column of cells (32 x 16 or 64 x 7, chosen per box: Tile) and marches through a chunk of z-planes. Every plane of every
// halo-read array arrives in shared memory as a (TX+4) x (TY+4) tile through ONE TMA tiled load
// (cp.async.bulk.tensor.4d, box dims (x, y, 1 plane, 1 array)) signalled on an mbarrier; NST planes are in
// flight so HBM latency never meets a warp. A thread owns two x-adjacent cells (16-byte shared loads and
// 16-byte coalesced global stores) and NEVER re-reads a plane: the 4th-order Laplacian (S2) is applied in
// scatter form — when plane p arrives its in-plane part goes to the accumulator of output plane p and its
// value to the accumulators of p-2, p-1, p+1, p+2 — so the z-direction lives in registers and each shared
// value is loaded once. Output plane p-2 is complete when plane p has arrived.
// Algorithmic traffic per cell and field (doubles): STAGE_12 reads u, rho, writes Y2r, Y3r (4);
// STAGE_34 reads u, rho, Y2r, Y3r, writes u_new, rho_new [, Y4r] (6 or 7). 10-11 per RK4 step.
// Neighbouring z-chunks march in OPPOSITE directions away from / towards their common boundary, so the 4
// halo planes two chunks share are requested at the same time and the second request hits L2.
#include <cuda.h>

#include <cstdlib>
#include <cstring>
#include <type_traits>

#include "kernels.h"
#include "launch_cfg.h"
#include "pdl.h"

namespace sc {

void launch_stage_direct(const StageArgs& a, cudaStream_t st);
int stage_tile_variant(const BoxView& b, int F);

namespace {

// Tile of cells per CTA column, chosen per box (stage_tile_variant): 32 x 16 — 256 threads, halo tile 36 x 20 — or
// 64 x 7 — 224 threads, halo tile 68 x 11. The second exists for boxes like 256^3, where 32 x 16 gives 128 columns x 2
// z-chunks = 256 CTAs on the 296 resident slots of 148 SMs (40 SMs then carry one CTA and the launch lasts as long as
// the SMs that carry two), while 64 x 7 gives 4 x 37 = 148 columns x 2 chunks = two CTAs on EVERY SM, all marching
// in lock step: 136.5 -> 130.9 us per launch although its halo is larger (1.67x the interior instead of 1.41x).
template <int TX_, int TY_> struct Tile {
  static constexpr int TX = TX_, TY = TY_;
  static constexpr int HX = TX + 4, HY = TY + 4;      // halo tile
  static constexpr int NTHR = (TX / 2) * TY;          // two x-adjacent cells per thread
  static constexpr int TILE_BYTES = HX * HY * 8;      // what one TMA tiled load writes
  static constexpr int TILE_DOUBLES = (TILE_BYTES + 127) / 128 * 16;  // distance between tiles in shared memory (128-byte aligned)
};
using TileA = Tile<32, 16>;
using TileB = Tile<64, 7>;
// Tile B's 224 compute threads leave room for a PRODUCER warp inside the 256-thread, 128-register budget of two CTAs per
// SM: warp 7 does nothing but wait for a ring stage to be released (an mbarrier the 7 compute warps arrive on when they
// have read it) and refill it by TMA. The compute warps then never meet in a CTA barrier: they drift up to NST - 1
// planes apart inside a CTA while the CTAs of neighbouring columns stay together (the ring depth bounds the drift).
template <class T> struct Spec { static constexpr bool WS = false; static constexpr int THREADS = T::NTHR; };
template <> struct Spec<TileB> { static constexpr bool WS = true; static constexpr int THREADS = TileB::NTHR + 32; };
constexpr int NST = 4;                       // planes in flight

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
  } while (!ok);
}
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, int c3,
                                            uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, "
      "%5}], [%6];" ::"r"(dst),
      "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar)
      : "memory");
}

struct TmaStageParams {
  BoxView b;
  int F, nchunks, chunk, write_Y4r;
  int a_yn, a_Y2r, a_Y3r;
  const double* yn;
  double* Y2r;
  double* Y3r;
  double* Y4r;
  double* ynew;
  double dt;
  double w[3];  // 1 / (12 dx_a^2)
  const double* S;  // coupled systems: F arrays A*(first stage operand), then F arrays A*(second), from couple_matvec
};

// values of one array around the thread's two cells (x, x+1) in the current plane
struct Nbr {
  double2 xa, xb, xc;          // row y: columns x-2..x+3
  double2 ym2, ym1, yp1, yp2;  // columns x, x+1 of rows y-2, y-1, y+1, y+2
};
template <int HX>
__device__ __forceinline__ Nbr load_nbr(const double* tile, int tx, int ty) {
  Nbr n;
  const double2* r = reinterpret_cast<const double2*>(tile + (ty + 2) * HX + 2 * tx);
  n.xa = r[0]; n.xb = r[1]; n.xc = r[2];
  n.ym2 = *reinterpret_cast<const double2*>(tile + (ty + 0) * HX + 2 * tx + 2);
  n.ym1 = *reinterpret_cast<const double2*>(tile + (ty + 1) * HX + 2 * tx + 2);
  n.yp1 = *reinterpret_cast<const double2*>(tile + (ty + 3) * HX + 2 * tx + 2);
  n.yp2 = *reinterpret_cast<const double2*>(tile + (ty + 4) * HX + 2 * tx + 2);
  return n;
}
template <int HX>
__device__ __forceinline__ double2 load_centre(const double* tile, int tx, int ty) {
  return *reinterpret_cast<const double2*>(tile + (ty + 2) * HX + 2 * tx + 2);
}
__device__ __forceinline__ double2 fma2(double c, double2 a, double2 b) {
  return make_double2(fma(c, a.x, b.x), fma(c, a.y, b.y));
}
__device__ __forceinline__ Nbr axpy(double c, const Nbr& r, const Nbr& u) {  // u + c r
  Nbr n;
  n.xa = fma2(c, r.xa, u.xa); n.xb = fma2(c, r.xb, u.xb); n.xc = fma2(c, r.xc, u.xc);
  n.ym2 = fma2(c, r.ym2, u.ym2); n.ym1 = fma2(c, r.ym1, u.ym1);
  n.yp1 = fma2(c, r.yp1, u.yp1); n.yp2 = fma2(c, r.yp2, u.yp2);
  return n;
}
// in-plane part of the 13-point Laplacian at the two cells: wx d_xx + wy d_yy - 30 wz centre
__device__ __forceinline__ double2 inplane(const Nbr& n, double wx, double wy, double c30) {
  const double x0 = 16.0 * (n.xa.y + n.xb.y) - (n.xa.x + n.xc.x);
  const double x1 = 16.0 * (n.xb.x + n.xc.x) - (n.xa.y + n.xc.y);
  const double y0 = 16.0 * (n.ym1.x + n.yp1.x) - (n.ym2.x + n.yp2.x);
  const double y1 = 16.0 * (n.ym1.y + n.yp1.y) - (n.ym2.y + n.yp2.y);
  return make_double2(fma(wx, x0, fma(wy, y0, -c30 * n.xb.x)), fma(wx, x1, fma(wy, y1, -c30 * n.xb.y)));
}

// Scatter one arrived plane into the five pending accumulators. R = arrival index mod 5 (compile time), so
// slot (R + d) mod 5 belongs to output plane (arrival + d). The slot of arrival + 2 is created here.
template <int R>
__device__ __forceinline__ void scatter(double2 (&acc)[5], double2 centre_term, double2 zc) {
  acc[(R + 3) % 5].x -= zc.x;                      acc[(R + 3) % 5].y -= zc.y;
  acc[(R + 4) % 5].x = fma(16.0, zc.x, acc[(R + 4) % 5].x);
  acc[(R + 4) % 5].y = fma(16.0, zc.y, acc[(R + 4) % 5].y);
  acc[R].x += centre_term.x;                       acc[R].y += centre_term.y;
  acc[(R + 1) % 5].x = fma(16.0, zc.x, acc[(R + 1) % 5].x);
  acc[(R + 1) % 5].y = fma(16.0, zc.y, acc[(R + 1) % 5].y);
  acc[(R + 2) % 5] = make_double2(-zc.x, -zc.y);
}

}  // namespace

template <int MODE, bool COUPLED, class T>
__global__ void __launch_bounds__(Spec<T>::THREADS, 2)
    stage_zmarch(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ TmaStageParams p) {
  constexpr int NH = MODE == STAGE_12 ? 2 : 3;  // halo-read arrays per plane
  constexpr int TX = T::TX, TY = T::TY, HX = T::HX, TILE_DOUBLES = T::TILE_DOUBLES;
  constexpr bool WS = Spec<T>::WS;
  pdl_enter();
  extern __shared__ unsigned char smraw[];
  // [NST][NH] tiles, 128-byte aligned for TMA, then NST mbarriers
  const uint32_t s0 = (smem_u32(smraw) + 127u) & ~127u;
  double* const tiles = reinterpret_cast<double*>(smraw + (s0 - smem_u32(smraw)));
  const uint32_t bar0 = s0 + NST * NH * TILE_DOUBLES * 8;

  const BoxView& b = p.b;
  const int tid = threadIdx.x, tx = tid % (TX / 2), ty = tid / (TX / 2);
  const int X0 = blockIdx.x * TX, Y0 = blockIdx.y * TY;
  const int f = blockIdx.z / p.nchunks, c = blockIdx.z % p.nchunks;
  const int zc0 = c * p.chunk, zc1 = min(b.n[2], zc0 + p.chunk);
  const int narr = zc1 - zc0 + 4;              // planes that arrive: the chunk plus 2 halo planes each side
  const int dir = (c & 1) ? 1 : -1;            // neighbouring chunks march in opposite directions
  const int zs = dir > 0 ? zc0 - 2 : zc1 + 1;  // first plane to arrive
  int arr[NH];
  arr[0] = p.a_yn + f;
  if (MODE == STAGE_12) arr[1] = p.a_yn + p.F + f;
  else { arr[1] = p.a_Y2r + f; arr[NH - 1] = p.a_Y3r + f; }

  auto issue = [&](int it) {  // one thread: arm the stage's mbarrier and request the plane's tiles
    const int st = it % NST;
    const uint32_t bar = bar0 + 8 * st;
    mbar_expect_tx(bar, NH * T::TILE_BYTES);
#pragma unroll
    for (int h = 0; h < NH; ++h)
      tma_load_4d(s0 + (st * NH + h) * TILE_DOUBLES * 8, &tmap, XOFF + X0 - 2, b.g + Y0 - 2, b.g + zs + dir * it,
                  arr[h], bar);
  };
  const uint32_t ebar0 = bar0 + 8 * NST;  // WS: the "stage released" barriers
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NST; ++s) {
      mbar_init(bar0 + 8 * s, 1);
      if (WS) mbar_init(ebar0 + 8 * s, T::NTHR / 32);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if (!WS)
      for (int it = 0; it < NST && it < narr; ++it) issue(it);
  }
  __syncthreads();
  if (WS && tid >= T::NTHR) {  // the producer warp: one lane feeds the ring for the whole march
    if (tid == T::NTHR) {
      for (int it = 0; it < narr; ++it) {
        if (it >= NST) mbar_wait(ebar0 + 8 * (it % NST), ((it / NST) - 1) & 1);
        issue(it);
      }
    }
    return;
  }

  const bool active = (X0 + 2 * tx < b.n[0]) && (Y0 + ty < b.n[1]);
  const long long cell0 = cell_offset(b, X0 + 2 * tx, Y0 + ty, 0);
  const double dt = p.dt, hdt = 0.5 * p.dt, third = 1.0 / 3.0, dt6 = p.dt / 6.0;
  // accumulator A collects Y2r (STAGE_12) / Y4r (STAGE_34); B collects Y3r / rho_new - Y4r/3
  const double sA = MODE == STAGE_12 ? hdt : dt, sB = MODE == STAGE_12 ? hdt : dt6;
  const double wxA = sA * p.w[0], wyA = sA * p.w[1], wzA = sA * p.w[2], cA = 30.0 * (wxA + wyA + wzA);
  const double wxB = sB * p.w[0], wyB = sB * p.w[1], wzB = sB * p.w[2], cB = 30.0 * (wxB + wyB + wzB);
  double2 accA[5], accB[5], Pu[5];
#pragma unroll
  for (int q = 0; q < 5; ++q) accA[q] = accB[q] = Pu[q] = make_double2(0.0, 0.0);
  const double* __restrict__ rho_g = p.yn + (long long)(p.F + f) * b.vol + cell0;
  double2 rho_nxt = make_double2(0.0, 0.0);
  (void)rho_g;
  // coupling terms (A W)_f of the two stage operands at the centre cells, read like rho_n: one plane ahead
  const double* __restrict__ s1_g = COUPLED ? p.S + (long long)f * b.vol + cell0 : nullptr;
  const double* __restrict__ s2_g = COUPLED ? p.S + (long long)(p.F + f) * b.vol + cell0 : nullptr;
  double2 s1_nxt = make_double2(0.0, 0.0), s2_nxt = s1_nxt;

  auto step = [&](auto Rc, int it) {
    constexpr int R = decltype(Rc)::value;
    const int st = it % NST;
    const bool inpl = it >= 2 && it < narr - 2;
    const int z = zs + dir * it;
    double2 rho_c = rho_nxt;
    const double2 s1_c = s1_nxt, s2_c = s2_nxt;
    {
      const int itn = it + 1;
      if (active && itn >= 2 && itn < narr - 2) {
        const long long zo = (long long)(z + dir) * b.plane;
        if (MODE == STAGE_34)  // rho_n is read at the centre only: plain global load, one plane ahead
          rho_nxt = __ldg(reinterpret_cast<const double2*>(rho_g + zo));
        if (COUPLED) {
          s1_nxt = __ldg(reinterpret_cast<const double2*>(s1_g + zo));
          s2_nxt = __ldg(reinterpret_cast<const double2*>(s2_g + zo));
        }
      }
    }
    mbar_wait(bar0 + 8 * st, (it / NST) & 1);
    const double* __restrict__ t0 = tiles + (st * NH) * TILE_DOUBLES;
    double2 ctA = make_double2(0.0, 0.0), ctB = ctA, zcA, zcB;
    if (MODE == STAGE_12) {
      if (inpl) {
        const Nbr u = load_nbr<HX>(t0, tx, ty), r = load_nbr<HX>(t0 + TILE_DOUBLES, tx, ty);
        const Nbr w = axpy(hdt, r, u);
        const double2 iu = inplane(u, wxA, wyA, cA), iw = inplane(w, wxB, wyB, cB);
        ctA = make_double2(r.xb.x + iu.x, r.xb.y + iu.y);
        ctB = make_double2(r.xb.x + iw.x, r.xb.y + iw.y);
        if (COUPLED) { ctA = fma2(hdt, s1_c, ctA); ctB = fma2(hdt, s2_c, ctB); }
        zcA = make_double2(wzA * u.xb.x, wzA * u.xb.y);
        zcB = make_double2(wzB * w.xb.x, wzB * w.xb.y);
      } else {
        const double2 uc = load_centre<HX>(t0, tx, ty), rc = load_centre<HX>(t0 + TILE_DOUBLES, tx, ty);
        const double2 wc = fma2(hdt, rc, uc);
        zcA = make_double2(wzA * uc.x, wzA * uc.y);
        zcB = make_double2(wzB * wc.x, wzB * wc.y);
      }
    } else {
      if (inpl) {
        const Nbr u = load_nbr<HX>(t0, tx, ty);
        const Nbr y2 = load_nbr<HX>(t0 + TILE_DOUBLES, tx, ty), y3 = load_nbr<HX>(t0 + 2 * TILE_DOUBLES, tx, ty);
        const Nbr w3 = axpy(hdt, y2, u), w4 = axpy(dt, y3, u);
        const double2 i3 = inplane(w3, wxA, wyA, cA), i4 = inplane(w4, wxB, wyB, cB);
        ctA = make_double2(rho_c.x + i3.x, rho_c.y + i3.y);
        const double prx = rho_c.x + (third * (y2.xb.x - rho_c.x) + (2.0 * third) * (y3.xb.x - rho_c.x)) - third * rho_c.x;
        const double pry = rho_c.y + (third * (y2.xb.y - rho_c.y) + (2.0 * third) * (y3.xb.y - rho_c.y)) - third * rho_c.y;
        ctB = make_double2(prx + i4.x, pry + i4.y);
        if (COUPLED) { ctA = fma2(dt, s1_c, ctA); ctB = fma2(dt6, s2_c, ctB); }
        Pu[R] = make_double2(fma(dt6, rho_c.x + 2.0 * (y2.xb.x + y3.xb.x), u.xb.x),
                             fma(dt6, rho_c.y + 2.0 * (y2.xb.y + y3.xb.y), u.xb.y));
        zcA = make_double2(wzA * w3.xb.x, wzA * w3.xb.y);
        zcB = make_double2(wzB * w4.xb.x, wzB * w4.xb.y);
      } else {
        const double2 uc = load_centre<HX>(t0, tx, ty);
        const double2 w3 = fma2(hdt, load_centre<HX>(t0 + TILE_DOUBLES, tx, ty), uc);
        const double2 w4 = fma2(dt, load_centre<HX>(t0 + 2 * TILE_DOUBLES, tx, ty), uc);
        zcA = make_double2(wzA * w3.x, wzA * w3.y);
        zcB = make_double2(wzB * w4.x, wzB * w4.y);
      }
    }
    scatter<R>(accA, ctA, zcA);
    scatter<R>(accB, ctB, zcB);
    if (it >= 4 && active) {  // output plane z - 2 dir is complete
      const long long o = (long long)f * b.vol + cell0 + (long long)(z - 2 * dir) * b.plane;
      const double2 a = accA[(R + 3) % 5], bb = accB[(R + 3) % 5];
      if (MODE == STAGE_12) {
        *reinterpret_cast<double2*>(p.Y2r + o) = a;
        *reinterpret_cast<double2*>(p.Y3r + o) = bb;
      } else {
        const double2 pu = Pu[(R + 3) % 5];
        *reinterpret_cast<double2*>(p.ynew + o) = make_double2(fma(dt6, a.x, pu.x), fma(dt6, a.y, pu.y));
        *reinterpret_cast<double2*>(p.ynew + (long long)p.F * b.vol + o) =
            make_double2(fma(third, a.x, bb.x), fma(third, a.y, bb.y));
        if (p.write_Y4r) *reinterpret_cast<double2*>(p.Y4r + o) = a;
      }
    }
    if (WS) {         // release stage st: the producer refills it once all compute warps have
      __syncwarp();
      if ((tid & 31) == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(ebar0 + 8 * st) : "memory");
    } else {
      __syncthreads();  // every thread is done with stage st: refill it with the plane NST arrivals ahead
      if (tid == 0 && it + NST < narr) issue(it + NST);
    }
  };

  for (int it0 = 0; it0 < narr; it0 += 5) {
    step(std::integral_constant<int, 0>{}, it0);
    if (it0 + 1 < narr) step(std::integral_constant<int, 1>{}, it0 + 1);
    if (it0 + 2 < narr) step(std::integral_constant<int, 2>{}, it0 + 2);
    if (it0 + 3 < narr) step(std::integral_constant<int, 3>{}, it0 + 3);
    if (it0 + 4 < narr) step(std::integral_constant<int, 4>{}, it0 + 4);
  }
}

// ---- host ------------------------------------------------------------------------------------------
namespace {

using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled() {
  static EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) != cudaSuccess ||
        qr != cudaDriverEntryPointSuccess) {
      cudaGetLastError();
      p = nullptr;
    }
    return reinterpret_cast<EncodeTiledFn>(p);
  }();
  return fn;
}

template <int MODE, class T>
size_t stage_smem() { return (size_t)NST * (MODE == STAGE_12 ? 2 : 3) * T::TILE_DOUBLES * 8 + 2 * NST * 8 + 128; }

// z-chunks per column of tx x ty cells: enough CTAs to fill the machine in whole waves, as few halo planes as possible.
// *cost_out: waves x (planes marched + pipeline fill), the launch's length in plane-steps of one CTA.
int pick_chunks_impl(const BoxView& b, int F, int ctas_per_sm, int halo_planes, int tx = 32, int ty = 16,
                     double* cost_out = nullptr) {
  static const int forced = [] { const char* e = getenv("SC_ZCHUNKS"); return e ? atoi(e) : 0; }();
  const int nsm = device_sm_count();
  const long long cols = (long long)((b.n[0] + tx - 1) / tx) * ((b.n[1] + ty - 1) / ty) * F;
  const long long slots = (long long)nsm * ctas_per_sm;
  int best = 1;
  double best_cost = 1e300;
  const int maxch = b.n[2] / 8 > 1 ? b.n[2] / 8 : 1;
  for (int nch = 1; nch <= maxch; ++nch) {
    if (forced > 0 && nch != (forced < b.n[2] ? forced : b.n[2])) continue;
    const int ch = (b.n[2] + nch - 1) / nch;
    const long long ctas = cols * ((b.n[2] + ch - 1) / ch);
    const long long waves = (ctas + slots - 1) / slots;
    const double cost = (double)waves * (ch + halo_planes + 6);  // time ~ waves x (planes marched + pipeline fill)
    if (cost < best_cost - 1e-9) { best_cost = cost; best = nch; }
  }
  if (cost_out) *cost_out = best_cost;
  return best;
}

template <class T>
double tile_cost(const BoxView& b, int F) {
  // a CTA's time per plane grows with its cells; the larger halo of a flatter tile costs about a third of its share
  // (measured on 256^3: 64 x 7 against 32 x 16, see Tile)
  double planes = 0.0;
  pick_chunks_impl(b, F, 2, 4, T::TX, T::TY, &planes);
  const double halo = (double)(T::HX * T::HY) / (T::TX * T::TY);
  return planes * T::TX * T::TY * (1.0 + 0.3 * (halo - 1.0));
}

template <int MODE, bool COUPLED, class T>
void launch_zmarch(const StageArgs& a, cudaStream_t st) {
  ensure_dynamic_smem(stage_zmarch<MODE, COUPLED, T>, stage_smem<MODE, T>());
  TmaStageParams p{};
  p.b = a.b;
  p.F = a.F;
  p.nchunks = pick_chunks_impl(a.b, a.F, 2, 4, T::TX, T::TY);
  p.chunk = (a.b.n[2] + p.nchunks - 1) / p.nchunks;
  p.nchunks = (a.b.n[2] + p.chunk - 1) / p.chunk;
  p.write_Y4r = a.write_Y4r;
  p.a_yn = a.a_yn; p.a_Y2r = a.a_Y2r; p.a_Y3r = a.a_Y3r;
  p.yn = a.yn; p.Y2r = a.Y2r; p.Y3r = a.Y3r; p.Y4r = a.Y4r; p.ynew = a.ynew;
  p.dt = a.dt;
  for (int d = 0; d < 3; ++d) p.w[d] = a.inv12dx2[d];
  p.S = a.S;
  dim3 grd((a.b.n[0] + T::TX - 1) / T::TX, (a.b.n[1] + T::TY - 1) / T::TY, p.nchunks * a.F);
  launch_pdl(stage_zmarch<MODE, COUPLED, T>, grd, dim3(Spec<T>::THREADS), stage_smem<MODE, T>(), st,
             *static_cast<const CUtensorMap*>(a.tmap), p);
}
template <int MODE, bool COUPLED>
void launch_zmarch_v(const StageArgs& a, cudaStream_t st) {
  if (a.tile_variant) launch_zmarch<MODE, COUPLED, TileB>(a, st);  // the tile the box's tensor map was built for
  else launch_zmarch<MODE, COUPLED, TileA>(a, st);
}

}  // namespace

// ---- coupled systems: the pointwise F x F product -------------------------------------------------------
// d_t rho_f = Lap u_f + sum_q A_fq u_q (PAPER.md:222-226 with BASELINE config 4's coupling, S21/S22). The
// Laplacian acts field by field, the coupling cell by cell across ALL fields; they are split accordingly: this
// kernel forms, at every interior cell, the coupling terms of the two stage operands W1, W2 of the following
// z-march launch,
//   STAGE_12:  W1 = u_n,               W2 = u_n + dt/2 rho_n
//   STAGE_34:  W1 = u_n + dt/2 Y2r,    W2 = u_n + dt Y3r
// S[f] = sum_q A_fq W1_q,  S[F + f] = sum_q A_fq W2_q, and the z-march kernel adds them at the centre cell.
// One thread per cell: all F operand pairs in registers (every global load issued up front), A in the
// constant bank (kernel parameter). 2 F^2 FMA per cell against (2|3) F reads + 2 F writes.
namespace {
template <int FB> struct CoupleMatrix { double a[FB * FB]; };  // row-major, zero-padded to FB x FB

// The matrix travels as a KERNEL PARAMETER (up to 8 KB; parameters may be 32 KB since CUDA 12.1): with both
// loops unrolled every A_fq is an immediate constant-bank operand of its FMA — no shared-memory traffic at
// all (the shared-memory version spent one broadcast LDS per FMA pair and ran at 40-53 % of DRAM peak).
template <int MODE, int FB>
__global__ void __launch_bounds__(128)
    couple_matvec(const __grid_constant__ TmaStageParams p, const __grid_constant__ CoupleMatrix<FB> A) {
  const BoxView& b = p.b;
  const int F = p.F;
  const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 4 + threadIdx.y, k = blockIdx.z;
  if (i >= b.n[0] || j >= b.n[1]) return;
  const long long o = cell_offset(b, i, j, k);
  const double hdt = 0.5 * p.dt;
  double w1[FB], w2[FB];
#pragma unroll
  for (int q = 0; q < FB; ++q) {
    if (q < F) {
      const double u = __ldg(p.yn + (long long)q * b.vol + o);
      if (MODE == STAGE_12) {
        w1[q] = u;
        w2[q] = fma(hdt, __ldg(p.yn + (long long)(F + q) * b.vol + o), u);
      } else {
        w1[q] = fma(hdt, __ldg(p.Y2r + (long long)q * b.vol + o), u);
        w2[q] = fma(p.dt, __ldg(p.Y3r + (long long)q * b.vol + o), u);
      }
    } else {
      w1[q] = w2[q] = 0.0;
    }
  }
  double* __restrict__ S = const_cast<double*>(p.S);
#pragma unroll
  for (int f = 0; f < FB; ++f) {
    if (f < F) {
      double s1 = 0.0, s2 = 0.0;
#pragma unroll
      for (int q = 0; q < FB; ++q) {
        s1 = fma(A.a[f * FB + q], w1[q], s1);
        s2 = fma(A.a[f * FB + q], w2[q], s2);
      }
      S[(long long)f * b.vol + o] = s1;
      S[(long long)(F + f) * b.vol + o] = s2;
    }
  }
}

template <int MODE, int FB>
void launch_couple_fb(const TmaStageParams& p, const double* A_host, cudaStream_t st) {
  CoupleMatrix<FB> m;
  for (int r = 0; r < FB; ++r)
    for (int c = 0; c < FB; ++c) m.a[r * FB + c] = (r < p.F && c < p.F) ? A_host[r * p.F + c] : 0.0;
  dim3 blk(32, 4, 1), grd((p.b.n[0] + 31) / 32, (p.b.n[1] + 3) / 4, p.b.n[2]);
  couple_matvec<MODE, FB><<<grd, blk, 0, st>>>(p, m);
}

template <int MODE>
void launch_couple_mode(const TmaStageParams& p, const double* A_host, cudaStream_t st) {
  if (p.F <= 8) launch_couple_fb<MODE, 8>(p, A_host, st);
  else if (p.F <= 16) launch_couple_fb<MODE, 16>(p, A_host, st);
  else if (p.F <= 24) launch_couple_fb<MODE, 24>(p, A_host, st);
  else launch_couple_fb<MODE, 32>(p, A_host, st);
}

void launch_couple_matvec(const StageArgs& a, cudaStream_t st) {
  TmaStageParams p{};
  p.b = a.b;
  p.F = a.F;
  p.yn = a.yn; p.Y2r = a.Y2r; p.Y3r = a.Y3r;
  p.dt = a.dt;
  p.S = a.S;
  if (a.mode == STAGE_12) launch_couple_mode<STAGE_12>(p, a.A_host, st);
  else launch_couple_mode<STAGE_34>(p, a.A_host, st);
}
}  // namespace

int stage_pick_chunks(const BoxView& b, int F, int ctas_per_sm, int halo_planes, int tx, int ty) {
  return pick_chunks_impl(b, F, ctas_per_sm, halo_planes, tx, ty);
}

// which tile the stage kernels use on this box (0: 32 x 16, 1: 64 x 7): a function of the box and the device only, so
// that the tensor map built at creation and every later launch agree. SC_STAGE_TILE=0|1 forces it (A/B checks).
int stage_tile_variant(const BoxView& b, int F) {
  static const int forced = [] { const char* e = getenv("SC_STAGE_TILE"); return e ? atoi(e) : -1; }();
  if (forced >= 0) return forced ? 1 : 0;
  return tile_cost<TileB>(b, F) < 0.97 * tile_cost<TileA>(b, F) ? 1 : 0;
}

void stage_box_dims(int variant, unsigned box[4]) {
  box[0] = variant ? TileB::HX : TileA::HX;
  box[1] = variant ? TileB::HY : TileA::HY;
  box[2] = 1;
  box[3] = 1;
}

bool make_box_tensor_map_tma(const BoxView& b, int narrays, void* base, const unsigned bx[4], int l2_promotion,
                             bool swizzle64, void* out_map128) {
  EncodeTiledFn enc = encode_tiled();
  if (!enc) return false;
  if (b.px > (1 << 30) || (reinterpret_cast<uintptr_t>(base) & 15)) return false;
  const cuuint64_t dims[4] = {(cuuint64_t)b.px, (cuuint64_t)b.py, (cuuint64_t)b.pz, (cuuint64_t)narrays};
  const cuuint64_t strides[3] = {(cuuint64_t)b.px * 8, (cuuint64_t)b.plane * 8, (cuuint64_t)b.vol * 8};
  const cuuint32_t box[4] = {bx[0], bx[1], bx[2], bx[3]};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  CUtensorMap m;
  const CUresult r = enc(&m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE,
                         swizzle64 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_NONE,
                         l2_promotion == 256 ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B
                                             : (l2_promotion == 128 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B
                                                                    : CU_TENSOR_MAP_L2_PROMOTION_NONE),
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return false;
  static_assert(sizeof(CUtensorMap) == 128, "CUtensorMap is 128 bytes");
  memcpy(out_map128, &m, 128);
  return true;
}

int launch_stage_tma(const StageArgs& a, cudaStream_t st) {
  if (!a.tmap || (a.A && !(a.S && a.A_host))) { launch_stage_direct(a, st); return 1; }
  if (a.A) {  // coupling terms first (pointwise F x F product over all fields), then the per-field z-march
    launch_couple_matvec(a, st);
    if (a.mode == STAGE_12) launch_zmarch_v<STAGE_12, true>(a, st);
    else launch_zmarch_v<STAGE_34, true>(a, st);
  } else {
    if (a.mode == STAGE_12) launch_zmarch_v<STAGE_12, false>(a, st);
    else launch_zmarch_v<STAGE_34, false>(a, st);
  }
  return a.A ? 2 : 1;
}

}  // namespace sc
