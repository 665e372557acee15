// stage_gen_tma.cu — tuned stage kernel of the general path for the wide stencils ("eighth-order
// finite differences and fifth-order KO dissipation" for every spacetime run; eq 36 with r = 8: ninth-order), sm_100a.
// One launch = one RK stage of one box, the arithmetic of stage_gen.cu:
//   k_u = R + Q U,   k_rho = Lap_h U + Q R,   then the integrator's stage combine (kernels.h: StageKOArgs)
// with Lap_h of radius RL (2: 4th order, 4: 8th order) and Q of radius RQ (0: none, 3: delta^6, 5: delta^10).
//
// Same data movement as stage_ko_tma.cu — a CTA owns a 32 x 16 column and marches a z-chunk, every plane of the two
// halo-read arrays arrives as one TMA tiled load each into an mbarrier ring, the z-stencils live in registers in scatter
// form (an arriving plane adds its in-plane part to its own output plane and its centre value, times the z weights, to
// the 2H neighbouring output planes, H = max(RL, RQ); output plane p - H is complete when plane p has arrived). Tile
// 64 x 7 cells (4 x 37 = 148 columns of a 256^2 plane: one CTA on every SM), 224 threads, two x-adjacent cells per thread (every shared load is 16 bytes), one CTA per SM with the
// whole register file (2 (2H + 1) double2 accumulators per thread), a 6-deep ring. Measured on the way (256^3, fd 8 +
// delta^6 / delta^10): one cell per thread, 512 threads: 252 / 323 us, ncu: `mio_throttle` 2.7 stall cycles per issue
// (30 8-byte shared loads per thread and plane); this form: 254 / 277 us; the direct-load stage_gen: 368 / 421 us. A
// barrier-free ring hand-off (274 us) and a deeper ring (254 us) did not help.
#include <cuda.h>

#include <type_traits>
#include <utility>

#include "kernels.h"
#include "launch_cfg.h"

namespace sc {

int stage_pick_chunks(const BoxView& b, int F, int ctas_per_sm, int halo_planes, int tx, int ty);

namespace {

constexpr int GTX = 64, GTY = 7, GNTHR = (GTX / 2) * GTY;  // two x-adjacent cells per thread: every shared load is 16 bytes
constexpr int GNST = 6;  // planes in flight

template <int H> struct TileGeo {
  static constexpr int HXE = (H + 1) & ~1;                 // x halo on the left, rounded up to even: the TMA x coordinate stays even
  static constexpr int HX = GTX + 2 * HXE, HY = GTY + 2 * H;
  static constexpr int DOUBLES = HX * HY;
  static constexpr int STRIDE = (DOUBLES * 8 + 127) / 128 * 128;  // bytes between tiles (TMA destinations are 128-byte aligned)
};

__device__ __forceinline__ uint32_t smem_u32s(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_wait_s(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
  } while (!ok);
}

struct GenTmaParams {
  BoxView b;
  int F, nchunks, chunk;
  int a_Yu, a_Yr;
  const double* yn_u;
  const double* yn_r;
  const double* A2u; const double* A2r;   // combine operands (centre only), see stage_ko_tma.cu: KoParams
  const double* A3u; const double* A3r;
  const double* A4u; const double* A4r;
  double c2, c3, c4;
  double* outU; double* outR;
  double* Ku; double* Kr;
  double adt;
  double w[3];   // 1 / (12 dx_a^2)
  double ko[3];  // sigma / (64 dx_a) or sigma / (1024 dx_a); 0 without dissipation
};

// centred-stencil weights at distance m: 12 h^2 x the second difference; the dissipation's delta^(2 RQ)
template <int RL> __device__ __forceinline__ constexpr double lapw(int m) {
  if (RL == 2) return m == 0 ? -30.0 : (m == 1 ? 16.0 : -1.0);
  return m == 0 ? 12.0 * (-205.0 / 72.0) : (m == 1 ? 12.0 * 8.0 / 5.0 : (m == 2 ? -12.0 / 5.0 : (m == 3 ? 12.0 * 8.0 / 315.0 : -12.0 / 560.0)));
}
template <int RQ> __device__ __forceinline__ constexpr double disw(int m) {
  if (RQ == 3) return m == 0 ? -20.0 : (m == 1 ? 15.0 : (m == 2 ? -6.0 : 1.0));
  return m == 0 ? -252.0 : (m == 1 ? 210.0 : (m == 2 ? -120.0 : (m == 3 ? 45.0 : (m == 4 ? -10.0 : 1.0))));
}

template <class Fn, int... Rs>
__device__ __forceinline__ void unrolled_steps(Fn& fn, int it0, int narr, std::integer_sequence<int, Rs...>) {
  ((it0 + Rs < narr ? (fn(std::integral_constant<int, Rs>{}, it0 + Rs), 0) : 0), ...);
}

}  // namespace

template <int RL, int RQ, bool COMBINE>
__global__ void __launch_bounds__(GNTHR, 1)
    stage_gen_zmarch(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ GenTmaParams p) {
  constexpr int H = RL > RQ ? RL : RQ, NS = 2 * H + 1;
  using G = TileGeo<H>;
  extern __shared__ unsigned char smraw[];
  const uint32_t s0 = (smem_u32s(smraw) + 127u) & ~127u;
  unsigned char* const tiles = smraw + (s0 - smem_u32s(smraw));
  const uint32_t bar0 = s0 + GNST * 2 * G::STRIDE;

  const BoxView& b = p.b;
  const int tid = threadIdx.x, tx = tid % (GTX / 2), ty = tid / (GTX / 2);
  const int X0 = blockIdx.x * GTX, Y0 = blockIdx.y * GTY;
  const int f = blockIdx.z / p.nchunks, c = blockIdx.z % p.nchunks;
  const int zc0 = c * p.chunk, zc1 = min(b.n[2], zc0 + p.chunk);
  const int narr = zc1 - zc0 + 2 * H;
  const int dir = (c & 1) ? 1 : -1;
  const int zs = dir > 0 ? zc0 - H : zc1 + H - 1;

  auto issue = [&](int it) {
    const int st = it % GNST;
    const uint32_t bar = bar0 + 8 * st;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(2 * G::DOUBLES * 8) : "memory");
#pragma unroll
    for (int h = 0; h < 2; ++h)
      asm volatile(
          "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, "
          "%4, %5}], [%6];" ::"r"(s0 + (st * 2 + h) * G::STRIDE),
          "l"(&tmap), "r"(XOFF + X0 - G::HXE), "r"(b.g + Y0 - H), "r"(b.g + zs + dir * it),
          "r"((h ? p.a_Yr : p.a_Yu) + f), "r"(bar)
          : "memory");
  };
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < GNST; ++s)
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar0 + 8 * s), "r"(1));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    for (int it = 0; it < GNST && it < narr; ++it) issue(it);
  }
  __syncthreads();

  const bool active = (X0 + 2 * tx < b.n[0]) && (Y0 + ty < b.n[1]);
  const long long cell0 = (long long)f * b.vol + cell_offset(b, X0 + 2 * tx, Y0 + ty, 0);
  const double wx = p.w[0], wy = p.w[1], wz = p.w[2], kx = p.ko[0], ky = p.ko[1], kz = p.ko[2];
  double2 accU[NS], accR[NS];
#pragma unroll
  for (int q = 0; q < NS; ++q) accU[q] = accR[q] = make_double2(0.0, 0.0);
  const double2 zero2 = make_double2(0.0, 0.0);
  double2 n_un = zero2, n_rn = zero2, n_u2 = zero2, n_r2 = zero2, n_u3 = zero2, n_r3 = zero2, n_u4 = zero2, n_r4 = zero2;
  auto ld2 = [](const double* q) { return __ldg(reinterpret_cast<const double2*>(q)); };

  auto step = [&](auto Rc, int it) {
    constexpr int R = decltype(Rc)::value;
    const int st = it % GNST;
    const bool inpl = it >= H && it < narr - H;
    const int z = zs + dir * it;
    const double2 un = n_un, rn = n_rn, u2 = n_u2, r2 = n_r2, u3 = n_u3, r3 = n_r3, u4 = n_u4, r4 = n_r4;
    if (active && it + 1 >= 2 * H && it + 1 < narr) {  // the next iteration completes plane z + dir - H dir
      const long long o = cell0 + (long long)(z - (H - 1) * dir) * b.plane;
      n_un = ld2(p.yn_u + o);
      n_rn = ld2(p.yn_r + o);
      if (COMBINE) {
        if (p.c2 != 0.0) { n_u2 = ld2(p.A2u + o); n_r2 = ld2(p.A2r + o); }
        if (p.c3 != 0.0) { n_u3 = ld2(p.A3u + o); n_r3 = ld2(p.A3r + o); }
        if (p.c4 != 0.0) { n_u4 = ld2(p.A4u + o); n_r4 = ld2(p.A4r + o); }
      }
    }
    mbar_wait_s(bar0 + 8 * st, (it / GNST) & 1);
    // the thread's two cells (x, x + 1) sit at double2 index 0 of cU / cR; row neighbours at double2 offsets, rows HX apart
    const double* __restrict__ tU = reinterpret_cast<const double*>(tiles + (st * 2) * G::STRIDE) + (ty + H) * G::HX + 2 * tx + G::HXE;
    const double* __restrict__ tR = reinterpret_cast<const double*>(tiles + (st * 2 + 1) * G::STRIDE) + (ty + H) * G::HX + 2 * tx + G::HXE;
    auto at2 = [](const double* q, int off) { return *reinterpret_cast<const double2*>(q + off); };
    const double2 uc = at2(tU, 0), rc = at2(tR, 0);
    double2 ctU = zero2, ctR = zero2;
    if (inpl) {
      // row values x-4 .. x+5 (x-6 .. x+7 for H = 5) as double2: flat index q <-> x - HR + q, HR = even radius
      constexpr int HR = (H + 1) & ~1, NV = HR + 1;
      double2 vu[NV], vr[NV];
#pragma unroll
      for (int q = 0; q < NV; ++q) { vu[q] = at2(tU, 2 * q - HR); if (RQ > 0) vr[q] = at2(tR, 2 * q - HR); }
      auto flat = [&](const double2 (&v)[NV], int q) { return (q & 1) ? v[q >> 1].y : v[q >> 1].x; };
      double2 lx = zero2, ly = zero2, qux = zero2, quy = zero2, qrx = zero2, qry = zero2;
#pragma unroll
      for (int m = 1; m <= H; ++m) {
        // cell 0 sits at flat HR, cell 1 at flat HR + 1
        const double2 ux = make_double2(flat(vu, HR - m) + flat(vu, HR + m), flat(vu, HR + 1 - m) + flat(vu, HR + 1 + m));
        const double2 um = at2(tU, -m * G::HX), up = at2(tU, m * G::HX);
        const double2 uy = make_double2(um.x + up.x, um.y + up.y);
        if (m <= RL) {
          lx.x = fma(lapw<RL>(m), ux.x, lx.x); lx.y = fma(lapw<RL>(m), ux.y, lx.y);
          ly.x = fma(lapw<RL>(m), uy.x, ly.x); ly.y = fma(lapw<RL>(m), uy.y, ly.y);
        }
        if (RQ > 0 && m <= RQ) {
          const double2 rx = make_double2(flat(vr, HR - m) + flat(vr, HR + m), flat(vr, HR + 1 - m) + flat(vr, HR + 1 + m));
          const double2 rm = at2(tR, -m * G::HX), rp = at2(tR, m * G::HX);
          const double2 ry = make_double2(rm.x + rp.x, rm.y + rp.y);
          qux.x = fma(disw<RQ>(m), ux.x, qux.x); qux.y = fma(disw<RQ>(m), ux.y, qux.y);
          quy.x = fma(disw<RQ>(m), uy.x, quy.x); quy.y = fma(disw<RQ>(m), uy.y, quy.y);
          qrx.x = fma(disw<RQ>(m), rx.x, qrx.x); qrx.y = fma(disw<RQ>(m), rx.y, qrx.y);
          qry.x = fma(disw<RQ>(m), ry.x, qry.x); qry.y = fma(disw<RQ>(m), ry.y, qry.y);
        }
      }
      const double lapc = lapw<RL>(0) * (wx + wy + wz);
      const double2 lU = make_double2(fma(wx, lx.x, fma(wy, ly.x, lapc * uc.x)), fma(wx, lx.y, fma(wy, ly.y, lapc * uc.y)));
      double2 qU = zero2, qR = zero2;
      if (RQ > 0) {
        const double qc = disw<RQ>(0) * (kx + ky + kz);
        qU = make_double2(fma(kx, qux.x, fma(ky, quy.x, qc * uc.x)), fma(kx, qux.y, fma(ky, quy.y, qc * uc.y)));
        qR = make_double2(fma(kx, qrx.x, fma(ky, qry.x, qc * rc.x)), fma(kx, qrx.y, fma(ky, qry.y, qc * rc.y)));
      }
      ctU = make_double2(rc.x + qU.x, rc.y + qU.y);
      ctR = make_double2(lU.x + qR.x, lU.y + qR.y);
    }
    // scatter: slot (R + d) mod NS belongs to output plane (arrival + d); the slot of arrival + H is created here
#pragma unroll
    for (int d = -H; d <= H; ++d) {
      const int m = d < 0 ? -d : d;
      const int slot = ((R + d) % NS + NS) % NS;
      double2 zu = zero2, zr = zero2;
      if (d == 0) { zu = ctU; zr = ctR; }
      else {
        if (RQ > 0 && m <= RQ) {
          const double cq = kz * disw<RQ>(m);
          zu = make_double2(cq * uc.x, cq * uc.y);
          zr = make_double2(cq * rc.x, cq * rc.y);
        }
        if (m <= RL) { const double cl = wz * lapw<RL>(m); zr.x = fma(cl, uc.x, zr.x); zr.y = fma(cl, uc.y, zr.y); }
      }
      if (d == H) { accU[slot] = zu; accR[slot] = zr; }
      else { accU[slot].x += zu.x; accU[slot].y += zu.y; accR[slot].x += zr.x; accR[slot].y += zr.y; }
    }
    if (it >= 2 * H && active) {  // output plane z - H dir is complete
      const long long o = cell0 + (long long)(z - H * dir) * b.plane;
      constexpr int done = ((R - H) % NS + NS) % NS;
      const double2 ku = accU[done], kr = accR[done];
      auto st2 = [](double* q, double2 v) { *reinterpret_cast<double2*>(q) = v; };
      if (!COMBINE) {
        st2(p.outU + o, make_double2(fma(p.adt, ku.x, un.x), fma(p.adt, ku.y, un.y)));
        st2(p.outR + o, make_double2(fma(p.adt, kr.x, rn.x), fma(p.adt, kr.y, rn.y)));
      } else {
        if (p.outU) {
          st2(p.outU + o, make_double2(un.x + ((p.c2 * (u2.x - un.x) + p.c4 * (u4.x - un.x)) + p.c3 * (u3.x - un.x)) + p.adt * ku.x,
                                       un.y + ((p.c2 * (u2.y - un.y) + p.c4 * (u4.y - un.y)) + p.c3 * (u3.y - un.y)) + p.adt * ku.y));
          st2(p.outR + o, make_double2(rn.x + ((p.c2 * (r2.x - rn.x) + p.c4 * (r4.x - rn.x)) + p.c3 * (r3.x - rn.x)) + p.adt * kr.x,
                                       rn.y + ((p.c2 * (r2.y - rn.y) + p.c4 * (r4.y - rn.y)) + p.c3 * (r3.y - rn.y)) + p.adt * kr.y));
        }
        if (p.Ku) { st2(p.Ku + o, ku); st2(p.Kr + o, kr); }
      }
    }
    __syncthreads();
    if (tid == 0 && it + GNST < narr) issue(it + GNST);
  };

  for (int it0 = 0; it0 < narr; it0 += NS) unrolled_steps(step, it0, narr, std::make_integer_sequence<int, NS>{});
}

// ---- host ------------------------------------------------------------------------------------------
void stagegen_box_dims(int H, unsigned box[4]) {
  box[0] = H == 5 ? TileGeo<5>::HX : TileGeo<4>::HX;
  box[1] = H == 5 ? TileGeo<5>::HY : TileGeo<4>::HY;
  box[2] = 1;
  box[3] = 1;
}

namespace {
template <int RL, int RQ, bool COMBINE>
void launch_gen(const StageKOArgs& a, GenTmaParams p, cudaStream_t st) {
  constexpr int H = RL > RQ ? RL : RQ;
  constexpr size_t smem = (size_t)GNST * 2 * TileGeo<H>::STRIDE + GNST * 8 + 128;
  ensure_dynamic_smem(stage_gen_zmarch<RL, RQ, COMBINE>, smem);
  p.nchunks = stage_pick_chunks(a.b, a.F, 1, 2 * H, GTX, GTY);
  p.chunk = (a.b.n[2] + p.nchunks - 1) / p.nchunks;
  p.nchunks = (a.b.n[2] + p.chunk - 1) / p.chunk;
  dim3 grd((a.b.n[0] + GTX - 1) / GTX, (a.b.n[1] + GTY - 1) / GTY, p.nchunks * a.F);
  stage_gen_zmarch<RL, RQ, COMBINE><<<grd, GNTHR, smem, st>>>(*static_cast<const CUtensorMap*>(a.tmap), p);
}
template <int RL, int RQ>
void launch_gen_c(const StageKOArgs& a, const GenTmaParams& p, bool combine, cudaStream_t st) {
  if (combine) launch_gen<RL, RQ, true>(a, p, st);
  else launch_gen<RL, RQ, false>(a, p, st);
}
}  // namespace

// 8th-order differences with no, fifth- or ninth-order dissipation (tile halo 4 or 5: the tensor map of the box says which)
bool stage_gen_tma_takes(const StageKOArgs& a) {
  const int H = a.ko_order == 9 ? 5 : 4;
  return a.tmap && !a.A && a.fd_order == 8 && a.b.g >= H;
}

void launch_stage_gen_tma(const StageKOArgs& a, cudaStream_t st) {
  GenTmaParams p{};
  p.b = a.b;
  p.F = a.F;
  p.a_Yu = a.a_Yu; p.a_Yr = a.a_Yr;
  p.yn_u = a.yn_u; p.yn_r = a.yn_r;
  p.A2u = a.U2; p.A2r = a.R2; p.A3u = a.U3; p.A3r = a.R3; p.A4u = a.Yu; p.A4r = a.Yr;
  p.outU = a.outU; p.outR = a.outR;
  p.Ku = a.K4u; p.Kr = a.K4r;
  for (int d = 0; d < 3; ++d) { p.w[d] = a.inv12dx2[d]; p.ko[d] = a.ko_order ? a.ko[d] : 0.0; }
  const int S = a.integrator, s = a.stage;
  bool combine = false;
  if (s > S) { combine = true; p.outU = p.outR = nullptr; }
  else if (S == 4 && s == 4) { combine = true; p.c2 = 1.0 / 3.0; p.c3 = 2.0 / 3.0; p.c4 = 1.0 / 3.0; p.adt = a.dt / 6.0; }
  else if (S == 3 && s == 2) { combine = true; p.c4 = -2.0; p.adt = 2.0 * a.dt; }
  else if (S == 3 && s == 3) { combine = true; p.c2 = 1.0; p.c4 = 1.0 / 3.0; p.adt = a.dt / 6.0; p.Ku = a.K3u; p.Kr = a.K3r; }
  else if (S == 2 && s == 2) { combine = true; p.adt = a.dt; }
  else p.adt = (S == 4 && s == 3 ? 1.0 : 0.5) * a.dt;
  if (a.ko_order == 9) launch_gen_c<4, 5>(a, p, combine, st);
  else if (a.ko_order == 5) launch_gen_c<4, 3>(a, p, combine, st);
  else launch_gen_c<4, 0>(a, p, combine, st);
}

}  // namespace sc
