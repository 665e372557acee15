// stage_ko_tma.cu — tuned stage kernel of the dissipative (Kreiss-Oliger) path, sm_100a: the z-march of
// stage_tma.cu with radius-3 halos. One launch = one RK4 stage of one box (stage_ko.cu states the arithmetic):
//   k_u = R + Q U,   k_rho = Lap_h U + Q R,   Q y = sigma/64 sum_i delta_i^6 y / h_i         (eqs 35-36)
//   stages 1..3:  Y_{s+1} = y_n + a_s dt k        stage 4:  y_{n+1} = y_n + [(Y_2-y_n) + 2 (Y_3-y_n) + (Y_4-y_n)]/3 + dt/6 k_4
// A CTA owns a 32 x 16 column and marches a z-chunk; every plane of the two halo-read arrays (U_s, R_s) arrives
// as a (32+8) x (16+6) tile through one TMA tiled load each (the tile starts 4 cells left of the column so that
// its fp64 x coordinate stays even — odd coordinates fault, see ghost_tma.cu) into a 4-deep mbarrier ring.
// Both 7-point (Q) and 5-point (Lap) z-stencils live in registers in scatter form: an arriving plane adds its
// in-plane part to the accumulators of its own output plane and its centre value, times the z weights, to the
// accumulators of the 6 neighbouring output planes; output plane p-3 is complete when plane p has arrived.
// Centre-only operands (y_n; Y_2, Y_3, Y_4 in stage 4) are plain global loads issued one plane ahead.
#include <cuda.h>

#include <type_traits>

#include "kernels.h"
#include "launch_cfg.h"

namespace sc {

int stage_pick_chunks(const BoxView& b, int F, int ctas_per_sm, int halo_planes, int tx, int ty);

namespace {

// Tile of cells per CTA column: 32 x 16 or 64 x 7, the same choice per box as stage_tma.cu (stage_tile_variant: on
// 256^3 the second makes 148 columns, i.e. whole CTAs-per-SM multiples on 148 SMs with all columns in lock step)
template <int TX_, int TY_> struct TileK {
  static constexpr int TX = TX_, TY = TY_;
  static constexpr int HXK = TX + 8, HYK = TY + 6;      // tile: x from X0-4 (even start), y from Y0-3
  static constexpr int NTHR = (TX / 2) * TY;            // two x-adjacent cells per thread
  static constexpr int TILE_BYTES = HXK * HYK * 8;      // what one TMA tiled load writes
  static constexpr int TILEK = (TILE_BYTES + 127) / 128 * 16;  // doubles between tiles in shared memory (128-byte aligned)
};
using TileKA = TileK<32, 16>;
using TileKB = TileK<64, 7>;
constexpr int NSTK = 4;                        // planes in flight

__device__ __forceinline__ uint32_t smem_u32k(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_wait_k(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
  } while (!ok);
}

struct KoParams {
  BoxView b;
  int F, nchunks, chunk;
  int a_Yu, a_Yr;        // array indices (field 0) of the stage vector's u- and rho-part in the tensor map
  const double* yn_u;    // centre-only operands and outputs: field-0 arrays
  const double* yn_r;
  // combine stage (FINAL): out = y_n + c2 (A2 - y_n) + c3 (A3 - y_n) + c4 (A4 - y_n) + adt k, centre-only operands A2..A4
  // (null with a zero coefficient); RK4 stage 4: (Y_2, Y_3, Y_4; 1/3, 2/3, 1/3; dt/6); RK3 stage 2: (-, -, Y_2; -2; 2 dt);
  // RK3 stage 3: (Y_2, -, Y_3; 1, 1/3; dt/6); RK2 stage 2: (dt); RK3's extra slope: no out, k only
  const double* U2; const double* U3; const double* R2; const double* R3;
  const double* Y4u; const double* Y4r;   // the centre of the stage's own input again (global, L2-resident)
  double c2, c3, c4;
  double* outU; double* outR;             // null: the slope only
  double* K4u; double* K4r;               // where the slope k is kept, or null
  double adt;            // a_s dt (simple stages) or the weight of k in the combine
  double w[3];           // 1 / (12 dx_a^2)
  double ko[3];          // sigma / (64 dx_a)
};

// values of one array around the thread's two cells (x, x+1) in the current plane
struct Nbr3 {
  double2 xa, xb, xc, xd, xe;                   // row y: columns x-4 .. x+5
  double2 ym3, ym2, ym1, yp1, yp2, yp3;         // columns x, x+1 of rows y-3 .. y+3
};
template <int HXK>
__device__ __forceinline__ Nbr3 load_nbr3(const double* tile, int tx, int ty) {
  Nbr3 n;
  const double2* r = reinterpret_cast<const double2*>(tile + (ty + 3) * HXK + 2 * tx);
  n.xa = r[0]; n.xb = r[1]; n.xc = r[2]; n.xd = r[3]; n.xe = r[4];
  const double* c = tile + 2 * tx + 4;
  n.ym3 = *reinterpret_cast<const double2*>(c + (ty + 0) * HXK);
  n.ym2 = *reinterpret_cast<const double2*>(c + (ty + 1) * HXK);
  n.ym1 = *reinterpret_cast<const double2*>(c + (ty + 2) * HXK);
  n.yp1 = *reinterpret_cast<const double2*>(c + (ty + 4) * HXK);
  n.yp2 = *reinterpret_cast<const double2*>(c + (ty + 5) * HXK);
  n.yp3 = *reinterpret_cast<const double2*>(c + (ty + 6) * HXK);
  return n;
}
template <int HXK>
__device__ __forceinline__ double2 load_centre3(const double* tile, int tx, int ty) {
  return *reinterpret_cast<const double2*>(tile + (ty + 3) * HXK + 2 * tx + 4);
}
// delta^6 along x and y at the two cells
__device__ __forceinline__ double2 d6x(const Nbr3& n) {
  return make_double2((n.xa.y + n.xd.y) - 6.0 * (n.xb.x + n.xd.x) + 15.0 * (n.xb.y + n.xc.y) - 20.0 * n.xc.x,
                      (n.xb.x + n.xe.x) - 6.0 * (n.xb.y + n.xd.y) + 15.0 * (n.xc.x + n.xd.x) - 20.0 * n.xc.y);
}
__device__ __forceinline__ double2 d6y(const Nbr3& n) {
  return make_double2((n.ym3.x + n.yp3.x) - 6.0 * (n.ym2.x + n.yp2.x) + 15.0 * (n.ym1.x + n.yp1.x) - 20.0 * n.xc.x,
                      (n.ym3.y + n.yp3.y) - 6.0 * (n.ym2.y + n.yp2.y) + 15.0 * (n.ym1.y + n.yp1.y) - 20.0 * n.xc.y);
}
// 12 h^2 x the 4th-order second derivative along x and y (S2)
__device__ __forceinline__ double2 d2x(const Nbr3& n) {
  return make_double2(16.0 * (n.xb.y + n.xc.y) - (n.xb.x + n.xd.x) - 30.0 * n.xc.x,
                      16.0 * (n.xc.x + n.xd.x) - (n.xb.y + n.xd.y) - 30.0 * n.xc.y);
}
__device__ __forceinline__ double2 d2y(const Nbr3& n) {
  return make_double2(16.0 * (n.ym1.x + n.yp1.x) - (n.ym2.x + n.yp2.x) - 30.0 * n.xc.x,
                      16.0 * (n.ym1.y + n.yp1.y) - (n.ym2.y + n.yp2.y) - 30.0 * n.xc.y);
}
__device__ __forceinline__ double2 add2(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 fma2k(double c, double2 a, double2 b) {
  return make_double2(fma(c, a.x, b.x), fma(c, a.y, b.y));
}
__device__ __forceinline__ double2 mul2(double c, double2 a) { return make_double2(c * a.x, c * a.y); }

// Scatter one arrived plane into the seven pending accumulators. R = arrival index mod 7 (compile time): slot
// (R + d) mod 7 belongs to output plane (arrival + d). z1, z2, z3 = the plane's contribution to the outputs at
// distance 1, 2, 3; ct to its own. The slot of arrival + 3 is created here.
template <int R>
__device__ __forceinline__ void scatter7(double2 (&acc)[7], double2 ct, double2 z1, double2 z2, double2 z3) {
  acc[(R + 4) % 7] = add2(acc[(R + 4) % 7], z3);
  acc[(R + 5) % 7] = add2(acc[(R + 5) % 7], z2);
  acc[(R + 6) % 7] = add2(acc[(R + 6) % 7], z1);
  acc[R] = add2(acc[R], ct);
  acc[(R + 1) % 7] = add2(acc[(R + 1) % 7], z1);
  acc[(R + 2) % 7] = add2(acc[(R + 2) % 7], z2);
  acc[(R + 3) % 7] = z3;
}

}  // namespace

// (stage 4 keeps 8 more centre operands in flight per cell pair: one CTA per SM with the full register file;
// the 4-deep TMA ring and the one-plane-ahead global loads still cover the memory latency)
// FINAL: 0 = simple stage (out = y_n + adt k), 1 = full combine (up to three more centre operands; one CTA per SM),
// 2 = light combine (the stage's own input as the only extra operand: RK3 stage 2, RK2 stage 2, RK3's extra slope)
template <int FINAL, class T>
__global__ void __launch_bounds__(T::NTHR, FINAL == 1 ? 1 : 2)
    stage_ko_zmarch(const __grid_constant__ CUtensorMap tmap, const __grid_constant__ KoParams p) {
  constexpr int TX = T::TX, TY = T::TY, HXK = T::HXK, TILEK = T::TILEK;
  extern __shared__ unsigned char smraw[];
  // [NSTK][2] tiles (U, R), 128-byte aligned for TMA, then NSTK mbarriers
  const uint32_t s0 = (smem_u32k(smraw) + 127u) & ~127u;
  double* const tiles = reinterpret_cast<double*>(smraw + (s0 - smem_u32k(smraw)));
  const uint32_t bar0 = s0 + NSTK * 2 * TILEK * 8;

  const BoxView& b = p.b;
  const int tid = threadIdx.x, tx = tid % (TX / 2), ty = tid / (TX / 2);
  const int X0 = blockIdx.x * TX, Y0 = blockIdx.y * TY;
  const int f = blockIdx.z / p.nchunks, c = blockIdx.z % p.nchunks;
  const int zc0 = c * p.chunk, zc1 = min(b.n[2], zc0 + p.chunk);
  const int narr = zc1 - zc0 + 6;              // planes that arrive: the chunk plus 3 halo planes each side
  const int dir = (c & 1) ? 1 : -1;            // neighbouring chunks march in opposite directions
  const int zs = dir > 0 ? zc0 - 3 : zc1 + 2;  // first plane to arrive

  auto issue = [&](int it) {  // one thread: arm the stage's mbarrier and request the plane's two tiles
    const int st = it % NSTK;
    const uint32_t bar = bar0 + 8 * st;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(2 * T::TILE_BYTES) : "memory");
#pragma unroll
    for (int h = 0; h < 2; ++h)
      asm volatile(
          "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, "
          "%4, %5}], [%6];" ::"r"(s0 + (st * 2 + h) * TILEK * 8),
          "l"(&tmap), "r"(XOFF + X0 - 4), "r"(b.g + Y0 - 3), "r"(b.g + zs + dir * it),
          "r"((h ? p.a_Yr : p.a_Yu) + f), "r"(bar)
          : "memory");
  };
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NSTK; ++s)
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar0 + 8 * s), "r"(1));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    for (int it = 0; it < NSTK && it < narr; ++it) issue(it);
  }
  __syncthreads();

  const bool active = (X0 + 2 * tx < b.n[0]) && (Y0 + ty < b.n[1]);
  const long long cell0 = (long long)f * b.vol + cell_offset(b, X0 + 2 * tx, Y0 + ty, 0);
  const double wx = p.w[0], wy = p.w[1], wz = p.w[2], kx = p.ko[0], ky = p.ko[1], kz = p.ko[2];
  double2 accU[7], accR[7];
#pragma unroll
  for (int q = 0; q < 7; ++q) accU[q] = accR[q] = make_double2(0.0, 0.0);
  // centre-only operands of the NEXT completed output plane
  const double2 zero2 = make_double2(0.0, 0.0);
  double2 n_un = zero2, n_rn = zero2, n_u2 = zero2, n_u3 = zero2, n_r2 = zero2, n_r3 = zero2, n_u4 = zero2, n_r4 = zero2;

  auto step = [&](auto Rc, int it) {
    constexpr int R = decltype(Rc)::value;
    const int st = it % NSTK;
    const bool inpl = it >= 3 && it < narr - 3;
    const int z = zs + dir * it;
    // operands of the output plane this iteration completes (requested one iteration ago)
    const double2 un = n_un, rn = n_rn, u2 = n_u2, u3 = n_u3, r2 = n_r2, r3 = n_r3, u4 = n_u4, r4 = n_r4;
    if (active && it + 1 >= 6 && it + 1 < narr) {  // next iteration completes plane z - 2 dir
      const long long o = cell0 + (long long)(z - 2 * dir) * b.plane;
      n_un = __ldg(reinterpret_cast<const double2*>(p.yn_u + o));
      n_rn = __ldg(reinterpret_cast<const double2*>(p.yn_r + o));
      if (FINAL == 2 && p.c4 != 0.0) {
        n_u4 = __ldg(reinterpret_cast<const double2*>(p.Y4u + o));
        n_r4 = __ldg(reinterpret_cast<const double2*>(p.Y4r + o));
      }
      if (FINAL == 1) {
        if (p.c2 != 0.0) {
          n_u2 = __ldg(reinterpret_cast<const double2*>(p.U2 + o));
          n_r2 = __ldg(reinterpret_cast<const double2*>(p.R2 + o));
        }
        if (p.c3 != 0.0) {
          n_u3 = __ldg(reinterpret_cast<const double2*>(p.U3 + o));
          n_r3 = __ldg(reinterpret_cast<const double2*>(p.R3 + o));
        }
        if (p.c4 != 0.0) {
          n_u4 = __ldg(reinterpret_cast<const double2*>(p.Y4u + o));
          n_r4 = __ldg(reinterpret_cast<const double2*>(p.Y4r + o));
        }
      }
    }
    mbar_wait_k(bar0 + 8 * st, (it / NSTK) & 1);
    const double* __restrict__ tU = tiles + (st * 2) * TILEK;
    const double* __restrict__ tR = tU + TILEK;
    double2 ctU = zero2, ctR = zero2, uc, rc;
    if (inpl) {
      const Nbr3 U = load_nbr3<HXK>(tU, tx, ty);
      const Nbr3 Rr = load_nbr3<HXK>(tR, tx, ty);
      uc = U.xc; rc = Rr.xc;
      const double2 qU = fma2k(kx, d6x(U), fma2k(ky, d6y(U), mul2(-20.0 * kz, uc)));
      const double2 qR = fma2k(kx, d6x(Rr), fma2k(ky, d6y(Rr), mul2(-20.0 * kz, rc)));
      const double2 lU = fma2k(wx, d2x(U), fma2k(wy, d2y(U), mul2(-30.0 * wz, uc)));
      ctU = add2(rc, qU);
      ctR = add2(lU, qR);
    } else {
      uc = load_centre3<HXK>(tU, tx, ty);
      rc = load_centre3<HXK>(tR, tx, ty);
    }
    // z contributions of this plane: Q on U -> k_u;  Lap on U and Q on R -> k_rho
    scatter7<R>(accU, ctU, mul2(15.0 * kz, uc), mul2(-6.0 * kz, uc), mul2(kz, uc));
    scatter7<R>(accR, ctR, fma2k(16.0 * wz, uc, mul2(15.0 * kz, rc)), fma2k(-wz, uc, mul2(-6.0 * kz, rc)), mul2(kz, rc));
    if (it >= 6 && active) {  // output plane z - 3 dir is complete
      const long long o = cell0 + (long long)(z - 3 * dir) * b.plane;
      const double2 ku = accU[(R + 4) % 7], kr = accR[(R + 4) % 7];
      if (!FINAL) {
        *reinterpret_cast<double2*>(p.outU + o) = fma2k(p.adt, ku, un);
        *reinterpret_cast<double2*>(p.outR + o) = fma2k(p.adt, kr, rn);
      } else if (FINAL == 2) {
        if (p.outU) {
          const double c4 = p.c4;
          *reinterpret_cast<double2*>(p.outU + o) = make_double2(un.x + c4 * (u4.x - un.x) + p.adt * ku.x,
                                                                 un.y + c4 * (u4.y - un.y) + p.adt * ku.y);
          *reinterpret_cast<double2*>(p.outR + o) = make_double2(rn.x + c4 * (r4.x - rn.x) + p.adt * kr.x,
                                                                 rn.y + c4 * (r4.y - rn.y) + p.adt * kr.y);
        }
        if (p.K4u) {
          *reinterpret_cast<double2*>(p.K4u + o) = ku;
          *reinterpret_cast<double2*>(p.K4r + o) = kr;
        }
      } else {
        if (p.outU) {
          const double c2 = p.c2, c3 = p.c3, c4 = p.c4;
          *reinterpret_cast<double2*>(p.outU + o) = make_double2(
              un.x + ((c2 * (u2.x - un.x) + c4 * (u4.x - un.x)) + c3 * (u3.x - un.x)) + p.adt * ku.x,
              un.y + ((c2 * (u2.y - un.y) + c4 * (u4.y - un.y)) + c3 * (u3.y - un.y)) + p.adt * ku.y);
          *reinterpret_cast<double2*>(p.outR + o) = make_double2(
              rn.x + ((c2 * (r2.x - rn.x) + c4 * (r4.x - rn.x)) + c3 * (r3.x - rn.x)) + p.adt * kr.x,
              rn.y + ((c2 * (r2.y - rn.y) + c4 * (r4.y - rn.y)) + c3 * (r3.y - rn.y)) + p.adt * kr.y);
        }
        if (p.K4u) {
          *reinterpret_cast<double2*>(p.K4u + o) = ku;
          *reinterpret_cast<double2*>(p.K4r + o) = kr;
        }
      }
    }
    __syncthreads();  // every thread is done with stage st: refill it with the plane NSTK arrivals ahead
    if (tid == 0 && it + NSTK < narr) issue(it + NSTK);
  };

  for (int it0 = 0; it0 < narr; it0 += 7) {
    step(std::integral_constant<int, 0>{}, it0);
    if (it0 + 1 < narr) step(std::integral_constant<int, 1>{}, it0 + 1);
    if (it0 + 2 < narr) step(std::integral_constant<int, 2>{}, it0 + 2);
    if (it0 + 3 < narr) step(std::integral_constant<int, 3>{}, it0 + 3);
    if (it0 + 4 < narr) step(std::integral_constant<int, 4>{}, it0 + 4);
    if (it0 + 5 < narr) step(std::integral_constant<int, 5>{}, it0 + 5);
    if (it0 + 6 < narr) step(std::integral_constant<int, 6>{}, it0 + 6);
  }
}

// ---- host ------------------------------------------------------------------------------------------
void stageko_box_dims(int variant, unsigned box[4]) {
  box[0] = variant ? TileKB::HXK : TileKA::HXK;
  box[1] = variant ? TileKB::HYK : TileKA::HYK;
  box[2] = 1;
  box[3] = 1;
}

template <int FINAL, class T>
static void launch_ko_zmarch_t(const StageKOArgs& a, const KoParams& p0, cudaStream_t st) {
  constexpr size_t smem = (size_t)NSTK * 2 * T::TILEK * 8 + NSTK * 8 + 128;
  ensure_dynamic_smem(stage_ko_zmarch<FINAL, T>, smem);
  KoParams p = p0;
  p.nchunks = stage_pick_chunks(a.b, a.F, FINAL == 1 ? 1 : 2, 6, T::TX, T::TY);
  p.chunk = (a.b.n[2] + p.nchunks - 1) / p.nchunks;
  p.nchunks = (a.b.n[2] + p.chunk - 1) / p.chunk;
  dim3 grd((a.b.n[0] + T::TX - 1) / T::TX, (a.b.n[1] + T::TY - 1) / T::TY, p.nchunks * a.F);
  stage_ko_zmarch<FINAL, T><<<grd, T::NTHR, smem, st>>>(*static_cast<const CUtensorMap*>(a.tmap), p);
}
template <int FINAL>
static void launch_ko_zmarch(const StageKOArgs& a, const KoParams& p0, cudaStream_t st) {
  if (a.tile_variant) launch_ko_zmarch_t<FINAL, TileKB>(a, p0, st);  // the tile the box's tensor map was built for
  else launch_ko_zmarch_t<FINAL, TileKA>(a, p0, st);
}

// the tuned kernel takes uncoupled systems whose box has a tensor map, 4th-order differences, no or fifth-order
// dissipation, any integrator; on a radiative level 0 the boundary points are redone by the direct kernel afterwards
// (dispatch.cu). Everything else goes to stage_gen.
bool stage_ko_tma_takes(const StageKOArgs& a) {
  return a.tmap && !a.A && a.fd_order == 4 && (a.ko_order == 0 || a.ko_order == 5) && a.b.g >= 3;
}

void launch_stage_ko_tma(const StageKOArgs& a, cudaStream_t st) {
  KoParams p{};
  p.b = a.b;
  p.F = a.F;
  p.a_Yu = a.a_Yu; p.a_Yr = a.a_Yr;
  p.yn_u = a.yn_u; p.yn_r = a.yn_r;
  p.U2 = a.U2; p.U3 = a.U3; p.R2 = a.R2; p.R3 = a.R3;
  p.Y4u = a.Yu; p.Y4r = a.Yr;
  p.outU = a.outU; p.outR = a.outR;
  p.K4u = a.K4u; p.K4r = a.K4r;
  for (int d = 0; d < 3; ++d) { p.w[d] = a.inv12dx2[d]; p.ko[d] = a.ko_order ? a.ko[d] : 0.0; }
  const int S = a.integrator, s = a.stage;
  bool combine = false;
  if (s > S) {                       // RK3: k_4 = M y_{n+1} only
    combine = true;
    p.outU = p.outR = nullptr;
  } else if (S == 4 && s == 4) {
    combine = true; p.c2 = 1.0 / 3.0; p.c3 = 2.0 / 3.0; p.c4 = 1.0 / 3.0; p.adt = a.dt / 6.0;
  } else if (S == 3 && s == 2) {     // Y_3 = y_n - 2 (Y_2 - y_n) + 2 dt k_2
    combine = true; p.c4 = -2.0; p.adt = 2.0 * a.dt;
  } else if (S == 3 && s == 3) {     // y_{n+1} = y_n + (Y_2 - y_n) + (Y_3 - y_n)/3 + dt/6 k_3;  k_3 kept where a child reads it
    combine = true; p.c2 = 1.0; p.c4 = 1.0 / 3.0; p.adt = a.dt / 6.0;
    p.K4u = a.K3u; p.K4r = a.K3r;
  } else if (S == 2 && s == 2) {
    combine = true; p.adt = a.dt;
  } else {
    p.adt = (S == 4 && s == 3 ? 1.0 : 0.5) * a.dt;
  }
  if (!combine) launch_ko_zmarch<0>(a, p, st);
  else if (p.c2 == 0.0 && p.c3 == 0.0) launch_ko_zmarch<2>(a, p, st);
  else launch_ko_zmarch<1>(a, p, st);
}

}  // namespace sc
