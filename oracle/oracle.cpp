// oracle.cpp — TEST INFRASTRUCTURE, not product code.
//
// A plain, slow, obviously-correct CPU implementation (fp64, C++17, optional OpenMP over k-planes) of
// what libsubcycle's hot path computes: one Berger–Oliger subcycled RK4 step over a nested-box AMR
// hierarchy with dense-output ghost fill (arXiv 2503.09629; citations are PAPER.md line numbers).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load
// it. It shares no code, header, table or constant with the CUDA path (it does not include
// include/subcycle.h) and follows the paper's equations in the paper's order and notation:
//
//   RK4, eqs (1)-(9) ....................... PAPER.md:54-75     -> rk4_level_step()
//   dense output b_i(theta), eqs (10)-(13) . PAPER.md:79-91     -> b_coeff()
//   time derivatives, eq (14) .............. PAPER.md:93-96     -> dense_stage()
//   ghost stage vectors, eqs (15)-(18) ..... PAPER.md:98-109    -> dense_stage()
//   recursion, steps 1-7 ................... PAPER.md:111-119   -> advance()
//   wave system, eqs (39)-(40) ............. PAPER.md:222-226   -> rhs()
//   Kreiss-Oliger dissipation, eqs (35)-(36) PAPER.md:194-204   -> add_dissipation()
//   same-level ghost exchange .............. PAPER.md:20, 347   -> sibling_exchange()
//   8th-order finite differences ........... PAPER.md:125       -> rhs() with fd_order = 8 (NEXT-3)
//   RK2 / RK3 subcycling ................... PAPER.md:359       -> rk_level_step(), b_coeff_rk3/2(), dense_stage_rk3/2() (NEXT-4, S28)
//   radiative (Sommerfeld) outer boundary .. PAPER.md:52, 113, 192 -> radiative_rhs() (NEXT-4, S29)
//   ninth-order KO dissipation, r = 8 ...... PAPER.md:125, eq 36 -> add_dissipation() with ko_order = 9 (NEXT-3)
//   interpolation that follows the stencil, vertex-centred grids with injection -> interp_* (NEXT-3, S30, S31)
//
// Where the paper is silent the readings S1..S24 of DESIGN.md apply (cell-centred grids S1, 4th-order
// centred Laplacian S2, quartic Lagrange prolongation S3, quintic Lagrange restriction S4, parent-step
// h in f_y y'' S5, periodic level 0 S9, non-subcycled mode S11/S15). Interpolation weights are computed
// here from the Lagrange formula, not tabulated; tests pin them to the rational values.
//
// Pins (tests/test_oracle_*.py, run with -m "not gpu"): dense-output invariants and the rational
// coefficient table; scalar-ODE stage-order test; closed-form single-level amplification matrix;
// polynomial exactness of prolongation / restriction / Laplacian; brute-force ghost index map;
// plane-wave convergence ladder (order ~4); subcycled-vs-uniform agreement; linearity; and the COMPOSITE
// multi-level step (dense-output fills at theta = 0 and 1/2, stage formulas, restrictions, both modes) against
// the exact solution u = r^2 + 3 t^2, rho = 6 t, which every operator reproduces to rounding
// (test_composite_scheme_exact_for_quadratic_solution); the same-level ghost exchange by decomposition
// invariance (a level cut into abutting boxes reproduces the uncut level bit for bit) and the same exact
// solution through abutting / edge-touching / near siblings (tests/test_oracle_siblings.py). What stays unpinned at bit level is only the
// composite step on data the operators do NOT reproduce exactly; there the oracle is the definition and the
// convergence ladder bounds it.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// The arithmetic type of everything below. The oracle is fp64 as shipped (`real` = double; the C interface at the end
// of the file is double in and out in every build). Compiling the SAME source with -DORACLE_LONG_DOUBLE (x86 long
// double: 64-bit mantissa, 11 more bits than fp64) gives the reference of higher precision that tests use to measure
// how far an fp64 evaluation of this definition lies from its exact-arithmetic value at a given depth (S27):
// state, slopes, weights and every accumulator are then long double. Constants are written so that they are exact in
// either type (2/3 as real(2)/real(3), never as the quotient of two double literals).
#ifdef ORACLE_LONG_DOUBLE
using real = long double;
#else
using real = double;
#endif

constexpr int kStencilRadius = 2;

// ---------------------------------------------------------------------------------------------
// dense output, eqs (10)-(18)
// ---------------------------------------------------------------------------------------------

// m-th theta-derivative (m = 0..3) of b_i(theta), i = 1..4; eqs (11)-(13).
real b_coeff(int i, int m, real th) {
  switch (i) {
    case 1:  // b1 = th - 3/2 th^2 + 2/3 th^3
      if (m == 0) return th - 1.5 * th * th + (real(2) / real(3)) * th * th * th;
      if (m == 1) return 1.0 - 3.0 * th + 2.0 * th * th;
      if (m == 2) return -3.0 + 4.0 * th;
      return 4.0;
    case 2:
    case 3:  // b2 = b3 = th^2 - 2/3 th^3
      if (m == 0) return th * th - (real(2) / real(3)) * th * th * th;
      if (m == 1) return 2.0 * th - 2.0 * th * th;
      if (m == 2) return 2.0 - 4.0 * th;
      return -4.0;
    default:  // b4 = -1/2 th^2 + 2/3 th^3
      if (m == 0) return -0.5 * th * th + (real(2) / real(3)) * th * th * th;
      if (m == 1) return -th + 2.0 * th * th;
      if (m == 2) return -1.0 + 4.0 * th;
      return 4.0;
  }
}

// Value that a refinement-boundary ghost cell of the child takes for RK "stage" of a child step that
// starts at parent progress theta, evaluated at ONE parent cell from the parent's y_n (= y_old) and
// k_1..k_4, which were computed with the parent's step hp. The child's step is h = hp/2 (S10).
//   stage 1..4: Y_1..Y_4 by eqs (15)-(18) with y, y', y'', y''' from eqs (10),(14) at theta, and
//               f_y y'' = 4 (k3 - k2) / hp^2 (reading S5: the parent's step);
//   stage 5:    y at "theta" by eq (10) alone (the caller passes theta + 1/2).
real dense_stage(int stage, real theta, real hp, real y_old, const real k[4]) {
  real y = y_old, d1 = 0.0, d2 = 0.0, d3 = 0.0;
  real s0 = 0.0;
  for (int i = 1; i <= 4; ++i) {
    s0 += b_coeff(i, 0, theta) * k[i - 1];
    d1 += b_coeff(i, 1, theta) * k[i - 1];
    d2 += b_coeff(i, 2, theta) * k[i - 1];
    d3 += b_coeff(i, 3, theta) * k[i - 1];
  }
  y = y_old + hp * s0;  // eq (10)
  d2 = d2 / hp;         // eq (14), m = 2
  d3 = d3 / (hp * hp);  // eq (14), m = 3
  if (stage == 1 || stage == 5) return y;  // eq (15) / eq (10)
  const real h = 0.5 * hp;               // child step
  const real fyy = 4.0 * (k[2] - k[1]) / (hp * hp);
  if (stage == 2) return y + 0.5 * h * d1;                                      // eq (16)
  if (stage == 3) return y + 0.5 * h * d1 + 0.25 * h * h * d2 + (h * h * h / 16.0) * (d3 - fyy);  // (17)
  return y + h * d1 + 0.5 * h * h * d2 + (h * h * h / 8.0) * (d3 + fyy);        // eq (18)
}

// ---------------------------------------------------------------------------------------------
// NEXT-4 ("extending it to RK2 and RK3 is straightforward"), reading S28. The extension repeats
// the construction of eqs (10)-(18) for the lower-order integrators:
//   RK3 = Kutta's third-order method:  k1 = f(Y1), k2 = f(Y2), k3 = f(Y3),
//         Y1 = y_n,  Y2 = y_n + h/2 k1,  Y3 = y_n - h k1 + 2 h k2,  y_{n+1} = y_n + h/6 (k1 + 4 k2 + k3);
//   RK2 = the midpoint method:         Y1 = y_n,  Y2 = y_n + h/2 k1,  y_{n+1} = y_n + h k2.
// Dense output (the analogue of eqs 10-13). RK4's eq (10) is a continuous extension one order below the method
// (local error O(h^4)). A three-stage third-order method has no such extension from k1..k3 alone (four order
// conditions, three polynomials), so a level that has a child evaluates one more slope, k4 = f(y_{n+1}), after
// its update (the child cannot start before y_{n+1} exists anyway); with c = (0, 1/2, 1, 1) the four conditions
//   sum b_i = theta,  sum b_i c_i = theta^2/2,  sum b_i c_i^2 = theta^3/3,  sum_i b_i sum_j a_ij c_j = theta^3/6
// have the unique solution
//   RK3:  b1 = theta - 3/2 theta^2 + 2/3 theta^3,  b2 = 2 theta^2 - 4/3 theta^3,
//         b3 = 1/2 theta^2 - 1/3 theta^3,          b4 = theta^3 - theta^2            (b(1) = (1/6, 2/3, 1/6, 0))
//   RK2:  b1 = theta - theta^2,  b2 = theta^2      (two conditions, two polynomials: full order from k1, k2)
// Ghost stage vectors (the analogue of eqs 15-18: Taylor expansion of the child's own stage values in its step h
// to the order the dense output supports; derivatives by eq 14 from the parent; D1, D2, D3 = first, second, third
// time derivative of y):
//   RK3:  Y1 = y,  Y2 = y + h/2 D1,  Y3 = y + h D1 + h^2 D2 + h^3/4 (D3 - f_y D2),   f_y D2 = 2 (k3 - k4) / hp^2
//         (k2 = D1 + h/2 D2 + h^2/8 (D3 - f_y D2) + O(h^3) in Y3 = y - h k1 + 2 h k2; the parent's
//          k3 - k4 = f(y + hp D1 + hp^2 D2 + ..) - f(y + hp D1 + hp^2/2 D2 + ..) = hp^2/2 f_y D2 + O(hp^3))
//   RK2:  Y1 = y,  Y2 = y + h/2 D1
// ---------------------------------------------------------------------------------------------
real b_coeff_rk3(int i, int m, real th) {
  switch (i) {
    case 1:
      if (m == 0) return th - 1.5 * th * th + (real(2) / real(3)) * th * th * th;
      if (m == 1) return 1.0 - 3.0 * th + 2.0 * th * th;
      if (m == 2) return -3.0 + 4.0 * th;
      return 4.0;
    case 2:
      if (m == 0) return 2.0 * th * th - (real(4) / real(3)) * th * th * th;
      if (m == 1) return 4.0 * th - 4.0 * th * th;
      if (m == 2) return 4.0 - 8.0 * th;
      return -8.0;
    case 3:
      if (m == 0) return 0.5 * th * th - (real(1) / real(3)) * th * th * th;
      if (m == 1) return th - th * th;
      if (m == 2) return 1.0 - 2.0 * th;
      return -2.0;
    default:
      if (m == 0) return th * th * th - th * th;
      if (m == 1) return 3.0 * th * th - 2.0 * th;
      if (m == 2) return 6.0 * th - 2.0;
      return 6.0;
  }
}
real b_coeff_rk2(int i, int m, real th) {
  if (i == 1) return m == 0 ? th - th * th : (m == 1 ? 1.0 - 2.0 * th : (m == 2 ? -2.0 : 0.0));
  return m == 0 ? th * th : (m == 1 ? 2.0 * th : (m == 2 ? 2.0 : 0.0));
}
// stage = 1..3 (RK3) / 1..2 (RK2): the ghost value of Y_stage; stage 5: y at `theta` by the dense output alone.
// RK3: k[0..2] = k1..k3 of the parent's step, k[3] = k4 = f(y_{n+1}).
real dense_stage_rk3(int stage, real theta, real hp, real y_old, const real k[4]) {
  real s0 = 0.0, d1 = 0.0, d2 = 0.0, d3 = 0.0;
  for (int i = 1; i <= 4; ++i) {
    s0 += b_coeff_rk3(i, 0, theta) * k[i - 1];
    d1 += b_coeff_rk3(i, 1, theta) * k[i - 1];
    d2 += b_coeff_rk3(i, 2, theta) * k[i - 1];
    d3 += b_coeff_rk3(i, 3, theta) * k[i - 1];
  }
  const real y = y_old + hp * s0;  // the analogue of eq (10)
  d2 = d2 / hp;                      // eq (14), m = 2
  d3 = d3 / (hp * hp);               // eq (14), m = 3
  if (stage == 1 || stage == 5) return y;
  const real h = 0.5 * hp;  // child step
  if (stage == 2) return y + 0.5 * h * d1;
  const real fyy = 2.0 * (k[2] - k[3]) / (hp * hp);
  return y + h * d1 + h * h * d2 + (h * h * h / 4.0) * (d3 - fyy);
}
real dense_stage_rk2(int stage, real theta, real hp, real y_old, const real k[2]) {
  real s0 = 0.0, d1 = 0.0;
  for (int i = 1; i <= 2; ++i) {
    s0 += b_coeff_rk2(i, 0, theta) * k[i - 1];
    d1 += b_coeff_rk2(i, 1, theta) * k[i - 1];
  }
  const real y = y_old + hp * s0;
  if (stage == 1 || stage == 5) return y;
  return y + 0.5 * (0.5 * hp) * d1;
}
real dense_stage_any(int integrator, int stage, real theta, real hp, real y_old, const real* k) {
  if (integrator == 3) return dense_stage_rk3(stage, theta, hp, y_old, k);
  if (integrator == 2) return dense_stage_rk2(stage, theta, hp, y_old, k);
  return dense_stage(stage, theta, hp, y_old, k);
}

// ---------------------------------------------------------------------------------------------
// spatial operators
// ---------------------------------------------------------------------------------------------

// Lagrange basis weights: value at x of the polynomial through (nodes[m], f_m) = sum_m w[m] f_m.
void lagrange_weights(const real* nodes, int n, real x, real* w) {
  for (int m = 0; m < n; ++m) {
    real v = 1.0;
    for (int q = 0; q < n; ++q)
      if (q != m) v *= (x - nodes[q]) / (nodes[m] - nodes[q]);
    w[m] = v;
  }
}

// Prolongation (S3): quartic through the 5 parent cells J-2..J+2 (centres at offsets -2..2 in units of
// the parent spacing) evaluated at the fine centre: -1/4 (parity 0) or +1/4 (parity 1).
void prolong_weights(int parity, real w[5]) {
  const real nodes[5] = {-2.0, -1.0, 0.0, 1.0, 2.0};
  lagrange_weights(nodes, 5, parity ? 0.25 : -0.25, w);
}

// Restriction (S4): quintic through the 6 fine cells 2J-2..2J+3, whose centres sit at -2.5..+2.5 fine
// spacings from the parent centre, evaluated at the parent centre.
void restrict_weights(real r[6]) {
  const real nodes[6] = {-2.5, -1.5, -0.5, 0.5, 1.5, 2.5};
  lagrange_weights(nodes, 6, 0.0, r);
}

// NEXT-3 variants of the two operators (readings S30, S31). `interp` = 0: the operators above (S3, S4);
// 1: operators whose order follows the 8th-order stencil of PAPER.md:125 (9-point prolongation, 10-point
// restriction). `vertex` = 1: vertex-centred grids (grid point i of level l sits at xlo + i dx_l): fine point 2J
// coincides with parent point J, so restriction is INJECTION and even fine points copy their parent; odd fine
// points 2J+1 sit midway between parents J and J+1 and take the Lagrange interpolant through parents J-2..J+3
// (interp 0, sextic-accurate) or J-4..J+5 (interp 1). All weights from the Lagrange formula.
struct Interp {
  int np = 5, omin = -2;   // prolongation: parent offsets omin .. omin + np - 1 around J = floor(I / 2)
  real w[2][10];         // [parity of the fine index][offset - omin]
  int nr = 6, rmin = -2;   // restriction: fine offsets rmin .. rmin + nr - 1 around 2J
  real r[10];
  int reach() const { return std::max(-omin, omin + np - 1); }  // parent cells the footprint extends beyond J
};
Interp make_interp(int interp, int vertex) {
  Interp P;
  real nodes[10];
  if (!vertex) {
    P.np = interp ? 9 : 5;
    P.omin = -(P.np / 2);
    for (int m = 0; m < P.np; ++m) nodes[m] = real(P.omin + m);
    lagrange_weights(nodes, P.np, -0.25, P.w[0]);
    lagrange_weights(nodes, P.np, +0.25, P.w[1]);
    P.nr = interp ? 10 : 6;
    P.rmin = -(P.nr / 2 - 1);
    // fine cell 2J + q has its centre at (q - 1/2) fine spacings from the parent centre J
    for (int m = 0; m < P.nr; ++m) nodes[m] = real(P.rmin + m) - 0.5;
    lagrange_weights(nodes, P.nr, 0.0, P.r);
  } else {
    P.np = interp ? 10 : 6;
    P.omin = -(P.np / 2 - 1);
    for (int m = 0; m < P.np; ++m) { nodes[m] = real(P.omin + m); P.w[0][m] = (P.omin + m == 0) ? 1.0 : 0.0; }
    lagrange_weights(nodes, P.np, 0.5, P.w[1]);
    P.nr = 1;
    P.rmin = 0;
    P.r[0] = 1.0;
  }
  return P;
}

inline int floor_div2(int a) { return (a >= 0) ? a / 2 : -((-a + 1) / 2); }
inline int pos_mod(int a, int n) { int r = a % n; return r < 0 ? r + n : r; }

// ---------------------------------------------------------------------------------------------
// hierarchy
// ---------------------------------------------------------------------------------------------
struct Field {  // one padded array of one box: index (i,j,k) in [-g, n+g)
  int n[3] = {0, 0, 0}, g = 0;
  std::vector<real> v;
  void init(const int nn[3], int gg) {
    for (int a = 0; a < 3; ++a) n[a] = nn[a];
    g = gg;
    v.assign(size_t(n[0] + 2 * g) * (n[1] + 2 * g) * (n[2] + 2 * g), 0.0);
  }
  inline size_t idx(int i, int j, int k) const {
    return size_t(i + g) + size_t(n[0] + 2 * g) * (size_t(j + g) + size_t(n[1] + 2 * g) * size_t(k + g));
  }
  inline real& at(int i, int j, int k) { return v[idx(i, j, k)]; }
  inline real at(int i, int j, int k) const { return v[idx(i, j, k)]; }
};

struct BoxData {
  int level = 0, lo[3] = {0, 0, 0}, n[3] = {0, 0, 0};
  int parent = -1;  // index into Hier::boxes of the containing box on level-1
  // per component c in [0, 2F): current state y, stage vector Y, start-of-step state y_old, slopes k1..k4
  std::vector<Field> y, Y, y_old, k[4];
};

struct Hier {
  int nlevels = 0, g = 3, F = 1;
  int domain[3] = {0, 0, 0};
  real xlo[3], xhi[3];
  std::vector<real> A;  // F*F coupling or empty
  real sigma = 0.0;     // Kreiss-Oliger dissipation strength (eqs 35-36); 0 = none
  int fd_order = 4;       // order of the centred finite differences of the RHS: 4 (S2) or 8 (NEXT-3)
  int ko_order = 5;       // 5: delta^6 (eq 36 with r = 4); 9: delta^10 (eq 36 with r = 8, "ninth-order")
  int integrator = 4;     // 4: RK4 (eqs 1-9); 3: Kutta's RK3; 2: midpoint RK2
  int outer_bc = 0;       // level 0: 0 = periodic (S9); 1 = radiative / Sommerfeld
  int interp = 0, vertex = 0;  // interpolation operators and grid centring (make_interp)
  Interp P = make_interp(0, 0);
  std::vector<BoxData> boxes;
  std::vector<std::vector<int>> level_boxes;
  real time = 0.0;
  real dx(int level, int a) const { return (xhi[a] - xlo[a]) / (real(domain[a]) * real(1 << level)); }
};

inline bool is_interior(const BoxData& b, int i, int j, int k) {
  return i >= 0 && i < b.n[0] && j >= 0 && j < b.n[1] && k >= 0 && k < b.n[2];
}

// ---------------------------------------------------------------------------------------------
// Kreiss-Oliger dissipation: d_t y -> RHS + Q y for EVERY evolved variable (eq 35),
//   Q y = (-1)^{r/2} sigma / 2^{r+2} sum_i h_i^{r+1} D_{i+}^{r/2+1} D_{i-}^{r/2+1} y          (eq 36)
// with r = 4 the order of the finite differences of the RHS (S2): (D+ D-)^3 y = delta^6 y / h^6,
//   delta^6 y = y[-3] - 6 y[-2] + 15 y[-1] - 20 y[0] + 15 y[+1] - 6 y[+2] + y[+3],
// so Q y = sigma / 64 sum_i delta_i^6 y / h_i. Uses all 3 ghost layers.
// ---------------------------------------------------------------------------------------------
void add_dissipation(const Hier& H, const BoxData& b, const std::vector<Field>& Y, std::vector<Field>& kout) {
  const int V = 2 * H.F;
  if (H.ko_order == 9) {
    // eq (36) with r = 8 ("ninth-order KO dissipation"): (-1)^4 sigma / 2^10 sum_i h_i^9 (D+ D-)^5 y
    //   = sigma / 1024 sum_i delta_i^10 y / h_i,  delta^10 = (1, -10, 45, -120, 210, -252, 210, -120, 45, -10, 1). 5 ghost layers.
    static const real d10[11] = {1.0, -10.0, 45.0, -120.0, 210.0, -252.0, 210.0, -120.0, 45.0, -10.0, 1.0};
    real c[3];
    for (int a = 0; a < 3; ++a) c[a] = H.sigma / (1024.0 * H.dx(b.level, a));
    for (int v = 0; v < V; ++v) {
      const Field& y = Y[v];
      Field& kv = kout[v];
#pragma omp parallel for schedule(static)
      for (int k = 0; k < b.n[2]; ++k)
        for (int j = 0; j < b.n[1]; ++j)
          for (int i = 0; i < b.n[0]; ++i) {
            real sx = 0.0, sy = 0.0, sz = 0.0;
            for (int m = -5; m <= 5; ++m) {
              sx += d10[m + 5] * y.at(i + m, j, k);
              sy += d10[m + 5] * y.at(i, j + m, k);
              sz += d10[m + 5] * y.at(i, j, k + m);
            }
            kv.at(i, j, k) += c[0] * sx + c[1] * sy + c[2] * sz;
          }
    }
    return;
  }
  real c[3];
  for (int a = 0; a < 3; ++a) c[a] = H.sigma / (64.0 * H.dx(b.level, a));
  for (int v = 0; v < V; ++v) {
    const Field& y = Y[v];
    Field& kv = kout[v];
#pragma omp parallel for schedule(static)
    for (int k = 0; k < b.n[2]; ++k)
      for (int j = 0; j < b.n[1]; ++j)
        for (int i = 0; i < b.n[0]; ++i) {
          const real d6x = y.at(i - 3, j, k) - 6.0 * y.at(i - 2, j, k) + 15.0 * y.at(i - 1, j, k) - 20.0 * y.at(i, j, k) +
                             15.0 * y.at(i + 1, j, k) - 6.0 * y.at(i + 2, j, k) + y.at(i + 3, j, k);
          const real d6y = y.at(i, j - 3, k) - 6.0 * y.at(i, j - 2, k) + 15.0 * y.at(i, j - 1, k) - 20.0 * y.at(i, j, k) +
                             15.0 * y.at(i, j + 1, k) - 6.0 * y.at(i, j + 2, k) + y.at(i, j + 3, k);
          const real d6z = y.at(i, j, k - 3) - 6.0 * y.at(i, j, k - 2) + 15.0 * y.at(i, j, k - 1) - 20.0 * y.at(i, j, k) +
                             15.0 * y.at(i, j, k + 1) - 6.0 * y.at(i, j, k + 2) + y.at(i, j, k + 3);
          kv.at(i, j, k) += c[0] * d6x + c[1] * d6y + c[2] * d6z;
        }
  }
}

// ---------------------------------------------------------------------------------------------
// NEXT-4: radiative (Sommerfeld) outer boundary, PAPER.md:52 ("outgoing wave conditions"), :113 (step 1: "using
// the physical boundary condition ... at the boundary"), :192 (NewRadX, outgoing boundary conditions applied to
// the dynamical variables). Reading S29: the cells of the level-0 box within g cells of a domain face are
// BOUNDARY POINTS; there every evolved variable y obeys, at every RK stage,
//     d_t y = - v0 [ (x^i / r) d_i y + (y - y_inf) / r ],     v0 = 1, y_inf = 0,
// with d_i y the second-order difference that fits in the box: centred where both neighbours exist, the one-sided
// three-point formula on the outermost layer. x = cell centre (grid point for vertex-centred grids), r = |x|.
// The boundary points are evolved by the same RK stages as the interior; ghost cells of level 0 are not used.
// ---------------------------------------------------------------------------------------------
void radiative_rhs(const Hier& H, const BoxData& b, const std::vector<Field>& Y, std::vector<Field>& kout) {
  const int V = 2 * H.F, nb = H.g;
  real dx[3];
  for (int a = 0; a < 3; ++a) dx[a] = H.dx(b.level, a);
  const real shift = H.vertex ? 0.0 : 0.5;
  for (int v = 0; v < V; ++v) {
    const Field& y = Y[v];
    Field& kv = kout[v];
#pragma omp parallel for schedule(static)
    for (int k = 0; k < b.n[2]; ++k)
      for (int j = 0; j < b.n[1]; ++j)
        for (int i = 0; i < b.n[0]; ++i) {
          const int idx[3] = {i, j, k};
          bool zone = false;
          for (int a = 0; a < 3; ++a)
            if (idx[a] < nb || idx[a] >= b.n[a] - nb) zone = true;
          if (!zone) continue;
          real x[3], d[3];
          for (int a = 0; a < 3; ++a) {
            x[a] = H.xlo[a] + (real(b.lo[a] + idx[a]) + shift) * dx[a];
            int e[3] = {0, 0, 0};
            e[a] = 1;
            auto Yat = [&](int m) { return y.at(i + m * e[0], j + m * e[1], k + m * e[2]); };
            if (idx[a] == 0) d[a] = (-3.0 * Yat(0) + 4.0 * Yat(1) - Yat(2)) / (2.0 * dx[a]);
            else if (idx[a] == b.n[a] - 1) d[a] = (3.0 * Yat(0) - 4.0 * Yat(-1) + Yat(-2)) / (2.0 * dx[a]);
            else d[a] = (Yat(1) - Yat(-1)) / (2.0 * dx[a]);
          }
          const real r = std::sqrt(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]);
          kv.at(i, j, k) = -((x[0] * d[0] + x[1] * d[1] + x[2] * d[2]) / r + y.at(i, j, k) / r);
        }
  }
}

// ---------------------------------------------------------------------------------------------
// right-hand side f(Y): k_u = rho ; k_rho = Lap_h u + A u   (eqs 39-40 + BASELINE cfg 4; S2)
// 4th-order centred second derivative (-1, 16, -30, 16, -1)/(12 dx^2) per axis.
// ---------------------------------------------------------------------------------------------
void rhs(const Hier& H, const BoxData& b, const std::vector<Field>& Y, std::vector<Field>& kout) {
  const int F = H.F;
  real inv12dx2[3];
  for (int a = 0; a < 3; ++a) {
    const real d = H.dx(b.level, a);
    inv12dx2[a] = 1.0 / (12.0 * d * d);
  }
  for (int f = 0; f < F; ++f) {
    const Field& u = Y[f];
    const Field& rho = Y[F + f];
    Field& ku = kout[f];
    Field& kr = kout[F + f];
#pragma omp parallel for schedule(static)
    for (int k = 0; k < b.n[2]; ++k)
      for (int j = 0; j < b.n[1]; ++j)
        for (int i = 0; i < b.n[0]; ++i) {
          const real dxx = (-u.at(i - 2, j, k) + 16.0 * u.at(i - 1, j, k) - 30.0 * u.at(i, j, k) +
                              16.0 * u.at(i + 1, j, k) - u.at(i + 2, j, k)) * inv12dx2[0];
          const real dyy = (-u.at(i, j - 2, k) + 16.0 * u.at(i, j - 1, k) - 30.0 * u.at(i, j, k) +
                              16.0 * u.at(i, j + 1, k) - u.at(i, j + 2, k)) * inv12dx2[1];
          const real dzz = (-u.at(i, j, k - 2) + 16.0 * u.at(i, j, k - 1) - 30.0 * u.at(i, j, k) +
                              16.0 * u.at(i, j, k + 1) - u.at(i, j, k + 2)) * inv12dx2[2];
          if (H.fd_order == 8) {  // the paper's BBH discretisation: 8th-order centred, 9 points per axis
            static const real c8[9] = {real(-1) / real(560), real(8) / real(315), real(-1) / real(5), real(8) / real(5), real(-205) / real(72),
                                       real(8) / real(5),    real(-1) / real(5),  real(8) / real(315), real(-1) / real(560)};
            real sx = 0.0, sy = 0.0, sz = 0.0;
            for (int m = -4; m <= 4; ++m) {
              sx += c8[m + 4] * u.at(i + m, j, k);
              sy += c8[m + 4] * u.at(i, j + m, k);
              sz += c8[m + 4] * u.at(i, j, k + m);
            }
            real src8 = 0.0;
            if (!H.A.empty())
              for (int q = 0; q < F; ++q) src8 += H.A[size_t(f) * F + q] * Y[q].at(i, j, k);
            ku.at(i, j, k) = rho.at(i, j, k);
            kr.at(i, j, k) = sx * 12.0 * inv12dx2[0] + sy * 12.0 * inv12dx2[1] + sz * 12.0 * inv12dx2[2] + src8;
            continue;
          }
          real src = 0.0;
          if (!H.A.empty())
            for (int q = 0; q < F; ++q) src += H.A[size_t(f) * F + q] * Y[q].at(i, j, k);
          ku.at(i, j, k) = rho.at(i, j, k);
          kr.at(i, j, k) = dxx + dyy + dzz + src;
        }
  }
  if (H.sigma != 0.0) add_dissipation(H, b, Y, kout);
  if (H.outer_bc == 1 && b.level == 0) radiative_rhs(H, b, Y, kout);  // boundary points: overrides the interior formulas
}

// ---------------------------------------------------------------------------------------------
// ghost fills
// ---------------------------------------------------------------------------------------------

// Level 0 (S9): every ghost cell takes the value of the interior cell at the periodically wrapped index.
void periodic_fill(const BoxData& b, std::vector<Field>& Y) {
  for (Field& f : Y) {
    const int g = f.g;
#pragma omp parallel for schedule(static)
    for (int k = -g; k < b.n[2] + g; ++k)
      for (int j = -g; j < b.n[1] + g; ++j)
        for (int i = -g; i < b.n[0] + g; ++i) {
          if (is_interior(b, i, j, k)) continue;
          f.at(i, j, k) = f.at(pos_mod(i, b.n[0]), pos_mod(j, b.n[1]), pos_mod(k, b.n[2]));
        }
  }
}

// Spatial prolongation of a parent-cell field C (stored over the parent box, interior valid) into the
// ghost cells of the child array `dst` (S3; variants: make_interp). Direct triple sum, x innermost then y then z.
void prolong_into_ghosts(const Hier& H, const BoxData& child, const BoxData& par, const Field& C, Field& dst) {
  const Interp& P = H.P;
  const int g = dst.g;
#pragma omp parallel for schedule(static)
  for (int k = -g; k < child.n[2] + g; ++k)
    for (int j = -g; j < child.n[1] + g; ++j)
      for (int i = -g; i < child.n[0] + g; ++i) {
        if (is_interior(child, i, j, k)) continue;
        const int I[3] = {child.lo[0] + i, child.lo[1] + j, child.lo[2] + k};  // level-global fine index
        int J[3], p[3];
        for (int a = 0; a < 3; ++a) {
          const int Jg = floor_div2(I[a]);  // containing parent cell (global)
          p[a] = I[a] - 2 * Jg;             // 0: fine centre at -dx_p/4, 1: at +dx_p/4 (vertex grids: 0 = on the parent point)
          J[a] = Jg - par.lo[a];            // parent-box-local
        }
        real sz = 0.0;
        for (int c = 0; c < P.np; ++c) {
          real sy = 0.0;
          for (int bb = 0; bb < P.np; ++bb) {
            real sx = 0.0;
            for (int a = 0; a < P.np; ++a) sx += P.w[p[0]][a] * C.at(J[0] + P.omin + a, J[1] + P.omin + bb, J[2] + P.omin + c);
            sy += P.w[p[1]][bb] * sx;
          }
          sz += P.w[p[2]][c] * sy;
        }
        dst.at(i, j, k) = sz;
      }
}

// fill(l, stage, theta) for a level >= 1 box in SUBCYCLED mode: evaluate the
// parent's dense output at every parent cell (combine), then prolong once into the child's ghosts.
void dense_ghost_fill(const Hier& H, const BoxData& child, const BoxData& par, std::vector<Field>& dst,
                      int stage, real theta, real hp) {
  Field C;
  C.init(par.n, H.g);
  // parent cells any ghost cell of the child can reach: ceil(g/2) cells beyond the child's coverage
  // plus the 2-cell interpolation radius (all inside the parent's interior by the nesting rule S13)
  const int reach = (H.g + 1) / 2 + H.P.reach();
  int lo[3], hi[3];
  for (int a = 0; a < 3; ++a) {
    lo[a] = child.lo[a] / 2 - par.lo[a] - reach;
    hi[a] = (child.lo[a] + child.n[a]) / 2 - par.lo[a] + reach;
  }
  for (int c = 0; c < 2 * H.F; ++c) {
#pragma omp parallel for schedule(static)
    for (int k = lo[2]; k < hi[2]; ++k)
      for (int j = lo[1]; j < hi[1]; ++j)
        for (int i = lo[0]; i < hi[0]; ++i) {
          const real kk[4] = {par.k[0][c].at(i, j, k), par.k[1][c].at(i, j, k), par.k[2][c].at(i, j, k),
                                par.k[3][c].at(i, j, k)};
          C.at(i, j, k) = dense_stage_any(H.integrator, stage, theta, hp, par.y_old[c].at(i, j, k), kk);
        }
    prolong_into_ghosts(H, child, par, C, dst[c]);
  }
}

// Restriction (PAPER.md:119 step 7, S4): every parent cell whose children lie in the child's interior
// takes the quintic interpolant of the child's y (reads up to 2 child ghost layers; variants: make_interp —
// 10-point: 4 layers; vertex-centred: injection of the coincident fine point).
void restrict_to_parent(const Hier& H, const BoxData& child, BoxData& par) {
  const Interp& P = H.P;
  const int J0[3] = {child.lo[0] / 2 - par.lo[0], child.lo[1] / 2 - par.lo[1], child.lo[2] / 2 - par.lo[2]};
  const int nc[3] = {child.n[0] / 2, child.n[1] / 2, child.n[2] / 2};
  for (int c = 0; c < 2 * H.F; ++c) {
    const Field& yc = child.y[c];
    Field& yp = par.y[c];
#pragma omp parallel for schedule(static)
    for (int K = 0; K < nc[2]; ++K)
      for (int J = 0; J < nc[1]; ++J)
        for (int I = 0; I < nc[0]; ++I) {
          real sz = 0.0;
          for (int cc = 0; cc < P.nr; ++cc) {
            real sy = 0.0;
            for (int bb = 0; bb < P.nr; ++bb) {
              real sx = 0.0;
              for (int a = 0; a < P.nr; ++a)
                sx += P.r[a] * yc.at(2 * I + P.rmin + a, 2 * J + P.rmin + bb, 2 * K + P.rmin + cc);
              sy += P.r[bb] * sx;
            }
            sz += P.r[cc] * sy;
          }
          yp.at(J0[0] + I, J0[1] + J, J0[2] + K) = sz;
        }
  }
}

// Same-level ghost exchange (NEXT-2; the ghost zones at a refinement boundary are the same
// zones an inter-process boundary uses). Boxes of one level may abut or sit closer than a ghost width: every
// ghost cell of a box that lies in the INTERIOR of a sibling box takes the sibling's value of the same array
// (the same stage vector at the same time), replacing whatever the refinement-boundary fill wrote there. A
// level cut into abutting boxes therefore computes exactly what the uncut level computes.
void sibling_exchange(Hier& H, int level, std::vector<Field> BoxData::*which) {
  const int g = H.g;
  for (int ia : H.level_boxes[level])
    for (int ib : H.level_boxes[level]) {
      if (ia == ib) continue;
      BoxData& A = H.boxes[ia];
      const BoxData& B = H.boxes[ib];
      int lo[3], hi[3];  // level-global index range of  padded(A) n interior(B)
      bool empty = false;
      for (int a = 0; a < 3; ++a) {
        lo[a] = std::max(A.lo[a] - g, B.lo[a]);
        hi[a] = std::min(A.lo[a] + A.n[a] + g, B.lo[a] + B.n[a]);
        if (hi[a] <= lo[a]) empty = true;
      }
      if (empty) continue;
      for (size_t c = 0; c < (A.*which).size(); ++c)
        for (int k = lo[2]; k < hi[2]; ++k)
          for (int j = lo[1]; j < hi[1]; ++j)
            for (int i = lo[0]; i < hi[0]; ++i)
              (A.*which)[c].at(i - A.lo[0], j - A.lo[1], k - A.lo[2]) =
                  (B.*which)[c].at(i - B.lo[0], j - B.lo[1], k - B.lo[2]);
    }
}

// ---------------------------------------------------------------------------------------------
// time stepping
// ---------------------------------------------------------------------------------------------
void axpy_interior(const BoxData& b, std::vector<Field>& out, const std::vector<Field>& y0, real a,
                   const std::vector<Field>& kk) {
  for (size_t c = 0; c < out.size(); ++c) {
#pragma omp parallel for schedule(static)
    for (int k = 0; k < b.n[2]; ++k)
      for (int j = 0; j < b.n[1]; ++j)
        for (int i = 0; i < b.n[0]; ++i) out[c].at(i, j, k) = y0[c].at(i, j, k) + a * kk[c].at(i, j, k);
  }
}

void fill(Hier& H, int level, std::vector<Field> BoxData::*which, int stage, real theta, real dt) {
  for (int ib : H.level_boxes[level]) {
    BoxData& b = H.boxes[ib];
    if (level == 0) { if (H.outer_bc == 0) periodic_fill(b, b.*which); }  // radiative: no ghosts, boundary points evolve
    else dense_ghost_fill(H, b, H.boxes[b.parent], b.*which, stage, theta, 2.0 * dt);
  }
  sibling_exchange(H, level, which);
}

// Stage vector Y_{s+1} from y_n and the slopes so far, and the final update, on the interior of one box, for the
// integrator in use: RK4 eqs (5), (7)-(9); RK3 / RK2 the tableaux of reading S28 (see b_coeff_rk3).
void next_stage_vector(const Hier& H, BoxData& b, int s, real dt) {
  if (H.integrator == 4) {
    const real a_s[3] = {0.5, 0.5, 1.0};
    axpy_interior(b, b.Y, b.y_old, a_s[s - 1] * dt, b.k[s - 1]);  // eqs (7)-(9)
    return;
  }
  if (s == 1) { axpy_interior(b, b.Y, b.y_old, 0.5 * dt, b.k[0]); return; }  // Y2 = y_n + h/2 k1 (RK3 and RK2)
  for (size_t c = 0; c < b.Y.size(); ++c) {                                  // RK3: Y3 = y_n - h k1 + 2 h k2
#pragma omp parallel for schedule(static)
    for (int k = 0; k < b.n[2]; ++k)
      for (int j = 0; j < b.n[1]; ++j)
        for (int i = 0; i < b.n[0]; ++i)
          b.Y[c].at(i, j, k) = b.y_old[c].at(i, j, k) + dt * (-b.k[0][c].at(i, j, k) + 2.0 * b.k[1][c].at(i, j, k));
  }
}
void final_update(const Hier& H, BoxData& b, real dt) {
  for (int c = 0; c < 2 * H.F; ++c) {
#pragma omp parallel for schedule(static)
    for (int k = 0; k < b.n[2]; ++k)
      for (int j = 0; j < b.n[1]; ++j)
        for (int i = 0; i < b.n[0]; ++i) {
          if (H.integrator == 4)
            b.y[c].at(i, j, k) = b.y_old[c].at(i, j, k) +
                                 (dt / 6.0) * (b.k[0][c].at(i, j, k) + 2.0 * b.k[1][c].at(i, j, k) +
                                               2.0 * b.k[2][c].at(i, j, k) + b.k[3][c].at(i, j, k));  // eq (5)
          else if (H.integrator == 3)
            b.y[c].at(i, j, k) = b.y_old[c].at(i, j, k) +
                                 (dt / 6.0) * (b.k[0][c].at(i, j, k) + 4.0 * b.k[1][c].at(i, j, k) + b.k[2][c].at(i, j, k));
          else
            b.y[c].at(i, j, k) = b.y_old[c].at(i, j, k) + dt * b.k[1][c].at(i, j, k);
        }
  }
}

// One RK step of all boxes of one level (RK4: eqs 1-9), ghosts by fill(); theta = where this step starts
// inside the parent's step (0 or 1/2; ignored on level 0).
void rk4_level_step(Hier& H, int level, real dt, real theta) {
  const int S = H.integrator;  // number of stages: RK4 4, RK3 3, RK2 2
  for (int ib : H.level_boxes[level]) {
    BoxData& b = H.boxes[ib];
    b.y_old = b.y;  // y_n
  }
  fill(H, level, &BoxData::y_old, 1, theta, dt);  // eq (15): Y_1 = y_n also in the ghosts
  for (int ib : H.level_boxes[level]) H.boxes[ib].Y = H.boxes[ib].y_old;  // eq (6)
  for (int s = 1; s <= S; ++s) {
    for (int ib : H.level_boxes[level]) rhs(H, H.boxes[ib], H.boxes[ib].Y, H.boxes[ib].k[s - 1]);  // (1)-(4)
    if (s < S) {
      for (int ib : H.level_boxes[level]) next_stage_vector(H, H.boxes[ib], s, dt);
      fill(H, level, &BoxData::Y, s + 1, theta, dt);  // eqs (16)-(18) in the ghosts
    }
  }
  for (int ib : H.level_boxes[level]) final_update(H, H.boxes[ib], dt);
  fill(H, level, &BoxData::y, 5, theta + 0.5, dt);  // eq (10) at theta + 1/2 in the ghosts
  if (S == 3 && level + 1 < H.nlevels)  // RK3 (S28): the slope at the new state completes the dense output the child reads
    for (int ib : H.level_boxes[level]) rhs(H, H.boxes[ib], H.boxes[ib].y, H.boxes[ib].k[3]);
}

// Steps 1-7.
void advance(Hier& H, int level, real dt, real theta) {
  rk4_level_step(H, level, dt, theta);
  if (level + 1 < H.nlevels) {
    advance(H, level + 1, 0.5 * dt, 0.0);
    advance(H, level + 1, 0.5 * dt, 0.5);
    for (int ib : H.level_boxes[level + 1]) restrict_to_parent(H, H.boxes[ib], H.boxes[H.boxes[ib].parent]);
  }
}

// Non-subcycled mode (S11, S15): all levels take the same step dt; refinement ghosts are the plain
// spatial prolongation of the parent's SAME stage vector; restriction once per step, finest first.
void same_time_fill(Hier& H, int level, std::vector<Field> BoxData::*which) {
  for (int ib : H.level_boxes[level]) {
    BoxData& b = H.boxes[ib];
    if (level == 0) { if (H.outer_bc == 0) periodic_fill(b, b.*which); continue; }
    const BoxData& par = H.boxes[b.parent];
    for (int c = 0; c < 2 * H.F; ++c) prolong_into_ghosts(H, b, par, (par.*which)[c], (b.*which)[c]);
  }
  sibling_exchange(H, level, which);
}

void uniform_step(Hier& H, real dt) {
  const int L = H.nlevels, S = H.integrator;
  for (BoxData& b : H.boxes) b.y_old = b.y;
  for (int l = 0; l < L; ++l) same_time_fill(H, l, &BoxData::y_old);
  for (BoxData& b : H.boxes) b.Y = b.y_old;
  for (int s = 1; s <= S; ++s) {
    for (BoxData& b : H.boxes) rhs(H, b, b.Y, b.k[s - 1]);
    if (s < S) {
      for (BoxData& b : H.boxes) next_stage_vector(H, b, s, dt);
      for (int l = 0; l < L; ++l) same_time_fill(H, l, &BoxData::Y);
    }
  }
  for (BoxData& b : H.boxes) final_update(H, b, dt);
  for (int l = 0; l < L; ++l) same_time_fill(H, l, &BoxData::y);
  for (int l = L - 1; l >= 1; --l)
    for (int ib : H.level_boxes[l]) restrict_to_parent(H, H.boxes[ib], H.boxes[H.boxes[ib].parent]);
}

// preconditions the loops above rely on (S13)
bool validate(Hier& H, char* msg, size_t cap) {
  auto fail = [&](const char* m) { snprintf(msg, cap, "%s", m); return false; };
  if (H.nlevels < 1 || H.boxes.empty()) return fail("no levels");
  if (H.g < kStencilRadius || H.g > 8) return fail("ghost width");
  if (H.level_boxes[0].size() != 1) return fail("level 0 must be one box");
  const BoxData& b0 = H.boxes[H.level_boxes[0][0]];
  for (int a = 0; a < 3; ++a)
    if (b0.lo[a] != 0 || b0.n[a] != H.domain[a] || b0.n[a] < H.g) return fail("level 0 must cover the domain");
  const int margin = (H.g + 1) / 2 + H.P.reach();
  for (int l = 1; l < H.nlevels; ++l) {
    if (H.level_boxes[l].empty()) return fail("empty level");
    for (int ib : H.level_boxes[l]) {
      BoxData& b = H.boxes[ib];
      b.parent = -1;
      for (int a = 0; a < 3; ++a)
        if ((b.lo[a] & 1) || (b.n[a] & 1) || b.n[a] < 8) return fail("box lo/n must be even, n >= 8");
      for (int ip : H.level_boxes[l - 1]) {
        const BoxData& p = H.boxes[ip];
        bool inside = true;
        for (int a = 0; a < 3; ++a) {
          const int plo = b.lo[a] / 2 - p.lo[a], phi = (b.lo[a] + b.n[a]) / 2 - p.lo[a];
          if (plo < margin || phi > p.n[a] - margin) inside = false;
        }
        if (inside) { b.parent = ip; break; }
      }
      if (b.parent < 0) return fail("box not properly nested in a parent box");
      for (int jb : H.level_boxes[l]) {
        if (jb == ib) continue;
        const BoxData& o = H.boxes[jb];
        bool disjoint = false;  // interiors must not overlap; any distance (abutting included) is fine
        for (int a = 0; a < 3; ++a)
          if (b.lo[a] >= o.lo[a] + o.n[a] || o.lo[a] >= b.lo[a] + b.n[a]) disjoint = true;
        if (!disjoint) return fail("sibling boxes overlap");
      }
    }
  }
  return true;
}

BoxData* get_box(Hier* H, int level, int box) {
  if (!H || level < 0 || level >= H->nlevels) return nullptr;
  if (box < 0 || box >= int(H->level_boxes[level].size())) return nullptr;
  return &H->boxes[H->level_boxes[level][box]];
}

thread_local char g_err[256] = "";

}  // namespace

// ---------------------------------------------------------------------------------------------
// C interface (loaded with ctypes by oracle/__init__.py)
// ---------------------------------------------------------------------------------------------
extern "C" {

const char* oc_last_error() { return g_err; }

void oc_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

int oc_max_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// unit-level entry points used by the pins
double oc_b(int i, int m, double theta) { return b_coeff(i, m, theta); }
double oc_dense_stage(int stage, double theta, double hp, double y_old, const double* k4) {
  const real k[4] = {k4[0], k4[1], k4[2], k4[3]};
  return dense_stage(stage, theta, hp, y_old, k);
}
void oc_prolong_weights(int parity, double* w5) {
  real w[5];
  prolong_weights(parity, w);
  for (int m = 0; m < 5; ++m) w5[m] = double(w[m]);
}
void oc_restrict_weights(double* r6) {
  real r[6];
  restrict_weights(r);
  for (int m = 0; m < 6; ++m) r6[m] = double(r[m]);
}
// sizeof of the arithmetic type of this build (8: the fp64 oracle; 16: the long double reference of DESIGN.md S27)
int oc_real_bytes() { return int(sizeof(real)); }

void* oc_create(int nlevels, int nboxes, const int* box_level, const int* box_lo, const int* box_n, int ghost,
                int nfields, const int* domain_cells, const double* xlo, const double* xhi,
                const double* coupling) {
  Hier* H = new Hier;
  H->nlevels = nlevels;
  H->g = ghost;
  H->F = nfields;
  for (int a = 0; a < 3; ++a) { H->domain[a] = domain_cells[a]; H->xlo[a] = xlo[a]; H->xhi[a] = xhi[a]; }
  if (coupling) H->A.assign(coupling, coupling + size_t(nfields) * nfields);
  if (nlevels < 1 || nlevels > 30 || nboxes < 1 || nfields < 1) {
    snprintf(g_err, sizeof g_err, "bad sizes");
    delete H;
    return nullptr;
  }
  H->level_boxes.resize(nlevels);
  H->boxes.resize(nboxes);
  for (int ib = 0; ib < nboxes; ++ib) {
    BoxData& b = H->boxes[ib];
    b.level = box_level[ib];
    if (b.level < 0 || b.level >= nlevels || (ib > 0 && b.level < box_level[ib - 1])) {
      snprintf(g_err, sizeof g_err, "boxes must be sorted by level");
      delete H;
      return nullptr;
    }
    for (int a = 0; a < 3; ++a) { b.lo[a] = box_lo[3 * ib + a]; b.n[a] = box_n[3 * ib + a]; }
    H->level_boxes[b.level].push_back(ib);
  }
  if (!validate(*H, g_err, sizeof g_err)) { delete H; return nullptr; }
  for (BoxData& b : H->boxes) {
    const int V = 2 * nfields;
    b.y.resize(V); b.Y.resize(V); b.y_old.resize(V);
    for (int s = 0; s < 4; ++s) b.k[s].resize(V);
    for (int c = 0; c < V; ++c) {
      b.y[c].init(b.n, ghost); b.Y[c].init(b.n, ghost); b.y_old[c].init(b.n, ghost);
      for (int s = 0; s < 4; ++s) b.k[s][c].init(b.n, ghost);
    }
  }
  return H;
}

void oc_destroy(void* h) { delete static_cast<Hier*>(h); }

// Kreiss-Oliger strength sigma of eq (36); needs ghost width >= 3. Returns 0, or -1 with oc_last_error set.
int oc_set_dissipation(void* h, double sigma) {
  Hier* H = static_cast<Hier*>(h);
  if (!H || !(sigma >= 0.0) || (sigma != 0.0 && H->g < (H->ko_order == 9 ? 5 : 3))) {
    snprintf(g_err, sizeof g_err, "dissipation needs sigma >= 0 and ghost width >= 3");
    return -1;
  }
  H->sigma = sigma;
  return 0;
}

// Order of the centred finite differences of the RHS: 4 (default, S2) or 8 (reads 4 ghost layers).
// The dissipation order is a separate option (oc_set_options: the paper runs 8th-order differences with FIFTH-
// order dissipation, while eq 36 ties it to r). Returns 0, or -1 with oc_last_error set.
int oc_set_fd_order(void* h, int order) {
  Hier* H = static_cast<Hier*>(h);
  if (!H || (order != 4 && order != 8) || (order == 8 && H->g < 4)) {
    snprintf(g_err, sizeof g_err, "fd order must be 4, or 8 with ghost width >= 4");
    return -1;
  }
  H->fd_order = order;
  return 0;
}

// NEXT-3 / NEXT-4 options, set right after oc_create (before any state is evolved). Returns 0, or -1 with oc_last_error:
//   integrator 4 | 3 | 2;  outer_bc 0 periodic | 1 radiative;  ko_order 5 | 9 (0: eq 36's r = fd_order -> 5 | 9);
//   interp 0 (S3/S4) | 1 (follows the 8th-order stencil);  vertex 0 | 1.
int oc_set_options(void* h, int integrator, int outer_bc, int ko_order, int interp, int vertex) {
  Hier* H = static_cast<Hier*>(h);
  if (!H) return -1;
  if (integrator == 0) integrator = 4;
  if (ko_order == 0) ko_order = H->fd_order == 8 ? 9 : 5;
  const int ko_layers = ko_order == 9 ? 5 : 3;
  if ((integrator != 4 && integrator != 3 && integrator != 2) || (outer_bc != 0 && outer_bc != 1) ||
      (ko_order != 5 && ko_order != 9) || (interp != 0 && interp != 1) || (vertex != 0 && vertex != 1)) {
    snprintf(g_err, sizeof g_err, "bad option value");
    return -1;
  }
  if (H->sigma != 0.0 && H->g < ko_layers) { snprintf(g_err, sizeof g_err, "dissipation order %d reads %d ghost layers", ko_order, ko_layers); return -1; }
  H->integrator = integrator;
  H->outer_bc = outer_bc;
  H->ko_order = ko_order;
  H->interp = interp;
  H->vertex = vertex;
  H->P = make_interp(interp, vertex);
  if (H->P.nr > 1 && -H->P.rmin > H->g) { snprintf(g_err, sizeof g_err, "restriction reads %d ghost layers", -H->P.rmin); return -1; }
  if (!validate(*H, g_err, sizeof g_err)) return -1;  // the nesting margin depends on the footprint
  return 0;
}
void oc_interp_weights(int interp, int vertex, int* np, int* omin, double* w0, double* w1, int* nr, int* rmin, double* r) {
  const Interp P = make_interp(interp, vertex);
  *np = P.np; *omin = P.omin; *nr = P.nr; *rmin = P.rmin;
  for (int m = 0; m < P.np; ++m) { w0[m] = P.w[0][m]; w1[m] = P.w[1][m]; }
  for (int m = 0; m < P.nr; ++m) r[m] = P.r[m];
}
double oc_b_rk(int integrator, int i, int m, double theta) {
  return integrator == 3 ? b_coeff_rk3(i, m, theta) : (integrator == 2 ? b_coeff_rk2(i, m, theta) : b_coeff(i, m, theta));
}
double oc_dense_stage_rk(int integrator, int stage, double theta, double hp, double y_old, const double* k) {
  const int nk = integrator == 2 ? 2 : 4;  // slopes the formulas of this integrator read (RK3: k_1..k_3 and k_4 = f(y_{n+1}))
  real kr[4] = {0, 0, 0, 0};
  for (int s = 0; s < nk; ++s) kr[s] = k[s];
  return dense_stage_any(integrator, stage, theta, hp, y_old, kr);
}

int oc_set_state(void* h, int level, int box, int comp, const double* src) {
  Hier* H = static_cast<Hier*>(h);
  BoxData* b = get_box(H, level, box);
  if (!b || !src || comp < 0 || comp >= 2 * H->F) return -1;
  size_t q = 0;
  for (int k = 0; k < b->n[2]; ++k)
    for (int j = 0; j < b->n[1]; ++j)
      for (int i = 0; i < b->n[0]; ++i) b->y[comp].at(i, j, k) = src[q++];
  return 0;
}

// slot: 0 = y (current), 1 = y_old, 2..5 = k_1..k_4; padded != 0 -> include ghosts
int oc_read(void* h, int level, int box, int slot, int comp, int padded, double* dst) {
  Hier* H = static_cast<Hier*>(h);
  BoxData* b = get_box(H, level, box);
  if (!b || !dst || comp < 0 || comp >= 2 * H->F || slot < 0 || slot > 5) return -1;
  const Field& f = slot == 0 ? b->y[comp] : slot == 1 ? b->y_old[comp] : b->k[slot - 2][comp];
  const int e = padded ? H->g : 0;
  size_t q = 0;
  for (int k = -e; k < b->n[2] + e; ++k)
    for (int j = -e; j < b->n[1] + e; ++j)
      for (int i = -e; i < b->n[0] + e; ++i) dst[q++] = f.at(i, j, k);
  return 0;
}

int oc_step(void* h, double dt_coarse, int subcycling) {
  Hier* H = static_cast<Hier*>(h);
  if (!H || !(dt_coarse == dt_coarse)) return -1;
  if (subcycling) {
    advance(*H, 0, dt_coarse, 0.0);
  } else {
    const int nsub = 1 << (H->nlevels - 1);
    for (int q = 0; q < nsub; ++q) uniform_step(*H, dt_coarse / double(nsub));
  }
  H->time += dt_coarse;
  return 0;
}

double oc_time(void* h) { return static_cast<Hier*>(h)->time; }

// Ghost index map of a level >= 1 box: canonical order (k, j, i over the padded box, interior skipped);
// 7 ints per ghost cell: i, j, k (box-local), pi, pj, pk (parent-box-local), parity bits px|py<<1|pz<<2.
long long oc_ghost_map(void* h, int level, int box, int* out, unsigned long long cap) {
  Hier* H = static_cast<Hier*>(h);
  BoxData* b = get_box(H, level, box);
  if (!b || level < 1) return -1;
  const BoxData& par = H->boxes[b->parent];
  const int g = H->g;
  long long cnt = 0;
  for (int k = -g; k < b->n[2] + g; ++k)
    for (int j = -g; j < b->n[1] + g; ++j)
      for (int i = -g; i < b->n[0] + g; ++i) {
        if (is_interior(*b, i, j, k)) continue;
        if (out && (unsigned long long)(7 * (cnt + 1)) <= cap) {
          const int loc[3] = {i, j, k};
          int* o = out + 7 * cnt;
          int bits = 0;
          for (int a = 0; a < 3; ++a) {
            const int I = b->lo[a] + loc[a];
            const int Jg = floor_div2(I);
            o[a] = loc[a];
            o[3 + a] = Jg - par.lo[a];
            bits |= (I - 2 * Jg) << a;
          }
          o[6] = bits;
        }
        ++cnt;
      }
  return cnt;
}

}  // extern "C"
