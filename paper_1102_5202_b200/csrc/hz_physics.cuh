// hz_physics.cuh -- per-point device arithmetic of the GRMHD substep (sm_100a, fp64 and fp32).
//
// Every function restates a formula of DESIGN.md section 3 (readings O1-O8 of the paper's
// pipeline) for one cell or one face, in registers.  Nothing here touches memory;
// the kernels in hz_kernels.cuh decide what is staged where.  This file shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>

namespace hz {

constexpr int NV = 9;   // rho|D, ut^i|S_i, p|tau, B^i, psi
constexpr int NM = 10;  // alpha, beta^i, gamma_xx xy xz yy yz zz
constexpr int NG = 2;   // ghost layers per active side: the MC stencil (R16)

enum { RHO = 0, UX = 1, UY = 2, UZ = 3, PR = 4, BX = 5, BY = 6, BZ = 7, PSI = 8 };
enum { AL = 0, BEX = 1, BEY = 2, BEZ = 3, GXX = 4, GXY = 5, GXZ = 6, GYY = 7, GYZ = 8, GZZ = 9 };

// Run-time parameters in the arithmetic type of the kernels.
template <typename T>
struct Par {
  T Gam;       // Gamma
  T gg1;       // Gamma/(Gamma-1)
  T g1g;       // (Gamma-1)/Gamma
  T rho_atm, p_atm;
  T rho_thr;   // rho_atm*(1+atm_tol)
  T kappa;
  T c2p_tol;
  T ih[3];     // 1/dx, 1/dy, 1/dz
  int c2p_maxit;
  int c2p_scheme;  // 0: Newton on Z, 1: Newton on (Z, v^2)
  int energy_var;  // 0: slot 4 of U is tau; 1: the paper's -sqrt(-g) T^t_t / sqrt(gamma) (R1b)
  int cleaning;
};

// ---- scalar helpers -----------------------------------------------------------------------------
// Reciprocal, division and square roots without the library's special-case branches: every operand
// on this path is a normal, finite, positive-scale number (densities, determinants, 1 - v^2 a^2 ...).
// fp64: hardware seed (MUFU.RCP64H, ~20 bits) + one cubic Newton step (error ~2^-60) and, for the
// quotient, one residual correction; results agree with IEEE division to the last bit or two.
// fp32: the hardware approximations (1-2 ulp), far inside the fp32 parity tolerance.
__device__ __forceinline__ double rcp_(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x, y, 1.0);
  const double e2 = fma(e, e, e);
  return fma(y, e2, y);
}
__device__ __forceinline__ float rcp_(float x) {
  float y;
  asm("rcp.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ double div_(double a, double b) {
  const double y = rcp_(b);
  const double q = a * y;
  const double r = fma(-b, q, a);
  return fma(y, r, q);
}
__device__ __forceinline__ float div_(float a, float b) {
  float q;
  asm("div.approx.f32 %0, %1, %2;" : "=f"(q) : "f"(a), "f"(b));
  return q;
}
// fp64 reciprocal square root and square root of a POSITIVE, finite, normal argument (Lorentz factors, metric
// determinants, 1 - v^2 of an accepted Newton trial): hardware seed (MUFU.RSQ64H, >= 20 bits) + one third-order
// step (relative error ~1e-18 before rounding), and for the root one residual correction.  No special cases: a
// zero or negative argument gives inf / NaN, which the callers' finite checks treat as a failed trial.  The
// library routines (sqrt, rsqrt) spend twice the instructions on the cases that cannot occur here.
__device__ __forceinline__ double rsqrt_(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double t = x * y;
  const double e = fma(-t, y, 1.0);
  const double p = fma(0.375, e, 0.5);
  return fma(y * e, p, y);
}
__device__ __forceinline__ double sqrt_(double x) {
  const double y = rsqrt_(x);
  const double s = x * y;
  const double r = fma(-s, s, x);
  return fma(r * 0.5, y, s);
}
// square root of an argument that may be exactly zero
__device__ __forceinline__ double sqrt0_(double x) { return sqrt(x); }
__device__ __forceinline__ float sqrt_(float x) {
  float y;
  asm("sqrt.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float sqrt0_(float x) { return sqrt_(x); }
__device__ __forceinline__ float rsqrt_(float x) {
  float y;
  asm("rsqrt.approx.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ double abs_(double x) { return fabs(x); }
__device__ __forceinline__ float abs_(float x) { return fabsf(x); }
// fp64 min/max as one compare and a select (no NaN fix-up: operands here are never NaN by construction,
// and a NaN state is caught by the finite checks of the primitive recovery)
__device__ __forceinline__ double min_(double a, double b) { return a < b ? a : b; }
__device__ __forceinline__ float min_(float a, float b) { return fminf(a, b); }
__device__ __forceinline__ double max_(double a, double b) { return a > b ? a : b; }
__device__ __forceinline__ float max_(float a, float b) { return fmaxf(a, b); }
__device__ __forceinline__ bool finite_(double x) { return isfinite(x); }
__device__ __forceinline__ bool finite_(float x) { return isfinite(x); }

// ---- two fp32 values in one register pair: the left and the right state of a face together ------------
// Blackwell issues packed fp32 arithmetic (PTX add/mul/fma.f32x2, SASS FADD2 / FMUL2 / FFMA2) at the flop rate of
// the scalar forms but in half the issue slots, and the fp32 kernel is bound by issue slots (profiles/
// r01_substep.md).  The two states of a face run the same code on different data, so the fp32 face item
// evaluates them as one F2 stream.  Transcendentals, min/max and selects stay per component.
struct F2 {
  float2 v;
  __device__ __forceinline__ F2() {}
  __device__ __forceinline__ F2(float a) { v = make_float2(a, a); }
  __device__ __forceinline__ F2(float a, float b) { v = make_float2(a, b); }
};
__device__ __forceinline__ F2 mk2(float2 x) { F2 r; r.v = x; return r; }
__device__ __forceinline__ F2 operator+(F2 a, F2 b) { return mk2(__fadd2_rn(a.v, b.v)); }
__device__ __forceinline__ F2 operator-(F2 a, F2 b) { return mk2(__fadd2_rn(a.v, make_float2(-b.v.x, -b.v.y))); }
__device__ __forceinline__ F2 operator*(F2 a, F2 b) { return mk2(__fmul2_rn(a.v, b.v)); }
__device__ __forceinline__ F2 operator-(F2 a) { return F2(-a.v.x, -a.v.y); }
__device__ __forceinline__ F2 operator+(float a, F2 b) { return F2(a) + b; }
__device__ __forceinline__ F2 operator+(F2 a, float b) { return a + F2(b); }
__device__ __forceinline__ F2 operator-(float a, F2 b) { return F2(a) - b; }
__device__ __forceinline__ F2 operator-(F2 a, float b) { return a - F2(b); }
__device__ __forceinline__ F2 operator*(float a, F2 b) { return F2(a) * b; }
__device__ __forceinline__ F2 operator*(F2 a, float b) { return a * F2(b); }
__device__ __forceinline__ F2& operator+=(F2& a, F2 b) { a = a + b; return a; }
__device__ __forceinline__ F2 rsqrt_(F2 a) { return F2(rsqrt_(a.v.x), rsqrt_(a.v.y)); }
__device__ __forceinline__ F2 sqrt_(F2 a) { return F2(sqrt_(a.v.x), sqrt_(a.v.y)); }
__device__ __forceinline__ F2 sqrt0_(F2 a) { return sqrt_(a); }
__device__ __forceinline__ F2 rcp_(F2 a) { return F2(rcp_(a.v.x), rcp_(a.v.y)); }
__device__ __forceinline__ F2 div_(F2 a, F2 b) { return a * rcp_(b); }
__device__ __forceinline__ F2 div_(float a, F2 b) { return F2(a) * rcp_(b); }
__device__ __forceinline__ F2 min_(F2 a, F2 b) { return F2(fminf(a.v.x, b.v.x), fminf(a.v.y, b.v.y)); }
__device__ __forceinline__ F2 max_(F2 a, F2 b) { return F2(fmaxf(a.v.x, b.v.x), fmaxf(a.v.y, b.v.y)); }

// Lower an index with the symmetric 3-metric stored as g6 = (xx, xy, xz, yy, yz, zz).
template <typename S, typename T>
__device__ __forceinline__ void lower(const S* g6, const T* a, T* l) {
  l[0] = g6[0] * a[0] + g6[1] * a[1] + g6[2] * a[2];
  l[1] = g6[1] * a[0] + g6[3] * a[1] + g6[4] * a[2];
  l[2] = g6[2] * a[0] + g6[4] * a[1] + g6[5] * a[2];
}
template <typename T>
__device__ __forceinline__ T dot3(const T* a, const T* b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

// Cofactors of the symmetric 3-metric in the same packed order; det by the first column.
template <typename T>
__device__ __forceinline__ T cofactors(const T* g, T* c) {
  c[0] = g[3] * g[5] - g[4] * g[4];
  c[1] = g[4] * g[2] - g[1] * g[5];
  c[2] = g[1] * g[4] - g[3] * g[2];
  c[3] = g[0] * g[5] - g[2] * g[2];
  c[4] = g[1] * g[2] - g[0] * g[4];
  c[5] = g[0] * g[3] - g[1] * g[1];
  return g[0] * c[0] + g[1] * c[1] + g[2] * c[2];
}
// Index of component (k, d) in the packed symmetric order.
__host__ __device__ constexpr int sym(int k, int d) {
  return k == d ? (k == 0 ? 0 : (k == 1 ? 3 : 5)) : (k + d == 1 ? 1 : (k + d == 2 ? 2 : 4));
}
// sqrt(gamma) of a packed 3-metric.
template <typename T>
__device__ __forceinline__ T sqrt_det(const T* g) {
  T c[6];
  return sqrt_(cofactors(g, c));
}

// MC-limited slope (O4): zero at extrema, else the smallest of twice
// each one-sided difference and the centred difference, with the sign of the differences.
template <typename T>
__device__ __forceinline__ T mc_slope(T qm, T q0, T qp) {
  T dm = q0 - qm, dp = qp - q0;
  T s = min_(min_(2 * abs_(dm), 2 * abs_(dp)), abs_(dm + dp) * T(0.5));
  s = dp > 0 ? s : -s;
  return dm * dp <= 0 ? T(0) : s;
}
// fp64: the same function without 64-bit selects (each costs two FSEL after a DSETP).  For differences of
// one sign the minimum is the centred value unless one difference exceeds three times the other, so:
// start from the centred value, overwrite it under a predicate with twice the smaller difference,
// zero it when the sign bits differ (a zero difference already gives zero through the second rule).
template <>
__device__ __forceinline__ double mc_slope<double>(double qm, double q0, double qp) {
  const double dm = q0 - qm, dp = qp - q0;
  double s;
  asm("{\n"
      ".reg .pred p, q, r;\n"
      ".reg .f64 c, am3, ap3, adm, adp;\n"
      ".reg .b32 lo, hm, hp, x;\n"
      "add.f64 c, %1, %2;\n"
      "mul.f64 c, c, 0d3FE0000000000000;\n"
      "abs.f64 adm, %1;\n"
      "abs.f64 adp, %2;\n"
      "mul.f64 am3, adm, 0d4008000000000000;\n"
      "mul.f64 ap3, adp, 0d4008000000000000;\n"
      "setp.gt.f64 p, adp, am3;\n"
      "setp.gt.f64 q, adm, ap3;\n"
      "mov.b64 {lo, hm}, %1;\n"
      "mov.b64 {lo, hp}, %2;\n"
      "xor.b32 x, hm, hp;\n"
      "setp.lt.s32 r, x, 0;\n"
      "mov.f64 %0, c;\n"
      "@p add.f64 %0, %1, %1;\n"
      "@q add.f64 %0, %2, %2;\n"
      "@r mov.f64 %0, 0d0000000000000000;\n"
      "}"
      : "=d"(s)
      : "d"(dm), "d"(dp));
  return s;
}

// Half the MC slope in fp64 with the fewest fp64-pipe instructions (the marching loop forms q -/+ half slope).
// For differences of one sign the limiter returns the centred slope unless one difference exceeds three times the
// other; so: start from a quarter of the sum, overwrite it with the smaller difference when the sign of
// |dp| - 3 |dm| (or |dm| - 3 |dp|), read off the high word of one fused multiply-add, says so, and zero it when the
// sign bits of the two differences differ.  (A test value that is positive but below 2^-1022 counts as not
// positive: the two candidates then agree to that size.)
__device__ __forceinline__ double mc_half_slope(double qm, double q0, double qp) {
  const double dm = q0 - qm, dp = qp - q0;
  double s;
  asm("{\n"
      ".reg .pred p, q, r;\n"
      ".reg .f64 adm, adp, t1, t2;\n"
      ".reg .b32 lo, hm, hp, h1, h2, x;\n"
      "add.f64 %0, %1, %2;\n"
      "mul.f64 %0, %0, 0d3FD0000000000000;\n"
      "abs.f64 adm, %1;\n"
      "abs.f64 adp, %2;\n"
      "fma.rn.f64 t1, adm, 0dC008000000000000, adp;\n"
      "fma.rn.f64 t2, adp, 0dC008000000000000, adm;\n"
      "mov.b64 {lo, h1}, t1;\n"
      "mov.b64 {lo, h2}, t2;\n"
      "setp.gt.s32 p, h1, 0;\n"
      "setp.gt.s32 q, h2, 0;\n"
      "mov.b64 {lo, hm}, %1;\n"
      "mov.b64 {lo, hp}, %2;\n"
      "xor.b32 x, hm, hp;\n"
      "setp.lt.s32 r, x, 0;\n"
      "@p mov.f64 %0, %1;\n"
      "@q mov.f64 %0, %2;\n"
      "@r mov.f64 %0, 0d0000000000000000;\n"
      "}"
      : "=d"(s)
      : "d"(dm), "d"(dp));
  return s;
}
__device__ __forceinline__ float mc_half_slope(float qm, float q0, float qp) { return 0.5f * mc_slope(qm, q0, qp); }

// Two MC slopes at once (fp32): differences and doublings packed; per component three min / max and one sign copy.
// min.xorsign.abs returns min(|a|, |b|) with the sign sign(a) xor sign(b): negative exactly when the two
// differences have opposite signs, so clamping min(that, |centred|) at zero from below IS the "zero at extrema"
// rule, and a zero difference gives zero as well; the sign of the result is that of the differences.
__device__ __forceinline__ float mc_slope_xs(float dm2, float dp2, float c) {
  float m;
  asm("min.xorsign.abs.f32 %0, %1, %2;" : "=f"(m) : "f"(dm2), "f"(dp2));
  return copysignf(fmaxf(fminf(m, fabsf(c)), 0.0f), dp2);
}
__device__ __forceinline__ F2 mc_slope(F2 qm, F2 q0, F2 qp) {
  const F2 dm = q0 - qm, dp = qp - q0;
  const F2 dm2 = dm * 2.0f, dp2 = dp * 2.0f, c = (dm + dp) * 0.5f;
  return F2(mc_slope_xs(dm2.v.x, dp2.v.x, c.v.x), mc_slope_xs(dm2.v.y, dp2.v.y, c.v.y));
}

// PPM (O4b / R5b): Colella-Woodward edge values on a uniform mesh, built on the
// monotonised-central slopes above, made monotone, without contact steepening or flattening.
// Edges of the cell with value q0, from the interface values l, r on its two sides.
template <typename T>
__device__ __forceinline__ void ppm_monotone(T q0, T& l, T& r) {
  if ((r - q0) * (q0 - l) <= 0) {
    l = q0; r = q0;
  } else {
    const T d = r - l, m = q0 - (l + r) * T(0.5);
    if (d * m > d * d * T(1.0 / 6.0)) l = 3 * q0 - 2 * r;
    else if (d * m < -(d * d) * T(1.0 / 6.0)) r = 3 * q0 - 2 * l;
  }
}
// The two states of the face between cells 0 and 1 from the six cells -2 .. 3:
// qL = right edge of cell 0, qR = left edge of cell 1.
template <typename T>
__device__ __forceinline__ void ppm_face(T qm2, T qm1, T q0, T q1, T q2, T q3, T& qL, T& qR) {
  const T dm1 = mc_slope(qm2, qm1, q0), d0 = mc_slope(qm1, q0, q1);
  const T d1 = mc_slope(q0, q1, q2), d2 = mc_slope(q1, q2, q3);
  const T s6 = T(1.0 / 6.0);
  T am = qm1 + (q0 - qm1) * T(0.5) - (d0 - dm1) * s6;   // interface -1/2
  T ac = q0 + (q1 - q0) * T(0.5) - (d1 - d0) * s6;      // interface +1/2: the face
  T ap = q1 + (q2 - q1) * T(0.5) - (d2 - d1) * s6;      // interface +3/2
  T l0 = am, r0 = ac, l1 = ac, r1 = ap;
  ppm_monotone(q0, l0, r0);
  ppm_monotone(q1, l1, r1);
  qL = r0;
  qR = l1;
}

// ---- R1b: the paper's energy variable -------------------------------------------
// -sqrt(-g) T^t_t = sqrt(gamma) [alpha (tau + D) - beta^j S_j]; source-free on a fixed metric.  The two maps
// swap slot 4 of an undensitised (D, S_j, tau, ...) vector -- or, the map being linear, of a coordinate-flux
// vector -- between tau and that variable on the metric m.
template <typename T, typename S>
__device__ __forceinline__ T tau_to_energy(const T* u, const S* m) {
  return m[AL] * (u[4] + u[0]) - (m[BEX] * u[1] + m[BEY] * u[2] + m[BEZ] * u[3]);
}
template <typename T>
__device__ __forceinline__ T energy_to_tau(const T* u, const T* m) {
  return div_(u[4] + (m[BEX] * u[1] + m[BEY] * u[2] + m[BEZ] * u[3]), m[AL]) - u[0];
}

// ---- O1: everything one primitive state defines on a given metric -------------------------------
template <typename T>
struct State {
  T W, iW, v[3], vl[3], v2, rhoh, Bl[3], B2, Bv, b2, pstar;
  T D, S[3], tau;
};

// q = (rho, ut^i, p, B^i, psi); m = met10.  PAPER.md:60 (variables), :74 (w(u) algebraic).
template <typename T>
__device__ __forceinline__ void eval_state(const T* q, const T* m, const Par<T>& par, State<T>& s) {
  T utl[3];
  lower(m + GXX, q + UX, utl);
  T ut2 = dot3(q + UX, utl);
  s.W = sqrt_(1 + ut2);
  s.iW = rcp_(s.W);
#pragma unroll
  for (int i = 0; i < 3; i++) { s.v[i] = q[UX + i] * s.iW; s.vl[i] = utl[i] * s.iW; }
  s.v2 = ut2 * s.iW * s.iW;
  s.rhoh = q[RHO] + par.gg1 * q[PR];
  lower(m + GXX, q + BX, s.Bl);
  s.B2 = dot3(q + BX, s.Bl);
  s.Bv = dot3(q + BX, s.vl);
  s.b2 = s.B2 * s.iW * s.iW + s.Bv * s.Bv;
  s.pstar = q[PR] + s.b2 * T(0.5);
  T Z = s.rhoh * s.W * s.W;
  s.D = q[RHO] * s.W;
#pragma unroll
  for (int j = 0; j < 3; j++) s.S[j] = (Z + s.B2) * s.vl[j] - s.Bv * s.Bl[j];
  s.tau = Z - q[PR] + (s.B2 * (1 + s.v2) - s.Bv * s.Bv) * T(0.5) - s.D;
}

// prim -> undensitised conserved (D, S_j, tau, B^k, psi).
template <typename T>
__device__ __forceinline__ void prim2con(const T* q, const T* m, const Par<T>& par, T* w) {
  State<T> s;
  eval_state(q, m, par, s);
  w[0] = s.D; w[1] = s.S[0]; w[2] = s.S[1]; w[3] = s.S[2]; w[4] = s.tau;
  w[5] = q[BX]; w[6] = q[BY]; w[7] = q[BZ]; w[8] = q[PSI];
}

// ---- O2 + O3: coordinate flux and coordinate signal speeds of one state along D ------------------
// gid[k] = gamma^{kD} of the face metric.  PAPER.md:52-56 (eq. 2 in 3+1 variables), :78.
template <typename T, int D>
__device__ __forceinline__ void flux_speeds(const T* q, const T* m, const T* gid, const Par<T>& par,
                                            T* U, T* F, T& lm, T& lp) {
  State<T> s;
  eval_state(q, m, par, s);
  const T al = m[AL], be = m[BEX + D];
  const T vt = al * s.v[D] - be;  // alpha (v^D - beta^D/alpha)
  const T Bd = q[BX + D];
  U[0] = s.D; U[1] = s.S[0]; U[2] = s.S[1]; U[3] = s.S[2]; U[4] = s.tau;
  U[5] = q[BX]; U[6] = q[BY]; U[7] = q[BZ]; U[8] = q[PSI];
  F[0] = s.D * vt;
  const T aBd = al * Bd * s.iW;
#pragma unroll
  for (int j = 0; j < 3; j++) {
    T bj = s.Bl[j] * s.iW + s.W * s.Bv * s.vl[j];
    F[1 + j] = s.S[j] * vt - bj * aBd;
  }
  F[1 + D] += al * s.pstar;
  F[4] = s.tau * vt + al * s.pstar * s.v[D] - al * s.Bv * Bd;
  if (par.cleaning) {
#pragma unroll
    for (int k = 0; k < 3; k++) F[5 + k] = vt * q[BX + k] - al * s.v[k] * Bd + al * gid[k] * q[PSI];
    F[8] = al * Bd - be * q[PSI];
  } else {
#pragma unroll
    for (int k = 0; k < 3; k++) F[5 + k] = vt * q[BX + k] - (al * s.v[k] - m[BEX + k]) * Bd;
    F[8] = 0;
  }
  // one fast-speed bound through the relativistic addition formula (R7)
  T cs2 = div_(par.Gam * q[PR], s.rhoh);
  T vA2 = div_(s.b2, s.rhoh + s.b2);
  T a2 = cs2 + vA2 - cs2 * vA2;
  a2 = min_(max_(a2, T(0)), T(1));
  T den = 1 - s.v2 * a2;
  T disc = a2 * (1 - s.v2) * (den * gid[D] - (1 - a2) * s.v[D] * s.v[D]);
  T sq = sqrt0_(max_(disc, T(0)));
  T aod = div_(al, den);
  T vd = s.v[D] * (1 - a2);
  lp = aod * (vd + sq) - be;
  lm = aod * (vd - sq) - be;
  if (par.cleaning) {  // light cone of the (B^D, psi) subsystem
    T c = al * sqrt_(gid[D]);
    lp = max_(lp, -be + c);
    lm = min_(lm, -be - c);
  }
}

// ---- O8: primitive recovery, Newton-Raphson on Z = rho h W^2 (R10, R11) -------
template <typename T>
struct C2P { T D, S2, B2, SB, E; };

template <typename T>
__device__ __forceinline__ void c2p_eval(T Z, const C2P<T>& c, const Par<T>& par, T& v2, T& f, T& df) {
  // one reciprocal r = 1/(Z (Z + B^2)) serves 1/Z, 1/(Z + B^2) and their powers; one reciprocal square root
  // serves sqrt(1 - v^2) and D / (2 sqrt(1 - v^2))
  const T ZB = Z + c.B2;
  const T SB2 = c.SB * c.SB;
  const T Z2 = Z * Z;
  const T r = rcp_(Z * ZB);
  const T iZ = ZB * r;
  const T iZ2 = iZ * iZ;
  // (the powers of r are applied one factor at a time: r^3 alone overflows fp32 for Z ~ 1e-7)
  v2 = (c.S2 * Z2 + SB2 * (c.B2 + 2 * Z)) * r * r;
  const T omv = 1 - v2;
  const T rs = rsqrt_(omv);
  const T sq = omv * rs;
  const T p = par.g1g * (Z * omv - c.D * sq);
  f = Z - p + c.B2 * (1 + v2) * T(0.5) - SB2 * T(0.5) * iZ2 - c.E;
  const T dv2 = -2 * (c.S2 * Z2 * Z + SB2 * (3 * Z2 + 3 * Z * c.B2 + c.B2 * c.B2)) * r * r * r;
  df = 1 - par.g1g * omv - par.g1g * (c.D * rs * T(0.5) - Z) * dv2 + c.B2 * dv2 * T(0.5) + SB2 * iZ2 * iZ;
}

// v^2(Z) alone: what the accepted last step still needs (its f and f' would never be used)
template <typename T>
__device__ __forceinline__ T c2p_v2(T Z, const C2P<T>& c) {
  const T r = rcp_(Z * (Z + c.B2));
  return (c.S2 * Z * Z + c.SB * c.SB * (c.B2 + 2 * Z)) * r * r;
}
// fp32 only: the residual f carries a round-off of eps (Z + B^2), so the Newton step cannot shrink below a few
// eps of that scale.  A step that has stopped shrinking while it is below STALL_EPS machine epsilons of the scale
// has found the root to working precision: it is accepted, counted (hz_diag.c2p_stalled) and the iteration ends.
constexpr float C2P_STALL_EPS = 64.0f * 1.1920929e-7f;

// w: undensitised conserved; gi: inverse 3-metric (packed); Zg: guess.  Returns 0 on success, 1 on failure;
// `stalled` is set when the fp32 round-off rule above ended the iteration.
template <typename T>
__device__ __forceinline__ int con2prim_1d(const T* w, const T* m, const T* gi, const Par<T>& par, T Zg, T* q, int& iters,
                                           int& stalled) {
  C2P<T> c;
  T Su[3], Bl[3];
  lower(gi, w + 1, Su);
  lower(m + GXX, w + 5, Bl);
  c.D = w[0];
  c.S2 = dot3(w + 1, Su);
  c.B2 = dot3(w + 5, Bl);
  c.SB = dot3(w + 1, w + 5);
  c.E = w[4] + w[0];
  iters = 0;
  if (!(c.D > 0) || !finite_(c.D) || !finite_(c.S2) || !finite_(c.E) || !finite_(c.B2)) return 1;
  T Z = Zg;
  if (!(Z > 0) || !finite_(Z)) Z = c.E + c.D;
  if (!(Z > 0)) Z = c.D;
  T v2, f, df;
  // move into the region v^2(Z) < 1 (v^2 falls monotonically with Z)
  for (int k = 0; k < 200; k++) {
    c2p_eval(Z, c, par, v2, f, df);
    if (v2 < 1 && finite_(f)) break;
    Z = 2 * Z;
  }
  if (!(v2 < 1)) return 1;
  bool ok = false;
  T dZ = Z, dZprev = Z;
  for (int it = 1; it <= par.c2p_maxit; it++) {
    iters = it;
    T Zn = Z - div_(f, df);
    // fp64: |dZ| <= tol Z (R11).  fp32: the test is made against Z + B^2 (see C2P_STALL_EPS).
    // A step that already meets the tolerance is the last one: only v^2 at the new point is still needed.
    if (finite_(Zn) && Zn > 0 && abs_(Zn - Z) <= par.c2p_tol * (sizeof(T) == 4 ? Zn + c.B2 : Zn)) {
      const T v2n = c2p_v2(Zn, c);
      if (v2n < 1) { Z = Zn; v2 = v2n; ok = true; break; }
    }
    T v2n, fn, dfn;
    int halv = 0;
    for (;;) {  // keep Z > 0 and v^2 < 1 by halving the step
      bool good = finite_(Zn) && Zn > 0;
      if (good) {
        c2p_eval(Zn, c, par, v2n, fn, dfn);
        good = v2n < 1 && finite_(fn) && finite_(dfn);
      }
      if (good) break;
      if (++halv > 40) return 1;
      Zn = (Z + Zn) * T(0.5);
    }
    dZprev = dZ;
    dZ = abs_(Zn - Z);
    Z = Zn; v2 = v2n; f = fn; df = dfn;
    const T scale = sizeof(T) == 4 ? Z + c.B2 : Z;
    if (dZ <= par.c2p_tol * scale) { ok = true; break; }   // (a halved step that lands within the tolerance)
    if (sizeof(T) == 4 && it >= 2 && dZ >= dZprev && dZ <= T(C2P_STALL_EPS) * scale) { ok = true; stalled = 1; break; }
  }
  if (!ok) return 1;
  const T omv = 1 - v2;
  const T sq = sqrt_(omv);
  const T W = rcp_(sq);
  q[RHO] = c.D * sq;
  q[PR] = par.g1g * (Z * omv - c.D * sq);
  const T iZB = rcp_(Z + c.B2);
  const T sbz = div_(c.SB, Z) * iZB;
#pragma unroll
  for (int i = 0; i < 3; i++) {
    q[UX + i] = W * (Su[i] * iZB + sbz * w[5 + i]);
    q[BX + i] = w[5 + i];
  }
  q[PSI] = w[8];
  if (!finite_(q[RHO]) || !finite_(q[PR]) || !finite_(W)) return 1;
  return 0;
}

// ---- O8b: the same root by Newton on the two unknowns (Z, v^2) ("2D_W"; R10b) ----
//   g1 = v2 - V(Z),  g2 = Z - p(Z, v2) + B^2 (1 + v2)/2 - SB^2/(2 Z^2) - E,  Jacobian [[-V', 1], [a, b]]
template <typename T>
__device__ __forceinline__ int con2prim_2d(const T* w, const T* m, const T* gi, const Par<T>& par, T Zg, T* q, int& iters,
                                           int& stalled) {
  C2P<T> c;
  T Su[3], Bl[3];
  lower(gi, w + 1, Su);
  lower(m + GXX, w + 5, Bl);
  c.D = w[0];
  c.S2 = dot3(w + 1, Su);
  c.B2 = dot3(w + 5, Bl);
  c.SB = dot3(w + 1, w + 5);
  c.E = w[4] + w[0];
  iters = 0;
  if (!(c.D > 0) || !finite_(c.D) || !finite_(c.S2) || !finite_(c.E) || !finite_(c.B2)) return 1;
  T Z = Zg;
  if (!(Z > 0) || !finite_(Z)) Z = c.E + c.D;
  if (!(Z > 0)) Z = c.D;
  T v2, f, df;
  for (int k = 0; k < 200; k++) {  // start inside v^2 < 1
    c2p_eval(Z, c, par, v2, f, df);
    if (v2 < 1 && finite_(f)) break;
    Z = 2 * Z;
  }
  if (!(v2 < 1)) return 1;
  const T SB2 = c.SB * c.SB;
  bool ok = false;
  T dZ = Z, dv = 1, dZprev = Z;
  for (int it = 1; it <= par.c2p_maxit; it++) {
    iters = it;
    const T ZB = Z + c.B2, Z2 = Z * Z;
    const T iZ = rcp_(Z), iZB = rcp_(ZB);
    const T iZ2 = iZ * iZ, iZB2 = iZB * iZB;
    const T V = (c.S2 * Z2 + SB2 * (c.B2 + 2 * Z)) * iZ2 * iZB2;
    const T dV = -2 * (c.S2 * Z2 * Z + SB2 * (3 * Z2 + 3 * Z * c.B2 + c.B2 * c.B2)) * (iZ2 * iZ) * (iZB2 * iZB);
    const T omv = 1 - v2, sq = sqrt_(omv);
    const T p = par.g1g * (Z * omv - c.D * sq);
    const T g1 = v2 - V;
    const T g2 = Z - p + c.B2 * (1 + v2) * T(0.5) - SB2 * T(0.5) * iZ2 - c.E;
    const T a = 1 - par.g1g * omv + SB2 * iZ2 * iZ;
    const T b = -par.g1g * (-Z + div_(c.D, 2 * sq)) + c.B2 * T(0.5);
    dZ = div_(-g2 + b * g1, a + b * dV);
    dv = -g1 + dV * dZ;
    // trial point: a linearised v2 outside [0, 1) is put back on the curve v2 = V(Z); a trial that is still
    // unphysical halves the step
    T Zn, vn;
    int halv = 0;
    for (;;) {
      Zn = Z + dZ; vn = v2 + dv;
      bool good = finite_(Zn) && Zn > 0;
      if (good && !(finite_(vn) && vn >= 0 && vn < 1)) {
        const T ZBn = Zn + c.B2;
        vn = div_(c.S2 * Zn * Zn + SB2 * (c.B2 + 2 * Zn), Zn * Zn * ZBn * ZBn);
      }
      good = good && finite_(vn) && vn >= 0 && vn < 1;
      if (good) break;
      if (++halv > 40) return 1;
      dZ = dZ * T(0.5); dv = dv * T(0.5);
    }
    dv = vn - v2;
    Z = Zn; v2 = vn;
    const T scale = sizeof(T) == 4 ? Z + c.B2 : Z;   // fp32: see con2prim_1d
    if (abs_(dZ) <= par.c2p_tol * scale && abs_(dv) <= par.c2p_tol) { ok = true; break; }
    if (sizeof(T) == 4 && it >= 2 && abs_(dZ) >= dZprev && abs_(dZ) <= T(C2P_STALL_EPS) * scale &&
        abs_(dv) <= T(C2P_STALL_EPS)) { ok = true; stalled = 1; break; }
    dZprev = abs_(dZ);
  }
  if (!ok) return 1;
  const T omv = 1 - v2;
  const T sq = sqrt_(omv);
  const T W = rcp_(sq);
  q[RHO] = c.D * sq;
  q[PR] = par.g1g * (Z * omv - c.D * sq);
  const T iZB = rcp_(Z + c.B2);
  const T sbz = div_(c.SB, Z) * iZB;
#pragma unroll
  for (int i = 0; i < 3; i++) {
    q[UX + i] = W * (Su[i] * iZB + sbz * w[5 + i]);
    q[BX + i] = w[5 + i];
  }
  q[PSI] = w[8];
  if (!finite_(q[RHO]) || !finite_(q[PR]) || !finite_(W)) return 1;
  return 0;
}

template <typename T>
__device__ __forceinline__ int con2prim(const T* w, const T* m, const T* gi, const Par<T>& par, T Zg, T* q, int& iters,
                                        int& stalled) {
  if (par.c2p_scheme == 1) return con2prim_2d(w, m, gi, par, Zg, q, iters, stalled);   // uniform over the launch
  return con2prim_1d(w, m, gi, par, Zg, q, iters, stalled);
}

}  // namespace hz
