// hzo.cpp -- CPU ORACLE for the HORIZON per-substep GRMHD update.  TEST INFRASTRUCTURE ONLY
// (see hzo.h).  Plain nested loops, fp64, one function per step of PAPER.md:74-80; OpenMP on
// the outer cell loop only.  No blocking, fusion or reordering.  Shares nothing with the CUDA path.
//
// Each function cites the passage of the paper it follows and the reading (restated
// in DESIGN.md) that supplies the discrete formula the paper does not print.
//
// Pins (tests/test_oracle_*.py) and what stays "parity unpinned": the CFL choice (R13), the floor
// thresholds (R11), the face-metric average (R8) and the centred source stencil (R9) are conventions
// with nothing external to pin them; everything else is pinned as listed in DESIGN.md.  The cleaning rows of
// compute_rhs (flux rows of O2 and the four metric-derivative source terms of O6 / R14) and the ghost fill
// (O9 / R15) are pinned by tests/test_oracle_cleaning.py: convergence to the non-conservative form of the
// equations with spectrally exact derivatives on a space-dependent background, and the padded arrays read back.
#include "hzo.h"

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef HZO_REAL
#define HZO_REAL double
#endif
typedef HZO_REAL real;

// Thin wrappers so an operation-counting scalar type can replace double (flop count).
#ifndef HZO_CUSTOM_REAL
static inline real r_sqrt(real x) { return std::sqrt(x); }
static inline real r_abs(real x) { return std::fabs(x); }
static inline real r_min(real a, real b) { return a < b ? a : b; }
static inline real r_max(real a, real b) { return a > b ? a : b; }
static inline bool r_finite(real x) { return std::isfinite(x); }
static inline double r_val(real x) { return x; }
#endif

namespace {

const int NV = 9;   // rho/D, ut/S (3), p/tau, B (3), psi
const int NM = 10;  // alpha, beta (3), gamma_ij (6)
const int NG = 2;   // ghost layers per active side (MC stencil, reading R16)

struct Met { real al, be[3], g[3][3]; };
struct Geo { real det, sq, gi[3][3]; };  // det gamma, sqrt(gamma), gamma^{ij}
struct Prim { real rho, ut[3], p, B[3], psi; };
struct Cons { real D, S[3], tau, B[3], psi; };

Met load_met(const double* m) {
  Met r;
  r.al = m[0];
  for (int i = 0; i < 3; i++) r.be[i] = m[1 + i];
  r.g[0][0] = m[4]; r.g[0][1] = r.g[1][0] = m[5]; r.g[0][2] = r.g[2][0] = m[6];
  r.g[1][1] = m[7]; r.g[1][2] = r.g[2][1] = m[8]; r.g[2][2] = m[9];
  return r;
}
Prim load_prim(const double* q) {
  Prim r;
  r.rho = q[0]; r.ut[0] = q[1]; r.ut[1] = q[2]; r.ut[2] = q[3]; r.p = q[4];
  r.B[0] = q[5]; r.B[1] = q[6]; r.B[2] = q[7]; r.psi = q[8];
  return r;
}
void store_prim(const Prim& r, double* q) {
  q[0] = r_val(r.rho); q[1] = r_val(r.ut[0]); q[2] = r_val(r.ut[1]); q[3] = r_val(r.ut[2]);
  q[4] = r_val(r.p); q[5] = r_val(r.B[0]); q[6] = r_val(r.B[1]); q[7] = r_val(r.B[2]); q[8] = r_val(r.psi);
}
Cons load_cons(const double* w) {
  Cons r;
  r.D = w[0]; r.S[0] = w[1]; r.S[1] = w[2]; r.S[2] = w[3]; r.tau = w[4];
  r.B[0] = w[5]; r.B[1] = w[6]; r.B[2] = w[7]; r.psi = w[8];
  return r;
}
void store_cons(const Cons& r, double* w) {
  w[0] = r_val(r.D); w[1] = r_val(r.S[0]); w[2] = r_val(r.S[1]); w[3] = r_val(r.S[2]);
  w[4] = r_val(r.tau); w[5] = r_val(r.B[0]); w[6] = r_val(r.B[1]); w[7] = r_val(r.B[2]); w[8] = r_val(r.psi);
}

// det, sqrt(det) and inverse of the spatial 3-metric (plain cofactor formula).
Geo geometry(const Met& m) {
  const real (*g)[3] = m.g;
  Geo r;
  real c00 = g[1][1] * g[2][2] - g[1][2] * g[2][1];
  real c01 = g[1][2] * g[2][0] - g[1][0] * g[2][2];
  real c02 = g[1][0] * g[2][1] - g[1][1] * g[2][0];
  real c11 = g[0][0] * g[2][2] - g[0][2] * g[2][0];
  real c12 = g[0][1] * g[2][0] - g[0][0] * g[2][1];
  real c22 = g[0][0] * g[1][1] - g[0][1] * g[1][0];
  r.det = g[0][0] * c00 + g[0][1] * c01 + g[0][2] * c02;
  r.sq = r_sqrt(r.det);
  r.gi[0][0] = c00 / r.det; r.gi[0][1] = r.gi[1][0] = c01 / r.det; r.gi[0][2] = r.gi[2][0] = c02 / r.det;
  r.gi[1][1] = c11 / r.det; r.gi[1][2] = r.gi[2][1] = c12 / r.det; r.gi[2][2] = c22 / r.det;
  return r;
}

// Quantities every flux / source / wave-speed evaluation needs from one primitive state.
struct Aux {
  real W, v[3], vl[3], v2, h, Bl[3], B2, Bv, b2, pstar, rhoh;
};
Aux aux_of(const Prim& q, const Met& m, real Gam) {
  Aux a;
  real utl[3], ut2 = 0;
  for (int i = 0; i < 3; i++) {
    utl[i] = 0;
    for (int j = 0; j < 3; j++) utl[i] += m.g[i][j] * q.ut[j];
    ut2 += q.ut[i] * utl[i];
  }
  a.W = r_sqrt(1 + ut2);
  for (int i = 0; i < 3; i++) { a.v[i] = q.ut[i] / a.W; a.vl[i] = utl[i] / a.W; }
  a.v2 = ut2 / (a.W * a.W);
  a.h = 1 + Gam / (Gam - 1) * q.p / q.rho;
  a.rhoh = q.rho * a.h;
  a.B2 = 0; a.Bv = 0;
  for (int i = 0; i < 3; i++) {
    a.Bl[i] = 0;
    for (int j = 0; j < 3; j++) a.Bl[i] += m.g[i][j] * q.B[j];
    a.B2 += q.B[i] * a.Bl[i];
    a.Bv += q.B[i] * a.vl[i];
  }
  a.b2 = a.B2 / (a.W * a.W) + a.Bv * a.Bv;
  a.pstar = q.p + a.b2 / 2;
  return a;
}

// O1.  prim -> cons, PAPER.md:74 ("The relation w(u) is algebraic"), variables of PAPER.md:60.
Cons prim2con(const Prim& q, const Met& m, real Gam) {
  Aux a = aux_of(q, m, Gam);
  Cons w;
  real Z = a.rhoh * a.W * a.W;
  w.D = q.rho * a.W;
  for (int j = 0; j < 3; j++) w.S[j] = (Z + a.B2) * a.vl[j] - a.Bv * a.Bl[j];
  w.tau = Z - q.p + (a.B2 * (1 + a.v2) - a.Bv * a.Bv) / 2 - w.D;
  for (int k = 0; k < 3; k++) w.B[k] = q.B[k];
  w.psi = q.psi;
  return w;
}

// O2.  Coordinate flux in direction d: alpha*F^d for D, S_j, tau (eq. 2 in 3+1
// variables) and the cleaning rows for B^k, psi (reading R14).  Not times sqrt(gamma).
// Reading R1b: the paper's own energy variable.  PAPER.md:54, 60 evolves sqrt(-g) T^t_t; with the 3+1
// variables  -sqrt(-g) T^t_t = sqrt(gamma) [ alpha (tau + D) - beta^j S_j ]  (checked in O1).  For a
// time-independent metric its source sqrt(-g) T^kappa_lambda Gamma^lambda_{t kappa} vanishes, so it is
// conserved exactly.  These two maps swap slot 4 of an undensitised (D, S_j, tau, ..) vector (or of a
// flux vector, the map being linear) between tau and that variable, on a given metric.
void tau_to_energy(double* u9, const Met& m) {
  real e = m.al * (real(u9[4]) + real(u9[0]));
  for (int j = 0; j < 3; j++) e = e - m.be[j] * real(u9[1 + j]);
  u9[4] = r_val(e);
}
void energy_to_tau(double* u9, const Met& m) {
  real t = real(u9[4]);
  for (int j = 0; j < 3; j++) t = t + m.be[j] * real(u9[1 + j]);
  u9[4] = r_val(t / m.al - real(u9[0]));
}

void flux_of(int d, const Prim& q, const Met& m, const Geo& geo, real Gam, int cleaning, real* F) {
  Aux a = aux_of(q, m, Gam);
  Cons w = prim2con(q, m, Gam);
  real vt = m.al * a.v[d] - m.be[d];  // alpha*vtilde^d = alpha v^d - beta^d
  real ab0 = a.W * a.Bv;              // alpha b^0
  F[0] = w.D * vt;
  for (int j = 0; j < 3; j++) {
    real bj = a.Bl[j] / a.W + a.W * a.Bv * a.vl[j];
    F[1 + j] = w.S[j] * vt + (j == d ? m.al * a.pstar : real(0)) - m.al * bj * q.B[d] / a.W;
  }
  F[4] = w.tau * vt + m.al * a.pstar * a.v[d] - m.al * ab0 * q.B[d] / a.W;
  if (cleaning) {
    for (int k = 0; k < 3; k++)
      F[5 + k] = vt * q.B[k] - m.al * a.v[k] * q.B[d] + m.al * geo.gi[k][d] * q.psi;
    F[8] = m.al * q.B[d] - m.be[d] * q.psi;
  } else {
    for (int k = 0; k < 3; k++)
      F[5 + k] = vt * q.B[k] - (m.al * a.v[k] - m.be[k]) * q.B[d];
    F[8] = 0;
  }
}

// O3.  "approximate maximal wave speeds", reading R7: one fast-speed bound a^2 put
// through the relativistic velocity addition; coordinate speeds (contain alpha and -beta^d).
void wavespeeds(int d, const Prim& q, const Met& m, const Geo& geo, real Gam, int cleaning,
                real* lm, real* lp) {
  Aux a = aux_of(q, m, Gam);
  real cs2 = Gam * q.p / a.rhoh;
  real vA2 = a.b2 / (a.rhoh + a.b2);
  real a2 = cs2 + vA2 - cs2 * vA2;
  a2 = r_min(r_max(a2, real(0)), real(1));
  real den = 1 - a.v2 * a2;
  real disc = a2 * (1 - a.v2) * (den * geo.gi[d][d] - (1 - a2) * a.v[d] * a.v[d]);
  disc = r_max(disc, real(0));
  real sq = r_sqrt(disc);
  *lp = m.al / den * (a.v[d] * (1 - a2) + sq) - m.be[d];
  *lm = m.al / den * (a.v[d] * (1 - a2) - sq) - m.be[d];
  if (cleaning) {  // light cone of the (B^d, psi) subsystem
    real c = m.al * r_sqrt(geo.gi[d][d]);
    *lp = r_max(*lp, -m.be[d] + c);
    *lm = r_min(*lm, -m.be[d] - c);
  }
}

// O4.  MC-limited slope ("TVD reconstruction with an MC limiter"; reading R6).
real mc_slope(real qm, real q0, real qp) {
  real dm = q0 - qm, dp = qp - q0;
  if (dm * dp <= 0) return 0;
  real s = r_min(r_min(2 * r_abs(dm), 2 * r_abs(dp)), r_abs(dm + dp) / 2);
  return dp > 0 ? s : -s;
}

// O5.  HLLE flux through one face: needs only F(u_L), F(u_R) and the speeds.
// Returns Phi = sqrt(gamma_f) * Fhat.
// O4b.  PPM ("choice between TVD ... MC limiter, and PPM"; reading R5b): the piecewise
// parabolic reconstruction of Colella & Woodward on a uniform mesh, without contact steepening and without
// flattening.  For cell 0 with neighbours q[-2..2] (array q5 = q_{-2}, q_{-1}, q_0, q_1, q_2):
//   slopes     d_i = the monotonised-central slope of O4 at cells -1, 0, 1
//   interfaces a_{i+1/2} = q_i + (q_{i+1} - q_i)/2 - (d_{i+1} - d_i)/6
//   edges      aL = a_{-1/2}, aR = a_{+1/2}, then made monotone:
//              (aR - q0)(q0 - aL) <= 0                      -> aL = aR = q0   (local extremum: flat)
//              (aR - aL)(q0 - (aL + aR)/2) >  (aR - aL)^2/6 -> aL = 3 q0 - 2 aR
//              (aR - aL)(q0 - (aL + aR)/2) < -(aR - aL)^2/6 -> aR = 3 q0 - 2 aL
void ppm_edges(const real* q5, real* aL, real* aR) {
  real dm = mc_slope(q5[0], q5[1], q5[2]);
  real d0 = mc_slope(q5[1], q5[2], q5[3]);
  real dp = mc_slope(q5[2], q5[3], q5[4]);
  real l = q5[1] + (q5[2] - q5[1]) / 2 - (d0 - dm) / 6;
  real r = q5[2] + (q5[3] - q5[2]) / 2 - (dp - d0) / 6;
  real q0 = q5[2];
  if ((r - q0) * (q0 - l) <= 0) {
    l = q0; r = q0;
  } else {
    real d = r - l, m = q0 - (l + r) / 2;
    if (d * m > d * d / 6) l = 3 * q0 - 2 * r;
    else if (d * m < -(d * d) / 6) r = 3 * q0 - 2 * l;
  }
  *aL = l; *aR = r;
}

void hlle(int d, const Prim& qL, const Prim& qR, const Met& mf, real Gam, int cleaning, real* Phi, int energy_var = 0) {
  Geo geo = geometry(mf);
  real FL[NV], FR[NV], lmL, lpL, lmR, lpR;
  flux_of(d, qL, mf, geo, Gam, cleaning, FL);
  flux_of(d, qR, mf, geo, Gam, cleaning, FR);
  wavespeeds(d, qL, mf, geo, Gam, cleaning, &lmL, &lpL);
  wavespeeds(d, qR, mf, geo, Gam, cleaning, &lmR, &lpR);
  double uL[NV], uR[NV];
  store_cons(prim2con(qL, mf, Gam), uL);
  store_cons(prim2con(qR, mf, Gam), uR);
  if (energy_var) {  // R1b: state and flux of the paper's energy variable, with the face metric
    double fl[NV], fr[NV];
    for (int c = 0; c < NV; c++) { fl[c] = r_val(FL[c]); fr[c] = r_val(FR[c]); }
    // flux_of returns coordinate fluxes alpha F; the map is linear, so it applies to them as to the state
    tau_to_energy(uL, mf); tau_to_energy(uR, mf); tau_to_energy(fl, mf); tau_to_energy(fr, mf);
    FL[4] = fl[4]; FR[4] = fr[4];
  }
  real lp = r_max(real(0), r_max(lpL, lpR));
  real lm = r_min(real(0), r_min(lmL, lmR));
  for (int c = 0; c < NV; c++) {
    real f;
    if (lp - lm > 1e-300)
      f = (lp * FL[c] - lm * FR[c] + lp * lm * (real(uR[c]) - real(uL[c]))) / (lp - lm);
    else
      f = (FL[c] + FR[c]) / 2;
    Phi[c] = geo.sq * f;
  }
  if (!cleaning) Phi[8] = 0;
}

// O6 (fluid part).  alpha*sqrt(gamma)*Sigma for S_j and tau: the Gamma term of PAPER.md:54 (eq. 2),
// written as 1/2 T^{mu nu} d_j g_{mu nu}; Sigma(tau) by the stationary-metric identity (reading R9).
// dm[j] holds the derivative along j of (alpha, beta^i, gamma_ik) in a Met.
void fluid_source(const Prim& q, const Met& m, const Met dm[3], real Gam, real* src4) {
  Geo geo = geometry(m);
  Aux a = aux_of(q, m, Gam);
  real al = m.al;
  // four-velocity and magnetic four-vector, contravariant
  real u[4], b[4];
  u[0] = a.W / al;
  b[0] = a.W * a.Bv / al;
  for (int i = 0; i < 3; i++) {
    real vti = a.v[i] - m.be[i] / al;
    u[1 + i] = a.W * vti;
    b[1 + i] = q.B[i] / a.W + a.W * a.Bv * vti;
  }
  // inverse 4-metric
  real gu[4][4];
  gu[0][0] = -1 / (al * al);
  for (int i = 0; i < 3; i++) {
    gu[0][1 + i] = gu[1 + i][0] = m.be[i] / (al * al);
    for (int j = 0; j < 3; j++) gu[1 + i][1 + j] = geo.gi[i][j] - m.be[i] * m.be[j] / (al * al);
  }
  real T[4][4];
  for (int mu = 0; mu < 4; mu++)
    for (int nu = 0; nu < 4; nu++)
      T[mu][nu] = (a.rhoh + a.b2) * u[mu] * u[nu] + a.pstar * gu[mu][nu] - b[mu] * b[nu];
  real bl[3];  // beta_i
  for (int i = 0; i < 3; i++) { bl[i] = 0; for (int k = 0; k < 3; k++) bl[i] += m.g[i][k] * m.be[k]; }
  real T0l[3];     // T^0_i = beta_i T^{00} + gamma_ik T^{0k}
  real Tml[3][3];  // T^i_j = beta_j T^{i0} + gamma_jk T^{ik}
  for (int i = 0; i < 3; i++) {
    T0l[i] = bl[i] * T[0][0];
    for (int k = 0; k < 3; k++) T0l[i] += m.g[i][k] * T[0][1 + k];
  }
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) {
      Tml[i][j] = bl[j] * T[1 + i][0];
      for (int k = 0; k < 3; k++) Tml[i][j] += m.g[j][k] * T[1 + i][1 + k];
    }
  real SigS[3];
  for (int j = 0; j < 3; j++) {
    real bbdg = 0, t0bdg = 0, t0db = 0, tdg = 0;
    for (int k = 0; k < 3; k++)
      for (int l = 0; l < 3; l++) bbdg += m.be[k] * m.be[l] * dm[j].g[k][l];
    for (int i = 0; i < 3; i++)
      for (int k = 0; k < 3; k++) t0bdg += T[0][1 + i] * m.be[k] * dm[j].g[i][k];
    for (int i = 0; i < 3; i++) t0db += T0l[i] * dm[j].be[i];
    for (int i = 0; i < 3; i++)
      for (int k = 0; k < 3; k++) tdg += T[1 + i][1 + k] * dm[j].g[i][k];
    SigS[j] = T[0][0] * (bbdg / 2 - al * dm[j].al) + t0bdg + t0db + tdg / 2;
  }
  real bS = 0, Tdb = 0, T0da = 0;
  for (int j = 0; j < 3; j++) bS += m.be[j] * SigS[j];
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) Tdb += Tml[i][j] * dm[i].be[j];
  for (int i = 0; i < 3; i++) T0da += T[0][1 + i] * dm[i].al;
  real SigTau = (bS + Tdb) / al - T0da;
  real f = al * geo.sq;
  for (int j = 0; j < 3; j++) src4[j] = f * SigS[j];
  src4[3] = f * SigTau;
}

// O8.  con2prim residual f(Z), Z = rho h W^2 (PAPER.md:80 "Newton-Raphson", :128; reading R10).
struct C2PIn { real D, S2, B2, SB, E; };
void c2p_eval(real Z, const C2PIn& c, real Gam, real* v2, real* f, real* df) {
  real ZB = Z + c.B2;
  *v2 = (c.S2 * Z * Z + c.SB * c.SB * (c.B2 + 2 * Z)) / (Z * Z * ZB * ZB);
  real omv = 1 - *v2;
  real sq = r_sqrt(omv);
  real gg = (Gam - 1) / Gam;
  real p = gg * (Z * omv - c.D * sq);
  *f = Z - p + c.B2 * (1 + *v2) / 2 - c.SB * c.SB / (2 * Z * Z) - c.E;
  real dv2 = -2 * (c.S2 * Z * Z * Z + c.SB * c.SB * (3 * Z * Z + 3 * Z * c.B2 + c.B2 * c.B2)) /
             (Z * Z * Z * ZB * ZB * ZB);
  *df = 1 - gg * omv - gg * (-Z + c.D / (2 * sq)) * dv2 + c.B2 * dv2 / 2 + c.SB * c.SB / (Z * Z * Z);
}
C2PIn c2p_input(const Cons& w, const Met& m, const Geo& geo) {
  C2PIn c;
  c.D = w.D;
  c.S2 = 0; c.B2 = 0; c.SB = 0;
  for (int i = 0; i < 3; i++) {
    for (int j = 0; j < 3; j++) {
      c.S2 += geo.gi[i][j] * w.S[i] * w.S[j];
      c.B2 += m.g[i][j] * w.B[i] * w.B[j];
    }
    c.SB += w.S[i] * w.B[i];
  }
  c.E = w.tau + w.D;
  return c;
}
// Newton iteration on Z.  Returns 0 on convergence (prim filled, floors NOT applied), 1 on failure.
int con2prim_2d(const Cons& w, const Met& m, const hzo_params& par, real Zguess, Prim* out, int* iters);
int con2prim(const Cons& w, const Met& m, const hzo_params& par, real Zguess, Prim* out, int* iters) {
  if (par.c2p_scheme == 1) return con2prim_2d(w, m, par, Zguess, out, iters);
  Geo geo = geometry(m);
  C2PIn c = c2p_input(w, m, geo);
  real Gam = par.gamma_ad;
  *iters = 0;
  if (!(w.D > 0) || !r_finite(w.D) || !r_finite(c.S2) || !r_finite(c.E) || !r_finite(c.B2)) return 1;
  real Z = Zguess;
  if (!(Z > 0) || !r_finite(Z)) Z = c.E + c.D;  // built-in guess when none is supplied
  if (!(Z > 0)) Z = c.D;
  real v2, f, df;
  // move into the region v^2(Z) < 1 (v^2 decreases monotonically with Z)
  for (int k = 0; k < 200; k++) {
    c2p_eval(Z, c, Gam, &v2, &f, &df);
    if (v2 < 1 && r_finite(f)) break;
    Z = 2 * Z;
  }
  if (!(v2 < 1)) return 1;
  bool ok = false;
  for (int it = 1; it <= par.c2p_maxit; it++) {
    *iters = it;
    real Zn = Z - f / df;
    real v2n, fn, dfn;
    int halv = 0;
    for (;;) {  // keep Z > 0 and v^2 < 1 by halving the step
      bool good = r_finite(Zn) && Zn > 0;
      if (good) {
        c2p_eval(Zn, c, Gam, &v2n, &fn, &dfn);
        good = v2n < 1 && r_finite(fn) && r_finite(dfn);
      }
      if (good) break;
      if (++halv > 40) return 1;
      Zn = (Z + Zn) / 2;
    }
    real dZ = r_abs(Zn - Z);
    Z = Zn; v2 = v2n; f = fn; df = dfn;
    if (dZ <= par.c2p_tol * Z) { ok = true; break; }
  }
  if (!ok) return 1;
  real omv = 1 - v2;
  real W = 1 / r_sqrt(omv);
  Prim q;
  q.rho = c.D / W;
  q.p = (Gam - 1) / Gam * (Z * omv - c.D * r_sqrt(omv));
  for (int i = 0; i < 3; i++) {
    real Su = 0;
    for (int j = 0; j < 3; j++) Su += geo.gi[i][j] * w.S[j];
    real vi = Su / (Z + c.B2) + c.SB * w.B[i] / (Z * (Z + c.B2));
    q.ut[i] = W * vi;
    q.B[i] = w.B[i];
  }
  q.psi = w.psi;
  if (!r_finite(q.rho) || !r_finite(q.p) || !r_finite(W)) return 1;
  *out = q;
  return 0;
}

// O8b.  The same root by a Newton iteration on TWO unknowns (Z, v^2) -- reading R10b of PAPER.md:128
// ("1D_P or 2D_W methods from Noble et al."): the unknown v^2 is not eliminated but iterated with Z,
//   g1(Z, v2) = v2 - V(Z) = 0,   V(Z) = [S^2 Z^2 + SB^2 (B^2 + 2Z)] / [Z^2 (Z + B^2)^2]
//   g2(Z, v2) = Z - p(Z, v2) + B^2 (1 + v2)/2 - SB^2/(2 Z^2) - E = 0,   p = (G-1)/G [Z (1 - v2) - D sqrt(1 - v2)]
// with the 2x2 Jacobian  [[-V'(Z), 1], [dg2/dZ, dg2/dv2]].  Same root as O8 (it is unique), other iterates.
int con2prim_2d(const Cons& w, const Met& m, const hzo_params& par, real Zguess, Prim* out, int* iters) {
  Geo geo = geometry(m);
  C2PIn c = c2p_input(w, m, geo);
  real Gam = par.gamma_ad, gg = (Gam - 1) / Gam;
  *iters = 0;
  if (!(w.D > 0) || !r_finite(w.D) || !r_finite(c.S2) || !r_finite(c.E) || !r_finite(c.B2)) return 1;
  real Z = Zguess;
  if (!(Z > 0) || !r_finite(Z)) Z = c.E + c.D;
  if (!(Z > 0)) Z = c.D;
  real V, f1d, df1d;
  for (int k = 0; k < 200; k++) {   // start inside v^2 < 1
    c2p_eval(Z, c, Gam, &V, &f1d, &df1d);
    if (V < 1 && r_finite(f1d)) break;
    Z = 2 * Z;
  }
  if (!(V < 1)) return 1;
  real v2 = V;
  bool ok = false;
  for (int it = 1; it <= par.c2p_maxit; it++) {
    *iters = it;
    real ZB = Z + c.B2, SB2 = c.SB * c.SB;
    real Vz = (c.S2 * Z * Z + SB2 * (c.B2 + 2 * Z)) / (Z * Z * ZB * ZB);
    real dV = -2 * (c.S2 * Z * Z * Z + SB2 * (3 * Z * Z + 3 * Z * c.B2 + c.B2 * c.B2)) / (Z * Z * Z * ZB * ZB * ZB);
    real omv = 1 - v2, sq = r_sqrt(omv);
    real p = gg * (Z * omv - c.D * sq);
    real g1 = v2 - Vz;
    real g2 = Z - p + c.B2 * (1 + v2) / 2 - SB2 / (2 * Z * Z) - c.E;
    real a = 1 - gg * omv + SB2 / (Z * Z * Z);                 // dg2/dZ
    real b = -gg * (-Z + c.D / (2 * sq)) + c.B2 / 2;           // dg2/dv2
    real dZ = (-g2 + b * g1) / (a + b * dV);
    real dv = -g1 + dV * dZ;
    // Trial point.  Far from the root the linearised v2 can leave [0, 1) (V is steep at small Z): such a
    // trial is put back on the curve v2 = V(Z); a trial that is still unphysical halves the step.
    real Zn, vn;
    int halv = 0;
    for (;;) {
      Zn = Z + dZ; vn = v2 + dv;
      bool good = r_finite(Zn) && Zn > 0;
      if (good && !(r_finite(vn) && vn >= 0 && vn < 1)) {
        real ZBn = Zn + c.B2;
        vn = (c.S2 * Zn * Zn + SB2 * (c.B2 + 2 * Zn)) / (Zn * Zn * ZBn * ZBn);
      }
      good = good && r_finite(vn) && vn >= 0 && vn < 1;
      if (good) break;
      if (++halv > 40) return 1;
      dZ = dZ / 2; dv = dv / 2;
    }
    dv = vn - v2;
    Z = Zn; v2 = vn;
    if (r_abs(dZ) <= par.c2p_tol * Z && r_abs(dv) <= par.c2p_tol) { ok = true; break; }
  }
  if (!ok) return 1;
  real omv = 1 - v2;
  real W = 1 / r_sqrt(omv);
  Prim q;
  q.rho = c.D / W;
  q.p = gg * (Z * omv - c.D * r_sqrt(omv));
  for (int i = 0; i < 3; i++) {
    real Su = 0;
    for (int j = 0; j < 3; j++) Su += geo.gi[i][j] * w.S[j];
    real vi = Su / (Z + c.B2) + c.SB * w.B[i] / (Z * (Z + c.B2));
    q.ut[i] = W * vi;
    q.B[i] = w.B[i];
  }
  q.psi = w.psi;
  if (!r_finite(q.rho) || !r_finite(q.p) || !r_finite(W)) return 1;
  *out = q;
  return 0;
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// Grid context
// ------------------------------------------------------------------------------------------------
struct hzo_ctx {
  hzo_grid G;
  hzo_params par;
  int n[3], g[3], N[3];   // interior, ghost width, padded extent per axis
  size_t ncell;           // padded cells
  double h[3];
  std::vector<double> met[NM], P[NV], U[NV], U0[NV], R[NV];
  bool have_metric, have_prim;
  int stage;              // next RK stage 0,1,2
  long long c2p_fail, atm_reset, p_floor;
  int c2p_maxit_seen;

  size_t idx(int i, int j, int k) const {
    return ((size_t)(k + g[2]) * N[1] + (j + g[1])) * N[0] + (i + g[0]);
  }
  size_t stride(int d) const { return d == 0 ? 1 : (d == 1 ? (size_t)N[0] : (size_t)N[0] * N[1]); }
  void metric_at(size_t c, double* m10) const { for (int q = 0; q < NM; q++) m10[q] = met[q][c]; }
  void prim_at(size_t c, double* p9) const { for (int q = 0; q < NV; q++) p9[q] = P[q][c]; }
};

namespace {

// O9.  Ghost fill (paper silent; reading R15): periodic wrap or zero-gradient copy, axis by axis so
// edges and corners are filled too.
void fill_ghosts(const hzo_ctx* c, std::vector<double>* F, int nf) {
  for (int d = 0; d < 3; d++) {
    if (c->g[d] == 0) continue;
    int nd = c->n[d];
    for (int f = 0; f < nf; f++) {
      std::vector<double>& a = F[f];
      // loop over the full padded extent of the other two axes (those already filled)
      int lo[3], hi[3];
      for (int e = 0; e < 3; e++) { lo[e] = -c->g[e]; hi[e] = c->n[e] + c->g[e]; }
      lo[d] = 0; hi[d] = 1;
      for (int k = lo[2]; k < hi[2]; k++)
        for (int j = lo[1]; j < hi[1]; j++)
          for (int i = lo[0]; i < hi[0]; i++) {
            int ijk[3] = {i, j, k};
            for (int s = 1; s <= c->g[d]; s++) {
              int src_lo, src_hi;
              if (c->G.bc[d] == HZO_BC_PERIODIC) {
                src_lo = ((-s) % nd + nd) % nd;
                src_hi = (nd - 1 + s) % nd;
              } else {
                src_lo = 0;
                src_hi = nd - 1;
              }
              int a3[3] = {ijk[0], ijk[1], ijk[2]}, b3[3] = {ijk[0], ijk[1], ijk[2]};
              a3[d] = -s; b3[d] = src_lo;
              a[c->idx(a3[0], a3[1], a3[2])] = a[c->idx(b3[0], b3[1], b3[2])];
              a3[d] = nd - 1 + s; b3[d] = src_hi;
              a[c->idx(a3[0], a3[1], a3[2])] = a[c->idx(b3[0], b3[1], b3[2])];
            }
          }
    }
  }
}

Met met_at(const hzo_ctx* c, size_t id) {
  double m10[NM];
  c->metric_at(id, m10);
  return load_met(m10);
}
Prim prim_at(const hzo_ctx* c, size_t id) {
  double p9[NV];
  c->prim_at(id, p9);
  return load_prim(p9);
}

// O4 + O5 for the face between cell `id` and its +d neighbour: MC-reconstructed L/R states of all
// nine primitives, face floors, face metric = arithmetic mean (reading R8), HLLE.
void face_flux(const hzo_ctx* c, int d, size_t id, real* Phi) {
  size_t s = c->stride(d);
  double qL[NV], qR[NV];
  for (int q = 0; q < NV; q++) {
    const double* a = c->P[q].data();
    if (c->par.recon == 1) {  // O4b: right edge of the cell below the face, left edge of the cell above it
      real w5[5], lo, hi;
      for (int t = 0; t < 5; t++) w5[t] = a[id + (size_t)t * s - 2 * s];
      ppm_edges(w5, &lo, &hi);
      qL[q] = r_val(hi);
      for (int t = 0; t < 5; t++) w5[t] = a[id + (size_t)t * s - s];
      ppm_edges(w5, &lo, &hi);
      qR[q] = r_val(lo);
      continue;
    }
    real sl = mc_slope(a[id - s], a[id], a[id + s]);
    real sr = mc_slope(a[id], a[id + s], a[id + 2 * s]);
    qL[q] = r_val(real(a[id]) + sl / 2);
    qR[q] = r_val(real(a[id + s]) - sr / 2);
  }
  Prim L = load_prim(qL), Rr = load_prim(qR);
  L.rho = r_max(L.rho, real(c->par.rho_atm)); L.p = r_max(L.p, real(c->par.p_atm));
  Rr.rho = r_max(Rr.rho, real(c->par.rho_atm)); Rr.p = r_max(Rr.p, real(c->par.p_atm));
  double mf[NM];
  for (int q = 0; q < NM; q++) mf[q] = 0.5 * (c->met[q][id] + c->met[q][id + s]);
  hlle(d, L, Rr, load_met(mf), c->par.gamma_ad, c->par.cleaning, Phi, c->par.energy_var);
}

// O5 (flux difference) + O6 (sources): R = L(U) on interior cells.
void compute_rhs(hzo_ctx* c) {
  const int nx = c->n[0], ny = c->n[1], nz = c->n[2];
  for (int q = 0; q < NV; q++) std::fill(c->R[q].begin(), c->R[q].end(), 0.0);
  // flux differences, one direction after the other; face arrays are plain temporaries
  for (int d = 0; d < 3; d++) {
    if (c->g[d] == 0) continue;  // inactive direction (PAPER.md:126 two-dimensional meshes)
    std::vector<double> Phi[NV];
    for (int q = 0; q < NV; q++) Phi[q].assign(c->ncell, 0.0);
    int lo[3] = {0, 0, 0};
    lo[d] = -1;  // face i+1/2 stored at cell i, i = -1 .. n-1
#pragma omp parallel for schedule(static) collapse(2)
    for (int k = lo[2]; k < nz; k++)
      for (int j = lo[1]; j < ny; j++)
        for (int i = lo[0]; i < nx; i++) {
          size_t id = c->idx(i, j, k);
          real ph[NV];
          face_flux(c, d, id, ph);
          for (int q = 0; q < NV; q++) Phi[q][id] = r_val(ph[q]);
        }
    size_t s = c->stride(d);
#pragma omp parallel for schedule(static) collapse(2)
    for (int k = 0; k < nz; k++)
      for (int j = 0; j < ny; j++)
        for (int i = 0; i < nx; i++) {
          size_t id = c->idx(i, j, k);
          for (int q = 0; q < NV; q++) c->R[q][id] -= (Phi[q][id] - Phi[q][id - s]) / c->h[d];
        }
  }
  // sources
  const int cleaning = c->par.cleaning;
#pragma omp parallel for schedule(static) collapse(2)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t id = c->idx(i, j, k);
        Met m = met_at(c, id);
        Prim q = prim_at(c, id);
        Met dm[3];
        real dQ[3] = {0, 0, 0};  // sum_j d_j(alpha sqrt(gamma) gamma^{kj}), k = 0..2
        real dRb = 0;            // sum_j d_j(sqrt(gamma) beta^j)
        for (int d = 0; d < 3; d++) {
          if (c->g[d] == 0) {
            std::memset(&dm[d], 0, sizeof(Met));
            continue;
          }
          size_t s = c->stride(d);
          Met mp = met_at(c, id + s), mm = met_at(c, id - s);
          real i2h = 1 / (2 * c->h[d]);
          dm[d].al = (mp.al - mm.al) * i2h;
          for (int a = 0; a < 3; a++) {
            dm[d].be[a] = (mp.be[a] - mm.be[a]) * i2h;
            for (int b = 0; b < 3; b++) dm[d].g[a][b] = (mp.g[a][b] - mm.g[a][b]) * i2h;
          }
          if (cleaning) {
            Geo gp = geometry(mp), gm = geometry(mm);
            for (int kk = 0; kk < 3; kk++)
              dQ[kk] += (mp.al * gp.sq * gp.gi[kk][d] - mm.al * gm.sq * gm.gi[kk][d]) * i2h;
            dRb += (gp.sq * mp.be[d] - gm.sq * mm.be[d]) * i2h;
          }
        }
        real src4[4];
        fluid_source(q, m, dm, c->par.gamma_ad, src4);
        if (c->par.energy_var) src4[3] = 0;   // R1b: no source for sqrt(-g) T^t_t on a fixed metric
        for (int a = 0; a < 4; a++) c->R[1 + a][id] += r_val(src4[a]);
        if (cleaning) {  // O6 cleaning sources (reading R14), not multiplied by alpha
          Geo geo = geometry(m);
          for (int kk = 0; kk < 3; kk++) {
            real adv = 0;
            for (int jj = 0; jj < 3; jj++) adv += q.B[jj] * dm[jj].be[kk];
            c->R[5 + kk][id] += r_val(-geo.sq * adv + q.psi * dQ[kk]);
          }
          real Bda = 0;
          for (int jj = 0; jj < 3; jj++) Bda += q.B[jj] * dm[jj].al;
          c->R[8][id] += r_val(geo.sq * Bda - q.psi * dRb - m.al * c->par.kappa * geo.sq * q.psi);
        } else {
          c->R[8][id] = 0;
        }
      }
}

// O8 + floors for every interior cell; U is overwritten where a floor acted (reading R11).
void recover_primitives(hzo_ctx* c) {
  const int nx = c->n[0], ny = c->n[1], nz = c->n[2];
  long long nfail = 0, natm = 0, npfl = 0;
  int itmax = 0;
#pragma omp parallel for schedule(static) collapse(2) reduction(+ : nfail, natm, npfl) reduction(max : itmax)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t id = c->idx(i, j, k);
        Met m = met_at(c, id);
        Geo geo = geometry(m);
        double w9[NV];
        for (int q = 0; q < NV; q++) w9[q] = c->U[q][id] / r_val(geo.sq);
        if (!c->par.cleaning) w9[8] = 0;
        if (c->par.energy_var) energy_to_tau(w9, m);
        Cons w = load_cons(w9);
        Prim old = prim_at(c, id);
        Aux a = aux_of(old, m, c->par.gamma_ad);
        real Zg = a.rhoh * a.W * a.W;  // guess from the previous primitives of this cell
        Prim q;
        int it = 0;
        int fail = con2prim(w, m, c->par, Zg, &q, &it);
        if (it > itmax) itmax = it;
        bool reset = false, pfl = false;
        if (fail) { nfail++; reset = true; }
        else if (q.rho < c->par.rho_atm * (1 + c->par.atm_tol)) reset = true;
        if (reset) {
          natm++;
          q.rho = c->par.rho_atm; q.p = c->par.p_atm;
          for (int a3 = 0; a3 < 3; a3++) { q.ut[a3] = 0; q.B[a3] = w.B[a3]; }
          q.psi = w.psi;
        } else if (q.p < c->par.p_atm) {
          npfl++; pfl = true;
          q.p = c->par.p_atm;
        }
        double p9[NV];
        store_prim(q, p9);
        for (int v = 0; v < NV; v++) c->P[v][id] = p9[v];
        if (reset || pfl) {
          double u9[NV];
          store_cons(prim2con(q, m, c->par.gamma_ad), u9);
          if (c->par.energy_var) tau_to_energy(u9, m);
          for (int v = 0; v < NV; v++) c->U[v][id] = r_val(geo.sq) * u9[v];
        }
      }
  c->c2p_fail += nfail; c->atm_reset += natm; c->p_floor += npfl;
  if (itmax > c->c2p_maxit_seen) c->c2p_maxit_seen = itmax;
}

// O7.  One substep of Shu-Osher SSP-RK3 ("third-order Runge-Kutta"; reading R12).
void substep(hzo_ctx* c, double dt) {
  const int nx = c->n[0], ny = c->n[1], nz = c->n[2];
  compute_rhs(c);
  const int st = c->stage;
  if (st == 0)
    for (int q = 0; q < NV; q++) c->U0[q] = c->U[q];
#pragma omp parallel for schedule(static) collapse(2)
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        size_t id = c->idx(i, j, k);
        for (int q = 0; q < NV; q++) {
          double u1 = c->U[q][id] + dt * c->R[q][id];
          if (st == 0) c->U[q][id] = u1;
          else if (st == 1) c->U[q][id] = 0.75 * c->U0[q][id] + 0.25 * u1;
          else c->U[q][id] = (1.0 / 3.0) * c->U0[q][id] + (2.0 / 3.0) * u1;
        }
      }
  recover_primitives(c);
  fill_ghosts(c, c->P, NV);
  c->stage = (st + 1) % 3;
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// C ABI
// ------------------------------------------------------------------------------------------------
extern "C" {

int hzo_prim2con_point(const double* prim9, const double* met10, double gamma_ad, double* cons9) {
  store_cons(prim2con(load_prim(prim9), load_met(met10), gamma_ad), cons9);
  return 0;
}
int hzo_con2prim_point(const double* cons9, const double* met10, const hzo_params* par, double Zguess,
                       double* prim9, int* iters) {
  Prim q;
  int it = 0;
  int r = con2prim(load_cons(cons9), load_met(met10), *par, Zguess, &q, &it);
  if (iters) *iters = it;
  if (r == 0) store_prim(q, prim9);
  return r;
}
double hzo_c2p_residual_point(double Z, const double* cons9, const double* met10, double gamma_ad) {
  Met m = load_met(met10);
  Geo geo = geometry(m);
  C2PIn c = c2p_input(load_cons(cons9), m, geo);
  real v2, f, df;
  c2p_eval(Z, c, gamma_ad, &v2, &f, &df);
  if (!(v2 < 1)) return NAN;
  return r_val(f);
}
int hzo_flux_point(int d, const double* prim9, const double* met10, double gamma_ad, int cleaning,
                   double* flux9) {
  Met m = load_met(met10);
  real F[NV];
  flux_of(d, load_prim(prim9), m, geometry(m), gamma_ad, cleaning, F);
  for (int q = 0; q < NV; q++) flux9[q] = r_val(F[q]);
  return 0;
}
int hzo_wavespeed_point(int d, const double* prim9, const double* met10, double gamma_ad, int cleaning,
                        double* lam) {
  Met m = load_met(met10);
  real lm, lp;
  wavespeeds(d, load_prim(prim9), m, geometry(m), gamma_ad, cleaning, &lm, &lp);
  lam[0] = r_val(lm); lam[1] = r_val(lp);
  return 0;
}
double hzo_mc_slope(double qm, double q0, double qp) { return r_val(mc_slope(qm, q0, qp)); }
void hzo_ppm_edges(const double* q5, double* aL, double* aR) {
  real w5[5], l, r;
  for (int t = 0; t < 5; t++) w5[t] = q5[t];
  ppm_edges(w5, &l, &r);
  *aL = r_val(l); *aR = r_val(r);
}
int hzo_hlle_point(int d, const double* primL, const double* primR, const double* met10, double gamma_ad,
                   int cleaning, double* phi9) {
  real Phi[NV];
  hlle(d, load_prim(primL), load_prim(primR), load_met(met10), gamma_ad, cleaning, Phi);
  for (int q = 0; q < NV; q++) phi9[q] = r_val(Phi[q]);
  return 0;
}
int hzo_source_point(const double* prim9, const double* met10, const double* dmet30, double gamma_ad,
                     double* src4) {
  Met dm[3];
  for (int j = 0; j < 3; j++) dm[j] = load_met(dmet30 + 10 * j);
  real s[4];
  fluid_source(load_prim(prim9), load_met(met10), dm, gamma_ad, s);
  for (int a = 0; a < 4; a++) src4[a] = r_val(s[a]);
  return 0;
}

int hzo_default_params(hzo_params* p) {
  if (!p) return HZO_EINVAL;
  p->gamma_ad = 4.0 / 3.0;
  p->rho_atm = 1e-12; p->p_atm = 1e-14; p->atm_tol = 1e-3;
  p->cleaning = 1; p->kappa = 1.0;
  p->c2p_maxit = 30; p->c2p_tol = 1e-13; p->c2p_scheme = 0; p->energy_var = 0; p->recon = 0;
  return HZO_OK;
}

int hzo_create(const hzo_grid* G, const hzo_params* par, hzo_ctx** out) {
  if (!G || !out) return HZO_EINVAL;
  if (G->nx < 1 || G->ny < 1 || G->nz < 1 || !(G->dx > 0) || !(G->dy > 0) || !(G->dz > 0)) return HZO_EINVAL;
  const int n3[3] = {G->nx, G->ny, G->nz};
  for (int d = 0; d < 3; d++) {
    if (G->bc[d] != HZO_BC_PERIODIC && G->bc[d] != HZO_BC_OUTFLOW) return HZO_EINVAL;
  }
  hzo_ctx* c = new (std::nothrow) hzo_ctx();
  if (!c) return HZO_ENOMEM;
  c->G = *G;
  if (par) c->par = *par; else hzo_default_params(&c->par);
  if (!(c->par.gamma_ad > 1) || c->par.c2p_maxit < 1) { delete c; return HZO_EINVAL; }
  const int ng = c->par.recon == 1 ? 3 : NG;   // PPM reaches one cell further than MC (reading R16)
  for (int d = 0; d < 3; d++)
    if (n3[d] > 1 && n3[d] < ng) { delete c; return HZO_EINVAL; }
  c->h[0] = G->dx; c->h[1] = G->dy; c->h[2] = G->dz;
  c->ncell = 1;
  for (int d = 0; d < 3; d++) {
    c->n[d] = n3[d];
    c->g[d] = n3[d] > 1 ? ng : 0;
    c->N[d] = c->n[d] + 2 * c->g[d];
    c->ncell *= (size_t)c->N[d];
  }
  try {
    for (int q = 0; q < NM; q++) c->met[q].assign(c->ncell, 0.0);
    for (int q = 0; q < NV; q++) {
      c->P[q].assign(c->ncell, 0.0); c->U[q].assign(c->ncell, 0.0);
      c->U0[q].assign(c->ncell, 0.0); c->R[q].assign(c->ncell, 0.0);
    }
  } catch (...) { delete c; return HZO_ENOMEM; }
  c->have_metric = c->have_prim = false;
  c->stage = 0;
  c->c2p_fail = c->atm_reset = c->p_floor = 0;
  c->c2p_maxit_seen = 0;
  *out = c;
  return HZO_OK;
}
int hzo_destroy(hzo_ctx* c) { delete c; return HZO_OK; }

int hzo_set_metric(hzo_ctx* c, const double* alpha, const double* beta3, const double* gamma6) {
  if (!c || !alpha || !beta3 || !gamma6) return HZO_EINVAL;
  const size_t n = (size_t)c->n[0] * c->n[1] * c->n[2];
  for (int k = 0; k < c->n[2]; k++)
    for (int j = 0; j < c->n[1]; j++)
      for (int i = 0; i < c->n[0]; i++) {
        size_t s = ((size_t)k * c->n[1] + j) * c->n[0] + i, id = c->idx(i, j, k);
        double m10[NM];
        m10[0] = alpha[s];
        for (int a = 0; a < 3; a++) m10[1 + a] = beta3[a * n + s];
        for (int a = 0; a < 6; a++) m10[4 + a] = gamma6[a * n + s];
        Met m = load_met(m10);
        Geo geo = geometry(m);
        bool ok = m.al > 0 && r_finite(m.al) && geo.det > 0 && r_finite(geo.det) && m.g[0][0] > 0 &&
                  m.g[0][0] * m.g[1][1] - m.g[0][1] * m.g[0][1] > 0;
        for (int a = 0; a < NM; a++) ok = ok && std::isfinite(m10[a]);
        if (!ok) return HZO_EINVAL;
        for (int a = 0; a < NM; a++) c->met[a][id] = m10[a];
      }
  fill_ghosts(c, c->met, NM);
  c->have_metric = true;
  c->have_prim = false;
  return HZO_OK;
}

int hzo_set_primitives(hzo_ctx* c, const double* prim8) {
  if (!c || !prim8) return HZO_EINVAL;
  if (!c->have_metric) return HZO_ESTATE;
  const size_t n = (size_t)c->n[0] * c->n[1] * c->n[2];
  for (int k = 0; k < c->n[2]; k++)
    for (int j = 0; j < c->n[1]; j++)
      for (int i = 0; i < c->n[0]; i++) {
        size_t s = ((size_t)k * c->n[1] + j) * c->n[0] + i, id = c->idx(i, j, k);
        Met m = met_at(c, id);
        double a8[8];
        for (int q = 0; q < 8; q++) { a8[q] = prim8[q * n + s]; if (!std::isfinite(a8[q])) return HZO_EINVAL; }
        real v2 = 0;
        for (int a = 0; a < 3; a++) for (int b = 0; b < 3; b++) v2 += m.g[a][b] * a8[1 + a] * a8[1 + b];
        if (!(a8[0] > 0) || a8[4] < 0 || !(v2 < 1)) return HZO_EINVAL;
        real W = 1 / r_sqrt(1 - v2);
        Prim q;
        q.rho = a8[0]; q.p = a8[4]; q.psi = 0;
        for (int a = 0; a < 3; a++) { q.ut[a] = W * a8[1 + a]; q.B[a] = a8[5 + a]; }
        double p9[NV], u9[NV];
        store_prim(q, p9);
        store_cons(prim2con(q, m, c->par.gamma_ad), u9);
        if (c->par.energy_var) tau_to_energy(u9, m);
        real sq = geometry(m).sq;
        for (int v = 0; v < NV; v++) { c->P[v][id] = p9[v]; c->U[v][id] = r_val(sq) * u9[v]; }
      }
  fill_ghosts(c, c->P, NV);
  c->have_prim = true;
  c->stage = 0;
  c->c2p_fail = c->atm_reset = c->p_floor = 0;
  c->c2p_maxit_seen = 0;
  return HZO_OK;
}

int hzo_substeps(hzo_ctx* c, double dt, int nsub) {
  if (!c || nsub < 0 || !(dt > 0)) return HZO_EINVAL;
  if (!c->have_metric || !c->have_prim) return HZO_ESTATE;
  for (int s = 0; s < nsub; s++) substep(c, dt);
  return HZO_OK;
}
int hzo_step(hzo_ctx* c, double dt, int n) {
  if (!c || n < 0) return HZO_EINVAL;
  if (c->stage != 0) return HZO_ESTATE;
  return hzo_substeps(c, dt, 3 * n);
}

int hzo_get_primitives(hzo_ctx* c, double* prim8) {
  if (!c || !prim8) return HZO_EINVAL;
  if (!c->have_prim) return HZO_ESTATE;
  const size_t n = (size_t)c->n[0] * c->n[1] * c->n[2];
  for (int k = 0; k < c->n[2]; k++)
    for (int j = 0; j < c->n[1]; j++)
      for (int i = 0; i < c->n[0]; i++) {
        size_t s = ((size_t)k * c->n[1] + j) * c->n[0] + i, id = c->idx(i, j, k);
        Met m = met_at(c, id);
        Prim q = prim_at(c, id);
        Aux a = aux_of(q, m, c->par.gamma_ad);
        prim8[0 * n + s] = r_val(q.rho);
        for (int d = 0; d < 3; d++) prim8[(1 + d) * n + s] = r_val(a.v[d]);
        prim8[4 * n + s] = r_val(q.p);
        for (int d = 0; d < 3; d++) prim8[(5 + d) * n + s] = r_val(q.B[d]);
      }
  return HZO_OK;
}
int hzo_get_psi(hzo_ctx* c, double* psi) {
  if (!c || !psi) return HZO_EINVAL;
  for (int k = 0; k < c->n[2]; k++)
    for (int j = 0; j < c->n[1]; j++)
      for (int i = 0; i < c->n[0]; i++)
        psi[((size_t)k * c->n[1] + j) * c->n[0] + i] = c->P[8][c->idx(i, j, k)];
  return HZO_OK;
}
static int copy_out(hzo_ctx* c, std::vector<double>* F, double* out9) {
  const size_t n = (size_t)c->n[0] * c->n[1] * c->n[2];
  for (int q = 0; q < NV; q++)
    for (int k = 0; k < c->n[2]; k++)
      for (int j = 0; j < c->n[1]; j++)
        for (int i = 0; i < c->n[0]; i++)
          out9[q * n + ((size_t)k * c->n[1] + j) * c->n[0] + i] = F[q][c->idx(i, j, k)];
  return HZO_OK;
}
int hzo_get_conserved(hzo_ctx* c, double* cons9) {
  if (!c || !cons9) return HZO_EINVAL;
  if (!c->have_prim) return HZO_ESTATE;
  return copy_out(c, c->U, cons9);
}
int hzo_get_rhs(hzo_ctx* c, double* rhs9) {
  if (!c || !rhs9) return HZO_EINVAL;
  if (!c->have_prim) return HZO_ESTATE;
  compute_rhs(c);
  return copy_out(c, c->R, rhs9);
}

// Test accessors (no arithmetic of the method): the cleaning scalar is not part of the API's prim8 (it starts
// at 0), so the pins of the cleaning rows of compute_rhs set a manufactured psi here; and the ghost-fill pins
// read one padded array back.
int hzo_set_psi(hzo_ctx* c, const double* psi) {
  if (!c || !psi) return HZO_EINVAL;
  if (!c->have_prim) return HZO_ESTATE;
  for (int k = 0; k < c->n[2]; k++)
    for (int j = 0; j < c->n[1]; j++)
      for (int i = 0; i < c->n[0]; i++) {
        size_t id = c->idx(i, j, k);
        double v = psi[((size_t)k * c->n[1] + j) * c->n[0] + i];
        if (!std::isfinite(v)) return HZO_EINVAL;
        c->P[8][id] = v;
        c->U[8][id] = r_val(geometry(met_at(c, id)).sq) * v;
      }
  fill_ghosts(c, c->P, NV);
  return HZO_OK;
}
int hzo_padded_extent(const hzo_ctx* c, int* N3, int* g3) {
  if (!c || !N3 || !g3) return HZO_EINVAL;
  for (int d = 0; d < 3; d++) { N3[d] = c->N[d]; g3[d] = c->g[d]; }
  return HZO_OK;
}
int hzo_get_padded(hzo_ctx* c, int which, int field, double* out) {   // which: 0 primitives (9), 1 metric (10)
  if (!c || !out || (which != 0 && which != 1) || field < 0 || field >= (which == 0 ? NV : NM)) return HZO_EINVAL;
  if (which == 0 ? !c->have_prim : !c->have_metric) return HZO_ESTATE;
  const std::vector<double>& a = which == 0 ? c->P[field] : c->met[field];
  for (size_t t = 0; t < c->ncell; t++) out[t] = a[t];
  return HZO_OK;
}

// O10.  Diagnostics (PAPER.md:170-174 global reductions): plain loops, long double accumulation.
int hzo_diagnostics(hzo_ctx* c, hzo_diag* out) {
  if (!c || !out) return HZO_EINVAL;
  if (!c->have_prim) return HZO_ESTATE;
  long double sum[NV] = {0};
  long double l1 = 0;
  double dmax = 0, smax = 0;
  const double dV = c->h[0] * c->h[1] * c->h[2];
  size_t ncells = 0;
  for (int k = 0; k < c->n[2]; k++)
    for (int j = 0; j < c->n[1]; j++)
      for (int i = 0; i < c->n[0]; i++) {
        size_t id = c->idx(i, j, k);
        ncells++;
        for (int q = 0; q < NV; q++) sum[q] += (long double)c->U[q][id];
        Met m = met_at(c, id);
        Geo geo = geometry(m);
        Prim q = prim_at(c, id);
        double div = 0;
        for (int d = 0; d < 3; d++) {
          if (c->g[d] == 0) continue;
          size_t s = c->stride(d);
          double bp = r_val(geometry(met_at(c, id + s)).sq) * c->P[5 + d][id + s];
          double bm = r_val(geometry(met_at(c, id - s)).sq) * c->P[5 + d][id - s];
          div += (bp - bm) / (2 * c->h[d]);
          real lm, lp;
          wavespeeds(d, q, m, geo, c->par.gamma_ad, c->par.cleaning, &lm, &lp);
          double sp = std::fmax(std::fabs(r_val(lm)), std::fabs(r_val(lp))) / c->h[d];
          if (sp > smax) smax = sp;
        }
        div /= r_val(geo.sq);
        if (std::fabs(div) > dmax) dmax = std::fabs(div);
        l1 += std::fabs(div);
      }
  out->sumD = (double)(sum[0] * dV); out->sumSx = (double)(sum[1] * dV); out->sumSy = (double)(sum[2] * dV);
  out->sumSz = (double)(sum[3] * dV); out->sumTau = (double)(sum[4] * dV);
  out->sumBx = (double)(sum[5] * dV); out->sumBy = (double)(sum[6] * dV); out->sumBz = (double)(sum[7] * dV);
  out->sumPsi = (double)(sum[8] * dV);
  out->divB_max = dmax;
  out->divB_L1 = (double)(l1 / (long double)ncells);
  out->max_speed_over_dx = smax;
  out->c2p_fail = c->c2p_fail; out->atm_reset = c->atm_reset; out->p_floor = c->p_floor;
  out->c2p_maxit_seen = c->c2p_maxit_seen;
  return HZO_OK;
}

int hzo_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}
const char* hzo_strerror(int e) {
  switch (e) {
    case HZO_OK: return "ok";
    case HZO_EINVAL: return "invalid argument or unphysical input";
    case HZO_ENOMEM: return "out of memory";
    case HZO_ESTATE: return "call out of order (metric/primitives not set, or mid-step)";
    default: return "unknown error";
  }
}

}  // extern "C"
