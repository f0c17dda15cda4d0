// hz_substep.cuh -- one Runge-Kutta substep as ONE kernel (rows a1-a9 of DESIGN.md section 2).
//
// Blocks are persistent (one per SM) and take tiles of TX x TY x TZ cells in the order of a list (blocks of
// neighbouring tiles, hz_lib.cu: make_tile_order).  Per tile:
//   Stage-in : one thread issues two TMA box loads (cp.async.bulk.tensor.4d): the 9 primitives of the
//              tile with an NG-cell halo (2 for MC, 3 for PPM) and the 10 metric components with a 1-cell
//              halo (16 bytes of halo along x in both, so every box row starts 16-byte aligned) land in
//              shared memory; everyone waits on one mbarrier.  The loads of the NEXT tile are issued as
//              soon as phase 1 is over and fly during phase 2.
//   Phase 1  : work items, one warp each, on a static schedule.  Face items: 32 faces of one
//              direction, every face of the tile exactly once -- reconstruction (MC or PPM), face metric,
//              left/right states, HLLE; the flux Phi goes to shared memory, never to HBM.
//              Source items: the geometric and cleaning sources of 32 cells; they need no
//              flux.  One block barrier ends the phase.
//   Phase 2  : one cell per thread: flux difference of its six faces + sources from shared memory (the flux
//              buffers are released through an mbarrier, waited on before the next tile's phase 1), Runge-
//              Kutta stage, Newton-Raphson recovery with the atmosphere floors,
//              then U and P are written -- P also into the ghost cells that mirror this cell (DESIGN.md
//              O9), so no boundary kernel runs.  P is double-buffered: neighbours still read the old
//              primitives while this block writes the new ones.  In the mixed mode
//              this phase runs in fp64 on fp32 data.
//
// The face flux is written ONCE, for a sweep along axis 0: a sweep along axis d reads the vector and
// metric components cyclically rotated by d (and stores the momentum and field fluxes rotated back).
// The general mode compiles that body once, with d a run-time value -- the unfused kernel, with six
// copies of it, was bound by instruction-cache misses (profiles/r01_naive.md); the fast mode (cleaning on),
// whose body is half the size, is instantiated per axis for the MC reconstruction.
#pragma once
#include <cuda.h>  // CUtensorMap (type only; the encoder is fetched through the runtime, see hz_lib.cu)

#include "hz_kernels.cuh"

namespace hz {

// Tile shape, threads per block (= cells per tile) and x halo of the staged boxes.  TMA wants the first
// element of every box row on a 16-byte boundary, so the x halo is 16 bytes: 2 doubles or 4 floats.
// R = 0: MC-limited linear reconstruction, 2 ghost layers; R = 1: PPM, 3 ghost layers (R5, R5b, R16).
// PPM's wider halo makes the staged boxes bigger, so its tiles are smaller.
// NT may exceed the cells of a tile: the extra warps take work items of phase 1 only.
#ifndef HZ_NT_D0
#define HZ_NT_D0 256
#endif
#ifndef HZ_NT_D1
#define HZ_NT_D1 256
#endif
#ifndef HZ_NT_F1
#define HZ_NT_F1 512
#endif
template <typename T, int R> struct Tile;
template <> struct Tile<double, 0> { static constexpr int TX = 8, TY = 8, TZ = 4, NT = HZ_NT_D0, HX = 2; };
template <> struct Tile<float, 0> { static constexpr int TX = 16, TY = 8, TZ = 4, NT = 512, HX = 4; };
template <> struct Tile<double, 1> { static constexpr int TX = 8, TY = 4, TZ = 4, NT = HZ_NT_D1, HX = 4; };
template <> struct Tile<float, 1> { static constexpr int TX = 8, TY = 8, TZ = 4, NT = HZ_NT_F1, HX = 4; };

template <typename T, int R>
struct TileGeom {
  static constexpr int NG = R == 1 ? 3 : 2;  // ghost layers = halo of the staged primitives
  static constexpr int TX = Tile<T, R>::TX, TY = Tile<T, R>::TY, TZ = Tile<T, R>::TZ, NT = Tile<T, R>::NT, HX = Tile<T, R>::HX;
  static constexpr int NC = TX * TY * TZ;
  static constexpr int NFX = (TX + 1) * TY * TZ, NFY = TX * (TY + 1) * TZ, NFZ = TX * TY * (TZ + 1);
  static constexpr int NF = NFX + NFY + NFZ;
  static constexpr int WX = (NFX + 31) / 32, WY = (NFY + 31) / 32, WZ = (NFZ + 31) / 32;  // warp items per direction
  // (the last item of a direction may be partly empty)
  static_assert(NC <= NT && NT % 32 == 0 && NC % 32 == 0, "phase 2 maps one cell to one thread of the first NC");
  static_assert(TY % 4 == 0, "the row swizzle permutes groups of four rows");
  static_assert(HX >= NG && (HX * sizeof(T)) % 16 == 0, "x halo: at least NG cells and 16-byte box rows starts");
  // staged boxes: primitives with halo 2, metric with halo 1; both with halo HX along x (same x origin)
  static constexpr int BX = TX + 2 * HX, BY = TY + 2 * NG, BZ = TZ + 2 * NG;
  static constexpr int MY = TY + 2, MZ = TZ + 2;
  static constexpr int PFS = BX * BY * BZ;  // field stride of the staged primitives
  static constexpr int MFS = BX * MY * MZ;  // field stride of the staged metric
  static_assert((BX * sizeof(T)) % 16 == 0, "TMA box rows must be multiples of 16 bytes");
  static constexpr size_t align128(size_t x) { return (x + 127) / 128 * 128; }
  static constexpr size_t OFF_P = 0;
  static constexpr size_t OFF_M = align128(OFF_P + (size_t)NV * PFS * sizeof(T));
  static constexpr size_t OFF_F = align128(OFF_M + (size_t)NM * MFS * sizeof(T));
  static constexpr size_t OFF_R = align128(OFF_F + (size_t)NV * NF * sizeof(T));
  static constexpr size_t OFF_BAR = align128(OFF_R + (size_t)(NV - 1) * NC * sizeof(T));  // two mbarriers (8 B each)
  static constexpr size_t SMEM = OFF_BAR + 16;
  static_assert(SMEM <= 227 * 1024, "tile does not fit the 227 KB of shared memory a block may use");
  static constexpr int NFACE_TASKS = WX + WY + WZ, NSRC_TASKS = NC / 32;  // phase-1 work items (one warp each)
  static constexpr unsigned TX_BYTES = (unsigned)((NV * PFS + NM * MFS) * sizeof(T));
};

// FAST = 1 instantiates the kernel for the configuration every BASELINE workload runs -- cleaning on, energy slot
// tau -- with both switches known at compile time; FAST = 0 keeps them run-time (cleaning off, R1b).
template <int FAST, typename P> __device__ __forceinline__ bool cleaning_(const P& par) {
  if constexpr (FAST) return true; else return par.cleaning != 0;
}
template <int FAST, typename P> __device__ __forceinline__ bool evar_(const P& par) {
  if constexpr (FAST) return false; else return par.energy_var != 0;
}

// packed index of gamma_{(d+a)%3, (d+b)%3} for (a,b) = 00 01 02 11 12 22
__device__ __forceinline__ int rot6(int d, int a) {
  // d = 0: 0 1 2 3 4 5;  d = 1: 3 4 1 5 2 0;  d = 2: 5 2 4 0 1 3   (4 bits each)
  const unsigned tab = d == 0 ? 0x543210u : (d == 1 ? 0x025143u : 0x310425u);
  return (int)((tab >> (4 * a)) & 15u);
}
__device__ __forceinline__ int rot3(int d, int a) { const int s = d + a; return s >= 3 ? s - 3 : s; }

// ---- TMA + mbarrier (sm_90+ PTX; SASS: UTMALDG, SYNCS) ---------------------------------------------
__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  unsigned done = 0;
  while (!done) {
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
  }
}
// 4D box (x, y, z, field) of a padded SoA array -> shared memory, completion on `bar`
__device__ __forceinline__ void tma_load_4d(unsigned dst, const CUtensorMap* map, unsigned bar, int c0, int c1, int c2,
                                            int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3)
      : "memory");
}

// ---- O1-O3 for one state in the frame of the sweep (axis 0 = sweep axis) ---------------------------
// q = (rho, ut^0..2, p, B^0..2, psi), m = (alpha, beta^0..2, g00 g01 g02 g11 g12 g22), gi0[k] = gamma^{k0}.
// U: undensitised conserved; F: coordinate flux along axis 0; lm, lp: coordinate signal speeds.
// T is the value type (double, float, or F2 = the left and the right state as one packed fp32 stream),
// S the scalar type of the face metric and the parameters, which both states share.
template <typename T, typename S>
__device__ __forceinline__ void state_flux0(const T* q, const S* m, const S* gi0, const Par<S>& par,
                                            T* U, T* F, T& lm, T& lp) {
  const S* g = m + GXX;
  T utl[3], Bl[3];
  lower(g, q + UX, utl);
  lower(g, q + BX, Bl);
  const T ut2 = dot3(q + UX, utl);
  const T W2 = 1 + ut2;
  const T iW = rsqrt_(W2);
  const T W = W2 * iW;
  const T iW2 = iW * iW;
  const T v2 = ut2 * iW2;
  const T rhoh = q[RHO] + par.gg1 * q[PR];
  const T B2 = dot3(q + BX, Bl);
  const T Bv = dot3(q + BX, utl) * iW;
  const T b2 = B2 * iW2 + Bv * Bv;
  const T pstar = q[PR] + b2 * T(0.5);
  const T Z = rhoh * W2;
  const T D = q[RHO] * W;
  const T ZB = Z + B2;
  const S al = m[AL], be = m[BEX];
  const T v0 = q[UX] * iW;
  const T vt = al * v0 - be;
  const T B0 = q[BX];
  const T aBd = al * B0 * iW;   // alpha B^0 / W
  const T WBv = W * Bv;
  const T ap = al * pstar;
  U[0] = D;
  F[0] = D * vt;
#pragma unroll
  for (int j = 0; j < 3; j++) {
    const T vlj = utl[j] * iW;
    const T Sj = ZB * vlj - Bv * Bl[j];
    const T bj = Bl[j] * iW + WBv * vlj;
    U[1 + j] = Sj;
    F[1 + j] = Sj * vt - bj * aBd;
  }
  F[1] += ap;
  const T tau = Z - q[PR] + (B2 * (1 + v2) - Bv * Bv) * T(0.5) - D;
  U[4] = tau;
  F[4] = tau * vt + ap * v0 - al * Bv * B0;
  const T psi = q[PSI];
#pragma unroll
  for (int k = 0; k < 3; k++) U[5 + k] = q[BX + k];
  U[8] = psi;
  if (par.cleaning) {
    const T apsi = al * psi;
    F[5] = -be * B0 + apsi * gi0[0];
#pragma unroll
    for (int k = 1; k < 3; k++) F[5 + k] = vt * q[BX + k] - al * (q[UX + k] * iW) * B0 + apsi * gi0[k];
    F[8] = al * B0 - be * psi;
  } else {
    F[5] = 0;
#pragma unroll
    for (int k = 1; k < 3; k++) F[5 + k] = vt * q[BX + k] - (al * (q[UX + k] * iW) - m[BEX + k]) * B0;
    F[8] = 0;
  }
  if (par.energy_var) {  // R1b: state and coordinate flux of the paper's energy variable on the face metric
    U[4] = tau_to_energy(U, m);
    F[4] = tau_to_energy(F, m);
  }
  // fast-speed bound a^2 = c_s^2 + v_A^2 - c_s^2 v_A^2 = (Gamma p + b^2)/(rho h + b^2)   (R7)
  T a2 = div_(par.Gam * q[PR] + b2, rhoh + b2);
  a2 = min_(max_(a2, T(0)), T(1));
  const T den = 1 - v2 * a2;
  const T disc = a2 * (1 - v2) * (den * gi0[0] - (1 - a2) * v0 * v0);
  const T sq = sqrt0_(max_(disc, T(0)));
  const T aod = div_(al, den);
  const T vd = v0 * (1 - a2);
  lp = aod * (vd + sq) - be;
  lm = aod * (vd - sq) - be;
}

// ---- the same state in the fast mode (cleaning on, energy slot = tau): its share of the HLLE flux ------
// With cleaning on the signal speeds of a face are the light cone of the (B^d, psi) subsystem: the fluid's
// fast-speed bound of O3 is the coordinate speed of a signal that moves with a <= 1 in the fluid frame, so it
// never leaves that cone, and max / min with it return the cone itself ("light-cone
// speeds").  The HLLE weights then depend on the face metric only, the flux is linear in (U, F) of each
// side with known weights, and each state adds  C = cF F + cU U  without U, F or the fluid speeds ever
// existing as vectors: with k = cF vt + cU every advected row is (row of U) * k plus its pressure / field term.
template <typename T, typename S>
__device__ __forceinline__ void state_contrib0(const T* q, const S* m, const S* gi0, const Par<S>& par, T cF, T cU,
                                               T* C) {
  const S* g = m + GXX;
  T utl[3], Bl[3];
  lower(g, q + UX, utl);
  lower(g, q + BX, Bl);
  const T ut2 = dot3(q + UX, utl);
  const T W2 = 1 + ut2;
  const T iW = rsqrt_(W2);
  const T W = W2 * iW;
  const T iW2 = iW * iW;
  const T v2 = ut2 * iW2;
  const T rhoh = q[RHO] + par.gg1 * q[PR];
  const T B2 = dot3(q + BX, Bl);
  const T Bv = dot3(q + BX, utl) * iW;
  const T Bv2 = Bv * Bv;
  const T b2 = B2 * iW2 + Bv2;
  const T Z = rhoh * W2;
  const T D = q[RHO] * W;
  const T ZB = Z + B2;
  const S al = m[AL], be = m[BEX];
  const T v0 = q[UX] * iW;
  const T k = cF * (al * v0 - be) + cU;
  const T B0 = q[BX];
  const T aBd = al * B0 * iW;   // alpha B^0 / W
  const T cFa = cF * aBd;
  const T WBv = W * Bv;
  const T cap = cF * (al * (q[PR] + b2 * T(0.5)));   // cF alpha p*
  C[0] = D * k;
#pragma unroll
  for (int j = 0; j < 3; j++) {
    const T vlj = utl[j] * iW;
    const T Sj = ZB * vlj - Bv * Bl[j];
    const T bj = Bl[j] * iW + WBv * vlj;
    C[1 + j] = Sj * k - cFa * bj;
  }
  C[1] = C[1] + cap;
  const T tau = Z - q[PR] + (B2 * (1 + v2) - Bv2) * T(0.5) - D;
  C[4] = tau * k + cap * v0 - cFa * WBv;   // alpha Bv B^0 = (alpha B^0 / W) (W Bv)
  const T psi = q[PSI];
  const T capsi = cF * (al * psi);
  C[5] = capsi * gi0[0] + (cU - cF * be) * B0;
#pragma unroll
  for (int c = 1; c < 3; c++) C[5 + c] = q[BX + c] * k + capsi * gi0[c] - cFa * q[UX + c];
  C[8] = cF * (al * B0 - be * psi) + cU * psi;
}

// ---- a1-a4 for one face of a sweep along axis d, everything read from the staged tile ---------------
// sPc / sMc: staged primitives / metric at the cell on the MINUS side of the face (field 0);
// sp / sm: element stride of axis d inside the two boxes.
// Phi comes out in the sweep frame: Phi[1+a] belongs to S_{(d+a)%3}, Phi[5+a] to B^{(d+a)%3}.
template <typename T, int R, int FAST>
__device__ __forceinline__ void face_flux_rot(const T* __restrict__ sPc, const T* __restrict__ sMc, int sp, int sm,
                                              int d, const Par<T>& par, T* Phi) {
  using G = TileGeom<T, R>;
  // face metric: mean of the two cells (R8), components rotated into the sweep frame
  T mf[NM];
  mf[AL] = T(0.5) * (sMc[0] + sMc[sm]);
#pragma unroll
  for (int c = 0; c < 3; c++) {
    const T* b = sMc + (BEX + rot3(d, c)) * G::MFS;
    mf[BEX + c] = T(0.5) * (b[0] + b[sm]);
  }
#pragma unroll
  for (int c = 0; c < 6; c++) {
    const T* b = sMc + (GXX + rot6(d, c)) * G::MFS;
    mf[GXX + c] = T(0.5) * (b[0] + b[sm]);
  }
  const T* g = mf + GXX;
  // first column of the cofactor matrix, determinant, gamma^{k0}
  const T c0 = g[3] * g[5] - g[4] * g[4];
  const T c1 = g[4] * g[2] - g[1] * g[5];
  const T c2 = g[1] * g[4] - g[3] * g[2];
  const T det = g[0] * c0 + g[1] * c1 + g[2] * c2;
  const T idet = rcp_(det);
  const T sqg = sqrt_(det);
  const T gi0[3] = {c0 * idet, c1 * idet, c2 * idet};
  // MC reconstruction (O4) of the 9 primitives, rotated
  T qL[NV], qR[NV];
#pragma unroll
  for (int q = 0; q < NV; q++) {
    const int f = (q >= UX && q <= UZ) ? UX + rot3(d, q - UX) : ((q >= BX && q <= BZ) ? BX + rot3(d, q - BX) : q);
    const T* a = sPc + f * G::PFS;
    if (R == 1) {  // PPM (O4b): right edge of the cell below the face, left edge of the cell above it
      ppm_face(a[-2 * sp], a[-sp], a[0], a[sp], a[2 * sp], a[3 * sp], qL[q], qR[q]);
    } else {
      const T qm = a[-sp], q0 = a[0], q1 = a[sp], q2 = a[2 * sp];
      if constexpr (sizeof(T) == 4) {  // fp32: the slopes of the two cells as one packed pair
        const F2 e = F2(q0, q1) + F2(0.5f, -0.5f) * mc_slope(F2(qm, q0), F2(q0, q1), F2(q1, q2));
        qL[q] = e.v.x;
        qR[q] = e.v.y;
      } else {
        qL[q] = q0 + mc_half_slope(qm, q0, q1);
        qR[q] = q1 - mc_half_slope(q0, q1, q2);
      }
    }
  }
  qL[RHO] = max_(qL[RHO], par.rho_atm); qL[PR] = max_(qL[PR], par.p_atm);
  qR[RHO] = max_(qR[RHO], par.rho_atm); qR[PR] = max_(qR[PR], par.p_atm);
  if constexpr (FAST) {
    // cleaning on: the light cone bounds every signal, so the HLLE weights are functions of the face metric
    const T c = mf[AL] * sqrt_(gi0[0]);
    const T lp = max_(c - mf[BEX], T(0)), lm = min_(-c - mf[BEX], T(0));
    const T sw = div_(sqg, lp - lm);           // lp - lm >= 2 c > 0
    const T cFL = sw * lp, cFR = -(sw * lm), cUU = sw * lp * lm;
    if constexpr (sizeof(T) == 4) {  // fp32: both states as one packed stream
      F2 q2[NV], C2[NV];
#pragma unroll
      for (int v = 0; v < NV; v++) q2[v] = F2(qL[v], qR[v]);
      state_contrib0(q2, mf, gi0, par, F2(cFL, cFR), F2(-cUU, cUU), C2);
#pragma unroll
      for (int v = 0; v < NV; v++) Phi[v] = C2[v].v.x + C2[v].v.y;
    } else {
      T CR[NV];
      state_contrib0(qL, mf, gi0, par, cFL, -cUU, Phi);
      state_contrib0(qR, mf, gi0, par, cFR, cUU, CR);
#pragma unroll
      for (int v = 0; v < NV; v++) Phi[v] += CR[v];
    }
    return;
  }
  T UL[NV], FL[NV], UR[NV], FR[NV], lmL, lpL, lmR, lpR;
  if constexpr (sizeof(T) == 4) {  // fp32: both states as one packed stream (F2, hz_physics.cuh)
    F2 q2[NV], U2[NV], Fx2[NV], lm2, lp2;
#pragma unroll
    for (int v = 0; v < NV; v++) q2[v] = F2(qL[v], qR[v]);
    state_flux0(q2, mf, gi0, par, U2, Fx2, lm2, lp2);
#pragma unroll
    for (int v = 0; v < NV; v++) { UL[v] = U2[v].v.x; UR[v] = U2[v].v.y; FL[v] = Fx2[v].v.x; FR[v] = Fx2[v].v.y; }
    lmL = lm2.v.x; lmR = lm2.v.y; lpL = lp2.v.x; lpR = lp2.v.y;
  } else {
    state_flux0(qL, mf, gi0, par, UL, FL, lmL, lpL);
    state_flux0(qR, mf, gi0, par, UR, FR, lmR, lpR);
  }
  T lp = max_(lpL, lpR), lm = min_(lmL, lmR);
  if (par.cleaning) {  // light cone of the (B^d, psi) subsystem (O3)
    const T c = mf[AL] * sqrt_(gi0[0]);
    lp = max_(lp, c - mf[BEX]);
    lm = min_(lm, -c - mf[BEX]);
  }
  lp = max_(lp, T(0));
  lm = min_(lm, T(0));
  const T w = lp - lm;
  if (w > T(1e-30)) {
    const T sw = div_(sqg, w), ll = lp * lm;
#pragma unroll
    for (int q = 0; q < NV; q++) Phi[q] = sw * (lp * FL[q] - lm * FR[q] + ll * (UR[q] - UL[q]));
  } else {
#pragma unroll
    for (int q = 0; q < NV; q++) Phi[q] = sqg * T(0.5) * (FL[q] + FR[q]);
  }
  if (!par.cleaning) Phi[8] = 0;
}

// ---- a6 at one cell: geometric and cleaning sources in the 3+1 form of the stress-energy contraction,
// accumulated ONE AXIS AT A TIME.  With A^{ik} = (rho h + b^2) ut^i ut^k + p* gamma^{ik} - Bt^i Bt^k
// (ut^i = W v^i the stored primitive, Bt^i = B^i / W + (B.v) ut^i), S_i, S^i the momentum density and
// E = tau + D, the contraction (1/2) T^{mu nu} d_j g_{mu nu} and the stationary-metric identity of O6 become
//   alpha Sigma(S_j) = alpha (1/2) A^{ik} d_j gamma_ik + S_i d_j beta^i - E d_j alpha
//   alpha Sigma(tau) = beta^j (1/2) A^{ik} d_j gamma_ik + A^{jl} gamma_lk d_j beta^k - S^j d_j alpha
// (T^{00} beta^i beta^k + 2 T^{0(i} beta^{k)} + T^{ik} = A^{ik}, alpha T^0_i = S_i, alpha^2 T^{00} = E: the same
// numbers as the T^{mu nu} d_j g_{mu nu} contraction up to rounding, with half the arithmetic and no division by the lapse).  Every term is
// a sum over the axis of differentiation, so the ten metric differences of one axis are formed, used and dropped
// before the next axis is touched.
// sPc / sMc: staged primitives / metric at the cell; sRc: its slot in sR; clc: its entry of the static cleaning
// coefficients of k_clean_static (field stride fs); gmask: bit j set = axis j active.
template <typename T, int R, int FAST>
__device__ __forceinline__ void source_cell(const T* __restrict__ sPc, const T* __restrict__ sMc, T* __restrict__ sRc,
                                           const T* __restrict__ clc, long long fs, int gmask, T gg1, T kappa, T ih0, T ih1,
                                           T ih2, int cleaning, int evar) {
  using G = TileGeom<T, R>;
  T q[NV], m[NM];
#pragma unroll
  for (int v = 0; v < NV; v++) q[v] = sPc[v * G::PFS];
#pragma unroll
  for (int v = 0; v < NM; v++) m[v] = sMc[v * G::MFS];
  const T* g = m + GXX;
  T cf[6];
  const T det = cofactors(g, cf);
  const T sq = sqrt_(det);
  const T idet = rcp_(det);
  // O1 at the cell
  T utl[3], Bl[3];
  lower(g, q + UX, utl);
  lower(g, q + BX, Bl);
  const T ut2 = dot3(q + UX, utl);
  const T W2 = 1 + ut2;
  const T iW = rsqrt_(W2);
  const T iW2 = iW * iW;
  const T rhoh = q[RHO] + gg1 * q[PR];
  const T B2 = dot3(q + BX, Bl);
  const T Bv = dot3(q + BX, utl) * iW;         // B.v
  const T b2 = B2 * iW2 + Bv * Bv;
  const T pstar = q[PR] + b2 * T(0.5);
  const T hb = rhoh + b2;
  const T Z = rhoh * W2;
  const T ZB = (Z + B2) * iW;                  // (Z + B^2) / W : S = ZB ut - Bv B with either index position
  const T E = Z - q[PR] + (B2 * (1 + ut2 * iW2) - Bv * Bv) * T(0.5);   // tau + D
  T Bt[3], Sl[3], Su[3];
#pragma unroll
  for (int i = 0; i < 3; i++) {
    Bt[i] = q[BX + i] * iW + Bv * q[UX + i];
    Sl[i] = ZB * utl[i] - Bv * Bl[i];
    Su[i] = ZB * q[UX + i] - Bv * q[BX + i];
  }
  const T pg = pstar * idet;                   // p* gamma^{ik} = p* cof_ik / det
  T A[6];                                      // packed (xx xy xz yy yz zz)
#pragma unroll
  for (int i = 0; i < 3; i++)
#pragma unroll
    for (int k = i; k < 3; k++) A[sym(i, k)] = hb * q[UX + i] * q[UX + k] + pg * cf[sym(i, k)] - Bt[i] * Bt[k];
  const T al = m[AL];
  const T* be = m + BEX;
  T Rs[NV];
  T sT = 0, adv[3] = {0, 0, 0}, Bda = 0;
  Rs[1] = Rs[2] = Rs[3] = 0;
#pragma unroll
  for (int j = 0; j < 3; j++) {
    if (((gmask >> j) & 1) == 0) continue;
    asm volatile("" ::: "memory");   // one axis at a time: keeps the staged loads of the next axis behind this one
    const int st = j == 0 ? 1 : (j == 1 ? G::BX : G::BX * G::MY);
    const T h = T(0.5) * (j == 0 ? ih0 : (j == 1 ? ih1 : ih2));
    T d[NM];   // twice the centred difference times the spacing: the factor h = 1 / (2 dx) is applied to the sums
#pragma unroll
    for (int v = 0; v < NM; v++) d[v] = sMc[v * G::MFS + st] - sMc[v * G::MFS - st];
    const T* dg = d + GXX;
    const T Gj = T(0.5) * (A[0] * dg[0] + A[3] * dg[3] + A[5] * dg[5]) + A[1] * dg[1] + A[2] * dg[2] + A[4] * dg[4];
    Rs[1 + j] = (sq * h) * (al * Gj + dot3(Sl, d + BEX) - E * d[AL]);
    // row j of A lowered with gamma: A^{jl} gamma_lk
    const T row[3] = {A[sym(j, 0)], A[sym(j, 1)], A[sym(j, 2)]};
    T rl[3];
    lower(g, row, rl);
    sT += h * (be[j] * Gj + dot3(rl, d + BEX) - Su[j] * d[AL]);
    const T Bh = q[BX + j] * h;
#pragma unroll
    for (int k = 0; k < 3; k++) adv[k] += Bh * d[BEX + k];
    Bda += Bh * d[AL];
  }
  Rs[4] = sq * sT;
  // cleaning sources (R14), not multiplied by alpha; clc: the static coefficients of k_clean_static
  if (FAST || cleaning) {
    const T psi = q[PSI];
#pragma unroll
    for (int k = 0; k < 3; k++) Rs[5 + k] = -sq * adv[k] + psi * clc[k * fs];
    Rs[8] = sq * Bda - psi * clc[3 * fs] - m[AL] * kappa * sq * psi;
  } else {
    Rs[5] = Rs[6] = Rs[7] = Rs[8] = 0;
  }
  if (!FAST && evar) Rs[4] = 0;  // R1b: no source on a fixed metric
#pragma unroll
  for (int v = 1; v < NV; v++) sRc[(v - 1) * G::NC] = Rs[v];
}
// ---- a9 fused: store the primitives of cell (i,j,k) and of every ghost cell that mirrors it --------
// Ghost images of interior coordinate c along axis d (O9): periodic -- c + n if c < ng, c - n if
// c >= n - ng; zero gradient -- the edge cell fills the ng layers beyond it; external sides get none.
__device__ __forceinline__ int image_count(const Layout& L, int d, int c) {
  if (L.g[d] == 0) return 0;
  const int n = L.n[d];
  if (L.bc[d] == 0) return (c < L.ng) + (c >= n - L.ng);
  if (c == 0 && bc_side(L.bc[d], 0) == 1) return L.ng;
  if (c == n - 1 && bc_side(L.bc[d], 1) == 1) return L.ng;
  return 0;
}
// t = 0 is the cell itself, t = 1 .. image_count its images
__device__ __forceinline__ int image_coord(const Layout& L, int d, int c, int t) {
  if (t == 0) return c;
  const int n = L.n[d];
  if (L.bc[d] == 0) return (t == 1 && c < L.ng) ? c + n : c - n;
  return c == 0 ? -t : n - 1 + t;
}
// ---- halo exchange fused into the substep ("peer stores") ----------
// A slab whose neighbour's primitive buffers are mapped into this process (another context on this GPU, a peer
// GPU of this process, or a CUDA-IPC mapping of another process's buffer; hz_peer_attach) stores the cells within
// NG of that cut -- and their x / y ghost images -- straight into the neighbour's ghost planes while it writes its
// own: no pack kernel, no transfer, no unpack kernel.  dst[s]: the neighbour's primitive set that this substep
// writes (side s: 0 below, 1 above), 0 = no neighbour mapped; fs[s]: its field stride; nz0: interior planes of the
// neighbour below.  The two slabs have the same extent in x and y, hence the same row and plane strides.
template <typename T, int PEER> struct PeerArg {};
template <typename T> struct PeerArg<T, 1> { T* dst[2]; long long fs[2]; int nz0; };

template <typename T, int PEER = 0>
__device__ __forceinline__ void store_prims_with_images(const Layout& L, T* __restrict__ Pout, int i, int j, int k,
                                                        const T* q, const PeerArg<T, PEER>& peer = PeerArg<T, PEER>()) {
  const long long id0 = L.idx(i, j, k);
#pragma unroll
  for (int v = 0; v < NV; v++) Pout[v * L.fs + id0] = q[v];
  const int ci = image_count(L, 0, i), cj = image_count(L, 1, j), ck = image_count(L, 2, k);
  if constexpr (PEER) {
#pragma unroll   // (static index into the kernel parameter: a run-time one would copy it to local memory)
    for (int s = 0; s < 2; s++) {
      if (peer.dst[s] == nullptr || !(s == 0 ? k < L.ng : k >= L.n[2] - L.ng)) continue;
      const int kp = s == 0 ? peer.nz0 + k : k - L.n[2];   // this plane in the neighbour's coordinates: a ghost plane
      for (int b = 0; b <= cj; b++)
        for (int a = 0; a <= ci; a++) {
          const long long id = (long long)(kp + L.g[2]) * L.sz + (long long)(image_coord(L, 1, j, b) + L.g[1]) * L.pitch +
                               (image_coord(L, 0, i, a) + L.ox);
#pragma unroll
          for (int v = 0; v < NV; v++) peer.dst[s][v * peer.fs[s] + id] = q[v];
        }
    }
  }
  if ((ci | cj | ck) == 0) return;   // not within reach of a boundary: the common case
  for (int c = 0; c <= ck; c++)
    for (int b = 0; b <= cj; b++)
      for (int a = 0; a <= ci; a++) {
        if ((a | b | c) == 0) continue;
        const long long id = L.idx(image_coord(L, 0, i, a), image_coord(L, 1, j, b), image_coord(L, 2, k, c));
#pragma unroll
        for (int v = 0; v < NV; v++) Pout[v * L.fs + id] = q[v];
      }
}

// Row swizzle against shared-memory bank conflicts.  A warp item covers rows of TX cells; staged box rows
// are BX = TX + 2 HX elements = 24 words apart, so rows b and b+1 read by one half-warp (fp64) or one
// warp (fp32) overlap in 8 banks, while rows b and b+2 (48 words apart) do not.  Lanes that would take
// rows (0,1,2,3) of a group of four take rows (0,2,1,3) instead: bits 0 and 1 of the row index swap.
__device__ __forceinline__ int swz(int b) { return (b & ~3) | ((b & 1) << 1) | ((b >> 1) & 1); }

// n / N for 0 <= n < NMAX and a compile-time N: shift or multiply-shift, never a division
template <int N, int NMAX>
__device__ __forceinline__ int cdiv(int n) {
  if ((N & (N - 1)) == 0) {
    int sh = 0;
    while ((1 << sh) < N) sh++;
    return n >> sh;
  }
  constexpr unsigned M = 65536 / N + 1;
  static_assert((long long)NMAX * ((long long)M * N - 65536) < 65536 && (long long)NMAX * M < (1ll << 32),
                "cdiv: multiply-shift not exact on this range");
  return (int)(((unsigned)n * M) >> 16);
}

// ---- the work items of phase 1 ----------------------------------------------------------------------
// Face item: 32 consecutive faces of one direction -> Phi into sF.
#ifndef HZ_FACE_ORDER
#define HZ_FACE_ORDER 1
#endif
#ifndef HZ_AXIS_COPIES_R
#define HZ_AXIS_COPIES_R 0   // per-axis copies for the MC body only (the PPM body is twice the size)
#endif
template <typename T, int R, int FAST, int DD = -1>
__device__ __forceinline__ void face_task(const Layout& L, const Par<T>& par, const T* sP, const T* sM, T* sF, int task,
                                          int lane, int x0, int y0, int z0) {
  using G = TileGeom<T, R>;
  if constexpr (DD < 0 && FAST && R == HZ_AXIS_COPIES_R) {
    // One copy of the face item per sweep axis where the body is small (the fast mode): the rotated component and
    // stride selections become immediates (fp32 +10 %, fp64 +1 %).  The general mode keeps ONE copy with a
    // run-time axis: its body is twice the size, and three of it overflow the instruction cache
    // (profiles/r01_naive.md).
    const int dd = (task >= G::WX) + (task >= G::WX + G::WY);
    if (dd == 0) face_task<T, R, FAST, 0>(L, par, sP, sM, sF, task, lane, x0, y0, z0);
    else if (dd == 1) face_task<T, R, FAST, 1>(L, par, sP, sM, sF, task, lane, x0, y0, z0);
    else face_task<T, R, FAST, 2>(L, par, sP, sM, sF, task, lane, x0, y0, z0);
    return;
  }
  int d = DD >= 0 ? DD : (task >= G::WX) + (task >= G::WX + G::WY);
  // general mode: hide the value of d so the compiler does not clone the body per axis
  if constexpr (DD < 0) asm volatile("" : "+r"(d));
  const int off = d == 0 ? 0 : (d == 1 ? G::NFX : G::NFX + G::NFY);                 // first face of d in sF
  const int f = (task - (d == 0 ? 0 : (d == 1 ? G::WX : G::WX + G::WY))) * 32 + lane;  // face number within d
  // (no L.g[d]: indexing a kernel parameter with a run-time d makes the compiler copy it to local memory)
  if ((d == 0 ? L.g[0] : (d == 1 ? L.g[1] : L.g[2])) == 0) return;
  if (f >= (d == 0 ? G::NFX : (d == 1 ? G::NFY : G::NFZ))) return;                     // partly empty last item
  // face coordinates inside the tile: f = (c * e1 + b) * e0 + a with e0 = TX (+1 for x faces),
  // e1 = TY (+1 for y faces); the quotients by multiply-shift (d is a run-time value here)
  const int e0 = G::TX + (d == 0), e1 = G::TY + (d == 1);
  // Which face a lane takes.  MC tiles: the faces of a direction are numbered so that a warp item is whole rows of TX
  // faces and a (half-)warp takes rows b, b + 2 of ONE plane (swz below): the faces with a < TX and b < TY first, as
  // the cells are (f < NC), then the TY * TZ x faces with a = TX or the TX * TZ y faces with b = TY.  (Numbered along
  // rows of TX + 1 x faces or planes of TY + 1 y rows, the rows drifted against the half-warps: the x and y items
  // took 1.76 shared-memory wavefronts per ideal one.)  The PPM tiles keep the plain numbering: their fp32 box rows
  // are 16 words, and an item of a = TX faces alone would hit two banks (measured: -6 %).
  int a, b0, c;
  if (HZ_FACE_ORDER && R == 0) {
    if (d == 2 || f < G::NC) {
      const int r = cdiv<G::TX, G::NF>(f);
      a = f - r * G::TX;
      c = cdiv<G::TY, G::NF>(r);
      b0 = r - c * G::TY;
    } else if (d == 0) {
      const int g = f - G::NC;
      a = G::TX;
      c = cdiv<G::TY, G::NF>(g);
      b0 = g - c * G::TY;
    } else {
      const int g = f - G::NC;
      c = cdiv<G::TX, G::NF>(g);
      a = g - c * G::TX;
      b0 = G::TY;
    }
  } else {
    const int r = d == 0 ? cdiv<G::TX + 1, G::NF>(f) : cdiv<G::TX, G::NF>(f);
    a = f - r * e0;
    c = d == 1 ? cdiv<G::TY + 1, G::NF>(r) : cdiv<G::TY, G::NF>(r);
    b0 = r - c * e1;
  }
  const int b = b0 < (G::TY & ~3) ? swz(b0) : b0;   // the extra y face (b0 = TY) keeps its row
  // the face lies between cell (a,b,c) - e_d and cell (a,b,c)
  const bool valid = x0 + a < L.n[0] + (d == 0) && y0 + b < L.n[1] + (d == 1) && z0 + c < L.n[2] + (d == 2);
  if (!valid) return;
  const int sp = d == 0 ? 1 : (d == 1 ? G::BX : G::BX * G::BY);
  const int sm = d == 0 ? 1 : (d == 1 ? G::BX : G::BX * G::MY);
  const T* sPc = sP + ((c + G::NG) * G::BY + (b + G::NG)) * G::BX + (a + G::HX) - sp;
  const T* sMc = sM + ((c + 1) * G::MY + (b + 1)) * G::BX + (a + G::HX) - sm;
  T Phi[NV];
  face_flux_rot<T, R, FAST>(sPc, sMc, sp, sm, d, par, Phi);
  T* o = sF + off + (c * e1 + b) * e0 + a;
  o[0] = Phi[0];
  o[4 * G::NF] = Phi[4];
  o[8 * G::NF] = Phi[8];
#pragma unroll
  for (int c3 = 0; c3 < 3; c3++) {
    const int t = rot3(d, c3);
    o[(1 + t) * G::NF] = Phi[1 + c3];
    o[(5 + t) * G::NF] = Phi[5 + c3];
  }
}

// Source item: the geometric and cleaning sources (a6) of 32 cells -> sR[(q-1) * NC + cell], q = 1..8
// (the D equation has no source).  Needs no flux, so it fills the scheduling gaps of the face items.
template <typename T, int R, int FAST>
__device__ __forceinline__ void source_task(const Layout& L, const Par<T>& par, const T* sP, const T* sM, T* sR,
                                            const T* __restrict__ cln, int cell, int x0, int y0, int z0) {
  using G = TileGeom<T, R>;
  const int a = cell % G::TX, r = cell / G::TX;
  const int b = swz(r % G::TY), c = r / G::TY;
  if (x0 + a >= L.n[0] || y0 + b >= L.n[1] || z0 + c >= L.n[2]) return;
  const T* sPc = sP + ((c + G::NG) * G::BY + (b + G::NG)) * G::BX + (a + G::HX);
  const T* sMc = sM + ((c + 1) * G::MY + (b + 1)) * G::BX + (a + G::HX);
  const int gmask = (L.g[0] ? 1 : 0) | (L.g[1] ? 2 : 0) | (L.g[2] ? 4 : 0);
  source_cell<T, R, FAST>(sPc, sMc, sR + cell, cln + L.idx(x0 + a, y0 + b, z0 + c), L.fs, gmask, par.gg1, par.kappa,
                          par.ih[0], par.ih[1], par.ih[2], par.cleaning, par.energy_var);
}

// One thread: the two TMA boxes of `tile` (primitives, metric), completion on `bar`.
template <typename T, int R>
__device__ __forceinline__ void issue_loads(const CUtensorMap* tmP, const CUtensorMap* tmM, const Layout& L, T* sP, T* sM,
                                            unsigned bar, int tile, int ntx, int nty) {
  using G = TileGeom<T, R>;
  const int tx = tile % ntx, r = tile / ntx;
  const int x0 = tx * G::TX, y0 = (r % nty) * G::TY, z0 = (r / nty) * G::TZ;
  mbar_expect_tx(bar, G::TX_BYTES);
  // storage coordinates of tile-local cell (-HX,-2,-2) / (-HX,-1,-1); out-of-range parts are zero-filled
  tma_load_4d(smem_addr(sP), tmP, bar, x0 + L.ox - G::HX, y0 + L.g[1] - G::NG, z0 + L.g[2] - G::NG, 0);
  tma_load_4d(smem_addr(sM), tmM, bar, x0 + L.ox - G::HX, y0 + L.g[1] - 1, z0 + L.g[2] - 1, 0);
}

// ---- the kernel: persistent blocks, one tile per iteration ----------------------------------------
// stage 0: Uout = Uin + dt L;  1: Uout = 3/4 U0 + 1/4 (Uin + dt L);  2: Uout = 1/3 U0 + 2/3 (Uin + dt L)
// Uin and Uout are the SAME buffer in stages 1 and 2 (no __restrict__ on them): the update is in place, which is
// safe because a thread reads only its own cell of U, once, before it writes it.
// tmP / tmM: tensor maps of the current primitives and of the metric as 4D arrays (x, y, z, field).
// Tiles are numbered x fastest; block b takes the tiles order[b], order[b + gridDim.x], ...  While a block is in phase 2
// of one tile, the TMA loads of its next tile are already in flight (the staged boxes are dead by then).
// T2 is the arithmetic type of phase 2.  T2 = T: pure fp64 or pure fp32.  T = float with
// T2 = double is the paper's mixed mode: storage, reconstruction and face fluxes in
// fp32; flux difference, Runge-Kutta combine and the primitive recovery in fp64.
// PEER = 1: the instantiation for slabs with mapped neighbours (peer stores, above); `peer` is an empty struct otherwise.
template <typename T, typename T2, int R, int FAST, int PEER = 0>
__global__ void __launch_bounds__(Tile<T, R>::NT, 1)
k_substep(const __grid_constant__ CUtensorMap tmP, const __grid_constant__ CUtensorMap tmM, Layout L, Par<T> par,
          Par<T2> par2, const T* __restrict__ cln, const T* Uin, const T* __restrict__ U0, T* Uout,
          T* __restrict__ Pout, int stage, T2 dt, unsigned long long* __restrict__ counters, int ntx, int nty,
          int ntiles, const int* __restrict__ order, const PeerArg<T, PEER> peer = PeerArg<T, PEER>()) {
  using G = TileGeom<T, R>;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  T* sP = reinterpret_cast<T*>(smem_raw + G::OFF_P);  // sP[field][z][y][x], halo 2 (HX in x)
  T* sM = reinterpret_cast<T*>(smem_raw + G::OFF_M);  // sM[field][z][y][x], halo 1 (HX in x)
  T* sF = reinterpret_cast<T*>(smem_raw + G::OFF_F);  // sF[q * NF + face]
  T* sR = reinterpret_cast<T*>(smem_raw + G::OFF_R);  // sR[(q-1) * NC + cell]
  const unsigned bar = smem_addr(smem_raw + G::OFF_BAR);       // the staged boxes of a tile have landed
  const unsigned bar2 = smem_addr(smem_raw + G::OFF_BAR + 8);  // every warp has read the fluxes and sources of a tile
  const int lane = threadIdx.x & 31;

  if (threadIdx.x == 0) { mbar_init(bar, 1); mbar_init(bar2, G::NT / 32); }
  __syncthreads();
  if (threadIdx.x == 0 && (int)blockIdx.x < ntiles) issue_loads<T, R>(&tmP, &tmM, L, sP, sM, bar, order[blockIdx.x], ntx, nty);

  // this thread's cell of phase 2 (one cell per thread), tile-local
  const bool has_cell = G::NT == G::NC || (int)threadIdx.x < G::NC;   // warp-uniform
  const int ctid = has_cell ? (int)threadIdx.x : 0;
  const int ca = ctid % G::TX, cr = ctid / G::TX;
  const int cb = swz(cr % G::TY), cc = cr / G::TY;
  const T* sPc = sP + ((cc + G::NG) * G::BY + (cb + G::NG)) * G::BX + (ca + G::HX);
  const T* sMc = sM + ((cc + 1) * G::MY + (cb + 1)) * G::BX + (ca + G::HX);
  int fail = 0, reset = 0, pfl = 0, it = 0, nstall = 0;
  unsigned parity = 0;
  int tile_next = (int)blockIdx.x < ntiles ? order[blockIdx.x] : 0;   // tile numbers are fetched one tile ahead

#pragma unroll 1
  for (int ti = blockIdx.x; ti < ntiles; ti += gridDim.x, parity ^= 1u) {
    // order[]: the sequence in which the tiles are taken (hz_lib.cu: blocks of neighbouring tiles, so that the halo
    // a tile shares with its neighbours is still in L2 when they ask for it); tile numbers are x fastest
    // (the load of the next number is in flight during phase 1: read at the top of its own iteration it cost 1 % of
    // the kernel in long-scoreboard stalls)
    const int tile = tile_next;
    tile_next = ti + (int)gridDim.x < ntiles ? order[ti + gridDim.x] : 0;
    const int tx = tile % ntx, tr = tile / ntx;
    const int x0 = tx * G::TX, y0 = (tr % nty) * G::TY, z0 = (tr / nty) * G::TZ;
    const int ci = x0 + ca, cj = y0 + cb, ck = z0 + cc;
    const bool cell_ok = has_cell && ci < L.n[0] && cj < L.n[1] && ck < L.n[2];
    const long long id = L.idx(ci, cj, ck);
    mbar_wait(bar, parity);
    // sF / sR may be overwritten once every warp is through phase 2a of the previous tile.  That is an mbarrier the
    // warps arrive at after 2a and wait on here, not a __syncthreads after 2a: a warp that has its right-hand
    // sides goes straight on to the Newton iteration (pure arithmetic) while others are still reading fluxes
    // (bound by shared-memory latency), and the two kinds of work overlap across the warps of the block.
    if (ti != (int)blockIdx.x) mbar_wait(bar2, parity ^ 1u);

    // ---- phase 1: face items, then source items ----
    // Static schedule: the items of a tile cost the same from tile to tile.  General rule: warp w takes face items
    // w, w + NW, ...; the source items go to the warps that got one face item fewer.  (A shared-memory work queue
    // with atomics measured 3 % slower: its fetches sat in 6 % of the stall samples.)
    if constexpr (sizeof(T) == 8 && G::NFACE_TASKS == 28 && G::NSRC_TASKS == 8 && G::NT == 256) {
      // fp64 MC tile, 28 + 8 items on 8 warps.  A source item has fewer instructions than a face item but issues them
      // more slowly (one dependent chain per thread), so the two take about the same time (measured 448 : 494), and
      // what matters is the mix on each of the four schedulers (warp w runs on scheduler w mod 4): warps 0-3 take
      // five face items each, warps 4-7 two face items and two source items -- every scheduler then has one warp bound
      // by the fp64 pipe and one bound by latency: +5 % against the rule below, which balances item counts.  (The
      // assignment that minimises the longest warp for fixed item durations leaves two warps with source items only:
      // -16 %; handing a warp consecutive items, all of one sweep axis: -10 %.)
      const int warp = threadIdx.x >> 5;
      // (one call site for both halves: a second one would put a second copy of the z face body into the kernel)
      const int t0 = warp < 4 ? warp : 16 + warp, t1 = warp < 4 ? 20 : 28;
#pragma unroll 1
      for (int t = t0; t < t1; t += 4) face_task<T, R, FAST>(L, par, sP, sM, sF, t, lane, x0, y0, z0);
      if (warp >= 4) {
#pragma unroll 1
        for (int t = warp - 4; t < 8; t += 4) source_task<T, R, FAST>(L, par, sP, sM, sR, cln, t * 32 + lane, x0, y0, z0);
      }
    } else {
      constexpr int NW = G::NT / 32, REM = G::NFACE_TASKS % NW;
      const int warp = threadIdx.x >> 5;
#pragma unroll 1
      for (int t = warp; t < G::NFACE_TASKS; t += NW) face_task<T, R, FAST>(L, par, sP, sM, sF, t, lane, x0, y0, z0);
      if (REM == 0 || warp >= REM) {
#pragma unroll 1
        for (int t = REM == 0 ? warp : warp - REM; t < G::NSRC_TASKS; t += REM == 0 ? NW : NW - REM)
          source_task<T, R, FAST>(L, par, sP, sM, sR, cln, t * 32 + lane, x0, y0, z0);
      }
    }
    // inputs of this thread's cell: conserved state from HBM (latency overlaps the barrier wait), metric and
    // the Newton guess Z = rho h W^2 of the previous primitives from the staged boxes (free for the next
    // tile afterwards)
    // (in the mixed mode, where phase 2 needs fp64 registers at 128 per thread, the early request would only be
    // spilled and read back: there U is requested in phase 2a, where it overlaps the flux read)
    constexpr bool EARLY_U = sizeof(T2) == sizeof(T);
    T u[NV], m[NM];
    T2 Zg = 0;
    if (EARLY_U && cell_ok) {
#pragma unroll
      for (int v = 0; v < NV; v++) u[v] = Uin[v * L.fs + id];
    }
    if (has_cell) {
#pragma unroll
      for (int v = 0; v < NM; v++) m[v] = sMc[v * G::MFS];
      T2 ut[3], utl[3], g2[6];
#pragma unroll
      for (int a3 = 0; a3 < 3; a3++) ut[a3] = (T2)sPc[(UX + a3) * G::PFS];
#pragma unroll
      for (int a6 = 0; a6 < 6; a6++) g2[a6] = (T2)m[GXX + a6];
      lower(g2, ut, utl);
      Zg = ((T2)sPc[RHO * G::PFS] + par2.gg1 * (T2)sPc[PR * G::PFS]) * (1 + dot3(ut, utl));
    }
    __syncthreads();  // all fluxes and sources are in shared memory; nobody reads sP / sM any more
    if (threadIdx.x == 0 && ti + (int)gridDim.x < ntiles)
      issue_loads<T, R>(&tmP, &tmM, L, sP, sM, bar, tile_next, ntx, nty);

    // ---- phase 2: one cell per thread, arithmetic in T2 ----
    // 2a: right-hand side from the fluxes and sources in shared memory and the Euler stage u + dt L; after the
    // barrier below sF / sR are free, so a warp that finishes 2b early goes straight on to the next tile's work
    // queue (the Newton iteration counts differ from cell to cell, and no barrier follows them).  The state at
    // the start of the step (stages 1, 2) is requested here and used after the barrier.
    T2 un[NV];
    T u0[NV];
    if (cell_ok) {
      if constexpr (!EARLY_U) {
#pragma unroll
        for (int v = 0; v < NV; v++) u[v] = Uin[v * L.fs + id];
      }
      if (stage != 0) {
#pragma unroll
        for (int v = 0; v < NV; v++) u0[v] = U0[v * L.fs + id];
      }
      T2 Rh[NV];
      Rh[0] = 0;
#pragma unroll
      for (int v = 1; v < NV; v++) Rh[v] = (T2)sR[(v - 1) * G::NC + ctid];
      if (L.g[0]) {
        const T2 ih = par2.ih[0];
        const T* o = sF + (cc * G::TY + cb) * (G::TX + 1) + ca;
#pragma unroll
        for (int v = 0; v < NV; v++) Rh[v] -= ((T2)o[v * G::NF + 1] - (T2)o[v * G::NF]) * ih;
      }
      if (L.g[1]) {
        const T2 ih = par2.ih[1];
        const T* o = sF + G::NFX + (cc * (G::TY + 1) + cb) * G::TX + ca;
#pragma unroll
        for (int v = 0; v < NV; v++) Rh[v] -= ((T2)o[v * G::NF + G::TX] - (T2)o[v * G::NF]) * ih;
      }
      if (L.g[2]) {
        const T2 ih = par2.ih[2];
        const T* o = sF + G::NFX + G::NFY + (cc * G::TY + cb) * G::TX + ca;
#pragma unroll
        for (int v = 0; v < NV; v++) Rh[v] -= ((T2)o[v * G::NF + G::TX * G::TY] - (T2)o[v * G::NF]) * ih;
      }
      if (!cleaning_<FAST>(par2)) Rh[8] = 0;
#pragma unroll
      for (int v = 0; v < NV; v++) un[v] = (T2)u[v] + dt * Rh[v];
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(bar2);   // this warp has read sF / sR (waited on before the next tile's phase 1)
    if (cell_ok) {  // 2b
      // a7: Runge-Kutta stage combine
      if (stage != 0) {
        const T2 wa = stage == 1 ? T2(0.75) : T2(1.0 / 3.0), wb = stage == 1 ? T2(0.25) : T2(2.0 / 3.0);
#pragma unroll
        for (int v = 0; v < NV; v++) un[v] = wa * (T2)u0[v] + wb * un[v];
      }
      // a8: primitive recovery and floors
      T2 m2[NM];
#pragma unroll
      for (int v = 0; v < NM; v++) m2[v] = (T2)m[v];
      T2 cf[6], gi[6];
      const T2 det = cofactors(m2 + GXX, cf);
      const T2 sq = sqrt_(det);
      const T2 idet = rcp_(det);
#pragma unroll
      for (int a6 = 0; a6 < 6; a6++) gi[a6] = cf[a6] * idet;
      const T2 isq = rcp_(sq);
      T2 w[NV];
#pragma unroll
      for (int v = 0; v < NV; v++) w[v] = un[v] * isq;
      if (!cleaning_<FAST>(par2)) w[8] = 0;
      if (evar_<FAST>(par2)) w[4] = energy_to_tau(w, m2);
      T2 qn[NV];
      int its = 0, stl = 0;
      const int fl = con2prim(w, m2, gi, par2, Zg, qn, its, stl);
      nstall += stl;
      it = its > it ? its : it;
      bool rs = fl != 0;
      if (!rs && qn[RHO] < par2.rho_thr) rs = true;
      bool pf = false;
      if (rs) {
        qn[RHO] = par2.rho_atm; qn[PR] = par2.p_atm;
#pragma unroll
        for (int a3 = 0; a3 < 3; a3++) { qn[UX + a3] = 0; qn[BX + a3] = w[5 + a3]; }
        qn[PSI] = w[8];
      } else if (qn[PR] < par2.p_atm) {
        pf = true;
        qn[PR] = par2.p_atm;
      }
      if (rs || pf) {
        T2 uf[NV];
        prim2con(qn, m2, par2, uf);
        if (evar_<FAST>(par2)) uf[4] = tau_to_energy(uf, m2);
#pragma unroll
        for (int v = 0; v < NV; v++) un[v] = sq * uf[v];
      }
      fail += fl != 0; reset += rs; pfl += pf;
      T qs[NV];
#pragma unroll
      for (int v = 0; v < NV; v++) {
        Uout[v * L.fs + id] = (T)un[v];
        qs[v] = (T)qn[v];
      }
      store_prims_with_images<T, PEER>(L, Pout, ci, cj, ck, qs, peer);
    }
  }
  // warp-level reduction of the counters: [0] c2p_fail, [1] atm_reset, [2] p_floor, [3] max iterations,
  // [4] recoveries ended by the fp32 round-off rule
  const unsigned full = 0xffffffffu;
  const int nf = __reduce_add_sync(full, fail), nr = __reduce_add_sync(full, reset), np = __reduce_add_sync(full, pfl);
  const int mi = __reduce_max_sync(full, it), ns = __reduce_add_sync(full, nstall);
  if (lane == 0) {
    if (nf) atomicAdd(counters + 0, (unsigned long long)nf);
    if (nr) atomicAdd(counters + 1, (unsigned long long)nr);
    if (np) atomicAdd(counters + 2, (unsigned long long)np);
    if (ns) atomicAdd(counters + 4, (unsigned long long)ns);
    if ((unsigned long long)mi > counters[3]) atomicMax(counters + 3, (unsigned long long)mi);
  }
}

}  // namespace hz
