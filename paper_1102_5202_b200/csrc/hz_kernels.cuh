// hz_kernels.cuh -- the kernels of one Runge-Kutta substep and of the set/get/diagnostic calls.
//
// The substep itself is the one fused kernel of hz_substep.cuh; here are the ghost fill used by
// hz_set_metric / hz_set_primitives, the pack / unpack kernels of the set / get calls and the
// reductions of hz_diagnostics.  All kernels are templated on the arithmetic type (double / float).
#pragma once
#include "hz_layout.cuh"
#include "hz_physics.cuh"

namespace hz {

constexpr int NDIAG = 16;      // doubles per block partial of the diagnostics reduction

// interior linear index -> (i, j, k), x fastest
__device__ __forceinline__ void cell_of(const Layout& L, long long t, int& i, int& j, int& k) {
  i = (int)(t % L.n[0]);
  long long r = t / L.n[0];
  j = (int)(r % L.n[1]);
  k = (int)(r / L.n[1]);
}

template <typename T>
__device__ __forceinline__ void load_fields(const T* __restrict__ F, long long fs, long long id, int nf, T* out) {
#pragma unroll
  for (int q = 0; q < NM; q++)
    if (q < nf) out[q] = F[q * fs + id];
}

// ---- ghost fill (O9 / R15): periodic wrap or zero-gradient copy, any number of fields ---
template <typename T>
__global__ void k_fill_ghosts(Layout L, T* __restrict__ F, int nf) {
  const long long ntot = (long long)L.N[0] * L.N[1] * L.N[2];
  long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= ntot) return;
  int c[3];
  c[0] = (int)(t % L.N[0]) - L.g[0];
  long long r = t / L.N[0];
  c[1] = (int)(r % L.N[1]) - L.g[1];
  c[2] = (int)(r / L.N[1]) - L.g[2];
  int s[3];
  bool ghost = false;
#pragma unroll
  for (int d = 0; d < 3; d++) {
    const int n = L.n[d];
    if (c[d] < 0 || c[d] >= n) {
      if (bc_side(L.bc[d], c[d] < 0 ? 0 : 1) == 2) return;  // external side: filled by hz_halo_unpack
      ghost = true;
      s[d] = L.bc[d] == 0 ? ((c[d] % n) + n) % n : (c[d] < 0 ? 0 : n - 1);
    } else {
      s[d] = c[d];
    }
  }
  if (!ghost) return;
  const long long dst = L.idx(c[0], c[1], c[2]), src = L.idx(s[0], s[1], s[2]);
  for (int f = 0; f < nf; f++) F[f * L.fs + dst] = F[f * L.fs + src];
}

// ---- hz_halo_pack / hz_halo_unpack: ng whole padded z planes of nf fields <-> one contiguous buffer ----
// k0: first storage plane; buffer layout [field][plane][y][x] with the padded extents of the context.
template <typename T>
__global__ void k_halo_copy(Layout L, T* __restrict__ F, int nf, int k0, T* __restrict__ buf, int unpack) {
  const long long per = (long long)L.ng * L.sz, tot = per * nf;
  for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < tot; e += (long long)gridDim.x * blockDim.x) {
    const long long f = e / per, r = e - f * per;
    T* cell = F + f * L.fs + (long long)k0 * L.sz + r;
    if (unpack) *cell = buf[e]; else buf[e] = *cell;
  }
}

// ---- static coefficients of the cleaning sources (O6 / R14) -----------------------------------
// cln[k] = sum_j d_j(alpha sqrt(gamma) gamma^{kj}), k = x y z;  cln[3] = sum_j d_j(sqrt(gamma) beta^j), centred
// differences of the stored metric at interior cells.  The metric is fixed, so this runs once per
// hz_set_metric (and again when ghost planes of the metric arrive through hz_halo_unpack).
template <typename T>
__global__ void k_clean_static(Layout L, const T* __restrict__ met, T* __restrict__ cln) {
  const long long n = L.ncell();
  long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  int i, j, k;
  cell_of(L, t, i, j, k);
  const long long id = L.idx(i, j, k);
  T dQ[3] = {0, 0, 0}, dRb = 0;
#pragma unroll
  for (int d = 0; d < 3; d++) {
    if (L.g[d] == 0) continue;
    const long long s = L.stride(d);
    const T i2h = T(0.5) * (T)(1.0 / L.h[d]);
    T mp[NM], mm[NM];
    load_fields(met, L.fs, id + s, NM, mp);
    load_fields(met, L.fs, id - s, NM, mm);
    T cp[6], cm[6];
    const T dp = cofactors(mp + GXX, cp), dn = cofactors(mm + GXX, cm);
    const T sp = sqrt_(dp), sn = sqrt_(dn);
    const T ap = div_(mp[AL], sp), am = div_(mm[AL], sn);  // alpha sqrt(gamma) gamma^{kd} = alpha cof_kd / sqrt(gamma)
#pragma unroll
    for (int kk = 0; kk < 3; kk++) dQ[kk] += (ap * cp[sym(kk, d)] - am * cm[sym(kk, d)]) * i2h;
    dRb += (sp * mp[BEX + d] - sn * mm[BEX + d]) * i2h;
  }
#pragma unroll
  for (int kk = 0; kk < 3; kk++) cln[kk * L.fs + id] = dQ[kk];
  cln[3 * L.fs + id] = dRb;
}

// ---- hz_fma_peak: what the plain FMA pipe sustains (the denominator of the ALU roofline) ----
// 16 independent accumulators per thread, `iters` trips of 16 FMAs each; nothing but FMAs in the loop.
template <typename T>
__global__ void __launch_bounds__(256) k_fma_peak(T* __restrict__ out, int iters, T a, T b) {
  T acc[16];
#pragma unroll
  for (int i = 0; i < 16; i++) acc[i] = (T)(threadIdx.x + i);
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 16; i++) acc[i] = acc[i] * a + b;
  }
  T s = 0;
#pragma unroll
  for (int i = 0; i < 16; i++) s += acc[i];
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// ---- hz_set_metric: interior-only planes -> padded SoA, with validation -------------------------
template <typename T>
__global__ void k_pack_metric(Layout L, const T* __restrict__ alpha, const T* __restrict__ beta3,
                              const T* __restrict__ gamma6, T* __restrict__ met, int* __restrict__ err) {
  const long long n = L.ncell();
  long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  int i, j, k;
  cell_of(L, t, i, j, k);
  T m[NM];
  m[0] = alpha[t];
#pragma unroll
  for (int a = 0; a < 3; a++) m[1 + a] = beta3[a * n + t];
#pragma unroll
  for (int a = 0; a < 6; a++) m[4 + a] = gamma6[a * n + t];
  T c[6];
  T det = cofactors(m + GXX, c);
  bool ok = m[AL] > 0 && det > 0 && m[GXX] > 0 && c[5] > 0;
#pragma unroll
  for (int a = 0; a < NM; a++) ok = ok && finite_(m[a]);
  ok = ok && finite_(det);
  if (!ok) atomicOr(err, 1);
  const long long id = L.idx(i, j, k);
#pragma unroll
  for (int a = 0; a < NM; a++) met[a * L.fs + id] = m[a];
}

// ---- hz_set_primitives: (rho, v^i, p, B^i) -> stored primitives (W v^i, psi = 0) and sqrt(gamma) U
template <typename T>
__global__ void k_pack_prims(Layout L, Par<T> par, const T* __restrict__ prim8, const T* __restrict__ met,
                             T* __restrict__ P, T* __restrict__ U, int* __restrict__ err) {
  const long long n = L.ncell();
  long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  int i, j, k;
  cell_of(L, t, i, j, k);
  const long long id = L.idx(i, j, k);
  T m[NM];
  load_fields(met, L.fs, id, NM, m);
  T a8[8];
  bool ok = true;
#pragma unroll
  for (int q = 0; q < 8; q++) { a8[q] = prim8[q * n + t]; ok = ok && finite_(a8[q]); }
  T vl[3];
  lower(m + GXX, a8 + 1, vl);
  T v2 = dot3(a8 + 1, vl);
  ok = ok && a8[0] > 0 && !(a8[4] < 0) && v2 < 1;
  if (!ok) { atomicOr(err, 1); return; }
  T W = rcp_(sqrt_(1 - v2));
  T q[NV];
  q[RHO] = a8[0]; q[PR] = a8[4]; q[PSI] = 0;
#pragma unroll
  for (int a = 0; a < 3; a++) { q[UX + a] = W * a8[1 + a]; q[BX + a] = a8[5 + a]; }
  T w[NV];
  prim2con(q, m, par, w);
  if (par.energy_var) w[4] = tau_to_energy(w, m);
  T sq = sqrt_det(m + GXX);
#pragma unroll
  for (int v = 0; v < NV; v++) { P[v * L.fs + id] = q[v]; U[v * L.fs + id] = sq * w[v]; }
}

// ---- hz_get_primitives ---------------------------------------------------------------------------
template <typename T>
__global__ void k_unpack_prims(Layout L, const T* __restrict__ P, const T* __restrict__ met, T* __restrict__ prim8) {
  const long long n = L.ncell();
  long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  int i, j, k;
  cell_of(L, t, i, j, k);
  const long long id = L.idx(i, j, k);
  T g[6], q[NV];
#pragma unroll
  for (int a = 0; a < 6; a++) g[a] = met[(GXX + a) * L.fs + id];
  load_fields(P, L.fs, id, NV, q);
  T utl[3];
  lower(g, q + UX, utl);
  T iW = rcp_(sqrt_(1 + dot3(q + UX, utl)));
  prim8[0 * n + t] = q[RHO];
#pragma unroll
  for (int d = 0; d < 3; d++) prim8[(1 + d) * n + t] = q[UX + d] * iW;
  prim8[4 * n + t] = q[PR];
#pragma unroll
  for (int d = 0; d < 3; d++) prim8[(5 + d) * n + t] = q[BX + d];
}

// nf padded fields starting at field f0 -> interior-only planes
template <typename T>
__global__ void k_unpack_fields(Layout L, const T* __restrict__ F, int f0, int nf, T* __restrict__ out) {
  const long long n = L.ncell();
  long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n) return;
  int i, j, k;
  cell_of(L, t, i, j, k);
  const long long id = L.idx(i, j, k);
  for (int f = 0; f < nf; f++) out[f * n + t] = F[(f0 + f) * L.fs + id];
}

// ---- a10: global reductions with warp shuffles ---------------------------------
// Block partial layout: [0..8] sums of U, [9] sum |divB|, [10] max |divB|, [11] max speed/dx
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
  return v;
}

template <typename T>
__global__ void __launch_bounds__(256) k_diag(Layout L, Par<T> par, const T* __restrict__ P, const T* __restrict__ U,
                                              const T* __restrict__ met, double* __restrict__ partials) {
  const long long n = L.ncell();
  double acc[12];
#pragma unroll
  for (int a = 0; a < 12; a++) acc[a] = 0;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (long long)gridDim.x * blockDim.x) {
    int i, j, k;
    cell_of(L, t, i, j, k);
    const long long id = L.idx(i, j, k);
#pragma unroll
    for (int v = 0; v < NV; v++) acc[v] += (double)U[v * L.fs + id];
    T m[NM], q[NV];
    load_fields(met, L.fs, id, NM, m);
    load_fields(P, L.fs, id, NV, q);
    T c[6];
    const T det = cofactors(m + GXX, c);
    const T sq = sqrt_(det), idet = rcp_(det);
    double div = 0, smax = 0;
#pragma unroll
    for (int d = 0; d < 3; d++) {
      if (L.g[d] == 0) continue;
      const long long s = L.stride(d);
      T gp[6], gm[6];
#pragma unroll
      for (int a = 0; a < 6; a++) { gp[a] = met[(GXX + a) * L.fs + id + s]; gm[a] = met[(GXX + a) * L.fs + id - s]; }
      const double bp = (double)sqrt_det(gp) * (double)P[(BX + d) * L.fs + id + s];
      const double bm = (double)sqrt_det(gm) * (double)P[(BX + d) * L.fs + id - s];
      div += (bp - bm) / (2 * L.h[d]);
      T gid[3], Uu[NV], Ff[NV], lm, lp;
#pragma unroll
      for (int kk = 0; kk < 3; kk++) gid[kk] = c[sym(kk, d)] * idet;
      if (d == 0) flux_speeds<T, 0>(q, m, gid, par, Uu, Ff, lm, lp);
      if (d == 1) flux_speeds<T, 1>(q, m, gid, par, Uu, Ff, lm, lp);
      if (d == 2) flux_speeds<T, 2>(q, m, gid, par, Uu, Ff, lm, lp);
      smax = fmax(smax, fmax(fabs((double)lm), fabs((double)lp)) / L.h[d]);
    }
    div /= (double)sq;
    acc[9] += fabs(div);
    acc[10] = fmax(acc[10], fabs(div));
    acc[11] = fmax(acc[11], smax);
  }
  __shared__ double sh[8][12];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int a = 0; a < 12; a++) {
    double v = a < 10 ? warp_sum(acc[a]) : warp_max(acc[a]);
    if (lane == 0) sh[wid][a] = v;
  }
  __syncthreads();
  if (threadIdx.x < 12) {
    const int a = threadIdx.x;
    double v = sh[0][a];
    for (int w = 1; w < 8; w++) v = a < 10 ? v + sh[w][a] : fmax(v, sh[w][a]);
    partials[(long long)blockIdx.x * NDIAG + a] = v;
  }
}

// one block: fold the block partials in a fixed order (deterministic result)
__global__ void k_diag_final(const double* __restrict__ partials, int nblocks, double* __restrict__ out) {
  const int a = threadIdx.x;
  if (a >= 12) return;
  double v = partials[a];
  for (int b = 1; b < nblocks; b++) {
    const double p = partials[(long long)b * NDIAG + a];
    v = a < 10 ? v + p : fmax(v, p);
  }
  out[a] = v;
}

}  // namespace hz
