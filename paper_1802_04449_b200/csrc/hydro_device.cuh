// hydro_device.cuh -- per-cell device building blocks of the CLVisc step (sm_100a).
//
// Everything here is written from /root/reference/PAPER.md (arXiv:1802.04449) and the readings in
// DESIGN.md; nothing is shared with oracle/.  Templated on the arithmetic type R (double / float).
//
//   eos_*          EoS lookup (EOSI PAPER.md:251, tables :253-259; table rule DESIGN.md A16)
//   signal_speed   local maximum propagation speed c_{i+1/2} (A6)
//   kt_div         KT flux difference H_{i+1/2} - H_{i-1/2} for one field (Eq.40-44)
//   is_source      Israel-Stewart source S_pi (Eq.33-38; signs DESIGN.md A1, A2)
//   rootfind       T_id^{tau mu} -> e, u~^i (Eq.51/54; A7, A8)
//   limit_pi       pi limiter (A14)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace clv {

// field order inside a state buffer
enum { F_E = 0, F_UX = 1, F_UY = 2, F_UN = 3, F_PI = 4 };
// symmetric (mu,nu) -> pi component
__constant__ int c_pidx[4][4] = {{0, 1, 2, 3}, {1, 4, 5, 6}, {2, 5, 7, 8}, {3, 6, 8, 9}};

template <typename R>
struct EosDev {
  int kind, n;
  R e_min, e_max, inv_e_min, inv_e_max;
  R P0_slope;       // P[0]/e_min                       (below-table branch)
  R P_top, T_bot, T_top;
  R conf_T_scale;   // 1/(c_sb*hbarc)   : T = hbarc * (e*conf_T_scale)^{1/4}
  R hbarc;
  float log2_emin, inv_dlog2;
  const R* node;    // [n]   e_k
  const R* P;       // [n]   P_k
  const R* cs2;     // [n-1] (P_{k+1}-P_k)/(e_{k+1}-e_k)
  const R* T;       // [n]
  const R* dTde;    // [n-1]
};

// device diagnostics block.  Non-negative doubles are stored as their bit pattern so
// that an unsigned 64-bit atomicMax orders them.
struct DiagDev {
  unsigned long long cfl[2][3];
  unsigned long long emax[2];
  unsigned long long n_floor, n_clamp, n_limit, n_nan, n_unconv;
};

template <typename R> __device__ __forceinline__ R rsqrt_(R x);
template <> __device__ __forceinline__ double rsqrt_<double>(double x) { return 1.0 / sqrt(x); }
template <> __device__ __forceinline__ float rsqrt_<float>(float x) { return 1.0f / sqrtf(x); }
template <typename R> __device__ __forceinline__ R sqrt_(R x);
template <> __device__ __forceinline__ double sqrt_<double>(double x) { return sqrt(x); }
template <> __device__ __forceinline__ float sqrt_<float>(float x) { return sqrtf(x); }
// Fast reciprocal / square roots for the production kernels (kernel 1 keeps the IEEE forms above): hardware seed plus
// Newton steps, no slow path.  fp64: rcp.approx / rsqrt.approx give ~20 bits, two Newton steps reach <= 2 ulp (the
// IEEE division and sqrt cost 25-30 instructions and a subroutine call each; ~15 of them sit on the per-plane critical
// path of the tile kernel).  fp32: the .approx instructions themselves (<= 2 ulp).
__device__ __forceinline__ double frcp_(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double e = fma(-x, y, 1.0);
  y = fma(y, e, y);
  e = fma(-x, y, 1.0);
  return fma(y, e, y);
}
__device__ __forceinline__ float frcp_(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ double frsqrt_(double x) {      // x > 0
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double h = 0.5 * y, e = fma(-(x * y), h, 0.5);
  y = fma(y, e, y);
  h = 0.5 * y; e = fma(-(x * y), h, 0.5);
  return fma(y, e, y);
}
__device__ __forceinline__ float frsqrt_(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ double fsqrt_(double x) {       // x >= 0
  const double y = frsqrt_(x > 0.0 ? x : 1.0);
  const double s = x * y;
  return fma(fma(-s, s, x), 0.5 * y, s);                   // one correction step on s = x rsqrt(x)
}
__device__ __forceinline__ float fsqrt_(float x) {
  float y;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
template <typename R> __device__ __forceinline__ R abs_(R x) { return x < R(0) ? -x : x; }
template <typename R> __device__ __forceinline__ R max_(R a, R b) { return a > b ? a : b; }
template <typename R> __device__ __forceinline__ R min_(R a, R b) { return a < b ? a : b; }

// ---------------------------------------------------------------------------------------------
// EoS
// ---------------------------------------------------------------------------------------------
template <typename R>
__device__ __forceinline__ int eos_bracket(const EosDev<R>& q, R e) {
  // first guess from a single-precision log2 (no double log on the hot path), then one exact
  // correction step against the node values: the bracket satisfies node[k] <= e < node[k+1].
  int k = (int)((__log2f((float)e) - q.log2_emin) * q.inv_dlog2);
  k = max(0, min(k, q.n - 2));
  if (e < __ldg(q.node + k)) k = max(k - 1, 0);
  else if (e >= __ldg(q.node + k + 1)) k = min(k + 1, q.n - 2);
  return k;
}

// P(e) and c_s^2(e)
template <typename R>
__device__ __forceinline__ void eos_P(const EosDev<R>& q, R e, R& P, R& cs2) {
  if (q.kind == 0) { P = e * R(1.0 / 3.0); cs2 = R(1.0 / 3.0); return; }
  if (e <= q.e_min) { P = q.P0_slope * e; cs2 = q.P0_slope; return; }
  if (e >= q.e_max) { P = q.P_top + (e - q.e_max) * R(1.0 / 3.0); cs2 = R(1.0 / 3.0); return; }
  const int k = eos_bracket(q, e);
  cs2 = __ldg(q.cs2 + k);
  P = __ldg(q.P + k) + (e - __ldg(q.node + k)) * cs2;
}

// T(e) in GeV (only needed at the cell centre, for 1/tau_pi)
template <typename R>
__device__ __forceinline__ R eos_T(const EosDev<R>& q, R e) {
  if (q.kind == 0) return q.hbarc * sqrt_(sqrt_(max_(e, R(0)) * q.conf_T_scale));
  if (e <= q.e_min) return q.T_bot * sqrt_(sqrt_(max_(e, R(0)) * q.inv_e_min));
  if (e >= q.e_max) return q.T_top * sqrt_(sqrt_(e * q.inv_e_max));
  const int k = eos_bracket(q, e);
  return __ldg(q.T + k) + (e - __ldg(q.node + k)) * __ldg(q.dTde + k);
}

// ---------------------------------------------------------------------------------------------
// Signal speed along one axis (A6): va = v_a, v2 = |v|^2.
// ---------------------------------------------------------------------------------------------
template <typename R>
__device__ __forceinline__ R signal_speed(R va, R v2, R cs2) {
  const R cs = sqrt_(cs2);
  const R disc = (R(1) - v2) * (R(1) - v2 * cs2 - va * va * (R(1) - cs2));
  return (abs_(va) * (R(1) - cs2) + cs * sqrt_(max_(disc, R(0)))) / (R(1) - v2 * cs2);
}

// ---------------------------------------------------------------------------------------------
// KT flux difference for one field along one axis.
// q[0..4], f[0..4]: conserved variable and its flux at i-2..i+2; cl, cr: face speeds at i-1/2, i+1/2.
// Slopes are generalised minmod (A4) of both Q and F (A5).  Returns H_{i+1/2} - H_{i-1/2}.
// ---------------------------------------------------------------------------------------------
template <typename R>
__device__ __forceinline__ R minmod_slope(R dm, R dp, R theta) {
  // minmod(theta*dm, (dm+dp)/2, theta*dp): non-zero only when dm, dp have the same sign, and the central
  // difference then shares it.
  const R a = theta * dm, c = theta * dp, b = R(0.5) * (dm + dp);
  const R m = min_(min_(abs_(a), abs_(c)), abs_(b));
  const bool pos = (dm > R(0)) && (dp > R(0)), neg = (dm < R(0)) && (dp < R(0));
  return pos ? m : (neg ? -m : R(0));
}

template <typename R>
__device__ __forceinline__ R kt_div(const R q[5], const R f[5], R cl, R cr, R theta) {
  const R dq0 = q[1] - q[0], dq1 = q[2] - q[1], dq2 = q[3] - q[2], dq3 = q[4] - q[3];
  const R df0 = f[1] - f[0], df1 = f[2] - f[1], df2 = f[3] - f[2], df3 = f[4] - f[3];
  const R sq1 = minmod_slope(dq0, dq1, theta), sq2 = minmod_slope(dq1, dq2, theta),
          sq3 = minmod_slope(dq2, dq3, theta);
  const R sf1 = minmod_slope(df0, df1, theta), sf2 = minmod_slope(df1, df2, theta),
          sf3 = minmod_slope(df2, df3, theta);
  // face i+1/2: left state from cell i (index 2), right state from cell i+1 (index 3)   Eq.41-44
  const R Hr = R(0.5) * ((f[3] - R(0.5) * sf3) + (f[2] + R(0.5) * sf2)) -
               R(0.5) * cr * ((q[3] - R(0.5) * sq3) - (q[2] + R(0.5) * sq2));
  const R Hl = R(0.5) * ((f[2] - R(0.5) * sf2) + (f[1] + R(0.5) * sf1)) -
               R(0.5) * cl * ((q[2] - R(0.5) * sq2) - (q[1] + R(0.5) * sq1));
  return Hr - Hl;
}

// ---------------------------------------------------------------------------------------------
// Israel-Stewart source (Eq.33 with lambda_2 = lambda_3 = 0), tilde components.
//   tau_pi = c_tau eta_v/(T s)  (paper: c_tau = 5; inv_ctau = 1/c_tau),  lambda_1 = lam1_hat / e
//   ut[4]      u~^mu at the cell
//   grad[m][n] nabla~_m u~^n  (Eq.22, 24-26 already added by the caller)
//   pi[10], e, P, T; out S[10] += source
// ---------------------------------------------------------------------------------------------
template <typename R>
__device__ __forceinline__ void is_source(const R ut[4], const R grad[4][4], const R pi[10], R e, R P, R T,
                                          R inv_5etas_hbarc, bool milne, R inv_tau, R S[10], R inv_ctau = R(0.2),
                                          R lam1_hat = R(0)) {
  const R gm[4] = {R(1), R(-1), R(-1), R(-1)};
  const R theta_exp = grad[0][0] + grad[1][1] + grad[2][2] + grad[3][3];
  R Du[4];
#pragma unroll
  for (int n = 0; n < 4; ++n)
    Du[n] = ut[0] * grad[0][n] + ut[1] * grad[1][n] + ut[2] * grad[2][n] + ut[3] * grad[3][n];
  const R inv_taupi = T * inv_5etas_hbarc;      // 1/tau_pi = T s/(c_tau eta_v)  (c_tau = 5)
  const R eta_over_taupi = (e + P) * inv_ctau;  // eta_v/tau_pi = (e+P)/c_tau
  const int IDX[4][4] = {{0, 1, 2, 3}, {1, 4, 5, 6}, {2, 5, 7, 8}, {3, 6, 8, 9}};
  R w[4];
#pragma unroll
  for (int n = 0; n < 4; ++n)
    w[n] = pi[IDX[n][0]] * Du[0] - pi[IDX[n][1]] * Du[1] - pi[IDX[n][2]] * Du[2] - pi[IDX[n][3]] * Du[3];
#pragma unroll
  for (int m = 0; m < 4; ++m)
#pragma unroll
    for (int n = m; n < 4; ++n) {
      // sigma~^{mn} = nabla~^m u^n + nabla~^n u^m - u^m Du^n - u^n Du^m - (2/3)(g^{mn} - u^m u^n) theta
      const R sig = gm[m] * grad[m][n] + gm[n] * grad[n][m] - ut[m] * Du[n] - ut[n] * Du[m] -
                    R(2.0 / 3.0) * ((m == n ? gm[m] : R(0)) - ut[m] * ut[n]) * theta_exp;
      const R p = pi[IDX[m][n]];
      R src = eta_over_taupi * sig - p * inv_taupi - p * theta_exp * R(1.0 / 3.0);
      // (u^m pi^{n b} + u^n pi^{m b}) g_{b a} Du^a with w^n = pi^{n b} g_{b a} Du^a formed once per row
      src -= ut[m] * w[n] + ut[n] * w[m];
      if (milne) {
        R I = R(0);   // Eq.35-38 in the general form (A2)
        if (m == 0) I += pi[IDX[3][n]];
        if (m == 3) I += pi[IDX[0][n]];
        if (n == 0) I += pi[IDX[m][3]];
        if (n == 3) I += pi[IDX[m][0]];
        src -= (p * ut[0] + I * ut[3]) * inv_tau;
      }
      S[IDX[m][n]] += src;
    }
  // lambda_1 term (Eq.4 / Eq.33): -(lambda_1/tau_pi) pi~^{<mu}_lambda pi~^{nu>lambda}.
  // X^{ab} = pi^{a l} g_{l k} pi^{k b};  Delta X Delta = X - u w^T - w u^T + u u^T s  with  w^a = X^{ab} u_b,
  // s = u_a X^{ab} u_b;  the traceless part subtracts 1/3 Delta^{mn} (g_{ab} X^{ab} - s).
  if (lam1_hat != R(0)) {
    R X[4][4], wv[4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
      for (int b = a; b < 4; ++b) {
        X[a][b] = pi[IDX[a][0]] * pi[IDX[0][b]] - pi[IDX[a][1]] * pi[IDX[1][b]] - pi[IDX[a][2]] * pi[IDX[2][b]] -
                  pi[IDX[a][3]] * pi[IDX[3][b]];
        X[b][a] = X[a][b];
      }
    R sx = R(0), tr = R(0);
#pragma unroll
    for (int a = 0; a < 4; ++a) {
      wv[a] = X[a][0] * ut[0] - X[a][1] * ut[1] - X[a][2] * ut[2] - X[a][3] * ut[3];
      tr += gm[a] * X[a][a];
    }
#pragma unroll
    for (int a = 0; a < 4; ++a) sx += gm[a] * ut[a] * wv[a];
    const R coef = lam1_hat / e * inv_taupi, third = (tr - sx) * R(1.0 / 3.0);
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
      for (int n = m; n < 4; ++n) {
        const R proj = X[m][n] - ut[m] * wv[n] - wv[m] * ut[n] + ut[m] * ut[n] * sx -
                       ((m == n ? gm[m] : R(0)) - ut[m] * ut[n]) * third;
        S[IDX[m][n]] -= coef * proj;
      }
  }
}

// ---------------------------------------------------------------------------------------------
// Root-find (Eq.51/54; A7, A8).  M0 = T_id^{tau tau}, Mi = T_id^{tau i}.  e_start: warm start.
// Branch-uniform: fixed iteration count, updates by select.  flags: bit0 floored, bit1 clamped, bit2
// residual above tolerance, bit3 NaN input.
// ---------------------------------------------------------------------------------------------
template <typename R>
__device__ __forceinline__ void rootfind(const EosDev<R>& eos, R M0, R Mx, R My, R Mn, R e_start, int iters,
                                         R e_floor, R v_max, R& e_out, R& ux, R& uy, R& un, unsigned& flags) {
  if (!(M0 == M0) || !(Mx == Mx) || !(My == My) || !(Mn == Mn)) flags |= 8u;
  if (!(M0 > e_floor)) {
    e_out = e_floor; ux = uy = un = R(0); flags |= 1u;
    return;
  }
  R M2 = Mx * Mx + My * My + Mn * Mn;
  const R lim = v_max * M0;
  if (M2 > lim * lim) {
    const R sc = lim * rsqrt_(M2);
    Mx *= sc; My *= sc; Mn *= sc; M2 = lim * lim; flags |= 2u;
  }
  R e;
  if (eos.kind == 0) {
    // closed form for P = e/3:  e = -M0 + sqrt(4 M0^2 - 3 M^2) = 3 (M0^2 - M^2)/(M0 + sqrt(M0^2 + 3 (M0^2 - M^2)))
    const R d = M0 * M0 - M2;
    e = R(3) * d / (M0 + sqrt_(M0 * M0 + R(3) * d));
  } else {
    const R tol = (sizeof(R) == 8) ? R(1e-15) : R(2e-7);
    R lo = R(0), hi = M0;
    e = e_start;
    if (!(e > lo && e < hi)) e = M0 - M2 / (M0 + M0 * R(1.0 / 3.0));
    if (!(e > lo && e < hi)) e = R(0.5) * M0;
    R g = R(0);
    for (int it = 0; it < iters; ++it) {
      R P, cs2;
      eos_P(eos, e, P, cs2);
      const R inv = R(1) / (M0 + P);
      g = M0 - M2 * inv - e;                        // strictly decreasing in e
      const R dg = M2 * cs2 * inv * inv - R(1);
      if (g > R(0)) lo = e; else hi = e;
      R en = e - g / dg;
      // the Newton step moves towards the root from the side just recorded, so it may land ON the other
      // bracket end (root at M0 when M -> 0): accept the closed interval, bisect only outside it
      if (!(en >= lo && en <= hi)) en = R(0.5) * (lo + hi);
      e = (abs_(g) > tol * M0) ? en : e;
    }
    {
      R P, cs2;
      eos_P(eos, e, P, cs2);
      g = M0 - M2 / (M0 + P) - e;
      if (abs_(g) > R(1e3) * tol * M0) flags |= 4u;
    }
  }
  if (e < e_floor) { e = e_floor; flags |= 1u; }
  R P, cs2;
  eos_P(eos, e, P, cs2);
  const R iw = R(1) / (M0 + P);
  const R vx = Mx * iw, vy = My * iw, vn = Mn * iw;
  const R gam = rsqrt_(R(1) - (vx * vx + vy * vy + vn * vn));
  ux = gam * vx; uy = gam * vy; un = gam * vn;
  e_out = e;
}

// pi limiter (A14): scale pi~ so that sqrt|pi~^{mn} pi~_{mn}| <= xi sqrt(e^2 + 3 P^2).
template <typename R>
__device__ __forceinline__ void limit_pi(const EosDev<R>& eos, R xi, R e, R pi[10], unsigned& flags) {
  if (!(xi > R(0))) return;
  R P, cs2;
  eos_P(eos, e, P, cs2);
  const R pp = pi[0] * pi[0] - R(2) * (pi[1] * pi[1] + pi[2] * pi[2] + pi[3] * pi[3]) + pi[4] * pi[4] +
               pi[7] * pi[7] + pi[9] * pi[9] + R(2) * (pi[5] * pi[5] + pi[6] * pi[6] + pi[8] * pi[8]);
  const R mag2 = abs_(pp);
  const R lim2 = xi * xi * (e * e + R(3) * P * P);
  if (mag2 > lim2) {
    const R r = sqrt_(lim2) * rsqrt_(mag2);
#pragma unroll
    for (int m = 0; m < 10; ++m) pi[m] *= r;
    flags |= 16u;
  }
}

// ---------------------------------------------------------------------------------------------
// Block-level reductions (warp shuffle, then one atomic per warp).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void atomic_max_nonneg(unsigned long long* addr, double v) {
  // v >= 0 (or NaN, which is dropped)
  if (v > 0.0) atomicMax(addr, (unsigned long long)__double_as_longlong(v));
}

__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

__device__ __forceinline__ void count_flags(DiagDev* d, unsigned flags) {
  const unsigned any = __ballot_sync(0xffffffffu, flags != 0);
  if (any == 0) return;
  const unsigned b0 = __ballot_sync(0xffffffffu, flags & 1u), b1 = __ballot_sync(0xffffffffu, flags & 2u),
                 b2 = __ballot_sync(0xffffffffu, flags & 4u), b3 = __ballot_sync(0xffffffffu, flags & 8u),
                 b4 = __ballot_sync(0xffffffffu, flags & 16u);
  const int lane = (threadIdx.x + threadIdx.y * blockDim.x + threadIdx.z * blockDim.x * blockDim.y) & 31;
  if (lane == 0) {
    if (b0) atomicAdd(&d->n_floor, (unsigned long long)__popc(b0));
    if (b1) atomicAdd(&d->n_clamp, (unsigned long long)__popc(b1));
    if (b2) atomicAdd(&d->n_unconv, (unsigned long long)__popc(b2));
    if (b3) atomicAdd(&d->n_nan, (unsigned long long)__popc(b3));
    if (b4) atomicAdd(&d->n_limit, (unsigned long long)__popc(b4));
  }
}

}  // namespace clv
