// hydro_stage_tiled.cuh -- "kernel 2": the production stage kernel.
//
// Same fused stage as hydro_stage_ref.cuh (one launch per RK2 stage, one thread per cell), re-organised
// around what the ncu profile of kernel 1 showed (profiles/round1_v1_ref_kernel.md: fp64 pipe 30 %,
// 15 k instructions per cell, 255 registers, 12 % occupancy):
//   * EXTENDED STATE: the producing kernel appends P, u^tau and the three signal speeds c_x, c_y, c_eta
//     of every cell to the state it writes (5 extra words), so the 13-point star is READ, never
//     re-derived: no EoS lookup, sqrt or division per stencil point (kernel 1 re-derives them 15 times).
//   * cheap generalised minmod: 2 compares + 3 arithmetic fp64 instructions, sign logic on the integer pipe.
//   * the overall factor tau of Q_T, F_T (Eq.18) is applied once to the flux difference, not per point.
//   * warp-uniform early exit of the Newton iteration (no intra-warp divergence).
#pragma once
#include "hydro_stage_ref.cuh"

namespace clv {

// extended-state field slots, counted from the end of the evolved fields (nf = 4 ideal / 14 viscous)
enum { X_P = 0, X_G = 1, X_CX = 2, X_CY = 3, X_CN = 4, X_COUNT = 5 };

__device__ __forceinline__ bool same_sign(double a, double b) {
  return (__double2hiint(a) ^ __double2hiint(b)) >= 0;
}
__device__ __forceinline__ bool same_sign(float a, float b) { return (__float_as_int(a) ^ __float_as_int(b)) >= 0; }
__device__ __forceinline__ double copysign_(double m, double s) { return copysign(m, s); }
__device__ __forceinline__ float copysign_(float m, float s) { return copysignf(m, s); }
__device__ __forceinline__ double fabs_(double x) { return fabs(x); }
__device__ __forceinline__ float fabs_(float x) { return fabsf(x); }
__device__ __forceinline__ double fmin_(double a, double b) { return fmin(a, b); }
__device__ __forceinline__ float fmin_(float a, float b) { return fminf(a, b); }

// minmod(theta dm, (dm+dp)/2, theta dp) = sign * min(theta min(|dm|,|dp|), |dm+dp|/2) when dm, dp share a sign
template <typename R>
__device__ __forceinline__ R minmod_fast(R dm, R dp, R theta) {
  const R m1 = fmin_(fabs_(dm), fabs_(dp));
  const R m = fmin_(theta * m1, R(0.5) * fabs_(dm + dp));
  return same_sign(dm, dp) ? copysign_(m, dm) : R(0);
}

// 2 (H_{i+1/2} - H_{i-1/2}) for one field (the factor 1/2 of Eq.41 is folded into the caller's scale)
template <typename R>
__device__ __forceinline__ R kt_div2(const R q[5], const R f[5], R cl, R cr, R theta) {
  const R dq0 = q[1] - q[0], dq1 = q[2] - q[1], dq2 = q[3] - q[2], dq3 = q[4] - q[3];
  const R df0 = f[1] - f[0], df1 = f[2] - f[1], df2 = f[3] - f[2], df3 = f[4] - f[3];
  const R hq1 = R(0.5) * minmod_fast(dq0, dq1, theta), hq2 = R(0.5) * minmod_fast(dq1, dq2, theta),
          hq3 = R(0.5) * minmod_fast(dq2, dq3, theta);
  const R hf1 = R(0.5) * minmod_fast(df0, df1, theta), hf2 = R(0.5) * minmod_fast(df1, df2, theta),
          hf3 = R(0.5) * minmod_fast(df2, df3, theta);
  const R Hr = ((f[3] - hf3) + (f[2] + hf2)) - cr * ((q[3] - hq3) - (q[2] + hq2));
  const R Hl = ((f[2] - hf2) + (f[1] + hf1)) - cl * ((q[2] - hq2) - (q[1] + hq1));
  return Hr - Hl;
}

// signal speeds of one cell along the three axes from u~ (A6); cs2 from the EoS at the cell
template <typename R>
__device__ __forceinline__ void signal_speeds3(R g, R ux, R uy, R un, R cs2, R& cx, R& cy, R& cn) {
  const R ig = R(1) / g;
  const R ig2 = ig * ig;                                  // 1 - v^2 = 1/gamma^2
  const R v2 = (ux * ux + uy * uy + un * un) * ig2;
  const R cs = sqrt_(cs2), omc = R(1) - cs2;
  const R D = R(1) / (R(1) - v2 * cs2), base = R(1) - v2 * cs2, csg = cs * ig;
  const R vx = ux * ig, vy = uy * ig, vn = un * ig;
  cx = (fabs_(vx) * omc + csg * sqrt_(max_(base - vx * vx * omc, R(0)))) * D;
  cy = (fabs_(vy) * omc + csg * sqrt_(max_(base - vy * vy * omc, R(0)))) * D;
  cn = (fabs_(vn) * omc + csg * sqrt_(max_(base - vn * vn * omc, R(0)))) * D;
}

// Root-find (Eq.51/54; A7, A8) with a warp-uniform iteration count: every lane runs the same number of
// Newton steps (the warp leaves the loop when all 32 lanes have converged), so there is no divergence.
// Must be called by all lanes of the warp.  Also returns P, c_s^2 at the root and u~^tau.
template <typename R>
__device__ __forceinline__ void rootfind_warp(const EosDev<R>& eos, R M0, R Mx, R My, R Mn, R e_start, int iters,
                                              R e_floor, R v_max, R& e_out, R& P_out, R& cs2_out, R& ux, R& uy,
                                              R& un, R& g_out, unsigned& flags) {
  if (!(M0 == M0) || !(Mx == Mx) || !(My == My) || !(Mn == Mn)) flags |= 8u;
  const bool vac = !(M0 > e_floor);
  if (vac) { flags |= 1u; M0 = R(1); Mx = My = Mn = R(0); }
  R M2 = Mx * Mx + My * My + Mn * Mn;
  const R lim = v_max * M0;
  if (M2 > lim * lim) {
    const R sc = lim * rsqrt_(M2);
    Mx *= sc; My *= sc; Mn *= sc; M2 = lim * lim; flags |= 2u;
  }
  R e, P, cs2;
  if (eos.kind == 0) {
    const R d = M0 * M0 - M2;
    e = R(3) * d / (M0 + sqrt_(M0 * M0 + R(3) * d));
    P = e * R(1.0 / 3.0); cs2 = R(1.0 / 3.0);
  } else {
    const R tol = (sizeof(R) == 8) ? R(1e-15) : R(2e-7);
    R lo = R(0), hi = M0;
    e = e_start;
    if (!(e > lo && e < hi)) e = M0 - M2 / (M0 + M0 * R(1.0 / 3.0));
    if (!(e > lo && e < hi)) e = R(0.5) * M0;
    for (int it = 0; it < iters; ++it) {
      eos_P(eos, e, P, cs2);
      const R inv = R(1) / (M0 + P);
      const R g = M0 - M2 * inv - e;
      const bool conv = !(abs_(g) > tol * M0);
      if (__all_sync(0xffffffffu, conv)) break;
      const R dg = M2 * cs2 * inv * inv - R(1);
      if (g > R(0)) lo = e; else hi = e;
      R en = e - g / dg;
      if (!(en >= lo && en <= hi)) en = R(0.5) * (lo + hi);
      e = conv ? e : en;
    }
    eos_P(eos, e, P, cs2);
    const R g = M0 - M2 / (M0 + P) - e;
    if (abs_(g) > R(1e3) * tol * M0) flags |= 4u;
  }
  if (vac) e = R(0);
  if (e < e_floor) {
    e = e_floor; flags |= 1u;
    eos_P(eos, e, P, cs2);
  }
  const R iw = R(1) / (M0 + P);
  const R vx = Mx * iw, vy = My * iw, vn = Mn * iw;
  const R gam = rsqrt_(R(1) - (vx * vx + vy * vy + vn * vn));
  ux = gam * vx; uy = gam * vy; un = gam * vn;
  e_out = e; P_out = P; cs2_out = cs2;
  // u~^tau consistent with the stored u~^i (what a consumer would recompute): sqrt(1 + u.u)
  g_out = sqrt_(R(1) + ux * ux + uy * uy + un * un);
}

// pi limiter (A14) with P(e) supplied
template <typename R>
__device__ __forceinline__ void limit_pi_P(R xi, R e, R P, R pi[10], unsigned& flags) {
  if (!(xi > R(0))) return;
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

template <typename R, bool VISC, int MODE>
__global__ void __launch_bounds__(256, 2) stage_fused_kernel(const StageArgs<R> a) {
  constexpr bool USE_PI = VISC && (MODE != 0);
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  const bool active = (i < a.nx) && (j < a.ny);
  const int ic = active ? i : 0, jc = active ? j : 0;
  const long long sf = a.sf;
  const long long c = (long long)k * a.sz + (long long)jc * a.px + ic;
  const R* __restrict__ in = a.in;
  const R* __restrict__ inx = a.in + a.xo;                  // extended slots of the input state

  // ---- cell-centre state ------------------------------------------------------------------------
  const R e_c = in[c];
  R ut[4];
  ut[1] = in[sf + c]; ut[2] = in[2 * sf + c]; ut[3] = in[3 * sf + c];
  ut[0] = inx[X_G * sf + c];
  const R P_c = inx[X_P * sf + c];
  R pic[10];
#pragma unroll
  for (int m = 0; m < 10; ++m) pic[m] = USE_PI ? in[(F_PI + m) * sf + c] : R(0);

  R S[14];
#pragma unroll
  for (int m = 0; m < 14; ++m) S[m] = R(0);
  R grad[4][4];
#pragma unroll
  for (int m = 0; m < 4; ++m)
#pragma unroll
    for (int n = 0; n < 4; ++n) grad[m][n] = R(0);
  R cfl0 = R(0), cfl1 = R(0), cfl2 = R(0);
  const R tf = a.milne ? a.tau : R(1);

  // ---- KT flux divergence, axes x, y, eta (Eq.40; A22) -------------------------------------------
#pragma unroll 1
  for (int ax = 0; ax < 3; ++ax) {
    const int n_ax = ax == 0 ? a.nx : (ax == 1 ? a.ny : a.nz);
    const int pos = ax == 0 ? ic : (ax == 1 ? jc : k);
    const long long stride = ax == 0 ? 1 : (ax == 1 ? (long long)a.px : a.sz);
    const long long base = c - (long long)pos * stride;
    long long idx[5];
#pragma unroll
    for (int p = 0; p < 5; ++p) idx[p] = base + (long long)bmap(pos + p - 2, n_ax, a.bc[ax]) * stride;
    const R* __restrict__ cax = inx + (X_CX + ax) * sf;   // signal speed along this axis
    const R* __restrict__ uax = in + (1 + ax) * sf;        // u~^a

    R g[5], ua[5];
    R cl, cr;
    {
      const R c1 = cax[idx[1]], c2 = cax[idx[2]], c3 = cax[idx[3]];
      cl = max_(c1, c2); cr = max_(c2, c3);
      const R cv = c2 * a.h * a.scale[ax];
      if (ax == 0) cfl0 = cv; else if (ax == 1) cfl1 = cv; else cfl2 = cv;
    }
#pragma unroll
    for (int p = 0; p < 5; ++p) { g[p] = inx[X_G * sf + idx[p]]; ua[p] = uax[idx[p]]; }
    const R sc_pi = R(0.5) * a.scale[ax], sc_T = sc_pi * tf;

    {
      // T fields: Q^mu/tau = T_f^{tau mu}, F_a^mu/tau = T_f^{a mu}   (Eq.27, Eq.39)
      R wq[5], wa[5], Pp[5], uu[3][5];
#pragma unroll
      for (int p = 0; p < 5; ++p) {
        Pp[p] = inx[X_P * sf + idx[p]];
        const R w = in[idx[p]] + Pp[p];
        wq[p] = w * g[p]; wa[p] = w * ua[p];
        uu[0][p] = in[sf + idx[p]]; uu[1][p] = in[2 * sf + idx[p]]; uu[2][p] = in[3 * sf + idx[p]];
      }
#pragma unroll
      for (int mu = 0; mu < 4; ++mu) {
        R q[5], f[5];
        const R* __restrict__ pt = in + (F_PI + c_pidx[0][mu]) * sf;
        const R* __restrict__ pa = in + (F_PI + c_pidx[ax + 1][mu]) * sf;
#pragma unroll
        for (int p = 0; p < 5; ++p) {
          const R umu = mu == 0 ? g[p] : uu[mu == 0 ? 0 : mu - 1][p];
          R tq = wq[p] * umu - (mu == 0 ? Pp[p] : R(0));
          R tfl = wa[p] * umu + (mu == ax + 1 ? Pp[p] : R(0));
          if (USE_PI) { tq += pt[idx[p]]; tfl += pa[idx[p]]; }
          q[p] = tq; f[p] = tfl;
        }
        S[mu] -= kt_div2(q, f, cl, cr, a.theta) * sc_T;
      }
      if (USE_PI) {
        // spatial rows of nabla~_mu u~^nu by central differences (A9); eta row divided by tau (Eq.22)
        const R d0 = (g[3] - g[1]) * sc_pi, d1 = (uu[0][3] - uu[0][1]) * sc_pi, d2 = (uu[1][3] - uu[1][1]) * sc_pi,
                d3 = (uu[2][3] - uu[2][1]) * sc_pi;
#pragma unroll
        for (int r = 0; r < 3; ++r)
          if (ax == r) { grad[r + 1][0] = d0; grad[r + 1][1] = d1; grad[r + 1][2] = d2; grad[r + 1][3] = d3; }
      }
    }
    // pi fields: Q = u^tau pi, F_a = u^a pi   (Eq.29)
    if (USE_PI) {
#pragma unroll
      for (int m = 0; m < 10; ++m) {
        const R* __restrict__ pm = in + (F_PI + m) * sf;
        R q[5], f[5];
#pragma unroll
        for (int p = 0; p < 5; ++p) {
          const R v = pm[idx[p]];
          q[p] = g[p] * v; f[p] = ua[p] * v;
        }
        S[4 + m] -= kt_div2(q, f, cl, cr, a.theta) * sc_pi;
      }
    }
  }

  // ---- geometric source of T (Eq.31, sign A1) ---------------------------------------------------
  const R w_c = e_c + P_c;
  if (a.milne) {
    S[0] -= w_c * ut[3] * ut[3] + P_c + pic[9];      // -T_f^{eta eta}
    S[3] -= w_c * ut[0] * ut[3] + pic[3];            // -T_f^{tau eta}
  }

  // ---- state n at the centre (MODE 2 reads it; MODE 0/1: it is the star centre itself) -----------
  R e_n = e_c, un_[4] = {ut[0], ut[1], ut[2], ut[3]}, pin[10], P_n = P_c;
#pragma unroll
  for (int m = 0; m < 10; ++m) pin[m] = pic[m];
  if (MODE == 2) {
    const R* __restrict__ sn = a.sn;
    e_n = sn[c];
    un_[1] = sn[sf + c]; un_[2] = sn[2 * sf + c]; un_[3] = sn[3 * sf + c];
    un_[0] = sn[a.xo + X_G * sf + c];
    P_n = sn[a.xo + X_P * sf + c];
#pragma unroll
    for (int m = 0; m < 10; ++m) pin[m] = VISC ? sn[(F_PI + m) * sf + c] : R(0);
  }

  R gdiv = R(1), gst = R(1);
  if (USE_PI) {
    if (MODE == 1) {
      const R* __restrict__ up = a.uprev;
      const R sx = R(2) * ut[1] - up[c], sy = R(2) * ut[2] - up[sf + c], sn_ = R(2) * ut[3] - up[2 * sf + c];
      const R gs2 = R(1) + sx * sx + sy * sy + sn_ * sn_;
      gst = sqrt_(gs2);
      const R g2 = R(1) + ut[1] * ut[1] + ut[2] * ut[2] + ut[3] * ut[3];
      grad[0][0] = (gs2 - g2) / (gst + ut[0]) * a.inv_h;      // (u*^tau - u^tau)/h without cancellation
      grad[0][1] = (sx - ut[1]) * a.inv_h; grad[0][2] = (sy - ut[2]) * a.inv_h; grad[0][3] = (sn_ - ut[3]) * a.inv_h;
      gdiv = gst;
    } else {
      gst = a.gstar[c];
      const R g12 = R(1) + ut[1] * ut[1] + ut[2] * ut[2] + ut[3] * ut[3];
      const R gn2 = R(1) + un_[1] * un_[1] + un_[2] * un_[2] + un_[3] * un_[3];
      grad[0][0] = (g12 - gn2) / (ut[0] + un_[0]) * a.inv_h;
      grad[0][1] = (ut[1] - un_[1]) * a.inv_h; grad[0][2] = (ut[2] - un_[2]) * a.inv_h;
      grad[0][3] = (ut[3] - un_[3]) * a.inv_h;
      gdiv = ut[0];
    }
    if (a.milne) {
      grad[3][0] += ut[3] * a.inv_tau;    // Eq.25
      grad[3][3] += ut[0] * a.inv_tau;    // Eq.26
    }
    const R T_c = eos_T(a.eos, e_c);
    is_source(ut, grad, pic, e_c, P_c, T_c, a.inv_5etas_hbarc, a.milne != 0, a.inv_tau, S + 4);
  }

  const R w_n = e_n + P_n;
  R QTn[4];
  QTn[0] = a.tf_n * (w_n * un_[0] * un_[0] - P_n + pin[0]);
  QTn[1] = a.tf_n * (w_n * un_[0] * un_[1] + pin[1]);
  QTn[2] = a.tf_n * (w_n * un_[0] * un_[2] + pin[2]);
  QTn[3] = a.tf_n * (w_n * un_[0] * un_[3] + pin[3]);

  R pnew[10], M[4];
  const R ig = R(1) / gdiv;
  if (MODE != 2) {
#pragma unroll
    for (int m = 0; m < 10; ++m) pnew[m] = USE_PI ? (un_[0] * pin[m] + a.h * S[4 + m]) * ig : R(0);    // Eq.49
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) M[mu] = (QTn[mu] + a.h * S[mu]) * a.inv_tf_1 - pnew[mu];              // Eq.50-51
  } else {
#pragma unroll
    for (int m = 0; m < 10; ++m)
      pnew[m] = USE_PI ? R(0.5) * (un_[0] * pin[m] + gst * pic[m] + a.h * S[4 + m]) * ig : R(0);         // Eq.52
    R QT1[4];
    QT1[0] = a.tf_1 * (w_c * ut[0] * ut[0] - P_c + pic[0]);
    QT1[1] = a.tf_1 * (w_c * ut[0] * ut[1] + pic[1]);
    QT1[2] = a.tf_1 * (w_c * ut[0] * ut[2] + pic[2]);
    QT1[3] = a.tf_1 * (w_c * ut[0] * ut[3] + pic[3]);
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) M[mu] = R(0.5) * (QTn[mu] + QT1[mu] + a.h * S[mu]) * a.inv_tf_1 - pnew[mu];  // Eq.53-54
  }

  // ---- root-find (Eq.51/54), warp-uniform iteration count --------------------------------------------
  unsigned flags = 0;
  R e_new, P_new, cs2_new, ux_new, uy_new, un_new, g_new;
  rootfind_warp(a.eos, M[0], M[1], M[2], M[3], e_c, a.root_iters, a.e_floor, a.v_max, e_new, P_new, cs2_new, ux_new,
                uy_new, un_new, g_new, flags);
  if (USE_PI) limit_pi_P(a.xi, e_new, P_new, pnew, flags);

  // ---- write state + extended slots ----------------------------------------------------------------
  if (active) {
    R* __restrict__ out = a.out;
    if (MODE == 0) {
      out[c] = R(2) * ut[1] - ux_new; out[sf + c] = R(2) * ut[2] - uy_new; out[2 * sf + c] = R(2) * ut[3] - un_new;
    } else {
      R cx, cy, cn;
      signal_speeds3(g_new, ux_new, uy_new, un_new, cs2_new, cx, cy, cn);
      out[c] = e_new; out[sf + c] = ux_new; out[2 * sf + c] = uy_new; out[3 * sf + c] = un_new;
      if (VISC) {
#pragma unroll
        for (int m = 0; m < 10; ++m) out[(F_PI + m) * sf + c] = pnew[m];
        if (MODE == 1) a.gstar[c] = gst;
      }
      R* __restrict__ ox = out + a.xo;
      ox[X_P * sf + c] = P_new; ox[X_G * sf + c] = g_new;
      ox[X_CX * sf + c] = cx; ox[X_CY * sf + c] = cy; ox[X_CN * sf + c] = cn;
    }
  }

  // ---- reductions (row a10) --------------------------------------------------------------------------
  if (MODE != 0) {
    if (!active) flags = 0;
    count_flags(a.diag, flags);
    const int lane = (threadIdx.x + threadIdx.y * blockDim.x) & 31;
    if (MODE == 1) {
      const double r0 = warp_max(active ? (double)cfl0 : 0.0), r1 = warp_max(active ? (double)cfl1 : 0.0),
                   r2 = warp_max(active ? (double)cfl2 : 0.0);
      if (lane == 0) {
        atomic_max_nonneg(&a.diag->cfl[a.slot][0], r0);
        atomic_max_nonneg(&a.diag->cfl[a.slot][1], r1);
        atomic_max_nonneg(&a.diag->cfl[a.slot][2], r2);
      }
    } else {
      const double r = warp_max(active ? (double)e_new : 0.0);
      if (lane == 0) atomic_max_nonneg(&a.diag->emax[a.slot], r);
    }
    if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && threadIdx.x == 0 && threadIdx.y == 0) {
      if (MODE == 1) a.diag->emax[a.slot] = 0ull;
      else { a.diag->cfl[a.slot ^ 1][0] = 0ull; a.diag->cfl[a.slot ^ 1][1] = 0ull; a.diag->cfl[a.slot ^ 1][2] = 0ull; }
    }
  }
}

template <typename R, bool VISC, int MODE>
void launch_stage_tiled(const StageArgs<R>& a, cudaStream_t stream) {
  dim3 block(32, 8, 1);
  dim3 grid((a.nx + 31) / 32, (a.ny + 7) / 8, a.nz);
  stage_fused_kernel<R, VISC, MODE><<<grid, block, 0, stream>>>(a);
}

}  // namespace clv
