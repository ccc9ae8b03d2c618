// hydro_stage_update.cuh -- the per-cell tail of an RK2 stage, shared by the stage kernels.
//
// Given the KT flux divergence S_KT (14 words) of a cell, this adds the geometric source of T (Eq.31), forms the time
// row of nabla~_mu u~^nu (A10), adds the Israel-Stewart source (Eq.33-38), applies the stage update (Eq.49-54 in the
// Shu-Osher bookkeeping, A26), runs the root-find (Eq.51/54) and the pi limiter (A14).
// One copy of this bookkeeping serves the fused per-cell kernel (hydro_stage_fused.cuh) and the tile kernel
// (hydro_stage_tile.cuh).
//   MODE 1: RHS on state n at tau_n, time derivative from u* = 2u^n - u^{n-1}; produces state ' and u*^tau.
//   MODE 2: RHS on state ' at tau_{n+1}, time derivative (u' - u^n)/h; Heun average; produces state n+1.
//   MODE 0: bootstrap of u^{-1} (A23): ideal-fluid Euler predictor (pi dropped).
#pragma once
#include "hydro_device.cuh"

namespace clv {

template <typename R>
struct Cell {
  R e, P;
  R u[4];      // u~^mu, u[0] = u~^tau
  R pi[10];
  R Pi, nb;    // bulk pressure, net-baryon density (used by the extended kernels only)
};

// A: any argument struct with the members milne, inv_tau, tf_n, tf_1, inv_tf_1, h, inv_h, xi, e_floor, v_max,
// root_iters, inv_5etas_hbarc, inv_ctau, lam1, eos.
//   S[14]      in: S_KT (T fields 0..3, pi fields 4..13); clobbered
//   c          the state the RHS was evaluated on (n in MODE 0/1, ' in MODE 2)
//   n          state n at the cell (MODE 2; ignored otherwise)
//   grad       rows 1..3 = spatial rows of nabla~_mu u~^nu (eta row already divided by tau); row 0 is filled here
//   up[3]      MODE 1: u~^i at n-1;  gst: MODE 1 out: u*^tau, MODE 2 in: u*^tau of stage 1
//   o          out: new e, P, u~, pi~;  cs2_o: c_s^2 at the new e
// Root-find (Eq.51/54; A7, A8) with a warp-uniform iteration count: every lane runs the same number of
// Newton steps (the warp leaves the loop when all 32 lanes have converged), so there is no divergence
// (the paper's "no way to tackle").  Must be called by all lanes of the warp.  Also returns
// P, c_s^2 at the root and u~^tau.
// Pib: bulk pressure carried through the root-find, e = M0 - M^2/(M0 + max(P(e) + Pi, 0)); P_out and
// cs2_out stay those of P(e).
template <typename R>
__device__ __forceinline__ void rootfind_warp(const EosDev<R>& eos, R M0, R Mx, R My, R Mn, R e_start, int iters,
                                              R e_floor, R v_max, R& e_out, R& P_out, R& cs2_out, R& ux, R& uy,
                                              R& un, R& g_out, unsigned& flags, R Pib = R(0), bool with_bulk = false) {
  if (!(M0 == M0) || !(Mx == Mx) || !(My == My) || !(Mn == Mn)) flags |= 8u;
  const bool vac = !(M0 > e_floor);
  if (vac) { flags |= 1u; M0 = R(1); Mx = My = Mn = R(0); }
  R M2 = Mx * Mx + My * My + Mn * Mn;
  const R lim = v_max * M0;
  if (M2 > lim * lim) {
    const R sc = lim * frsqrt_(M2);
    Mx *= sc; My *= sc; Mn *= sc; M2 = lim * lim; flags |= 2u;
  }
  R e, P, cs2;
  if (eos.kind == 0 && !with_bulk) {
    const R d = M0 * M0 - M2;
    e = R(3) * d * frcp_(M0 + fsqrt_(M0 * M0 + R(3) * d));
    P = e * R(1.0 / 3.0); cs2 = R(1.0 / 3.0);
  } else {
    const R tol = (sizeof(R) == 8) ? R(1e-15) : R(2e-7);
    const R tol2 = (sizeof(R) == 8) ? R(1e-9) : R(1e-4);
    R lo = R(0), hi = M0;
    e = e_start;
    if (!(e > lo && e < hi)) e = M0 - M2 * frcp_(M0 + M0 * R(1.0 / 3.0));
    if (!(e > lo && e < hi)) e = R(0.5) * M0;
    for (int it = 0; it < iters; ++it) {
      eos_P(eos, e, P, cs2);
      R Pt = P;
      if (with_bulk) { Pt = P + Pib; if (Pt < R(0)) { Pt = R(0); cs2 = R(0); } }      // A32: max(P + Pi, 0)
      const R inv = frcp_(M0 + Pt);
      const R g = M0 - M2 * inv - e;
      const bool conv = !(abs_(g) > tol * M0);
      if (__all_sync(0xffffffffu, conv)) break;
      const R dg = M2 * cs2 * inv * inv - R(1);
      if (g > R(0)) lo = e; else hi = e;
      R en = e - g * frcp_(dg);
      if (!(en >= lo && en <= hi)) en = R(0.5) * (lo + hi);
      e = conv ? e : en;
      // Newton converges quadratically on the (piecewise linear, convex) g: a step taken from a residual
      // below sqrt(tol) lands below tol, so the warp can leave without another evaluation
      if (__all_sync(0xffffffffu, !(abs_(g) > tol2 * M0))) break;
    }
    eos_P(eos, e, P, cs2);
    const R g = M0 - M2 * frcp_(M0 + (with_bulk ? max_(P + Pib, R(0)) : P)) - e;
    if (abs_(g) > R(1e3) * tol * M0) flags |= 4u;
  }
  if (vac) e = R(0);
  if (e < e_floor) {
    e = e_floor; flags |= 1u;
    eos_P(eos, e, P, cs2);
  }
  const R iw = frcp_(M0 + (with_bulk ? max_(P + Pib, R(0)) : P));
  const R vx = Mx * iw, vy = My * iw, vn = Mn * iw;
  const R gam = frsqrt_(R(1) - (vx * vx + vy * vy + vn * vn));
  ux = gam * vx; uy = gam * vy; un = gam * vn;
  e_out = e; P_out = P; cs2_out = cs2;
  // u~^tau consistent with the stored u~^i (what a consumer would recompute): sqrt(1 + u.u)
  g_out = fsqrt_(R(1) + ux * ux + uy * uy + un * un);
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
    const R r = fsqrt_(lim2 * frcp_(mag2));
#pragma unroll
    for (int m = 0; m < 10; ++m) pi[m] *= r;
    flags |= 16u;
  }
}

// XT: S[14], S[15] hold the KT divergences of (u~^tau Pi, u~^a Pi) and of (n u~^tau, n u~^a); tf_rhs is the
// factor tau of the RHS evaluation that turns the latter into S_N,tot (A31); c.Pi, c.nb, n.Pi, n.nb are read and o.Pi,
// o.nb written; a.zeta_over_eta = (zeta/s)/(eta_v/s) (A30).
template <typename R, bool VISC, int MODE, bool XT = false, typename A>
__device__ __forceinline__ void stage_update(const A& a, R S[], const Cell<R>& c, const Cell<R>& n, R grad[4][4],
                                             const R up[3], R& gst, Cell<R>& o, R& cs2_o, unsigned& flags,
                                             R tf_rhs = R(1)) {
  constexpr bool USE_PI = VISC && (MODE != 0);
  const R* ut = c.u;
  // ---- geometric source of T (Eq.31, sign A1) ---------------------------------------------------
  const R Pc = XT ? c.P + c.Pi : c.P;       // A28: P + Pi wherever the pressure enters T_f
  const R w_c = c.e + Pc;
  if (a.milne) {
    S[0] -= w_c * ut[3] * ut[3] + Pc + (USE_PI ? c.pi[9] : R(0));      // -T_f^{eta eta}
    S[3] -= w_c * ut[0] * ut[3] + (USE_PI ? c.pi[3] : R(0));            // -T_f^{tau eta}
  }
  // state n at the centre: the RHS state itself in MODE 0/1
  const Cell<R>& sn = (MODE == 2) ? n : c;

  R gdiv = R(1);      // u~^tau that divides Q_pi in this stage (A11)
  if (USE_PI) {
    // time row of the gradient (A10)
    if (MODE == 1) {
      const R sx = R(2) * ut[1] - up[0], sy = R(2) * ut[2] - up[1], sn_ = R(2) * ut[3] - up[2];
      const R gs2 = R(1) + sx * sx + sy * sy + sn_ * sn_;
      gst = fsqrt_(gs2);
      const R g2 = R(1) + ut[1] * ut[1] + ut[2] * ut[2] + ut[3] * ut[3];
      grad[0][0] = (gs2 - g2) * frcp_(gst + ut[0]) * a.inv_h;      // (u*^tau - u^tau)/h without cancellation
      grad[0][1] = (sx - ut[1]) * a.inv_h; grad[0][2] = (sy - ut[2]) * a.inv_h; grad[0][3] = (sn_ - ut[3]) * a.inv_h;
      gdiv = gst;
    } else {
      const R g12 = R(1) + ut[1] * ut[1] + ut[2] * ut[2] + ut[3] * ut[3];
      const R gn2 = R(1) + sn.u[1] * sn.u[1] + sn.u[2] * sn.u[2] + sn.u[3] * sn.u[3];
      grad[0][0] = (g12 - gn2) * frcp_(ut[0] + sn.u[0]) * a.inv_h;
      grad[0][1] = (ut[1] - sn.u[1]) * a.inv_h; grad[0][2] = (ut[2] - sn.u[2]) * a.inv_h;
      grad[0][3] = (ut[3] - sn.u[3]) * a.inv_h;
      gdiv = ut[0];
    }
    if (a.milne) {
      grad[3][0] += ut[3] * a.inv_tau;    // Eq.25
      grad[3][3] += ut[0] * a.inv_tau;    // Eq.26
    }
    const R T_c = eos_T(a.eos, c.e);
    is_source(ut, grad, c.pi, c.e, c.P, T_c, a.inv_5etas_hbarc, a.milne != 0, a.inv_tau, S + 4, a.inv_ctau, a.lam1);
    if constexpr (XT) {   // S_Pi (A29, A30): -(Pi + zeta theta)/tau_Pi - Pi theta / 3 - u~^tau Pi / tau, tau_Pi = tau_pi
      const R theta = grad[0][0] + grad[1][1] + grad[2][2] + grad[3][3];
      R src = -c.Pi * (T_c * a.inv_5etas_hbarc) - a.zeta_over_eta * ((c.e + c.P) * a.inv_ctau) * theta -
              c.Pi * theta * R(1.0 / 3.0);
      if (a.milne) src -= c.Pi * ut[0] * a.inv_tau;
      S[14] += src;
    }
  }

  // Q_T^n = tf_n T_f^{tau mu}(state n)
  const R Pn = XT ? sn.P + sn.Pi : sn.P;
  const R w_n = sn.e + Pn;
  R QTn[4];
  QTn[0] = a.tf_n * (w_n * sn.u[0] * sn.u[0] - Pn + (USE_PI ? sn.pi[0] : R(0)));
  QTn[1] = a.tf_n * (w_n * sn.u[0] * sn.u[1] + (USE_PI ? sn.pi[1] : R(0)));
  QTn[2] = a.tf_n * (w_n * sn.u[0] * sn.u[2] + (USE_PI ? sn.pi[2] : R(0)));
  QTn[3] = a.tf_n * (w_n * sn.u[0] * sn.u[3] + (USE_PI ? sn.pi[3] : R(0)));

  R M[4];
  const R ig = frcp_(gdiv);
  R Pb = R(0), QN = R(0);      // 8(f)-3: predicted / averaged Pi and Q_N (A26 bookkeeping, like pi and Q_T)
  if (XT) {
    const R QNn = a.tf_n * sn.nb * sn.u[0];
    if (MODE != 2) {
      Pb = (sn.u[0] * sn.Pi + a.h * S[14]) * ig;
      QN = QNn + a.h * tf_rhs * S[15];
    } else {
      Pb = R(0.5) * (sn.u[0] * sn.Pi + gst * c.Pi + a.h * S[14]) * ig;
      QN = R(0.5) * (QNn + a.tf_1 * c.nb * ut[0] + a.h * tf_rhs * S[15]);
    }
  }
  if (MODE != 2) {
#pragma unroll
    for (int m = 0; m < 10; ++m) o.pi[m] = USE_PI ? (sn.u[0] * sn.pi[m] + a.h * S[4 + m]) * ig : R(0);   // Eq.49
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) M[mu] = (QTn[mu] + a.h * S[mu]) * a.inv_tf_1 - o.pi[mu];              // Eq.50-51
  } else {
    // Eq.52-54 in Shu-Osher form (A26): Q^{n+1} = 1/2 [Q^n + Q(state') + h S(state')]
#pragma unroll
    for (int m = 0; m < 10; ++m)
      o.pi[m] = USE_PI ? R(0.5) * (sn.u[0] * sn.pi[m] + gst * c.pi[m] + a.h * S[4 + m]) * ig : R(0);     // Eq.52
    R QT1[4];
    QT1[0] = a.tf_1 * (w_c * ut[0] * ut[0] - Pc + (USE_PI ? c.pi[0] : R(0)));
    QT1[1] = a.tf_1 * (w_c * ut[0] * ut[1] + (USE_PI ? c.pi[1] : R(0)));
    QT1[2] = a.tf_1 * (w_c * ut[0] * ut[2] + (USE_PI ? c.pi[2] : R(0)));
    QT1[3] = a.tf_1 * (w_c * ut[0] * ut[3] + (USE_PI ? c.pi[3] : R(0)));
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) M[mu] = R(0.5) * (QTn[mu] + QT1[mu] + a.h * S[mu]) * a.inv_tf_1 - o.pi[mu];  // Eq.53-54
  }

  // ---- root-find (Eq.51/54), warp-uniform iteration count; pi limiter (A14) -----------------------
  rootfind_warp(a.eos, M[0], M[1], M[2], M[3], c.e, a.root_iters, a.e_floor, a.v_max, o.e, o.P, cs2_o, o.u[1], o.u[2],
                o.u[3], o.u[0], flags, Pb, XT);
  if (USE_PI) limit_pi_P(a.xi, o.e, o.P, o.pi, flags);
  if (XT) {
    if (a.xi > R(0)) {      // bulk limiter (A32): |Pi| <= xi P(e)
      const R lim = a.xi * o.P;
      if (abs_(Pb) > lim) Pb = Pb < R(0) ? -lim : lim;
    }
    o.Pi = Pb;
    // n = Q_N / (tau u~^tau) with u~^tau = sqrt(1 + u.u) of the new velocity
    o.nb = QN * a.inv_tf_1 * frcp_(o.u[0]);
  }
}

}  // namespace clv
