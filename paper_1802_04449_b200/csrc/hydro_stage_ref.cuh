// hydro_stage_ref.cuh -- "kernel 1": one thread per cell, 13-point star read straight from global
// memory through L1/L2.  Every step of the RK2 stage is fused in this one kernel (KT fluxes on three
// axes for 4 + 10 fields, geometric source, velocity gradients, Israel-Stewart source, stage update,
// root-find, pi limiter, CFL / e_max reductions): one launch per stage.  It is the simple, obviously
// structured CUDA statement of the method; the fused extended-state kernel (hydro_stage_fused.cuh) must agree with it.
//
// Stages (Eq.49-54; A10-A12, A26):
//   MODE 1: RHS on state n at tau_n, time derivative from u* = 2u^n - u^{n-1}; writes state ' and u*^tau.
//   MODE 2: RHS on state ' at tau_{n+1}, time derivative (u' - u^n)/h; Heun average; writes state n+1.
//   MODE 0: bootstrap of u^{-1} (A23): ideal-fluid Euler predictor, writes 2u^0 - u_id^1.
#pragma once
#include "hydro_device.cuh"

namespace clv {

template <typename R>
struct StageArgs {
  int nx, ny, nz;        // cells along x, y, eta_s
  // state-buffer layout [k][j][x-block][field][32]: element (field m, cell i,j,k) sits at
  //   k*sz + j*sy + (i>>5)*blk + m*32 + (i&31);   blk = 32 * (fields per buffer)
  int blk;               // elements per x-block (32 cells x all fields of the buffer)
  int gp;                // row pitch of the single-field gstar array (= 32 * x-blocks)
  long long sy, sz;      // row stride, plane stride (elements)
  int bc[3];             // 0 clamp (zero-gradient outflow), 1 periodic
  int milne;
  R tau, inv_tau;        // time level of this RHS evaluation
  R tf_n, tf_1;          // tau_n, tau_{n+1}   (both 1 in Cartesian mode)
  R inv_tf_1;
  R h, inv_h;
  R scale[3];            // 1/dx, 1/dy, 1/(tau deta)  (Eq.40)
  R theta, e_floor, xi, v_max;
  R inv_5etas_hbarc;     // 1/(c_tau (eta_v/s) hbarc), c_tau = 5 unless set (tau_pi = c_tau eta_v/(T s))
  R inv_ctau, lam1;      // 1/c_tau; lambda1_hat (lambda_1 = lambda1_hat / e)
  R zeta_over_eta;       // (zeta/s)/(eta_v/s); 0 without the extension
  int root_iters;
  const R* in;           // state whose 13-point star is read
  const R* sn;           // MODE 2: state n (cell centre only)
  const R* uprev;        // MODE 1: u~^i at n-1, 3 fields with stride sf
  R* gstar;              // u*^tau: written by MODE 1, read by MODE 2
  R* out;                // MODE 1: state '; MODE 2: state n+1; MODE 0: history (3 fields, stride sf)
  EosDev<R> eos;
  DiagDev* diag;
  int slot;              // parity slot of the per-step maxima
};

constexpr int FS = 32;   // field stride inside an x-block (elements)

__device__ __forceinline__ int bmap(int i, int n, int periodic) {
  if (periodic) { i = i % n; return i < 0 ? i + n : i; }
  return min(max(i, 0), n - 1);
}
__device__ __forceinline__ long long xoff(int i, int blk) { return (long long)(i >> 5) * blk + (i & 31); }
// offsets of the five points pos-2..pos+2 along axis ax through cell (i,j,k), boundary rule a11 applied
template <typename A>
__device__ __forceinline__ void star_offsets(const A& a, int ax, int i, int j, int k, long long idx[5]) {
#pragma unroll
  for (int p = 0; p < 5; ++p) {
    const int d = p - 2;
    const int ii = ax == 0 ? bmap(i + d, a.nx, a.bc[0]) : i;
    const int jj = ax == 1 ? bmap(j + d, a.ny, a.bc[1]) : j;
    const int kk = ax == 2 ? bmap(k + d, a.nz, a.bc[2]) : k;
    idx[p] = (long long)kk * a.sz + (long long)jj * a.sy + xoff(ii, a.blk);
  }
}

template <typename R, bool VISC, int MODE>
__global__ void __launch_bounds__(256) stage_ref_kernel(const StageArgs<R> a) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  const bool active = (i < a.nx) && (j < a.ny);
  const int ic = active ? i : 0, jc = active ? j : 0;
  const long long c = (long long)k * a.sz + (long long)jc * a.sy + xoff(ic, a.blk);
  const long long cg = ((long long)k * a.ny + jc) * a.gp + ic;      // gstar index
  const R* __restrict__ in = a.in;
  constexpr long long sf = FS;
  constexpr bool USE_PI = VISC && (MODE != 0);

  // ---- cell-centre state -------------------------------------------------------------------
  const R e_c = in[c];
  R ut[4];
  ut[1] = in[sf + c]; ut[2] = in[2 * sf + c]; ut[3] = in[3 * sf + c];
  ut[0] = sqrt_(R(1) + ut[1] * ut[1] + ut[2] * ut[2] + ut[3] * ut[3]);
  R pic[10];
#pragma unroll
  for (int m = 0; m < 10; ++m) pic[m] = USE_PI ? in[(F_PI + m) * sf + c] : R(0);
  R P_c, cs2_c;
  eos_P(a.eos, e_c, P_c, cs2_c);

  R S[14];
#pragma unroll
  for (int m = 0; m < 14; ++m) S[m] = R(0);
  R grad[4][4];
#pragma unroll
  for (int m = 0; m < 4; ++m)
#pragma unroll
    for (int n = 0; n < 4; ++n) grad[m][n] = R(0);
  R cfl0 = R(0), cfl1 = R(0), cfl2 = R(0);

  // ---- KT flux divergence, axes x, y, eta in this order (Eq.40; A22) ---------------------------
#pragma unroll 1
  for (int ax = 0; ax < 3; ++ax) {
    long long idx[5];
    star_offsets(a, ax, ic, jc, k, idx);

    R w[5], Pp[5], g[5], ux[5], uy[5], un[5], ua[5], cs[5];
#pragma unroll
    for (int p = 0; p < 5; ++p) {
      const R e = in[idx[p]];
      ux[p] = in[sf + idx[p]]; uy[p] = in[2 * sf + idx[p]]; un[p] = in[3 * sf + idx[p]];
      ua[p] = ax == 0 ? ux[p] : (ax == 1 ? uy[p] : un[p]);
      const R u2 = ux[p] * ux[p] + uy[p] * uy[p] + un[p] * un[p];
      g[p] = sqrt_(R(1) + u2);
      R cs2;
      eos_P(a.eos, e, Pp[p], cs2);
      w[p] = e + Pp[p];
      const R ig = R(1) / g[p];
      cs[p] = signal_speed(ua[p] * ig, u2 * ig * ig, cs2);
    }
    const R cl = max_(cs[1], cs[2]), cr = max_(cs[2], cs[3]);
    {
      const R cv = cs[2] * a.h * a.scale[ax];
      if (ax == 0) cfl0 = cv; else if (ax == 1) cfl1 = cv; else cfl2 = cv;
    }
    const R tf = a.milne ? a.tau : R(1);

    // T fields: Q^mu = tf T_f^{tau mu}, F_a^mu = tf T_f^{a mu}   (Eq.27, Eq.39)
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
      R q[5], f[5];
      const int ip_t = c_pidx[0][mu], ip_a = c_pidx[ax + 1][mu];
#pragma unroll
      for (int p = 0; p < 5; ++p) {
        const R umu = mu == 0 ? g[p] : (mu == 1 ? ux[p] : (mu == 2 ? uy[p] : un[p]));
        R tq = w[p] * g[p] * umu - (mu == 0 ? Pp[p] : R(0));
        R tfl = w[p] * ua[p] * umu + (mu == ax + 1 ? Pp[p] : R(0));
        if (USE_PI) {
          tq += in[(F_PI + ip_t) * sf + idx[p]];
          tfl += in[(F_PI + ip_a) * sf + idx[p]];
        }
        q[p] = tf * tq; f[p] = tf * tfl;
      }
      S[mu] -= kt_div(q, f, cl, cr, a.theta) * a.scale[ax];
    }
    // pi fields: Q = u^tau pi, F_a = u^a pi   (Eq.29)
    if (USE_PI) {
#pragma unroll
      for (int m = 0; m < 10; ++m) {
        R q[5], f[5];
#pragma unroll
        for (int p = 0; p < 5; ++p) {
          const R v = in[(F_PI + m) * sf + idx[p]];
          q[p] = g[p] * v; f[p] = ua[p] * v;
        }
        S[4 + m] -= kt_div(q, f, cl, cr, a.theta) * a.scale[ax];
      }
      // spatial rows of nabla~_mu u~^nu by central differences (A9); eta row divided by tau (Eq.22)
      const R inv2d = R(0.5) * a.scale[ax];
      const R d0 = (g[3] - g[1]) * inv2d, d1 = (ux[3] - ux[1]) * inv2d, d2 = (uy[3] - uy[1]) * inv2d,
              d3 = (un[3] - un[1]) * inv2d;
#pragma unroll
      for (int r = 0; r < 3; ++r)
        if (ax == r) { grad[r + 1][0] = d0; grad[r + 1][1] = d1; grad[r + 1][2] = d2; grad[r + 1][3] = d3; }
    }
  }

  // ---- geometric source of T (Eq.31, sign A1) -------------------------------------------------
  const R w_c = e_c + P_c;
  if (a.milne) {
    S[0] -= w_c * ut[3] * ut[3] + P_c + pic[9];      // -T_f^{eta eta}
    S[3] -= w_c * ut[0] * ut[3] + pic[3];            // -T_f^{tau eta}
  }

  // ---- stage bookkeeping -------------------------------------------------------------------------
  // state n at the centre (MODE 2 reads it; MODE 0/1 it is the star centre itself)
  R e_n = e_c, un_[4] = {ut[0], ut[1], ut[2], ut[3]}, pin[10], P_n = P_c;
#pragma unroll
  for (int m = 0; m < 10; ++m) pin[m] = pic[m];
  if (MODE == 2) {
    const R* __restrict__ sn = a.sn;
    e_n = sn[c];
    un_[1] = sn[sf + c]; un_[2] = sn[2 * sf + c]; un_[3] = sn[3 * sf + c];
    un_[0] = sqrt_(R(1) + un_[1] * un_[1] + un_[2] * un_[2] + un_[3] * un_[3]);
#pragma unroll
    for (int m = 0; m < 10; ++m) pin[m] = VISC ? sn[(F_PI + m) * sf + c] : R(0);
    R cs2;
    eos_P(a.eos, e_n, P_n, cs2);
  }

  R gdiv = R(1);      // u~^tau that divides Q_pi in this stage (A11)
  R gst = R(1);       // u*^tau
  if (USE_PI) {
    // time row of the gradient (A10)
    if (MODE == 1) {
      const R* __restrict__ up = a.uprev;
      const R sx = R(2) * ut[1] - up[c], sy = R(2) * ut[2] - up[sf + c], sn_ = R(2) * ut[3] - up[2 * sf + c];
      const R gs2 = R(1) + sx * sx + sy * sy + sn_ * sn_;
      gst = sqrt_(gs2);
      // (u*^tau - u^tau)/h without cancellation: (gs2 - g2)/(gst + g)
      const R g2 = R(1) + ut[1] * ut[1] + ut[2] * ut[2] + ut[3] * ut[3];
      grad[0][0] = (gs2 - g2) / (gst + ut[0]) * a.inv_h;
      grad[0][1] = (sx - ut[1]) * a.inv_h; grad[0][2] = (sy - ut[2]) * a.inv_h; grad[0][3] = (sn_ - ut[3]) * a.inv_h;
      gdiv = gst;
    } else {
      gst = a.gstar[cg];
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
    is_source(ut, grad, pic, e_c, P_c, T_c, a.inv_5etas_hbarc, a.milne != 0, a.inv_tau, S + 4, a.inv_ctau, a.lam1);
  }

  // Q_T^n = tf_n T_f^{tau mu}(state n)
  const R w_n = e_n + P_n;
  R QTn[4];
  QTn[0] = a.tf_n * (w_n * un_[0] * un_[0] - P_n + pin[0]);
  QTn[1] = a.tf_n * (w_n * un_[0] * un_[1] + pin[1]);
  QTn[2] = a.tf_n * (w_n * un_[0] * un_[2] + pin[2]);
  QTn[3] = a.tf_n * (w_n * un_[0] * un_[3] + pin[3]);

  R pnew[10], M[4];
  if (MODE != 2) {
    // Eq.49-51: Q' = Q^n + h S(n)
    const R ig = R(1) / gdiv;
#pragma unroll
    for (int m = 0; m < 10; ++m) pnew[m] = USE_PI ? (un_[0] * pin[m] + a.h * S[4 + m]) * ig : R(0);
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) M[mu] = (QTn[mu] + a.h * S[mu]) * a.inv_tf_1 - pnew[mu];
  } else {
    // Eq.52-54 in Shu-Osher form (A26): Q^{n+1} = 1/2 [Q^n + Q(state') + h S(state')]
    const R ig = R(1) / gdiv;
#pragma unroll
    for (int m = 0; m < 10; ++m)
      pnew[m] = USE_PI ? R(0.5) * (un_[0] * pin[m] + gst * pic[m] + a.h * S[4 + m]) * ig : R(0);
    R QT1[4];
    QT1[0] = a.tf_1 * (w_c * ut[0] * ut[0] - P_c + pic[0]);
    QT1[1] = a.tf_1 * (w_c * ut[0] * ut[1] + pic[1]);
    QT1[2] = a.tf_1 * (w_c * ut[0] * ut[2] + pic[2]);
    QT1[3] = a.tf_1 * (w_c * ut[0] * ut[3] + pic[3]);
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) M[mu] = R(0.5) * (QTn[mu] + QT1[mu] + a.h * S[mu]) * a.inv_tf_1 - pnew[mu];
  }

  unsigned flags = 0;
  R e_new, ux_new, uy_new, un_new;
  rootfind(a.eos, M[0], M[1], M[2], M[3], e_c, a.root_iters, a.e_floor, a.v_max, e_new, ux_new, uy_new, un_new,
           flags);
  if (USE_PI) limit_pi(a.eos, a.xi, e_new, pnew, flags);

  // ---- write -----------------------------------------------------------------------------------
  if (active) {
    R* __restrict__ out = a.out;
    if (MODE == 0) {
      out[c] = R(2) * ut[1] - ux_new; out[sf + c] = R(2) * ut[2] - uy_new; out[2 * sf + c] = R(2) * ut[3] - un_new;
    } else {
      out[c] = e_new; out[sf + c] = ux_new; out[2 * sf + c] = uy_new; out[3 * sf + c] = un_new;
      if (VISC) {
#pragma unroll
        for (int m = 0; m < 10; ++m) out[(F_PI + m) * sf + c] = pnew[m];
        if (MODE == 1) a.gstar[cg] = gst;
      }
    }
  }

  // ---- reductions (row a10) ----------------------------------------------------------------------
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
      // reset the slot the NEXT user will accumulate into (no kernel of this stage touches it)
      if (MODE == 1) a.diag->emax[a.slot] = 0ull;
      else { a.diag->cfl[a.slot ^ 1][0] = 0ull; a.diag->cfl[a.slot ^ 1][1] = 0ull; a.diag->cfl[a.slot ^ 1][2] = 0ull; }
    }
  }
}

}  // namespace clv
