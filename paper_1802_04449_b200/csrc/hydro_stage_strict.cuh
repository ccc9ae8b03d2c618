// hydro_stage_strict.cuh -- the strict reading of Eq.53 (A12).
//
// Eq.53 as printed evaluates the stage-2 right-hand side of T^{tau mu} with pi^{n+1} (the result of Eq.52), not with
// pi' -- "two sweeps in stage 2".  With hydro_opts.strict_eq53 = 1 stage 2 becomes three launches:
//   sweep A   the ordinary stage-2 kernel with the pi limiter off and a scratch diagnostics block: its pi slots hold the
//             unlimited pi^{n+1} of Eq.52 (its e, u~ are overwritten by sweep B);
//   sweep B   stage_strict_T_kernel: KT fluxes and geometric source of the four T fields on (e', u~', pi^{n+1}) --
//             13-point star of e', u~', P, c_a from the state ' buffer and of pi^{n+1} from the output buffer --, Heun
//             update of T (Shu-Osher form, A26), root-find; writes e, u~ and the derived words, not pi;
//   sweep C   stage_strict_limit_kernel: the pi limiter (A14) on pi^{n+1} with the new e, P, cell by cell.
// Sweep B reads only the pi slots of the output buffer and writes only the others, so there is no race.
// Same blocked extended store as kernels 2 and 4 (the only kernels the option is available for).
#pragma once
#include "hydro_stage_fused.cuh"

namespace clv {

template <typename R>
__global__ void __launch_bounds__(256, 2) stage_strict_T_kernel(const StageArgs<R> a, const R* __restrict__ pin) {
  constexpr int NF = 14, OX = NF * FS, sf = FS;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  const bool active = (i < a.nx) && (j < a.ny);
  const int ic = active ? i : 0, jc = active ? j : 0;
  const long long c = (long long)k * a.sz + (long long)jc * a.sy + xoff(ic, a.blk);
  const R tf = a.milne ? a.tau : R(1);
  const R th2 = R(2) * a.theta;
  R S[4] = {R(0), R(0), R(0), R(0)};

#pragma unroll
  for (int ax = 0; ax < 3; ++ax) {
    long long idx[5];
    star_offsets(a, ax, ic, jc, k, idx);
    const R* __restrict__ pp[5];
    const R* __restrict__ ppi[5];
#pragma unroll
    for (int p = 0; p < 5; ++p) { pp[p] = a.in + idx[p]; ppi[p] = pin + idx[p]; }
    const int o_ca = OX + (X_CX + ax) * FS;
    const R cl = max_(pp[1][o_ca], pp[2][o_ca]), cr = max_(pp[2][o_ca], pp[3][o_ca]);
    R g[5], wq[5], wa[5], Pp[5];
#pragma unroll
    for (int p = 0; p < 5; ++p) {
      g[p] = pp[p][OX + X_G * FS];
      Pp[p] = pp[p][OX + X_P * FS];
      const R w = pp[p][0] + Pp[p];
      wq[p] = w * g[p]; wa[p] = w * pp[p][(1 + ax) * FS];
    }
    const R sc_T = R(0.5) * a.scale[ax] * tf;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
      R q[5], f[5];
      const int o_t = (F_PI + mu) * FS, o_a = (F_PI + c_pidx[ax + 1][mu]) * FS;
#pragma unroll
      for (int p = 0; p < 5; ++p) {
        const R umu = mu == 0 ? g[p] : pp[p][mu * FS];
        q[p] = wq[p] * umu - (mu == 0 ? Pp[p] : R(0)) + ppi[p][o_t];
        f[p] = wa[p] * umu + (mu == ax + 1 ? Pp[p] : R(0)) + ppi[p][o_a];
      }
      S[mu] -= kt_div2(q, f, cl, cr, th2) * sc_T;
    }
  }

  // centre: state ' (RHS state), pi^{n+1}, state n
  const R* __restrict__ pc = a.in + c;
  const R* __restrict__ pn = pin + c;
  const R* __restrict__ sn = a.sn + c;
  const R e1 = pc[0], u1x = pc[sf], u1y = pc[2 * sf], u1n = pc[3 * sf], g1 = pc[OX + X_G * FS], P1 = pc[OX + X_P * FS];
  const R w1 = e1 + P1;
  if (a.milne) {      // Eq.31 (sign A1) with pi^{n+1}
    S[0] -= w1 * u1n * u1n + P1 + pn[(F_PI + 9) * FS];
    S[3] -= w1 * g1 * u1n + pn[(F_PI + 3) * FS];
  }
  const R en = sn[0], unx = sn[sf], uny = sn[2 * sf], unn = sn[3 * sf], gn = sn[OX + X_G * FS], Pn = sn[OX + X_P * FS];
  const R wn = en + Pn;
  const R un4[4] = {gn, unx, uny, unn}, u14[4] = {g1, u1x, u1y, u1n};
  R M[4];
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) {
    const R QTn = a.tf_n * (wn * gn * un4[mu] - (mu == 0 ? Pn : R(0)) + sn[(F_PI + mu) * FS]);
    const R QT1 = a.tf_1 * (w1 * g1 * u14[mu] - (mu == 0 ? P1 : R(0)) + pc[(F_PI + mu) * FS]);
    M[mu] = R(0.5) * (QTn + QT1 + a.h * S[mu]) * a.inv_tf_1 - pn[(F_PI + mu) * FS];      // Eq.53-54 (A26 form)
  }
  unsigned flags = 0;
  R e_new, P_new, cs2_new, ux, uy, un, g_new;
  rootfind_warp(a.eos, M[0], M[1], M[2], M[3], e1, a.root_iters, a.e_floor, a.v_max, e_new, P_new, cs2_new, ux, uy, un,
                g_new, flags);
  if (active) {
    R* __restrict__ out = a.out + c;
    R cx, cy, cn;
    signal_speeds3(g_new, ux, uy, un, cs2_new, cx, cy, cn);
    out[0] = e_new; out[sf] = ux; out[2 * sf] = uy; out[3 * sf] = un;
    out[OX + X_P * FS] = P_new; out[OX + X_G * FS] = g_new;
    out[OX + X_CX * FS] = cx; out[OX + X_CY * FS] = cy; out[OX + X_CN * FS] = cn;
  } else {
    flags = 0;
  }
  count_flags(a.diag, flags);
  const int lane = (threadIdx.x + threadIdx.y * blockDim.x) & 31;
  const double r = warp_max(active ? (double)e_new : 0.0);
  if (lane == 0) atomic_max_nonneg(&a.diag->emax[a.slot], r);
  if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && threadIdx.x == 0 && threadIdx.y == 0) {
    a.diag->cfl[a.slot ^ 1][0] = 0ull; a.diag->cfl[a.slot ^ 1][1] = 0ull; a.diag->cfl[a.slot ^ 1][2] = 0ull;
  }
}

// sweep C: pi <- limiter(pi; e, P) cell by cell in the output buffer (A14)
template <typename R>
__global__ void __launch_bounds__(256) stage_strict_limit_kernel(const StageArgs<R> a) {
  constexpr int OX = 14 * FS;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  const bool active = (i < a.nx) && (j < a.ny);
  const int ic = active ? i : 0, jc = active ? j : 0;
  R* __restrict__ o = a.out + ((long long)k * a.sz + (long long)jc * a.sy + xoff(ic, a.blk));
  R pi[10];
#pragma unroll
  for (int m = 0; m < 10; ++m) pi[m] = o[(F_PI + m) * FS];
  unsigned flags = 0;
  limit_pi_P(a.xi, o[0], o[OX + X_P * FS], pi, flags);
  if (active && flags) {
#pragma unroll
    for (int m = 0; m < 10; ++m) o[(F_PI + m) * FS] = pi[m];
  }
  count_flags(a.diag, active ? flags : 0u);
}

}  // namespace clv
