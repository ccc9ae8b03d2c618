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
};

// A: any argument struct with the members milne, inv_tau, tf_n, tf_1, inv_tf_1, h, inv_h, xi, e_floor, v_max,
// root_iters, inv_5etas_hbarc, eos.
//   S[14]      in: S_KT (T fields 0..3, pi fields 4..13); clobbered
//   c          the state the RHS was evaluated on (n in MODE 0/1, ' in MODE 2)
//   n          state n at the cell (MODE 2; ignored otherwise)
//   grad       rows 1..3 = spatial rows of nabla~_mu u~^nu (eta row already divided by tau); row 0 is filled here
//   up[3]      MODE 1: u~^i at n-1;  gst: MODE 1 out: u*^tau, MODE 2 in: u*^tau of stage 1
//   o          out: new e, P, u~, pi~;  cs2_o: c_s^2 at the new e
template <typename R, bool VISC, int MODE, typename A>
__device__ __forceinline__ void stage_update(const A& a, R S[14], const Cell<R>& c, const Cell<R>& n, R grad[4][4],
                                             const R up[3], R& gst, Cell<R>& o, R& cs2_o, unsigned& flags);

}  // namespace clv
