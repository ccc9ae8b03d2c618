// hydro_freezeout.cuh -- freeze-out hypersurface elements between two stored time levels.
//
// PAPER.md:268 (text under Eq.55): "d Sigma_mu is a freeze-out hyper-surface element determined by the constant
// freeze-out temperature T_f or constant freeze-out energy density e_f"; the finder runs on the GPU next
// to the e_max reduction that stops the evolution, so the full field never leaves the device.  The paper does not print
// the finder (it cites its Ref.[64]); reading A27: the cuboidal surface.  Every grid point of every stored
// level owns the 4-D cell centred on it; a point is HOT when e >= e_frz; the surface is the set of faces between a hot
// and a cold 4-D cell:
//   dir 0       cell c hot at level a and cold at level b (or the reverse): w = (e_frz - e_a)/(e_b - e_a),
//               tau* = tau_a + w dtau_out, dSigma~ = s (tau* dx dy deta, 0, 0, 0), s = +1 if hot at level a
//   dir 1,2,3   cells c and c + e_axis differ at level b: w = (e_frz - e_b(c))/(e_b(c+) - e_b(c)), position moved by
//               w * spacing along the axis, dSigma~_x = s tau_b dtau_out dy deta, dSigma~_y = s tau_b dtau_out dx deta,
//               dSigma~_eta = s dtau_out dx dy (tilde components, Eq.22), s = +1 if c is hot
// with u~^i and pi~ interpolated linearly with the weight w and u~^tau = sqrt(1 + u~.u~).  Cartesian geometry: tau -> 1.
// Outflow axes have no face across the domain edge; periodic axes wrap.  One thread per cell; an element is appended
// with one atomicAdd on the element counter and carries the key ((slab * 4 + dir) * N + cell), which is unique, so the
// (unordered) output can be compared after sorting by key.  Row: 22 doubles
//   [0:4] tau, x, y, eta   [4:8] dSigma~_mu   [8:11] u~^i   [11] u~^tau   [12:22] pi~
// The arithmetic is fp64 in both precisions (the levels are converted on load), every product and sum rounded
// separately (no FMA contraction), so that the fp64 result can be compared bit for bit.
#pragma once
#include <cuda_runtime.h>

namespace clv {

constexpr int FRZ_WORDS = 22;

struct FrzCounters {             // device block at the head of the freeze-out workspace
  unsigned long long n_elem;     // elements appended since hydro_freezeout_begin (including those that did not fit)
  unsigned long long n_hot_b;    // hot cells of the last level b
};

struct FrzArgs {
  int nx, ny, nz;
  int bc[3];
  int milne;
  long long N;
  double dx, dy, de;
  double tau_a, tau_b, e_frz;
  long long slab;
  long long capacity;
  FrzCounters* cnt;
  long long* keys;
  double* rows;
};

__device__ __forceinline__ double frz_centre(int i, int n, double d) {
  return __dmul_rn(__dsub_rn((double)i, __dmul_rn(0.5, (double)(n - 1))), d);
}
__device__ __forceinline__ double frz_mix(double w, double a, double b) {      // (1 - w) a + w b
  return __dadd_rn(__dmul_rn(__dsub_rn(1.0, w), a), __dmul_rn(w, b));
}

// level = (e [N], u~^mu [4][N], pi~ [10][N]) in the user layout (what hydro_read returns)
template <typename R>
__global__ void __launch_bounds__(256) freezeout_kernel(const FrzArgs a, const R* __restrict__ ea,
                                                        const R* __restrict__ ua, const R* __restrict__ pa,
                                                        const R* __restrict__ eb, const R* __restrict__ ub,
                                                        const R* __restrict__ pb) {
  const long long cu = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const bool in = cu < a.N;
  const long long c = in ? cu : 0;
  const int i = (int)(c % a.nx), j = (int)((c / a.nx) % a.ny), k = (int)(c / ((long long)a.nx * a.ny));
  const double e_a = (double)ea[c], e_b = (double)eb[c];
  const bool hot_a = e_a >= a.e_frz, hot_b = e_b >= a.e_frz;
  const double dt = __dsub_rn(a.tau_b, a.tau_a);
  const double xc = frz_centre(i, a.nx, a.dx), yc = frz_centre(j, a.ny, a.dy), zc = frz_centre(k, a.nz, a.de);

  auto emit = [&](int dir, const double pos[4], const double dS[4], double w, const R* __restrict__ u0,
                  const R* __restrict__ p0, long long c0, const R* __restrict__ u1, const R* __restrict__ p1,
                  long long c1) {
    const unsigned long long at = atomicAdd(&a.cnt->n_elem, 1ull);
    if ((long long)at >= a.capacity) return;
    a.keys[at] = (a.slab * 4 + dir) * a.N + c;
    double* __restrict__ r = a.rows + at * FRZ_WORDS;
#pragma unroll
    for (int m = 0; m < 4; ++m) { r[m] = pos[m]; r[4 + m] = dS[m]; }
    double ui[3];
#pragma unroll
    for (int m = 0; m < 3; ++m) {
      ui[m] = frz_mix(w, (double)u0[(m + 1) * a.N + c0], (double)u1[(m + 1) * a.N + c1]);
      r[8 + m] = ui[m];
    }
    r[11] = sqrt(__dadd_rn(__dadd_rn(__dadd_rn(1.0, __dmul_rn(ui[0], ui[0])), __dmul_rn(ui[1], ui[1])),
                           __dmul_rn(ui[2], ui[2])));
#pragma unroll
    for (int m = 0; m < 10; ++m) r[12 + m] = frz_mix(w, (double)p0[m * a.N + c0], (double)p1[m * a.N + c1]);
  };

  if (in && hot_a != hot_b) {      // time-like face of the cell
    const double w = __ddiv_rn(__dsub_rn(a.e_frz, e_a), __dsub_rn(e_b, e_a));
    const double ts = __dadd_rn(a.tau_a, __dmul_rn(w, dt));
    const double s = hot_a ? 1.0 : -1.0;
    const double tf = a.milne ? ts : 1.0;
    const double pos[4] = {ts, xc, yc, zc};
    const double dS[4] = {__dmul_rn(__dmul_rn(__dmul_rn(__dmul_rn(s, tf), a.dx), a.dy), a.de), 0.0, 0.0, 0.0};
    emit(0, pos, dS, w, ua, pa, c, ub, pb, c);
  }
  if (in) {
#pragma unroll
    for (int axis = 0; axis < 3; ++axis) {
      const int n_ax = axis == 0 ? a.nx : (axis == 1 ? a.ny : a.nz);
      const int c_ax = axis == 0 ? i : (axis == 1 ? j : k);
      int up = c_ax + 1;
      if (up >= n_ax) {
        if (!a.bc[axis] || n_ax < 2) continue;
        up = 0;
      }
      const long long stride = axis == 0 ? 1 : (axis == 1 ? a.nx : (long long)a.nx * a.ny);
      const long long c2 = c + (long long)(up - c_ax) * stride;
      const double e2 = (double)eb[c2];
      const bool hot2 = e2 >= a.e_frz;
      if (hot_b == hot2) continue;
      const double w = __ddiv_rn(__dsub_rn(a.e_frz, e_b), __dsub_rn(e2, e_b));
      const double s = hot_b ? 1.0 : -1.0;
      const double tf = a.milne ? a.tau_b : 1.0;
      double pos[4] = {a.tau_b, xc, yc, zc};
      const double sp = axis == 0 ? a.dx : (axis == 1 ? a.dy : a.de);
      pos[1 + axis] = __dadd_rn(pos[1 + axis], __dmul_rn(w, sp));
      double dS[4] = {0.0, 0.0, 0.0, 0.0};
      if (axis == 0) dS[1] = __dmul_rn(__dmul_rn(__dmul_rn(__dmul_rn(s, tf), dt), a.dy), a.de);
      else if (axis == 1) dS[2] = __dmul_rn(__dmul_rn(__dmul_rn(__dmul_rn(s, tf), dt), a.dx), a.de);
      else dS[3] = __dmul_rn(__dmul_rn(__dmul_rn(s, dt), a.dx), a.dy);
      emit(1 + axis, pos, dS, w, ub, pb, c, ub, pb, c2);
    }
  }
  // hot cells of level b: the stop criterion (e_max < e_frz  <=>  no hot cell), one atomic per warp
  const unsigned hot = __ballot_sync(0xffffffffu, in && hot_b);
  if ((threadIdx.x & 31) == 0 && hot) atomicAdd(&a.cnt->n_hot_b, (unsigned long long)__popc(hot));
}

}  // namespace clv
