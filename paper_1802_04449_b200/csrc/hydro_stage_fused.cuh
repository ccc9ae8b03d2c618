// hydro_stage_fused.cuh -- "kernel 2": the production stage kernel (fused stage on the extended state).
//
// Same fused stage as hydro_stage_ref.cuh (one launch per RK2 stage, one thread per cell), re-organised
// around what the ncu profile of kernel 1 showed (profiles/round1_kernel1.md: fp64 pipe 30 %,
// 15 k instructions per cell, 255 registers, 12 % occupancy):
//   * EXTENDED STATE: the producing kernel appends P, u^tau and the three signal speeds c_x, c_y, c_eta
//     of every cell to the state it writes (5 extra words), so the 13-point star is READ, never
//     re-derived: no EoS lookup, sqrt or division per stencil point (kernel 1 re-derives them 15 times).
//   * cheap generalised minmod (hmm4): 4 fp64-pipe instructions + selects on the integer pipe; fp32: FMNMX clamp form.
//   * the overall factor tau of Q_T, F_T (Eq.18) is applied once to the flux difference, not per point.
//   * warp-uniform early exit of the Newton iteration (no intra-warp divergence).
#pragma once
#include "hydro_stage_ref.cuh"
#include "hydro_stage_update.cuh"

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

// hmm4(dm, dp) = 4 x the half slope = 2 minmod(theta dm, (dm+dp)/2, theta dp)
//              = the smaller in magnitude of (2 theta s, dm + dp), s = the smaller in magnitude of (dm, dp), when dm and
//                dp share a sign, else 0.  th2 = 2 theta.  The callers fold the factor 1/4 into an FMA.
// fp64: both candidates carry the sign already, so there is no sign word to build: 5 fp64-pipe instructions (2 DSETP,
// DADD, 2 DMUL) + 7 on the integer pipe (4 selects, xor, compare, select of the 1/0 factor); the round-1 form spent
// 7 + 7 (profiles/round2_kernels.md).  fp32: clamp form on FMNMX / FMNMX3, 7 instructions and no integer logic.
__device__ __forceinline__ double hmm4(double dm, double dp, double th2) {
  const bool same = (__double2hiint(dm) ^ __double2hiint(dp)) >= 0;
  const double s = fabs(dm) < fabs(dp) ? dm : dp;
  const double t = s * th2;
  const double h = dm + dp;
  const double m = fabs(t) < fabs(h) ? t : h;
  // times 1 or 0: measured faster on B200 than zeroing with two selects (14.60 vs 14.78 ms per step) or zeroing s early
  return m * __hiloint2double(same ? 0x3ff00000 : 0, 0);
}
__device__ __forceinline__ float hmm4(float dm, float dp, float th2) {
  // t = 2 theta min(|dm|, |dp|) when the signs agree, else 0:  max(min(dm,dp), -max(dm,dp), 0)
  const float p = fminf(dm, dp), q = fmaxf(dm, dp);
  float t0, r;
  asm("max.f32 %0, %1, %2, %3;" : "=f"(t0) : "f"(p), "f"(-q), "f"(0.0f));
  const float t = t0 * th2;
  asm("min.f32 %0, %1, %2;" : "=f"(r) : "f"(fmaxf(dm + dp, -t)), "f"(t));      // clamp(dm + dp, -t, t)
  return r;
}

// 2 (H_{i+1/2} - H_{i-1/2}) for one field (the factor 1/2 of Eq.41 is folded into the caller's scale)
template <typename R>
__device__ __forceinline__ R kt_div2(const R q[5], const R f[5], R cl, R cr, R th2) {
  const R dq0 = q[1] - q[0], dq1 = q[2] - q[1], dq2 = q[3] - q[2], dq3 = q[4] - q[3];
  const R df0 = f[1] - f[0], df1 = f[2] - f[1], df2 = f[3] - f[2], df3 = f[4] - f[3];
  const R mq1 = hmm4(dq0, dq1, th2), mq2 = hmm4(dq1, dq2, th2), mq3 = hmm4(dq2, dq3, th2);
  const R mf1 = hmm4(df0, df1, th2), mf2 = hmm4(df1, df2, th2), mf3 = hmm4(df2, df3, th2);
  // Hr - Hl with the f-part collected (half slopes h = m/4):
  //   (f3 + f2 - hf3 + hf2) - (f2 + f1 - hf2 + hf1) = (df1 + df2) - (hf3 + hf1) + 2 hf2
  const R fpart = R(0.5) * mf2 + (R(-0.25) * (mf3 + mf1) + (df1 + df2));
  const R qr = R(-0.25) * (mq3 + mq2) + dq2, ql = R(-0.25) * (mq2 + mq1) + dq1;
  return fpart - cr * qr + cl * ql;
}

// ---- packed fp32 pairs (sm_100a add/mul/fma.f32x2 -> FADD2 / FMUL2 / FFMA2): two fields per instruction -------------
// The fp32 stage is bound by instruction issue (profiles/round2_kernels.md), so the arithmetic of the two fields of a
// trip is issued as one packed instruction; min/max stay scalar (there is no packed FMNMX).
#ifndef CLV_PACK32
#define CLV_PACK32 1
#endif
struct F2 { float x, y; };
__device__ __forceinline__ unsigned long long pk_(F2 a) {
  unsigned long long r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.x), "f"(a.y)); return r;
}
__device__ __forceinline__ F2 up_(unsigned long long r) {
  F2 a; asm("mov.b64 {%0, %1}, %2;" : "=f"(a.x), "=f"(a.y) : "l"(r)); return a;
}
__device__ __forceinline__ F2 bc2(float s) { F2 a = {s, s}; return a; }
__device__ __forceinline__ F2 add2(F2 a, F2 b) {
  unsigned long long r; asm("add.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk_(a)), "l"(pk_(b))); return up_(r);
}
__device__ __forceinline__ F2 sub2(F2 a, F2 b) { const F2 nb = {-b.x, -b.y}; return add2(a, nb); }
__device__ __forceinline__ F2 mul2(F2 a, F2 b) {
  unsigned long long r; asm("mul.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk_(a)), "l"(pk_(b))); return up_(r);
}
__device__ __forceinline__ F2 fma2(F2 a, F2 b, F2 c) {
  unsigned long long r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(pk_(a)), "l"(pk_(b)), "l"(pk_(c)));
  return up_(r);
}
__device__ __forceinline__ F2 hmm4_2(F2 dm, F2 dp, F2 th2) {
  float t0x, t0y, rx, ry;
  asm("max.f32 %0, %1, %2, %3;" : "=f"(t0x) : "f"(fminf(dm.x, dp.x)), "f"(-fmaxf(dm.x, dp.x)), "f"(0.0f));
  asm("max.f32 %0, %1, %2, %3;" : "=f"(t0y) : "f"(fminf(dm.y, dp.y)), "f"(-fmaxf(dm.y, dp.y)), "f"(0.0f));
  const F2 t0 = {t0x, t0y};
  const F2 t = mul2(t0, th2), s = add2(dm, dp);
  asm("min.f32 %0, %1, %2;" : "=f"(rx) : "f"(fmaxf(s.x, -t.x)), "f"(t.x));
  asm("min.f32 %0, %1, %2;" : "=f"(ry) : "f"(fmaxf(s.y, -t.y)), "f"(t.y));
  const F2 r = {rx, ry};
  return r;
}
// kt_div2 for a pair of fields
__device__ __forceinline__ F2 kt_div2_2(const F2 q[5], const F2 f[5], F2 cl, F2 ncr, F2 th2) {
  const F2 dq0 = sub2(q[1], q[0]), dq1 = sub2(q[2], q[1]), dq2 = sub2(q[3], q[2]), dq3 = sub2(q[4], q[3]);
  const F2 df0 = sub2(f[1], f[0]), df1 = sub2(f[2], f[1]), df2 = sub2(f[3], f[2]), df3 = sub2(f[4], f[3]);
  const F2 mq1 = hmm4_2(dq0, dq1, th2), mq2 = hmm4_2(dq1, dq2, th2), mq3 = hmm4_2(dq2, dq3, th2);
  const F2 mf1 = hmm4_2(df0, df1, th2), mf2 = hmm4_2(df1, df2, th2), mf3 = hmm4_2(df2, df3, th2);
  const F2 fpart = fma2(bc2(0.5f), mf2, fma2(bc2(-0.25f), add2(mf3, mf1), add2(df1, df2)));
  const F2 qr = fma2(bc2(-0.25f), add2(mq3, mq2), dq2), ql = fma2(bc2(-0.25f), add2(mq2, mq1), dq1);
  return fma2(cl, ql, fma2(ncr, qr, fpart));      // ncr = -cr
}

// signal speeds of one cell along the three axes from u~ (A6); cs2 from the EoS at the cell
template <typename R>
__device__ __forceinline__ void signal_speeds3(R g, R ux, R uy, R un, R cs2, R& cx, R& cy, R& cn) {
  const R ig = frcp_(g);
  const R ig2 = ig * ig;                                  // 1 - v^2 = 1/gamma^2
  const R v2 = (ux * ux + uy * uy + un * un) * ig2;
  const R cs = fsqrt_(cs2), omc = R(1) - cs2;
  const R D = frcp_(R(1) - v2 * cs2), base = R(1) - v2 * cs2, csg = cs * ig;
  const R vx = ux * ig, vy = uy * ig, vn = un * ig;
  cx = (fabs_(vx) * omc + csg * fsqrt_(max_(base - vx * vx * omc, R(0)))) * D;
  cy = (fabs_(vy) * omc + csg * fsqrt_(max_(base - vy * vy * omc, R(0)))) * D;
  cn = (fabs_(vn) * omc + csg * fsqrt_(max_(base - vn * vn * omc, R(0)))) * D;
}

#ifndef CLV_PFD
#define CLV_PFD 1        // prefetch distance in trips
#endif
#ifndef CLV_PFZ
#define CLV_PFZ 1        // L1 prefetch of the eta_s-neighbour planes one trip ahead (they are the loads that miss L1)
#endif
__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }
#ifndef CLV_MINB
#define CLV_MINB 2
#endif
#ifndef CLV_MINB32
#define CLV_MINB32 2     // fp32 blocks per SM; with the unrolled axis loop 2 (128 registers, no spills) measured 9.25 ms
                         // per step against 9.9 (3 blocks, 80 registers) and 9.5 (4 blocks, 64 registers)
#endif
// KT flux difference (Eq.40-44) of every evolved field along axis AX from the five-point star pp[0..4] of the extended
// state (pp[2] = the cell itself).  T fields: S[0..3] -= ...; pi fields: the thread-private shared-memory slots
// slot0[m * SSTR] (SSTR = threads per block; INIT: first axis, "=" instead of "-=").  cfl = c_a h / Delta_a of the cell.  Shared by the per-cell
// kernel (three axes) and the marching kernel (x and y; hydro_stage_march.cuh).  FSTR = element stride between the
// fields of a point (32 in the blocked global store; the plane size of a shared-memory tile).
// EXT: two more pi-like fields follow the ten pi components -- the bulk pressure Pi (Q = u^tau Pi,
// F_a = u^a Pi, Eq.30) and the net-baryon density n (Q_N / tau = n u^tau, F_a / tau = n u^a, Eq.28; the factor tau is
// applied by the stage tail) -- and Pi adds to the pressure in the T fields (A28).
template <typename R, bool USE_PI, int AX, bool INIT, int OX, int FSTR = FS, bool EXT = false, int SSTR = 256, typename A,
          int NS>
__device__ __forceinline__ void axis_flux(const A& a, const R* __restrict__ const (&pp)[5], R th2, R tf, R (&S)[NS],
                                          R* slot0, R& cfl) {
  constexpr int NTRIP = (EXT && USE_PI) ? 6 : 5;      // pi-like fields, two per trip
  const int o_ua = (1 + AX) * FSTR, o_ca = OX + (X_CX + AX) * FSTR;
  if (CLV_PFZ && USE_PI && AX == 2) {      // first pi trip of this axis: in flight behind the T-field part
#pragma unroll
    for (int p = 0; p < 5; ++p)
      if (p != 2) {
#pragma unroll
        for (int m = 0; m < 2 * CLV_PFD; ++m) prefetch_l1(pp[p] + (F_PI + m) * FSTR);
      }
  }

  R g[5], ua[5];
  R cl, cr;
  {
    const R c1 = pp[1][o_ca], c2 = pp[2][o_ca], c3 = pp[3][o_ca];
    cl = max_(c1, c2); cr = max_(c2, c3);
    cfl = c2 * a.h * a.scale[AX];
  }
#pragma unroll
  for (int p = 0; p < 5; ++p) { g[p] = pp[p][OX + X_G * FSTR]; ua[p] = pp[p][o_ua]; }
  const R sc_pi = R(0.5) * a.scale[AX], sc_T = sc_pi * tf;

  {
    // T fields: Q^mu/tau = T_f^{tau mu}, F_a^mu/tau = T_f^{a mu}   (Eq.27, Eq.39)
    R wq[5], wa[5], Pp[5];
#pragma unroll
    for (int p = 0; p < 5; ++p) {
      Pp[p] = pp[p][OX + X_P * FSTR];
      if (EXT && USE_PI) Pp[p] += pp[p][(F_PI + 10) * FSTR];      // P + Pi (A28)
      const R w = pp[p][0] + Pp[p];
      wq[p] = w * g[p]; wa[p] = w * ua[p];
    }
    if constexpr (CLV_PACK32 && sizeof(R) == 4) {
      // packed pairs (mu = 0,1) and (2,3): Q, F and the whole flux difference as f32x2
#pragma unroll
      for (int hp = 0; hp < 2; ++hp) {
        const int m0 = 2 * hp, m1 = m0 + 1;
        const int o_t0 = (F_PI + m0) * FSTR, o_t1 = (F_PI + m1) * FSTR;
        const int o_a0 = (F_PI + c_pidx[AX + 1][m0]) * FSTR, o_a1 = (F_PI + c_pidx[AX + 1][m1]) * FSTR;
        F2 q[5], f[5];
#pragma unroll
        for (int p = 0; p < 5; ++p) {
          const F2 um = {m0 == 0 ? (float)g[p] : (float)pp[p][m0 * FSTR], (float)pp[p][m1 * FSTR]};
          F2 cq = {m0 == 0 ? -(float)Pp[p] : 0.0f, 0.0f};
          F2 cf = {m0 == AX + 1 ? (float)Pp[p] : 0.0f, m1 == AX + 1 ? (float)Pp[p] : 0.0f};
          if (USE_PI) {
            cq.x += (float)pp[p][o_t0]; cq.y += (float)pp[p][o_t1];
            cf.x += (float)pp[p][o_a0]; cf.y += (float)pp[p][o_a1];
          }
          q[p] = fma2(bc2((float)wq[p]), um, cq); f[p] = fma2(bc2((float)wa[p]), um, cf);
        }
        const F2 d = kt_div2_2(q, f, bc2((float)cl), bc2(-(float)cr), bc2((float)th2));
        S[m0] -= R(d.x) * sc_T; S[m1] -= R(d.y) * sc_T;
      }
    } else {
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) {
      R q[5], f[5];
      const int o_t = (F_PI + (mu == 0 ? 0 : mu)) * FSTR;            // pi^{tau mu}: components 0..3
      const int o_a = (F_PI + c_pidx[AX + 1][mu]) * FSTR;            // pi^{a mu} (a constant-memory lookup measured
                                                                   // faster than a constexpr index here)
#pragma unroll
      for (int p = 0; p < 5; ++p) {
        const R umu = mu == 0 ? g[p] : pp[p][mu * FSTR];
        R tq = wq[p] * umu - (mu == 0 ? Pp[p] : R(0));
        R tfl = wa[p] * umu + (mu == AX + 1 ? Pp[p] : R(0));
        if (USE_PI) { tq += pp[p][o_t]; tfl += pp[p][o_a]; }
        q[p] = tq; f[p] = tfl;
      }
      S[mu] -= kt_div2(q, f, cl, cr, th2) * sc_T;
    }
    }
  }
  // pi fields: Q = u^tau pi, F_a = u^a pi   (Eq.29)
  if (USE_PI) {
    // two fields per trip: their 12 minmod chains interleave (ILP for the 4 warps per scheduler), the field
    // offsets inside a trip are immediates and the five star pointers are bumped once per trip
    const R* __restrict__ pq[5];
#pragma unroll
    for (int p = 0; p < 5; ++p) pq[p] = pp[p] + F_PI * FSTR;
    R* slot = slot0;
    if constexpr (CLV_PACK32 && sizeof(R) == 4) {
      F2 g2[5], ua2[5];
#pragma unroll
      for (int p = 0; p < 5; ++p) { g2[p] = bc2((float)g[p]); ua2[p] = bc2((float)ua[p]); }
      const F2 cl2 = bc2((float)cl), ncr2 = bc2(-(float)cr), th22 = bc2((float)th2);
#pragma unroll 1
      for (int t = 0; t < NTRIP; ++t) {
        F2 q[5], f[5];
        if (CLV_PFZ && AX == 2) {
#pragma unroll
          for (int p = 0; p < 5; ++p)
            if (p != 2) { prefetch_l1(pq[p] + CLV_PFD * 2 * FSTR); prefetch_l1(pq[p] + (CLV_PFD * 2 + 1) * FSTR); }
        }
#pragma unroll
        for (int p = 0; p < 5; ++p) {
          const F2 v = {(float)pq[p][0], (float)pq[p][FSTR]};
          q[p] = mul2(g2[p], v); f[p] = mul2(ua2[p], v);
          pq[p] += 2 * FSTR;
        }
        const F2 d = kt_div2_2(q, f, cl2, ncr2, th22);
        const R da = R(d.x) * sc_pi, db = R(d.y) * sc_pi;
        slot[0] = INIT ? -da : slot[0] - da;
        slot[SSTR] = INIT ? -db : slot[SSTR] - db;
        slot += 2 * SSTR;
      }
    } else {
#pragma unroll 1
    for (int t = 0; t < NTRIP; ++t) {
      R qa[5], fa[5], qb[5], fb[5];
      if (CLV_PFZ && AX == 2) {      // next trip's fields on the four off-centre planes
#pragma unroll
        for (int p = 0; p < 5; ++p)
          if (p != 2) { prefetch_l1(pq[p] + CLV_PFD * 2 * FSTR); prefetch_l1(pq[p] + (CLV_PFD * 2 + 1) * FSTR); }
      }
#pragma unroll
      for (int p = 0; p < 5; ++p) {
        const R va = pq[p][0], vb = pq[p][FSTR];
        qa[p] = g[p] * va; fa[p] = ua[p] * va;
        qb[p] = g[p] * vb; fb[p] = ua[p] * vb;
        pq[p] += 2 * FSTR;
      }
      const R da = kt_div2(qa, fa, cl, cr, th2) * sc_pi;
      const R db = kt_div2(qb, fb, cl, cr, th2) * sc_pi;
      slot[0] = INIT ? -da : slot[0] - da;
      slot[SSTR] = INIT ? -db : slot[SSTR] - db;
      slot += 2 * SSTR;
    }
    }
  }
}

// EXT: the 16-word cell of PAPER.md:614 -- fields 14 (bulk pressure Pi) and 15 (net-baryon density n)
// follow the ten pi components; viscous runs only.
template <typename R, bool VISC, int MODE, bool EXT = false>
__global__ void __launch_bounds__(256, (sizeof(R) == 4 ? CLV_MINB32 : CLV_MINB)) stage_fused_kernel(const StageArgs<R> a) {
  static_assert(!EXT || VISC, "the bulk / baryon extension rides on the viscous path");
  constexpr bool USE_PI = VISC && (MODE != 0);
  constexpr bool XT = EXT && USE_PI;                // the extension is active in this launch (not in the bootstrap)
  constexpr int NPI = XT ? 12 : 10;                 // pi-like fields
  constexpr int NF = VISC ? (EXT ? 16 : 14) : 4;    // evolved fields of a buffer; extended slots follow
  constexpr int OX = NF * FS;                       // element offset of the extended slots inside an x-block
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const int j = blockIdx.y * blockDim.y + threadIdx.y;
  const int k = blockIdx.z;
  const bool active = (i < a.nx) && (j < a.ny);
  const int ic = active ? i : 0, jc = active ? j : 0;
  constexpr int sf = FS;
  const long long c = (long long)k * a.sz + (long long)jc * a.sy + xoff(ic, a.blk);
  const long long cg = ((long long)k * a.ny + jc) * a.gp + ic;
  const R* __restrict__ in = a.in;
  const R* __restrict__ pc = a.in + c;              // this cell: field m at pc[m * FS] (immediate offsets)

  // S_KT of the ten pi fields accumulates in thread-private shared-memory slots, so that the pi-field loop
  // can stay rolled (its ~200-instruction body then lives in the L0 instruction cache)
  __shared__ R sS[USE_PI ? NPI * 256 : 1];
  const int tid = threadIdx.y * 32 + threadIdx.x;
  R S[16];
#pragma unroll
  for (int m = 0; m < 16; ++m) S[m] = R(0);
  R cfl0 = R(0), cfl1 = R(0), cfl2 = R(0);
  const R tf = a.milne ? a.tau : R(1);
  const R th2 = R(2) * a.theta;

  // ---- KT flux divergence, axes x, y, eta (Eq.40; A22) -------------------------------------------
  // fully unrolled: with ax a compile-time constant every field offset and the P delta^{a mu} select are
  // immediates (measured 17.2 -> 15.6 ms per step; the ~100 KB of code is streamed
  // through the instruction cache three axis-bodies in a row, each with its own L0-resident pi loop)
#pragma unroll
  for (int ax = 0; ax < 3; ++ax) {
    long long idx[5];
    star_offsets(a, ax, ic, jc, k, idx);
    const R* __restrict__ pp[5];
#pragma unroll
    for (int p = 0; p < 5; ++p) pp[p] = in + idx[p];
    if (ax == 0) axis_flux<R, USE_PI, 0, true, OX, FS, XT>(a, pp, th2, tf, S, &sS[tid], cfl0);
    else if (ax == 1) axis_flux<R, USE_PI, 1, false, OX, FS, XT>(a, pp, th2, tf, S, &sS[tid], cfl1);
    else axis_flux<R, USE_PI, 2, false, OX, FS, XT>(a, pp, th2, tf, S, &sS[tid], cfl2);
  }
  if (USE_PI) {
#pragma unroll
    for (int m = 0; m < NPI; ++m) S[4 + m] = sS[m * 256 + tid];
  }

  // ---- cell-centre state (re-read after the flux loop: L1 hits, keeps the loop's register set small) ---
  Cell<R> cc, cn_;
  cc.e = pc[0];
  cc.u[1] = pc[sf]; cc.u[2] = pc[2 * sf]; cc.u[3] = pc[3 * sf];
  cc.u[0] = pc[OX + X_G * FS];
  cc.P = pc[OX + X_P * FS];
#pragma unroll
  for (int m = 0; m < 10; ++m) cc.pi[m] = USE_PI ? pc[(F_PI + m) * FS] : R(0);
  cc.Pi = XT ? pc[(F_PI + 10) * FS] : R(0); cc.nb = XT ? pc[(F_PI + 11) * FS] : R(0);

  // spatial rows of nabla~_mu u~^nu by central differences (A9); eta row divided by tau (Eq.22)
  R grad[4][4];
#pragma unroll
  for (int m = 0; m < 4; ++m)
#pragma unroll
    for (int n = 0; n < 4; ++n) grad[m][n] = R(0);
  if (USE_PI) {
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) {
      const int im = ax == 0 ? bmap(ic - 1, a.nx, a.bc[0]) : ic, ip = ax == 0 ? bmap(ic + 1, a.nx, a.bc[0]) : ic;
      const int jm = ax == 1 ? bmap(jc - 1, a.ny, a.bc[1]) : jc, jp = ax == 1 ? bmap(jc + 1, a.ny, a.bc[1]) : jc;
      const int km = ax == 2 ? bmap(k - 1, a.nz, a.bc[2]) : k, kp = ax == 2 ? bmap(k + 1, a.nz, a.bc[2]) : k;
      const R* __restrict__ qm = in + ((long long)km * a.sz + (long long)jm * a.sy + xoff(im, a.blk));
      const R* __restrict__ qp = in + ((long long)kp * a.sz + (long long)jp * a.sy + xoff(ip, a.blk));
      const R sc = R(0.5) * a.scale[ax];
      grad[ax + 1][0] = (qp[OX + X_G * FS] - qm[OX + X_G * FS]) * sc;
      grad[ax + 1][1] = (qp[sf] - qm[sf]) * sc;
      grad[ax + 1][2] = (qp[2 * sf] - qm[2 * sf]) * sc;
      grad[ax + 1][3] = (qp[3 * sf] - qm[3 * sf]) * sc;
    }
  }

  // ---- state n at the centre (MODE 2 reads it; MODE 0/1: it is the star centre itself) -----------
  if (MODE == 2) {
    const R* __restrict__ sn = a.sn + c;
    cn_.e = sn[0];
    cn_.u[1] = sn[sf]; cn_.u[2] = sn[2 * sf]; cn_.u[3] = sn[3 * sf];
    cn_.u[0] = sn[OX + X_G * FS];
    cn_.P = sn[OX + X_P * FS];
#pragma unroll
    for (int m = 0; m < 10; ++m) cn_.pi[m] = VISC ? sn[(F_PI + m) * FS] : R(0);
    cn_.Pi = XT ? sn[(F_PI + 10) * FS] : R(0); cn_.nb = XT ? sn[(F_PI + 11) * FS] : R(0);
  }
  R up3[3] = {R(0), R(0), R(0)};
  R gst = R(1);
  if (USE_PI) {
    if (MODE == 1) {
      const R* __restrict__ up = a.uprev + c;
      up3[0] = up[0]; up3[1] = up[sf]; up3[2] = up[2 * sf];
    } else {
      gst = a.gstar[cg];
    }
  }

  // ---- sources, stage update, root-find, limiter (hydro_stage_update.cuh) -------------------------
  unsigned flags = 0;
  Cell<R> nw;
  R cs2_new;
  stage_update<R, VISC, MODE, XT>(a, S, cc, cn_, grad, up3, gst, nw, cs2_new, flags, tf);
  const R* ut = cc.u;
  const R e_new = nw.e, P_new = nw.P, ux_new = nw.u[1], uy_new = nw.u[2], un_new = nw.u[3], g_new = nw.u[0];
  const R* pnew = nw.pi;

  // ---- write state + extended slots ----------------------------------------------------------------
  if (active) {
    R* __restrict__ out = a.out + c;
    if (MODE == 0) {
      out[0] = R(2) * ut[1] - ux_new; out[sf] = R(2) * ut[2] - uy_new; out[2 * sf] = R(2) * ut[3] - un_new;
    } else {
      R cx, cy, cn;
      signal_speeds3(g_new, ux_new, uy_new, un_new, cs2_new, cx, cy, cn);
      out[0] = e_new; out[sf] = ux_new; out[2 * sf] = uy_new; out[3 * sf] = un_new;
      if (VISC) {
#pragma unroll
        for (int m = 0; m < 10; ++m) out[(F_PI + m) * FS] = pnew[m];
        if (XT) { out[(F_PI + 10) * FS] = nw.Pi; out[(F_PI + 11) * FS] = nw.nb; }
        if (MODE == 1) a.gstar[cg] = gst;
      }
      out[OX + X_P * FS] = P_new; out[OX + X_G * FS] = g_new;
      out[OX + X_CX * FS] = cx; out[OX + X_CY * FS] = cy; out[OX + X_CN * FS] = cn;
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

template <typename R, bool VISC, int MODE, bool EXT = false>
void launch_stage_fused(const StageArgs<R>& a, cudaStream_t stream) {
  dim3 block(32, 8, 1);
  dim3 grid((a.nx + 31) / 32, (a.ny + 7) / 8, a.nz);
  stage_fused_kernel<R, VISC, MODE, EXT><<<grid, block, 0, stream>>>(a);
}

}  // namespace clv
