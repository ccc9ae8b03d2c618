// hydro_stage_tile.cuh -- "kernel 3": the tile / marching stage kernel (default).
//
// One launch per RK2 stage, like kernels 1 and 2, but every limited slope and every KT face flux is computed ONCE
// and shared by the cells that use it (kernels 1/2: every slope 3x, every face 2x; profiles/round1_kernel2.md).
//
//   * State buffers are plain SoA with two ghost layers per side: [field][nz+4][ny+4][pitch], 14 words per cell
//     (e, u~^x, u~^y, u~^eta, pi~[10]); nothing derived is stored ("16 floats per cell").
//   * A block owns a 32 x 8 xy tile and MARCHES along eta_s through a z-chunk.  Each plane of the tile with its
//     2-cell halo (36 x 12 points x 14 fields) arrives by ONE TMA box load (cp.async.bulk.tensor.4d + mbarrier)
//     into a 4-stage shared-memory ring: the point the paper could not reach for want of local memory
//     (7^3 block, 56 KB) -- a B200 SM has 227 KB.
//   * eta_s direction: a register pipeline per column.  When plane p arrives, the slope of cell p-1, the face
//     p-3/2 and the flux difference of cell k = p-2 are completed from the kept left state (Q^l, F^l) and face flux
//     of the previous step: one slope and one face per cell per field.
//   * x direction: lanes of a warp are 32 consecutive x cells; left/right states and face fluxes travel by warp
//     shuffle; the two halo cells on each side are handled once per tile row by one warp (x-halo pass).
//   * y direction: warps are rows; left/right states travel through a double-buffered shared-memory exchange, one
//     block barrier per field; the rows -1 and 8 are handled by the first / last warp (warp-uniform branch).
//   * P, u~^tau and the signal speeds c_x, c_y, c_eta are derived once per loaded point (interior: on arrival of its
//     plane; halo: in the halo passes), never stored in HBM.
//   * Boundaries (row a11): the producing kernel writes the ghost cells itself (clamp: copies of the edge cell;
//     periodic: copies of the opposite edge), so the TMA boxes never need an index map.
// The tail of the stage (sources, update, root-find, limiter) is hydro_stage_update.cuh, shared with kernel 2.
//
// Citations: KT scheme PAPER.md:193-213 (Eq.40-44); sources :161-183 (Eq.31-38); RK2 :225-239 (Eq.49-54).
#pragma once
#include <cuda.h>

#include "hydro_stage_fused.cuh"
#include "hydro_stage_update.cuh"

namespace clv {

constexpr int TX = 32, TY = 8, HALO = 2;
constexpr int SX = TX + 2 * HALO, SY = TY + 2 * HALO;   // 36 x 12 points per plane of a tile
constexpr int FST = SX * SY;                            // field stride inside a ring stage (elements)
constexpr int NSTAGE = 4;
constexpr int TILE_THREADS = TX * TY;
constexpr int XHW = 5;                                  // the warp that runs the x-halo pass

template <typename R>
struct TileArgs {
  int nx, ny, nz;
  // ghosted SoA buffer: element(field f, cell i,j,k) = f*pf + (k+2)*pz + (j+2)*py + (i+2)
  long long py, pz, pf;
  int bc[3];
  int milne;
  R tau, inv_tau, tf_n, tf_1, inv_tf_1, h, inv_h;
  R scale[3];
  R theta, e_floor, xi, v_max, inv_5etas_hbarc;
  int root_iters;
  const R* sn;       // MODE 2: state n (centre only)
  const R* uprev;    // MODE 1: u~^i at n-1 (3 fields, stride pf)
  R* gstar;          // u*^tau (one field)
  R* out;            // MODE 1: state '; MODE 2: state n+1; MODE 0: history (3 fields, stride pf)
  EosDev<R> eos;
  DiagDev* diag;
  int slot;
  int ntx, nty, nchunk, chunk;   // tiles in x, y; z-chunks and planes per chunk
};

// symmetric (mu, nu) -> pi component 0..9 (order tt, tx, ty, tn, xx, xy, xn, yy, yn, nn); folds after unrolling
__device__ __forceinline__ constexpr int pidx_f(int m, int n) {
  const int lo = m < n ? m : n, hi = m < n ? n : m;
  return lo == 0 ? hi : (lo == 1 ? 3 + hi : (lo == 2 ? 5 + hi : 9));
}

// ---- shared memory of a block --------------------------------------------------------------------------------------
template <typename R, int NFL, int NFS>
struct TileSmem {
  R ring[NSTAGE][NFL][SY][SX];      // TMA destinations; NFL * 432 * sizeof(R) is a multiple of 128 bytes
  R yx[2][4][TY][TX];               // y exchange: Q^l, F^l, Q^r, F^r of the interior rows, double-buffered per field
  R yaux[3][SY][TX];                // g, P, c_y of rows -2..9 (interior columns)
  R xh[NFS][2][2][TY];              // x-halo: [field][side][Q state, F state][row]  (side 0: Q^l of cell -1; 1: Q^r of cell 32)
  R xaux[3][2][TY];                 // g, P, c_x of cell -1 (side 0) and cell 32 (side 1)
  unsigned long long bar[NSTAGE];
};

// ---- TMA / mbarrier primitives (PTX) -------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// one 4-D box {36, 12, 1, NFL} of the ghosted state buffer -> one ring stage
__device__ __forceinline__ void tma_load_plane(void* dst, const CUtensorMap* map, unsigned long long* bar, int x, int y,
                                               int z) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(z), "r"(0) : "memory");
}

// ---- per-point quantities ------------------------------------------------------------------------------------------
template <typename R>
struct PtAux {      // what Q and F_a of every field need at a point
  R g, ua, P, wg, wua;
};
template <typename R>
__device__ __forceinline__ PtAux<R> pt_aux(R e, R g, R ua, R P) {
  PtAux<R> x;
  x.g = g; x.ua = ua; x.P = P;
  const R w = e + P;
  x.wg = w * g; x.wua = w * ua;
  return x;
}
// Q and F_a of evolved field f at a point whose raw words sit at pt[field * FST]  (Eq.27, 29, 39; the factor tau of
// the T fields is applied to the flux difference).  ax = axis of the flux; f and ax are compile-time after unrolling.
template <typename R, bool USE_PI>
__device__ __forceinline__ void qf(const R* __restrict__ pt, const PtAux<R>& x, int f, int ax, R& Q, R& Fl) {
  if (f < 4) {
    const R umu = f == 0 ? x.g : pt[f * FST];
    Q = x.wg * umu; Fl = x.wua * umu;
    if (f == 0) Q -= x.P;
    if (f == ax + 1) Fl += x.P;
    if (USE_PI) { Q += pt[(4 + pidx_f(0, f)) * FST]; Fl += pt[(4 + pidx_f(ax + 1, f)) * FST]; }
  } else {
    const R v = pt[f * FST];
    Q = x.g * v; Fl = x.ua * v;
  }
}
// half-slope states of a cell: Q^l = Q + s/2 (left state of its upper face), Q^r = Q - s/2   (Eq.43-44, A4)
template <typename R>
__device__ __forceinline__ void lr(R Qm, R Q0, R Qp, R theta, R& L, R& Rr) {
  const R s = hmm(Q0 - Qm, Qp - Q0, theta);
  L = Q0 + s; Rr = Q0 - s;
}
// 2 H_{i+1/2} from the left state of cell i and the right state of cell i+1   (Eq.41-42, A5)
template <typename R>
__device__ __forceinline__ R face2(R QL, R FL, R QRn, R FRn, R c) { return (FL + FRn) - c * (QRn - QL); }

__device__ __forceinline__ double shfl_up_(double v) { return __shfl_up_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ float shfl_up_(float v) { return __shfl_up_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ double shfl_dn_(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ float shfl_dn_(float v) { return __shfl_down_sync(0xffffffffu, v, 1); }

template <typename R>
struct PlaneAux {   // derived once per column when its plane arrives
  R g, P, cx, cy, cn;
};

// g, P, c_s^2 of a raw point
template <typename R>
__device__ __forceinline__ void derive(const EosDev<R>& eos, const R* __restrict__ pt, R& e, R& ux, R& uy, R& un, R& g,
                                       R& P, R& cs2) {
  e = pt[0]; ux = pt[FST]; uy = pt[2 * FST]; un = pt[3 * FST];
  g = sqrt_(R(1) + ux * ux + uy * uy + un * un);
  eos_P(eos, e, P, cs2);
}

// ghost positions of axis extent n that mirror cell i (boundary rule a11): up to four of {-2, -1, n, n+1}
__device__ __forceinline__ int ghost_list(int i, int n, int periodic, int out[4]) {
  int cnt = 0;
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    const int gidx = t < 2 ? t - 2 : n + (t - 2);
    if (bmap(gidx, n, periodic) == i) out[cnt++] = gidx;
  }
  return cnt;
}

// =====================================================================================================================
template <typename R, bool VISC, int MODE>
__global__ void __launch_bounds__(TILE_THREADS, 1)
stage_tile_kernel(const TileArgs<R> a, const __grid_constant__ CUtensorMap tmap) {
  constexpr bool USE_PI = VISC && (MODE != 0);
  constexpr int NFS = USE_PI ? 14 : 4;          // evolved fields whose fluxes are formed
  constexpr int NFL = NFS;                      // fields per TMA box (the tensor map carries the same count)
  using Smem = TileSmem<R, NFL, NFS>;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(smem_raw);

  const int lane = threadIdx.x & 31, row = threadIdx.x >> 5, tid = threadIdx.x;
  // block -> (tile x, tile y, z chunk); x fastest so that concurrently running blocks share halos in L2
  int b = blockIdx.x;
  const int tx = b % a.ntx; b /= a.ntx;
  const int ty = b % a.nty; b /= a.nty;
  const int kc0 = b * a.chunk, kc1 = min(kc0 + a.chunk, a.nz);
  const int X0 = tx * TX, Y0 = ty * TY;
  const int i = X0 + lane, j = Y0 + row;
  const bool active = (i < a.nx) && (j < a.ny);
  constexpr unsigned STAGE_BYTES = NFL * FST * sizeof(R);

  const int p_first = kc0 - 2, p_last = kc1 + 1;
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NSTAGE; ++s) mbar_init(&sm.bar[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NSTAGE; ++s) {
      const int p = p_first + s;
      if (p <= p_last) {
        mbar_expect_tx(&sm.bar[p & 3], STAGE_BYTES);
        tma_load_plane(&sm.ring[p & 3][0][0][0], &tmap, &sm.bar[p & 3], X0, Y0, p + HALO);
      }
    }
  }

  // ---- per-thread state that lives across planes --------------------------------------------------------------------
  R S[14];                          // S_KT of the centre cell
  R QLk[NFS], FLk[NFS], Hk[NFS];    // eta pipeline: left state of cell p-2 -> p-1, and 2 H of the last face
#pragma unroll
  for (int f = 0; f < NFS; ++f) { QLk[f] = R(0); FLk[f] = R(0); Hk[f] = R(0); }
#pragma unroll
  for (int f = 0; f < 14; ++f) S[f] = R(0);
  PlaneAux<R> h1 = {R(1), R(0), R(0), R(0), R(0)}, h2 = h1;      // planes p-1 and p-2
  R km1[4] = {R(1), R(0), R(0), R(0)};                            // u~^mu of plane k-1
  const R tf = a.milne ? a.tau : R(1);
  const R sc_eta = R(0.5) * a.scale[2], sc_x = R(0.5) * a.scale[0], sc_y = R(0.5) * a.scale[1];
  unsigned flags_acc = 0;
  R cfl0 = R(0), cfl1 = R(0), cfl2 = R(0), emax = R(0);

  const int own = (row + HALO) * SX + (lane + HALO);     // own point inside a field plane of a stage

  for (int p = p_first; p <= p_last; ++p) {
    const int it = p - p_first;
    mbar_wait(&sm.bar[p & 3], (unsigned)((it >> 2) & 1));
    const R* __restrict__ rp = &sm.ring[p & 3][0][0][0] + own;
    const R* __restrict__ r1 = &sm.ring[(p - 1) & 3][0][0][0] + own;     // plane p-1 = k+1
    const R* __restrict__ r2 = &sm.ring[(p - 2) & 3][0][0][0] + own;     // plane p-2 = k

    // ---- arrival of plane p: derived quantities of the own column ---------------------------------------------------
    PlaneAux<R> hp;
    R e_p, ux_p, uy_p, un_p;
    {
      R cs2;
      derive(a.eos, rp, e_p, ux_p, uy_p, un_p, hp.g, hp.P, cs2);
      signal_speeds3(hp.g, ux_p, uy_p, un_p, cs2, hp.cx, hp.cy, hp.cn);
    }

    // ---- eta pipeline: slope of cell p-1, face p-3/2, flux difference of cell k = p-2 ---------------------------------
    if (p >= kc0) {
      const PtAux<R> xp = pt_aux(e_p, hp.g, un_p, hp.P);
      const PtAux<R> x1 = pt_aux(r1[0], h1.g, r1[3 * FST], h1.P);
      const PtAux<R> x2 = pt_aux(r2[0], h2.g, r2[3 * FST], h2.P);
      const R cface = max_(h2.cn, h1.cn);
#pragma unroll
      for (int f = 0; f < NFS; ++f) {
        R Qp, Fp, Q1, F1, Q2, F2, QL1, QR1, FL1, FR1;
        qf<R, USE_PI>(rp, xp, f, 2, Qp, Fp);
        qf<R, USE_PI>(r1, x1, f, 2, Q1, F1);
        qf<R, USE_PI>(r2, x2, f, 2, Q2, F2);
        lr(Q2, Q1, Qp, a.theta, QL1, QR1);
        lr(F2, F1, Fp, a.theta, FL1, FR1);
        const R Hn = face2(QLk[f], FLk[f], QR1, FR1, cface);
        S[f] = -(Hn - Hk[f]) * (f < 4 ? sc_eta * tf : sc_eta);
        QLk[f] = QL1; FLk[f] = FL1; Hk[f] = Hn;
      }
    }

    // ---- centre plane k = p-2: x and y fluxes, sources, update, root-find, store -------------------------------------
    if (p - 2 >= kc0) {
      const int k = p - 2;
      const R* __restrict__ rk = r2;
      const R e0 = rk[0], ux0 = rk[FST], uy0 = rk[2 * FST], un0 = rk[3 * FST];
      const R g0 = h2.g, P0 = h2.P;
      const R* __restrict__ ringk = &sm.ring[k & 3][0][0][0];

      // (1) own g, P, c_y for the y neighbours
      sm.yaux[0][row + HALO][lane] = g0; sm.yaux[1][row + HALO][lane] = P0; sm.yaux[2][row + HALO][lane] = h2.cy;
      // (2) the four halo rows: first and last warp, two rows each (warp-uniform branch)
      if (row == 0 || row == TY - 1) {
#pragma unroll
        for (int t = 0; t < 2; ++t) {
          const int sy = row == 0 ? t : SY - 2 + t;
          R e, ux, uy, un, g, P, cs2, cx, cy, cn;
          derive(a.eos, ringk + sy * SX + lane + HALO, e, ux, uy, un, g, P, cs2);
          signal_speeds3(g, ux, uy, un, cs2, cx, cy, cn);
          sm.yaux[0][sy][lane] = g; sm.yaux[1][sy][lane] = P; sm.yaux[2][sy][lane] = cy;
        }
      }
      // (3) x-halo pass: one warp computes, for all rows, the left state of cell -1 and the right state of cell 32
      if (row == XHW && lane < 2 * TY) {
        const int r = lane & (TY - 1), side = lane / TY;
        const int sx_in = side ? TX + HALO : HALO - 1, sx_out = side ? TX + HALO + 1 : 0, sx_adj = side ? TX + HALO - 1 : HALO;
        const R* __restrict__ rowp = ringk + (r + HALO) * SX;
        R e, ux, uy, un, g, P, cs2, cx, cy, cn;
        derive(a.eos, rowp + sx_in, e, ux, uy, un, g, P, cs2);
        signal_speeds3(g, ux, uy, un, cs2, cx, cy, cn);
        sm.xaux[0][side][r] = g; sm.xaux[1][side][r] = P; sm.xaux[2][side][r] = cx;
        const PtAux<R> xin = pt_aux(e, g, ux, P);
        derive(a.eos, rowp + sx_out, e, ux, uy, un, g, P, cs2);
        const PtAux<R> xout = pt_aux(e, g, ux, P);
        derive(a.eos, rowp + sx_adj, e, ux, uy, un, g, P, cs2);
        const PtAux<R> xadj = pt_aux(e, g, ux, P);
        // along +x the three points are (out, in, adj) on the left side and (adj, in, out) on the right side
        const R* __restrict__ pm = rowp + (side ? sx_adj : sx_out);
        const R* __restrict__ pp = rowp + (side ? sx_out : sx_adj);
        const PtAux<R> xm = side ? xadj : xout, xpl = side ? xout : xadj;
#pragma unroll 2
        for (int f = 0; f < NFS; ++f) {
          R Qm, Fm, Q0, F0, Qp, Fp, QL, QR, FL, FR;
          qf<R, USE_PI>(pm, xm, f, 0, Qm, Fm);
          qf<R, USE_PI>(rowp + sx_in, xin, f, 0, Q0, F0);
          qf<R, USE_PI>(pp, xpl, f, 0, Qp, Fp);
          lr(Qm, Q0, Qp, a.theta, QL, QR);
          lr(Fm, F0, Fp, a.theta, FL, FR);
          sm.xh[f][side][0][r] = side ? QR : QL;
          sm.xh[f][side][1][r] = side ? FR : FL;
        }
      }
      __syncthreads();

      // ---- x direction: states and faces by warp shuffle --------------------------------------------------------------
      R gxm = shfl_up_(g0), Pxm = shfl_up_(P0), cxm = shfl_up_(h2.cx);
      R gxp = shfl_dn_(g0), Pxp = shfl_dn_(P0), cxp = shfl_dn_(h2.cx);
      if (lane == 0) { gxm = sm.xaux[0][0][row]; Pxm = sm.xaux[1][0][row]; cxm = sm.xaux[2][0][row]; }
      if (lane == TX - 1) { gxp = sm.xaux[0][1][row]; Pxp = sm.xaux[1][1][row]; cxp = sm.xaux[2][1][row]; }
      {
        const PtAux<R> x0 = pt_aux(e0, g0, ux0, P0);
        const PtAux<R> xm = pt_aux(rk[-1], gxm, rk[FST - 1], Pxm);
        const PtAux<R> xpl = pt_aux(rk[1], gxp, rk[FST + 1], Pxp);
        const R cl = max_(cxm, h2.cx), cr = max_(h2.cx, cxp);
#pragma unroll
        for (int f = 0; f < NFS; ++f) {
          R Qm, Fm, Q0, F0, Qp, Fp, QL, QR, FL, FR;
          qf<R, USE_PI>(rk - 1, xm, f, 0, Qm, Fm);
          qf<R, USE_PI>(rk, x0, f, 0, Q0, F0);
          qf<R, USE_PI>(rk + 1, xpl, f, 0, Qp, Fp);
          lr(Qm, Q0, Qp, a.theta, QL, QR);
          lr(Fm, F0, Fp, a.theta, FL, FR);
          R QRn = shfl_dn_(QR), FRn = shfl_dn_(FR);
          if (lane == TX - 1) { QRn = sm.xh[f][1][0][row]; FRn = sm.xh[f][1][1][row]; }
          const R Hr = face2(QL, FL, QRn, FRn, cr);
          R Hl = shfl_up_(Hr);
          if (lane == 0) Hl = face2(sm.xh[f][0][0][row], sm.xh[f][0][1][row], QR, FR, cl);
          S[f] -= (Hr - Hl) * (f < 4 ? sc_x * tf : sc_x);
        }
      }

      // ---- y direction: states through the shared-memory exchange, one barrier per field ------------------------------
      const R gym = sm.yaux[0][row + HALO - 1][lane], Pym = sm.yaux[1][row + HALO - 1][lane],
              cym = sm.yaux[2][row + HALO - 1][lane];
      const R gyp = sm.yaux[0][row + HALO + 1][lane], Pyp = sm.yaux[1][row + HALO + 1][lane],
              cyp = sm.yaux[2][row + HALO + 1][lane];
      {
        const PtAux<R> y0 = pt_aux(e0, g0, uy0, P0);
        const PtAux<R> ym = pt_aux(rk[-SX], gym, rk[2 * FST - SX], Pym);
        const PtAux<R> ypl = pt_aux(rk[SX], gyp, rk[2 * FST + SX], Pyp);
        const R cd = max_(cym, h2.cy), cu = max_(h2.cy, cyp);
        // outer halo row of the first / last warp (row -2 or 9)
        const int so = row == 0 ? -2 * SX : 2 * SX;
        const int syo = row == 0 ? 0 : SY - 1;
        PtAux<R> yo = y0;
        if (row == 0 || row == TY - 1) yo = pt_aux(rk[so], sm.yaux[0][syo][lane], rk[2 * FST + so], sm.yaux[1][syo][lane]);
        int buf = 0;
#pragma unroll
        for (int f = 0; f < NFS; ++f) {
          R Qm, Fm, Q0, F0, Qp, Fp, QL, QR, FL, FR;
          qf<R, USE_PI>(rk - SX, ym, f, 1, Qm, Fm);
          qf<R, USE_PI>(rk, y0, f, 1, Q0, F0);
          qf<R, USE_PI>(rk + SX, ypl, f, 1, Qp, Fp);
          lr(Qm, Q0, Qp, a.theta, QL, QR);
          lr(Fm, F0, Fp, a.theta, FL, FR);
          sm.yx[buf][0][row][lane] = QL; sm.yx[buf][1][row][lane] = FL;
          sm.yx[buf][2][row][lane] = QR; sm.yx[buf][3][row][lane] = FR;
          R QLn = R(0), FLn = R(0), QRn = R(0), FRn = R(0);
          if (row == 0) {              // left state of row -1 from rows -2, -1, 0
            R Qo, Fo, t0, t1;
            qf<R, USE_PI>(rk + so, yo, f, 1, Qo, Fo);
            lr(Qo, Qm, Q0, a.theta, QLn, t0);
            lr(Fo, Fm, F0, a.theta, FLn, t1);
          }
          if (row == TY - 1) {         // right state of row 8 from rows 7, 8, 9
            R Qo, Fo, t0, t1;
            qf<R, USE_PI>(rk + so, yo, f, 1, Qo, Fo);
            lr(Q0, Qp, Qo, a.theta, t0, QRn);
            lr(F0, Fp, Fo, a.theta, t1, FRn);
          }
          __syncthreads();
          if (row != TY - 1) { QRn = sm.yx[buf][2][row + 1][lane]; FRn = sm.yx[buf][3][row + 1][lane]; }
          if (row != 0) { QLn = sm.yx[buf][0][row - 1][lane]; FLn = sm.yx[buf][1][row - 1][lane]; }
          const R Hu = face2(QL, FL, QRn, FRn, cu);
          const R Hd = face2(QLn, FLn, QR, FR, cd);
          S[f] -= (Hu - Hd) * (f < 4 ? sc_y * tf : sc_y);
          buf ^= 1;
        }
      }

      // ---- cell-centre state, velocity gradients (A9) -----------------------------------------------------------------
      Cell<R> cc, cn_;
      cc.e = e0; cc.P = P0; cc.u[0] = g0; cc.u[1] = ux0; cc.u[2] = uy0; cc.u[3] = un0;
#pragma unroll
      for (int m = 0; m < 10; ++m) cc.pi[m] = USE_PI ? rk[(4 + m) * FST] : R(0);
      R grad[4][4];
#pragma unroll
      for (int m = 0; m < 4; ++m)
#pragma unroll
        for (int n = 0; n < 4; ++n) grad[m][n] = R(0);
      if (USE_PI) {
        grad[1][0] = (gxp - gxm) * sc_x;
        grad[2][0] = (gyp - gym) * sc_y;
        grad[3][0] = (h1.g - km1[0]) * sc_eta;
#pragma unroll
        for (int n = 1; n < 4; ++n) {
          grad[1][n] = (rk[n * FST + 1] - rk[n * FST - 1]) * sc_x;
          grad[2][n] = (rk[n * FST + SX] - rk[n * FST - SX]) * sc_y;
          grad[3][n] = (r1[n * FST] - km1[n]) * sc_eta;
        }
      }
      const int ic = active ? i : 0, jc = active ? j : 0;
      const long long cell = (long long)(k + HALO) * a.pz + (long long)(jc + HALO) * a.py + (ic + HALO);
      if (MODE == 2) {
        const R* __restrict__ sn = a.sn + cell;
        cn_.e = sn[0]; cn_.u[1] = sn[a.pf]; cn_.u[2] = sn[2 * a.pf]; cn_.u[3] = sn[3 * a.pf];
        cn_.u[0] = sqrt_(R(1) + cn_.u[1] * cn_.u[1] + cn_.u[2] * cn_.u[2] + cn_.u[3] * cn_.u[3]);
        R cs2n;
        eos_P(a.eos, cn_.e, cn_.P, cs2n);
#pragma unroll
        for (int m = 0; m < 10; ++m) cn_.pi[m] = VISC ? sn[(4 + m) * a.pf] : R(0);
      }
      R up3[3] = {R(0), R(0), R(0)};
      R gst = R(1);
      if (USE_PI) {
        if (MODE == 1) {
          const R* __restrict__ up = a.uprev + cell;
          up3[0] = up[0]; up3[1] = up[a.pf]; up3[2] = up[2 * a.pf];
        } else {
          gst = a.gstar[cell];
        }
      }

      // ---- sources, stage update, root-find, limiter (hydro_stage_update.cuh) -----------------------------------------
      unsigned flags = 0;
      Cell<R> nw;
      R cs2_new;
      stage_update<R, VISC, MODE>(a, S, cc, cn_, grad, up3, gst, nw, cs2_new, flags);

      // ---- store the new state and its ghost images (boundary rule a11) -----------------------------------------------
      if (active) {
        R* __restrict__ out = a.out + cell;
        if (MODE == 0) {
          out[0] = R(2) * ux0 - nw.u[1]; out[a.pf] = R(2) * uy0 - nw.u[2]; out[2 * a.pf] = R(2) * un0 - nw.u[3];
        } else {
          int gl[12];
          int ng[3] = {0, 0, 0};
          if (i < 2 || i >= a.nx - 2) ng[0] = ghost_list(i, a.nx, a.bc[0], gl);
          if (j < 2 || j >= a.ny - 2) ng[1] = ghost_list(j, a.ny, a.bc[1], gl + 4);
          if (k < 2 || k >= a.nz - 2) ng[2] = ghost_list(k, a.nz, a.bc[2], gl + 8);
          auto put = [&](int f, R v) {
            R* __restrict__ o = out + (long long)f * a.pf;
            o[0] = v;
            for (int t = 0; t < ng[0]; ++t) o[gl[t] - i] = v;
            for (int t = 0; t < ng[1]; ++t) o[(long long)(gl[4 + t] - j) * a.py] = v;
            for (int t = 0; t < ng[2]; ++t) o[(long long)(gl[8 + t] - k) * a.pz] = v;
          };
          put(0, nw.e); put(1, nw.u[1]); put(2, nw.u[2]); put(3, nw.u[3]);
          if (VISC) {
#pragma unroll
            for (int m = 0; m < 10; ++m) put(4 + m, nw.pi[m]);
            if (MODE == 1) a.gstar[cell] = gst;
          }
        }
      }
      if (MODE != 0) {
        if (!active) flags = 0;
        count_flags(a.diag, flags);
        if (active) {
          if (MODE == 1) {
            cfl0 = max_(cfl0, h2.cx * a.h * a.scale[0]); cfl1 = max_(cfl1, h2.cy * a.h * a.scale[1]);
            cfl2 = max_(cfl2, h2.cn * a.h * a.scale[2]);
          } else {
            emax = max_(emax, nw.e);
          }
        }
      }
    }

    // ---- rotate the per-column history; free the stage of plane p-2 and refill it with plane p+2 ----------------------
    if (it >= 2) { km1[0] = h2.g; km1[1] = r2[FST]; km1[2] = r2[2 * FST]; km1[3] = r2[3 * FST]; }
    h2 = h1; h1 = hp;
    __syncthreads();
    if (tid == 0 && it >= 2 && p + 2 <= p_last) {
      mbar_expect_tx(&sm.bar[(p + 2) & 3], STAGE_BYTES);
      tma_load_plane(&sm.ring[(p + 2) & 3][0][0][0], &tmap, &sm.bar[(p + 2) & 3], X0, Y0, p + 2 + HALO);
    }
  }

  // ---- reductions (row a10): one atomic per warp per block ------------------------------------------------------------
  if (MODE != 0) {
    if (MODE == 1) {
      const double r0 = warp_max((double)cfl0), r1m = warp_max((double)cfl1), r2m = warp_max((double)cfl2);
      if (lane == 0) {
        atomic_max_nonneg(&a.diag->cfl[a.slot][0], r0);
        atomic_max_nonneg(&a.diag->cfl[a.slot][1], r1m);
        atomic_max_nonneg(&a.diag->cfl[a.slot][2], r2m);
      }
    } else {
      const double r = warp_max((double)emax);
      if (lane == 0) atomic_max_nonneg(&a.diag->emax[a.slot], r);
    }
    if (blockIdx.x == 0 && tid == 0) {
      // reset the slot the NEXT user will accumulate into (no kernel of this stage touches it)
      if (MODE == 1) a.diag->emax[a.slot] = 0ull;
      else { a.diag->cfl[a.slot ^ 1][0] = 0ull; a.diag->cfl[a.slot ^ 1][1] = 0ull; a.diag->cfl[a.slot ^ 1][2] = 0ull; }
    }
  }
}

template <typename R, bool VISC, int MODE>
cudaError_t launch_stage_tile(const TileArgs<R>& a, const CUtensorMap& tmap, cudaStream_t stream) {
  constexpr bool USE_PI = VISC && (MODE != 0);
  constexpr int NFS = USE_PI ? 14 : 4;
  const size_t smem = sizeof(TileSmem<R, NFS, NFS>);
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(stage_tile_kernel<R, VISC, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  const unsigned nblocks = (unsigned)(a.ntx * a.nty * a.nchunk);
  stage_tile_kernel<R, VISC, MODE><<<nblocks, TILE_THREADS, smem, stream>>>(a, tmap);
  return cudaGetLastError();
}

}  // namespace clv
