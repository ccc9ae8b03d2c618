// hydro_stage_tile.cuh -- "kernel 3": the tile / marching stage kernel (default).
//
// One launch per RK2 stage, like kernels 1 and 2, but every limited slope and every KT face flux is computed ONCE
// and shared by the cells that use it (kernels 1/2: every slope 3x, every face 2x; profiles/round1_kernel2.md).
//
//   * State buffers are plain SoA with two ghost layers per side: [field][nz+4][ny+4][pitch], 14 words per cell
//     (e, u~^x, u~^y, u~^eta, pi~[10]); nothing derived is stored ("16 floats per cell").
//   * A block owns a 32 x 8 xy tile and MARCHES along eta_s through a z-chunk.  Each plane of the tile with its
//     2-cell halo (36 x 12 points x 14 fields) arrives by ONE TMA box load (cp.async.bulk.tensor.4d + mbarrier)
//     into a 3-stage shared-memory ring: the point the paper could not reach for want of local memory
//     (7^3 block, 56 KB) -- a B200 SM has 227 KB.
//   * eta_s direction: a register pipeline per column.  When plane p arrives, the slope of cell p-1, the face
//     p-3/2 and the flux difference of cell k = p-2 are completed from the kept left state (Q^l, F^l) and face flux
//     of the previous step: one slope and one face per cell per field.
//   * x direction: lanes of a warp are 32 consecutive x cells; left/right states and face fluxes travel by warp
//     shuffle.
//   * y direction: warps are rows; left/right states travel through a double-buffered shared-memory exchange, one
//     block barrier per PAIR of fields (two fields per trip: their minmod chains interleave).
//   * The halo cells (x: -2, -1, 32, 33; y: rows -2, -1, 8, 9) are served by small warp-sized TASKS spread over
//     warps 1..5: five tasks per plane derive g, P, c of the 160 halo points, five tasks per trip form the states of
//     the cells just outside the tile for the next trip's fields.
//   * P, u~^tau and the signal speeds c_x, c_y, c_eta are derived once per loaded point (interior: on arrival of its
//     plane; halo: in the halo passes), never stored in HBM.
//   * Boundaries (row a11): the producing kernel writes the ghost cells itself (clamp: copies of the edge cell;
//     periodic: copies of the opposite edge), so the TMA boxes never need an index map.
//   * The loops over the 4 T fields and the 10 pi fields are ROLLED: their bodies (~250 instructions) stay in the
//     instruction cache (fully unrolled, the 10 k-instruction kernel stalled 4.8 warps per issue on instruction
//     fetch, profiles/round2_kernel3.md).  The per-column state that must survive from field to field and from plane
//     to plane -- the eta pipeline (Q^l, F^l, H per field) and the 14 flux sums -- is therefore indexed at run time
//     and lives in TENSOR MEMORY: each thread owns 112 (fp64) / 56 (fp32) 32-bit columns of its TMEM lane
//     (tcgen05.st / tcgen05.ld, shape 32x32b), because 4 ring stages of fp64 planes leave no shared memory for it
//     and registers cannot be indexed.  No tensor-core instruction is issued; TMEM is used as a private scratchpad.
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
constexpr int NSTAGE = 3;
constexpr int TILE_THREADS = TX * TY;

template <typename R>
struct TileArgs {
  int nx, ny, nz;
  // ghosted SoA buffer: element(field f, cell i,j,k) = f*pf + (k+2)*pz + (j+2)*py + (i+2)
  long long py, pz, pf;
  int bc[3];
  int milne;
  R tau, inv_tau, tf_n, tf_1, inv_tf_1, h, inv_h;
  R scale[3];
  R theta, e_floor, xi, v_max, inv_5etas_hbarc, inv_ctau, lam1;
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
  R yx[2][2][4][TY][TX];            // y exchange [buffer][field of the trip][Q^l, F^l, Q^r, F^r][row][lane]
  R yaux[3][SY][TX];                // g, P, c_y of rows -2..9 (interior columns)
  R xaux[3][2][2][TY];              // g, P, c_x of the x-halo cells [side][0 inner, 1 outer][row]
  R xh[2][2][2][2][TY];             // x-halo states [trip parity][field of the trip][side][Q, F][row]
                                    //   side 0: Q^l, F^l of cell -1;  side 1: Q^r, F^r of cell 32
  R yh[3][2][2][2][TX];             // y-halo states [trip mod 3][field of the trip][side][Q, F][lane]  (rows -1 / 8)
  unsigned long long bar[NSTAGE];
  unsigned tmem_base;               // written by tcgen05.alloc
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
// Q and F_a of an evolved field at a point whose raw words sit at pt[field * FST]  (Eq.27, 29, 39; the factor tau of
// the T fields is applied to the flux difference).  AX = axis of the flux.  The field index is a run-time value.
//   T field mu:   Q = (e+P) g u^mu - P delta^{mu tau} + pi^{tau mu},   F_a = (e+P) u^a u^mu + P delta^{a mu} + pi^{a mu}
//   pi field m:   Q = g pi_m,   F_a = u^a pi_m
template <typename R, bool USE_PI, int AX, bool IS_T>
__device__ __forceinline__ void qf(const R* __restrict__ pt, const PtAux<R>& x, int f, R& Q, R& Fl) {
  if (IS_T) {
    const R umu = f == 0 ? x.g : pt[f * FST];
    Q = x.wg * umu; Fl = x.wua * umu;
    if (f == 0) Q -= x.P;
    if (f == AX + 1) Fl += x.P;
    if (USE_PI) { Q += pt[(4 + f) * FST]; Fl += pt[(4 + pidx_f(AX + 1, f)) * FST]; }
  } else {
    const R v = pt[f * FST];
    Q = x.g * v; Fl = x.ua * v;
  }
}
// half-slope states of a cell: Q^l = Q + s/2 (left state of its upper face), Q^r = Q - s/2   (Eq.43-44, A4)
template <typename R>
__device__ __forceinline__ void lr(R Qm, R Q0, R Qp, R th2, R& L, R& Rr) {
  const R s4 = hmm4(Q0 - Qm, Qp - Q0, th2);      // 4 x the half slope
  L = R(0.25) * s4 + Q0; Rr = R(-0.25) * s4 + Q0;
}
// 2 H_{i+1/2} from the left state of cell i and the right state of cell i+1   (Eq.41-42, A5)
template <typename R>
__device__ __forceinline__ R face2(R QL, R FL, R QRn, R FRn, R c) { return (FL + FRn) - c * (QRn - QL); }

__device__ __forceinline__ double shfl_up_(double v) { return __shfl_up_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ float shfl_up_(float v) { return __shfl_up_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ double shfl_dn_(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ float shfl_dn_(float v) { return __shfl_down_sync(0xffffffffu, v, 1); }

// ---- tensor memory as a per-thread scratchpad -------------------------------------------------------------------------
// Shape 32x32b: lane l of warp w reads / writes TMEM lane 32 (w % 4) + l, so every thread owns one TMEM lane segment.
// The two warps that share a lane quadrant (w and w + 4) use disjoint column ranges.
__device__ __forceinline__ void tm_st(unsigned addr, double v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(addr), "r"(__double2loint(v)),
               "r"(__double2hiint(v)) : "memory");
}
__device__ __forceinline__ void tm_st(unsigned addr, float v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(addr), "r"(__float_as_int(v)) : "memory");
}
// three consecutive values (issue the loads, then one wait; the wait carries the registers so that no use can be
// scheduled before it)
__device__ __forceinline__ void tm_ld3(unsigned addr, double& a, double& b, double& c) {
  int r0, r1, r2, r3, r4, r5;
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
               : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr) : "memory");
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(r4), "=r"(r5) : "r"(addr + 4) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" : "+r"(r0), "+r"(r1), "+r"(r2), "+r"(r3), "+r"(r4), "+r"(r5)::"memory");
  a = __hiloint2double(r1, r0); b = __hiloint2double(r3, r2); c = __hiloint2double(r5, r4);
}
__device__ __forceinline__ void tm_ld3(unsigned addr, float& a, float& b, float& c) {
  int r0, r1, r2;
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(r0), "=r"(r1) : "r"(addr) : "memory");
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(r2) : "r"(addr + 2) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" : "+r"(r0), "+r"(r1), "+r"(r2)::"memory");
  a = __int_as_float(r0); b = __int_as_float(r1); c = __int_as_float(r2);
}
__device__ __forceinline__ void tm_ld1(unsigned addr, double& a) {
  int r0, r1;
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(r0), "=r"(r1) : "r"(addr) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" : "+r"(r0), "+r"(r1)::"memory");
  a = __hiloint2double(r1, r0);
}
__device__ __forceinline__ void tm_ld1(unsigned addr, float& a) {
  int r0;
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(r0) : "r"(addr) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" : "+r"(r0)::"memory");
  a = __int_as_float(r0);
}
// issue only (no wait): the caller batches several loads in front of one tm_wait_ld
__device__ __forceinline__ void tm_ld_issue(unsigned addr, int& lo, int& hi) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(lo), "=r"(hi) : "r"(addr) : "memory");
}
__device__ __forceinline__ void tm_ld_issue(unsigned addr, int& lo) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(lo) : "r"(addr) : "memory");
}
__device__ __forceinline__ void tm_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// Private per-thread store of NV values of type R in tensor memory.  Word layout of a thread (W = words per value):
//   [ kept: 3 values per field (Q^l, F^l, 2H) ][ S: one value per field ]
template <typename R>
struct PrivTmem {
  static constexpr int W = sizeof(R) / 4;
  static constexpr int COLS_PER_THREAD = 14 * 4 * W;          // 112 (fp64) / 56 (fp32)
  static constexpr int ALLOC_COLS = 2 * COLS_PER_THREAD <= 128 ? 128 : 256;
  unsigned base;
  __device__ __forceinline__ void init(unsigned tmem_base, int warp) {
    base = tmem_base + ((unsigned)(32 * (warp & 3)) << 16) + (unsigned)((warp >> 2) * COLS_PER_THREAD);
  }
  __device__ __forceinline__ void get_kept(int f, R& ql, R& fl, R& h) const { tm_ld3(base + f * 3 * W, ql, fl, h); }
  __device__ __forceinline__ void put_kept(int f, R ql, R fl, R h) const {
    tm_st(base + f * 3 * W, ql); tm_st(base + (f * 3 + 1) * W, fl); tm_st(base + (f * 3 + 2) * W, h);
  }
  __device__ __forceinline__ void put_S(int f, R v) const { tm_st(base + (42 + f) * W, v); }
  __device__ __forceinline__ void get_S(int f, R& v) const { tm_ld1(base + (42 + f) * W, v); }
  // all flux sums with one wait
  template <int N>
  __device__ __forceinline__ void get_S_all(R (&S)[14]) const {
    int lo[N], hi[N];
#pragma unroll
    for (int f = 0; f < N; ++f) {
      if (W == 2) tm_ld_issue(base + (42 + f) * W, lo[f], hi[f]);
      else { tm_ld_issue(base + (42 + f) * W, lo[f]); hi[f] = 0; }
    }
    tm_wait_ld();
#pragma unroll
    for (int f = 0; f < N; ++f) {
      // the empty asm ties the register to a point after the wait
      asm volatile("" : "+r"(lo[f]), "+r"(hi[f]));
      if (W == 2) S[f] = (R)__hiloint2double(hi[f], lo[f]);
      else S[f] = (R)__int_as_float(lo[f]);
    }
  }
};

template <typename R>
struct PlaneAux {   // derived once per column when its plane arrives
  R g, P, cx, cy, cn;
};

// g, P, c_s^2 of a raw point
template <typename R>
__device__ __forceinline__ void derive(const EosDev<R>& eos, const R* __restrict__ pt, R& e, R& ux, R& uy, R& un, R& g,
                                       R& P, R& cs2) {
  e = pt[0]; ux = pt[FST]; uy = pt[2 * FST]; un = pt[3 * FST];
  g = fsqrt_(R(1) + ux * ux + uy * uy + un * un);
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
__global__ void __launch_bounds__(TILE_THREADS, (sizeof(R) == 4 ? 2 : 1))
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
        mbar_expect_tx(&sm.bar[s], STAGE_BYTES);
        tma_load_plane(&sm.ring[s][0][0][0], &tmap, &sm.bar[s], X0, Y0, p + HALO);
      }
    }
  }

  // ---- tensor memory: the per-thread scratchpad (allocated by warp 0, which also frees it) ------------------------------
  using Priv = PrivTmem<R>;
  if (row == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&sm.tmem_base)),
                 "r"((unsigned)Priv::ALLOC_COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  Priv priv;
  priv.init(sm.tmem_base, row);
#pragma unroll 1
  for (int f = 0; f < NFS; ++f) { priv.put_kept(f, R(0), R(0), R(0)); priv.put_S(f, R(0)); }
  tm_wait_st();

  // ---- per-thread state that lives across planes --------------------------------------------------------------------
  PlaneAux<R> h1 = {R(1), R(0), R(0), R(0), R(0)}, h2 = h1;      // planes p-1 and p-2
  R km1[4] = {R(1), R(0), R(0), R(0)};                            // u~^mu of plane k-1
  const R tf = a.milne ? a.tau : R(1);
  const R th2 = R(2) * a.theta;
  const R sc_eta = R(0.5) * a.scale[2], sc_x = R(0.5) * a.scale[0], sc_y = R(0.5) * a.scale[1];
  R cfl0 = R(0), cfl1 = R(0), cfl2 = R(0), emax = R(0);

  const int own = (row + HALO) * SX + (lane + HALO);     // own point inside a field plane of a stage
  const bool edge_lo = row == 0, edge_hi = row == TY - 1;
  constexpr int NTRIP = NFS / 2;                         // two fields per trip: T fields trips 0-1, pi fields 2-6
  int sp = 0, s1 = 2, s2 = 1;                            // ring stages of planes p, p-1, p-2  (p - p_first mod 3)

  for (int p = p_first; p <= p_last; ++p) {
    const int it = p - p_first;
    mbar_wait(&sm.bar[sp], (unsigned)((it / 3) & 1));
    const R* __restrict__ rp = &sm.ring[sp][0][0][0] + own;
    const R* __restrict__ r1 = &sm.ring[s1][0][0][0] + own;     // plane p-1 = k+1
    const R* __restrict__ rk = &sm.ring[s2][0][0][0] + own;     // plane p-2 = k
    bool released = false;

    // ---- arrival of plane p: derived quantities of the own column ---------------------------------------------------
    PlaneAux<R> hp;
    R e_p, ux_p, uy_p, un_p;
    {
      R cs2;
      derive(a.eos, rp, e_p, ux_p, uy_p, un_p, hp.g, hp.P, cs2);
      signal_speeds3(hp.g, ux_p, uy_p, un_p, cs2, hp.cx, hp.cy, hp.cn);
    }
    const R ux0 = rk[FST], uy0 = rk[2 * FST], un0 = rk[3 * FST];      // (garbage before plane k exists: unused then)

    if (p >= kc0) {
      const bool centre = p - 2 >= kc0;        // block-uniform
      const int k = p - 2;
      const R e0 = rk[0];
      const R g0 = h2.g, P0 = h2.P;
      const R* __restrict__ ringk = &sm.ring[s2][0][0][0];
      R gxm = g0, Pxm = P0, cxm = h2.cx, gxp = g0, Pxp = P0, cxp = h2.cx;
      R gym = g0, Pym = P0, cym = h2.cy, gyp = g0, Pyp = P0, cyp = h2.cy;

      // ---- halo tasks (warps 1..5, one warp-sized task each) ----------------------------------------------------------
      // states of the cells just outside the tile for the two fields fa, fa+1 of trip t
      auto halo_states = [&](int t) {
        const int fa = 2 * t;
        if (row == 1) {                  // x: lane = (field of the trip, side, row)
          const int slot = lane >> 4, side = (lane >> 3) & 1, r = lane & (TY - 1), f = fa + slot;
          const int sx_in = side ? TX + HALO : HALO - 1;
          const R* __restrict__ pt = ringk + (r + HALO) * SX + sx_in;
          // along +x: (outer, inner, interior cell 0) on the left, (interior cell 31, inner, outer) on the right
          const int cin = side ? TX - 1 : 0;
          const PtAux<R> xin = pt_aux(pt[0], sm.xaux[0][side][0][r], pt[FST], sm.xaux[1][side][0][r]);
          const PtAux<R> xout = pt_aux(pt[side ? 1 : -1], sm.xaux[0][side][1][r], pt[FST + (side ? 1 : -1)], sm.xaux[1][side][1][r]);
          const PtAux<R> xadj = pt_aux(pt[side ? -1 : 1], sm.yaux[0][r + HALO][cin], pt[FST + (side ? -1 : 1)], sm.yaux[1][r + HALO][cin]);
          const PtAux<R> xm = side ? xadj : xout, xpl = side ? xout : xadj;
          R Qm, Fm, Q0, F0, Qp, Fp, QL, QR, FL, FR;
          if (f < 4) {
            qf<R, USE_PI, 0, true>(pt - 1, xm, f, Qm, Fm); qf<R, USE_PI, 0, true>(pt, xin, f, Q0, F0);
            qf<R, USE_PI, 0, true>(pt + 1, xpl, f, Qp, Fp);
          } else {
            qf<R, USE_PI, 0, false>(pt - 1, xm, f, Qm, Fm); qf<R, USE_PI, 0, false>(pt, xin, f, Q0, F0);
            qf<R, USE_PI, 0, false>(pt + 1, xpl, f, Qp, Fp);
          }
          lr(Qm, Q0, Qp, th2, QL, QR);
          lr(Fm, F0, Fp, th2, FL, FR);
          sm.xh[t & 1][slot][side][0][r] = side ? QR : QL;
          sm.xh[t & 1][slot][side][1][r] = side ? FR : FL;
        } else if (row >= 2 && row <= 5) {     // y: warp = (side, field of the trip), lanes along x
          const int side = (row - 2) >> 1, slot = (row - 2) & 1, f = fa + slot;
          const int sy_in = side ? SY - 2 : 1;
          const R* __restrict__ pt = ringk + sy_in * SX + lane + HALO;
          const PtAux<R> ya = pt_aux(pt[-SX], sm.yaux[0][sy_in - 1][lane], pt[2 * FST - SX], sm.yaux[1][sy_in - 1][lane]);
          const PtAux<R> yb = pt_aux(pt[0], sm.yaux[0][sy_in][lane], pt[2 * FST], sm.yaux[1][sy_in][lane]);
          const PtAux<R> yc = pt_aux(pt[SX], sm.yaux[0][sy_in + 1][lane], pt[2 * FST + SX], sm.yaux[1][sy_in + 1][lane]);
          R Qm, Fm, Q0, F0, Qp, Fp, QL, QR, FL, FR;
          if (f < 4) {
            qf<R, USE_PI, 1, true>(pt - SX, ya, f, Qm, Fm); qf<R, USE_PI, 1, true>(pt, yb, f, Q0, F0);
            qf<R, USE_PI, 1, true>(pt + SX, yc, f, Qp, Fp);
          } else {
            qf<R, USE_PI, 1, false>(pt - SX, ya, f, Qm, Fm); qf<R, USE_PI, 1, false>(pt, yb, f, Q0, F0);
            qf<R, USE_PI, 1, false>(pt + SX, yc, f, Qp, Fp);
          }
          lr(Qm, Q0, Qp, th2, QL, QR);
          lr(Fm, F0, Fp, th2, FL, FR);
          sm.yh[t % 3][slot][side][0][lane] = side ? QR : QL;
          sm.yh[t % 3][slot][side][1][lane] = side ? FR : FL;
        }
      };

      if (centre) {
        // own g, P, c_y for the y neighbours and the halo tasks
        sm.yaux[0][row + HALO][lane] = g0; sm.yaux[1][row + HALO][lane] = P0; sm.yaux[2][row + HALO][lane] = h2.cy;
        // derived quantities of the 160 halo points: five tasks
        if (row >= 1 && row <= 5) {
          int sy, sx;
          if (row == 1) {          // the 32 x-halo points: lane = (side, depth, row)
            const int side = lane >> 4, depth = (lane >> 3) & 1, r = lane & (TY - 1);
            sy = r + HALO; sx = side ? TX + HALO + depth : HALO - 1 - depth;
          } else {                 // one y-halo row
            sy = row == 2 ? 0 : (row == 3 ? 1 : (row == 4 ? SY - 2 : SY - 1)); sx = lane + HALO;
          }
          R e, ux, uy, un, g, P, cs2, cx, cy, cn;
          derive(a.eos, ringk + sy * SX + sx, e, ux, uy, un, g, P, cs2);
          signal_speeds3(g, ux, uy, un, cs2, cx, cy, cn);
          if (row == 1) {
            const int side = lane >> 4, depth = (lane >> 3) & 1, r = lane & (TY - 1);
            sm.xaux[0][side][depth][r] = g; sm.xaux[1][side][depth][r] = P; sm.xaux[2][side][depth][r] = cx;
          } else {
            sm.yaux[0][sy][lane] = g; sm.yaux[1][sy][lane] = P; sm.yaux[2][sy][lane] = cy;
          }
        }
        __syncthreads();
        halo_states(0);
        // neighbour quantities: x by shuffle (edges from the x-halo cells), y from the shared rows
        gxm = shfl_up_(g0); Pxm = shfl_up_(P0); cxm = shfl_up_(h2.cx);
        gxp = shfl_dn_(g0); Pxp = shfl_dn_(P0); cxp = shfl_dn_(h2.cx);
        if (lane == 0) { gxm = sm.xaux[0][0][0][row]; Pxm = sm.xaux[1][0][0][row]; cxm = sm.xaux[2][0][0][row]; }
        if (lane == TX - 1) { gxp = sm.xaux[0][1][0][row]; Pxp = sm.xaux[1][1][0][row]; cxp = sm.xaux[2][1][0][row]; }
        gym = sm.yaux[0][row + HALO - 1][lane]; Pym = sm.yaux[1][row + HALO - 1][lane]; cym = sm.yaux[2][row + HALO - 1][lane];
        gyp = sm.yaux[0][row + HALO + 1][lane]; Pyp = sm.yaux[1][row + HALO + 1][lane]; cyp = sm.yaux[2][row + HALO + 1][lane];
        __syncthreads();
      }
      // the tail of this plane reads the cell's state n (stage 2) or history (stage 1) from global memory: start those
      // lines moving towards L1 now, behind the flux trips
      const int ic = active ? i : 0, jc = active ? j : 0;
      const long long cell = (long long)(k + HALO) * a.pz + (long long)(jc + HALO) * a.py + (ic + HALO);
      if (centre && (lane & 15) == 0) {      // one request per 128-byte line of the row
        if (MODE == 2) {
#pragma unroll
          for (int f = 0; f < (VISC ? 14 : 4); ++f) asm volatile("prefetch.global.L1 [%0];" ::"l"(a.sn + cell + f * a.pf));
          if (USE_PI) asm volatile("prefetch.global.L1 [%0];" ::"l"(a.gstar + cell));
        } else if (MODE == 1 && USE_PI) {
#pragma unroll
          for (int f = 0; f < 3; ++f) asm volatile("prefetch.global.L1 [%0];" ::"l"(a.uprev + cell + f * a.pf));
        }
      }
      // point quantities of the three stencils (eta: planes p, p-1, p-2; x: i-1, i, i+1; y: j-1, j, j+1)
      const PtAux<R> zp = pt_aux(e_p, hp.g, un_p, hp.P);
      const PtAux<R> z1 = pt_aux(r1[0], h1.g, r1[3 * FST], h1.P);
      const PtAux<R> z2 = pt_aux(e0, g0, un0, P0);
      const PtAux<R> x0 = pt_aux(e0, g0, ux0, P0);
      const PtAux<R> xm = pt_aux(rk[-1], gxm, rk[FST - 1], Pxm);
      const PtAux<R> xpl = pt_aux(rk[1], gxp, rk[FST + 1], Pxp);
      const PtAux<R> y0 = pt_aux(e0, g0, uy0, P0);
      const PtAux<R> ym = pt_aux(rk[-SX], gym, rk[2 * FST - SX], Pym);
      const PtAux<R> ypl = pt_aux(rk[SX], gyp, rk[2 * FST + SX], Pyp);
      const R cface = max_(h2.cn, h1.cn);
      const R cl = max_(cxm, h2.cx), cr = max_(h2.cx, cxp);
      const R cd = max_(cym, h2.cy), cu = max_(h2.cy, cyp);

      // first half of a field: eta pipeline step, x flux difference, y states into the exchange buffer
      auto phase_a = [&](auto is_t_tag, int f, int t, int slot, R& Sf, R& QLy, R& FLy, R& QRy, R& FRy) {
        constexpr bool IS_T = decltype(is_t_tag)::value;
        const R tfac = IS_T ? tf : R(1);
        {   // eta: slope of cell p-1, face p-3/2, flux difference of cell k = p-2
          R Qp, Fp, Q1, F1, Q2, F2, QL1, QR1, FL1, FR1, QLk, FLk, Hk;
          priv.get_kept(f, QLk, FLk, Hk);
          qf<R, USE_PI, 2, IS_T>(rp, zp, f, Qp, Fp);
          qf<R, USE_PI, 2, IS_T>(r1, z1, f, Q1, F1);
          qf<R, USE_PI, 2, IS_T>(rk, z2, f, Q2, F2);
          lr(Q2, Q1, Qp, th2, QL1, QR1);
          lr(F2, F1, Fp, th2, FL1, FR1);
          const R Hn = face2(QLk, FLk, QR1, FR1, cface);
          Sf = -(Hn - Hk) * (sc_eta * tfac);
          priv.put_kept(f, QL1, FL1, Hn);
        }
        if (centre) {
          {   // x: states and faces by warp shuffle
            R Qm, Fm, Q0, F0, Qp, Fp, QL, QR, FL, FR;
            qf<R, USE_PI, 0, IS_T>(rk - 1, xm, f, Qm, Fm);
            qf<R, USE_PI, 0, IS_T>(rk, x0, f, Q0, F0);
            qf<R, USE_PI, 0, IS_T>(rk + 1, xpl, f, Qp, Fp);
            lr(Qm, Q0, Qp, th2, QL, QR);
            lr(Fm, F0, Fp, th2, FL, FR);
            R QRn = shfl_dn_(QR), FRn = shfl_dn_(FR);
            if (lane == TX - 1) { QRn = sm.xh[t & 1][slot][1][0][row]; FRn = sm.xh[t & 1][slot][1][1][row]; }
            const R Hr = face2(QL, FL, QRn, FRn, cr);
            R Hl = shfl_up_(Hr);
            if (lane == 0) Hl = face2(sm.xh[t & 1][slot][0][0][row], sm.xh[t & 1][slot][0][1][row], QR, FR, cl);
            Sf -= (Hr - Hl) * (sc_x * tfac);
          }
          {   // y: states of the own cell
            R Qm, Fm, Q0, F0, Qp, Fp;
            qf<R, USE_PI, 1, IS_T>(rk - SX, ym, f, Qm, Fm);
            qf<R, USE_PI, 1, IS_T>(rk, y0, f, Q0, F0);
            qf<R, USE_PI, 1, IS_T>(rk + SX, ypl, f, Qp, Fp);
            lr(Qm, Q0, Qp, th2, QLy, QRy);
            lr(Fm, F0, Fp, th2, FLy, FRy);
            sm.yx[t & 1][slot][0][row][lane] = QLy; sm.yx[t & 1][slot][1][row][lane] = FLy;
            sm.yx[t & 1][slot][2][row][lane] = QRy; sm.yx[t & 1][slot][3][row][lane] = FRy;
          }
        }
      };
      // second half (after the barrier): y faces from the neighbours' states
      auto phase_b = [&](auto is_t_tag, int f, int t, int slot, R Sf, R QLy, R FLy, R QRy, R FRy) {
        constexpr bool IS_T = decltype(is_t_tag)::value;
        const R tfac = IS_T ? tf : R(1);
        R QRn, FRn, QLn, FLn;
        if (!edge_hi) { QRn = sm.yx[t & 1][slot][2][row + 1][lane]; FRn = sm.yx[t & 1][slot][3][row + 1][lane]; }
        else { QRn = sm.yh[t % 3][slot][1][0][lane]; FRn = sm.yh[t % 3][slot][1][1][lane]; }
        if (!edge_lo) { QLn = sm.yx[t & 1][slot][0][row - 1][lane]; FLn = sm.yx[t & 1][slot][1][row - 1][lane]; }
        else { QLn = sm.yh[t % 3][slot][0][0][lane]; FLn = sm.yh[t % 3][slot][0][1][lane]; }
        const R Hu = face2(QLy, FLy, QRn, FRn, cu);
        const R Hd = face2(QLn, FLn, QRy, FRy, cd);
        Sf -= (Hu - Hd) * (sc_y * tfac);
        priv.put_S(f, Sf);
      };
      auto trip = [&](auto is_t_tag, int t) {
        const int fa = 2 * t;
        R Sa, Sb, QLa, FLa, QRa, FRa, QLb, FLb, QRb, FRb;
        phase_a(is_t_tag, fa, t, 0, Sa, QLa, FLa, QRa, FRa);
        phase_a(is_t_tag, fa + 1, t, 1, Sb, QLb, FLb, QRb, FRb);
        if (centre) {
          if (t + 1 < NTRIP) halo_states(t + 1);
          __syncthreads();
          phase_b(is_t_tag, fa, t, 0, Sa, QLa, FLa, QRa, FRa);
          phase_b(is_t_tag, fa + 1, t, 1, Sb, QLb, FLb, QRb, FRb);
        }
      };
#pragma unroll
      for (int t = 0; t < 2; ++t) trip(std::true_type{}, t);      // unrolled: the T-field index is a constant
      if (USE_PI) {
#pragma unroll 1
        for (int t = 2; t < NTRIP; ++t) trip(std::false_type{}, t);
      }
      tm_wait_st();

      // ---- centre plane k: sources, update, root-find, store ----------------------------------------------------------
      if (centre) {
        R S[14];
#pragma unroll
        for (int f = NFS; f < 14; ++f) S[f] = R(0);
        priv.template get_S_all<NFS>(S);
        Cell<R> cc, cn_;
        cc.e = e0; cc.P = P0; cc.u[0] = g0; cc.u[1] = ux0; cc.u[2] = uy0; cc.u[3] = un0;
#pragma unroll
        for (int m = 0; m < 10; ++m) cc.pi[m] = USE_PI ? rk[(4 + m) * FST] : R(0);
        R grad[4][4];
#pragma unroll
        for (int m = 0; m < 4; ++m)
#pragma unroll
          for (int n = 0; n < 4; ++n) grad[m][n] = R(0);
        if (USE_PI) {      // spatial rows of nabla~_mu u~^nu by central differences (A9); eta row divided by tau (Eq.22)
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
        // everything the tail needs from plane k is in registers: free its ring stage for plane p+1 now, so that the
        // TMA load runs behind the sources / root-find instead of a fourth ring stage
        __syncthreads();
        released = true;
        if (tid == 0 && p + 1 <= p_last) {
          mbar_expect_tx(&sm.bar[s2], STAGE_BYTES);
          tma_load_plane(&sm.ring[s2][0][0][0], &tmap, &sm.bar[s2], X0, Y0, p + 1 + HALO);
        }
        if (MODE == 2) {
          const R* __restrict__ sn = a.sn + cell;
          cn_.e = sn[0]; cn_.u[1] = sn[a.pf]; cn_.u[2] = sn[2 * a.pf]; cn_.u[3] = sn[3 * a.pf];
#pragma unroll
          for (int m = 0; m < 10; ++m) cn_.pi[m] = VISC ? sn[(4 + m) * a.pf] : R(0);
          cn_.u[0] = fsqrt_(R(1) + cn_.u[1] * cn_.u[1] + cn_.u[2] * cn_.u[2] + cn_.u[3] * cn_.u[3]);
          R cs2n;
          eos_P(a.eos, cn_.e, cn_.P, cs2n);
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
        unsigned flags = 0;
        Cell<R> nw;
        R cs2_new;
        stage_update<R, VISC, MODE>(a, S, cc, cn_, grad, up3, gst, nw, cs2_new, flags);

        // store the new state and its ghost images (boundary rule a11)
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
    }

    // ---- rotate the per-column history and the ring; a stage that was not released above is released here ------------
    if (it >= 2) { km1[0] = h2.g; km1[1] = ux0; km1[2] = uy0; km1[3] = un0; }
    h2 = h1; h1 = hp;
    if (!released) {
      __syncthreads();
      if (tid == 0 && it >= 2 && p + 1 <= p_last) {
        mbar_expect_tx(&sm.bar[s2], STAGE_BYTES);
        tma_load_plane(&sm.ring[s2][0][0][0], &tmap, &sm.bar[s2], X0, Y0, p + 1 + HALO);
      }
    }
    { const int t = s2; s2 = s1; s1 = sp; sp = t; }
  }
  // free the tensor memory (same warp that allocated it; all loads are complete: every thread has waited on them)
  __syncthreads();
  if (row == 0) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(sm.tmem_base), "r"((unsigned)Priv::ALLOC_COLS)
                 : "memory");
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
