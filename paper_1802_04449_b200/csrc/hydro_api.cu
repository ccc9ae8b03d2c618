// hydro_api.cu -- context object and C ABI (include/clvisc_hydro.h) of the B200-native CLVisc step.
//
// Host side only sequences launches: every arithmetic step of the path runs in the CUDA kernels of
// hydro_stage_*.cuh / the load & read kernels below.  There is no CPU fallback.
//
// Workspace layout (caller-allocated device memory, 256-byte aligned pieces):
//   [diag 256 B][EoS tables 5 x kMaxEosNodes x elem][buf A][buf B][buf X][gstar]
// (each buf = nf evolved fields + 5 extended slots P, u^tau, c_x, c_y, c_eta used by kernel 2)
// buf A/B alternate as "state n" / "state n-1 (its u~^i is the history) -> state n+1"; buf X holds the
// stage-1 state '.  Each buf holds nft = nf + 5 fields (nf = 4 ideal, 14 viscous) in the blocked layout
// [k][j][x-block][field][32]: the 32 x-consecutive cells of one field are contiguous (one 256-byte / 128-byte
// warp transaction), and all fields of those 32 cells follow each other, so that inside a kernel the field
// offset is a compile-time immediate and a cell's whole state lies in one 4.8 KB stretch of DRAM.
// buf X (+gstar) doubles as the staging area for host-memory load/read between steps.
//
// Kernel 3 (the tile kernel) uses a different field store: plain SoA with two ghost layers per side,
//   [field][nz+4][ny+4][pitch]   (pitch = nx+4 rounded up to 16 bytes), nf = 4 / 14 fields and nothing derived,
// addressed by TMA tensor maps (one per buffer and box depth) that hydro_create encodes.
#include "../../include/clvisc_hydro.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "hydro_stage_ref.cuh"
#include "hydro_stage_fused.cuh"
#include "hydro_stage_tile.cuh"
#include "hydro_stage_march.cuh"
#include "hydro_freezeout.cuh"
#include "hydro_stage_strict.cuh"

namespace clv {

constexpr int kMaxEosNodes = 1 << 16;
constexpr double kHbarc = 0.1973269804;   // GeV fm (A18)

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct Layout {
  int soa;               // 0: blocked layout of kernels 1/2; 1: ghosted SoA of kernel 3
  long long py, pz, pf;  // soa: row, plane and field strides (elements)
  int nxb, blk, gp;      // x-blocks per row, elements per x-block (32 * nft), gstar row pitch
  long long sy, sz;      // row and plane strides (elements)
  long long nelem;       // elements of one state buffer
  int nf, nft;
  size_t elem;
  size_t off_diag, off_eos, off_buf[3], off_gstar, total;
};

// kernel 0 = the fastest one as measured on B200 (round 2, profiles/round2_bench.md): the marching
// per-cell kernel (4) from about 5e5 cells on (301x301x201: fp64 11.8 ms per step against 14.4 for kernel 2 and 15.7 for
// kernel 3, fp32 6.05 against 7.5 and 8.0; 201x201x105: 3.04 against 3.46 ms); below that a block that walks along eta_s
// leaves SMs idle and the per-cell kernel (2) wins (40x36x24: 0.063 against 0.111 ms; 33x33x17 ideal: 0.84 against 1.96 ms
// for 40 steps).  Kernels 2 and 4 share the field store, so the choice does not change the workspace.
static int resolve_kernel(int kernel, int precision, long long cells = 1ll << 40) {
  (void)precision;
  if (kernel != 0) return kernel;
  return cells >= 500000 ? 4 : 2;
}

static bool make_layout(const hydro_grid* g, int precision, double eta_s, int kernel, Layout* L, bool ext = false) {
  if (!g || g->nx < 1 || g->ny < 1 || g->nz < 1) return false;
  if (precision != 64 && precision != 32) return false;
  if ((long long)g->nx * g->ny * g->nz > (1ll << 36)) return false;
  // launch-grid limits of kernels 1/2 (gridDim.y, gridDim.z) and of the TMA coordinates of kernel 3
  if (g->nz > 65535 || g->ny > 8 * 65535 || g->nx > (1 << 30)) return false;
  L->elem = precision == 64 ? 8 : 4;
  L->nf = eta_s > 0.0 ? (ext ? 16 : 14) : 4;      // ext: the 16-word cell
  L->soa = resolve_kernel(kernel, precision) == 3 ? 1 : 0;
  if (L->soa) {
    const int per16 = 16 / (int)L->elem;
    L->py = ((long long)g->nx + 2 * HALO + per16 - 1) / per16 * per16;
    L->pz = L->py * (g->ny + 2 * HALO);
    L->pf = L->pz * (g->nz + 2 * HALO);
    L->nft = L->nf; L->nxb = 0; L->blk = 0; L->gp = 0; L->sy = 0; L->sz = 0;
    L->nelem = L->pf * L->nf;
    size_t off = 0;
    L->off_diag = off; off += 256;
    L->off_eos = off; off += align_up((size_t)5 * kMaxEosNodes * L->elem, 256);
    for (int b = 0; b < 3; ++b) { L->off_buf[b] = off; off += align_up((size_t)L->nelem * L->elem, 256); }
    L->off_gstar = off; off += align_up((size_t)L->pf * L->elem, 256);
    L->total = off;
    return true;
  }
  L->nft = L->nf + X_COUNT;     // + extended slots P, u^tau, c_x, c_y, c_eta
  L->nxb = (g->nx + 31) / 32;
  L->blk = 32 * L->nft;
  L->gp = 32 * L->nxb;
  L->sy = (long long)L->nxb * L->blk;
  L->sz = (long long)g->ny * L->sy;
  L->nelem = (long long)g->nz * L->sz;
  size_t off = 0;
  L->off_diag = off; off += 256;
  L->off_eos = off; off += align_up((size_t)5 * kMaxEosNodes * L->elem, 256);
  for (int b = 0; b < 3; ++b) { L->off_buf[b] = off; off += align_up((size_t)L->nelem * L->elem, 256); }
  L->off_gstar = off; off += align_up((size_t)g->nz * g->ny * L->gp * L->elem, 256);
  L->total = off;
  return true;
}

// ---------------------------------------------------------------------------------------------
// load / read kernels (user layout: unpadded [comp][nz][ny][nx])
// ---------------------------------------------------------------------------------------------
template <typename R>
struct IoArgs {
  int nx, ny, nz, blk;
  long long sy, sz, N;
  R e_floor, v_max;
  EosDev<R> eos;
  DiagDev* diag;
};

template <typename R, bool VISC, bool EXT = false>
__global__ void __launch_bounds__(256) load_kernel(IoArgs<R> a, const R* __restrict__ T, const R* __restrict__ pi,
                                                   R* __restrict__ st, const R* __restrict__ Pib = nullptr,
                                                   const R* __restrict__ nb = nullptr) {
  const long long cu = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const bool active = cu < a.N;
  const long long cc = active ? cu : 0;
  const int i = (int)(cc % a.nx), j = (int)((cc / a.nx) % a.ny), k = (int)(cc / ((long long)a.nx * a.ny));
  const long long c = (long long)k * a.sz + (long long)j * a.sy + xoff(i, a.blk);
  R p[10];
#pragma unroll
  for (int m = 0; m < 10; ++m) p[m] = (VISC && pi) ? pi[m * a.N + cc] : R(0);
  R M[4];
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) M[mu] = T[mu * a.N + cc] - p[mu];    // T_id = T - pi  (Eq.51)
  unsigned flags = 0;
  R e, ux, uy, un, P, cs2, g;
  // warp-uniform Newton with early exit (round 1 ran 64 fixed iterations here: 6.7 ms at 301x301x201)
  // T is the full tensor, the root-find carries the bulk pressure (A28, A32)
  const R Pb = (EXT && Pib) ? Pib[cc] : R(0);
  rootfind_warp(a.eos, M[0], M[1], M[2], M[3], R(-1), 64, a.e_floor, a.v_max, e, P, cs2, ux, uy, un, g, flags, Pb, EXT);
  if (active) {
    st[c] = e; st[FS + c] = ux; st[2 * FS + c] = uy; st[3 * FS + c] = un;
    if (VISC) {
#pragma unroll
      for (int m = 0; m < 10; ++m) st[(F_PI + m) * FS + c] = p[m];
    }
    if (EXT) { st[(F_PI + 10) * FS + c] = Pb; st[(F_PI + 11) * FS + c] = nb ? nb[cc] : R(0); }
    // extended slots read by kernel 2
    R cx, cy, cn;
    signal_speeds3(g, ux, uy, un, cs2, cx, cy, cn);
    R* __restrict__ sx = st + (VISC ? (EXT ? 16 : 14) : 4) * FS + c;
    sx[X_P * FS] = P; sx[X_G * FS] = g;
    sx[X_CX * FS] = cx; sx[X_CY * FS] = cy; sx[X_CN * FS] = cn;
  } else {
    flags = 0;
  }
  count_flags(a.diag, flags);
  const double r = warp_max(active ? (double)e : 0.0);
  if ((threadIdx.x & 31) == 0) atomic_max_nonneg(&a.diag->emax[1], r);
}

template <typename R, bool VISC>
__global__ void __launch_bounds__(256) read_kernel(IoArgs<R> a, const R* __restrict__ st, R* __restrict__ e,
                                                   R* __restrict__ u, R* __restrict__ pi) {
  const long long cu = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (cu >= a.N) return;
  const int i = (int)(cu % a.nx), j = (int)((cu / a.nx) % a.ny), k = (int)(cu / ((long long)a.nx * a.ny));
  const long long c = (long long)k * a.sz + (long long)j * a.sy + xoff(i, a.blk);
  if (e) e[cu] = st[c];
  if (u) {
    const R ux = st[FS + c], uy = st[2 * FS + c], un = st[3 * FS + c];
    u[cu] = sqrt_(R(1) + ux * ux + uy * uy + un * un);
    u[a.N + cu] = ux; u[2 * a.N + cu] = uy; u[3 * a.N + cu] = un;
  }
  if (pi) {
#pragma unroll
    for (int m = 0; m < 10; ++m) pi[m * a.N + cu] = VISC ? st[(F_PI + m) * FS + c] : R(0);
  }
}

// pad (dir = 0: user -> internal) or unpad (dir = 1) three history fields
// bulk pressure and net-baryon density of the state (fields 14, 15 of the 16-word cell)
template <typename R>
__global__ void __launch_bounds__(256) read_ext_kernel(IoArgs<R> a, const R* __restrict__ st, R* __restrict__ Pib,
                                                       R* __restrict__ nb) {
  const long long cu = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (cu >= a.N) return;
  const int i = (int)(cu % a.nx), j = (int)((cu / a.nx) % a.ny), k = (int)(cu / ((long long)a.nx * a.ny));
  const long long c = (long long)k * a.sz + (long long)j * a.sy + xoff(i, a.blk);
  if (Pib) Pib[cu] = st[(F_PI + 10) * FS + c];
  if (nb) nb[cu] = st[(F_PI + 11) * FS + c];
}

template <typename R>
__global__ void __launch_bounds__(256) history_kernel(IoArgs<R> a, R* __restrict__ hist, R* __restrict__ user,
                                                      int dir) {
  const long long cu = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (cu >= a.N) return;
  const int i = (int)(cu % a.nx), j = (int)((cu / a.nx) % a.ny), k = (int)(cu / ((long long)a.nx * a.ny));
  const long long c = (long long)k * a.sz + (long long)j * a.sy + xoff(i, a.blk);
#pragma unroll
  for (int m = 0; m < 3; ++m) {
    if (dir == 0) hist[m * FS + c] = user[m * a.N + cu];
    else user[m * a.N + cu] = hist[m * FS + c];
  }
}

// ---- the same three kernels for the ghosted SoA layout of kernel 3 ---------------------------------------------------
template <typename R>
struct SoaArgs {
  int nx, ny, nz;
  long long py, pz, pf, N;
  int bc[3];
  R e_floor, v_max;
  EosDev<R> eos;
  DiagDev* diag;
};

// store v at (field f, cell i,j,k) and at the ghost positions that mirror the cell (boundary rule a11)
template <typename R>
__device__ __forceinline__ void soa_put(const SoaArgs<R>& a, R* __restrict__ st, int f, int i, int j, int k, R v,
                                        const int* gl, const int* ng) {
  R* __restrict__ o = st + (long long)f * a.pf + (long long)(k + HALO) * a.pz + (long long)(j + HALO) * a.py + (i + HALO);
  o[0] = v;
  for (int t = 0; t < ng[0]; ++t) o[gl[t] - i] = v;
  for (int t = 0; t < ng[1]; ++t) o[(long long)(gl[4 + t] - j) * a.py] = v;
  for (int t = 0; t < ng[2]; ++t) o[(long long)(gl[8 + t] - k) * a.pz] = v;
}

template <typename R, bool VISC>
__global__ void __launch_bounds__(256) load_kernel_soa(SoaArgs<R> a, const R* __restrict__ T, const R* __restrict__ pi,
                                                       R* __restrict__ st) {
  const long long cu = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const bool active = cu < a.N;
  const long long cc = active ? cu : 0;
  const int i = (int)(cc % a.nx), j = (int)((cc / a.nx) % a.ny), k = (int)(cc / ((long long)a.nx * a.ny));
  R p[10];
#pragma unroll
  for (int m = 0; m < 10; ++m) p[m] = (VISC && pi) ? pi[m * a.N + cc] : R(0);
  R M[4];
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) M[mu] = T[mu * a.N + cc] - p[mu];    // T_id = T - pi  (Eq.51)
  unsigned flags = 0;
  R e, P, cs2, ux, uy, un, g;
  rootfind_warp(a.eos, M[0], M[1], M[2], M[3], R(-1), 64, a.e_floor, a.v_max, e, P, cs2, ux, uy, un, g, flags);
  if (active) {
    int gl[12], ng[3];
    ng[0] = ghost_list(i, a.nx, a.bc[0], gl);
    ng[1] = ghost_list(j, a.ny, a.bc[1], gl + 4);
    ng[2] = ghost_list(k, a.nz, a.bc[2], gl + 8);
    soa_put(a, st, 0, i, j, k, e, gl, ng); soa_put(a, st, 1, i, j, k, ux, gl, ng);
    soa_put(a, st, 2, i, j, k, uy, gl, ng); soa_put(a, st, 3, i, j, k, un, gl, ng);
    if (VISC) {
#pragma unroll
      for (int m = 0; m < 10; ++m) soa_put(a, st, 4 + m, i, j, k, p[m], gl, ng);
    }
  } else {
    flags = 0;
  }
  count_flags(a.diag, flags);
  const double r = warp_max(active ? (double)e : 0.0);
  if ((threadIdx.x & 31) == 0) atomic_max_nonneg(&a.diag->emax[1], r);
}

template <typename R, bool VISC>
__global__ void __launch_bounds__(256) read_kernel_soa(SoaArgs<R> a, const R* __restrict__ st, R* __restrict__ e,
                                                       R* __restrict__ u, R* __restrict__ pi) {
  const long long cu = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (cu >= a.N) return;
  const int i = (int)(cu % a.nx), j = (int)((cu / a.nx) % a.ny), k = (int)(cu / ((long long)a.nx * a.ny));
  const R* __restrict__ c = st + (long long)(k + HALO) * a.pz + (long long)(j + HALO) * a.py + (i + HALO);
  if (e) e[cu] = c[0];
  if (u) {
    const R ux = c[a.pf], uy = c[2 * a.pf], un = c[3 * a.pf];
    u[cu] = sqrt_(R(1) + ux * ux + uy * uy + un * un);
    u[a.N + cu] = ux; u[2 * a.N + cu] = uy; u[3 * a.N + cu] = un;
  }
  if (pi) {
#pragma unroll
    for (int m = 0; m < 10; ++m) pi[m * a.N + cu] = VISC ? c[(4 + m) * a.pf] : R(0);
  }
}

// pad (dir = 0: user -> internal) or unpad (dir = 1) three history fields (no ghosts: the history is read at the
// cell centre only)
template <typename R>
__global__ void __launch_bounds__(256) history_kernel_soa(SoaArgs<R> a, R* __restrict__ hist, R* __restrict__ user,
                                                          int dir) {
  const long long cu = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (cu >= a.N) return;
  const int i = (int)(cu % a.nx), j = (int)((cu / a.nx) % a.ny), k = (int)(cu / ((long long)a.nx * a.ny));
  R* __restrict__ c = hist + (long long)(k + HALO) * a.pz + (long long)(j + HALO) * a.py + (i + HALO);
#pragma unroll
  for (int m = 0; m < 3; ++m) {
    if (dir == 0) c[m * a.pf] = user[m * a.N + cu];
    else user[m * a.N + cu] = c[m * a.pf];
  }
}

}  // namespace clv

using namespace clv;

struct hydro_ctx {
  hydro_grid grid;
  double dtau, tau0, eta_s;
  int precision, visc, kernel, strict, ext;
  int half;          // 1 between hydro_stage(1) and hydro_stage(2)
  double zeta_s;
  double theta, e_floor, xi, v_max, lambda1_hat, c_tau;
  int root_iters;
  Layout L;
  char* ws;
  void* buf[3];
  int cur, prev;     // indices of state n / state n-1 in buf[0..1]; buf[2] is state '
  void* gstar;
  DiagDev* diag;
  EosDev<double> eos64;
  EosDev<float> eos32;
  cudaStream_t stream;
  long long step;
  long long launches;
  bool loaded;
  // kernel 3: TMA tensor maps of the three state buffers with box depth nf ([b][0]) and 4 ([b][1]); tiling
  CUtensorMap tmap[3][2];
  int ntx, nty, nchunk, chunk;
  int march_chunk;   // kernel 4: eta_s planes per block
  // freeze-out surface finder: caller-owned workspace [counters 256 B][level 0][level 1], each level
  // = e, u~^mu[4], pi~[10] in the user layout; level[frz_a] is the stored level a
  char* frz_ws;
  void* frz_level[2];
  int frz_a;
  double frz_e, frz_tau_a;
  long long frz_slab;
};

namespace {

template <typename R> const EosDev<R>& eos_of(const hydro_ctx* c);
template <> const EosDev<double>& eos_of<double>(const hydro_ctx* c) { return c->eos64; }
template <> const EosDev<float>& eos_of<float>(const hydro_ctx* c) { return c->eos32; }

// ---- kernel 3 host side: tensor maps, tiling, argument block ----------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// 4-D map (x, y, z, field) of one ghosted SoA buffer with box {36, 12, 1, nbox}
int make_tmap(const hydro_ctx* c, void* base, int nbox, CUtensorMap* out) {
  static EncodeTiledFn encode = nullptr;
  if (!encode) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess || !fn) {
      (void)cudaGetLastError();
      return HYDRO_ECUDA;
    }
    encode = reinterpret_cast<EncodeTiledFn>(fn);
  }
  const Layout& L = c->L;
  const cuuint64_t dims[4] = {(cuuint64_t)(c->grid.nx + 2 * HALO), (cuuint64_t)(c->grid.ny + 2 * HALO),
                              (cuuint64_t)(c->grid.nz + 2 * HALO), (cuuint64_t)nbox};
  const cuuint64_t strides[3] = {(cuuint64_t)L.py * L.elem, (cuuint64_t)L.pz * L.elem, (cuuint64_t)L.pf * L.elem};
  const cuuint32_t box[4] = {(cuuint32_t)SX, (cuuint32_t)SY, 1u, (cuuint32_t)nbox};
  const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
  const CUresult r = encode(out, L.elem == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, base,
                            dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                            CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? HYDRO_OK : HYDRO_ECUDA;
}

// z-chunks per tile column: fill the SMs in whole waves while keeping the 4-plane pipeline warm-up per chunk small
void choose_tiling(hydro_ctx* c, int nsm) {
  c->ntx = (c->grid.nx + TX - 1) / TX;
  c->nty = (c->grid.ny + TY - 1) / TY;
  const long long tiles = (long long)c->ntx * c->nty;
  const int nz = c->grid.nz;
  double best = -1.0;
  for (int cand = 1; cand <= nz && cand <= 256; ++cand) {
    const int chunk = (nz + cand - 1) / cand, nchunk = (nz + chunk - 1) / chunk;
    const long long blocks = tiles * nchunk;
    const long long waves = (blocks + nsm - 1) / nsm;
    const double eff = (double)blocks / (double)(waves * nsm) * (double)chunk / ((double)chunk + 1.5);
    if (eff > best * 1.0001) { best = eff; c->chunk = chunk; c->nchunk = nchunk; }
  }
}

template <typename R>
TileArgs<R> tile_args(const hydro_ctx* c, double tau_rhs, double tau_n, double tau_1) {
  TileArgs<R> a;
  memset(&a, 0, sizeof(a));
  const bool milne = c->grid.geometry == 0;
  a.nx = c->grid.nx; a.ny = c->grid.ny; a.nz = c->grid.nz;
  a.py = c->L.py; a.pz = c->L.pz; a.pf = c->L.pf;
  for (int d = 0; d < 3; ++d) a.bc[d] = c->grid.bc[d];
  a.milne = milne ? 1 : 0;
  a.tau = (R)tau_rhs; a.inv_tau = (R)(1.0 / tau_rhs);
  a.tf_n = (R)(milne ? tau_n : 1.0); a.tf_1 = (R)(milne ? tau_1 : 1.0); a.inv_tf_1 = (R)(milne ? 1.0 / tau_1 : 1.0);
  a.h = (R)c->dtau; a.inv_h = (R)(1.0 / c->dtau);
  a.scale[0] = (R)(1.0 / c->grid.dx); a.scale[1] = (R)(1.0 / c->grid.dy);
  a.scale[2] = (R)(milne ? 1.0 / (tau_rhs * c->grid.deta) : 1.0 / c->grid.deta);
  a.theta = (R)c->theta; a.e_floor = (R)c->e_floor; a.xi = (R)c->xi; a.v_max = (R)c->v_max;
  a.inv_5etas_hbarc = (R)(c->visc ? 1.0 / (c->c_tau * c->eta_s * kHbarc) : 0.0);
  a.inv_ctau = (R)(1.0 / c->c_tau); a.lam1 = (R)c->lambda1_hat;
  a.root_iters = c->root_iters;
  a.eos = eos_of<R>(c);
  a.diag = c->diag;
  a.ntx = c->ntx; a.nty = c->nty; a.nchunk = c->nchunk; a.chunk = c->chunk;
  return a;
}

template <typename R, bool VISC, int MODE>
int launch_tile(hydro_ctx* c, const TileArgs<R>& a, int buf_in) {
  constexpr bool USE_PI = VISC && (MODE != 0);
  const CUtensorMap& map = c->tmap[buf_in][(USE_PI || !c->visc) ? 0 : 1];
  const cudaError_t e = launch_stage_tile<R, VISC, MODE>(a, map, c->stream);
  c->launches += 1;
  return e == cudaSuccess ? HYDRO_OK : HYDRO_ECUDA;
}

template <typename R>
SoaArgs<R> soa_args(const hydro_ctx* c) {
  SoaArgs<R> a;
  a.nx = c->grid.nx; a.ny = c->grid.ny; a.nz = c->grid.nz;
  a.py = c->L.py; a.pz = c->L.pz; a.pf = c->L.pf; a.N = (long long)a.nx * a.ny * a.nz;
  for (int d = 0; d < 3; ++d) a.bc[d] = c->grid.bc[d];
  a.e_floor = (R)c->e_floor; a.v_max = (R)c->v_max;
  a.eos = eos_of<R>(c);
  a.diag = c->diag;
  return a;
}

template <typename R>
int upload_eos(hydro_ctx* c, const hydro_eos* eos, EosDev<R>* q) {
  memset(q, 0, sizeof(*q));
  q->kind = eos->kind;
  q->hbarc = (R)kHbarc;
  q->conf_T_scale = (R)(1.0 / (eos->c_sb * kHbarc));
  if (eos->kind == 0) return HYDRO_OK;
  const int n = eos->n;
  std::vector<double> node(n), cs2(n, 0.0), dT(n, 0.0);
  for (int k = 0; k < n; ++k) node[k] = eos->e_min * std::pow(eos->e_max / eos->e_min, double(k) / double(n - 1));
  for (int k = 0; k + 1 < n; ++k) {
    cs2[k] = (eos->P[k + 1] - eos->P[k]) / (node[k + 1] - node[k]);
    dT[k] = (eos->T[k + 1] - eos->T[k]) / (node[k + 1] - node[k]);
  }
  std::vector<R> h((size_t)5 * n);
  for (int k = 0; k < n; ++k) {
    h[k] = (R)node[k]; h[n + k] = (R)eos->P[k]; h[2 * n + k] = (R)cs2[k]; h[3 * n + k] = (R)eos->T[k];
    h[4 * n + k] = (R)dT[k];
  }
  R* d = reinterpret_cast<R*>(c->ws + c->L.off_eos);
  if (cudaMemcpyAsync(d, h.data(), h.size() * sizeof(R), cudaMemcpyHostToDevice, c->stream) != cudaSuccess)
    return HYDRO_ECUDA;
  if (cudaStreamSynchronize(c->stream) != cudaSuccess) return HYDRO_ECUDA;
  q->n = n;
  q->e_min = (R)node[0]; q->e_max = (R)node[n - 1];
  q->inv_e_min = (R)(1.0 / node[0]); q->inv_e_max = (R)(1.0 / node[n - 1]);
  q->P0_slope = (R)(eos->P[0] / eos->e_min);
  q->P_top = (R)eos->P[n - 1]; q->T_bot = (R)eos->T[0]; q->T_top = (R)eos->T[n - 1];
  q->log2_emin = (float)std::log2(eos->e_min);
  q->inv_dlog2 = (float)(double(n - 1) / std::log2(eos->e_max / eos->e_min));
  q->node = d; q->P = d + n; q->cs2 = d + 2 * n; q->T = d + 3 * n; q->dTde = d + 4 * n;
  return HYDRO_OK;
}

template <typename R>
IoArgs<R> io_args(const hydro_ctx* c) {
  IoArgs<R> a;
  a.nx = c->grid.nx; a.ny = c->grid.ny; a.nz = c->grid.nz; a.blk = c->L.blk;
  a.sy = c->L.sy; a.sz = c->L.sz; a.N = (long long)a.nx * a.ny * a.nz;
  a.e_floor = (R)c->e_floor; a.v_max = (R)c->v_max;
  a.eos = eos_of<R>(c);
  a.diag = c->diag;
  return a;
}

template <typename R>
StageArgs<R> stage_args(const hydro_ctx* c, double tau_rhs, double tau_n, double tau_1) {
  StageArgs<R> a;
  memset(&a, 0, sizeof(a));
  const bool milne = c->grid.geometry == 0;
  a.nx = c->grid.nx; a.ny = c->grid.ny; a.nz = c->grid.nz;
  a.blk = c->L.blk; a.gp = c->L.gp; a.sy = c->L.sy; a.sz = c->L.sz;
  for (int d = 0; d < 3; ++d) a.bc[d] = c->grid.bc[d];
  a.milne = milne ? 1 : 0;
  a.tau = (R)tau_rhs; a.inv_tau = (R)(1.0 / tau_rhs);
  a.tf_n = (R)(milne ? tau_n : 1.0); a.tf_1 = (R)(milne ? tau_1 : 1.0); a.inv_tf_1 = (R)(milne ? 1.0 / tau_1 : 1.0);
  a.h = (R)c->dtau; a.inv_h = (R)(1.0 / c->dtau);
  a.scale[0] = (R)(1.0 / c->grid.dx); a.scale[1] = (R)(1.0 / c->grid.dy);
  a.scale[2] = (R)(milne ? 1.0 / (tau_rhs * c->grid.deta) : 1.0 / c->grid.deta);
  a.theta = (R)c->theta; a.e_floor = (R)c->e_floor; a.xi = (R)c->xi; a.v_max = (R)c->v_max;
  a.inv_5etas_hbarc = (R)(c->visc ? 1.0 / (c->c_tau * c->eta_s * kHbarc) : 0.0);
  a.inv_ctau = (R)(1.0 / c->c_tau); a.lam1 = (R)c->lambda1_hat;
  a.zeta_over_eta = (R)((c->ext && c->visc) ? c->zeta_s / c->eta_s : 0.0);
  a.root_iters = c->root_iters;
  a.eos = eos_of<R>(c);
  a.diag = c->diag;
  return a;
}

template <typename R, bool VISC, int MODE>
int launch_stage(hydro_ctx* c, const StageArgs<R>& a) {
  if constexpr (VISC) {
    if (c->ext) {      // the 16-word cell, kernels 4 (marching) and 2 (per-cell; also the bootstrap)
      c->launches += 1;
      if constexpr (MODE != 0) {
        if (c->kernel == 4)
          return launch_stage_march<R, true, MODE, true>(a, c->march_chunk, c->stream) == cudaSuccess ? HYDRO_OK : HYDRO_ECUDA;
      }
      launch_stage_fused<R, true, MODE, true>(a, c->stream);
      return cudaGetLastError() == cudaSuccess ? HYDRO_OK : HYDRO_ECUDA;
    }
  }
  if (c->kernel == 4 && MODE != 0) {
    if constexpr (MODE != 0) {
      c->launches += 1;
      return launch_stage_march<R, VISC, MODE>(a, c->march_chunk, c->stream) == cudaSuccess ? HYDRO_OK : HYDRO_ECUDA;
    }
  } else if (c->kernel == 2 || c->kernel == 4) {      // the bootstrap of kernel 4 runs in the per-cell kernel (same store)
    launch_stage_fused<R, VISC, MODE>(a, c->stream);
  } else {
    dim3 block(32, 8, 1);
    dim3 grid((a.nx + 31) / 32, (a.ny + 7) / 8, a.nz);
    stage_ref_kernel<R, VISC, MODE><<<grid, block, 0, c->stream>>>(a);
  }
  c->launches += 1;
  return cudaGetLastError() == cudaSuccess ? HYDRO_OK : HYDRO_ECUDA;
}

template <typename R>
int do_bootstrap(hydro_ctx* c) {
  if (c->L.soa) {
    TileArgs<R> t = tile_args<R>(c, c->tau0, c->tau0, c->tau0 + c->dtau);
    t.out = static_cast<R*>(c->buf[c->prev]) + c->L.pf;      // u~^i slots (fields 1..3) of the history buffer
    t.slot = 0;
    return c->visc ? launch_tile<R, true, 0>(c, t, c->cur) : launch_tile<R, false, 0>(c, t, c->cur);
  }
  StageArgs<R> a = stage_args<R>(c, c->tau0, c->tau0, c->tau0 + c->dtau);
  a.in = static_cast<const R*>(c->buf[c->cur]);
  a.out = static_cast<R*>(c->buf[c->prev]) + FS;         // u~^i slots (fields 1..3) of the history buffer
  a.slot = 0;
  return c->visc ? launch_stage<R, true, 0>(c, a) : launch_stage<R, false, 0>(c, a);
}

// which: 0 = the whole RK2 step; 1 / 2 = one stage only (hydro_stage: blocked store, not with strict_eq53)
template <typename R>
int do_step(hydro_ctx* c, int which = 0) {
  const double tau_n = c->tau0 + (double)c->step * c->dtau, tau_1 = tau_n + c->dtau;
  const int slot = (int)(c->step & 1);
  R* cur = static_cast<R*>(c->buf[c->cur]);
  R* prev = static_cast<R*>(c->buf[c->prev]);
  R* X = static_cast<R*>(c->buf[2]);
  if (c->L.soa) {
    TileArgs<R> t1 = tile_args<R>(c, tau_n, tau_n, tau_1);
    t1.uprev = prev + c->L.pf; t1.gstar = static_cast<R*>(c->gstar); t1.out = X; t1.slot = slot;
    TileArgs<R> t2 = tile_args<R>(c, tau_1, tau_n, tau_1);
    t2.sn = cur; t2.gstar = static_cast<R*>(c->gstar); t2.out = prev; t2.slot = slot;
    int rc;
    if (c->visc) {
      rc = launch_tile<R, true, 1>(c, t1, c->cur);
      if (rc) return rc;
      rc = launch_tile<R, true, 2>(c, t2, 2);
    } else {
      rc = launch_tile<R, false, 1>(c, t1, c->cur);
      if (rc) return rc;
      rc = launch_tile<R, false, 2>(c, t2, 2);
    }
    if (rc) return rc;
    const int t = c->cur; c->cur = c->prev; c->prev = t;
    c->step += 1;
    return HYDRO_OK;
  }
  StageArgs<R> a1 = stage_args<R>(c, tau_n, tau_n, tau_1);
  a1.in = cur; a1.uprev = prev + FS; a1.gstar = static_cast<R*>(c->gstar); a1.out = X; a1.slot = slot;
  StageArgs<R> a2 = stage_args<R>(c, tau_1, tau_n, tau_1);
  a2.in = X; a2.sn = cur; a2.gstar = static_cast<R*>(c->gstar); a2.out = prev; a2.slot = slot;
  int rc;
  if (c->visc && c->strict) {
    // Eq.53 as printed (A12; hydro_stage_strict.cuh): sweep A = stage 2 without limiter into a scratch diag block,
    // sweep B = T fields on (e', u', pi^{n+1}), sweep C = limiter
    rc = launch_stage<R, true, 1>(c, a1);
    if (rc) return rc;
    StageArgs<R> a2a = a2;
    a2a.xi = R(0); a2a.diag = c->diag + 1;
    rc = launch_stage<R, true, 2>(c, a2a);
    if (rc) return rc;
    dim3 block(32, 8, 1);
    dim3 grid((a2.nx + 31) / 32, (a2.ny + 7) / 8, a2.nz);
    stage_strict_T_kernel<R><<<grid, block, 0, c->stream>>>(a2, prev);
    stage_strict_limit_kernel<R><<<grid, block, 0, c->stream>>>(a2);
    c->launches += 2;
    rc = cudaGetLastError() == cudaSuccess ? HYDRO_OK : HYDRO_ECUDA;
  } else if (c->visc) {
    rc = which == 2 ? HYDRO_OK : launch_stage<R, true, 1>(c, a1);
    if (rc) return rc;
    if (which != 1) rc = launch_stage<R, true, 2>(c, a2);
  } else {
    rc = which == 2 ? HYDRO_OK : launch_stage<R, false, 1>(c, a1);
    if (rc) return rc;
    if (which != 1) rc = launch_stage<R, false, 2>(c, a2);
  }
  if (rc) return rc;
  if (which == 1) { c->half = 1; return HYDRO_OK; }
  c->half = 0;
  const int t = c->cur; c->cur = c->prev; c->prev = t;
  c->step += 1;
  return HYDRO_OK;
}

template <typename R>
int do_load(hydro_ctx* c, const void* T, const void* pi, int mem, const void* Pib = nullptr, const void* nb = nullptr) {
  const long long N = (long long)c->grid.nx * c->grid.ny * c->grid.nz;
  const R* dT = static_cast<const R*>(T);
  const R* dpi = static_cast<const R*>(pi);
  const R* dPib = static_cast<const R*>(Pib);
  const R* dnb = static_cast<const R*>(nb);
  if (!c->visc) dpi = nullptr;
  if (!(c->ext && c->visc)) { dPib = nullptr; dnb = nullptr; }
  if (mem == HYDRO_MEM_HOST) {
    R* stage = static_cast<R*>(c->buf[2]);
    if (dPib) {
      if (cudaMemcpyAsync(stage + 14 * N, Pib, (size_t)N * sizeof(R), cudaMemcpyHostToDevice, c->stream) != cudaSuccess)
        return HYDRO_ECUDA;
      dPib = stage + 14 * N;
    }
    if (dnb) {
      if (cudaMemcpyAsync(stage + 15 * N, nb, (size_t)N * sizeof(R), cudaMemcpyHostToDevice, c->stream) != cudaSuccess)
        return HYDRO_ECUDA;
      dnb = stage + 15 * N;
    }
    if (cudaMemcpyAsync(stage, T, (size_t)4 * N * sizeof(R), cudaMemcpyHostToDevice, c->stream) != cudaSuccess)
      return HYDRO_ECUDA;
    dT = stage;
    if (dpi) {
      if (cudaMemcpyAsync(stage + 4 * N, pi, (size_t)10 * N * sizeof(R), cudaMemcpyHostToDevice, c->stream) !=
          cudaSuccess)
        return HYDRO_ECUDA;
      dpi = stage + 4 * N;
    }
  }
  if (cudaMemsetAsync(c->diag, 0, sizeof(DiagDev), c->stream) != cudaSuccess) return HYDRO_ECUDA;
  c->cur = 0; c->prev = 1; c->step = 0; c->half = 0;
  const unsigned nblk = (unsigned)((N + 255) / 256);
  if (c->L.soa) {
    SoaArgs<R> a = soa_args<R>(c);
    if (c->visc) load_kernel_soa<R, true><<<nblk, 256, 0, c->stream>>>(a, dT, dpi, static_cast<R*>(c->buf[c->cur]));
    else load_kernel_soa<R, false><<<nblk, 256, 0, c->stream>>>(a, dT, dpi, static_cast<R*>(c->buf[c->cur]));
  } else {
    IoArgs<R> a = io_args<R>(c);
    if (c->visc && c->ext)
      load_kernel<R, true, true><<<nblk, 256, 0, c->stream>>>(a, dT, dpi, static_cast<R*>(c->buf[c->cur]), dPib, dnb);
    else if (c->visc) load_kernel<R, true><<<nblk, 256, 0, c->stream>>>(a, dT, dpi, static_cast<R*>(c->buf[c->cur]));
    else load_kernel<R, false><<<nblk, 256, 0, c->stream>>>(a, dT, dpi, static_cast<R*>(c->buf[c->cur]));
  }
  c->launches += 1;
  if (cudaGetLastError() != cudaSuccess) return HYDRO_ECUDA;
  int rc = do_bootstrap<R>(c);
  if (rc) return rc;
  if (mem == HYDRO_MEM_HOST && cudaStreamSynchronize(c->stream) != cudaSuccess) return HYDRO_ECUDA;
  c->loaded = true;
  return HYDRO_OK;
}

template <typename R>
int do_read(hydro_ctx* c, void* e, void* u, void* pi, int mem) {
  const long long N = (long long)c->grid.nx * c->grid.ny * c->grid.nz;
  IoArgs<R> a = io_args<R>(c);
  const unsigned nb = (unsigned)((N + 255) / 256);
  const R* st = static_cast<const R*>(c->buf[c->cur]);
  auto run = [&](R* pe, R* pu, R* pp) -> int {
    if (c->L.soa) {
      SoaArgs<R> sa = soa_args<R>(c);
      if (c->visc) read_kernel_soa<R, true><<<nb, 256, 0, c->stream>>>(sa, st, pe, pu, pp);
      else read_kernel_soa<R, false><<<nb, 256, 0, c->stream>>>(sa, st, pe, pu, pp);
    } else if (c->visc) read_kernel<R, true><<<nb, 256, 0, c->stream>>>(a, st, pe, pu, pp);
    else read_kernel<R, false><<<nb, 256, 0, c->stream>>>(a, st, pe, pu, pp);
    c->launches += 1;
    return cudaGetLastError() == cudaSuccess ? HYDRO_OK : HYDRO_ECUDA;
  };
  if (mem == HYDRO_MEM_DEVICE) return run(static_cast<R*>(e), static_cast<R*>(u), static_cast<R*>(pi));
  // host: stage each requested piece through buf X (+gstar when viscous), one D2H copy per piece
  R* stage = static_cast<R*>(c->buf[2]);
  int rc = HYDRO_OK;
  if (e) {
    if ((rc = run(stage, nullptr, nullptr))) return rc;
    if (cudaMemcpyAsync(e, stage, (size_t)N * sizeof(R), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess)
      return HYDRO_ECUDA;
  }
  if (u) {
    R* s = c->visc ? stage + N : stage;
    if ((rc = run(nullptr, s, nullptr))) return rc;
    if (cudaMemcpyAsync(u, s, (size_t)4 * N * sizeof(R), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess)
      return HYDRO_ECUDA;
  }
  if (pi) {
    if (c->visc) {
      // the e and u pieces occupy 5N elements of the 14 sf available; pi (10N) does not fit behind them in
      // general, so wait for their copies to be issued in stream order and reuse the area from the start.
      if ((rc = run(nullptr, nullptr, stage))) return rc;
      if (cudaMemcpyAsync(pi, stage, (size_t)10 * N * sizeof(R), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess)
        return HYDRO_ECUDA;
    } else {
      if (cudaStreamSynchronize(c->stream) != cudaSuccess) return HYDRO_ECUDA;
      memset(pi, 0, (size_t)10 * N * sizeof(R));
    }
  }
  return cudaStreamSynchronize(c->stream) == cudaSuccess ? HYDRO_OK : HYDRO_ECUDA;
}

template <typename R>
int do_history(hydro_ctx* c, void* user, int mem, int dir) {
  const long long N = (long long)c->grid.nx * c->grid.ny * c->grid.nz;
  IoArgs<R> a = io_args<R>(c);
  const unsigned nb = (unsigned)((N + 255) / 256);
  R* hist = static_cast<R*>(c->buf[c->prev]) + (c->L.soa ? c->L.pf : (long long)FS);
  R* dev = static_cast<R*>(user);
  R* stage = static_cast<R*>(c->buf[2]);
  if (mem == HYDRO_MEM_HOST) {
    dev = stage;
    if (dir == 0 &&
        cudaMemcpyAsync(stage, user, (size_t)3 * N * sizeof(R), cudaMemcpyHostToDevice, c->stream) != cudaSuccess)
      return HYDRO_ECUDA;
  }
  if (c->L.soa) history_kernel_soa<R><<<nb, 256, 0, c->stream>>>(soa_args<R>(c), hist, dev, dir);
  else history_kernel<R><<<nb, 256, 0, c->stream>>>(a, hist, dev, dir);
  c->launches += 1;
  if (cudaGetLastError() != cudaSuccess) return HYDRO_ECUDA;
  if (mem == HYDRO_MEM_HOST) {
    if (dir == 1 &&
        cudaMemcpyAsync(user, stage, (size_t)3 * N * sizeof(R), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess)
      return HYDRO_ECUDA;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return HYDRO_ECUDA;
  }
  return HYDRO_OK;
}

// Pi and n of the current state to user arrays (device in place; host through buf X)
template <typename R>
int do_read_ext(hydro_ctx* c, void* Pib, void* nb, int mem) {
  const long long N = (long long)c->grid.nx * c->grid.ny * c->grid.nz;
  IoArgs<R> a = io_args<R>(c);
  const unsigned nblk = (unsigned)((N + 255) / 256);
  const R* st = static_cast<const R*>(c->buf[c->cur]);
  R* dP = static_cast<R*>(Pib);
  R* dn = static_cast<R*>(nb);
  R* stage = static_cast<R*>(c->buf[2]);
  if (mem == HYDRO_MEM_HOST) { dP = Pib ? stage : nullptr; dn = nb ? stage + N : nullptr; }
  read_ext_kernel<R><<<nblk, 256, 0, c->stream>>>(a, st, dP, dn);
  c->launches += 1;
  if (cudaGetLastError() != cudaSuccess) return HYDRO_ECUDA;
  if (mem == HYDRO_MEM_HOST) {
    if (Pib && cudaMemcpyAsync(Pib, dP, (size_t)N * sizeof(R), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess)
      return HYDRO_ECUDA;
    if (nb && cudaMemcpyAsync(nb, dn, (size_t)N * sizeof(R), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess)
      return HYDRO_ECUDA;
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return HYDRO_ECUDA;
  }
  return HYDRO_OK;
}

// freeze-out finder: bytes of one stored level; store the current state as level `which`
static size_t frz_level_bytes(const hydro_grid* g, int precision) {
  const size_t N = (size_t)g->nx * g->ny * g->nz;
  return align_up((size_t)15 * N * (precision == 64 ? 8 : 4), 256);
}
template <typename R>
int frz_store_level(hydro_ctx* c, int which) {
  const long long N = (long long)c->grid.nx * c->grid.ny * c->grid.nz;
  R* lv = static_cast<R*>(c->frz_level[which]);
  return do_read<R>(c, lv, lv + N, lv + 5 * N, HYDRO_MEM_DEVICE);
}

}  // namespace

extern "C" {

size_t hydro_workspace_bytes_ext(const hydro_grid* grid, int precision, double eta_over_s, int bulk_baryon) {
  if (!bulk_baryon) return hydro_workspace_bytes(grid, precision, eta_over_s);
  Layout L;
  if (!(eta_over_s > 0.0) || !make_layout(grid, precision, eta_over_s, 2, &L, true)) return 0;
  return L.total;
}

size_t hydro_workspace_bytes(const hydro_grid* grid, int precision, double eta_over_s) {
  // one figure for every kernel choice: the larger of the blocked (kernels 1/2) and the ghosted SoA (kernel 3) stores
  Layout L2, L3;
  if (!make_layout(grid, precision, eta_over_s, 2, &L2) || !make_layout(grid, precision, eta_over_s, 3, &L3)) return 0;
  return L2.total > L3.total ? L2.total : L3.total;
}

int hydro_create(hydro_ctx** out, const hydro_grid* grid, double dtau, double tau0, const hydro_eos* eos,
                 double eta_over_s, const hydro_opts* opts) {
  if (!out) return HYDRO_EINVAL;
  *out = nullptr;
  if (!grid || !eos || !opts) return HYDRO_EINVAL;
  Layout L;
  if (opts->kernel < 0 || opts->kernel > 4) return HYDRO_EINVAL;
  if (opts->strict_eq53 && eta_over_s > 0.0) {      // the strict sweeps exist for the blocked extended store only
    const int kk = resolve_kernel(opts->kernel, opts->precision);
    if (kk != 2 && kk != 4) return HYDRO_EINVAL;
  }
  const bool ext = opts->bulk_baryon != 0;
  if (ext) {      // viscous runs, blocked store (kernel 2), no strict Eq.53
    const int kk = resolve_kernel(opts->kernel, opts->precision);
    if (!(eta_over_s > 0.0) || (kk != 2 && kk != 4) || opts->strict_eq53 || !(opts->zeta_over_s >= 0.0)) return HYDRO_EINVAL;
  }
  if (!make_layout(grid, opts->precision, eta_over_s, ext ? 2 : opts->kernel, &L, ext)) return HYDRO_EINVAL;
  if (!(dtau > 0.0) || !(grid->dx > 0.0) || !(grid->dy > 0.0) || !(grid->deta > 0.0)) return HYDRO_EINVAL;
  if (grid->geometry != 0 && grid->geometry != 1) return HYDRO_EINVAL;
  if (grid->geometry == 0 && !(tau0 > 0.0)) return HYDRO_EINVAL;
  for (int d = 0; d < 3; ++d)
    if (grid->bc[d] != 0 && grid->bc[d] != 1) return HYDRO_EINVAL;
  if (!(eta_over_s >= 0.0)) return HYDRO_EINVAL;
  if (!(opts->minmod_theta >= 1.0 && opts->minmod_theta <= 2.0)) return HYDRO_EINVAL;
  if (!(opts->e_floor > 0.0)) return HYDRO_EINVAL;
  if (eos->kind != 0 && eos->kind != 1) return HYDRO_EINVAL;
  if (!(eos->c_sb > 0.0)) return HYDRO_EINVAL;
  if (eos->kind == 1) {
    if (eos->n < 2 || eos->n > kMaxEosNodes || !eos->P || !eos->T) return HYDRO_EINVAL;
    if (!(eos->e_min > 0.0) || !(eos->e_max > eos->e_min)) return HYDRO_EINVAL;
    for (int k = 0; k + 1 < eos->n; ++k)
      if (!(eos->P[k + 1] >= eos->P[k])) return HYDRO_EINVAL;   // monotone P keeps the root unique (A7)
  }
  if (!opts->workspace || opts->workspace_bytes < L.total || (reinterpret_cast<size_t>(opts->workspace) & 255))
    return HYDRO_ENOMEM;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { (void)cudaGetLastError(); return HYDRO_ECUDA; }
  {   // the workspace must be device memory of the CURRENT device (a host or wrong-GPU pointer would fault inside a kernel)
    cudaPointerAttributes pa;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaPointerGetAttributes(&pa, opts->workspace) != cudaSuccess) {
      (void)cudaGetLastError();
      return HYDRO_ECUDA;
    }
    if ((pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged) || (pa.type == cudaMemoryTypeDevice && pa.device != dev))
      return HYDRO_EINVAL;
  }

  hydro_ctx* c = new (std::nothrow) hydro_ctx();
  if (!c) return HYDRO_ENOMEM;
  c->grid = *grid; c->dtau = dtau; c->tau0 = tau0; c->eta_s = eta_over_s;
  c->precision = opts->precision; c->visc = eta_over_s > 0.0 ? 1 : 0;
  c->kernel = resolve_kernel(opts->kernel, opts->precision, (long long)grid->nx * grid->ny * grid->nz);
  c->strict = opts->strict_eq53 ? 1 : 0;
  c->ext = ext ? 1 : 0; c->zeta_s = ext ? opts->zeta_over_s : 0.0;
  c->theta = opts->minmod_theta; c->e_floor = opts->e_floor; c->xi = opts->pi_limit_xi;
  c->v_max = opts->v_max > 0.0 ? opts->v_max : 0.999;   // gamma <= 22.4 (A7)
  c->root_iters = opts->root_iters > 0 ? opts->root_iters : 6;
  c->lambda1_hat = opts->lambda1_hat;
  c->c_tau = opts->tau_pi_coeff > 0.0 ? opts->tau_pi_coeff : 5.0;
  c->L = L;
  c->ws = static_cast<char*>(opts->workspace);
  for (int b = 0; b < 3; ++b) c->buf[b] = c->ws + L.off_buf[b];
  c->gstar = c->ws + L.off_gstar;
  c->diag = reinterpret_cast<DiagDev*>(c->ws + L.off_diag);
  c->stream = static_cast<cudaStream_t>(opts->stream);
  c->cur = 0; c->prev = 1; c->step = 0; c->launches = 0; c->loaded = false;
  int rc = opts->precision == 64 ? upload_eos<double>(c, eos, &c->eos64) : upload_eos<float>(c, eos, &c->eos32);
  if (rc == HYDRO_OK && cudaMemsetAsync(c->diag, 0, sizeof(DiagDev), c->stream) != cudaSuccess) rc = HYDRO_ECUDA;
  if (rc == HYDRO_OK && c->kernel == 4) {
    if (L.sz >= (1ll << 31)) rc = HYDRO_EINVAL;      // kernel 4 keeps in-plane offsets in 32 bits
    int dev = 0, nsm = 148;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
      rc = HYDRO_ECUDA;
    c->march_chunk = march_chunk(grid->nx, grid->ny, grid->nz, nsm > 0 ? nsm : 148, opts->precision == 64 ? 2 : CLV_MARCH_MINB32);
  }
  if (rc == HYDRO_OK && L.soa) {
    int dev = 0, nsm = 148;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
      rc = HYDRO_ECUDA;
    choose_tiling(c, nsm > 0 ? nsm : 148);
    // ghost cells and pitch padding are read by the TMA boxes before anything writes them: start from zeros
    if (rc == HYDRO_OK && cudaMemsetAsync(c->buf[0], 0, (size_t)3 * align_up((size_t)L.nelem * L.elem, 256), c->stream) != cudaSuccess)
      rc = HYDRO_ECUDA;
    for (int b = 0; b < 3 && rc == HYDRO_OK; ++b) {
      rc = make_tmap(c, c->buf[b], L.nf, &c->tmap[b][0]);
      if (rc == HYDRO_OK) rc = make_tmap(c, c->buf[b], 4, &c->tmap[b][1]);
    }
  }
  if (rc != HYDRO_OK) { delete c; return rc; }
  *out = c;
  return HYDRO_OK;
}

int hydro_load(hydro_ctx* c, const void* T, const void* pi, int mem) {
  if (!c || !T || (mem != HYDRO_MEM_DEVICE && mem != HYDRO_MEM_HOST)) return HYDRO_EINVAL;
  return c->precision == 64 ? do_load<double>(c, T, pi, mem) : do_load<float>(c, T, pi, mem);
}

int hydro_load_ext(hydro_ctx* c, const void* T, const void* pi, const void* Pi, const void* n_b, int mem) {
  if (!c || !T || (mem != HYDRO_MEM_DEVICE && mem != HYDRO_MEM_HOST)) return HYDRO_EINVAL;
  if (!c->ext) return HYDRO_ESTATE;
  return c->precision == 64 ? do_load<double>(c, T, pi, mem, Pi, n_b) : do_load<float>(c, T, pi, mem, Pi, n_b);
}

int hydro_read_ext(hydro_ctx* c, void* Pi, void* n_b, int mem) {
  if (!c || (mem != HYDRO_MEM_DEVICE && mem != HYDRO_MEM_HOST)) return HYDRO_EINVAL;
  if (!c->loaded || !c->ext) return HYDRO_ESTATE;
  return c->precision == 64 ? do_read_ext<double>(c, Pi, n_b, mem) : do_read_ext<float>(c, Pi, n_b, mem);
}

int hydro_set_history(hydro_ctx* c, const void* u_prev, int mem) {
  if (!c || !u_prev || (mem != HYDRO_MEM_DEVICE && mem != HYDRO_MEM_HOST)) return HYDRO_EINVAL;
  if (!c->loaded) return HYDRO_ESTATE;
  void* p = const_cast<void*>(u_prev);
  return c->precision == 64 ? do_history<double>(c, p, mem, 0) : do_history<float>(c, p, mem, 0);
}

int hydro_read_history(hydro_ctx* c, void* u_prev, int mem) {
  if (!c || !u_prev || (mem != HYDRO_MEM_DEVICE && mem != HYDRO_MEM_HOST)) return HYDRO_EINVAL;
  if (!c->loaded) return HYDRO_ESTATE;
  return c->precision == 64 ? do_history<double>(c, u_prev, mem, 1) : do_history<float>(c, u_prev, mem, 1);
}

int hydro_stage(hydro_ctx* c, int stage) {
  if (!c || (stage != 1 && stage != 2)) return HYDRO_EINVAL;
  if (!c->loaded || c->half != stage - 1) return HYDRO_ESTATE;      // stage 1, then stage 2
  if (c->L.soa || c->strict) return HYDRO_EINVAL;
  return c->precision == 64 ? do_step<double>(c, stage) : do_step<float>(c, stage);
}

size_t hydro_plane_bytes(const hydro_ctx* c) { return (c && !c->L.soa) ? (size_t)c->L.sz * c->L.elem : 0; }

int hydro_planes(hydro_ctx* c, int which, int k0, int nk, void* buf, int dir, int mem) {
  if (!c || !buf || (which != 0 && which != 1) || (dir != 0 && dir != 1) || nk < 1 || k0 < 0 || k0 + nk > c->grid.nz ||
      (mem != HYDRO_MEM_DEVICE && mem != HYDRO_MEM_HOST))
    return HYDRO_EINVAL;
  if (!c->loaded) return HYDRO_ESTATE;
  if (c->L.soa) return HYDRO_EINVAL;
  char* base = static_cast<char*>(which == 0 ? c->buf[c->cur] : c->buf[2]) + (size_t)k0 * c->L.sz * c->L.elem;
  const size_t bytes = (size_t)nk * c->L.sz * c->L.elem;
  const cudaMemcpyKind kind = mem == HYDRO_MEM_DEVICE ? cudaMemcpyDeviceToDevice
                                                      : (dir == 0 ? cudaMemcpyDeviceToHost : cudaMemcpyHostToDevice);
  const cudaError_t e = dir == 0 ? cudaMemcpyAsync(buf, base, bytes, kind, c->stream)
                                 : cudaMemcpyAsync(base, buf, bytes, kind, c->stream);
  if (e != cudaSuccess) return HYDRO_ECUDA;
  if (mem == HYDRO_MEM_HOST && cudaStreamSynchronize(c->stream) != cudaSuccess) return HYDRO_ECUDA;
  return HYDRO_OK;
}

int hydro_step(hydro_ctx* c, int n) {
  if (!c || n < 0) return HYDRO_EINVAL;
  if (!c->loaded || c->half) return HYDRO_ESTATE;
  for (int s = 0; s < n; ++s) {
    const int rc = c->precision == 64 ? do_step<double>(c) : do_step<float>(c);
    if (rc) return rc;
  }
  return HYDRO_OK;
}

int hydro_read(hydro_ctx* c, void* e, void* u, void* pi, int mem) {
  if (!c || (mem != HYDRO_MEM_DEVICE && mem != HYDRO_MEM_HOST)) return HYDRO_EINVAL;
  if (!c->loaded) return HYDRO_ESTATE;
  return c->precision == 64 ? do_read<double>(c, e, u, pi, mem) : do_read<float>(c, e, u, pi, mem);
}


// ---- freeze-out hypersurface (hydro_freezeout.cuh) ----------------------------------------------------

// Freeze-out at constant temperature ("constant freeze-out temperature T_f or constant freeze-out energy
// density e_f"): T(e) of the EoS rule A16 is monotone, so T_f is an e_f.  Host arithmetic only (no device needed).
int hydro_eos_e_of_temperature(const hydro_eos* eos, double T, double* e_out) {
  if (!eos || !e_out || !(T > 0.0) || !(eos->c_sb > 0.0)) return HYDRO_EINVAL;
  if (eos->kind == 0) { *e_out = eos->c_sb * kHbarc * std::pow(T / kHbarc, 4.0); return HYDRO_OK; }
  if (eos->kind != 1 || eos->n < 2 || !eos->T || !(eos->e_min > 0.0) || !(eos->e_max > eos->e_min)) return HYDRO_EINVAL;
  const int n = eos->n;
  auto node = [&](int k) { return eos->e_min * std::pow(eos->e_max / eos->e_min, double(k) / double(n - 1)); };
  if (T <= eos->T[0]) { *e_out = eos->e_min * std::pow(T / eos->T[0], 4.0); return HYDRO_OK; }            // T = T_0 (e/e_min)^{1/4}
  if (T >= eos->T[n - 1]) { *e_out = eos->e_max * std::pow(T / eos->T[n - 1], 4.0); return HYDRO_OK; }
  int lo = 0, hi = n - 1;      // T[lo] <= T < T[hi]
  while (hi - lo > 1) {
    const int mid = (lo + hi) / 2;
    if (eos->T[mid] <= T) lo = mid; else hi = mid;
  }
  const double e0 = node(lo), e1 = node(lo + 1), dT = eos->T[lo + 1] - eos->T[lo];
  if (!(dT > 0.0)) return HYDRO_EINVAL;      // T must increase with e for the inverse to exist
  *e_out = e0 + (T - eos->T[lo]) * (e1 - e0) / dT;
  return HYDRO_OK;
}

size_t hydro_freezeout_bytes(const hydro_grid* grid, int precision) {
  if (!grid || grid->nx < 1 || grid->ny < 1 || grid->nz < 1 || (precision != 64 && precision != 32)) return 0;
  return 256 + 2 * frz_level_bytes(grid, precision);
}

int hydro_freezeout_begin(hydro_ctx* c, void* workspace, size_t bytes, double e_frz) {
  if (!c || !workspace || !(e_frz > 0.0)) return HYDRO_EINVAL;
  if (!c->loaded) return HYDRO_ESTATE;
  if (bytes < hydro_freezeout_bytes(&c->grid, c->precision) || (reinterpret_cast<size_t>(workspace) & 255))
    return HYDRO_ENOMEM;
  c->frz_ws = static_cast<char*>(workspace);
  c->frz_level[0] = c->frz_ws + 256;
  c->frz_level[1] = c->frz_ws + 256 + frz_level_bytes(&c->grid, c->precision);
  c->frz_a = 0; c->frz_e = e_frz; c->frz_slab = 0;
  c->frz_tau_a = c->tau0 + (double)c->step * c->dtau;
  if (cudaMemsetAsync(c->frz_ws, 0, 256, c->stream) != cudaSuccess) return HYDRO_ECUDA;
  return c->precision == 64 ? frz_store_level<double>(c, 0) : frz_store_level<float>(c, 0);
}

int hydro_freezeout_slab(hydro_ctx* c, long long* keys, double* rows, long long capacity, long long* n_total,
                         long long* n_hot) {
  if (!c || capacity < 0 || (capacity > 0 && (!keys || !rows))) return HYDRO_EINVAL;
  if (!c->loaded || !c->frz_ws) return HYDRO_ESTATE;
  const int b = c->frz_a ^ 1;
  int rc = c->precision == 64 ? frz_store_level<double>(c, b) : frz_store_level<float>(c, b);
  if (rc) return rc;
  FrzArgs a;
  memset(&a, 0, sizeof(a));
  a.nx = c->grid.nx; a.ny = c->grid.ny; a.nz = c->grid.nz;
  for (int d = 0; d < 3; ++d) a.bc[d] = c->grid.bc[d];
  a.milne = c->grid.geometry == 0 ? 1 : 0;
  a.N = (long long)a.nx * a.ny * a.nz;
  a.dx = c->grid.dx; a.dy = c->grid.dy; a.de = c->grid.deta;
  a.tau_a = c->frz_tau_a; a.tau_b = c->tau0 + (double)c->step * c->dtau; a.e_frz = c->frz_e;
  a.slab = c->frz_slab; a.capacity = capacity;
  a.cnt = reinterpret_cast<FrzCounters*>(c->frz_ws);
  a.keys = keys; a.rows = rows;
  if (cudaMemsetAsync(&a.cnt->n_hot_b, 0, sizeof(unsigned long long), c->stream) != cudaSuccess) return HYDRO_ECUDA;
  const unsigned nb = (unsigned)((a.N + 255) / 256);
  if (c->precision == 64) {
    const double* la = static_cast<const double*>(c->frz_level[c->frz_a]);
    const double* lb = static_cast<const double*>(c->frz_level[b]);
    freezeout_kernel<double><<<nb, 256, 0, c->stream>>>(a, la, la + a.N, la + 5 * a.N, lb, lb + a.N, lb + 5 * a.N);
  } else {
    const float* la = static_cast<const float*>(c->frz_level[c->frz_a]);
    const float* lb = static_cast<const float*>(c->frz_level[b]);
    freezeout_kernel<float><<<nb, 256, 0, c->stream>>>(a, la, la + a.N, la + 5 * a.N, lb, lb + a.N, lb + 5 * a.N);
  }
  c->launches += 1;
  if (cudaGetLastError() != cudaSuccess) return HYDRO_ECUDA;
  FrzCounters h;
  if (cudaMemcpyAsync(&h, a.cnt, sizeof(h), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) return HYDRO_ECUDA;
  if (cudaStreamSynchronize(c->stream) != cudaSuccess) return HYDRO_ECUDA;
  c->frz_a = b; c->frz_tau_a = a.tau_b; c->frz_slab += 1;
  if (n_total) *n_total = (long long)h.n_elem;
  if (n_hot) *n_hot = (long long)h.n_hot_b;
  return (long long)h.n_elem > capacity ? HYDRO_ENOMEM : HYDRO_OK;
}

int hydro_freezeout_run(hydro_ctx* c, int steps_per_slab, int max_slabs, long long* keys, double* rows,
                        long long capacity, long long* n_total, int* n_slabs) {
  if (!c || steps_per_slab < 1 || max_slabs < 0) return HYDRO_EINVAL;
  if (!c->loaded || !c->frz_ws) return HYDRO_ESTATE;
  int done = 0, rc = HYDRO_OK;
  long long hot = 1;
  while (done < max_slabs && hot > 0) {
    if ((rc = hydro_step(c, steps_per_slab))) break;
    rc = hydro_freezeout_slab(c, keys, rows, capacity, n_total, &hot);
    if (rc) break;
    done += 1;
  }
  if (n_slabs) *n_slabs = done;
  return rc;
}

int hydro_diag(hydro_ctx* c, hydro_diag_t* out) {
  if (!c || !out) return HYDRO_EINVAL;
  DiagDev d;
  if (cudaMemcpyAsync(&d, c->diag, sizeof(d), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess) return HYDRO_ECUDA;
  if (cudaStreamSynchronize(c->stream) != cudaSuccess) return HYDRO_ECUDA;
  const int slot = (int)((c->step + 1) & 1);    // slot of the last completed step ((step-1)&1); load uses 1
  auto as_double = [](unsigned long long b) { double v; memcpy(&v, &b, 8); return v; };
  out->tau = c->tau0 + (double)c->step * c->dtau;
  out->step = c->step;
  for (int a = 0; a < 3; ++a) out->cfl[a] = c->step > 0 ? as_double(d.cfl[slot][a]) : 0.0;
  out->e_max = as_double(d.emax[slot]);
  out->n_floor = (long long)d.n_floor; out->n_clamp = (long long)d.n_clamp;
  out->n_pi_limited = (long long)d.n_limit; out->n_nan = (long long)d.n_nan;
  out->n_root_unconverged = (long long)d.n_unconv;
  int warn = 0;
  if (out->cfl[0] + out->cfl[1] + out->cfl[2] > 1.0) warn |= HYDRO_WARN_CFL;
  if (d.n_nan) warn |= HYDRO_WARN_NAN;
  if (d.n_unconv) warn |= HYDRO_WARN_ROOT;
  return warn;
}

long long hydro_launch_count(const hydro_ctx* c) { return c ? c->launches : 0; }

int hydro_kernel(const hydro_ctx* c) { return c ? c->kernel : 0; }

void hydro_destroy(hydro_ctx* c) { delete c; }

const char* hydro_strerror(int code) {
  switch (code) {
    case HYDRO_OK: return "ok";
    case HYDRO_EINVAL: return "invalid argument";
    case HYDRO_ENOMEM: return "workspace too small or misaligned";
    case HYDRO_ECUDA: return "CUDA error (no usable device, or a launch/copy failed)";
    case HYDRO_ESTATE: return "call order error (hydro_load must come first)";
    default: return code > 0 ? "warning mask" : "unknown error";
  }
}

}  // extern "C"
