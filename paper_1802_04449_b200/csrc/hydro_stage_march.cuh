// hydro_stage_march.cuh -- "kernel 4": the per-cell fused stage kernel MARCHING along eta_s (default kernel).
//
// Same field store (blocked extended state, 19 words per cell), same x / y flux code (axis_flux) and same stage tail
// (hydro_stage_update.cuh) as kernel 2.  What changes follows the ncu profile of kernel 2 (profiles/round2_kernels.md:
// 43 % of the stall samples on the 28 % of the instructions that form the eta_s fluxes, because the four off-centre
// planes of the eta_s star miss L1; long-scoreboard stalls 2.3-3.2 warps per issue, L1 hit rate 53 %):
//   * a block owns a 32 x 8 column of cells and walks through a chunk of eta_s planes;
//   * the eta_s flux is a PIPELINE per column: when plane p comes into reach the limited slope of cell p-1 and the
//     KT face p-3/2 are formed ONCE (kernel 2: every eta slope three times, every face twice), and the flux difference
//     of cell k = p-2 is completed from the kept left state (Q^l, F^l) of cell p-2 and the kept face flux p-5/2;
//   * that kept state -- 3 values for each of the 14 evolved fields -- is indexed at run time by the rolled pi-field
//     loop, so it cannot sit in registers; it lives in TENSOR MEMORY (tcgen05.st / tcgen05.ld, 32x32b: every thread
//     owns a lane segment).  No tensor-core instruction is issued;
//   * the x and y stars of plane k (and the cell's own state) are read from a SHARED-MEMORY TILE: 36 x 12 points x 19
//     fields (65.7 KB fp64, two blocks per SM), filled with cp.async one plane ahead, behind the stage tail of the
//     previous plane -- the paper's local-memory block, which its GPU had no room for.  The
//     boundary rule a11 is applied to the source index of the copy, so the tile needs no special cases;
//   * fp32 only: the raw words of plane p are stashed in tensor memory next to the pipeline state, so the next eta_s step
//     reads plane p-1 from there and only ONE plane per step comes from global memory (fp64: measured slower, off);
//   * one block barrier per plane (two with the tile) keeps the 8 warps of a block on the same instruction-cache lines
//     of the ~90 KB loop body: without it "no instruction" stalls are 1.8 warps per issue, with it 0.19.
//   * fp64 only: L2 eviction hints (keep the first read of a plane for the tile fill two steps later; stream the rest).
// Measured at 301x301x201 (profiles/round2_bench.md): 11.3 ms per step fp64, 5.84 ms fp32 (kernel 2: 14.4 / 7.5).
// Citations: KT scheme PAPER.md:193-213 (Eq.40-44); RK2 :225-239 (Eq.49-54).
#pragma once
#include "hydro_stage_fused.cuh"
#include "hydro_stage_tile.cuh"      // PrivTmem, lr, face2

namespace clv {

#ifndef CLV_MARCH_PF
#define CLV_MARCH_PF 1      // prefetch of the own column of plane p+1: 1 into L1, 2 into L2, 0 none
#endif
#ifndef CLV_MARCH_SYNC
#define CLV_MARCH_SYNC 1    // block barrier per plane: keeps the warps of a block on the same instruction-cache lines
                            // (measured at 301x301x201: 15.7 -> 13.4 ms per step fp64, 7.6 -> 6.95 fp32; "no instruction"
                            // stalls 1.8 -> 0.19 warps per issue, profiles/round2_kernel4.md)
#endif

#ifndef CLV_MARCH_TILE
#define CLV_MARCH_TILE 1    // 1: the x / y stars of plane k are read from a shared-memory tile (32 x 8 cells + 2-cell halo,
                            // all fields) filled with cp.async one plane ahead, behind the stage tail of the previous plane
#endif
#ifndef CLV_MARCH_ETA_TILE
#define CLV_MARCH_ETA_TILE 1   // with the tile: the eta_s step takes plane p-2 (own column) from the tile too, so the tile
                               // is also filled for the two warm-up planes of a chunk
#endif
#ifndef CLV_MARCH_PF_TAIL
#define CLV_MARCH_PF_TAIL 0    // 1: L1 prefetch of what the stage tail reads at the cell (state n / history / u*^tau / plane
                               // k-1); measured neutral (11.84 vs 11.75 ms fp64), off
#endif
#ifndef CLV_MARCH_TY
#define CLV_MARCH_TY 8         // rows of cells per block (one warp per row)
#endif
constexpr int MTY = CLV_MARCH_TY, MT_NTHR = 32 * MTY;
constexpr int MT_SX = 36, MT_SY = MTY + 4, MT_FST = MT_SX * MT_SY;      // tile extents and field stride (elements)
constexpr int MT_NSLOT = (MT_FST + MT_NTHR - 1) / MT_NTHR;              // tile points copied per thread

__device__ __forceinline__ void cp_async_elem(double* dst_smem, const double* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_elem_hint(double* dst_smem, const double* src, unsigned long long pol) {
  asm volatile("cp.async.ca.shared.global.L2::cache_hint [%0], [%1], 8, %2;" ::"r"(smem_u32(dst_smem)), "l"(src), "l"(pol) : "memory");
}
__device__ __forceinline__ void cp_async_elem_hint(float* dst_smem, const float* src, unsigned long long pol) {
  asm volatile("cp.async.ca.shared.global.L2::cache_hint [%0], [%1], 4, %2;" ::"r"(smem_u32(dst_smem)), "l"(src), "l"(pol) : "memory");
}
__device__ __forceinline__ void cp_async_elem(float* dst_smem, const float* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory");
}
// two x-consecutive elements in one copy: 16 bytes (fp64; .cg: through L2 only, the tile does not pass through L1) / 8 bytes
__device__ __forceinline__ void cp_async_pair(double* dst_smem, const double* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_pair(float* dst_smem, const float* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst_smem)), "l"(src) : "memory");
}
// L2 eviction hints (createpolicy + ld/st .L2::cache_hint).  A plane is read twice by a block, two steps apart (own
// column in the eta_s step, then as the tile), and ncu shows 1.4 x the compulsory DRAM reads: the first read asks L2 to
// keep the lines (evict_last), the read-once operands of the stage tail and the output stores ask it not to (evict_first).
// Measured at 301x301x201 (fp64): 11.65 -> 11.29 ms per step, DRAM reads of stage 2 8.0 -> 6.7 GB (stage 1 4.9 -> 4.6), all
// DRAM bytes 1.80 -> 1.63 x algorithmic; fp32: 5.84 -> 5.91 ms, so the hints are on in fp64 only.
#ifndef CLV_MARCH_L2HINT
#define CLV_MARCH_L2HINT 2      // 0 off, 1 on, 2 on in fp64 only
#endif
__device__ __forceinline__ unsigned long long l2_policy(bool keep) {
  unsigned long long p;
  if (keep) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  else asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ double ldg_hint(const double* p, unsigned long long pol) {
  double v;
  asm volatile("ld.global.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(p), "l"(pol));
  return v;
}
__device__ __forceinline__ float ldg_hint(const float* p, unsigned long long pol) {
  float v;
  asm volatile("ld.global.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(v) : "l"(p), "l"(pol));
  return v;
}
__device__ __forceinline__ void stg_hint(double* p, double v, unsigned long long pol) {
  asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(p), "d"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ void stg_hint(float* p, float v, unsigned long long pol) {
  asm volatile("st.global.L2::cache_hint.f32 [%0], %1, %2;" ::"l"(p), "f"(v), "l"(pol) : "memory");
}
#ifndef CLV_MARCH_FILLHINT
#define CLV_MARCH_FILLHINT 0     // 1: the tile fill (second and last read of a plane by this block) asks L2 not to keep the lines
#endif
#ifndef CLV_MARCH_PAIRS
#define CLV_MARCH_PAIRS 0      // 1: tile fill in pairs of x-consecutive points (128-bit copies in fp64).  Measured at
                               // 301x301x201: 11.65-11.71 ms per step fp64 / 5.92 fp32 against 11.45 / 5.84 with one point per
                               // copy (whose warp request is one contiguous 256-byte stretch), so it is off
#endif

// ---- tensor memory as the per-thread store of the eta_s pipeline --------------------------------------------------------
// Per thread (one TMEM lane segment, 32x32b shape): for each of the 14 evolved fields FOUR values
//   [Q^l, F^l of cell p-2;  2H of face p-5/2;  the field's raw value at plane p-1 (the "stash")]
// and three more stashed words of plane p-1 (u~^tau, P, c_eta): 59 values = 118 (fp64) / 59 (fp32) columns; 8 warps share
// 4 lane quadrants, so a block allocates 256 / 128 columns.  The stash means that an eta_s step reads only ONE plane
// from global memory (plane p; p-1 comes from here, p-2 from the shared-memory tile).
// Measured at 301x301x201 (profiles/round2_bench.md): fp32 6.21 -> 6.06 ms per step, fp64 11.79 -> 12.03 (the TMEM round
// trips cost the fp64 kernel more than the L1 misses they replace), so the stash is on in fp32 only.
#ifndef CLV_MARCH_STASH
#define CLV_MARCH_STASH 2      // 0 off, 1 on, 2 on in fp32 only
#endif
template <int N> struct TmWords { unsigned w[N]; };
__device__ __forceinline__ void tm_ld_x(unsigned addr, TmWords<2>& v) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(v.w[0]), "=r"(v.w[1]) : "r"(addr) : "memory");
}
__device__ __forceinline__ void tm_ld_x(unsigned addr, TmWords<1>& v) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=r"(v.w[0]) : "r"(addr) : "memory");
}
__device__ __forceinline__ void tm_ld_x(unsigned addr, TmWords<4>& v) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
               : "=r"(v.w[0]), "=r"(v.w[1]), "=r"(v.w[2]), "=r"(v.w[3]) : "r"(addr) : "memory");
}
__device__ __forceinline__ void tm_ld_x(unsigned addr, TmWords<8>& v) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(v.w[0]), "=r"(v.w[1]), "=r"(v.w[2]), "=r"(v.w[3]), "=r"(v.w[4]), "=r"(v.w[5]), "=r"(v.w[6]), "=r"(v.w[7])
               : "r"(addr) : "memory");
}
__device__ __forceinline__ void tm_ld_x(unsigned addr, TmWords<16>& v) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
               : "=r"(v.w[0]), "=r"(v.w[1]), "=r"(v.w[2]), "=r"(v.w[3]), "=r"(v.w[4]), "=r"(v.w[5]), "=r"(v.w[6]), "=r"(v.w[7]),
                 "=r"(v.w[8]), "=r"(v.w[9]), "=r"(v.w[10]), "=r"(v.w[11]), "=r"(v.w[12]), "=r"(v.w[13]), "=r"(v.w[14]), "=r"(v.w[15])
               : "r"(addr) : "memory");
}
__device__ __forceinline__ void tm_st_x(unsigned addr, const TmWords<1>& v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(addr), "r"(v.w[0]) : "memory");
}
__device__ __forceinline__ void tm_st_x(unsigned addr, const TmWords<2>& v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(addr), "r"(v.w[0]), "r"(v.w[1]) : "memory");
}
__device__ __forceinline__ void tm_st_x(unsigned addr, const TmWords<4>& v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.w[0]), "r"(v.w[1]),
               "r"(v.w[2]), "r"(v.w[3]) : "memory");
}
__device__ __forceinline__ void tm_st_x(unsigned addr, const TmWords<8>& v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(addr), "r"(v.w[0]),
               "r"(v.w[1]), "r"(v.w[2]), "r"(v.w[3]), "r"(v.w[4]), "r"(v.w[5]), "r"(v.w[6]), "r"(v.w[7]) : "memory");
}
__device__ __forceinline__ void tm_st_x(unsigned addr, const TmWords<16>& v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
               ::"r"(addr), "r"(v.w[0]), "r"(v.w[1]), "r"(v.w[2]), "r"(v.w[3]), "r"(v.w[4]), "r"(v.w[5]), "r"(v.w[6]), "r"(v.w[7]),
               "r"(v.w[8]), "r"(v.w[9]), "r"(v.w[10]), "r"(v.w[11]), "r"(v.w[12]), "r"(v.w[13]), "r"(v.w[14]), "r"(v.w[15])
               : "memory");
}
// the wait ties the loaded registers to a point after it (no use can be scheduled before the wait)
template <int N> __device__ __forceinline__ void tm_wait_ld_x(TmWords<N>& v) {
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < N; ++i) asm volatile("" : "+r"(v.w[i]));
}
template <int N> __device__ __forceinline__ double tm_val(const TmWords<N>& v, int i, double) {
  return __hiloint2double((int)v.w[2 * i + 1], (int)v.w[2 * i]);
}
template <int N> __device__ __forceinline__ float tm_val(const TmWords<N>& v, int i, float) { return __uint_as_float(v.w[i]); }
template <int N> __device__ __forceinline__ void tm_set(TmWords<N>& v, int i, double x) {
  v.w[2 * i] = (unsigned)__double2loint(x); v.w[2 * i + 1] = (unsigned)__double2hiint(x);
}
template <int N> __device__ __forceinline__ void tm_set(TmWords<N>& v, int i, float x) { v.w[i] = __float_as_uint(x); }

template <typename R, int NFLD = 14>
struct MarchTmem {
  static constexpr int W = sizeof(R) / 4;
  static constexpr int NVAL = NFLD * 4 + (NFLD == 14 ? 3 : 0);           // 16 fields (8(f)-3): no stash, no aux words
  static constexpr int COLS_PER_THREAD = NVAL * W;                       // 118 (fp64) / 59 (fp32)
  static constexpr int WPQ = (MTY + 3) / 4;                              // warps per lane quadrant
  static constexpr int ALLOC_COLS = WPQ * COLS_PER_THREAD <= 64 ? 64 : (WPQ * COLS_PER_THREAD <= 128 ? 128 : (WPQ * COLS_PER_THREAD <= 256 ? 256 : 512));
  unsigned base;
  __device__ __forceinline__ void init(unsigned tmem_base, int warp) {
    base = tmem_base + ((unsigned)(32 * (warp & 3)) << 16) + (unsigned)((warp >> 2) * COLS_PER_THREAD);
  }
  __device__ __forceinline__ unsigned field(int f) const { return base + (unsigned)(f * 4 * W); }      // 4 values of field f
  __device__ __forceinline__ unsigned stash(int f) const { return base + (unsigned)((f * 4 + 3) * W); }
  __device__ __forceinline__ unsigned aux(int i) const { return base + (unsigned)((NFLD * 4 + i) * W); }   // 0 u~^tau, 1 P, 2 c_eta
  // three-value access (the build without the stash, CLV_MARCH_STASH = 0)
  __device__ __forceinline__ void get(int f, R& ql, R& fl, R& h) const { tm_ld3(field(f), ql, fl, h); }
  __device__ __forceinline__ void put(int f, R ql, R fl, R h) const {
    tm_st(field(f), ql); tm_st(field(f) + W, fl); tm_st(field(f) + 2 * W, h);
  }
};
template <int N, int M> __device__ __forceinline__ void tm_wait_ld_x(TmWords<N>& a, TmWords<M>& b) {
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < N; ++i) asm volatile("" : "+r"(a.w[i]));
#pragma unroll
  for (int i = 0; i < M; ++i) asm volatile("" : "+r"(b.w[i]));
}

#ifndef CLV_MARCH_MINB32
#define CLV_MARCH_MINB32 3      // fp32 blocks per SM: 3 (<= 85 registers) measured 6.28 ms per step against 6.8 with 2
#endif
// EXT: the 16-word cell -- fields 14 (Pi) and 15 (n) ride along as two more pi-like fields.
template <typename R, bool VISC, int MODE, bool TILE, bool EXT = false>
__global__ void __launch_bounds__(MT_NTHR, ((sizeof(R) == 4 ? CLV_MARCH_MINB32 : 2) * 8 / MTY > 0 ? (sizeof(R) == 4 ? CLV_MARCH_MINB32 : 2) * 8 / MTY : 1))
stage_march_kernel(const StageArgs<R> a, const int chunk) {
  static_assert(MODE == 1 || MODE == 2, "the bootstrap (MODE 0) runs in the per-cell kernel");
  constexpr bool USE_PI = VISC;
  static_assert(!EXT || VISC, "the bulk / baryon extension rides on the viscous path");
  constexpr int NF = VISC ? (EXT ? 16 : 14) : 4;
  constexpr int NPI = EXT ? 12 : 10, NTRIP = NPI / 2;      // pi-like fields, two per trip
  constexpr int OX = NF * FS;
  const int lane = threadIdx.x, row = threadIdx.y, tid = row * 32 + lane;
  const int i = blockIdx.x * 32 + lane, j = blockIdx.y * MTY + row;
  const bool active = (i < a.nx) && (j < a.ny);
  const int ic = active ? i : 0, jc = active ? j : 0;
  const int kc0 = blockIdx.z * chunk, kc1 = min(kc0 + chunk, a.nz);
  constexpr int sf = FS;
  const R* __restrict__ in = a.in;

  __shared__ R sS[USE_PI ? NPI * MT_NTHR : 1];
  __shared__ unsigned s_tmem;
  extern __shared__ __align__(16) unsigned char tile_raw[];      // TILE: R tile[NF + 5][12][36]
  R* const tile = reinterpret_cast<R*>(tile_raw);
  constexpr int NFT = NF + X_COUNT;
  using Priv = MarchTmem<R, EXT ? 16 : 14>;
  if (row == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)),
                 "r"((unsigned)Priv::ALLOC_COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  Priv priv;
  priv.init(s_tmem, row);

  // in-plane offsets (elements) of the x and y stars and of the column itself
  // (32-bit: hydro_create admits kernel 4 only when a plane has fewer than 2^31 elements)
  const int col = (int)(jc * a.sy + xoff(ic, a.blk));
  int offx[5], offy[5];
#pragma unroll
  for (int p = 0; p < 5; ++p) {
    offx[p] = (int)(jc * a.sy + xoff(bmap(ic + p - 2, a.nx, a.bc[0]), a.blk));
    offy[p] = (int)(bmap(jc + p - 2, a.ny, a.bc[1]) * a.sy + xoff(ic, a.blk));
  }
  const long long cg0 = (long long)jc * a.gp + ic;
  constexpr bool L2H = (CLV_MARCH_L2HINT == 1) || (CLV_MARCH_L2HINT == 2 && sizeof(R) == 8);
  const unsigned long long pol_keep = L2H ? l2_policy(true) : 0ull;
  const unsigned long long pol_once = L2H ? l2_policy(false) : 0ull;
#define LDK(ptr) (L2H ? ldg_hint((ptr), pol_keep) : *(ptr))
#define LD1(ptr) (L2H ? ldg_hint((ptr), pol_once) : *(ptr))
  // tile fill (boundary rule a11 applied to the source index, so the tile needs no special cases).  The 36 x 12 points
  // are copied as 18 x 12 PAIRS of x-consecutive points, one pair per thread and field: the tile starts at an even x
  // (32 bx - 2), pairs never straddle an x-block of the store, so a pair is one aligned 16-byte (fp64) / 8-byte (fp32)
  // cp.async -- unless the boundary rule maps its two points to non-consecutive cells (clamp at the domain edge, wrap),
  // in which case the two points are copied one by one.
  constexpr int NPAIR = MT_FST / 2, NPSLOT = (NPAIR + MT_NTHR - 1) / MT_NTHR;
  int tsrc[CLV_MARCH_PAIRS ? NPSLOT : MT_NSLOT], tsrc1[CLV_MARCH_PAIRS ? NPSLOT : 1];
  if (CLV_MARCH_PAIRS) {
#pragma unroll
    for (int s = 0; s < NPSLOT; ++s) {
      const int pr = min(tid + MT_NTHR * s, NPAIR - 1);
      const int r = pr / (MT_SX / 2), cx = 2 * (pr - r * (MT_SX / 2));
      const long long rowoff = bmap(blockIdx.y * MTY - 2 + r, a.ny, a.bc[1]) * a.sy;
      tsrc[s] = (int)(rowoff + xoff(bmap(blockIdx.x * 32 - 2 + cx, a.nx, a.bc[0]), a.blk));
      tsrc1[s] = (int)(rowoff + xoff(bmap(blockIdx.x * 32 - 2 + cx + 1, a.nx, a.bc[0]), a.blk));
    }
  } else {
#pragma unroll
    for (int s = 0; s < MT_NSLOT; ++s) {
      const int pos = min(tid + MT_NTHR * s, MT_FST - 1);
      const int r = pos / MT_SX, cx = pos - r * MT_SX;
      tsrc[s] = (int)(bmap(blockIdx.y * MTY - 2 + r, a.ny, a.bc[1]) * a.sy +
                      xoff(bmap(blockIdx.x * 32 - 2 + cx, a.nx, a.bc[0]), a.blk));
    }
  }
  auto fill_tile = [&](int kk) {
    const R* __restrict__ src = in + (long long)kk * a.sz;
    if (CLV_MARCH_PAIRS) {
#pragma unroll
      for (int s = 0; s < NPSLOT; ++s) {
        if (tid + MT_NTHR * s < NPAIR) {
          const R* __restrict__ g0 = src + tsrc[s];
          R* d0 = tile + 2 * (tid + MT_NTHR * s);
          if (tsrc1[s] == tsrc[s] + 1 && (tsrc[s] & 1) == 0) {
#pragma unroll
            for (int m = 0; m < NFT; ++m) cp_async_pair(d0 + m * MT_FST, g0 + m * FS);
          } else {
            const R* __restrict__ g1 = src + tsrc1[s];
#pragma unroll
            for (int m = 0; m < NFT; ++m) { cp_async_elem(d0 + m * MT_FST, g0 + m * FS); cp_async_elem(d0 + m * MT_FST + 1, g1 + m * FS); }
          }
        }
      }
    } else {
#pragma unroll
      for (int s = 0; s < MT_NSLOT; ++s) {
        if (tid + MT_NTHR * s < MT_FST) {
          const R* __restrict__ g0 = src + tsrc[s];
          R* d0 = tile + (tid + MT_NTHR * s);
#pragma unroll
          for (int m = 0; m < NFT; ++m) {
            if (CLV_MARCH_FILLHINT && L2H) cp_async_elem_hint(d0 + m * MT_FST, g0 + m * FS, pol_once);
            else cp_async_elem(d0 + m * MT_FST, g0 + m * FS);
          }
        }
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  constexpr bool ETILE = TILE && (CLV_MARCH_ETA_TILE != 0);
  if (TILE) fill_tile(ETILE ? bmap(kc0 - 2, a.nz, a.bc[2]) : kc0);
  const R* const town = tile + (row + 2) * MT_SX + (lane + 2);      // own point inside a field plane of the tile

  const R tf = a.milne ? a.tau : R(1);
  const R th2 = R(2) * a.theta;
  const R sc_pi = R(0.5) * a.scale[2], sc_T = sc_pi * tf;
  R cflm0 = R(0), cflm1 = R(0), cflm2 = R(0), emax = R(0);

  constexpr bool STASH = !EXT && ((CLV_MARCH_STASH == 1) || (CLV_MARCH_STASH == 2 && sizeof(R) == 4));
  if constexpr (STASH) {   // the stash starts with plane kc0-1
    const R* __restrict__ qm = in + (long long)bmap(kc0 - 1, a.nz, a.bc[2]) * a.sz + col;
    TmWords<Priv::W> v;
#pragma unroll
    for (int m = 0; m < NF; ++m) { tm_set(v, 0, qm[m * FS]); tm_st_x(priv.stash(m), v); }
    tm_set(v, 0, qm[OX + X_G * FS]); tm_st_x(priv.aux(0), v);
    tm_set(v, 0, qm[OX + X_P * FS]); tm_st_x(priv.aux(1), v);
    tm_set(v, 0, qm[OX + X_CN * FS]); tm_st_x(priv.aux(2), v);
    tm_wait_st();
  }
  for (int p = kc0; p <= kc1 + 1; ++p) {
    const int k = p - 2;
    const bool centre = p >= kc0 + 2;                      // block-uniform
    if (CLV_MARCH_SYNC && !TILE) __syncthreads();
    const R* __restrict__ q2 = in + (long long)bmap(p - 2, a.nz, a.bc[2]) * a.sz + col;    // plane p-2 (= k)
    const R* __restrict__ q1 = in + (long long)bmap(p - 1, a.nz, a.bc[2]) * a.sz + col;
    const R* __restrict__ q0 = in + (long long)bmap(p, a.nz, a.bc[2]) * a.sz + col;
    if (ETILE) {
      asm volatile("cp.async.wait_all;" ::: "memory");
      __syncthreads();                                     // tile(p-2) complete and visible
    }
    if (CLV_MARCH_PF && p + 1 <= kc1 + 1 && (lane & (sizeof(R) == 8 ? 15 : 31)) == 0) {
      const R* __restrict__ qn = in + (long long)bmap(p + 1, a.nz, a.bc[2]) * a.sz + col;
#pragma unroll
      for (int m = 0; m < NF + X_COUNT; ++m) {
        if (CLV_MARCH_PF == 1) prefetch_l1(qn + m * FS);
        else asm volatile("prefetch.global.L2 [%0];" ::"l"(qn + m * FS));
      }
    }

    if (CLV_MARCH_PF_TAIL && centre && (lane & (sizeof(R) == 8 ? 15 : 31)) == 0) {
      const long long cpf = (long long)k * a.sz + col;
      if (MODE == 2) {
#pragma unroll
        for (int m = 0; m < NF; ++m) prefetch_l1(a.sn + cpf + m * FS);
        prefetch_l1(a.sn + cpf + OX + X_G * FS); prefetch_l1(a.sn + cpf + OX + X_P * FS);
        if (USE_PI) prefetch_l1(a.gstar + (long long)k * a.ny * a.gp + cg0);
      } else if (USE_PI) {
#pragma unroll
        for (int m = 0; m < 3; ++m) prefetch_l1(a.uprev + cpf + m * FS);
      }
      if (USE_PI) {
        const R* __restrict__ zmp = in + (long long)bmap(k - 1, a.nz, a.bc[2]) * a.sz + col;
        prefetch_l1(zmp + FS); prefetch_l1(zmp + 2 * FS); prefetch_l1(zmp + 3 * FS); prefetch_l1(zmp + OX + X_G * FS);
      }
    }

    R S[16];
#pragma unroll
    for (int m = 0; m < 16; ++m) S[m] = R(0);
    R cfl2;
    // ---- eta_s pipeline step: slope of cell p-1, face p-3/2, flux difference of cell p-2 ---------------------------
    if constexpr (STASH) {
      // plane p from global memory, plane p-1 from the tensor-memory stash, plane p-2 from the tile
      constexpr int TW = Priv::W;
      using W1 = TmWords<TW>;
      using W4 = TmWords<4 * TW>;
      using W8 = TmWords<8 * TW>;
#define P2_LD(m) (ETILE ? town[(m) * MT_FST] : q2[(m) * FS])
      R g[3], ua[3], Pp[3], e3[3];
      g[0] = P2_LD(NF + X_G); ua[0] = P2_LD(3); Pp[0] = P2_LD(NF + X_P); e3[0] = P2_LD(0);
      const R c2 = P2_LD(NF + X_CN);
      g[2] = LDK(q0 + OX + X_G * FS); ua[2] = LDK(q0 + 3 * FS); Pp[2] = LDK(q0 + OX + X_P * FS); e3[2] = LDK(q0);
      const R cnew = LDK(q0 + OX + X_CN * FS);
      R c1;
      {
        W1 a0, a1, a2, s0, s3;      // u~^tau, P, c_eta, e (field 0), u~^eta (field 3) of plane p-1
        tm_ld_x(priv.aux(0), a0); tm_ld_x(priv.aux(1), a1); tm_ld_x(priv.aux(2), a2);
        tm_ld_x(priv.stash(0), s0); tm_ld_x(priv.stash(3), s3);
        tm_wait_ld_x(a0, a1); tm_wait_ld_x(a2, s0); tm_wait_ld_x(s3);
        g[1] = tm_val(a0, 0, R()); Pp[1] = tm_val(a1, 0, R()); c1 = tm_val(a2, 0, R()); e3[1] = tm_val(s0, 0, R());
        ua[1] = tm_val(s3, 0, R());
      }
      const R cface = max_(c2, c1);
      cfl2 = c2 * a.h * a.scale[2];
      {
        R wq[3], wa[3];
#pragma unroll
        for (int t = 0; t < 3; ++t) {
          const R w = e3[t] + Pp[t];
          wq[t] = w * g[t]; wa[t] = w * ua[t];
        }
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
          const int o_t = F_PI + mu, o_a = F_PI + c_pidx[3][mu];
          W4 k4; W1 st, sa;
          tm_ld_x(priv.field(mu), k4);
          if (USE_PI) { tm_ld_x(priv.stash(o_t), st); tm_ld_x(priv.stash(o_a), sa); tm_wait_ld_x(st, sa); }
          tm_wait_ld_x(k4);
          const R raw_p = LDK(q0 + mu * FS);      // field mu at plane p (e for mu = 0): the new stash
          R um[3];
          um[0] = mu == 0 ? g[0] : P2_LD(mu);
          um[1] = mu == 0 ? g[1] : tm_val(k4, 3, R());
          um[2] = mu == 0 ? g[2] : raw_p;
          R q[3], f[3];
#pragma unroll
          for (int t = 0; t < 3; ++t) {
            q[t] = wq[t] * um[t] - (mu == 0 ? Pp[t] : R(0));
            f[t] = wa[t] * um[t] + (mu == 3 ? Pp[t] : R(0));
          }
          if (USE_PI) {
            q[0] += P2_LD(o_t); f[0] += P2_LD(o_a);
            q[1] += tm_val(st, 0, R()); f[1] += tm_val(sa, 0, R());
            q[2] += LDK(q0 + o_t * FS); f[2] += LDK(q0 + o_a * FS);
          }
          const R QLk = tm_val(k4, 0, R()), FLk = tm_val(k4, 1, R()), Hk = tm_val(k4, 2, R());
          R QL1, QR1, FL1, FR1;
          lr(q[0], q[1], q[2], th2, QL1, QR1);
          lr(f[0], f[1], f[2], th2, FL1, FR1);
          const R Hn = face2(QLk, FLk, QR1, FR1, cface);
          S[mu] = -(Hn - Hk) * sc_T;
          W4 n4;
          tm_set(n4, 0, QL1); tm_set(n4, 1, FL1); tm_set(n4, 2, Hn); tm_set(n4, 3, raw_p);
          tm_st_x(priv.field(mu), n4);
        }
        // the three derived words of plane p
        W1 a0, a1, a2;
        tm_set(a0, 0, g[2]); tm_set(a1, 0, Pp[2]); tm_set(a2, 0, cnew);
        tm_st_x(priv.aux(0), a0); tm_st_x(priv.aux(1), a1); tm_st_x(priv.aux(2), a2);
      }
      if (USE_PI) {
        R* slot = &sS[tid];
#pragma unroll 1
        for (int t = 0; t < 5; ++t) {
          const int fa = F_PI + 2 * t;
          W8 k8;
          tm_ld_x(priv.field(fa), k8);
          const R va0 = P2_LD(fa), vb0 = P2_LD(fa + 1), va2 = LDK(q0 + fa * FS), vb2 = LDK(q0 + (fa + 1) * FS);
          tm_wait_ld_x(k8);
          const R va1 = tm_val(k8, 3, R()), vb1 = tm_val(k8, 7, R());
          R QL1, QR1, FL1, FR1;
          W8 n8;
          lr(g[0] * va0, g[1] * va1, g[2] * va2, th2, QL1, QR1);
          lr(ua[0] * va0, ua[1] * va1, ua[2] * va2, th2, FL1, FR1);
          const R Hna = face2(tm_val(k8, 0, R()), tm_val(k8, 1, R()), QR1, FR1, cface);
          tm_set(n8, 0, QL1); tm_set(n8, 1, FL1); tm_set(n8, 2, Hna); tm_set(n8, 3, va2);
          lr(g[0] * vb0, g[1] * vb1, g[2] * vb2, th2, QL1, QR1);
          lr(ua[0] * vb0, ua[1] * vb1, ua[2] * vb2, th2, FL1, FR1);
          const R Hnb = face2(tm_val(k8, 4, R()), tm_val(k8, 5, R()), QR1, FR1, cface);
          tm_set(n8, 4, QL1); tm_set(n8, 5, FL1); tm_set(n8, 6, Hnb); tm_set(n8, 7, vb2);
          tm_st_x(priv.field(fa), n8);
          slot[0] = -(Hna - tm_val(k8, 2, R())) * sc_pi;
          slot[MT_NTHR] = -(Hnb - tm_val(k8, 6, R())) * sc_pi;
          slot += 2 * MT_NTHR;
        }
      }
      tm_wait_st();
#undef P2_LD
    } else {
      // planes p and p-1 from global memory (L1 / L2), plane p-2 from the tile
      const R* __restrict__ pp[3] = {q2, q1, q0};
      // field m of plane p-2+t at the own column (t is a constant after unrolling)
#define ETA_LD(t, m) ((ETILE && (t) == 0) ? town[(m) * MT_FST] : ((t) == 2 ? LDK(pp[t] + (m) * FS) : pp[t][(m) * FS]))
      R g[3], ua[3];
#pragma unroll
      for (int t = 0; t < 3; ++t) { g[t] = ETA_LD(t, NF + X_G); ua[t] = ETA_LD(t, 3); }
      const R c2 = ETA_LD(0, NF + X_CN);
      const R cface = max_(c2, q1[OX + X_CN * FS]);
      cfl2 = c2 * a.h * a.scale[2];
      {
        R wq[3], wa[3], Pp[3];
#pragma unroll
        for (int t = 0; t < 3; ++t) {
          Pp[t] = ETA_LD(t, NF + X_P);
          if (EXT) Pp[t] += ETA_LD(t, F_PI + 10);      // P + Pi (A28)
          const R w = ETA_LD(t, 0) + Pp[t];
          wq[t] = w * g[t]; wa[t] = w * ua[t];
        }
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
          R q[3], f[3];
          const int o_t = F_PI + mu, o_a = F_PI + c_pidx[3][mu];
#pragma unroll
          for (int t = 0; t < 3; ++t) {
            const R umu = mu == 0 ? g[t] : ETA_LD(t, mu);
            R tq = wq[t] * umu - (mu == 0 ? Pp[t] : R(0));
            R tfl = wa[t] * umu + (mu == 3 ? Pp[t] : R(0));
            if (USE_PI) { tq += ETA_LD(t, o_t); tfl += ETA_LD(t, o_a); }
            q[t] = tq; f[t] = tfl;
          }
          R QLk, FLk, Hk, QL1, QR1, FL1, FR1;
          priv.get(mu, QLk, FLk, Hk);
          lr(q[0], q[1], q[2], th2, QL1, QR1);
          lr(f[0], f[1], f[2], th2, FL1, FR1);
          const R Hn = face2(QLk, FLk, QR1, FR1, cface);
          S[mu] = -(Hn - Hk) * sc_T;
          priv.put(mu, QL1, FL1, Hn);
        }
      }
      if (USE_PI) {
        R* slot = &sS[tid];
        // planes p-1 and p of the next trip's two fields are loaded one trip ahead (they come from L2 more often than not)
        R nxt[2][2] = {{ETA_LD(1, F_PI), ETA_LD(1, F_PI + 1)}, {ETA_LD(2, F_PI), ETA_LD(2, F_PI + 1)}};
#pragma unroll 1
        for (int t = 0; t < NTRIP; ++t) {
          const int fa = F_PI + 2 * t;
          R QLa, FLa, Ha, QLb, FLb, Hb;
          priv.get(fa, QLa, FLa, Ha);
          priv.get(fa + 1, QLb, FLb, Hb);
          R qa[3], fa_[3], qb[3], fb[3];
          const R cur[2][2] = {{nxt[0][0], nxt[0][1]}, {nxt[1][0], nxt[1][1]}};
          if (t < NTRIP - 1) {
            nxt[0][0] = ETA_LD(1, fa + 2); nxt[0][1] = ETA_LD(1, fa + 3);
            nxt[1][0] = ETA_LD(2, fa + 2); nxt[1][1] = ETA_LD(2, fa + 3);
          }
#pragma unroll
          for (int s = 0; s < 3; ++s) {
            const R va = s == 0 ? ETA_LD(0, fa) : cur[s - 1][0], vb = s == 0 ? ETA_LD(0, fa + 1) : cur[s - 1][1];
            qa[s] = g[s] * va; fa_[s] = ua[s] * va;
            qb[s] = g[s] * vb; fb[s] = ua[s] * vb;
          }
          R QL1, QR1, FL1, FR1;
          lr(qa[0], qa[1], qa[2], th2, QL1, QR1);
          lr(fa_[0], fa_[1], fa_[2], th2, FL1, FR1);
          const R Hna = face2(QLa, FLa, QR1, FR1, cface);
          priv.put(fa, QL1, FL1, Hna);
          lr(qb[0], qb[1], qb[2], th2, QL1, QR1);
          lr(fb[0], fb[1], fb[2], th2, FL1, FR1);
          const R Hnb = face2(QLb, FLb, QR1, FR1, cface);
          priv.put(fa + 1, QL1, FL1, Hnb);
          slot[0] = -(Hna - Ha) * sc_pi;
          slot[MT_NTHR] = -(Hnb - Hb) * sc_pi;
          slot += 2 * MT_NTHR;
        }
      }
      tm_wait_st();
#undef ETA_LD
    }
    if (!centre) {
      if (ETILE) { __syncthreads(); fill_tile(bmap(p - 1, a.nz, a.bc[2])); }
      continue;
    }

    // ---- x and y flux differences of cell k (five-point stars inside plane k) ---------------------------------------
    const R* __restrict__ plane = in + (long long)bmap(k, a.nz, a.bc[2]) * a.sz;
    R cfl0, cfl1;
    if (TILE) {
      if (!ETILE) {
        asm volatile("cp.async.wait_all;" ::: "memory");
        __syncthreads();                                   // tile(k) complete and visible
      }
      constexpr int OXT = NF * MT_FST;
      const R* __restrict__ pp[5];
#pragma unroll
      for (int t = 0; t < 5; ++t) pp[t] = town + (t - 2);
      axis_flux<R, USE_PI, 0, false, OXT, MT_FST, EXT, MT_NTHR>(a, pp, th2, tf, S, &sS[tid], cfl0);
#pragma unroll
      for (int t = 0; t < 5; ++t) pp[t] = town + (t - 2) * MT_SX;
      axis_flux<R, USE_PI, 1, false, OXT, MT_FST, EXT, MT_NTHR>(a, pp, th2, tf, S, &sS[tid], cfl1);
    } else {
      const R* __restrict__ pp[5];
#pragma unroll
      for (int t = 0; t < 5; ++t) pp[t] = plane + offx[t];
      axis_flux<R, USE_PI, 0, false, OX, FS, EXT, MT_NTHR>(a, pp, th2, tf, S, &sS[tid], cfl0);
#pragma unroll
      for (int t = 0; t < 5; ++t) pp[t] = plane + offy[t];
      axis_flux<R, USE_PI, 1, false, OX, FS, EXT, MT_NTHR>(a, pp, th2, tf, S, &sS[tid], cfl1);
    }
    if (USE_PI) {
#pragma unroll
      for (int m = 0; m < NPI; ++m) S[4 + m] = sS[m * MT_NTHR + tid];
    }

    // ---- cell-centre state, velocity gradients ------------------------------------------------------------------------
    Cell<R> cc, cn_;
    R grad[4][4];
#pragma unroll
    for (int m = 0; m < 4; ++m)
#pragma unroll
      for (int n = 0; n < 4; ++n) grad[m][n] = R(0);
    const R sc_x = R(0.5) * a.scale[0], sc_y = R(0.5) * a.scale[1], sc_n = R(0.5) * a.scale[2];
    // operands of the stage tail that come from global memory (state n / history / u*^tau at the cell, u~ of planes k+-1):
    // issued here, ahead of the tile barrier and the refill, so that their latency runs behind both
    const long long c = (long long)k * a.sz + col;
    const long long cg = (long long)k * a.ny * a.gp + cg0;
    if (MODE == 2) {
      const R* __restrict__ sn = a.sn + c;
      cn_.e = LD1(sn);
      cn_.u[1] = LD1(sn + sf); cn_.u[2] = LD1(sn + 2 * sf); cn_.u[3] = LD1(sn + 3 * sf);
      cn_.u[0] = LD1(sn + OX + X_G * FS);
      cn_.P = LD1(sn + OX + X_P * FS);
#pragma unroll
      for (int m = 0; m < 10; ++m) cn_.pi[m] = VISC ? LD1(sn + (F_PI + m) * FS) : R(0);
      cn_.Pi = EXT ? LD1(sn + (F_PI + 10) * FS) : R(0); cn_.nb = EXT ? LD1(sn + (F_PI + 11) * FS) : R(0);
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

    if (USE_PI) {      // eta_s row: planes k-1 and k+1 of the own column
      const R* __restrict__ zm = in + (long long)bmap(k - 1, a.nz, a.bc[2]) * a.sz + col;
      grad[3][0] = (q1[OX + X_G * FS] - zm[OX + X_G * FS]) * sc_n;
      grad[3][1] = (q1[sf] - zm[sf]) * sc_n;
      grad[3][2] = (q1[2 * sf] - zm[2 * sf]) * sc_n;
      grad[3][3] = (q1[3 * sf] - zm[3 * sf]) * sc_n;
    }
    if (TILE) {
      constexpr int OXT = NF * MT_FST;
      cc.e = town[0];
      cc.u[1] = town[MT_FST]; cc.u[2] = town[2 * MT_FST]; cc.u[3] = town[3 * MT_FST];
      cc.u[0] = town[OXT + X_G * MT_FST];
      cc.P = town[OXT + X_P * MT_FST];
#pragma unroll
      for (int m = 0; m < 10; ++m) cc.pi[m] = USE_PI ? town[(F_PI + m) * MT_FST] : R(0);
      cc.Pi = EXT ? town[(F_PI + 10) * MT_FST] : R(0); cc.nb = EXT ? town[(F_PI + 11) * MT_FST] : R(0);
      if (USE_PI) {
        grad[1][0] = (town[OXT + X_G * MT_FST + 1] - town[OXT + X_G * MT_FST - 1]) * sc_x;
        grad[2][0] = (town[OXT + X_G * MT_FST + MT_SX] - town[OXT + X_G * MT_FST - MT_SX]) * sc_y;
#pragma unroll
        for (int n = 1; n < 4; ++n) {
          grad[1][n] = (town[n * MT_FST + 1] - town[n * MT_FST - 1]) * sc_x;
          grad[2][n] = (town[n * MT_FST + MT_SX] - town[n * MT_FST - MT_SX]) * sc_y;
        }
      }
      __syncthreads();                                     // every warp is done with tile(k): refill it for plane k+1,
      if (ETILE) { if (p + 1 <= kc1 + 1) fill_tile(bmap(p - 1, a.nz, a.bc[2])); }
      else if (k + 1 < kc1) fill_tile(k + 1);              // behind the stage tail below and the next eta_s step
    } else {
      const R* __restrict__ pc = plane + col;
      cc.e = pc[0];
      cc.u[1] = pc[sf]; cc.u[2] = pc[2 * sf]; cc.u[3] = pc[3 * sf];
      cc.u[0] = pc[OX + X_G * FS];
      cc.P = pc[OX + X_P * FS];
#pragma unroll
      for (int m = 0; m < 10; ++m) cc.pi[m] = USE_PI ? pc[(F_PI + m) * FS] : R(0);
      cc.Pi = EXT ? pc[(F_PI + 10) * FS] : R(0); cc.nb = EXT ? pc[(F_PI + 11) * FS] : R(0);
      if (USE_PI) {
#pragma unroll
        for (int ax = 0; ax < 2; ++ax) {
          const R* __restrict__ qm = ax == 0 ? plane + offx[1] : plane + offy[1];
          const R* __restrict__ qp = ax == 0 ? plane + offx[3] : plane + offy[3];
          const R sc = ax == 0 ? sc_x : sc_y;
          grad[ax + 1][0] = (qp[OX + X_G * FS] - qm[OX + X_G * FS]) * sc;
          grad[ax + 1][1] = (qp[sf] - qm[sf]) * sc;
          grad[ax + 1][2] = (qp[2 * sf] - qm[2 * sf]) * sc;
          grad[ax + 1][3] = (qp[3 * sf] - qm[3 * sf]) * sc;
        }
      }
    }
    // ---- sources, stage update, root-find, limiter (hydro_stage_update.cuh) -----------------------------------------
    unsigned flags = 0;
    Cell<R> nw;
    R cs2_new;
    stage_update<R, VISC, MODE, EXT>(a, S, cc, cn_, grad, up3, gst, nw, cs2_new, flags, tf);

    if (active) {
      R* __restrict__ out = a.out + c;
      R cx, cy, cn;
      signal_speeds3(nw.u[0], nw.u[1], nw.u[2], nw.u[3], cs2_new, cx, cy, cn);
#define ST1(ptr, v) do { if (L2H) stg_hint((ptr), (v), pol_once); else *(ptr) = (v); } while (0)
      ST1(out, nw.e); ST1(out + sf, nw.u[1]); ST1(out + 2 * sf, nw.u[2]); ST1(out + 3 * sf, nw.u[3]);
      if (VISC) {
#pragma unroll
        for (int m = 0; m < 10; ++m) ST1(out + (F_PI + m) * FS, nw.pi[m]);
        if (EXT) { ST1(out + (F_PI + 10) * FS, nw.Pi); ST1(out + (F_PI + 11) * FS, nw.nb); }
        if (MODE == 1) a.gstar[cg] = gst;
      }
      ST1(out + OX + X_P * FS, nw.P); ST1(out + OX + X_G * FS, nw.u[0]);
      ST1(out + OX + X_CX * FS, cx); ST1(out + OX + X_CY * FS, cy); ST1(out + OX + X_CN * FS, cn);
#undef ST1
      if (MODE == 1) { cflm0 = max_(cflm0, cfl0); cflm1 = max_(cflm1, cfl1); cflm2 = max_(cflm2, cfl2); }
      else emax = max_(emax, nw.e);
    } else {
      flags = 0;
    }
    count_flags(a.diag, flags);
  }

  // the tensor memory goes back (the warp that allocated it frees it; every thread has waited on its accesses)
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (row == 0) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(s_tmem), "r"((unsigned)Priv::ALLOC_COLS)
                 : "memory");
  }

  // ---- reductions (row a10): one atomic per warp per block ------------------------------------------------------------
  if (MODE == 1) {
    const double r0 = warp_max((double)cflm0), r1 = warp_max((double)cflm1), r2 = warp_max((double)cflm2);
    if (lane == 0) {
      atomic_max_nonneg(&a.diag->cfl[a.slot][0], r0);
      atomic_max_nonneg(&a.diag->cfl[a.slot][1], r1);
      atomic_max_nonneg(&a.diag->cfl[a.slot][2], r2);
    }
  } else {
    const double r = warp_max((double)emax);
    if (lane == 0) atomic_max_nonneg(&a.diag->emax[a.slot], r);
  }
  if (blockIdx.x == 0 && blockIdx.y == 0 && blockIdx.z == 0 && tid == 0) {
    if (MODE == 1) a.diag->emax[a.slot] = 0ull;
    else { a.diag->cfl[a.slot ^ 1][0] = 0ull; a.diag->cfl[a.slot ^ 1][1] = 0ull; a.diag->cfl[a.slot ^ 1][2] = 0ull; }
  }
}

// planes per chunk: whole waves of the resident blocks, against the two pipeline warm-up planes of a chunk
inline int march_chunk(int nx, int ny, int nz, int nsm, int blocks_per_sm) {
  const long long tiles = (long long)((nx + 31) / 32) * ((ny + MTY - 1) / MTY);
  const long long slots = (long long)(blocks_per_sm * 8 / MTY > 0 ? blocks_per_sm * 8 / MTY : 1) * nsm;
  double best = -1.0;
  int best_chunk = nz;
  for (int nchunk = 1; nchunk <= nz; ++nchunk) {
    const int chunk = (nz + nchunk - 1) / nchunk;
    const long long blocks = tiles * ((nz + chunk - 1) / chunk);
    const long long waves = (blocks + slots - 1) / slots;
    const double eff = (double)blocks / (double)(waves * slots) * (double)chunk / ((double)chunk + 0.6);
    if (eff > best * 1.0001) { best = eff; best_chunk = chunk; }
  }
  return best_chunk;
}

template <typename R, bool VISC, int MODE, bool EXT = false>
cudaError_t launch_stage_march(const StageArgs<R>& a, int chunk, cudaStream_t stream) {
  constexpr bool TILE = CLV_MARCH_TILE != 0;
  constexpr int NFT = (VISC ? (EXT ? 16 : 14) : 4) + X_COUNT;
  const size_t smem = TILE ? (size_t)NFT * MT_FST * sizeof(R) : 0;
  static bool configured = false;
  if (TILE && !configured) {
    cudaError_t e = cudaFuncSetAttribute(stage_march_kernel<R, VISC, MODE, TILE, EXT>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  dim3 block(32, MTY, 1);
  dim3 grid((a.nx + 31) / 32, (a.ny + MTY - 1) / MTY, (a.nz + chunk - 1) / chunk);
  stage_march_kernel<R, VISC, MODE, TILE, EXT><<<grid, block, smem, stream>>>(a, chunk);
  return cudaGetLastError();
}

}  // namespace clv
