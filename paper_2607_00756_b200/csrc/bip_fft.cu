// Fused slice step of the parent columns for power-of-two grids (plumbing of bip_build_S2 / ADVANCETO / PEELTO):
//
//     S  <-  post . F^-1[ Pspec . F[ pre . S ] ]          (eq. 2, eq. 6, eq. 12; pre / post in {1, T_j, conj T_j})
//
// in THREE passes over the column instead of the eleven of the cuFFT route (load/convert, 2 x 2 cuFFT passes, spectrum
// multiply, store/convert, each reading and writing the whole column):
//
//   pass 1  rows:     load S[y][.] (x pre),  forward FFT along x in shared memory,           store      k_ms_rows<LN, fwd>
//   pass 2  columns:  load a tile of columns, forward FFT along y, x P(q) / G, inverse FFT along y, store   k_ms_cols<LN, LC>
//   pass 3  rows:     load, inverse FFT along x, (x post), store                                         k_ms_rows<LN, inv>
//
// i.e. 48 bytes of HBM traffic per pixel and slice step -- and 32 when slice steps follow one another on the same columns
// (a build, a cursor move over several slices, the exit multislice of Algorithm 3): pass 3 of step j and pass 1 of step
// j + 1 work on the same rows and run as ONE kernel (k_ms_rows_both; fft_slice_op leaves pass 3 owing, the next step or
// fft_flush runs it).  The forward transforms are decimation-in-frequency (natural order in, digit-reversed order out),
// the inverse ones decimation-in-time (digit-reversed in, natural out), so no reordering pass exists at all: the
// propagator -- separable, P(q) / G = Ey[q_y] Ex[q_x] -- is stored as two 1-D tables in the digit-reversed order of their axis.
// Butterflies are radix-8 in registers (radix 4 / 2 for the last stage), fp32 with round-to-nearest throughout.
// Every CONSTANT the data is multiplied by -- twiddles, sqrt(1/2), the propagator -- is held as a double-float pair
// hi + lo (hi = fp32(c), lo = fp32(c - hi)) and applied with the small terms first inside one FMA chain.  A twiddle
// rounded to fp32 alone has |w|^2 - 1 ~ +-6e-8, the same for every element that meets it, and those do NOT average out:
// measured, a plain-fp32 version of these kernels lost 3.5e-7 of the column norm^2 per slice (the same systematic loss
// cuFFT's C2C shows), i.e. 3.5e-6 of the summed intensity at 10 slices against a bound of 1e-6.  With double-float
// constants only the data roundings remain, and those are unbiased (tests/test_gpu_plumbing.py measures the drift of
// this route, of the fp64 cuFFT route and of plain cuFFT C2C).
#include <cmath>

#include "bip_internal.h"
#include "bip_fft.cuh"

namespace bip {

namespace {

using namespace fftdev;

// ---------------------------------------------------------------------------------------------------------------------
// Compile-time-sized transforms.  Everything about a stage -- its radix, the stride of its butterflies, the shared-memory
// offsets of its eight elements -- is a template constant, so the inner loops are loads, floating-point work and stores
// with immediate offsets (the run-time-sized version spent 45 % of its instructions on index arithmetic and a third of its
// shared-memory wavefronts on bank conflicts; profiles/r02_fft_ncu.md).
//
// Shared-memory layout of a line of N = 2^LN elements: element i lives at slot  i ^ g(i),  g = XOR of a 4-bit mask per set
// bit 4, 5, 6 of i (masks by LN mod 3, found by exhaustive search).  With it the 16 lanes of a half-warp hit 16 different
// 8-byte bank pairs in EVERY access pattern of the transform: contiguous runs (copies, long-stride stages), the
// short-stride radix-8 stages and the final radix-8 / 4 / 2 stage.  The map is XOR-linear, so the slot of element
// i0 + (k << LSUB) is slot(i0) ^ const_k.  A tile of columns adds a per-line key (c & 15) so that the same holds when the
// lanes of a warp run over 16 lines at one position.
// ---------------------------------------------------------------------------------------------------------------------
constexpr int NT = 256;                    // threads per block
constexpr int TILE_EL = 8192;              // elements per block tile (64 KB)

template <int LN> struct Swz {
  static constexpr uint32_t M4 = (LN % 3 == 1) ? 3u : 1u;
  static constexpr uint32_t M5 = (LN % 3 == 0) ? 2u : (LN % 3 == 1) ? 4u : 6u;
  static constexpr uint32_t M6 = (LN % 3 == 0) ? 12u : 8u;
};
template <int LN> __host__ __device__ constexpr uint32_t swz_g(uint32_t i) {
  return (LN > 4 ? ((i >> 4) & 1u) * Swz<LN>::M4 : 0u) ^ (LN > 5 ? ((i >> 5) & 1u) * Swz<LN>::M5 : 0u) ^
         (LN > 6 ? ((i >> 6) & 1u) * Swz<LN>::M6 : 0u);
}
template <int LN> __host__ __device__ constexpr uint32_t slot(uint32_t i) { return i ^ swz_g<LN>(i); }
// XOR key (4 bits) of line c of a column tile 2^lc columns wide.  16 or more columns: c & 15 -- the 16 lanes of a half-warp
// that run over 16 columns at one row hit 16 different slots.  Narrower tiles (long columns): a half-warp covers 2^lc
// columns x 2^(4-lc) consecutive rows (copies) or consecutive final-stage butterflies (the fused stage), whose row bits sit
// at the bottom resp. just above the butterfly's own bits; c is therefore XORed in twice, shifted above the row bits and
// unshifted, which keeps both patterns conflict-free.  A line shorter than 16 elements keeps the key inside the line.
template <int LN> __host__ __device__ constexpr uint32_t key_mask() { return LN >= 4 ? 15u : (1u << LN) - 1u; }
template <int LN> __host__ __device__ constexpr uint32_t line_key(uint32_t c, int lc) {
  return (lc >= 4 ? c : ((c << (4 - lc)) | (c & ((1u << (4 - lc)) - 1u)))) & key_mask<LN>();
}

// the tile: dynamic shared memory, always addressed as sm + offset so that every access is an LDS / STS with an
// immediate offset (its start is 1024-byte aligned: the bank of an offset is the bank of the address)
extern __shared__ __align__(1024) char sm[];
constexpr size_t tile_smem_bytes() { return (size_t)TILE_EL * sizeof(float2); }
__device__ __forceinline__ float2 lds2(uint32_t off) { return *reinterpret_cast<const float2*>(sm + off); }
__device__ __forceinline__ void sts2(uint32_t off, float2 v) { *reinterpret_cast<float2*>(sm + off) = v; }
// asynchronous 8-byte copy global -> shared (LDGSTS): no register staging, as many in flight as the loop issues
__device__ __forceinline__ void cp_async8(uint32_t off, const float2* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(sm + off)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory"); }

// radix-R butterfly with its twiddles: forward (DIF) butterfly then w_L^(j m); inverse (DIT) conj twiddle then butterfly
template <int R, bool INV, bool TW>
__device__ __forceinline__ void bfly(float2 (&x)[8], const float4 (&w)[8]) {
  if (INV && TW) {
#pragma unroll
    for (int m = 1; m < R; ++m) x[m] = cmulc_dd(x[m], w[m]);
  }
  dft_small<R, INV>(x);
  if (!INV && TW) {
#pragma unroll
    for (int m = 1; m < R; ++m) x[m] = cmul_dd(x[m], w[m]);
  }
}

// byte offsets of element k of a butterfly relative to element 0: an XOR part (the swizzle bits, and the k field itself
// when it lies inside the low index bits) and an ADD part (the k field above them) -- both compile-time constants
template <int LN, int LSUB> __host__ __device__ constexpr uint32_t xk(int k) {
  return LSUB >= 4 ? 8u * swz_g<LN>((uint32_t)k << LSUB) : 8u * slot<LN>((uint32_t)k << LSUB);
}
template <int LN, int LSUB> __host__ __device__ constexpr uint32_t ak(int k) { return LSUB >= 4 ? 8u * ((uint32_t)k << LSUB) : 0u; }

enum { IO_SMEM = 0, IO_GLOBAL = 1 };

// One radix-R stage on block length 2^LL of n_lines transforms of length 2^LN (lines 8 N bytes apart in the tile).
// Thread <-> butterfly position v, consecutive lanes = consecutive v; the thread keeps the twiddles of its position in
// registers and loops over the lines with them.  SRC / DST = IO_GLOBAL (only for the stage on the whole line, LL == LN):
// the elements are read from / written to global memory in natural order, line l at g + l N, times
// T[(line index mod ny) N + i] (tmode 1) or its conjugate (tmode 2) -- the row passes touch global memory directly in the
// stage whose butterflies stride over the whole row (unit stride across the lanes).  The T values of a line are requested
// before its butterfly, so that their latency hides behind it.  KEYED: line c carries the XOR key 8 (c & 15) (column tiles).
template <int LN, int LL, int R, bool INV, int SRC, int DST, bool KEYED>
__device__ __forceinline__ void stage(int n_lines, int lc, const float4* __restrict__ root, int tid, float2* __restrict__ g = nullptr,
                                      const float2* __restrict__ T = nullptr, int tmode = 0, int64_t line0_global = 0, int ny_mask = 0) {
  constexpr int LR = R == 8 ? 3 : R == 4 ? 2 : 1;
  constexpr int LSUB = LL - LR, SUB = 1 << LSUB, NV = 1 << (LN - LR), N = 1 << LN;
  constexpr int NVT = NV < NT ? NV : NT, LSTEP = NT / NVT;
  constexpr bool TW = R == 8 && LSUB > 0;
  static_assert((SRC == IO_SMEM && DST == IO_SMEM) || LL == LN, "global access only in the stage on the whole line");
  const float4* tw = root + tw_stage_off(LN, LL);
  const int l0 = tid / NVT;
  for (int v = tid % NVT; v < NV; v += NVT) {
    const int blk = v >> LSUB, j = v & (SUB - 1);
    const uint32_t i0 = ((uint32_t)blk << LL) + (uint32_t)j;
    float4 w[8];
    if (TW) {
#pragma unroll
      for (int m = 1; m < R; ++m) w[m] = __ldg(tw + ((m - 1) << LSUB) + j);
    }
    const uint32_t p0 = 8u * slot<LN>(i0);
    for (int line = l0; line < n_lines; line += LSTEP) {
      const uint32_t q = ((uint32_t)line * (8u * N) + p0) ^ (KEYED ? 8u * line_key<LN>((uint32_t)line, lc) : 0u);
      float2 x[8], t[8];
      if (SRC == IO_GLOBAL || DST == IO_GLOBAL) {
        if (tmode) {
          const float2* tp = T + (((line0_global + line) & ny_mask) << LN) + i0;
#pragma unroll
          for (int k = 0; k < R; ++k) t[k] = __ldg(tp + (k << LSUB));
        }
      }
      if (SRC == IO_GLOBAL) {
        const float2* gp = g + (int64_t)line * N + i0;
#pragma unroll
        for (int k = 0; k < R; ++k) x[k] = gp[k << LSUB];
        if (tmode) {
#pragma unroll
          for (int k = 0; k < R; ++k) x[k] = cmulf(x[k], make_float2(t[k].x, tmode == 2 ? -t[k].y : t[k].y));
        }
      } else {
#pragma unroll
        for (int k = 0; k < R; ++k) x[k] = lds2((q ^ xk<LN, LSUB>(k)) + ak<LN, LSUB>(k));
      }
      bfly<R, INV, TW>(x, w);
      if (DST == IO_GLOBAL) {
        float2* gp = g + (int64_t)line * N + i0;
        if (tmode) {
#pragma unroll
          for (int k = 0; k < R; ++k) x[k] = cmulf(x[k], make_float2(t[k].x, tmode == 2 ? -t[k].y : t[k].y));
        }
#pragma unroll
        for (int k = 0; k < R; ++k) gp[k << LSUB] = x[k];
      } else {
#pragma unroll
        for (int k = 0; k < R; ++k) sts2((q ^ xk<LN, LSUB>(k)) + ak<LN, LSUB>(k), x[k]);
      }
    }
  }
}

// radix sequence of a length-2^LN transform: LN / 3 radix-8 stages on L = N, N/8, ..., then radix 4 or 2 on what is left
template <int LN> struct Seq {
  static constexpr int N8 = LN / 3, REM = LN % 3, NS = N8 + (REM ? 1 : 0);
  static constexpr int RL = REM == 2 ? 4 : REM == 1 ? 2 : 8;         // radix of the last forward stage
  static constexpr int LRL = REM ? REM : 3;                         // its block length (log2): L == R
};

// forward stages S .. LAST (0-based, inclusive) of every line of the tile, a block barrier after each
template <int LN, bool KEYED, int S, int LAST>
__device__ __forceinline__ void fwd_stages(int n_lines, int lc, const float4* __restrict__ root, int tid) {
  if constexpr (S <= LAST) {
    if constexpr (S < Seq<LN>::N8) stage<LN, LN - 3 * S, 8, false, IO_SMEM, IO_SMEM, KEYED>(n_lines, lc, root, tid);
    else stage<LN, Seq<LN>::LRL, Seq<LN>::RL, false, IO_SMEM, IO_SMEM, KEYED>(n_lines, lc, root, tid);
    __syncthreads();
    fwd_stages<LN, KEYED, S + 1, LAST>(n_lines, lc, root, tid);
  }
}
// inverse stages S, S - 1, ..., FIRST (the forward stages backwards)
template <int LN, bool KEYED, int S, int FIRST>
__device__ __forceinline__ void inv_stages(int n_lines, int lc, const float4* __restrict__ root, int tid) {
  if constexpr (S >= FIRST) {
    if constexpr (S < Seq<LN>::N8) stage<LN, LN - 3 * S, 8, true, IO_SMEM, IO_SMEM, KEYED>(n_lines, lc, root, tid);
    else stage<LN, Seq<LN>::LRL, Seq<LN>::RL, true, IO_SMEM, IO_SMEM, KEYED>(n_lines, lc, root, tid);
    __syncthreads();
    inv_stages<LN, KEYED, S - 1, FIRST>(n_lines, lc, root, tid);
  }
}

// First row of a block's tile.  Row tiles are handed out column-interleaved -- consecutive blocks take the SAME rows of
// consecutive columns -- so that the blocks resident at one time read the same few rows of T_j (at 2048^2 a whole T_j slice,
// 32 MB, does not survive in L2 beside the streaming columns: 60 % of its reads went to DRAM in column-major order).  Grids with
// fewer rows than a tile keep the flat order (a tile then spans several columns).
template <int LN>
__device__ __forceinline__ int64_t tile_line0(int ny_mask) {
  constexpr int LINES = TILE_EL >> LN;
  const int ny = ny_mask + 1;
  if (LINES > ny) return (int64_t)blockIdx.x * LINES;
  const unsigned tiles_per_col = (unsigned)ny / LINES, n_cols = gridDim.x / tiles_per_col;
  const unsigned c = blockIdx.x % n_cols, r = blockIdx.x / n_cols;
  return (int64_t)c * ny + (int64_t)r * LINES;
}

// Passes 1 and 3: a block takes LINES = TILE_EL / nx consecutive rows of the flat [n_cols * ny][nx] array (rows of
// consecutive columns are consecutive in memory).  Forward: the first stage reads global memory (x pre, coalesced: its
// butterflies stride over the whole row) and the digit-reversed result leaves through a coalesced copy; inverse: an
// asynchronous coalesced copy comes first and the last stage (x post) writes global memory.
// tmode: 0 none, 1 multiply by T, 2 by conj T.
template <int LN, bool INV>
__global__ void __launch_bounds__(NT, 3) k_ms_rows(float2* __restrict__ S, const float2* __restrict__ T, int tmode, int64_t n_lines_total,
                                                  int ny_mask, const float4* __restrict__ rootx) {
  constexpr int N = 1 << LN, LINES = TILE_EL / N, NS = Seq<LN>::NS;
  const int tid = threadIdx.x;
  const int64_t line0 = tile_line0<LN>(ny_mask);
  const int n_lines = (int)min((int64_t)LINES, n_lines_total - line0);
  float2* g = S + line0 * N;
  const int n_el = n_lines << LN;
  // flat copy: element e of the tile at slot e ^ g(e); g depends on bits 4-6 of e only, i.e. on tid (NT is a multiple of 128)
  const uint32_t c0 = 8u * ((uint32_t)tid ^ swz_g<LN>((uint32_t)tid));
  if (!INV) {
    stage<LN, LN, 8, false, IO_GLOBAL, IO_SMEM, false>(n_lines, 0, rootx, tid, g, T, tmode, line0, ny_mask);
    __syncthreads();
    fwd_stages<LN, false, 1, NS - 1>(n_lines, 0, rootx, tid);
#pragma unroll 8
    for (int e = tid; e < n_el; e += NT) g[e] = lds2(c0 + 8u * (uint32_t)(e - tid));
  } else {
#pragma unroll 8
    for (int e = tid; e < n_el; e += NT) cp_async8(c0 + 8u * (uint32_t)(e - tid), g + e);
    cp_async_wait_all();
    __syncthreads();
    inv_stages<LN, false, NS - 1, 1>(n_lines, 0, rootx, tid);
    stage<LN, LN, 8, true, IO_SMEM, IO_GLOBAL, false>(n_lines, 0, rootx, tid, g, T, tmode, line0, ny_mask);
  }
}

// The stage on the whole line of the inverse transform of one slice step and of the forward transform of the NEXT one, in
// registers: conj twiddle, inverse butterfly, x post (of this step) x pre (of the next), forward butterfly, twiddle -- both
// butterflies work on the same eight elements i0 + k N/8.
template <int LN>
__device__ __forceinline__ void stage_both(int n_lines, const float4* __restrict__ root, int tid, const float2* __restrict__ Ta, int mode_a,
                                           const float2* __restrict__ Tb, int mode_b, int64_t line0_global, int ny_mask) {
  constexpr int LSUB = LN - 3, SUB = 1 << LSUB, NV = 1 << LSUB, N = 1 << LN;
  constexpr int NVT = NV < NT ? NV : NT, LSTEP = NT / NVT;
  constexpr bool TW = LSUB > 0;
  const float4* tw = root + tw_stage_off(LN, LN);
  const int l0 = tid / NVT;
  for (int v = tid % NVT; v < NV; v += NVT) {
    const uint32_t i0 = (uint32_t)v;
    float4 w[8];
    if (TW) {
#pragma unroll
      for (int m = 1; m < 8; ++m) w[m] = __ldg(tw + ((m - 1) << LSUB) + v);
    }
    const uint32_t p0 = 8u * slot<LN>(i0);
    for (int line = l0; line < n_lines; line += LSTEP) {
      const uint32_t q = (uint32_t)line * (8u * N) + p0;
      const int64_t trow = (((line0_global + line) & ny_mask) << LN) + i0;
      float2 x[8], t[8];
      if (mode_a) {
#pragma unroll
        for (int k = 0; k < 8; ++k) { t[k] = __ldg(Ta + trow + (k << LSUB)); if (mode_a == 2) t[k].y = -t[k].y; }
      }
      if (mode_b) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          float2 u = __ldg(Tb + trow + (k << LSUB));
          if (mode_b == 2) u.y = -u.y;
          t[k] = mode_a ? cmulf(t[k], u) : u;
        }
      }
#pragma unroll
      for (int k = 0; k < 8; ++k) x[k] = lds2((q ^ xk<LN, LSUB>(k)) + ak<LN, LSUB>(k));
      bfly<8, true, TW>(x, w);
      if (mode_a || mode_b) {
#pragma unroll
        for (int k = 0; k < 8; ++k) x[k] = cmulf(x[k], t[k]);
      }
      bfly<8, false, TW>(x, w);
#pragma unroll
      for (int k = 0; k < 8; ++k) sts2((q ^ xk<LN, LSUB>(k)) + ak<LN, LSUB>(k), x[k]);
    }
  }
  (void)SUB;
}

// Pass 3 of one slice step and pass 1 of the next on the same rows in one kernel (consecutive steps of a build, of a cursor
// move over several slices, of the exit multislice of Algorithm 3): k chained steps take 2 k + 1 passes instead of 3 k.
template <int LN>
__global__ void __launch_bounds__(NT, 3) k_ms_rows_both(float2* __restrict__ S, const float2* __restrict__ Ta, int mode_a, const float2* __restrict__ Tb,
                                                       int mode_b, int64_t n_lines_total, int ny_mask, const float4* __restrict__ rootx) {
  constexpr int N = 1 << LN, LINES = TILE_EL / N, NS = Seq<LN>::NS;
  const int tid = threadIdx.x;
  const int64_t line0 = tile_line0<LN>(ny_mask);
  const int n_lines = (int)min((int64_t)LINES, n_lines_total - line0);
  float2* g = S + line0 * N;
  const int n_el = n_lines << LN;
  const uint32_t c0 = 8u * ((uint32_t)tid ^ swz_g<LN>((uint32_t)tid));
#pragma unroll 8
  for (int e = tid; e < n_el; e += NT) cp_async8(c0 + 8u * (uint32_t)(e - tid), g + e);
  cp_async_wait_all();
  __syncthreads();
  inv_stages<LN, false, NS - 1, 1>(n_lines, 0, rootx, tid);
  stage_both<LN>(n_lines, rootx, tid, Ta, mode_a, Tb, mode_b, line0, ny_mask);
  __syncthreads();
  fwd_stages<LN, false, 1, NS - 1>(n_lines, 0, rootx, tid);
#pragma unroll 8
  for (int e = tid; e < n_el; e += NT) g[e] = lds2(c0 + 8u * (uint32_t)(e - tid));
}

// slot of row y of column c of a column tile (line c, key c & 15), in bytes
template <int LN> __device__ __forceinline__ uint32_t col_off(uint32_t c, uint32_t y, int lc) {
  return c * (8u << LN) + 8u * (slot<LN>(y) ^ line_key<LN>(c, lc));
}

// Pass 2: a tile of COLS = 2^LC columns (consecutive stored x positions) x ny rows per block.  Asynchronous coalesced copy
// in (lanes run over the columns), forward stages along y, then ONE stage that does the last forward butterfly, the spectrum
// multiply and the first inverse butterfly in registers -- both butterflies work on the same R consecutive elements.  The
// propagator is separable, P(q) / G = Ey[qy] Ex[qx] (eq. 2: the phase is a sum of a qy^2 and a qx^2 term): two 1-D tables in
// the digit-reversed order of their axis, conjugated when conj_p, instead of a G-entry table that falls out of L2 on a
// 2048^2 grid (64 MB, re-read from DRAM by every column: measured 3 x the DRAM reads of the pass).  Inverse stages,
// coalesced copy out.  LCT >= 0: the tile width is the compile-time 2^LCT (TILE_EL / ny columns: every grid with ny nx >= TILE_EL);
// LCT < 0: run-time width 2^lc_rt (small grids).
template <int LN, int LCT>
__global__ void __launch_bounds__(NT, 3) k_ms_cols(float2* __restrict__ S, const float4* __restrict__ Ey, const float4* __restrict__ Ex, int conj_p, int nx,
                                                  int lc_rt, const float4* __restrict__ rooty) {
  constexpr int N = 1 << LN, NS = Seq<LN>::NS, RL = Seq<LN>::RL;
  const int tid = threadIdx.x, lc = LCT >= 0 ? LCT : lc_rt, cols = 1 << lc;
  float2* col = S + (int64_t)blockIdx.y * N * nx + ((int64_t)blockIdx.x << lc);
  const int n_el = N << lc;
  if (cols <= NT) {
    const uint32_t c = (uint32_t)tid & (uint32_t)(cols - 1), yy = (uint32_t)tid >> lc, ystep = (uint32_t)NT >> lc;
    const float2* src = col + (int64_t)yy * nx + c;
#pragma unroll 8
    for (uint32_t y = yy; y < (uint32_t)N; y += ystep, src += (int64_t)ystep * nx) cp_async8(col_off<LN>(c, y, lc), src);
  } else {                                   // more columns than threads (short columns of a small grid)
    for (int i = tid; i < n_el; i += NT) cp_async8(col_off<LN>((uint32_t)i & (uint32_t)(cols - 1), (uint32_t)i >> lc, lc), col + (int64_t)(i >> lc) * nx + (i & (cols - 1)));
  }
  cp_async_wait_all();
  __syncthreads();
  fwd_stages<LN, true, 0, NS - 2>(cols, lc, rooty, tid);
  {
    const float4 w[8] = {};
    const uint32_t n_b = ((uint32_t)N / RL) << lc;                     // butterflies of the tile, lanes over the columns first
    const float4* ex = Ex + ((int64_t)blockIdx.x << lc);
    for (uint32_t u = (uint32_t)tid; u < n_b; u += NT) {
      const uint32_t cc = u & (uint32_t)(cols - 1), b = u >> lc;
      const uint32_t q = col_off<LN>(cc, b * RL, lc);
      const float4 px = __ldg(ex + cc);                                // a thread keeps its column when the tile is narrower than the block
      float4 py[8];
#pragma unroll
      for (int k = 0; k < RL; ++k) py[k] = __ldg(Ey + b * RL + k);
      float2 x[8];
#pragma unroll
      for (int k = 0; k < RL; ++k) x[k] = lds2(q ^ (8u * k));
      bfly<RL, false, false>(x, w);
#pragma unroll
      for (int k = 0; k < RL; ++k) x[k] = conj_p ? cmulc_dd(cmulc_dd(x[k], py[k]), px) : cmul_dd(cmul_dd(x[k], py[k]), px);
      bfly<RL, true, false>(x, w);
#pragma unroll
      for (int k = 0; k < RL; ++k) sts2(q ^ (8u * k), x[k]);
    }
  }
  __syncthreads();
  inv_stages<LN, true, NS - 2, 0>(cols, lc, rooty, tid);
  if (cols <= NT) {
    const uint32_t c = (uint32_t)tid & (uint32_t)(cols - 1), yy = (uint32_t)tid >> lc, ystep = (uint32_t)NT >> lc;
    float2* dst = col + (int64_t)yy * nx + c;
#pragma unroll 8
    for (uint32_t y = yy; y < (uint32_t)N; y += ystep, dst += (int64_t)ystep * nx) *dst = lds2(col_off<LN>(c, y, lc));
  } else {
    for (int i = tid; i < n_el; i += NT) col[(int64_t)(i >> lc) * nx + (i & (cols - 1))] = lds2(col_off<LN>((uint32_t)i & (uint32_t)(cols - 1), (uint32_t)i >> lc, lc));
  }
}

// Detector plane of Algorithm 3 (Alg. 1 lines 6-7): after the row pass (forward along x, stored order),
// forward FFT along y of a tile of columns of every channel field of one scan position and
//     out[rho][ky][kx] += sum_n |F psi_n|^2 / G
// at the TRUE frequency (ky, kx) of the stored position (permy / permx undo the digit reversal).  A block owns the
// (all y, its x tile) outputs of its scan position, so the read-modify-write needs no atomics.
template <int LN>
__global__ void __launch_bounds__(NT, 2) k_ms_cols_detect(const float2* __restrict__ F, int n_ch, float* __restrict__ out, float inv_G, int nx, int lc,
                                                         const float4* __restrict__ rooty, const int32_t* __restrict__ permy,
                                                         const int32_t* __restrict__ permx) {
  constexpr int N = 1 << LN, NS = Seq<LN>::NS;
  const int tid = threadIdx.x, cols = 1 << lc;
  const int64_t G = (int64_t)N * nx;
  const int x0 = blockIdx.x << lc, rho = blockIdx.y;
  float* acc = reinterpret_cast<float*>(sm + (size_t)TILE_EL * sizeof(float2));       // [N * cols], element i of the tile loop
  const int n_el = N << lc;
  for (int i = tid; i < n_el; i += NT) acc[i] = 0.f;
  for (int n = 0; n < n_ch; ++n) {
    const float2* col = F + ((int64_t)rho * n_ch + n) * G + x0;
    __syncthreads();
#pragma unroll 8
    for (int i = tid; i < n_el; i += NT) {
      const uint32_t y = (uint32_t)i >> lc, c = (uint32_t)i & (uint32_t)(cols - 1);
      cp_async8(col_off<LN>(c, y, lc), col + (int64_t)y * nx + c);
    }
    cp_async_wait_all();
    __syncthreads();
    fwd_stages<LN, true, 0, NS - 1>(cols, lc, rooty, tid);
    for (int i = tid; i < n_el; i += NT) {
      const uint32_t y = (uint32_t)i >> lc, c = (uint32_t)i & (uint32_t)(cols - 1);
      const float2 v = lds2(col_off<LN>(c, y, lc));
      acc[i] += v.x * v.x + v.y * v.y;
    }
  }
  float* o = out + (int64_t)rho * G;
  for (int i = tid; i < n_el; i += NT) {
    const int y = i >> lc, c = i & (cols - 1);
    const int64_t k = (int64_t)__ldg(permy + y) * nx + __ldg(permx + x0 + c);
    o[k] += acc[i] * inv_G;
  }
}

// ---- dispatch on the (power-of-two) transform length ----
#define BIP_FFT_SWITCH(ln, CALL)                                                                                        \
  switch (ln) {                                                                                                         \
    case 3: { constexpr int LN_ = 3; CALL; } break;   case 4: { constexpr int LN_ = 4; CALL; } break;                     \
    case 5: { constexpr int LN_ = 5; CALL; } break;   case 6: { constexpr int LN_ = 6; CALL; } break;                     \
    case 7: { constexpr int LN_ = 7; CALL; } break;   case 8: { constexpr int LN_ = 8; CALL; } break;                     \
    case 9: { constexpr int LN_ = 9; CALL; } break;   case 10: { constexpr int LN_ = 10; CALL; } break;                   \
    case 11: { constexpr int LN_ = 11; CALL; } break; case 12: { constexpr int LN_ = 12; CALL; } break;                   \
    default: return fail(ctx, BIP_ERR_UNSUPPORTED, "native FFT: length 2^%d outside 8 .. 4096", ln);                    \
  }

template <int LN> int32_t set_attrs(bip_ctx* ctx) {
  const int bytes = (int)tile_smem_bytes();
  BIP_CUDA(ctx, cudaFuncSetAttribute(k_ms_rows<LN, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  BIP_CUDA(ctx, cudaFuncSetAttribute(k_ms_rows<LN, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  BIP_CUDA(ctx, cudaFuncSetAttribute(k_ms_rows_both<LN>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  BIP_CUDA(ctx, cudaFuncSetAttribute(k_ms_cols<LN, 13 - LN>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  BIP_CUDA(ctx, cudaFuncSetAttribute(k_ms_cols<LN, -1>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  BIP_CUDA(ctx, cudaFuncSetAttribute(k_ms_cols_detect<LN>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes + TILE_EL * (int)sizeof(float)));
  return BIP_OK;
}

template <int LN, bool INV>
void launch_rows(bip_ctx* ctx, float2* S, const float2* T, int tmode, int64_t n_lines_total, int ny) {
  constexpr int LINES = TILE_EL >> LN;
  const int64_t blocks = (n_lines_total + LINES - 1) / LINES;
  k_ms_rows<LN, INV><<<(unsigned)blocks, NT, tile_smem_bytes(), ctx->stream>>>(S, T, tmode, n_lines_total, ny - 1, ctx->fft_rootx);
}

template <int LN>
void launch_rows_both(bip_ctx* ctx, float2* S, const float2* Ta, int mode_a, const float2* Tb, int mode_b, int64_t n_lines_total, int ny) {
  constexpr int LINES = TILE_EL >> LN;
  const int64_t blocks = (n_lines_total + LINES - 1) / LINES;
  k_ms_rows_both<LN><<<(unsigned)blocks, NT, tile_smem_bytes(), ctx->stream>>>(S, Ta, mode_a, Tb, mode_b, n_lines_total, ny - 1, ctx->fft_rootx);
}

}  // namespace

bool fft_supported(const bip_ctx* ctx) {
  return is_pow2(ctx->g.ny) && is_pow2(ctx->g.nx) && ctx->g.ny >= 8 && ctx->g.nx >= 8 && ctx->g.ny <= 4096 && ctx->g.nx <= 4096;
}

int32_t fft_init(bip_ctx* ctx) {
  const int ny = ctx->g.ny, nx = ctx->g.nx;
  const int64_t G = (int64_t)ny * nx;
  auto dd = [](double re, double im) { return dd_pair(re, im); };
  std::vector<float4> ry = make_twiddle_table(ny), rx = make_twiddle_table(nx), Ey(ny), Ex(nx);
  // Fresnel propagator P(q) = exp(-i pi lambda dz |q|^2) / G (eq. 2; no band limit) = Ey[qy] Ex[qx], each factor in the
  // stored (digit-reversed) order of its axis; the 1 / G of the unnormalised transform pair sits in Ey
  for (int py = 0; py < ny; ++py) {
    const int ky = dif_frequency(py, ny), hy = ky < (ny + 1) / 2 ? ky : ky - ny;
    const double qy = hy / ctx->g.ly, ph = -M_PI * ctx->g.lambda * ctx->g.dz * qy * qy;
    Ey[py] = dd(std::cos(ph) / (double)G, std::sin(ph) / (double)G);
  }
  for (int px = 0; px < nx; ++px) {
    const int kx = dif_frequency(px, nx), hx = kx < (nx + 1) / 2 ? kx : kx - nx;
    const double qx = hx / ctx->g.lx, ph = -M_PI * ctx->g.lambda * ctx->g.dz * qx * qx;
    Ex[px] = dd(std::cos(ph), std::sin(ph));
  }
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->fft_rooty, sizeof(float4) * ry.size(), "fft twiddles"));
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->fft_rootx, sizeof(float4) * rx.size(), "fft twiddles"));
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->fft_Ey, sizeof(float4) * ny, "propagator factor along y (digit-reversed order)"));
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->fft_Ex, sizeof(float4) * nx, "propagator factor along x (digit-reversed order)"));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->fft_rooty, ry.data(), sizeof(float4) * ry.size(), cudaMemcpyHostToDevice, ctx->stream));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->fft_rootx, rx.data(), sizeof(float4) * rx.size(), cudaMemcpyHostToDevice, ctx->stream));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->fft_Ey, Ey.data(), sizeof(float4) * ny, cudaMemcpyHostToDevice, ctx->stream));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->fft_Ex, Ex.data(), sizeof(float4) * nx, cudaMemcpyHostToDevice, ctx->stream));
  std::vector<int32_t> py(ny), px(nx);
  for (int i = 0; i < ny; ++i) py[i] = dif_frequency(i, ny);
  for (int i = 0; i < nx; ++i) px[i] = dif_frequency(i, nx);
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->fft_permy, sizeof(int32_t) * ny, "fft permutation"));
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->fft_permx, sizeof(int32_t) * nx, "fft permutation"));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->fft_permy, py.data(), sizeof(int32_t) * ny, cudaMemcpyHostToDevice, ctx->stream));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->fft_permx, px.data(), sizeof(int32_t) * nx, cudaMemcpyHostToDevice, ctx->stream));
  BIP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  // launch shapes: tiles of TILE_EL elements (64 KB): TILE_EL / nx rows per block in the row passes, min(nx, TILE_EL / ny)
  // columns per block in the column pass
  const int lnx = ilog2(nx), lny = ilog2(ny);
  ctx->fft_lines = TILE_EL / nx;
  ctx->fft_cols = std::min(nx, TILE_EL / ny);
  BIP_FFT_SWITCH(lnx, BIP_TRY(set_attrs<LN_>(ctx)));
  if (lny != lnx) BIP_FFT_SWITCH(lny, BIP_TRY(set_attrs<LN_>(ctx)));
  return BIP_OK;
}

// S <- post . F^-1[ P . F[ pre . S ] ] on n_cols columns (modes as in bip_multislice.cu: 0 = 1, 1 = T_j, 2 = conj T_j)
int32_t fft_slice_op(bip_ctx* ctx, float2* S, int n_cols, const float2* Tj, int pre, int conj_p, int post) {
  const int ny = ctx->g.ny, nx = ctx->g.nx;
  const int lnx = ilog2(nx), lny = ilog2(ny), lc = ilog2(ctx->fft_cols);
  const int64_t n_lines = (int64_t)n_cols * ny;
  // the inverse row pass of the previous step on the same columns is still owed (fft_flush): it runs together with this step's
  // forward row pass in one kernel
  FftPending& pd = ctx->fft_pending;
  if (pd.active && pd.S == S && pd.n_cols == n_cols) {
    BIP_FFT_SWITCH(lnx, (launch_rows_both<LN_>(ctx, S, pd.T, pd.post, Tj, pre, n_lines, ny)));
    pd.active = false;
  } else {
    BIP_TRY(fft_flush(ctx));
    BIP_FFT_SWITCH(lnx, (launch_rows<LN_, false>(ctx, S, Tj, pre, n_lines, ny)));
  }
  for (int c0 = 0; c0 < n_cols; c0 += 65535) {                // gridDim.y limit
    const int nc = std::min(65535, n_cols - c0);
    float2* Sc = S + (int64_t)c0 * ny * nx;
    const dim3 grid((unsigned)(nx >> lc), (unsigned)nc);
    if (lc == 13 - lny) {         // the compile-time tile width (every grid with ny nx >= TILE_EL)
      BIP_FFT_SWITCH(lny, (k_ms_cols<LN_, 13 - LN_><<<grid, NT, tile_smem_bytes(), ctx->stream>>>(Sc, ctx->fft_Ey, ctx->fft_Ex, conj_p, nx, lc, ctx->fft_rooty)));
    } else {
      BIP_FFT_SWITCH(lny, (k_ms_cols<LN_, -1><<<grid, NT, tile_smem_bytes(), ctx->stream>>>(Sc, ctx->fft_Ey, ctx->fft_Ex, conj_p, nx, lc, ctx->fft_rooty)));
    }
  }
  BIP_CUDA(ctx, cudaGetLastError());
  pd.S = S; pd.n_cols = n_cols; pd.T = Tj; pd.post = post; pd.active = true;      // pass 3 is owed: the next step on S or fft_flush runs it
  return BIP_OK;
}

// Run the inverse row pass that the last fft_slice_op left owing.  Every caller of a sequence of slice steps ends it with
// ms_flush (bip_api.cu: seek, bip_build_S2); fft_detect takes the owed pass into its own forward row pass.
int32_t fft_flush(bip_ctx* ctx) {
  FftPending& pd = ctx->fft_pending;
  if (!pd.active) return BIP_OK;
  pd.active = false;
  const int ny = ctx->g.ny, lnx = ilog2(ctx->g.nx);
  BIP_FFT_SWITCH(lnx, (launch_rows<LN_, true>(ctx, pd.S, pd.T, pd.post, (int64_t)pd.n_cols * ny, ny)));
  BIP_CUDA(ctx, cudaGetLastError());
  return BIP_OK;
}

// out[rho][ky][kx] += sum_n |F fields[rho][n]|^2 / G for n_rho scan positions x n_ch channel fields (destroys the fields)
int32_t fft_detect(bip_ctx* ctx, float2* fields, int n_rho, int n_ch, float* out) {
  const int ny = ctx->g.ny, nx = ctx->g.nx;
  const int lnx = ilog2(nx), lny = ilog2(ny), lc = ilog2(ctx->fft_cols);
  const int64_t G = (int64_t)ny * nx;
  FftPending& pd = ctx->fft_pending;
  if (pd.active && pd.S == fields && pd.n_cols == n_rho * n_ch) {      // the exit multislice's last inverse row pass + this forward one
    BIP_FFT_SWITCH(lnx, (launch_rows_both<LN_>(ctx, fields, pd.T, pd.post, nullptr, 0, (int64_t)n_rho * n_ch * ny, ny)));
    pd.active = false;
  } else {
    BIP_TRY(fft_flush(ctx));
    BIP_FFT_SWITCH(lnx, (launch_rows<LN_, false>(ctx, fields, nullptr, 0, (int64_t)n_rho * n_ch * ny, ny)));
  }
  const size_t smem_det = tile_smem_bytes() + (size_t)TILE_EL * sizeof(float);
  for (int r0 = 0; r0 < n_rho; r0 += 65535) {                 // gridDim.y limit
    const int nr = std::min(65535, n_rho - r0);
    const dim3 grid((unsigned)(nx >> lc), (unsigned)nr);
    BIP_FFT_SWITCH(lny, (k_ms_cols_detect<LN_><<<grid, NT, smem_det, ctx->stream>>>(fields + (int64_t)r0 * n_ch * G, n_ch, out + (int64_t)r0 * G,
                                                                                   (float)(1.0 / (double)G), nx, lc, ctx->fft_rooty,
                                                                                   ctx->fft_permy, ctx->fft_permx)));
  }
  BIP_CUDA(ctx, cudaGetLastError());
  return BIP_OK;
}

void fft_release(bip_ctx* ctx) {
  cudaFree(ctx->fft_rooty); cudaFree(ctx->fft_rootx); cudaFree(ctx->fft_Ey); cudaFree(ctx->fft_Ex); cudaFree(ctx->fft_permy); cudaFree(ctx->fft_permx);
  ctx->fft_rooty = ctx->fft_rootx = ctx->fft_Ey = ctx->fft_Ex = nullptr;
  ctx->fft_permy = ctx->fft_permx = nullptr;
}

}  // namespace bip
