// Device building blocks of the library's own power-of-two FFTs: the radix-8 / 4 / 2 butterflies and double-float constant
// products shared by both users, the per-stage twiddle tables, and the run-time-sized transform on padded shared-memory lines
// that bip_focal.cu uses for the Fresnel steps on padded windows (bip_fft.cu has its own compile-time-sized stages for the
// slice steps on the whole grid).
// See the header comment of bip_fft.cu for why every constant is a hi + lo pair.
#ifndef BIP_FFT_CUH_
#define BIP_FFT_CUH_

#include <cmath>
#include <cstdint>
#include <vector>
#include <cuda_runtime.h>

namespace bip {
namespace fftdev {

__device__ __forceinline__ float2 cmulf(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
// a * (hi + lo) with w = (hi.x, hi.y, lo.x, lo.y): the small products enter the FMA chain first, so they are part of the
// exact sum that each final FMA rounds once
__device__ __forceinline__ float2 cmul_dd(float2 a, float4 w) {
  return make_float2(fmaf(a.x, w.x, fmaf(-a.y, w.y, fmaf(a.x, w.z, -a.y * w.w))),
                     fmaf(a.x, w.y, fmaf(a.y, w.x, fmaf(a.x, w.w, a.y * w.z))));
}
__device__ __forceinline__ float2 cmulc_dd(float2 a, float4 w) {            // a * conj(hi + lo)
  return make_float2(fmaf(a.x, w.x, fmaf(a.y, w.y, fmaf(a.x, w.z, a.y * w.w))),
                     fmaf(a.y, w.x, fmaf(-a.x, w.y, fmaf(a.y, w.z, -a.x * w.w))));
}
__device__ __forceinline__ float mul_h(float v) {                            // v * sqrt(1/2), sqrt(1/2) = hi + lo
  return fmaf(v, 0.70710676908493042f, v * 1.2101617485e-8f);
}
__device__ __forceinline__ float2 caddf(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csubf(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 mul_mi(float2 a) { return make_float2(a.y, -a.x); }    // a * (-i)
__device__ __forceinline__ float2 mul_pi(float2 a) { return make_float2(-a.y, a.x); }    // a * (+i)

// R-point DFT in registers, X[m] = sum_k x[k] exp(-+ 2 pi i k m / R) (INV = false / true), unnormalised.
template <int R, bool INV>
__device__ __forceinline__ void dft_small(float2 (&x)[8]) {
  if (R == 2) {
    const float2 a = x[0], b = x[1];
    x[0] = caddf(a, b); x[1] = csubf(a, b);
  } else if (R == 4) {
    const float2 s02 = caddf(x[0], x[2]), d02 = csubf(x[0], x[2]), s13 = caddf(x[1], x[3]), d13 = csubf(x[1], x[3]);
    const float2 r = INV ? mul_pi(d13) : mul_mi(d13);          // -+ i (x1 - x3)
    x[0] = caddf(s02, s13); x[2] = csubf(s02, s13);
    x[1] = caddf(d02, r);   x[3] = csubf(d02, r);
  } else {
    float2 a[4], b[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) { a[k] = caddf(x[k], x[k + 4]); b[k] = csubf(x[k], x[k + 4]); }
    // b_k *= w8^k, w8 = exp(-+ i pi / 4)
    b[1] = INV ? make_float2(mul_h(b[1].x - b[1].y), mul_h(b[1].x + b[1].y)) : make_float2(mul_h(b[1].x + b[1].y), mul_h(b[1].y - b[1].x));
    b[2] = INV ? mul_pi(b[2]) : mul_mi(b[2]);
    b[3] = INV ? make_float2(mul_h(-b[3].x - b[3].y), mul_h(b[3].x - b[3].y)) : make_float2(mul_h(b[3].y - b[3].x), mul_h(-b[3].x - b[3].y));
    {
      const float2 s02 = caddf(a[0], a[2]), d02 = csubf(a[0], a[2]), s13 = caddf(a[1], a[3]), d13 = csubf(a[1], a[3]);
      const float2 r = INV ? mul_pi(d13) : mul_mi(d13);
      x[0] = caddf(s02, s13); x[4] = csubf(s02, s13); x[2] = caddf(d02, r); x[6] = csubf(d02, r);
    }
    {
      const float2 s02 = caddf(b[0], b[2]), d02 = csubf(b[0], b[2]), s13 = caddf(b[1], b[3]), d13 = csubf(b[1], b[3]);
      const float2 r = INV ? mul_pi(d13) : mul_mi(d13);
      x[1] = caddf(s02, s13); x[5] = csubf(s02, s13); x[3] = caddf(d02, r); x[7] = csubf(d02, r);
    }
  }
}

// Shared-memory index of element i of a line: one float2 of padding after every 8, so that the stride-8 and stride-64
// accesses of the later stages fall into different banks (a half-warp's 64-bit accesses then cover 16 distinct bank pairs).
__device__ __forceinline__ int pad_idx(int i) { return i + (i >> 3); }
__host__ __device__ constexpr int pad_len(int n) { return n + (n >> 3); }

// Twiddle tables are stored PER STAGE, transposed: for the radix-8 stage on block length L (sub = L / 8 > 1) the entry of
// output m (1..7) and position j (0..sub-1) is w_L^(j m) at  stage_off(L) + (m - 1) * sub + j, so that the lanes of a warp
// (consecutive j) read consecutive 16-byte entries.  (With one table of N-th roots indexed by j m N / L every lane of a
// warp hit its own cache line: the kernels were bound by the L1 data path, profiles/r02_fft_ncu.md.)
// stage_off: stages run L = N, N/8, N/64, ...; the table of stage L starts after those of all longer stages.
__host__ __device__ inline int tw_stage_off(int lN, int lL) {
  int off = 0;
  for (int l = lN; l > lL; l -= 3) off += 7 << (l - 3);
  return off;
}
__host__ __device__ inline int tw_table_len(int lN) {       // entries of all radix-8 stages with sub > 1
  int n = 0;
  for (int l = lN; l > 3; l -= 3) n += 7 << (l - 3);
  return n > 0 ? n : 1;
}

// One stage on block length L = 2^lL with radix R over all lines of the block.  Forward (DIF): butterfly, then twiddle
// w_L^(j m); inverse (DIT): conjugate twiddle, then inverse butterfly.  Element (line, i) lives at sm[line * pitch + pad_idx(i)].
// All sizes are powers of two: shifts and masks, no integer division.  A stage with L == R has j = 0 only: no twiddles
// (the radix-4 / radix-2 remainder stages are always of that kind).
template <int R, bool INV>
__device__ __forceinline__ void fft_stage(float2* sm, int lN, int lL, int n_lines, int pitch, const float4* __restrict__ root, int tid, int nthr) {
  constexpr int lR = R == 8 ? 3 : R == 4 ? 2 : 1;
  const int lsub = lL - lR, sub = 1 << lsub, lper = lN - lR, nv = 1 << lper;
  const float4* tw = root + tw_stage_off(lN, lL);
  // thread <-> butterfly position v inside a line (consecutive lanes = consecutive v: coalesced twiddle reads, conflict-free
  // shared-memory accesses); the thread keeps the 7 twiddles of its position in registers and loops over the LINES of the
  // block with them -- every line of a block needs the same twiddles, and fetching them per line made the twiddle reads
  // half of the L1 traffic of these kernels (profiles/r02_fft_ncu.md)
  const int lthr = 31 - __clz(nthr), lv = lthr < lper ? lthr : lper;       // nthr is a power of two
  const int line0 = tid >> lv, line_step = nthr >> lv;
  for (int v = tid & ((1 << lv) - 1); v < nv; v += 1 << lv) {
    const int blk = v >> lsub, j = v & (sub - 1);
    const int i0 = (blk << lL) + j;
    float4 w[8];
    if (R == 8 && lsub > 0) {
#pragma unroll
      for (int m = 1; m < R; ++m) w[m] = __ldg(tw + ((m - 1) << lsub) + j);
    }
    for (int line = line0; line < n_lines; line += line_step) {
      float2* p = sm + line * pitch;
      float2 x[8];
#pragma unroll
      for (int k = 0; k < R; ++k) x[k] = p[pad_idx(i0 + (k << lsub))];
      if (INV && R == 8 && lsub > 0) {
#pragma unroll
        for (int m = 1; m < R; ++m) x[m] = cmulc_dd(x[m], w[m]);
      }
      dft_small<R, INV>(x);
      if (!INV && R == 8 && lsub > 0) {
#pragma unroll
        for (int m = 1; m < R; ++m) x[m] = cmul_dd(x[m], w[m]);
      }
#pragma unroll
      for (int k = 0; k < R; ++k) p[pad_idx(i0 + (k << lsub))] = x[k];
    }
  }
}

// Whole transform of every line: radix sequence 8, 8, ..., then 4 or 2 (forward); the inverse runs the same stages backwards.
template <bool INV>
__device__ __forceinline__ void fft_lines(float2* sm, int lN, int n_lines, int pitch, const float4* __restrict__ root, int tid, int nthr) {
  if (!INV) {
    int lL = lN;
    for (; lL >= 3; lL -= 3) { fft_stage<8, false>(sm, lN, lL, n_lines, pitch, root, tid, nthr); __syncthreads(); }
    if (lL == 2) { fft_stage<4, false>(sm, lN, 2, n_lines, pitch, root, tid, nthr); __syncthreads(); }
    else if (lL == 1) { fft_stage<2, false>(sm, lN, 1, n_lines, pitch, root, tid, nthr); __syncthreads(); }
  } else {
    int lL = lN % 3;                                         // length left for the last forward stage: 2^0, 2^1 or 2^2
    if (lL == 2) { fft_stage<4, true>(sm, lN, 2, n_lines, pitch, root, tid, nthr); __syncthreads(); }
    else if (lL == 1) { fft_stage<2, true>(sm, lN, 1, n_lines, pitch, root, tid, nthr); __syncthreads(); }
    for (lL += 3; lL <= lN; lL += 3) { fft_stage<8, true>(sm, lN, lL, n_lines, pitch, root, tid, nthr); __syncthreads(); }
  }
}


}  // namespace fftdev

// host helpers
inline bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }
inline int ilog2(int n) { int l = 0; while ((1 << l) < n) ++l; return l; }
inline size_t smem_rows_bytes(int lines, int nx) { return (size_t)lines * fftdev::pad_len(nx) * sizeof(float2); }
inline size_t smem_cols_bytes(int cols, int ny) { return (size_t)cols * (fftdev::pad_len(ny) + 1) * sizeof(float2); }

// frequency index held at stored position `pos` after the forward (DIF) transform of length N
inline int dif_frequency(int pos, int N) {
  if (N == 1) return 0;
  const int r = N >= 8 ? 8 : N;
  const int sub = N / r;
  return r * dif_frequency(pos % sub, sub) + pos / sub;
}


// (hi, lo) double-float pair of a complex constant
inline float4 dd_pair(double re, double im) {
  const float hr = (float)re, hi = (float)im;
  return make_float4(hr, hi, (float)(re - (double)hr), (float)(im - (double)hi));
}


// per-stage transposed twiddle table of a length-N transform (see tw_stage_off): entries exp(-2 pi i j m / L)
inline std::vector<float4> make_twiddle_table(int N) {
  const int lN = ilog2(N);
  std::vector<float4> t((size_t)fftdev::tw_table_len(lN), make_float4(1.f, 0.f, 0.f, 0.f));
  for (int lL = lN; lL > 3; lL -= 3) {
    const int L = 1 << lL, sub = L >> 3, off = fftdev::tw_stage_off(lN, lL);
    for (int m = 1; m < 8; ++m)
      for (int j = 0; j < sub; ++j) {
        const double a = -2.0 * M_PI * (double)((int64_t)j * m % L) / (double)L;
        t[(size_t)off + (size_t)(m - 1) * sub + j] = dd_pair(std::cos(a), std::sin(a));
      }
  }
  return t;
}

}  // namespace bip
#endif  // BIP_FFT_CUH_
