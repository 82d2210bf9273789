// Tile-blocked, three-slice bf16 operand format of the tensor-core contractions (precision BIP_PREC_BF16X6).
//
// Why not plain 3xTF32: tcgen05.mma accumulates into TMEM with truncation (profiles/r01_tcgen05_rounding_probe.txt),
// which shrinks every amplitude by ~1.25e-8 per accumulating MMA and breaks the 1e-6 summed-intensity bound after a
// few dozen steps.  Here every real operand x of a row with power-of-two scale s (s >= max |x| of the row) is split
//
//     x / s = x1 + x2 + x3,   x1 = rint(128 x / s) / 128   (8-bit fixed point: an integer / 128, exact in bf16)
//                             x2 = bf16(x / s - x1),  x3 = bf16(x / s - x1 - x2)      (floating residuals)
//
// and a real product is x1 y1 + (x1 y2 + x2 y1) + (x1 y3 + x2 y2 + x3 y1): six kind::f16 (bf16) MMAs at twice the
// TF32 rate, i.e. the tensor time of 3xTF32.  The leading products x1 y1 are integers / 2^14, so their sum over a
// chunk of 256 k-elements (2 x 256 x 2^14 = 2^23 < 2^24) is EXACT in the fp32 accumulator -- no truncation, no
// bias; the chunk sums are added in fp32 round-to-nearest by the epilogue warps.  The small products (<= 2^-8 of
// the leading ones) go to a second accumulator, whose truncation is 2^-8 smaller and harmless.
//
// Memory layout (what one cp.async.bulk brings in): [batch][row tile of 128][k-step of 16][part 6][128 x 16 tile],
// part = (re1, re2, re3, im1, im2, im3), each 128 x 16 tile in the canonical K-major no-swizzle UMMA layout
// (8-row x 16-byte core matrices: SBO = 256 B between 8-row groups, LBO = 128 B between the two k halves).
#ifndef BIP_SLICED_CUH_
#define BIP_SLICED_CUH_

#include <cuda_bf16.h>
#include <cstdint>

namespace bip {

constexpr int SL_ROWS = 128;                       // rows per tile
constexpr int SL_K = 16;                           // k-elements per step (one kind::f16 MMA)
constexpr int SL_TILE_EL = SL_ROWS * SL_K;         // 2048 bf16 = 4 KB per part
constexpr int SL_PARTS = 6;
constexpr int SL_STEP_EL = SL_PARTS * SL_TILE_EL;  // 12288 bf16 = 24 KB per (row tile, k-step)

struct Sliced {
  __nv_bfloat16* base = nullptr;
  float* scale = nullptr;            // [batch][rows_pad] power-of-two row scale: value = stored * scale
  int64_t rows = 0, rows_pad = 0;    // valid rows; padded to a multiple of 128
  int64_t k = 0, ksteps = 0;         // valid k; ceil(k / 16)
  int64_t batch_stride = 0;          // bf16 elements between batch items (0 = shared by all)
  int64_t scale_batch_stride = 0;    // floats between batch items of `scale`
};

#ifdef __CUDACC__
// element offset of (row, k-group g of 8 consecutive k) for part 0; add part * SL_TILE_EL; 8 bf16 (16 B) contiguous
__device__ __forceinline__ int64_t sl_group_offset(const Sliced& S, int64_t row, int64_t g) {
  const int64_t tile = row >> 7, r = row & 127, ks = g >> 1, half = g & 1;
  return (tile * S.ksteps + ks) * SL_STEP_EL + (r >> 3) * 128 + half * 64 + (r & 7) * 8;
}

// power-of-two scale >= m (m >= 0); 1 for an all-zero row
__device__ __forceinline__ float sl_pow2_scale(float m) {
  if (!(m > 0.f)) return 1.f;
  int e;
  const float f = frexpf(m, &e);           // m = f 2^e, f in [0.5, 1)
  (void)f;
  return ldexpf(1.f, e);                   // 2^e > m  (>= m)
}

__device__ __forceinline__ void sl_split(float x, float inv_scale, __nv_bfloat16& s1, __nv_bfloat16& s2, __nv_bfloat16& s3) {
  const float t = x * inv_scale;           // exact: power of two
  const float a = rintf(t * 128.f) * (1.f / 128.f);
  const float r1 = t - a;                  // exact
  const __nv_bfloat16 b = __float2bfloat16_rn(r1);
  const float r2 = r1 - __bfloat162float(b);   // exact
  s1 = __float2bfloat16_rn(a);             // exact: |integer| <= 128 (or a little more) over 128
  s2 = b;
  s3 = __float2bfloat16_rn(r2);
}

// Split 8 consecutive complex values (re[8], im[8]) of one row and store the six 16-byte groups.
__device__ __forceinline__ void sl_store_group(const Sliced& S, int64_t batch, int64_t row, int64_t g, const float (&re)[8],
                                               const float (&im)[8], float inv_scale) {
  __align__(16) __nv_bfloat16 out[6][8];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    sl_split(re[j], inv_scale, out[0][j], out[1][j], out[2][j]);
    sl_split(im[j], inv_scale, out[3][j], out[4][j], out[5][j]);
  }
  __nv_bfloat16* p = S.base + batch * S.batch_stride + sl_group_offset(S, row, g);
#pragma unroll
  for (int part = 0; part < 6; ++part) *reinterpret_cast<uint4*>(p + part * SL_TILE_EL) = *reinterpret_cast<const uint4*>(out[part]);
}
#endif  // __CUDACC__

}  // namespace bip
#endif  // BIP_SLICED_CUH_
