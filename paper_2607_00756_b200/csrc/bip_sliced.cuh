// Tile-blocked, sliced 16-bit operand formats of the tensor-core contractions (precisions BIP_PREC_FP16X4 and
// BIP_PREC_BF16X6).
//
// Why not plain 3xTF32: tcgen05.mma accumulates into TMEM with truncation (profiles/r01_tcgen05_rounding_probe.txt),
// which shrinks every amplitude by ~1.25e-8 per accumulating MMA and breaks the 1e-6 summed-intensity bound after a
// few dozen steps.  Here every real operand x of a row with power-of-two scale s (s > max |x| of the row) is split
// into a LEADING fixed-point slice and floating residual slices:
//
//   FP16X4:  x / s = x1 + x2 (+ 2^-21),  x1 = rint(256 x / s) / 256  (an integer / 2^8, |integer| <= 256, exact in fp16)
//                                        x2 = fp16(x / s - x1)      (|x2| <= 2^-9, 11 significant bits)
//            real product = x1 y1 + (x1 y2 + x2 y1 + x2 y2): FOUR kind::f16 MMAs -- 2/3 of the tensor time of 3xTF32.
//   BF16X6:  x / s = x1 + x2 + x3,       x1 = rint(128 x / s) / 128, x2 = bf16(x / s - x1), x3 = bf16(x / s - x1 - x2)
//            real product = x1 y1 + (x1 y2 + x2 y1) + (x1 y3 + x2 y2 + x3 y1): SIX bf16 MMAs (the time of 3xTF32).
//
// The leading products x1 y1 are integers / 2^16 (FP16X4) or / 2^14 (BF16X6), so their sum over a chunk of 128
// (resp. 256) k-elements of the complex product (2 x 128 x 2^16 = 2^24) is EXACT in the fp32 accumulator -- no
// truncation, no bias; the chunk sums are added in fp32 round-to-nearest by the epilogue warps.  The small products
// (<= 2^-8 of the leading ones) go to a second accumulator, whose truncation is 2^-8 smaller and harmless.
//
// Y operands of the FP16X4 CTA-pair kernel carry two more parts, the NEGATED imaginary slices (-im1, -im2; the sign flip
// of an fp16 is exact): the kernel forms [Cr | Ci] with N = 256 MMAs, x_re . [y_re ; y_im] and x_im . [-y_im ; y_re],
// which halves the shared-memory operand reads per flop (bip_gemm_sliced.cu).
//
// Memory layout (what one cp.async.bulk brings in): [batch][row tile of 128][k-step of 16][part][128 x 16 tile],
// parts = (re1, re2, im1, im2) or (re1, re2, re3, im1, im2, im3), each 128 x 16 tile in the canonical K-major
// no-swizzle UMMA layout (8-row x 16-byte core matrices: SBO = 256 B between 8-row groups, LBO = 128 B between the
// two k halves).
#ifndef BIP_SLICED_CUH_
#define BIP_SLICED_CUH_

#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cstdint>

namespace bip {

constexpr int SL_ROWS = 128;                       // rows per tile
constexpr int SL_K = 16;                           // k-elements per step (one kind::f16 MMA)
constexpr int SL_TILE_EL = SL_ROWS * SL_K;         // 2048 16-bit elements = 4 KB per part

enum SlicedFmt : int32_t { SL_FMT_BF16X6 = 0, SL_FMT_FP16X4 = 1 };
__host__ __device__ constexpr int sl_parts(int fmt) { return fmt == SL_FMT_FP16X4 ? 4 : 6; }
__host__ __device__ constexpr int sl_step_el(int fmt) { return sl_parts(fmt) * SL_TILE_EL; }   // 16 KB / 24 KB per (row tile, k-step)

struct Sliced {
  uint16_t* base = nullptr;          // fp16 or bf16 bit patterns
  int32_t neg_im = 0;                // 1: two extra parts (-im1, -im2) after the regular ones (FP16X4 Y operands)
  float* scale = nullptr;            // [batch][rows_pad] power-of-two row scale: value = stored * scale
  int64_t rows = 0, rows_pad = 0;    // valid rows; padded to a multiple of 128
  int64_t k = 0, ksteps = 0;         // valid k; ceil(k / 16)
  int64_t batch_stride = 0;          // 16-bit elements between batch items (0 = shared by all)
  int64_t scale_batch_stride = 0;    // floats between batch items of `scale`
  int32_t fmt = SL_FMT_FP16X4;
};

__host__ __device__ inline int sl_parts_of(const Sliced& S) {
#ifdef BIP_TUNING
  return sl_parts(S.fmt) + (S.neg_im ? 2 : 0);
#else
  return sl_parts(S.fmt);                  // the shipped build never sets neg_im (N = 256 A/B variant only)
#endif
}
__host__ __device__ inline int sl_step_el_of(const Sliced& S) { return sl_parts_of(S) * SL_TILE_EL; }

#ifdef __CUDACC__
// element offset of (row, k-group g of 8 consecutive k) for part 0; add part * SL_TILE_EL; 8 elements (16 B) contiguous
__device__ __forceinline__ int64_t sl_group_offset(const Sliced& S, int64_t row, int64_t g) {
  const int64_t tile = row >> 7, r = row & 127, ks = g >> 1, half = g & 1;
  return (tile * S.ksteps + ks) * sl_step_el_of(S) + (r >> 3) * 128 + half * 64 + (r & 7) * 8;
}

// power-of-two scale > m (m >= 0); 1 for an all-zero row
__device__ __forceinline__ float sl_pow2_scale(float m) {
  if (!(m > 0.f)) return 1.f;
  int e;
  (void)frexpf(m, &e);                     // m = f 2^e, f in [0.5, 1)
  return ldexpf(1.f, e);                   // 2^e > m
}

__device__ __forceinline__ void sl_split_bf16(float x, float inv_scale, uint16_t& s1, uint16_t& s2, uint16_t& s3) {
  const float t = x * inv_scale;           // exact: power of two
  const float a = rintf(t * 128.f) * (1.f / 128.f);
  const float r1 = t - a;                  // exact
  const __nv_bfloat16 b = __float2bfloat16_rn(r1);
  const float r2 = r1 - __bfloat162float(b);   // exact
  s1 = __bfloat16_as_ushort(__float2bfloat16_rn(a));   // exact: |integer| <= 128 over 128
  s2 = __bfloat16_as_ushort(b);
  s3 = __bfloat16_as_ushort(__float2bfloat16_rn(r2));
}

__device__ __forceinline__ void sl_split_fp16(float x, float inv_scale, uint16_t& s1, uint16_t& s2) {
  const float t = x * inv_scale;           // exact: power of two
  const float a = rintf(t * 256.f) * (1.f / 256.f);
  s1 = __half_as_ushort(__float2half_rn(a));           // exact: |integer| <= 256 over 256
  s2 = __half_as_ushort(__float2half_rn(t - a));       // t - a exact, |t - a| <= 2^-9
}

// Split 8 consecutive complex values (re[8], im[8]) of one row and store the 16-byte group of every part.
__device__ __forceinline__ void sl_store_group(const Sliced& S, int64_t batch, int64_t row, int64_t g, const float (&re)[8],
                                               const float (&im)[8], float inv_scale) {
  uint16_t* p = S.base + batch * S.batch_stride + sl_group_offset(S, row, g);
  if (S.fmt == SL_FMT_FP16X4) {
    __align__(16) uint16_t out[4][8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      sl_split_fp16(re[j], inv_scale, out[0][j], out[1][j]);
      sl_split_fp16(im[j], inv_scale, out[2][j], out[3][j]);
    }
#pragma unroll
    for (int part = 0; part < 4; ++part) *reinterpret_cast<uint4*>(p + part * SL_TILE_EL) = *reinterpret_cast<const uint4*>(out[part]);
#ifdef BIP_TUNING                    // only the N = 256 A/B variant reads these parts; the shipped build never sets neg_im
    if (S.neg_im) {
#pragma unroll
      for (int part = 2; part < 4; ++part) {
        uint4 v = *reinterpret_cast<const uint4*>(out[part]);
        v.x ^= 0x80008000u; v.y ^= 0x80008000u; v.z ^= 0x80008000u; v.w ^= 0x80008000u;     // -im: flip the fp16 sign bits
        *reinterpret_cast<uint4*>(p + (part + 2) * SL_TILE_EL) = v;
      }
    }
#endif
  } else {
    __align__(16) uint16_t out[6][8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      sl_split_bf16(re[j], inv_scale, out[0][j], out[1][j], out[2][j]);
      sl_split_bf16(im[j], inv_scale, out[3][j], out[4][j], out[5][j]);
    }
#pragma unroll
    for (int part = 0; part < 6; ++part) *reinterpret_cast<uint4*>(p + part * SL_TILE_EL) = *reinterpret_cast<const uint4*>(out[part]);
  }
}
#endif  // __CUDACC__

}  // namespace bip
#endif  // BIP_SLICED_CUH_
