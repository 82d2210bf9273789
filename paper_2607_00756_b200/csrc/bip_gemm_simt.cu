// fp32 CUDA-core versions of the two contractions (steps a4-a5 and a7-a8 of SURVEY.md 8(a)).
// They are the A/B reference for the tcgen05 kernels (precision = BIP_PREC_FP32_SIMT): same operands (the split
// planes, read as hi + lo), same epilogues, plain tiled fp32 arithmetic.
#include "bip_internal.h"

namespace bip {

namespace {

constexpr int BM = 64, BN = 64, BK = 16, PAD = 1;

struct Tile {
  float2 X[BK][BM + PAD];
  float2 Y[BK][BN + PAD];
};

// Load a [64 rows][16 k] tile of a K-major split-plane operand into smem as complex fp32 (hi + lo).
__device__ __forceinline__ void load_tile(float2 (*dst)[BM + PAD], const Planes& P, int64_t base, int row0, int rows,
                                          int k0) {
  const int t = threadIdx.x;
  const int r = t >> 2, kq = (t & 3) * 4;
  float4 rh = make_float4(0, 0, 0, 0), rl = rh, ih = rh, il = rh;
  if (row0 + r < rows) {
    const int64_t o = base + (int64_t)(row0 + r) * P.ld + k0 + kq;
    rh = *reinterpret_cast<const float4*>(P.p[0] + o);
    rl = *reinterpret_cast<const float4*>(P.p[1] + o);
    ih = *reinterpret_cast<const float4*>(P.p[2] + o);
    il = *reinterpret_cast<const float4*>(P.p[3] + o);
  }
  dst[kq + 0][r] = make_float2(rh.x + rl.x, ih.x + il.x);
  dst[kq + 1][r] = make_float2(rh.y + rl.y, ih.y + il.y);
  dst[kq + 2][r] = make_float2(rh.z + rl.z, ih.z + il.z);
  dst[kq + 3][r] = make_float2(rh.w + rl.w, ih.w + il.w);
}

// C[4][4] += X . Y^T over one 64 x 64 x Kd tile product
__device__ __forceinline__ void tile_product(Tile& sm, const Planes& X, int64_t xbase, int m0, int M, const Planes& Y,
                                             int64_t ybase, int n0, int N, int Kd, float2 (&C)[4][4]) {
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  for (int k0 = 0; k0 < Kd; k0 += BK) {
    load_tile(sm.X, X, xbase, m0, M, k0);
    load_tile(sm.Y, Y, ybase, n0, N, k0);
    __syncthreads();
#pragma unroll
    for (int k = 0; k < BK; ++k) {
      float2 x[4], y[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) x[i] = sm.X[k][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) y[j] = sm.Y[k][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          C[i][j].x = fmaf(x[i].x, y[j].x, C[i][j].x);
          C[i][j].x = fmaf(-x[i].y, y[j].y, C[i][j].x);
          C[i][j].y = fmaf(x[i].x, y[j].y, C[i][j].y);
          C[i][j].y = fmaf(x[i].y, y[j].x, C[i][j].y);
        }
    }
    __syncthreads();
  }
}

__device__ __forceinline__ float tf32_hi(float x) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return __uint_as_float(r);
}

// a4 + a5: Psi[rho][s] = sum_b A[rho][b] R1t[s][b];  Phi_n[rho][s] = H_n[s] Psi[rho][s]  -> split planes
__global__ void __launch_bounds__(256) k_gemm1_simt(Gemm1Args g) {
  __shared__ Tile sm;
  const int atom = blockIdx.z;
  const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
  float2 C[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) C[i][j] = make_float2(0.f, 0.f);
  const int Kd = (g.n_ap + BK - 1) / BK * BK;
  tile_product(sm, g.A, 0, m0, g.n_rho, g.R1t, (int64_t)atom * g.R1t.batch_stride, n0, g.w2, Kd, C);
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  for (int n = 0; n < g.n_ch; ++n) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int rho = m0 + ty * 4 + i;
      if (rho >= g.n_rho) continue;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int s = n0 + tx * 4 + j;
        if (s >= g.w2) continue;
        const float2 h = g.H[(int64_t)n * g.w2 + s];
        const float re = h.x * C[i][j].x - h.y * C[i][j].y;
        const float im = h.x * C[i][j].y + h.y * C[i][j].x;
        const int64_t o = (int64_t)atom * g.Phi.batch_stride + (int64_t)n * g.phi_ch_stride + (int64_t)rho * g.Phi.ld + s;
        const float rh = tf32_hi(re), ih = tf32_hi(im);
        g.Phi.p[0][o] = rh; g.Phi.p[1][o] = tf32_hi(re - rh);
        g.Phi.p[2][o] = ih; g.Phi.p[3][o] = tf32_hi(im - ih);
      }
    }
  }
}

// a7 + a8: a_n[rho][d] = G^-1/2 sum_s Phi_n[rho][s] R2[d][s];  I += sum_n |a_n|^2 reduced per mode
__global__ void __launch_bounds__(256) k_gemm2_simt(Gemm2Args g) {
  __shared__ Tile sm;
  const int atom = blockIdx.z;
  const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  float P[4][4];
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) P[i][j] = 0.f;
  const int Kd = (g.w2 + BK - 1) / BK * BK;
  for (int n = 0; n < g.n_ch; ++n) {
    float2 C[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) C[i][j] = make_float2(0.f, 0.f);
    tile_product(sm, g.Phi, (int64_t)atom * g.Phi.batch_stride + (int64_t)n * g.phi_ch_stride, m0, g.n_rho, g.R2,
                 (int64_t)atom * g.R2.batch_stride, n0, g.n_det, Kd, C);
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
      for (int j = 0; j < 4; ++j) P[i][j] += C[i][j].x * C[i][j].x + C[i][j].y * C[i][j].y;
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int rho = m0 + ty * 4 + i;
    float rowsum = 0.f;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int d = n0 + tx * 4 + j;
      const float v = (rho < g.n_rho && d < g.n_det) ? P[i][j] * g.inv_G : 0.f;
      rowsum += v;
      if (rho < g.n_rho && d < g.n_det) {
        if (g.mode == BIP_MODE_CUBE) atomicAdd(reinterpret_cast<float*>(g.out) + (int64_t)rho * g.n_det + d, v);
        else if (g.mode != BIP_MODE_MAP)
          atomicAdd(reinterpret_cast<float*>(g.out) + (int64_t)rho * g.n_bins + g.bin_of_det[d], v);
      }
    }
    if (g.mode == BIP_MODE_MAP) {       // sum over the 16 threads that share this row (half a warp)
      rowsum += __shfl_xor_sync(0xffffffffu, rowsum, 8);
      rowsum += __shfl_xor_sync(0xffffffffu, rowsum, 4);
      rowsum += __shfl_xor_sync(0xffffffffu, rowsum, 2);
      rowsum += __shfl_xor_sync(0xffffffffu, rowsum, 1);
      if (tx == 0 && rho < g.n_rho) atomicAdd(reinterpret_cast<double*>(g.out) + rho, (double)rowsum);
    }
  }
}

}  // namespace

int32_t launch_gemm1_simt(bip_ctx* ctx, const Gemm1Args& a) {
  dim3 grid((unsigned)((a.w2 + BN - 1) / BN), (unsigned)((a.n_rho + BM - 1) / BM), (unsigned)a.n_atoms);
  k_gemm1_simt<<<grid, 256, 0, ctx->stream>>>(a);
  BIP_CUDA(ctx, cudaGetLastError());
  ctx->timing.kernel_launches++;
  return BIP_OK;
}

int32_t launch_gemm2_simt(bip_ctx* ctx, const Gemm2Args& a) {
  dim3 grid((unsigned)((a.n_det + BN - 1) / BN), (unsigned)((a.n_rho + BM - 1) / BM), (unsigned)a.n_atoms);
  k_gemm2_simt<<<grid, 256, 0, ctx->stream>>>(a);
  BIP_CUDA(ctx, cudaGetLastError());
  ctx->timing.kernel_launches++;
  return BIP_OK;
}

}  // namespace bip
