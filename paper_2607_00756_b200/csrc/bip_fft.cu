// Fused slice step of the parent columns for power-of-two grids (plumbing of bip_build_S2 / ADVANCETO / PEELTO):
//
//     S  <-  post . F^-1[ Pspec . F[ pre . S ] ]          (eq. 2, eq. 6, eq. 12; pre / post in {1, T_j, conj T_j})
//
// in THREE passes over the column instead of the eleven of the cuFFT route (load/convert, 2 x 2 cuFFT passes, spectrum
// multiply, store/convert, each reading and writing the whole column):
//
//   pass 1  rows:     load S[y][.] (x pre),  forward FFT along x in shared memory,           store
//   pass 2  columns:  load a tile of columns, forward FFT along y, x P(q) / G, inverse FFT along y, store
//   pass 3  rows:     load, inverse FFT along x, (x post), store
//
// i.e. 48 bytes of HBM traffic per pixel and slice step.  The forward transforms are decimation-in-frequency (natural
// order in, digit-reversed order out), the inverse ones decimation-in-time (digit-reversed in, natural out), so no
// reordering pass exists at all: the propagator table is stored once in the digit-reversed order of both axes.
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

__device__ __forceinline__ float2 apply_t(float2 v, const float2* __restrict__ T, int64_t i, int mode) {
  if (mode == 0) return v;
  float2 t = __ldg(T + i);
  if (mode == 2) t.y = -t.y;
  return cmulf(v, t);
}

// Passes 1 and 3: LINES rows per block.  tmode: 0 none, 1 multiply by T, 2 by conj T (before the forward transform /
// after the inverse one).
template <bool INV>
__global__ void __launch_bounds__(256, 3) k_ms_rows(float2* __restrict__ S, const float2* __restrict__ T, int tmode, int ny, int lnx, int lines,
                                                  const float4* __restrict__ rootx) {
  extern __shared__ float2 sm_rows[];
  const int nx = 1 << lnx, pitch = pad_len(nx);
  const int64_t G = (int64_t)ny * nx;
  float2* col = S + (int64_t)blockIdx.y * G;
  const int y0 = blockIdx.x * lines;
  const int n_lines = min(lines, ny - y0);
  const int tid = threadIdx.x, nthr = blockDim.x;
  for (int i = tid; i < (n_lines << lnx); i += nthr) {
    const int64_t g = (int64_t)y0 * nx + i;
    float2 v = col[g];
    if (!INV) v = apply_t(v, T, g, tmode);
    sm_rows[(i >> lnx) * pitch + pad_idx(i & (nx - 1))] = v;
  }
  __syncthreads();
  fft_lines<INV>(sm_rows, lnx, n_lines, pitch, rootx, tid, nthr);
  for (int i = tid; i < (n_lines << lnx); i += nthr) {
    const int64_t g = (int64_t)y0 * nx + i;
    float2 v = sm_rows[(i >> lnx) * pitch + pad_idx(i & (nx - 1))];
    if (INV) v = apply_t(v, T, g, tmode);
    col[g] = v;
  }
}

// Pass 2: a tile of `cols` columns (consecutive stored x positions) x ny rows per block; forward along y, spectrum
// multiply with the digit-reversed propagator table (conjugated when conj_p), inverse along y.
__global__ void __launch_bounds__(256, 3) k_ms_cols(float2* __restrict__ S, const float4* __restrict__ Pperm, int conj_p, int lny, int nx, int lcols,
                                                  const float4* __restrict__ rooty) {
  extern __shared__ float2 sm_cols[];
  const int ny = 1 << lny, cols = 1 << lcols;
  const int64_t G = (int64_t)ny * nx;
  float2* col = S + (int64_t)blockIdx.y * G;
  const int x0 = blockIdx.x << lcols;
  const int pitch = pad_len(ny) + 1;
  const int tid = threadIdx.x, nthr = blockDim.x;
  for (int i = tid; i < (ny << lcols); i += nthr) {
    const int y = i >> lcols, c = i & (cols - 1);
    sm_cols[c * pitch + pad_idx(y)] = col[(int64_t)y * nx + x0 + c];
  }
  __syncthreads();
  fft_lines<false>(sm_cols, lny, cols, pitch, rooty, tid, nthr);
  for (int i = tid; i < (ny << lcols); i += nthr) {
    const int y = i >> lcols, c = i & (cols - 1);
    const float4 p = __ldg(Pperm + (int64_t)y * nx + x0 + c);
    float2* e = sm_cols + c * pitch + pad_idx(y);
    *e = conj_p ? cmulc_dd(*e, p) : cmul_dd(*e, p);
  }
  __syncthreads();
  fft_lines<true>(sm_cols, lny, cols, pitch, rooty, tid, nthr);
  for (int i = tid; i < (ny << lcols); i += nthr) {
    const int y = i >> lcols, c = i & (cols - 1);
    col[(int64_t)y * nx + x0 + c] = sm_cols[c * pitch + pad_idx(y)];
  }
}

// Detector plane of Algorithm 3 (Alg. 1 lines 6-7): after the row pass (forward along x, stored order),
// forward FFT along y of a tile of columns of every channel field of one scan position and
//     out[rho][ky][kx] += sum_n |F psi_n|^2 / G
// at the TRUE frequency (ky, kx) of the stored position (permy / permx undo the digit reversal).  A block owns the
// (all y, its x tile) outputs of its scan position, so the read-modify-write needs no atomics.
__global__ void __launch_bounds__(256, 2) k_ms_cols_detect(const float2* __restrict__ F, int n_ch, float* __restrict__ out, float inv_G, int lny, int nx,
                                                         int lcols, const float4* __restrict__ rooty, const int32_t* __restrict__ permy,
                                                         const int32_t* __restrict__ permx) {
  extern __shared__ float2 sm_det[];
  const int ny = 1 << lny, cols = 1 << lcols;
  const int64_t G = (int64_t)ny * nx;
  const int x0 = blockIdx.x << lcols, rho = blockIdx.y;
  const int pitch = pad_len(ny) + 1;
  float* acc = reinterpret_cast<float*>(sm_det + (size_t)cols * pitch);       // [ny * cols], element i of the tile loop
  const int tid = threadIdx.x, nthr = blockDim.x;
  for (int i = tid; i < (ny << lcols); i += nthr) acc[i] = 0.f;
  for (int n = 0; n < n_ch; ++n) {
    const float2* col = F + ((int64_t)rho * n_ch + n) * G;
    __syncthreads();
    for (int i = tid; i < (ny << lcols); i += nthr) {
      const int y = i >> lcols, c = i & (cols - 1);
      sm_det[c * pitch + pad_idx(y)] = col[(int64_t)y * nx + x0 + c];
    }
    __syncthreads();
    fft_lines<false>(sm_det, lny, cols, pitch, rooty, tid, nthr);
    for (int i = tid; i < (ny << lcols); i += nthr) {
      const int y = i >> lcols, c = i & (cols - 1);
      const float2 v = sm_det[c * pitch + pad_idx(y)];
      acc[i] += v.x * v.x + v.y * v.y;
    }
  }
  float* o = out + (int64_t)rho * G;
  for (int i = tid; i < (ny << lcols); i += nthr) {
    const int y = i >> lcols, c = i & (cols - 1);
    const int64_t k = (int64_t)__ldg(permy + y) * nx + __ldg(permx + x0 + c);
    o[k] += acc[i] * inv_G;
  }
}

// threads per block: a power of two, a quarter of the butterflies of a stage (lines * N / 8), within 64 .. 256
int fft_threads(int lines, int n) {
  const int reuse = std::max(1, tune_int("BIP_TUNE_FFT_REUSE", 4));
  int t = 64;
  while (t < 256 && t * reuse < lines * n / 8) t <<= 1;
  return t;
}

}  // namespace

bool fft_supported(const bip_ctx* ctx) {
  return is_pow2(ctx->g.ny) && is_pow2(ctx->g.nx) && ctx->g.ny >= 8 && ctx->g.nx >= 8 && ctx->g.ny <= 4096 && ctx->g.nx <= 4096;
}

int32_t fft_init(bip_ctx* ctx) {
  const int ny = ctx->g.ny, nx = ctx->g.nx;
  const int64_t G = (int64_t)ny * nx;
  auto dd = [](double re, double im) { return dd_pair(re, im); };
  std::vector<float4> ry = make_twiddle_table(ny), rx = make_twiddle_table(nx), P(G);
  // Fresnel propagator P(q) = exp(-i pi lambda dz |q|^2) / G (eq. 2; no band limit), in the stored (digit-reversed) order
  for (int py = 0; py < ny; ++py) {
    const int ky = dif_frequency(py, ny), hy = ky < (ny + 1) / 2 ? ky : ky - ny;
    const double qy = hy / ctx->g.ly;
    for (int px = 0; px < nx; ++px) {
      const int kx = dif_frequency(px, nx), hx = kx < (nx + 1) / 2 ? kx : kx - nx;
      const double qx = hx / ctx->g.lx;
      const double ph = -M_PI * ctx->g.lambda * ctx->g.dz * (qy * qy + qx * qx);
      P[(int64_t)py * nx + px] = dd(std::cos(ph) / (double)G, std::sin(ph) / (double)G);
    }
  }
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->fft_rooty, sizeof(float4) * ry.size(), "fft twiddles"));
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->fft_rootx, sizeof(float4) * rx.size(), "fft twiddles"));
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->fft_P, sizeof(float4) * G, "propagator (digit-reversed order)"));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->fft_rooty, ry.data(), sizeof(float4) * ry.size(), cudaMemcpyHostToDevice, ctx->stream));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->fft_rootx, rx.data(), sizeof(float4) * rx.size(), cudaMemcpyHostToDevice, ctx->stream));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->fft_P, P.data(), sizeof(float4) * G, cudaMemcpyHostToDevice, ctx->stream));
  std::vector<int32_t> py(ny), px(nx);
  for (int i = 0; i < ny; ++i) py[i] = dif_frequency(i, ny);
  for (int i = 0; i < nx; ++i) px[i] = dif_frequency(i, nx);
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->fft_permy, sizeof(int32_t) * ny, "fft permutation"));
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->fft_permx, sizeof(int32_t) * nx, "fft permutation"));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->fft_permy, py.data(), sizeof(int32_t) * ny, cudaMemcpyHostToDevice, ctx->stream));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->fft_permx, px.data(), sizeof(int32_t) * nx, cudaMemcpyHostToDevice, ctx->stream));
  BIP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  // launch shapes: ~64 KB of rows or columns per block (at least 4 columns: whole 32-byte sectors), and a quarter as many
  // threads as butterflies per stage, so that every thread re-uses its twiddles over 4 lines (fft_stage)
  ctx->fft_lines = std::max(1, std::min(ny, tune_int("BIP_TUNE_FFT_ROW_EL", 8192) / nx));
  ctx->fft_cols = std::max(tune_int("BIP_TUNE_FFT_MINCOLS", 4), std::min(nx, tune_int("BIP_TUNE_FFT_COL_EL", 8192) / ny));
  BIP_CUDA(ctx, cudaFuncSetAttribute(k_ms_rows<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_rows_bytes(ctx->fft_lines, nx)));
  BIP_CUDA(ctx, cudaFuncSetAttribute(k_ms_rows<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_rows_bytes(ctx->fft_lines, nx)));
  const size_t smem_cols = smem_cols_bytes(ctx->fft_cols, ny);
  BIP_CUDA(ctx, cudaFuncSetAttribute(k_ms_cols, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_cols));
  BIP_CUDA(ctx, cudaFuncSetAttribute(k_ms_cols_detect, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(smem_cols + (size_t)ctx->fft_cols * ny * sizeof(float))));
  return BIP_OK;
}

// S <- post . F^-1[ P . F[ pre . S ] ] on n_cols columns (modes as in bip_multislice.cu: 0 = 1, 1 = T_j, 2 = conj T_j)
int32_t fft_slice_op(bip_ctx* ctx, float2* S, int n_cols, const float2* Tj, int pre, int conj_p, int post) {
  const int ny = ctx->g.ny, nx = ctx->g.nx;
  const int lines = ctx->fft_lines, cols = ctx->fft_cols;
  const int thr_rows = fft_threads(lines, nx), thr_cols = fft_threads(cols, ny);
  const size_t smem_rows = smem_rows_bytes(lines, nx), smem_cols = smem_cols_bytes(cols, ny);
  const int lnx = ilog2(nx), lny = ilog2(ny), lcols = ilog2(cols);
  for (int c0 = 0; c0 < n_cols; c0 += 65535) {                // gridDim.y limit
    const int nc = std::min(65535, n_cols - c0);
    float2* Sc = S + (int64_t)c0 * ny * nx;
    k_ms_rows<false><<<dim3((unsigned)((ny + lines - 1) / lines), (unsigned)nc), thr_rows, smem_rows, ctx->stream>>>(Sc, Tj, pre, ny, lnx, lines, ctx->fft_rootx);
    k_ms_cols<<<dim3((unsigned)(nx / cols), (unsigned)nc), thr_cols, smem_cols, ctx->stream>>>(Sc, ctx->fft_P, conj_p, lny, nx, lcols, ctx->fft_rooty);
    k_ms_rows<true><<<dim3((unsigned)((ny + lines - 1) / lines), (unsigned)nc), thr_rows, smem_rows, ctx->stream>>>(Sc, Tj, post, ny, lnx, lines, ctx->fft_rootx);
    BIP_CUDA(ctx, cudaGetLastError());
  }
  return BIP_OK;
}

// out[rho][ky][kx] += sum_n |F fields[rho][n]|^2 / G for n_rho scan positions x n_ch channel fields (destroys the fields)
int32_t fft_detect(bip_ctx* ctx, float2* fields, int n_rho, int n_ch, float* out) {
  const int ny = ctx->g.ny, nx = ctx->g.nx;
  const int lines = ctx->fft_lines, cols = ctx->fft_cols;
  const int thr_rows = fft_threads(lines, nx), thr_cols = fft_threads(cols, ny);
  const size_t smem_rows = smem_rows_bytes(lines, nx);
  const size_t smem_det = smem_cols_bytes(cols, ny) + (size_t)cols * ny * sizeof(float);
  const int lnx = ilog2(nx), lny = ilog2(ny), lcols = ilog2(cols);
  const int64_t G = (int64_t)ny * nx;
  for (int r0 = 0; r0 < n_rho; r0 += 4096) {                  // gridDim.y limit (n_ch fields per scan position)
    const int nr = std::min(4096, n_rho - r0);
    float2* Fc = fields + (int64_t)r0 * n_ch * G;
    for (int f0 = 0; f0 < nr * n_ch; f0 += 65535) {
      const int nf = std::min(65535, nr * n_ch - f0);
      k_ms_rows<false><<<dim3((unsigned)((ny + lines - 1) / lines), (unsigned)nf), thr_rows, smem_rows, ctx->stream>>>(Fc + (int64_t)f0 * G, nullptr, 0, ny, lnx, lines, ctx->fft_rootx);
    }
    k_ms_cols_detect<<<dim3((unsigned)(nx / cols), (unsigned)nr), thr_cols, smem_det, ctx->stream>>>(Fc, n_ch, out + (int64_t)r0 * G, (float)(1.0 / (double)G), lny, nx, lcols,
                                                                                                   ctx->fft_rooty, ctx->fft_permy, ctx->fft_permx);
    BIP_CUDA(ctx, cudaGetLastError());
  }
  return BIP_OK;
}

void fft_release(bip_ctx* ctx) {
  cudaFree(ctx->fft_rooty); cudaFree(ctx->fft_rootx); cudaFree(ctx->fft_P); cudaFree(ctx->fft_permy); cudaFree(ctx->fft_permx);
  ctx->fft_rooty = ctx->fft_rootx = ctx->fft_P = nullptr;
  ctx->fft_permy = ctx->fft_permx = nullptr;
}

}  // namespace bip
