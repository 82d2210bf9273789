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
// Butterflies are radix-8 in registers (radix 4 / 2 for the last stage), fp32 with round-to-nearest throughout and
// twiddles from a table of exact roots of unity computed in double -- every rounding is unbiased, so the column norms
// do not drift systematically (tests/test_gpu_plumbing.py measures the drift against the fp64 cuFFT route).
#include <cmath>

#include "bip_internal.h"

namespace bip {

namespace {

__device__ __forceinline__ float2 cmulf(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ float2 cmulcf(float2 a, float2 b) { return make_float2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }   // a conj(b)
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
    const float h = 0.70710678118654752440f;
    float2 a[4], b[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) { a[k] = caddf(x[k], x[k + 4]); b[k] = csubf(x[k], x[k + 4]); }
    // b_k *= w8^k, w8 = exp(-+ i pi / 4)
    b[1] = INV ? make_float2((b[1].x - b[1].y) * h, (b[1].x + b[1].y) * h) : make_float2((b[1].x + b[1].y) * h, (b[1].y - b[1].x) * h);
    b[2] = INV ? mul_pi(b[2]) : mul_mi(b[2]);
    b[3] = INV ? make_float2((-b[3].x - b[3].y) * h, (b[3].x - b[3].y) * h) : make_float2((b[3].y - b[3].x) * h, (-b[3].x - b[3].y) * h);
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

// One stage on block length L with radix R over all lines of the block.  Forward (DIF): butterfly, then twiddle
// w_L^(j m); inverse (DIT): conjugate twiddle, then inverse butterfly.  Element (line, i) lives at sm[line * pitch + i].
template <int R, bool INV>
__device__ __forceinline__ void fft_stage(float2* sm, int N, int L, int n_lines, int pitch, const float2* __restrict__ root, int tid, int nthr) {
  const int sub = L / R, per_line = N / R, tw_step = N / L;
  for (int u = tid; u < n_lines * per_line; u += nthr) {
    const int line = u / per_line, v = u - line * per_line;
    const int blk = v / sub, j = v - blk * sub;
    float2* p = sm + line * pitch + blk * L + j;
    float2 x[8];
#pragma unroll
    for (int k = 0; k < R; ++k) x[k] = p[k * sub];
    if (INV) {
#pragma unroll
      for (int m = 1; m < R; ++m) x[m] = cmulcf(x[m], __ldg(root + ((j * m * tw_step) & (N - 1))));
    }
    dft_small<R, INV>(x);
    if (!INV) {
#pragma unroll
      for (int m = 1; m < R; ++m) x[m] = cmulf(x[m], __ldg(root + ((j * m * tw_step) & (N - 1))));
    }
#pragma unroll
    for (int k = 0; k < R; ++k) p[k * sub] = x[k];
  }
}

// Whole transform of every line: radix sequence 8, 8, ..., then 4 or 2 (forward); the inverse runs the same stages backwards.
template <bool INV>
__device__ __forceinline__ void fft_lines(float2* sm, int N, int n_lines, int pitch, const float2* __restrict__ root, int tid, int nthr) {
  if (!INV) {
    int L = N;
    for (; L >= 8; L >>= 3) { fft_stage<8, false>(sm, N, L, n_lines, pitch, root, tid, nthr); __syncthreads(); }
    if (L == 4) { fft_stage<4, false>(sm, N, 4, n_lines, pitch, root, tid, nthr); __syncthreads(); }
    else if (L == 2) { fft_stage<2, false>(sm, N, 2, n_lines, pitch, root, tid, nthr); __syncthreads(); }
  } else {
    int L = N;
    while (L >= 8) L >>= 3;                                  // length left for the last forward stage: 1, 2 or 4
    if (L == 4) { fft_stage<4, true>(sm, N, 4, n_lines, pitch, root, tid, nthr); __syncthreads(); }
    else if (L == 2) { fft_stage<2, true>(sm, N, 2, n_lines, pitch, root, tid, nthr); __syncthreads(); }
    for (L = L * 8; L <= N; L <<= 3) { fft_stage<8, true>(sm, N, L, n_lines, pitch, root, tid, nthr); __syncthreads(); }
  }
}

__device__ __forceinline__ float2 apply_t(float2 v, const float2* __restrict__ T, int64_t i, int mode) {
  if (mode == 0) return v;
  float2 t = __ldg(T + i);
  if (mode == 2) t.y = -t.y;
  return cmulf(v, t);
}

// Passes 1 and 3: LINES rows per block.  tmode: 0 none, 1 multiply by T, 2 by conj T (before the forward transform /
// after the inverse one).
template <bool INV>
__global__ void __launch_bounds__(1024) k_ms_rows(float2* __restrict__ S, const float2* __restrict__ T, int tmode, int ny, int nx, int lines,
                                                  const float2* __restrict__ rootx) {
  extern __shared__ float2 sm_rows[];
  const int64_t G = (int64_t)ny * nx;
  float2* col = S + (int64_t)blockIdx.y * G;
  const int y0 = blockIdx.x * lines;
  const int n_lines = min(lines, ny - y0);
  const int tid = threadIdx.x, nthr = blockDim.x;
  for (int i = tid; i < n_lines * nx; i += nthr) {
    const int64_t g = (int64_t)y0 * nx + i;
    float2 v = col[g];
    if (!INV) v = apply_t(v, T, g, tmode);
    sm_rows[i] = v;
  }
  __syncthreads();
  fft_lines<INV>(sm_rows, nx, n_lines, nx, rootx, tid, nthr);
  for (int i = tid; i < n_lines * nx; i += nthr) {
    const int64_t g = (int64_t)y0 * nx + i;
    float2 v = sm_rows[i];
    if (INV) v = apply_t(v, T, g, tmode);
    col[g] = v;
  }
}

// Pass 2: a tile of `cols` columns (consecutive stored x positions) x ny rows per block; forward along y, spectrum
// multiply with the digit-reversed propagator table (conjugated when conj_p), inverse along y.
__global__ void __launch_bounds__(1024) k_ms_cols(float2* __restrict__ S, const float2* __restrict__ Pperm, int conj_p, int ny, int nx, int cols,
                                                  const float2* __restrict__ rooty) {
  extern __shared__ float2 sm_cols[];
  const int64_t G = (int64_t)ny * nx;
  float2* col = S + (int64_t)blockIdx.y * G;
  const int x0 = blockIdx.x * cols;
  const int pitch = ny + 1;
  const int tid = threadIdx.x, nthr = blockDim.x;
  for (int i = tid; i < ny * cols; i += nthr) {
    const int y = i / cols, c = i - y * cols;
    sm_cols[c * pitch + y] = col[(int64_t)y * nx + x0 + c];
  }
  __syncthreads();
  fft_lines<false>(sm_cols, ny, cols, pitch, rooty, tid, nthr);
  for (int i = tid; i < ny * cols; i += nthr) {
    const int y = i / cols, c = i - y * cols;
    float2 p = __ldg(Pperm + (int64_t)y * nx + x0 + c);
    if (conj_p) p.y = -p.y;
    sm_cols[c * pitch + y] = cmulf(sm_cols[c * pitch + y], p);
  }
  __syncthreads();
  fft_lines<true>(sm_cols, ny, cols, pitch, rooty, tid, nthr);
  for (int i = tid; i < ny * cols; i += nthr) {
    const int y = i / cols, c = i - y * cols;
    col[(int64_t)y * nx + x0 + c] = sm_cols[c * pitch + y];
  }
}

// Detector plane of Algorithm 3 (Alg. 1 lines 6-7): after the row pass (forward along x, stored order),
// forward FFT along y of a tile of columns of every channel field of one scan position and
//     out[rho][ky][kx] += sum_n |F psi_n|^2 / G
// at the TRUE frequency (ky, kx) of the stored position (permy / permx undo the digit reversal).  A block owns the
// (all y, its x tile) outputs of its scan position, so the read-modify-write needs no atomics.
__global__ void __launch_bounds__(1024) k_ms_cols_detect(const float2* __restrict__ F, int n_ch, float* __restrict__ out, float inv_G, int ny, int nx,
                                                         int cols, const float2* __restrict__ rooty, const int32_t* __restrict__ permy,
                                                         const int32_t* __restrict__ permx) {
  extern __shared__ float2 sm_det[];
  const int64_t G = (int64_t)ny * nx;
  const int x0 = blockIdx.x * cols, rho = blockIdx.y;
  const int pitch = ny + 1;
  float* acc = reinterpret_cast<float*>(sm_det + (size_t)cols * pitch);       // [ny * cols], element i of the tile loop
  const int tid = threadIdx.x, nthr = blockDim.x;
  for (int i = tid; i < ny * cols; i += nthr) acc[i] = 0.f;
  for (int n = 0; n < n_ch; ++n) {
    const float2* col = F + ((int64_t)rho * n_ch + n) * G;
    __syncthreads();
    for (int i = tid; i < ny * cols; i += nthr) {
      const int y = i / cols, c = i - y * cols;
      sm_det[c * pitch + y] = col[(int64_t)y * nx + x0 + c];
    }
    __syncthreads();
    fft_lines<false>(sm_det, ny, cols, pitch, rooty, tid, nthr);
    for (int i = tid; i < ny * cols; i += nthr) {
      const int y = i / cols, c = i - y * cols;
      const float2 v = sm_det[c * pitch + y];
      acc[i] += v.x * v.x + v.y * v.y;
    }
  }
  float* o = out + (int64_t)rho * G;
  for (int i = tid; i < ny * cols; i += nthr) {
    const int y = i / cols, c = i - y * cols;
    const int64_t k = (int64_t)__ldg(permy + y) * nx + __ldg(permx + x0 + c);
    o[k] += acc[i] * inv_G;
  }
}

bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

// frequency index held at stored position `pos` after the forward (DIF) transform of length N
int dif_frequency(int pos, int N) {
  if (N == 1) return 0;
  const int r = N >= 8 ? 8 : N;
  const int sub = N / r;
  return r * dif_frequency(pos % sub, sub) + pos / sub;
}

}  // namespace

bool fft_supported(const bip_ctx* ctx) {
  return is_pow2(ctx->g.ny) && is_pow2(ctx->g.nx) && ctx->g.ny >= 8 && ctx->g.nx >= 8 && ctx->g.ny <= 4096 && ctx->g.nx <= 4096;
}

int32_t fft_init(bip_ctx* ctx) {
  const int ny = ctx->g.ny, nx = ctx->g.nx;
  const int64_t G = (int64_t)ny * nx;
  std::vector<float2> ry(ny), rx(nx), P(G);
  for (int t = 0; t < ny; ++t) ry[t] = make_float2((float)std::cos(-2.0 * M_PI * t / ny), (float)std::sin(-2.0 * M_PI * t / ny));
  for (int t = 0; t < nx; ++t) rx[t] = make_float2((float)std::cos(-2.0 * M_PI * t / nx), (float)std::sin(-2.0 * M_PI * t / nx));
  // Fresnel propagator P(q) = exp(-i pi lambda dz |q|^2) / G (eq. 2; no band limit), in the stored (digit-reversed) order
  for (int py = 0; py < ny; ++py) {
    const int ky = dif_frequency(py, ny), hy = ky < (ny + 1) / 2 ? ky : ky - ny;
    const double qy = hy / ctx->g.ly;
    for (int px = 0; px < nx; ++px) {
      const int kx = dif_frequency(px, nx), hx = kx < (nx + 1) / 2 ? kx : kx - nx;
      const double qx = hx / ctx->g.lx;
      const double ph = -M_PI * ctx->g.lambda * ctx->g.dz * (qy * qy + qx * qx);
      P[(int64_t)py * nx + px] = make_float2((float)(std::cos(ph) / (double)G), (float)(std::sin(ph) / (double)G));
    }
  }
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->fft_rooty, sizeof(float2) * ny, "fft twiddles"));
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->fft_rootx, sizeof(float2) * nx, "fft twiddles"));
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->fft_P, sizeof(float2) * G, "propagator (digit-reversed order)"));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->fft_rooty, ry.data(), sizeof(float2) * ny, cudaMemcpyHostToDevice, ctx->stream));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->fft_rootx, rx.data(), sizeof(float2) * nx, cudaMemcpyHostToDevice, ctx->stream));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->fft_P, P.data(), sizeof(float2) * G, cudaMemcpyHostToDevice, ctx->stream));
  std::vector<int32_t> py(ny), px(nx);
  for (int i = 0; i < ny; ++i) py[i] = dif_frequency(i, ny);
  for (int i = 0; i < nx; ++i) px[i] = dif_frequency(i, nx);
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->fft_permy, sizeof(int32_t) * ny, "fft permutation"));
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->fft_permx, sizeof(int32_t) * nx, "fft permutation"));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->fft_permy, py.data(), sizeof(int32_t) * ny, cudaMemcpyHostToDevice, ctx->stream));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->fft_permx, px.data(), sizeof(int32_t) * nx, cudaMemcpyHostToDevice, ctx->stream));
  BIP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  // launch shapes: ~32 KB of rows per block, ~64 KB of columns per block (at least 4 columns: whole 32-byte sectors)
  ctx->fft_lines = std::max(1, std::min(ny, 4096 / nx));
  ctx->fft_cols = std::max(4, std::min(nx, 8192 / ny));
  const size_t smem_cols = (size_t)ctx->fft_cols * (ny + 1) * sizeof(float2);
  BIP_CUDA(ctx, cudaFuncSetAttribute(k_ms_cols, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_cols));
  BIP_CUDA(ctx, cudaFuncSetAttribute(k_ms_cols_detect, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(smem_cols + (size_t)ctx->fft_cols * ny * sizeof(float))));
  return BIP_OK;
}

// S <- post . F^-1[ P . F[ pre . S ] ] on n_cols columns (modes as in bip_multislice.cu: 0 = 1, 1 = T_j, 2 = conj T_j)
int32_t fft_slice_op(bip_ctx* ctx, float2* S, int n_cols, const float2* Tj, int pre, int conj_p, int post) {
  const int ny = ctx->g.ny, nx = ctx->g.nx;
  const int lines = ctx->fft_lines, cols = ctx->fft_cols;
  const int thr_rows = std::max(32, std::min(1024, lines * nx / 8)), thr_cols = std::max(32, std::min(1024, cols * ny / 8));
  const size_t smem_rows = (size_t)lines * nx * sizeof(float2), smem_cols = (size_t)cols * (ny + 1) * sizeof(float2);
  for (int c0 = 0; c0 < n_cols; c0 += 65535) {                // gridDim.y limit
    const int nc = std::min(65535, n_cols - c0);
    float2* Sc = S + (int64_t)c0 * ny * nx;
    k_ms_rows<false><<<dim3((unsigned)((ny + lines - 1) / lines), (unsigned)nc), thr_rows, smem_rows, ctx->stream>>>(Sc, Tj, pre, ny, nx, lines, ctx->fft_rootx);
    k_ms_cols<<<dim3((unsigned)(nx / cols), (unsigned)nc), thr_cols, smem_cols, ctx->stream>>>(Sc, ctx->fft_P, conj_p, ny, nx, cols, ctx->fft_rooty);
    k_ms_rows<true><<<dim3((unsigned)((ny + lines - 1) / lines), (unsigned)nc), thr_rows, smem_rows, ctx->stream>>>(Sc, Tj, post, ny, nx, lines, ctx->fft_rootx);
    BIP_CUDA(ctx, cudaGetLastError());
  }
  return BIP_OK;
}

// out[rho][ky][kx] += sum_n |F fields[rho][n]|^2 / G for n_rho scan positions x n_ch channel fields (destroys the fields)
int32_t fft_detect(bip_ctx* ctx, float2* fields, int n_rho, int n_ch, float* out) {
  const int ny = ctx->g.ny, nx = ctx->g.nx;
  const int lines = ctx->fft_lines, cols = ctx->fft_cols;
  const int thr_rows = std::max(32, std::min(1024, lines * nx / 8)), thr_cols = std::max(32, std::min(1024, cols * ny / 8));
  const size_t smem_rows = (size_t)lines * nx * sizeof(float2);
  const size_t smem_det = (size_t)cols * (ny + 1) * sizeof(float2) + (size_t)cols * ny * sizeof(float);
  const int64_t G = (int64_t)ny * nx;
  for (int r0 = 0; r0 < n_rho; r0 += 4096) {                  // gridDim.y limit (n_ch fields per scan position)
    const int nr = std::min(4096, n_rho - r0);
    float2* Fc = fields + (int64_t)r0 * n_ch * G;
    for (int f0 = 0; f0 < nr * n_ch; f0 += 65535) {
      const int nf = std::min(65535, nr * n_ch - f0);
      k_ms_rows<false><<<dim3((unsigned)((ny + lines - 1) / lines), (unsigned)nf), thr_rows, smem_rows, ctx->stream>>>(Fc + (int64_t)f0 * G, nullptr, 0, ny, nx, lines, ctx->fft_rootx);
    }
    k_ms_cols_detect<<<dim3((unsigned)(nx / cols), (unsigned)nr), thr_cols, smem_det, ctx->stream>>>(Fc, n_ch, out + (int64_t)r0 * G, (float)(1.0 / (double)G), ny, nx, cols,
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
