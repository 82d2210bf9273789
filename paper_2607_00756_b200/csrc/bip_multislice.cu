// Slice-by-slice multislice of the parent columns: S1 ADVANCETO (eq. 6) and S2 build / PEELTO
// (eq. 12).  cuFFT does the 2-D transforms (plumbing, timed separately from the contraction).
#include <cmath>
#include <cstring>

#include "bip_internal.h"

namespace bip {

namespace {

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// S[p][ry][rx] = exp(sign 2 pi i h_p.r/N) from the exact root-of-unity tables.
__global__ void k_plane_waves(float2* __restrict__ S, const int32_t* __restrict__ h, int ny, int nx,
                              const float2* __restrict__ rooty, const float2* __restrict__ rootx, int sign) {
  const int p = blockIdx.y;
  const int hy = ((h[2 * p] % ny) + ny) % ny, hx = ((h[2 * p + 1] % nx) + nx) % nx;
  const int64_t G = (int64_t)ny * nx;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < G; i += (int64_t)gridDim.x * blockDim.x) {
    const int ry = (int)(i / nx), rx = (int)(i % nx);
    float2 v = cmul(rooty[(int)(((int64_t)hy * ry) % ny)], rootx[(int)(((int64_t)hx * rx) % nx)]);
    if (sign < 0) v.y = -v.y;
    S[(int64_t)p * G + i] = v;
  }
}

// max | |T|^2 - 1 | over all pixels of all slices (non-negative floats order like their bit patterns)
__global__ void k_modulus_deviation(const float2* __restrict__ T, int64_t n, unsigned int* __restrict__ out) {
  float m = 0.f;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const float2 t = T[i];
    const float d = fabsf(t.x * t.x + t.y * t.y - 1.f);
    m = fmaxf(m, d == d ? d : 3.0e38f);               // NaN counts as a violation
  }
#pragma unroll
  for (int o = 16; o; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) atomicMax(out, __float_as_uint(m));
}

// The cuFFT route (grids that are not powers of two, and the A/B reference of the native slice step).
// cuFFT's single-precision C2C loses ~3e-7 of the norm^2 per forward+inverse pair, systematically (measured on
// B200 in round 1; tests/test_gpu_plumbing.py re-measures the drift of both variants); over tens of slices that alone breaks the 1e-6 summed-intensity bound.  The slice
// steps therefore run in double precision (Z2Z) on a chunk workspace and the columns are stored back as c64:
// the only rounding per slice is one unbiased round-to-nearest of the result.

// W[p][i] = (double) S[p][i] * (mode 0: 1, 1: T[i], 2: conj T[i])
__global__ void k_load_cols(double2* __restrict__ W, const float2* __restrict__ S, const float2* __restrict__ T,
                            int64_t G, int mode) {
  const int64_t p = blockIdx.y;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < G; i += (int64_t)gridDim.x * blockDim.x) {
    const float2 s = S[p * G + i];
    double2 v = make_double2(s.x, s.y);
    if (mode) {
      const float2 t = T[i];
      const double tr = t.x, ti = mode == 2 ? -(double)t.y : (double)t.y;
      v = make_double2(v.x * tr - v.y * ti, v.x * ti + v.y * tr);
    }
    W[p * G + i] = v;
  }
}

// W[p][i] *= (conj ? conj(P[i]) : P[i])   (P carries the 1/G of the unnormalised transform pair)
__global__ void k_mul_prop(double2* __restrict__ W, const double2* __restrict__ P, int64_t G, int conj_p) {
  const int64_t p = blockIdx.y;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < G; i += (int64_t)gridDim.x * blockDim.x) {
    const double2 f = P[i];
    const double fi = conj_p ? -f.y : f.y;
    const double2 v = W[p * G + i];
    W[p * G + i] = make_double2(v.x * f.x - v.y * fi, v.x * fi + v.y * f.x);
  }
}

// S[p][i] = (float) (W[p][i] * (mode 0: 1, 1: T[i], 2: conj T[i]))
__global__ void k_store_cols(float2* __restrict__ S, const double2* __restrict__ W, const float2* __restrict__ T,
                             int64_t G, int mode) {
  const int64_t p = blockIdx.y;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < G; i += (int64_t)gridDim.x * blockDim.x) {
    double2 v = W[p * G + i];
    if (mode) {
      const float2 t = T[i];
      const double tr = t.x, ti = mode == 2 ? -(double)t.y : (double)t.y;
      v = make_double2(v.x * tr - v.y * ti, v.x * ti + v.y * tr);
    }
    S[p * G + i] = make_float2((float)v.x, (float)v.y);
  }
}

int32_t get_plan(bip_ctx* ctx, int batch, cufftHandle* out) {
  auto it = ctx->plans.find(batch);
  if (it != ctx->plans.end()) { *out = it->second; return BIP_OK; }
  cufftHandle h;
  int n[2] = {ctx->g.ny, ctx->g.nx};
  cufftResult r = cufftPlanMany(&h, 2, n, nullptr, 1, ctx->g.ny * ctx->g.nx, nullptr, 1, ctx->g.ny * ctx->g.nx, CUFFT_Z2Z, batch);
  if (r != CUFFT_SUCCESS) return fail(ctx, r == CUFFT_ALLOC_FAILED ? BIP_ERR_OOM : BIP_ERR_CUDA, "cufftPlanMany(%dx%d, batch %d) failed: %d", ctx->g.ny, ctx->g.nx, batch, (int)r);
  r = cufftSetStream(h, ctx->stream);
  if (r != CUFFT_SUCCESS) return fail(ctx, BIP_ERR_CUDA, "cufftSetStream failed: %d", (int)r);
  ctx->plans[batch] = h;
  *out = h;
  return BIP_OK;
}

// One unitary slice operation on all columns of S:  S <- post . F^-1[ Pspec . F[ pre . S ] ]
//   pre / post: 0 = identity, 1 = T_j, 2 = conj T_j ;  conj_p: multiply the spectrum by conj(P) instead of P
int32_t slice_op(bip_ctx* ctx, float2* S, int n_cols, const float2* Tj, int pre, int conj_p, int post) {
  if (ctx->fft_native) return fft_slice_op(ctx, S, n_cols, Tj, pre, conj_p, post);
  BIP_TRY(fft_flush(ctx));                      // the backend was switched in the middle of a sequence
  const int64_t G = (int64_t)ctx->g.ny * ctx->g.nx;
  const int chunk = ctx->plan_batch;
  if (!ctx->ms_work) BIP_TRY(dev_alloc(ctx, &ctx->ms_work, (size_t)ctx->plan_batch * G * sizeof(double2), "multislice workspace"));
  double2* W = reinterpret_cast<double2*>(ctx->ms_work);
  const double2* P = reinterpret_cast<const double2*>(ctx->P_dev);
  for (int c0 = 0; c0 < n_cols; c0 += chunk) {
    const int nb = std::min(chunk, n_cols - c0);
    cufftHandle h;
    BIP_TRY(get_plan(ctx, nb, &h));
    float2* Sc = S + (int64_t)c0 * G;
    dim3 grid((unsigned)std::min<int64_t>((G + 255) / 256, 2048), (unsigned)nb);
    k_load_cols<<<grid, 256, 0, ctx->stream>>>(W, Sc, Tj, G, pre);
    cufftResult r = cufftExecZ2Z(h, reinterpret_cast<cufftDoubleComplex*>(W), reinterpret_cast<cufftDoubleComplex*>(W), CUFFT_FORWARD);
    if (r != CUFFT_SUCCESS) return fail(ctx, BIP_ERR_CUDA, "cufftExecZ2Z failed: %d", (int)r);
    k_mul_prop<<<grid, 256, 0, ctx->stream>>>(W, P, G, conj_p);
    r = cufftExecZ2Z(h, reinterpret_cast<cufftDoubleComplex*>(W), reinterpret_cast<cufftDoubleComplex*>(W), CUFFT_INVERSE);
    if (r != CUFFT_SUCCESS) return fail(ctx, BIP_ERR_CUDA, "cufftExecZ2Z failed: %d", (int)r);
    k_store_cols<<<grid, 256, 0, ctx->stream>>>(Sc, W, Tj, G, post);
    BIP_CUDA(ctx, cudaGetLastError());
  }
  return BIP_OK;
}

// out[f / n_ch][i] += |W[f][i]|^2 / G summed over the n_ch fields of a scan position (cuFFT route of ms_detect)
__global__ void k_detect_accum(const double2* __restrict__ W, int n_ch, float* __restrict__ out, double inv_G, int64_t G) {
  const int64_t rho = blockIdx.y;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < G; i += (int64_t)gridDim.x * blockDim.x) {
    double a = 0.0;
    for (int n = 0; n < n_ch; ++n) {
      const double2 v = W[(rho * n_ch + n) * G + i];
      a += v.x * v.x + v.y * v.y;
    }
    out[rho * G + i] += (float)(a * inv_G);
  }
}

}  // namespace

int32_t ms_exit_step(bip_ctx* ctx, float2* fields, int n, int32_t j) {
  const float2* Tj = ctx->T_dev + (int64_t)j * ctx->g.ny * ctx->g.nx;
  return slice_op(ctx, fields, n, Tj, /*pre=*/1, /*conj_p=*/0, /*post=*/0);      // psi <- P[T_j psi] (eq. 6 on a wavefield)
}

int32_t ms_flush(bip_ctx* ctx) { return fft_flush(ctx); }   // the cuFFT route never leaves a pass owing

int32_t ms_detect(bip_ctx* ctx, float2* fields, int n_rho, int n_ch, float* out) {
  if (ctx->fft_native) return fft_detect(ctx, fields, n_rho, n_ch, out);
  BIP_TRY(fft_flush(ctx));
  const int64_t G = (int64_t)ctx->g.ny * ctx->g.nx;
  if (!ctx->ms_work) BIP_TRY(dev_alloc(ctx, &ctx->ms_work, (size_t)ctx->plan_batch * G * sizeof(double2), "multislice workspace"));
  double2* W = reinterpret_cast<double2*>(ctx->ms_work);
  const int rho_chunk = std::max(1, ctx->plan_batch / n_ch);
  if (n_ch > ctx->plan_batch) return fail(ctx, BIP_ERR_UNSUPPORTED, "Algorithm 3 on the cuFFT route: %d channels exceed the transform batch %d", n_ch, ctx->plan_batch);
  for (int r0 = 0; r0 < n_rho; r0 += rho_chunk) {
    const int nr = std::min(rho_chunk, n_rho - r0), nf = nr * n_ch;
    cufftHandle h;
    BIP_TRY(get_plan(ctx, nf, &h));
    dim3 grid((unsigned)std::min<int64_t>((G + 255) / 256, 2048), (unsigned)nf);
    k_load_cols<<<grid, 256, 0, ctx->stream>>>(W, fields + (int64_t)r0 * n_ch * G, nullptr, G, 0);
    cufftResult r = cufftExecZ2Z(h, reinterpret_cast<cufftDoubleComplex*>(W), reinterpret_cast<cufftDoubleComplex*>(W), CUFFT_FORWARD);
    if (r != CUFFT_SUCCESS) return fail(ctx, BIP_ERR_CUDA, "cufftExecZ2Z failed: %d", (int)r);
    k_detect_accum<<<dim3(grid.x, (unsigned)nr), 256, 0, ctx->stream>>>(W, n_ch, out + (int64_t)r0 * G, 1.0 / (double)G, G);
    BIP_CUDA(ctx, cudaGetLastError());
  }
  return BIP_OK;
}

void ms_release(bip_ctx* ctx) {
  fft_release(ctx);
  for (auto& kv : ctx->plans) cufftDestroy(kv.second);
  ctx->plans.clear();
}

int32_t ms_init(bip_ctx* ctx) {
  const int ny = ctx->g.ny, nx = ctx->g.nx;
  const int64_t G = (int64_t)ny * nx;
  // exact roots of unity in double, rounded once to float
  std::vector<float2> ry(ny), rx(nx);
  for (int k = 0; k < ny; ++k) ry[k] = make_float2((float)std::cos(2.0 * M_PI * k / ny), (float)std::sin(2.0 * M_PI * k / ny));
  for (int k = 0; k < nx; ++k) rx[k] = make_float2((float)std::cos(2.0 * M_PI * k / nx), (float)std::sin(2.0 * M_PI * k / nx));
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->rooty_dev, sizeof(float2) * ny, "root table"));
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->rootx_dev, sizeof(float2) * nx, "root table"));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->rooty_dev, ry.data(), sizeof(float2) * ny, cudaMemcpyHostToDevice, ctx->stream));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->rootx_dev, rx.data(), sizeof(float2) * nx, cudaMemcpyHostToDevice, ctx->stream));
  // Fresnel propagator P(q) = exp(-i pi lambda dz |q|^2) (eq. 2), no band limit, with the 1/G of the
  // unnormalised cuFFT round trip folded in.
  std::vector<double2> P(G);
  for (int ky = 0; ky < ny; ++ky) {
    const int hy = ky < (ny + 1) / 2 ? ky : ky - ny;
    const double qy = hy / ctx->g.ly;
    for (int kx = 0; kx < nx; ++kx) {
      const int hx = kx < (nx + 1) / 2 ? kx : kx - nx;
      const double qx = hx / ctx->g.lx;
      const double ph = -M_PI * ctx->g.lambda * ctx->g.dz * (qy * qy + qx * qx);
      P[(int64_t)ky * nx + kx] = make_double2(std::cos(ph) / (double)G, std::sin(ph) / (double)G);
    }
  }
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->P_dev, sizeof(double2) * G, "propagator"));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->P_dev, P.data(), sizeof(double2) * G, cudaMemcpyHostToDevice, ctx->stream));
  BIP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  // cuFFT batch: at most 512 MB of double-precision workspace per call
  const int64_t col_bytes = G * (int64_t)sizeof(double2);
  ctx->plan_batch = (int)std::max<int64_t>(1, std::min<int64_t>(std::max(ctx->n_p1, ctx->n_p2), (512ll << 20) / col_bytes));
  ctx->plan_ok = true;
  // power-of-two grids take the native fused slice step (bip_fft.cu); any other grid the cuFFT route above
  if (fft_supported(ctx)) { BIP_TRY(fft_init(ctx)); ctx->fft_native = true; }
  return BIP_OK;
}

int32_t ms_max_modulus_deviation(bip_ctx* ctx, const float2* T, int64_t n, float* out) {
  unsigned int* d = nullptr;
  BIP_TRY(dev_alloc(ctx, (void**)&d, sizeof(unsigned int), "modulus check"));
  cudaMemsetAsync(d, 0, sizeof(unsigned int), ctx->stream);
  k_modulus_deviation<<<(unsigned)std::min<int64_t>((n + 255) / 256, 4096), 256, 0, ctx->stream>>>(T, n, d);
  unsigned int bits = 0;
  cudaError_t e = cudaMemcpyAsync(&bits, d, sizeof bits, cudaMemcpyDeviceToHost, ctx->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
  cudaFree(d);
  if (e != cudaSuccess) { cudaGetLastError(); return fail(ctx, BIP_ERR_CUDA, "modulus check: %s", cudaGetErrorString(e)); }
  std::memcpy(out, &bits, sizeof bits);
  return BIP_OK;
}

int32_t ms_plane_waves(bip_ctx* ctx, float2* S, const int32_t* h_dev, int32_t n, int sign) {
  const int64_t G = (int64_t)ctx->g.ny * ctx->g.nx;
  dim3 grid((unsigned)std::min<int64_t>((G + 255) / 256, 1024), (unsigned)n);
  k_plane_waves<<<grid, 256, 0, ctx->stream>>>(S, h_dev, ctx->g.ny, ctx->g.nx, ctx->rooty_dev, ctx->rootx_dev, sign);
  BIP_CUDA(ctx, cudaGetLastError());
  return BIP_OK;
}

int32_t ms_step_S1(bip_ctx* ctx, int32_t j, int dir) {
  const float2* Tj = ctx->T_dev + (int64_t)j * ctx->g.ny * ctx->g.nx;
  if (dir > 0) return slice_op(ctx, ctx->S1, ctx->n_p1, Tj, /*pre=*/1, /*conj_p=*/0, /*post=*/0);   // S <- P[T_j S]   (eq. 6)
  return slice_op(ctx, ctx->S1, ctx->n_p1, Tj, 0, 1, 2);                                             // S <- T_j* P*[S]
}

int32_t ms_step_S2(bip_ctx* ctx, int32_t j, int dir) {
  const float2* Tj = ctx->T_dev + (int64_t)j * ctx->g.ny * ctx->g.nx;
  if (dir < 0) return slice_op(ctx, ctx->S2, ctx->n_p2, Tj, 0, 0, 1);   // build / un-peel: S <- T_j P[S]  (eq. 12)
  return slice_op(ctx, ctx->S2, ctx->n_p2, Tj, 2, 1, 0);                // peel: S <- P*[T_j* S]
}

}  // namespace bip
