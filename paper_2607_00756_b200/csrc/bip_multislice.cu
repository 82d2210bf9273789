// Slice-by-slice multislice of the parent columns: S1 ADVANCETO (eq. 6) and S2 build / PEELTO
// (eq. 12).  cuFFT does the 2-D transforms (plumbing, timed separately from the contraction).
#include <cmath>
#include <map>

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

// S[p][i] *= (conj ? conj(F[i]) : F[i]) for a batch of columns; F is a single [G] field (T_j, or P/G).
__global__ void k_mul_field(float2* __restrict__ S, const float2* __restrict__ F, int64_t G, int conj_f) {
  const int64_t p = blockIdx.y;
  float2* col = S + p * G;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < G; i += (int64_t)gridDim.x * blockDim.x) {
    float2 f = F[i];
    if (conj_f) f.y = -f.y;
    col[i] = cmul(col[i], f);
  }
}

struct PlanCache {
  std::map<int, cufftHandle> plans;
};
std::map<const bip_ctx*, PlanCache>& plan_caches() {
  static std::map<const bip_ctx*, PlanCache> m;
  return m;
}

int32_t get_plan(bip_ctx* ctx, int batch, cufftHandle* out) {
  auto& pc = plan_caches()[ctx];
  auto it = pc.plans.find(batch);
  if (it != pc.plans.end()) { *out = it->second; return BIP_OK; }
  cufftHandle h;
  int n[2] = {ctx->g.ny, ctx->g.nx};
  cufftResult r = cufftPlanMany(&h, 2, n, nullptr, 1, ctx->g.ny * ctx->g.nx, nullptr, 1, ctx->g.ny * ctx->g.nx, CUFFT_C2C, batch);
  if (r != CUFFT_SUCCESS) return fail(ctx, r == CUFFT_ALLOC_FAILED ? BIP_ERR_OOM : BIP_ERR_CUDA, "cufftPlanMany(%dx%d, batch %d) failed: %d", ctx->g.ny, ctx->g.nx, batch, (int)r);
  r = cufftSetStream(h, ctx->stream);
  if (r != CUFFT_SUCCESS) return fail(ctx, BIP_ERR_CUDA, "cufftSetStream failed: %d", (int)r);
  pc.plans[batch] = h;
  *out = h;
  return BIP_OK;
}

int32_t fft_cols(bip_ctx* ctx, float2* S, int n_cols, int dir) {
  const int64_t G = (int64_t)ctx->g.ny * ctx->g.nx;
  const int chunk = ctx->plan_batch;
  for (int c0 = 0; c0 < n_cols; c0 += chunk) {
    const int nb = std::min(chunk, n_cols - c0);
    cufftHandle h;
    BIP_TRY(get_plan(ctx, nb, &h));
    cufftComplex* p = reinterpret_cast<cufftComplex*>(S + (int64_t)c0 * G);
    cufftResult r = cufftExecC2C(h, p, p, dir);
    if (r != CUFFT_SUCCESS) return fail(ctx, BIP_ERR_CUDA, "cufftExecC2C failed: %d", (int)r);
  }
  return BIP_OK;
}

int32_t mul_field(bip_ctx* ctx, float2* S, int n_cols, const float2* F, int conj_f) {
  const int64_t G = (int64_t)ctx->g.ny * ctx->g.nx;
  dim3 grid((unsigned)std::min<int64_t>((G + 255) / 256, 1024), (unsigned)n_cols);
  // gridDim.y is limited to 65535 columns, far above any parent count used here
  k_mul_field<<<grid, 256, 0, ctx->stream>>>(S, F, G, conj_f);
  BIP_CUDA(ctx, cudaGetLastError());
  return BIP_OK;
}

}  // namespace

void ms_release(bip_ctx* ctx) {
  auto it = plan_caches().find(ctx);
  if (it == plan_caches().end()) return;
  for (auto& kv : it->second.plans) cufftDestroy(kv.second);
  plan_caches().erase(it);
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
  std::vector<float2> P(G);
  for (int ky = 0; ky < ny; ++ky) {
    const int hy = ky < (ny + 1) / 2 ? ky : ky - ny;
    const double qy = hy / ctx->g.ly;
    for (int kx = 0; kx < nx; ++kx) {
      const int hx = kx < (nx + 1) / 2 ? kx : kx - nx;
      const double qx = hx / ctx->g.lx;
      const double ph = -M_PI * ctx->g.lambda * ctx->g.dz * (qy * qy + qx * qx);
      P[(int64_t)ky * nx + kx] = make_float2((float)(std::cos(ph) / (double)G), (float)(std::sin(ph) / (double)G));
    }
  }
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->P_dev, sizeof(float2) * G, "propagator"));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->P_dev, P.data(), sizeof(float2) * G, cudaMemcpyHostToDevice, ctx->stream));
  BIP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  // cuFFT batch: at most 256 MB of columns per call
  const int64_t col_bytes = G * (int64_t)sizeof(float2);
  ctx->plan_batch = (int)std::max<int64_t>(1, std::min<int64_t>(std::max(ctx->n_p1, ctx->n_p2), (256ll << 20) / col_bytes));
  ctx->plan_ok = true;
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
  const int64_t G = (int64_t)ctx->g.ny * ctx->g.nx;
  const float2* Tj = ctx->T_dev + (int64_t)j * G;
  if (dir > 0) {                     // S <- P[T_j S]
    BIP_TRY(mul_field(ctx, ctx->S1, ctx->n_p1, Tj, 0));
    BIP_TRY(fft_cols(ctx, ctx->S1, ctx->n_p1, CUFFT_FORWARD));
    BIP_TRY(mul_field(ctx, ctx->S1, ctx->n_p1, ctx->P_dev, 0));
    BIP_TRY(fft_cols(ctx, ctx->S1, ctx->n_p1, CUFFT_INVERSE));
  } else {                           // inverse: S <- T_j* P*[S]   (|T| = |P| = 1)
    BIP_TRY(fft_cols(ctx, ctx->S1, ctx->n_p1, CUFFT_FORWARD));
    BIP_TRY(mul_field(ctx, ctx->S1, ctx->n_p1, ctx->P_dev, 1));
    BIP_TRY(fft_cols(ctx, ctx->S1, ctx->n_p1, CUFFT_INVERSE));
    BIP_TRY(mul_field(ctx, ctx->S1, ctx->n_p1, Tj, 1));
  }
  return BIP_OK;
}

int32_t ms_step_S2(bip_ctx* ctx, int32_t j, int dir) {
  const int64_t G = (int64_t)ctx->g.ny * ctx->g.nx;
  const float2* Tj = ctx->T_dev + (int64_t)j * G;
  if (dir < 0) {                     // build / un-peel: S <- T_j P[S]   (absorbs slice j)
    BIP_TRY(fft_cols(ctx, ctx->S2, ctx->n_p2, CUFFT_FORWARD));
    BIP_TRY(mul_field(ctx, ctx->S2, ctx->n_p2, ctx->P_dev, 0));
    BIP_TRY(fft_cols(ctx, ctx->S2, ctx->n_p2, CUFFT_INVERSE));
    BIP_TRY(mul_field(ctx, ctx->S2, ctx->n_p2, Tj, 0));
  } else {                           // peel: S <- P*[T_j* S]            (sheds slice j)
    BIP_TRY(mul_field(ctx, ctx->S2, ctx->n_p2, Tj, 1));
    BIP_TRY(fft_cols(ctx, ctx->S2, ctx->n_p2, CUFFT_FORWARD));
    BIP_TRY(mul_field(ctx, ctx->S2, ctx->n_p2, ctx->P_dev, 1));
    BIP_TRY(fft_cols(ctx, ctx->S2, ctx->n_p2, CUFFT_INVERSE));
  }
  return BIP_OK;
}

}  // namespace bip
