// NEXT-4: S1 focal back-propagation to the scattering-centroid plane (section 2.2.3.1; reading c20 of
// DESIGN.md): the de-tilted parent envelopes on the padded window Omega+ are carried back to the centroid plane by a
// Fresnel step with the transfer function of their own carrier, interpolated there (eq. 15 / eq. 11), carried forward
// again beam by beam, re-tilted and cropped to the W x W window -- the R1^T operand of the probe GEMM.
//
//   k_slice_strength     m_j = sum_r |T_j(r) - 1|^2 (once per transmission set; centroid depths follow on the host)
//   k_window_fresnel     one block per window: 2-D FFT of the W_p x W_p envelope in shared memory (rows, transpose, rows),
//                        x exp(-i pi lambda d |q_w + q_h|^2) / W_p^2, inverse transform; double-float constants as in bip_fft.cu
//   k_env_colmax         row scales of the operand: power of two above max_b |E_b(s)|
//   k_env_to_r1t_sliced  re-tilt, crop Omega+ -> Omega, split into the sliced K-major operand R1^T[s][b]
#include <cmath>

#include "bip_internal.h"
#include "bip_fft.cuh"

namespace bip {

namespace {

using namespace fftdev;

__global__ void k_slice_strength(const float2* __restrict__ T, int64_t G, double* __restrict__ m) {
  const int j = blockIdx.y;
  double a = 0.0;
  for (int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; i < G; i += (int64_t)gridDim.x * blockDim.x) {
    const float2 t = T[(int64_t)j * G + i];
    const double dr = (double)t.x - 1.0, di = (double)t.y;
    a += dr * dr + di * di;
  }
#pragma unroll
  for (int o = 16; o; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
  if ((threadIdx.x & 31) == 0) atomicAdd(m + j, a);
}

// E[e] <- F_w^-1[ exp(-i pi lambda d |q_w + q_h|^2) F_w E[e] ] for window e; its carrier is beam h[e % n_beams].
// pld = pi lambda d (signed); q_w = k / (W_p pixel); stored positions after the forward transforms are digit-reversed (perm).
__global__ void __launch_bounds__(256, 2) k_window_fresnel(float2* __restrict__ E, const int32_t* __restrict__ h, int n_beams, int lW, double pld,
                                                         double inv_ly, double inv_lx, double inv_wy, double inv_wx,
                                                         const float4* __restrict__ root, const int32_t* __restrict__ perm) {
  extern __shared__ float2 sm_win[];
  const int Wp = 1 << lW, pitch = pad_len(Wp) + 1;
  float4* ea = reinterpret_cast<float4*>(sm_win + (size_t)Wp * pitch);     // [Wp] phase factors along y (hi, lo), with the 1 / W_p^2
  float4* eb = ea + Wp;                                                     // [Wp] along x
  const int tid = threadIdx.x, nthr = blockDim.x;
  float2* win = E + (int64_t)blockIdx.x * Wp * Wp;
  const int b = blockIdx.x % n_beams;
  const double qhy = (double)h[2 * b] * inv_ly, qhx = (double)h[2 * b + 1] * inv_lx;
  for (int i = tid; i < 2 * Wp; i += nthr) {
    const int pos = i & (Wp - 1), k = perm[pos], ks = k < Wp / 2 ? k : k - Wp;
    const bool is_y = i < Wp;
    const double q = (double)ks * (is_y ? inv_wy : inv_wx) + (is_y ? qhy : qhx);
    double sn, cs;
    sincos(-pld * q * q, &sn, &cs);
    const double sc = is_y ? 1.0 / ((double)Wp * (double)Wp) : 1.0;
    const float hr = (float)(cs * sc), hi = (float)(sn * sc);
    (is_y ? ea : eb)[pos] = make_float4(hr, hi, (float)(cs * sc - (double)hr), (float)(sn * sc - (double)hi));
  }
  for (int i = tid; i < Wp * Wp; i += nthr) sm_win[(i >> lW) * pitch + pad_idx(i & (Wp - 1))] = win[i];
  __syncthreads();
  auto transpose = [&]() {
    for (int i = tid; i < Wp * Wp; i += nthr) {
      const int r = i >> lW, c = i & (Wp - 1);
      if (r < c) {
        float2* p = sm_win + r * pitch + pad_idx(c);
        float2* q = sm_win + c * pitch + pad_idx(r);
        const float2 t = *p; *p = *q; *q = t;
      }
    }
    __syncthreads();
  };
  fft_lines<false>(sm_win, lW, Wp, pitch, root, tid, nthr);                // along x
  transpose();
  fft_lines<false>(sm_win, lW, Wp, pitch, root, tid, nthr);                // along y: element [x'][y']
  for (int i = tid; i < Wp * Wp; i += nthr) {
    const int xs = i >> lW, ys = i & (Wp - 1);
    float2* p = sm_win + xs * pitch + pad_idx(ys);
    *p = cmul_dd(cmul_dd(*p, ea[ys]), eb[xs]);
  }
  __syncthreads();
  fft_lines<true>(sm_win, lW, Wp, pitch, root, tid, nthr);
  transpose();
  fft_lines<true>(sm_win, lW, Wp, pitch, root, tid, nthr);
  for (int i = tid; i < Wp * Wp; i += nthr) win[i] = sm_win[(i >> lW) * pitch + pad_idx(i & (Wp - 1))];
}

// scale[s] = power of two above max_b |Env[b][s_pad]| for the W x W centre of the padded window
__global__ void k_env_colmax(const float2* __restrict__ Env, int n_beams, int w, int Wp, float* __restrict__ scale) {
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= w * w) return;
  const int o = (Wp - w) / 2, sp = (s / w + o) * Wp + (s % w) + o;
  float m = 0.f;
  for (int b = 0; b < n_beams; ++b) {
    const float2 v = Env[(int64_t)b * Wp * Wp + sp];
    m = fmaxf(m, v.x * v.x + v.y * v.y);
  }
  scale[s] = sl_pow2_scale(1.001f * sqrtf(m));
}

// R1^T[s][b] = exp(+2 pi i h_b.r/N) Env[b][s_pad], r = (origin + s) mod N: rows = window pixels, k = aperture beams.
// thread = (row s, group of 8 consecutive beams); lanes run over consecutive s (coalesced reads of Env, 128-byte stores).
__global__ void __launch_bounds__(256) k_env_to_r1t_sliced(const float2* __restrict__ Env, const int32_t* __restrict__ bh, int n_beams, int oy, int ox,
                                                           int w, int Wp, int ny, int nx, const float2* __restrict__ rooty,
                                                           const float2* __restrict__ rootx, Sliced out, int atom) {
  const int w2 = w * w;
  const int s = blockIdx.x * 32 + threadIdx.x, g = blockIdx.y * 8 + threadIdx.y;
  if (s >= w2 || g >= 2 * out.ksteps) return;
  const int sy = s / w, sx = s - sy * w, o = (Wp - w) / 2;
  int ry = oy + sy; if (ry >= ny) ry -= ny;
  int rx = ox + sx; if (rx >= nx) rx -= nx;
  const int sp = (sy + o) * Wp + sx + o;
  float re[8], im[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    const int b = g * 8 + j;
    re[j] = 0.f; im[j] = 0.f;
    if (b < n_beams) {
      const int hyp = ((bh[2 * b] % ny) + ny) % ny, hxp = ((bh[2 * b + 1] % nx) + nx) % nx;
      const float2 ty = rooty[(hyp * ry) % ny], tx = rootx[(hxp * rx) % nx];
      const float2 t = make_float2(ty.x * tx.x - ty.y * tx.y, ty.x * tx.y + ty.y * tx.x);
      const float2 v = Env[(int64_t)b * Wp * Wp + sp];
      re[j] = v.x * t.x - v.y * t.y; im[j] = v.x * t.y + v.y * t.x;
    }
  }
  sl_store_group(out, atom, s, g, re, im, 1.f / out.scale[(int64_t)atom * out.scale_batch_stride + s]);
}

}  // namespace

int32_t focal_padded_window(int32_t w) { int p = 1; while (p < w + 16) p <<= 1; return p; }

// m_j = sum_r |T_j - 1|^2 for every slice -> centroid distance d_i of every plane (host, double), reading c20
int32_t focal_init(bip_ctx* ctx) {
  const int nz = ctx->g.nz;
  const int64_t G = (int64_t)ctx->g.ny * ctx->g.nx;
  double* m_dev = nullptr;
  BIP_TRY(dev_alloc(ctx, (void**)&m_dev, sizeof(double) * nz, "slice strengths"));
  cudaMemsetAsync(m_dev, 0, sizeof(double) * nz, ctx->stream);
  k_slice_strength<<<dim3((unsigned)std::min<int64_t>((G + 255) / 256, 512), (unsigned)nz), 256, 0, ctx->stream>>>(ctx->T_dev, G, m_dev);
  std::vector<double> m(nz);
  cudaError_t e = cudaMemcpyAsync(m.data(), m_dev, sizeof(double) * nz, cudaMemcpyDeviceToHost, ctx->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
  cudaFree(m_dev);
  if (e != cudaSuccess) { cudaGetLastError(); return fail(ctx, BIP_ERR_CUDA, "slice strengths: %s", cudaGetErrorString(e)); }
  ctx->focal_d.assign(nz + 1, 0.0);
  double sm = 0.0, smz = 0.0;
  for (int i = 1; i <= nz; ++i) {
    sm += m[i - 1]; smz += m[i - 1] * ((i - 1) + 0.5) * ctx->g.dz;
    ctx->focal_d[i] = sm > 0.0 ? i * ctx->g.dz - smz / sm : 0.0;
  }
  return BIP_OK;
}

static int32_t window_tables(bip_ctx* ctx, int Wp, const float4** root, const int32_t** perm) {
  auto it = ctx->focal_tables.find(Wp);
  if (it == ctx->focal_tables.end()) {
    std::vector<float4> r = make_twiddle_table(Wp);
    std::vector<int32_t> p(Wp);
    for (int t = 0; t < Wp; ++t) p[t] = dif_frequency(t, Wp);
    void* rd = nullptr; void* pd = nullptr;
    BIP_TRY(dev_alloc(ctx, &rd, sizeof(float4) * r.size(), "window twiddles"));
    BIP_TRY(dev_alloc(ctx, &pd, sizeof(int32_t) * Wp, "window permutation"));
    BIP_CUDA(ctx, cudaMemcpyAsync(rd, r.data(), sizeof(float4) * r.size(), cudaMemcpyHostToDevice, ctx->stream));
    BIP_CUDA(ctx, cudaMemcpyAsync(pd, p.data(), sizeof(int32_t) * Wp, cudaMemcpyHostToDevice, ctx->stream));
    BIP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    it = ctx->focal_tables.emplace(Wp, std::make_pair(rd, pd)).first;
    const int Wmax = ctx->focal_tables.rbegin()->first;                 // opt in for the largest window seen so far
    const size_t smem = (size_t)Wmax * (pad_len(Wmax) + 1) * sizeof(float2) + 2 * (size_t)Wmax * sizeof(float4);
    BIP_CUDA(ctx, cudaFuncSetAttribute(k_window_fresnel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)std::max<size_t>(smem, 48 << 10)));
  }
  *root = reinterpret_cast<const float4*>(it->second.first);
  *perm = reinterpret_cast<const int32_t*>(it->second.second);
  return BIP_OK;
}

// Fresnel step over distance d (signed) of n_win envelopes [n_win][Wp][Wp]; window e carries beam h[e % n_beams]
int32_t focal_window_fresnel(bip_ctx* ctx, float2* E, int64_t n_win, const int32_t* h_dev, int n_beams, int Wp, double d) {
  const float4* root; const int32_t* perm;
  BIP_TRY(window_tables(ctx, Wp, &root, &perm));
  const int lW = ilog2(Wp);
  const size_t smem = (size_t)Wp * (pad_len(Wp) + 1) * sizeof(float2) + 2 * (size_t)Wp * sizeof(float4);
  const int thr = std::max(64, std::min(256, Wp * Wp / 32));       // a quarter of the butterflies per stage: twiddle re-use over 4 lines
  const double py = ctx->g.ly / ctx->g.ny, px = ctx->g.lx / ctx->g.nx;
  for (int64_t e0 = 0; e0 < n_win; e0 += (int64_t)n_beams * 1024) {          // whole beam sets per launch: e % n_beams stays the beam
    const int64_t ne = std::min<int64_t>((int64_t)n_beams * 1024, n_win - e0);
    k_window_fresnel<<<(unsigned)ne, thr, smem, ctx->stream>>>(E + e0 * Wp * Wp, h_dev, n_beams, lW, M_PI * ctx->g.lambda * d, 1.0 / ctx->g.ly,
                                                              1.0 / ctx->g.lx, 1.0 / (Wp * py), 1.0 / (Wp * px), root, perm);
    BIP_CUDA(ctx, cudaGetLastError());
    ctx->timing.kernel_launches++;
  }
  return BIP_OK;
}

int32_t focal_env_to_r1t(bip_ctx* ctx, const float2* Env, int32_t oy, int32_t ox, int32_t w, int32_t Wp, const Sliced& out, int32_t atom) {
  const int w2 = w * w;
  k_env_colmax<<<(unsigned)((w2 + 255) / 256), 256, 0, ctx->stream>>>(Env, ctx->n_ap, w, Wp, out.scale + (int64_t)atom * out.scale_batch_stride);
  dim3 grid((unsigned)((w2 + 31) / 32), (unsigned)((2 * out.ksteps + 7) / 8));
  k_env_to_r1t_sliced<<<grid, dim3(32, 8), 0, ctx->stream>>>(Env, ctx->ap_h_dev, ctx->n_ap, oy, ox, w, Wp, ctx->g.ny, ctx->g.nx, ctx->rooty_dev,
                                                            ctx->rootx_dev, out, atom);
  BIP_CUDA(ctx, cudaGetLastError());
  ctx->timing.kernel_launches += 2;
  return BIP_OK;
}

void focal_release(bip_ctx* ctx) {
  for (auto& kv : ctx->focal_tables) { cudaFree(kv.second.first); cudaFree(kv.second.second); }
  ctx->focal_tables.clear();
}

}  // namespace bip
