// Windowed column reconstruction (eq. 15; eq. 11) and illumination
// coefficients: steps a1, a2, a3, a6 of SURVEY.md 8(a).
#include "bip_internal.h"

namespace bip {

namespace {

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

__device__ __forceinline__ float tf32_hi(float x) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return __uint_as_float(r);
}

// exp(+2 pi i h.r/N) for non-negative reduced beam index (hyp, hxp) at global pixel (ry, rx): exact phase from the
// root tables, (h r mod N) reduced in integers (SURVEY "Phases exactly").
// a mod n for 0 <= a: a mask when n is a power of two (every BASELINE grid; the branch is uniform), else the division
__device__ __forceinline__ int mod_n(int a, int n) { return (n & (n - 1)) == 0 ? (a & (n - 1)) : a % n; }

// non-negative index of a signed beam component (|h| < n / 2 is checked when the beam lists are registered)
__device__ __forceinline__ int beam_idx(int h, int n) { return h < 0 ? h + n : h; }

__device__ __forceinline__ float2 tilt(const float2* __restrict__ rooty, const float2* __restrict__ rootx,
                                       int hyp, int hxp, int ry, int rx, int ny, int nx) {
  return cmul(rooty[mod_n(hyp * ry, ny)], rootx[mod_n(hxp * rx, nx)]);
}

// a1: D[a][p][s] = S_p(r) exp(-carrier 2 pi i h_p.r/N), r = (origin_a + s) mod N
__global__ void k_crop_detilt(const float2* __restrict__ S, const int32_t* __restrict__ ph, int carrier,
                              const int32_t* __restrict__ origin, int w, int ny, int nx,
                              const float2* __restrict__ rooty, const float2* __restrict__ rootx,
                              float2* __restrict__ D, int n_par, int shift) {
  const int a = blockIdx.z, p = blockIdx.y;
  const int w2 = w * w;
  const int oy = (origin[2 * a] - shift + ny) % ny, ox = (origin[2 * a + 1] - shift + nx) % nx;   // shift: margin of a padded window
  const int hyp = beam_idx(ph[2 * p], ny), hxp = beam_idx(ph[2 * p + 1], nx);
  const float2* col = S + (int64_t)p * ny * nx;
  float2* out = D + ((int64_t)a * n_par + p) * w2;
  for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < w2; s += gridDim.x * blockDim.x) {
    const int sy = s / w, sx = s - sy * w;
    int ry = oy + sy; if (ry >= ny) ry -= ny;
    int rx = ox + sx; if (rx >= nx) rx -= nx;
    float2 t = tilt(rooty, rootx, hyp, hxp, ry, rx, ny, nx);
    if (carrier > 0) t.y = -t.y;                       // remove the carrier: multiply by its conjugate
    out[s] = cmul(col[(int64_t)ry * nx + rx], t);
  }
}

// One reconstructed element: sum_j w_j D[idx_j][s], optional magnitude-preserving form, re-tilt.
__device__ __forceinline__ float2 recon_elem(const float2* __restrict__ Da, const int32_t* __restrict__ idx,
                                             const float* __restrict__ wt, int max_nn, int w2, int s, int recon,
                                             float2 t) {
  float zr = 0.f, zi = 0.f, mag = 0.f;
  for (int j = 0; j < max_nn; ++j) {
    const int p = idx[j];
    if (p < 0) break;
    const float wj = wt[j];
    const float2 d = Da[(int64_t)p * w2 + s];
    zr = fmaf(wj, d.x, zr);
    zi = fmaf(wj, d.y, zi);
    if (recon == BIP_RECON_MAGPHASE) mag = fmaf(wj, sqrtf(d.x * d.x + d.y * d.y), mag);
  }
  if (recon == BIP_RECON_MAGPHASE) {
    const float az = sqrtf(zr * zr + zi * zi);
    const float sc = az >= 1e-30f ? mag / az : 0.f;   // eq. 11; |z| < 1e-30 -> 0
    zr *= sc; zi *= sc;
  }
  return cmul(make_float2(zr, zi), t);
}

// a2 / a6 (row-major output [a][beam][s], K-major over s): grid (s-chunks, beams, atoms)
__global__ void k_recon_rows(const float2* __restrict__ D, int n_par, const int32_t* __restrict__ bh, int n_beams,
                             const int32_t* __restrict__ nn_idx, const float* __restrict__ nn_w, int max_nn,
                             int carrier, int recon, const int32_t* __restrict__ origin, int w, int ny, int nx,
                             const float2* __restrict__ rooty, const float2* __restrict__ rootx, Planes out) {
  const int a = blockIdx.z, b = blockIdx.y;
  const int w2 = w * w;
  __shared__ int32_t s_idx[BIP_MAX_NN];
  __shared__ float s_w[BIP_MAX_NN];
  if (threadIdx.x < max_nn) {
    s_idx[threadIdx.x] = nn_idx[(int64_t)b * max_nn + threadIdx.x];
    s_w[threadIdx.x] = nn_w[(int64_t)b * max_nn + threadIdx.x];
  }
  __syncthreads();
  const int oy = origin[2 * a], ox = origin[2 * a + 1];
  const int hyp = beam_idx(bh[2 * b], ny), hxp = beam_idx(bh[2 * b + 1], nx);
  const float2* Da = D + (int64_t)a * n_par * w2;
  const int64_t row = (int64_t)a * out.batch_stride + (int64_t)b * out.ld;
  for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < w2; s += gridDim.x * blockDim.x) {
    const int sy = s / w, sx = s - sy * w;
    int ry = oy + sy; if (ry >= ny) ry -= ny;
    int rx = ox + sx; if (rx >= nx) rx -= nx;
    float2 t = tilt(rooty, rootx, hyp, hxp, ry, rx, ny, nx);
    if (carrier < 0) t.y = -t.y;                       // restore the carrier exp(carrier 2 pi i h_b.r/N)
    const float2 v = recon_elem(Da, s_idx, s_w, max_nn, w2, s, recon, t);
    const float rh = tf32_hi(v.x), ih = tf32_hi(v.y);
    out.p[0][row + s] = rh; out.p[1][row + s] = tf32_hi(v.x - rh);
    out.p[2][row + s] = ih; out.p[3][row + s] = tf32_hi(v.y - ih);
  }
}

// a2 transposed output [a][s][beam] (K-major over beams, operand of the probe GEMM): 32 x 32 tiles through smem
__global__ void k_recon_transposed(const float2* __restrict__ D, int n_par, const int32_t* __restrict__ bh, int n_beams,
                                   const int32_t* __restrict__ nn_idx, const float* __restrict__ nn_w, int max_nn,
                                   int carrier, int recon, const int32_t* __restrict__ origin, int w, int ny, int nx,
                                   const float2* __restrict__ rooty, const float2* __restrict__ rootx, Planes out) {
  __shared__ float2 tile[32][33];
  const int a = blockIdx.z;
  const int w2 = w * w;
  const int b0 = blockIdx.y * 32, s0 = blockIdx.x * 32;
  const int oy = origin[2 * a], ox = origin[2 * a + 1];
  const float2* Da = D + (int64_t)a * n_par * w2;
  // compute: threadIdx.x <-> s (coalesced reads of D), threadIdx.y strides over beams
  for (int bb = threadIdx.y; bb < 32; bb += blockDim.y) {
    const int b = b0 + bb, s = s0 + threadIdx.x;
    float2 v = make_float2(0.f, 0.f);
    if (b < n_beams && s < w2) {
      const int sy = s / w, sx = s - sy * w;
      int ry = oy + sy; if (ry >= ny) ry -= ny;
      int rx = ox + sx; if (rx >= nx) rx -= nx;
      const int hyp = beam_idx(bh[2 * b], ny), hxp = beam_idx(bh[2 * b + 1], nx);
      float2 t = tilt(rooty, rootx, hyp, hxp, ry, rx, ny, nx);
      if (carrier < 0) t.y = -t.y;
      v = recon_elem(Da, nn_idx + (int64_t)b * max_nn, nn_w + (int64_t)b * max_nn, max_nn, w2, s, recon, t);
    }
    tile[bb][threadIdx.x] = v;
  }
  __syncthreads();
  // store: threadIdx.x <-> beam (coalesced writes)
  for (int ss = threadIdx.y; ss < 32; ss += blockDim.y) {
    const int s = s0 + ss, b = b0 + threadIdx.x;
    if (s < w2 && b < n_beams) {
      const float2 v = tile[threadIdx.x][ss];
      const int64_t o = (int64_t)a * out.batch_stride + (int64_t)s * out.ld + b;
      const float rh = tf32_hi(v.x), ih = tf32_hi(v.y);
      out.p[0][o] = rh; out.p[1][o] = tf32_hi(v.x - rh);
      out.p[2][o] = ih; out.p[3][o] = tf32_hi(v.y - ih);
    }
  }
}

// plain c64 output of one atom (debug / parity of a1-a2, a6)
__global__ void k_recon_c64(const float2* __restrict__ D, int n_par, const int32_t* __restrict__ bh, int n_beams,
                            const int32_t* __restrict__ nn_idx, const float* __restrict__ nn_w, int max_nn,
                            int carrier, int recon, const int32_t* __restrict__ origin, int atom, int w, int ny, int nx,
                            const float2* __restrict__ rooty, const float2* __restrict__ rootx, float2* __restrict__ out, int shift, int retilt) {
  const int b = blockIdx.y;
  const int w2 = w * w;
  const int oy = (origin[2 * atom] - shift + ny) % ny, ox = (origin[2 * atom + 1] - shift + nx) % nx;
  const int hyp = beam_idx(bh[2 * b], ny), hxp = beam_idx(bh[2 * b + 1], nx);
  for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < w2; s += gridDim.x * blockDim.x) {
    const int sy = s / w, sx = s - sy * w;
    int ry = oy + sy; if (ry >= ny) ry -= ny;
    int rx = ox + sx; if (rx >= nx) rx -= nx;
    float2 t = retilt ? tilt(rooty, rootx, hyp, hxp, ry, rx, ny, nx) : make_float2(1.f, 0.f);   // retilt == 0: the bare envelope
    if (carrier < 0) t.y = -t.y;
    out[(int64_t)b * w2 + s] = recon_elem(D, nn_idx + (int64_t)b * max_nn, nn_w + (int64_t)b * max_nn, max_nn, w2, s, recon, t);
  }
}

// a3: A[rho][b] = c_b exp(-2 pi i (hy rho_y / ny + hx rho_x / nx)), phase in double (rho may be any real)
__global__ void k_illumination(const double* __restrict__ rho, int n_rho, const int32_t* __restrict__ h,
                               const float2* __restrict__ c, int n_ap, int ny, int nx, Planes out) {
  const int r = blockIdx.y;
  const double py = rho[2 * r], px = rho[2 * r + 1];
  for (int b = blockIdx.x * blockDim.x + threadIdx.x; b < n_ap; b += gridDim.x * blockDim.x) {
    double t = (double)h[2 * b] * py / ny + (double)h[2 * b + 1] * px / nx;
    t -= rint(t);                                       // exact range reduction of the turn count
    double sn, cs;
    sincospi(-2.0 * t, &sn, &cs);
    const float2 cb = c[b];
    const float re = (float)((double)cb.x * cs - (double)cb.y * sn);
    const float im = (float)((double)cb.x * sn + (double)cb.y * cs);
    const int64_t o = (int64_t)r * out.ld + b;
    const float rh = tf32_hi(re), ih = tf32_hi(im);
    out.p[0][o] = rh; out.p[1][o] = tf32_hi(re - rh);
    out.p[2][o] = ih; out.p[3][o] = tf32_hi(im - ih);
  }
}


// ---- sliced-operand producers (precision BIP_PREC_BF16X6; layout and split in bip_sliced.cuh) ----

// scale[a][s] = power of two >= max_p |D[a][p][s]|: a bound of every reconstructed beam at window pixel s, because
// the natural-neighbour weights are a convex combination (eq. 8) in both eq. 15 and eq. 11.
__global__ void k_parent_colmax(const float2* __restrict__ D, int n_par, int w2, float* __restrict__ scale, int64_t scale_batch_stride) {
  const int a = blockIdx.y;
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= w2) return;
  const float2* Da = D + (int64_t)a * n_par * w2;
  float m = 0.f;
  for (int p = 0; p < n_par; ++p) {
    const float2 d = Da[(int64_t)p * w2 + s];
    m = fmaxf(m, d.x * d.x + d.y * d.y);
  }
  scale[(int64_t)a * scale_batch_stride + s] = sl_pow2_scale(1.001f * sqrtf(m));
}

// a2 as the K-major operand of the probe GEMM: rows = window pixels s, k = aperture beams b.
// thread = (row s, group of 8 consecutive beams); lanes run over consecutive s (coalesced reads of D, 128-byte stores).
__global__ void __launch_bounds__(256) k_recon_t_sliced(const float2* __restrict__ D, int n_par, const int32_t* __restrict__ bh, int n_beams,
                                 const int32_t* __restrict__ nn_idx, const float* __restrict__ nn_w, int max_nn, int carrier,
                                 int recon, const int32_t* __restrict__ origin, int w, int ny, int nx,
                                 const float2* __restrict__ rooty, const float2* __restrict__ rootx, Sliced out) {
  const int a = blockIdx.z;
  const int w2 = w * w;
  const int s = blockIdx.x * 32 + threadIdx.x, g = blockIdx.y * 8 + threadIdx.y;
  // neighbour lists of the block's 64 beams, read once per block instead of once per (beam, window pixel)
  __shared__ int32_t s_idx[64][BIP_MAX_NN];
  __shared__ float s_w[64][BIP_MAX_NN];
  __shared__ int32_t s_h[64][2];
  for (int i = threadIdx.y * 32 + threadIdx.x; i < 64 * max_nn; i += 256) {
    const int bb = i / max_nn, j = i - bb * max_nn, b = blockIdx.y * 64 + bb;
    s_idx[bb][j] = b < n_beams ? nn_idx[(int64_t)b * max_nn + j] : -1;
    s_w[bb][j] = b < n_beams ? nn_w[(int64_t)b * max_nn + j] : 0.f;
  }
  if (threadIdx.y < 2) {
    const int bb = threadIdx.y * 32 + threadIdx.x, b = blockIdx.y * 64 + bb;
    s_h[bb][0] = b < n_beams ? beam_idx(bh[2 * b], ny) : 0;
    s_h[bb][1] = b < n_beams ? beam_idx(bh[2 * b + 1], nx) : 0;
  }
  __syncthreads();
  if (s >= w2 || g >= 2 * out.ksteps) return;
  const int oy = origin[2 * a], ox = origin[2 * a + 1];
  const int sy = s / w, sx = s - sy * w;
  int ry = oy + sy; if (ry >= ny) ry -= ny;
  int rx = ox + sx; if (rx >= nx) rx -= nx;
  const float2* Da = D + (int64_t)a * n_par * w2;
  float re[8], im[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    const int b = g * 8 + j, bb = threadIdx.y * 8 + j;
    float2 v = make_float2(0.f, 0.f);
    if (b < n_beams) {
      float2 t = tilt(rooty, rootx, s_h[bb][0], s_h[bb][1], ry, rx, ny, nx);
      if (carrier < 0) t.y = -t.y;
      v = recon_elem(Da, s_idx[bb], s_w[bb], max_nn, w2, s, recon, t);
    }
    re[j] = v.x; im[j] = v.y;
  }
  sl_store_group(out, a, s, g, re, im, 1.f / out.scale[(int64_t)a * out.scale_batch_stride + s]);
}

// a6 as the K-major operand of the detector GEMM: rows = detector beams d, k = window pixels s.
// One block per (beam, atom): pass 1 finds the row maximum, pass 2 splits and stores.
// max_s |D[a][p][s]| of every parent window: one warp per (parent, atom).  Feeds the row scales of R2 below.
__global__ void __launch_bounds__(256) k_parent_rowmax(const float2* __restrict__ D, int n_par, int w2, float* __restrict__ pmax) {
  const int p = blockIdx.x * 8 + (threadIdx.x >> 5), a = blockIdx.y, lane = threadIdx.x & 31;
  if (p >= n_par) return;
  const float2* row = D + ((int64_t)a * n_par + p) * w2;
  float m = 0.f;
  for (int s = lane; s < w2; s += 32) { const float2 d = row[s]; m = fmaxf(m, d.x * d.x + d.y * d.y); }
#pragma unroll
  for (int o = 16; o; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if (lane == 0) pmax[(int64_t)a * n_par + p] = sqrtf(m);
}

__global__ void __launch_bounds__(256, 3) k_recon_rows_sliced(const float2* __restrict__ D, int n_par, const int32_t* __restrict__ bh, int n_beams,
                                    const int32_t* __restrict__ nn_idx, const float* __restrict__ nn_w, int max_nn, int carrier,
                                    int recon, const int32_t* __restrict__ origin, int w, int ny, int nx,
                                    const float2* __restrict__ rooty, const float2* __restrict__ rootx,
                                    const float* __restrict__ pmax, const float2* __restrict__ H, int n_ch,
                                    const float* __restrict__ hmax, Sliced out) {
  // One block per (8 consecutive beams, atom); thread = (row = t & 7, k-group lane = t >> 3).  The blocked slice layout
  // keeps the 16-byte groups of rows r .. r+7 of one k-group side by side, so the 8 row-lanes of a store instruction
  // fill one 128-byte line.  Single pass: the row scale is the power of two above sum_p w_p max_s |D_p[s]|, a bound on
  // |R2[d][s]| for both reconstructions (the weights are a convex combination, eq. 8; eq. 11 has magnitude
  // sum_p w_p |D_p|), so no element has to be evaluated twice to find the exact row maximum.
  const int a = blockIdx.y, r = threadIdx.x & 7, gl = threadIdx.x >> 3, b = blockIdx.x * 8 + r;
  const bool row_ok = b < n_beams;
  const int w2 = w * w;
  __shared__ int32_t s_idx[8][BIP_MAX_NN];
  __shared__ float s_w[8][BIP_MAX_NN];
  for (int i = threadIdx.x; i < 8 * max_nn; i += blockDim.x) {
    const int rr = i / max_nn, j = i - rr * max_nn, bb = blockIdx.x * 8 + rr;
    s_idx[rr][j] = bb < n_beams ? nn_idx[(int64_t)bb * max_nn + j] : -1;
    s_w[rr][j] = bb < n_beams ? nn_w[(int64_t)bb * max_nn + j] : 0.f;
  }
  __syncthreads();
  if (!row_ok) return;
  float bound = 0.f;
  for (int j = 0; j < max_nn; ++j) {
    const int p = s_idx[r][j];
    if (p < 0) break;
    bound = fmaf(s_w[r][j], __ldg(pmax + (int64_t)a * n_par + p), bound);
  }
  // H != NULL (coupling association, eq. 13): the rows written are H_n[s] R[b][s], row n * n_beams + b, n = 0 .. n_ch-1
  const int n_rep = H ? n_ch : 1;
  if (gl == 0)
    for (int n = 0; n < n_rep; ++n)
      out.scale[(int64_t)a * out.scale_batch_stride + (int64_t)n * n_beams + b] = sl_pow2_scale(1.001f * bound * (H ? hmax[n] : 1.f));
  const int oy = origin[2 * a], ox = origin[2 * a + 1];
  const int hyp = beam_idx(bh[2 * b], ny), hxp = beam_idx(bh[2 * b + 1], nx);
  const float2* Da = D + (int64_t)a * n_par * w2;
  const int n_groups = 2 * (int)out.ksteps;
  for (int g = gl; g < n_groups; g += 32) {
    // the 8 window pixels s0 .. s0 + 7 of this k-group: neighbours in the outer loop (index and weight read once per
    // group, the parent window read as 4 x 16 bytes), eq. 15 / eq. 11 sums in registers, then re-tilt
    const int s0 = g * 8;
    const bool whole = s0 + 8 <= w2;
    float zr[8], zi[8], mg[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) { zr[j] = 0.f; zi[j] = 0.f; mg[j] = 0.f; }
    for (int jn = 0; jn < max_nn; ++jn) {
      const int p = s_idx[r][jn];
      if (p < 0) break;
      const float wj = s_w[r][jn];
      const float2* dp = Da + (int64_t)p * w2 + s0;
      float2 d[8];
      if (whole) {                                   // w is even: rows of D and s0 are 16-byte aligned
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const float4 q = __ldg(reinterpret_cast<const float4*>(dp) + j);
          d[2 * j] = make_float2(q.x, q.y); d[2 * j + 1] = make_float2(q.z, q.w);
        }
      } else {
#pragma unroll
        for (int j = 0; j < 8; ++j) d[j] = s0 + j < w2 ? __ldg(dp + j) : make_float2(0.f, 0.f);
      }
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        zr[j] = fmaf(wj, d[j].x, zr[j]);
        zi[j] = fmaf(wj, d[j].y, zi[j]);
        if (recon == BIP_RECON_MAGPHASE) mg[j] = fmaf(wj, sqrtf(d[j].x * d[j].x + d[j].y * d[j].y), mg[j]);
      }
    }
    float re[8], im[8];
    int sy = s0 / w, sx = s0 - sy * w;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      float2 v = make_float2(0.f, 0.f);
      if (s0 + j < w2) {
        int ry = oy + sy; if (ry >= ny) ry -= ny;
        int rx = ox + sx; if (rx >= nx) rx -= nx;
        float2 t = tilt(rooty, rootx, hyp, hxp, ry, rx, ny, nx);
        if (carrier < 0) t.y = -t.y;
        float ar = zr[j], ai = zi[j];
        if (recon == BIP_RECON_MAGPHASE) {
          const float az = sqrtf(ar * ar + ai * ai);
          const float sc = az >= 1e-30f ? mg[j] / az : 0.f;   // eq. 11; |z| < 1e-30 -> 0
          ar *= sc; ai *= sc;
        }
        v = cmul(make_float2(ar, ai), t);
      }
      re[j] = v.x; im[j] = v.y;
      if (++sx == w) { sx = 0; ++sy; }
    }
    if (!H) {
      sl_store_group(out, a, b, g, re, im, 1.f / sl_pow2_scale(1.001f * bound));
    } else {
      for (int n = 0; n < n_ch; ++n) {
        float hr[8], hi[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const int s = g * 8 + j;
          const float2 h = s < w2 ? __ldg(H + (int64_t)n * w2 + s) : make_float2(0.f, 0.f);
          hr[j] = h.x * re[j] - h.y * im[j];
          hi[j] = h.x * im[j] + h.y * re[j];
        }
        sl_store_group(out, a, (int64_t)n * n_beams + b, g, hr, hi, 1.f / sl_pow2_scale(1.001f * bound * hmax[n]));
      }
    }
  }
}

// a3 as the K-major operand of the probe GEMM: rows = scan positions, k = aperture beams; every row has the scale
// `scale` >= max_b |c_b|.  thread = (rho, group of 8 beams), lanes over consecutive rho.
__global__ void __launch_bounds__(256) k_illumination_sliced(const double* __restrict__ rho, int n_rho, const int32_t* __restrict__ h,
                                      const float2* __restrict__ c, int n_ap, int ny, int nx, float scale, Sliced out) {
  const int r = blockIdx.x * 32 + threadIdx.x, g = blockIdx.y * 8 + threadIdx.y;
  if (r >= n_rho || g >= 2 * out.ksteps) return;
  const double py = rho[2 * r], px = rho[2 * r + 1];
  float re[8], im[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    const int b = g * 8 + j;
    re[j] = 0.f; im[j] = 0.f;
    if (b < n_ap) {
      double t = (double)h[2 * b] * py / ny + (double)h[2 * b + 1] * px / nx;
      t -= rint(t);
      double sn, cs;
      sincospi(-2.0 * t, &sn, &cs);
      const float2 cb = c[b];
      re[j] = (float)((double)cb.x * cs - (double)cb.y * sn);
      im[j] = (float)((double)cb.x * sn + (double)cb.y * cs);
    }
  }
  if (g == 0) out.scale[r] = scale;
  sl_store_group(out, 0, r, g, re, im, 1.f / scale);
}

}  // namespace

int32_t launch_crop_detilt(bip_ctx* ctx, const float2* S, const int32_t* ph_dev, int32_t n_par, int carrier,
                           const int32_t* origin_dev, int32_t n_atoms, int32_t w, float2* D, int32_t origin_shift) {
  dim3 grid((unsigned)((w * w + 255) / 256), (unsigned)n_par, (unsigned)n_atoms);
  k_crop_detilt<<<grid, 256, 0, ctx->stream>>>(S, ph_dev, carrier, origin_dev, w, ctx->g.ny, ctx->g.nx,
                                               ctx->rooty_dev, ctx->rootx_dev, D, n_par, origin_shift);
  BIP_CUDA(ctx, cudaGetLastError());
  ctx->timing.kernel_launches++;
  return BIP_OK;
}

int32_t launch_recon(bip_ctx* ctx, const float2* D, int32_t n_par, const int32_t* bh_dev, int32_t n_beams,
                     const int32_t* nn_idx, const float* nn_w, int32_t max_nn, int carrier, int recon,
                     const int32_t* origin_dev, int32_t n_atoms, int32_t w, bool transpose, Planes out) {
  const int w2 = w * w;
  if (!transpose) {
    for (int b0 = 0; b0 < n_beams; b0 += 65535) {     // gridDim.y limit
      const int nb = std::min(65535, n_beams - b0);
      Planes o = out;
      for (int k = 0; k < 4; ++k) o.p[k] += (int64_t)b0 * out.ld;
      dim3 grid((unsigned)((w2 + 255) / 256), (unsigned)nb, (unsigned)n_atoms);
      k_recon_rows<<<grid, 256, 0, ctx->stream>>>(D, n_par, bh_dev + 2 * (int64_t)b0, nb, nn_idx + (int64_t)b0 * max_nn,
                                                  nn_w + (int64_t)b0 * max_nn, max_nn, carrier, recon, origin_dev, w,
                                                  ctx->g.ny, ctx->g.nx, ctx->rooty_dev, ctx->rootx_dev, o);
      BIP_CUDA(ctx, cudaGetLastError());
      ctx->timing.kernel_launches++;
    }
  } else {
    dim3 grid((unsigned)((w2 + 31) / 32), (unsigned)((n_beams + 31) / 32), (unsigned)n_atoms);
    k_recon_transposed<<<grid, dim3(32, 8), 0, ctx->stream>>>(D, n_par, bh_dev, n_beams, nn_idx, nn_w, max_nn, carrier, recon,
                                                             origin_dev, w, ctx->g.ny, ctx->g.nx, ctx->rooty_dev,
                                                             ctx->rootx_dev, out);
    BIP_CUDA(ctx, cudaGetLastError());
    ctx->timing.kernel_launches++;
  }
  return BIP_OK;
}

int32_t launch_recon_c64(bip_ctx* ctx, const float2* D, int32_t n_par, const int32_t* bh_dev, int32_t n_beams,
                         const int32_t* nn_idx, const float* nn_w, int32_t max_nn, int carrier, int recon,
                         const int32_t* origin_dev, int32_t atom, int32_t w, float2* out, int32_t origin_shift, bool retilt) {
  for (int b0 = 0; b0 < n_beams; b0 += 65535) {
    const int nb = std::min(65535, n_beams - b0);
    dim3 grid((unsigned)((w * w + 255) / 256), (unsigned)nb);
    k_recon_c64<<<grid, 256, 0, ctx->stream>>>(D, n_par, bh_dev + 2 * (int64_t)b0, nb, nn_idx + (int64_t)b0 * max_nn,
                                               nn_w + (int64_t)b0 * max_nn, max_nn, carrier, recon, origin_dev, atom, w,
                                               ctx->g.ny, ctx->g.nx, ctx->rooty_dev, ctx->rootx_dev,
                                               out + (int64_t)b0 * w * w, origin_shift, retilt ? 1 : 0);
    BIP_CUDA(ctx, cudaGetLastError());
  }
  return BIP_OK;
}

int32_t launch_illumination(bip_ctx* ctx, const double* rho_dev, int32_t n_rho, Planes out) {
  for (int r0 = 0; r0 < n_rho; r0 += 65535) {
    const int nr = std::min(65535, n_rho - r0);
    Planes o = out;
    for (int k = 0; k < 4; ++k) o.p[k] += (int64_t)r0 * out.ld;
    dim3 grid((unsigned)((ctx->n_ap + 255) / 256), (unsigned)nr);
    k_illumination<<<grid, 256, 0, ctx->stream>>>(rho_dev + 2 * (int64_t)r0, nr, ctx->ap_h_dev, ctx->ap_c_dev, ctx->n_ap,
                                                  ctx->g.ny, ctx->g.nx, o);
    BIP_CUDA(ctx, cudaGetLastError());
  }
  return BIP_OK;
}


int32_t launch_recon_t_sliced(bip_ctx* ctx, const float2* D, int32_t n_par, const int32_t* bh_dev, int32_t n_beams,
                              const int32_t* nn_idx, const float* nn_w, int32_t max_nn, int carrier, int recon,
                              const int32_t* origin_dev, int32_t n_atoms, int32_t w, Sliced out) {
  const int w2 = w * w;
  dim3 g0((unsigned)((w2 + 255) / 256), (unsigned)n_atoms);
  k_parent_colmax<<<g0, 256, 0, ctx->stream>>>(D, n_par, w2, out.scale, out.scale_batch_stride);
  BIP_CUDA(ctx, cudaGetLastError());
  dim3 grid((unsigned)((w2 + 31) / 32), (unsigned)((2 * out.ksteps + 7) / 8), (unsigned)n_atoms);
  k_recon_t_sliced<<<grid, dim3(32, 8), 0, ctx->stream>>>(D, n_par, bh_dev, n_beams, nn_idx, nn_w, max_nn, carrier, recon, origin_dev,
                                                         w, ctx->g.ny, ctx->g.nx, ctx->rooty_dev, ctx->rootx_dev, out);
  BIP_CUDA(ctx, cudaGetLastError());
  ctx->timing.kernel_launches += 2;
  return BIP_OK;
}

int32_t launch_recon_rows_sliced(bip_ctx* ctx, const float2* D, int32_t n_par, const int32_t* bh_dev, int32_t n_beams,
                                 const int32_t* nn_idx, const float* nn_w, int32_t max_nn, int carrier, int recon,
                                 const int32_t* origin_dev, int32_t n_atoms, int32_t w, Sliced out, const float2* H, int32_t n_ch,
                                 const float* hmax) {
  BIP_TRY(ensure(ctx, ctx->Pmax, (size_t)n_atoms * n_par * sizeof(float), "parent window maxima"));
  float* pmax = reinterpret_cast<float*>(ctx->Pmax.p);
  for (int a0 = 0; a0 < n_atoms; a0 += 65535) {          // gridDim.y limit
    const int na = std::min(65535, n_atoms - a0);
    k_parent_rowmax<<<dim3((unsigned)((n_par + 7) / 8), (unsigned)na), 256, 0, ctx->stream>>>(D + (int64_t)a0 * n_par * w * w, n_par, w * w,
                                                                                              pmax + (int64_t)a0 * n_par);
    BIP_CUDA(ctx, cudaGetLastError());
    ctx->timing.kernel_launches++;
    Sliced o = out;
    o.base += (int64_t)a0 * out.batch_stride;
    o.scale += (int64_t)a0 * out.scale_batch_stride;
    dim3 grid((unsigned)((n_beams + 7) / 8), (unsigned)na);
    k_recon_rows_sliced<<<grid, 256, 0, ctx->stream>>>(D + (int64_t)a0 * n_par * w * w, n_par, bh_dev, n_beams, nn_idx, nn_w, max_nn, carrier,
                                                      recon, origin_dev + 2 * (int64_t)a0, w, ctx->g.ny, ctx->g.nx, ctx->rooty_dev,
                                                      ctx->rootx_dev, pmax + (int64_t)a0 * n_par, H, n_ch, hmax, o);
    BIP_CUDA(ctx, cudaGetLastError());
    ctx->timing.kernel_launches++;
  }
  return BIP_OK;
}

int32_t launch_illumination_sliced(bip_ctx* ctx, const double* rho_dev, int32_t n_rho, float scale, Sliced out) {
  dim3 grid((unsigned)((n_rho + 31) / 32), (unsigned)((2 * out.ksteps + 7) / 8));
  k_illumination_sliced<<<grid, dim3(32, 8), 0, ctx->stream>>>(rho_dev, n_rho, ctx->ap_h_dev, ctx->ap_c_dev, ctx->n_ap, ctx->g.ny,
                                                              ctx->g.nx, scale, out);
  BIP_CUDA(ctx, cudaGetLastError());
  return BIP_OK;
}

}  // namespace bip
