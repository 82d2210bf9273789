// C ABI of libbip (include/bip.h) and the plane-loop driver of Algorithm 5.
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>

#include "bip_internal.h"

namespace bip {

void ms_release(bip_ctx* ctx);

static thread_local std::string g_err;

int32_t fail(bip_ctx* ctx, int32_t status, const char* fmt, ...) {
  char buf[1024];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (ctx) ctx->err = buf;
  g_err = buf;
  return status;
}

int32_t dev_alloc(bip_ctx* ctx, void** p, size_t bytes, const char* what) {
  *p = nullptr;
  if (bytes == 0) bytes = 16;
  cudaError_t e = cudaMalloc(p, bytes);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return fail(ctx, e == cudaErrorMemoryAllocation ? BIP_ERR_OOM : BIP_ERR_CUDA, "cudaMalloc of %zu bytes for %s failed: %s",
                bytes, what, cudaGetErrorString(e));
  }
  return BIP_OK;
}

// Recycled device blocks for per-call objects: best fit among the context's released blocks (at most twice the request), else
// a fresh cudaMalloc.  Released blocks are kept until bip_destroy.
int32_t pool_alloc(bip_ctx* ctx, void** p, size_t bytes, const char* what) {
  if (bytes == 0) bytes = 16;
  int best = -1;
  for (int i = 0; i < (int)ctx->pool_free.size(); ++i) {
    const size_t sz = ctx->pool_free[i].second;
    if (sz >= bytes && sz <= 2 * bytes + 256 && (best < 0 || sz < ctx->pool_free[best].second)) best = i;
  }
  if (best >= 0) {
    *p = ctx->pool_free[best].first;
    ctx->pool_size[*p] = ctx->pool_free[best].second;
    ctx->pool_free.erase(ctx->pool_free.begin() + best);
    return BIP_OK;
  }
  BIP_TRY(dev_alloc(ctx, p, bytes, what));
  ctx->pool_size[*p] = bytes;
  return BIP_OK;
}

void pool_release(bip_ctx* ctx, void* p) {
  if (!p) return;
  auto it = ctx->pool_size.find(p);
  if (it == ctx->pool_size.end()) { cudaFree(p); return; }
  ctx->pool_free.emplace_back(p, it->second);
  ctx->pool_size.erase(it);
}

int32_t ensure(bip_ctx* ctx, DevBuf& b, size_t bytes, const char* what) {
  if (b.bytes >= bytes && b.p) return BIP_OK;
  if (b.p) { cudaStreamSynchronize(ctx->stream); cudaFree(b.p); b.p = nullptr; b.bytes = 0; }
  BIP_TRY(dev_alloc(ctx, &b.p, bytes, what));
  b.bytes = bytes;
  return BIP_OK;
}

static inline int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }

// Carve four planes [batch][rows][ld] out of one DevBuf (zero-filled when (re)allocated or when `zero`).
// The kernels that fill the planes write only the valid columns; the padding up to `ld` must read as zero, so the
// buffer is cleared whenever its layout (rows, cols, batch) changes.
static int32_t planes_in(bip_ctx* ctx, DevBuf& buf, Planes& P, int64_t rows, int64_t cols, int64_t batch, const char* what) {
  P.rows = rows;
  P.ld = round_up(cols, 32);
  P.batch_stride = rows * P.ld;
  const int64_t plane_floats = round_up(P.batch_stride * batch, 256);   // keep plane bases 1024 B aligned
  const void* before = buf.p;
  BIP_TRY(ensure(ctx, buf, (size_t)plane_floats * 4 * sizeof(float), what));
  const uint64_t sig = ((uint64_t)rows * 1000003ull + (uint64_t)cols) * 1000003ull + (uint64_t)batch;
  if (buf.p != before || buf.sig != sig) {
    if (P.ld != cols || buf.p != before) BIP_CUDA(ctx, cudaMemsetAsync(buf.p, 0, buf.bytes, ctx->stream));
    buf.sig = sig;
  }
  for (int k = 0; k < 4; ++k) P.p[k] = reinterpret_cast<float*>(buf.p) + k * plane_floats;
  return BIP_OK;
}

// Carve a sliced 16-bit operand [batch][rows][k] of format `fmt` out of one DevBuf.  Producers write every k-step of every valid row;
// the padding rows of the last row tile only have to be finite (they feed masked accumulator rows / columns), so the
// buffer is cleared when it is (re)allocated and never again.
static int32_t sliced_in(bip_ctx* ctx, DevBuf& buf, Sliced& S, int fmt, int64_t rows, int64_t k, int64_t batch, const char* what,
                         int64_t row_align = SL_ROWS, bool y_operand = false) {
  S.fmt = fmt;
  S.neg_im = y_operand && sliced_wide(fmt) ? 1 : 0;       // Y operands of the N = 256 kernel carry the negated imaginary slices
  S.rows = rows;
  S.rows_pad = round_up(rows, row_align);
  S.k = k;
  S.ksteps = (k + SL_K - 1) / SL_K;
  S.batch_stride = S.rows_pad / SL_ROWS * S.ksteps * sl_step_el_of(S);
  const void* before = buf.p;
  BIP_TRY(ensure(ctx, buf, (size_t)(S.batch_stride * std::max<int64_t>(batch, 1)) * sizeof(uint16_t), what));
  if (buf.p != before) BIP_CUDA(ctx, cudaMemsetAsync(buf.p, 0, buf.bytes, ctx->stream));
  S.base = reinterpret_cast<uint16_t*>(buf.p);
  return BIP_OK;
}

// a3, built on first use in the format the requested arithmetic reads.
static void free_illumination(bip_ctx* ctx);
static inline int sliced_fmt_of(int precision) { return precision == BIP_PREC_FP16X4 || precision == BIP_PREC_FP16X3 ? SL_FMT_FP16X4 : precision == BIP_PREC_BF16X6 ? SL_FMT_BF16X6 : -1; }

static int32_t ensure_illumination(bip_ctx* ctx, int precision) {
  const int fmt = sliced_fmt_of(precision);
  if (fmt >= 0) {
    if (ctx->A_sl.base && ctx->A_sl.fmt == fmt) return BIP_OK;
    if (ctx->A_sl.base) { cudaStreamSynchronize(ctx->stream); cudaFree(ctx->A_sl.base); cudaFree(ctx->A_sl.scale); ctx->A_sl = Sliced(); }
    Sliced A;
    DevBuf b;
    BIP_TRY(sliced_in(ctx, b, A, fmt, ctx->n_rho, ctx->n_ap, 1, "illumination matrix (sliced)", 2 * SL_ROWS));   // X operand: row-tile pairs
    A.batch_stride = 0;
    if (dev_alloc(ctx, (void**)&A.scale, (size_t)A.rows_pad * sizeof(float), "illumination row scales") != BIP_OK) { cudaFree(b.p); return BIP_ERR_OOM; }
    BIP_CUDA(ctx, cudaMemsetAsync(A.scale, 0, (size_t)A.rows_pad * sizeof(float), ctx->stream));
    A.scale_batch_stride = 0;
    int e = 0;
    std::frexp(1.0001f * ctx->ap_c_max, &e);
    ctx->A_sl = A;
    return launch_illumination_sliced(ctx, ctx->rho_dev, ctx->n_rho, ctx->ap_c_max > 0.f ? std::ldexp(1.f, e) : 1.f, A);
  }
  if (ctx->A.p[0]) return BIP_OK;
  Planes A;
  A.rows = ctx->n_rho; A.ld = round_up(ctx->n_ap, 32); A.batch_stride = 0;
  const int64_t plane_floats = round_up(A.rows * A.ld, 256);
  float* base = nullptr;
  BIP_TRY(dev_alloc(ctx, (void**)&base, (size_t)plane_floats * 4 * sizeof(float), "illumination matrix"));
  BIP_CUDA(ctx, cudaMemsetAsync(base, 0, (size_t)plane_floats * 4 * sizeof(float), ctx->stream));
  for (int k = 0; k < 4; ++k) A.p[k] = base + k * plane_floats;
  ctx->A = A;
  return launch_illumination(ctx, ctx->rho_dev, ctx->n_rho, A);
}

static void free_illumination(bip_ctx* ctx) {
  if (ctx->A.p[0]) { cudaFree(ctx->A.p[0]); ctx->A = Planes(); }
  if (ctx->A_sl.base) { cudaFree(ctx->A_sl.base); cudaFree(ctx->A_sl.scale); ctx->A_sl = Sliced(); }
}

template <class T>
static int32_t upload(bip_ctx* ctx, T** dst, const T* src, size_t n, const char* what) {
  BIP_TRY(dev_alloc(ctx, (void**)dst, n * sizeof(T), what));
  if (n) BIP_CUDA(ctx, cudaMemcpyAsync(*dst, src, n * sizeof(T), cudaMemcpyHostToDevice, ctx->stream));
  return BIP_OK;
}

// the same into a recycled block (edge tables: registered and cleared once per end-to-end step)
template <class T>
static int32_t upload_pooled(bip_ctx* ctx, T** dst, const T* src, size_t n, const char* what) {
  BIP_TRY(pool_alloc(ctx, (void**)dst, n * sizeof(T), what));
  if (n) BIP_CUDA(ctx, cudaMemcpyAsync(*dst, src, n * sizeof(T), cudaMemcpyHostToDevice, ctx->stream));
  return BIP_OK;
}

static int32_t check_weights(bip_ctx* ctx, const bip_weights* w, int32_t n_rows, int32_t n_parent, const char* what) {
  if (!w || !w->nn_idx || !w->nn_w) return fail(ctx, BIP_ERR_INVALID, "%s: weight table is NULL", what);
  if (w->n_rows != n_rows) return fail(ctx, BIP_ERR_INVALID, "%s: weight table has %d rows, expected %d", what, w->n_rows, n_rows);
  if (w->max_nn < 1 || w->max_nn > BIP_MAX_NN) return fail(ctx, BIP_ERR_INVALID, "%s: max_nn %d outside 1..%d", what, w->max_nn, BIP_MAX_NN);
  for (int32_t b = 0; b < n_rows; ++b) {
    double s = 0;
    bool ended = false;
    for (int j = 0; j < w->max_nn; ++j) {
      const int32_t p = w->nn_idx[(size_t)b * w->max_nn + j];
      const float v = w->nn_w[(size_t)b * w->max_nn + j];
      if (p < 0) { ended = true; continue; }
      if (ended) return fail(ctx, BIP_ERR_INVALID, "%s: row %d has an entry after the -1 padding", what, b);
      if (p >= n_parent) return fail(ctx, BIP_ERR_INVALID, "%s: row %d names parent %d >= %d", what, b, p, n_parent);
      if (!(v >= 0.f)) return fail(ctx, BIP_ERR_INVALID, "%s: row %d has a negative or NaN weight", what, b);
      s += v;
    }
    if (std::fabs(s - 1.0) > 1e-5) return fail(ctx, BIP_ERR_INVALID, "%s: row %d sums to %.8f, not 1", what, b, s);
  }
  return BIP_OK;
}


// w == NULL at the ABI: the library computes the Sibson table itself (eq. 8; "computed once per aperture
// and cached").  The Voronoi cells are clipped to 1024 qmax with qmax = the largest |q| of the beam set being
// reconstructed; parents = beams (every beam coincides with a parent) gives the identity table.
static int32_t auto_weights(bip_ctx* ctx, const bip_grid& g, int32_t n, const int32_t* h, int32_t n_par, const int32_t* par_h,
                            std::vector<int32_t>& idx, std::vector<float>& w, int32_t& max_nn) {
  double q2 = 0;
  for (int32_t b = 0; b < n; ++b) {
    const double qy = h[2 * b] / g.ly, qx = h[2 * b + 1] / g.lx;
    q2 = std::max(q2, qy * qy + qx * qx);
  }
  const double qmax = q2 > 0 ? std::sqrt(q2) : 1.0 / std::max(g.ly, g.lx);
  for (int32_t nn : {8, BIP_MAX_NN}) {
    idx.assign((size_t)n * nn, -1);
    w.assign((size_t)n * nn, 0.f);
    const int32_t st = bip_sibson(&g, n, h, n_par, par_h, qmax, nn, idx.data(), w.data());
    if (st == BIP_OK) { max_nn = nn; return BIP_OK; }
    if (nn == BIP_MAX_NN) return fail(ctx, st, "automatic Sibson table: %s", bip_last_error(nullptr));
  }
  return BIP_OK;
}

static uint64_t fnv1a(const void* data, size_t bytes) {
  const unsigned char* p = static_cast<const unsigned char*>(data);
  uint64_t hsh = 1469598103934665603ull;
  for (size_t i = 0; i < bytes; ++i) { hsh ^= p[i]; hsh *= 1099511628211ull; }
  return hsh;
}

static int32_t check_beams(bip_ctx* ctx, const bip_grid& g, int32_t n, const int32_t* h, const char* what) {
  if (n <= 0 || !h) return fail(ctx, BIP_ERR_INVALID, "%s: empty beam list", what);
  for (int32_t i = 0; i < n; ++i)
    if (2 * std::abs(h[2 * i]) >= g.ny || 2 * std::abs(h[2 * i + 1]) >= g.nx)
      return fail(ctx, BIP_ERR_INVALID, "%s: beam %d = (%d, %d) violates |h| < N/2", what, i, h[2 * i], h[2 * i + 1]);
  return BIP_OK;
}

struct Span {
  bip_ctx* ctx; SpanList* v; cudaEvent_t a, b;
  Span(bip_ctx* c, EventPool& pool, SpanList& vec) : ctx(c), v(&vec) {
    a = pool.get(); b = pool.get(); cudaEventRecord(a, c->stream);
  }
  ~Span() { cudaEventRecord(b, ctx->stream); v->push_back({a, b}); }
};

static float sum_ms(SpanList& v) {
  float t = 0;
  for (auto& p : v) { float ms = 0; if (cudaEventElapsedTime(&ms, p.first, p.second) == cudaSuccess) t += ms; }
  return t;
}

// Move the plane cursor.  S1 forward: eq. 6.  S1 backward: either the inverse steps T_j* P* (exact for |T| = 1, checked by
// bip_create) or a restart from the analytic plane waves of plane 0 followed by forward steps, whichever needs fewer
// slice steps -- the restart also discards the rounding accumulated by earlier passes.  S2 forward: the peel
// P*[T_j* .]; backward: the build recursion T_j P[.] itself (eq. 12), exact for any T.  A counter moves only after its
// step has been enqueued successfully.
static int32_t seek_S1(bip_ctx* ctx, int32_t plane) {
  if (!ctx->s1_built) return fail(ctx, BIP_ERR_STATE, "bip_build_S1 must run before the plane loop");
  if (plane < 0 || plane > ctx->g.nz) return fail(ctx, BIP_ERR_INVALID, "plane %d outside 0..%d", plane, ctx->g.nz);
  if (plane < ctx->plane1 && plane <= ctx->plane1 - plane) {
    BIP_TRY(ms_plane_waves(ctx, ctx->S1, ctx->p1_h_dev, ctx->n_p1, +1));
    ctx->plane1 = 0;
  }
  while (ctx->plane1 < plane) { BIP_TRY(ms_step_S1(ctx, ctx->plane1, +1)); ctx->plane1++; }
  while (ctx->plane1 > plane) { BIP_TRY(ms_step_S1(ctx, ctx->plane1 - 1, -1)); ctx->plane1--; }
  return ms_flush(ctx);
}

static int32_t seek(bip_ctx* ctx, int32_t plane) {
  if (!ctx->s1_built || !ctx->s2_built) return fail(ctx, BIP_ERR_STATE, "bip_build_S1 and bip_build_S2 must run before the plane loop");
  BIP_TRY(seek_S1(ctx, plane));
  while (ctx->plane2 < plane) { BIP_TRY(ms_step_S2(ctx, ctx->plane2, +1)); ctx->plane2++; }
  while (ctx->plane2 > plane) { BIP_TRY(ms_step_S2(ctx, ctx->plane2 - 1, -1)); ctx->plane2--; }
  return ms_flush(ctx);
}

// Steps a1-a8 on the sliced 16-bit operands (BIP_PREC_FP16X4 / BIP_PREC_BF16X6).
// NEXT-2: the coupling-matrix association (eq. 13 as printed; Alg. 4 lines 6-8) on the same kernels:
//   X1 = H_n R2 rows (n, d) [k = s],  Y1 = R1 rows b [k = s]   ->  M[(n, d)][b]  (GEMM, c64 out)       n_ch K B W^2
//   X2 = A rows rho [k = b],          Y2 = M rows (n, d) [k = b] ->  |a|^2 reduced per mode (GEMM2 epilogue; the
//   channels run as extra columns c = n K + d)                                                          N_rho n_ch K B
static int32_t contract_coupling(bip_ctx* ctx, Edge& e, const int32_t* org, int32_t nb, int mode, int recon, int fmt, bool drop_tiny,
                                 void* out, const Sliced& Ax, int32_t n_rows, int64_t rho_pad, const int32_t* row_idx_dev,
                                 int64_t row_idx_stride, double n_rows_total) {
  auto& sp = ctx->spans;
  const int w2 = e.w * e.w;
  const int64_t n_nd = (int64_t)e.n_ch * e.n_det;                 // rows (n, d) = n K + d
  Sliced R1r, HR2, Ms;
  BIP_TRY(ensure(ctx, ctx->D1, (size_t)nb * ctx->n_p1 * w2 * sizeof(float2), "D1 (de-tilted S1 windows)"));
  BIP_TRY(ensure(ctx, ctx->D2, (size_t)nb * ctx->n_p2 * w2 * sizeof(float2), "D2 (de-tilted S2 windows)"));
  BIP_TRY(sliced_in(ctx, ctx->R1r, R1r, fmt, ctx->n_ap, w2, nb, "R1 rows (coupling)", SL_ROWS, true));
  BIP_TRY(sliced_in(ctx, ctx->HR2, HR2, fmt, n_nd, w2, nb, "H_n R2 rows (coupling)", 2 * SL_ROWS));
  BIP_TRY(sliced_in(ctx, ctx->Ms, Ms, fmt, n_nd, ctx->n_ap, nb, "coupling matrix (sliced)", SL_ROWS, true));
  const int64_t m_ld = round_up(ctx->n_ap, 2);                   // even pitch: the GEMM epilogue stores pairs of complex values
  BIP_TRY(ensure(ctx, ctx->Mc, (size_t)nb * n_nd * m_ld * sizeof(float2), "coupling matrix"));
  const int64_t n_scale = (int64_t)nb * (R1r.rows_pad + HR2.rows_pad + Ms.rows_pad);
  BIP_TRY(ensure(ctx, ctx->Scl, (size_t)n_scale * sizeof(float), "row scales"));
  R1r.scale = reinterpret_cast<float*>(ctx->Scl.p);           R1r.scale_batch_stride = R1r.rows_pad;
  HR2.scale = R1r.scale + (int64_t)nb * R1r.rows_pad;         HR2.scale_batch_stride = HR2.rows_pad;
  Ms.scale = HR2.scale + (int64_t)nb * HR2.rows_pad;          Ms.scale_batch_stride = Ms.rows_pad;
  // a1-a2, a6: both reconstructions as rows over the window pixels; H_n folded into the S2 side
  BIP_TRY(launch_crop_detilt(ctx, ctx->S1, ctx->p1_h_dev, ctx->n_p1, +1, org, nb, e.w, (float2*)ctx->D1.p));
  BIP_TRY(launch_recon_rows_sliced(ctx, (const float2*)ctx->D1.p, ctx->n_p1, ctx->ap_h_dev, ctx->n_ap, ctx->w1_idx_dev, ctx->w1_w_dev,
                                   ctx->nn1, +1, recon, org, nb, e.w, R1r));
  BIP_TRY(launch_crop_detilt(ctx, ctx->S2, ctx->p2_h_dev, ctx->n_p2, -1, org, nb, e.w, (float2*)ctx->D2.p));
  BIP_TRY(launch_recon_rows_sliced(ctx, (const float2*)ctx->D2.p, ctx->n_p2, e.det_h_dev, e.n_det, e.nn_idx_dev, e.nn_w_dev, e.max_nn,
                                   -1, recon, org, nb, e.w, HR2, e.H_dev, e.n_ch, e.hmax_dev));
  // M[(n, d)][b] = sum_s (H_n R2)[(n, d)][s] R1[b][s]
  Gemm1SlArgs g1;
  g1.A = HR2; g1.R1t = R1r; g1.Psi = (float2*)ctx->Mc.p; g1.psi_ld = m_ld; g1.psi_batch_stride = n_nd * m_ld;
  g1.n_rho = (int32_t)n_nd; g1.w2 = ctx->n_ap; g1.n_atoms = nb; g1.drop_tiny = drop_tiny;
  BIP_TRY(launch_gemm1_sliced(ctx, g1));
  BIP_TRY(launch_quantize_phi(ctx, g1.Psi, g1.psi_ld, g1.psi_batch_stride, nullptr, Ms, (int32_t)n_nd, (int32_t)Ms.rows_pad, ctx->n_ap, 1, nb));
  // a[rho][(n, d)] = G^-1/2 sum_b A[rho][b] M[(n, d)][b]; |a|^2 reduced in the epilogue
  Gemm2SlArgs g2;
  g2.Phi = Ax; g2.R2 = Ms; g2.rows_pad = (int32_t)rho_pad;
  g2.n_rho = n_rows; g2.n_det = (int32_t)n_nd; g2.n_out_cols = e.n_det; g2.n_ch = 1; g2.n_atoms = nb;
  g2.row_idx = row_idx_dev; g2.row_idx_stride = row_idx_stride;
  g2.inv_G = (float)(1.0 / ((double)ctx->g.ny * ctx->g.nx));
  g2.mode = mode;
  g2.bin_of_det = mode == BIP_MODE_QEELS_X ? e.bin_of_det_x_dev : e.bin_of_det_y_dev;
  g2.n_bins = mode == BIP_MODE_QEELS_X ? (int)e.binx.size() : (int)e.biny.size();
  g2.out = out; g2.drop_tiny = drop_tiny;
  {
    Span s(ctx, sp.pool_map, sp.gemm2);
    BIP_TRY(launch_gemm2_sliced(ctx, g2));
  }
  ctx->timing.gemm2_launches++;
  ctx->timing.amplitudes += n_rows_total * e.n_ch * e.n_det;
  ctx->timing.flops += 8.0 * (double)n_nd * ctx->n_ap * ((double)nb * w2 + n_rows_total);
  return BIP_OK;
}

// Which association runs for this edge (bip_set_association): the cost model of include/bip.h.
static bool use_coupling(const bip_ctx* ctx, const Edge& e, double rows_per_site, size_t budget) {
  if (ctx->assoc == BIP_ASSOC_PROBE) return false;
  if (ctx->focal && ctx->assoc == BIP_ASSOC_AUTO) return false;       // focal back-propagation lives on the probe-first path
  const double w2 = (double)e.w * e.w, nd = (double)e.n_ch * e.n_det, B = ctx->n_ap;
  if (ctx->assoc == BIP_ASSOC_AUTO) {
    const double probe = rows_per_site * w2 * (B + nd), coup = nd * B * (w2 + rows_per_site);
    const double bytes = 8.0 * (nd * w2 + B * w2 + 2.0 * nd * B);
    return coup < probe && bytes < (double)budget;
  }
  return true;
}

// Steps a1-a4 for nb sites: S1 windows -> R1^T (sliced) -> probe at the atom Psi[site][rho][s] (c64, pitch w^2) in ctx->Psi.
// R1t must have been carved (sliced_in) and given its scales by the caller.
static int32_t probe_at_sites(bip_ctx* ctx, Edge& e, const int32_t* org, int32_t nb, int recon, bool drop_tiny, const Sliced& Ax,
                              int32_t n_rows, const Sliced& R1t, Gemm1SlArgs* g1_out) {
  const int w2 = e.w * e.w;
  BIP_TRY(ensure(ctx, ctx->Psi, (size_t)nb * n_rows * w2 * sizeof(float2), "Psi (probe at the atom)"));
  const double d_focal = ctx->focal ? ctx->focal_d[ctx->plane1] : 0.0;
  if (d_focal > 0.0) {
    // NEXT-4 (reading c20): per site, de-tilted parent envelopes on the padded window -> Fresnel step back to
    // the scattering-centroid plane -> NNW interpolation (eq. 15 / eq. 11) -> Fresnel step forward, beam by beam ->
    // re-tilt, crop, slice into R1^T
    const int Wp = focal_padded_window(e.w), shift = (Wp - e.w) / 2;
    if (Wp > std::min(ctx->g.ny, ctx->g.nx)) return fail(ctx, BIP_ERR_UNSUPPORTED, "focal back-propagation: padded window %d exceeds the grid", Wp);
    BIP_TRY(ensure(ctx, ctx->D1p, (size_t)ctx->n_p1 * Wp * Wp * sizeof(float2), "padded de-tilted S1 windows"));
    BIP_TRY(ensure(ctx, ctx->Env, (size_t)ctx->n_ap * Wp * Wp * sizeof(float2), "interpolated beam envelopes"));
    std::vector<int32_t> oh(2 * (size_t)nb);
    BIP_CUDA(ctx, cudaMemcpyAsync(oh.data(), org, sizeof(int32_t) * 2 * nb, cudaMemcpyDeviceToHost, ctx->stream));
    BIP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    for (int32_t a = 0; a < nb; ++a) {
      BIP_TRY(launch_crop_detilt(ctx, ctx->S1, ctx->p1_h_dev, ctx->n_p1, +1, org + 2 * (int64_t)a, 1, Wp, (float2*)ctx->D1p.p, shift));
      BIP_TRY(focal_window_fresnel(ctx, (float2*)ctx->D1p.p, ctx->n_p1, ctx->p1_h_dev, ctx->n_p1, Wp, -d_focal));
      BIP_TRY(launch_recon_c64(ctx, (const float2*)ctx->D1p.p, ctx->n_p1, ctx->ap_h_dev, ctx->n_ap, ctx->w1_idx_dev, ctx->w1_w_dev, ctx->nn1, +1,
                               recon, org + 2 * (int64_t)a, 0, Wp, (float2*)ctx->Env.p, shift, /*retilt=*/false));
      BIP_TRY(focal_window_fresnel(ctx, (float2*)ctx->Env.p, ctx->n_ap, ctx->ap_h_dev, ctx->n_ap, Wp, +d_focal));
      BIP_TRY(focal_env_to_r1t(ctx, (const float2*)ctx->Env.p, oh[2 * a], oh[2 * a + 1], e.w, Wp, R1t, a));
    }
  } else {
    BIP_TRY(ensure(ctx, ctx->D1, (size_t)nb * ctx->n_p1 * w2 * sizeof(float2), "D1 (de-tilted S1 windows)"));
    BIP_TRY(launch_crop_detilt(ctx, ctx->S1, ctx->p1_h_dev, ctx->n_p1, +1, org, nb, e.w, (float2*)ctx->D1.p));          // a1
    BIP_TRY(launch_recon_t_sliced(ctx, (const float2*)ctx->D1.p, ctx->n_p1, ctx->ap_h_dev, ctx->n_ap, ctx->w1_idx_dev, ctx->w1_w_dev,
                                  ctx->nn1, +1, recon, org, nb, e.w, R1t));                                                 // a2
  }
  Gemm1SlArgs g1;                                                                                                            // a3-a4
  g1.A = Ax; g1.R1t = R1t; g1.Psi = (float2*)ctx->Psi.p; g1.psi_ld = w2; g1.psi_batch_stride = (int64_t)n_rows * w2;
  g1.n_rho = n_rows; g1.w2 = w2; g1.n_atoms = nb; g1.drop_tiny = drop_tiny;
  BIP_TRY(launch_gemm1_sliced(ctx, g1));
  if (g1_out) *g1_out = g1;
  return BIP_OK;
}

// Crop mask: the number of scan rows inside every site's window, counted on the device once per (edge,
// crop setting, scan) and kept on the host -- the per-batch launches below are then sized without a device round trip.
static int32_t ensure_crop_counts(bip_ctx* ctx, Edge& e) {
  if (e.crop_counts_fy == ctx->crop_fy && e.crop_counts_fx == ctx->crop_fx && (int32_t)e.crop_counts.size() == e.n_atoms) return BIP_OK;
  e.crop_counts.assign(e.n_atoms, 0);
  if (e.n_atoms > 0) {
    BIP_TRY(ensure(ctx, ctx->RowIdx, (size_t)e.n_atoms * sizeof(int32_t), "crop-mask row counts"));
    int32_t* counts_dev = reinterpret_cast<int32_t*>(ctx->RowIdx.p);
    BIP_TRY(launch_crop_rows(ctx, e.origin_dev, e.n_atoms, e.w, nullptr, 0, counts_dev));
    BIP_CUDA(ctx, cudaMemcpyAsync(e.crop_counts.data(), counts_dev, (size_t)e.n_atoms * sizeof(int32_t), cudaMemcpyDeviceToHost, ctx->stream));
    BIP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  }
  e.crop_counts_fy = ctx->crop_fy; e.crop_counts_fx = ctx->crop_fx;
  return BIP_OK;
}

static int32_t contract_batch_sliced(bip_ctx* ctx, Edge& e, const int32_t* org, int32_t a0, int32_t nb, int mode, int recon, int fmt, bool drop_tiny,
                                     bool coupling, void* out) {
  auto& sp = ctx->spans;
  const int w2 = e.w * e.w;
  // scan rows of the contraction: all of them, or (crop mask) each site's own list, gathered into a per-site A operand
  const bool crop = ctx->crop_fy > 1 || ctx->crop_fx > 1;
  int32_t n_rows = ctx->n_rho;
  double n_rows_total = (double)ctx->n_rho * nb;
  const int32_t* row_idx_dev = nullptr;
  int64_t row_idx_stride = 0;
  int64_t rho_pad = round_up(ctx->n_rho, 2 * SL_ROWS);    // X operands are padded to pairs of row tiles (CTA-pair kernel)
  Sliced Ax = ctx->A_sl;
  if (crop) {
    // per-site scan-row lists on the device (k_crop_rows); their lengths are already on the host (ensure_crop_counts)
    const int64_t idx_stride = round_up(ctx->n_rho, 2 * SL_ROWS);
    BIP_TRY(ensure(ctx, ctx->RowIdx, ((size_t)nb * idx_stride + nb) * sizeof(int32_t), "crop-mask row lists"));
    int32_t* rows_dev = reinterpret_cast<int32_t*>(ctx->RowIdx.p);
    int32_t* counts_dev = rows_dev + (size_t)nb * idx_stride;
    BIP_TRY(launch_crop_rows(ctx, org, nb, e.w, rows_dev, idx_stride, counts_dev));
    n_rows = 1; n_rows_total = 0;
    for (int32_t a = a0; a < a0 + nb; ++a) { n_rows = std::max(n_rows, e.crop_counts[a]); n_rows_total += e.crop_counts[a]; }
    rho_pad = round_up(n_rows, 2 * SL_ROWS);
    row_idx_dev = rows_dev;
    row_idx_stride = idx_stride;
    Sliced Ac = ctx->A_sl;
    Ac.rows = n_rows; Ac.rows_pad = rho_pad;
    Ac.batch_stride = rho_pad / SL_ROWS * Ac.ksteps * sl_step_el_of(Ac);
    Ac.scale_batch_stride = rho_pad;
    const size_t op_bytes = (size_t)(Ac.batch_stride * nb) * sizeof(uint16_t), sc_bytes = (size_t)nb * rho_pad * sizeof(float);
    BIP_TRY(ensure(ctx, ctx->Acrop, op_bytes + sc_bytes, "illumination rows of the cropped scans"));
    Ac.base = reinterpret_cast<uint16_t*>(ctx->Acrop.p);
    Ac.scale = reinterpret_cast<float*>(reinterpret_cast<char*>(ctx->Acrop.p) + op_bytes);
    BIP_TRY(launch_gather_rows_sliced(ctx, ctx->A_sl, row_idx_dev, row_idx_stride, Ac, nb));
    Ax = Ac;
  }
  if (coupling)
    return contract_coupling(ctx, e, org, nb, mode, recon, fmt, drop_tiny, out, Ax, n_rows, rho_pad, row_idx_dev, row_idx_stride, n_rows_total);
  Sliced R1t, R2, Phi;
  BIP_TRY(ensure(ctx, ctx->D2, (size_t)nb * ctx->n_p2 * w2 * sizeof(float2), "D2 (de-tilted S2 windows)"));
  BIP_TRY(sliced_in(ctx, ctx->R1s, R1t, fmt, w2, ctx->n_ap, nb, "R1 (reconstructed S1 windows, sliced)", SL_ROWS, true));
  BIP_TRY(sliced_in(ctx, ctx->R2s, R2, fmt, e.n_det, w2, nb, "R2 (reconstructed S2 windows, sliced)", SL_ROWS, true));
  BIP_TRY(sliced_in(ctx, ctx->Phis, Phi, fmt, rho_pad * e.n_ch, w2, nb, "Phi (H_n psi, sliced)"));
  const int64_t psi_ld = w2;
  const int64_t n_scale = (int64_t)nb * (R1t.rows_pad + R2.rows_pad + Phi.rows_pad);
  BIP_TRY(ensure(ctx, ctx->Scl, (size_t)n_scale * sizeof(float), "row scales"));
  R1t.scale = reinterpret_cast<float*>(ctx->Scl.p);           R1t.scale_batch_stride = R1t.rows_pad;
  R2.scale = R1t.scale + (int64_t)nb * R1t.rows_pad;          R2.scale_batch_stride = R2.rows_pad;
  Phi.scale = R2.scale + (int64_t)nb * R2.rows_pad;           Phi.scale_batch_stride = Phi.rows_pad;

  // a1-a4: S1 windows -> R1^T[s][b] -> probe at the atom
  Gemm1SlArgs g1;
  BIP_TRY(probe_at_sites(ctx, e, org, nb, recon, drop_tiny, Ax, n_rows, R1t, &g1));
  // a5: times H_n, split into slices
  BIP_TRY(launch_quantize_phi(ctx, g1.Psi, psi_ld, g1.psi_batch_stride, e.H_dev, Phi, n_rows, (int32_t)rho_pad, w2, e.n_ch, nb));
  // a6: S2 windows -> R2[d][s]
  BIP_TRY(launch_crop_detilt(ctx, ctx->S2, ctx->p2_h_dev, ctx->n_p2, -1, org, nb, e.w, (float2*)ctx->D2.p));
  BIP_TRY(launch_recon_rows_sliced(ctx, (const float2*)ctx->D2.p, ctx->n_p2, e.det_h_dev, e.n_det, e.nn_idx_dev, e.nn_w_dev, e.max_nn,
                                   -1, recon, org, nb, e.w, R2));
  // a7-a8: detector projection and reduction
  Gemm2SlArgs g2;
  g2.Phi = Phi; g2.R2 = R2; g2.rows_pad = (int32_t)rho_pad;
  g2.n_rho = n_rows; g2.n_det = e.n_det; g2.n_ch = e.n_ch; g2.n_atoms = nb;
  g2.row_idx = row_idx_dev; g2.row_idx_stride = row_idx_stride;
  g2.inv_G = (float)(1.0 / ((double)ctx->g.ny * ctx->g.nx));
  g2.mode = mode;
  g2.bin_of_det = mode == BIP_MODE_QEELS_X ? e.bin_of_det_x_dev : e.bin_of_det_y_dev;
  g2.n_bins = mode == BIP_MODE_QEELS_X ? (int)e.binx.size() : (int)e.biny.size();
  g2.out = out; g2.drop_tiny = drop_tiny;
  {
    Span s(ctx, sp.pool_map, sp.gemm2);
    BIP_TRY(launch_gemm2_sliced(ctx, g2));
  }
  ctx->timing.gemm2_launches++;
  ctx->timing.amplitudes += n_rows_total * e.n_ch * e.n_det;
  ctx->timing.flops += 8.0 * n_rows_total * w2 * ((double)ctx->n_ap + (double)e.n_ch * e.n_det);
  return BIP_OK;
}

// Steps a1-a8 for atoms [a0, a0 + nb) of one edge, all sitting in the current plane.
static int32_t contract_batch(bip_ctx* ctx, Edge& e, const int32_t* origin_dev, int32_t a0, int32_t nb, int mode, int recon,
                              int precision, bool coupling, void* out) {
  auto& sp = ctx->spans;
  const int w2 = e.w * e.w;
  const int32_t* org = origin_dev + 2 * (int64_t)a0;
  if (sliced_fmt_of(precision) >= 0) return contract_batch_sliced(ctx, e, org, a0, nb, mode, recon, sliced_fmt_of(precision), precision == BIP_PREC_FP16X3, coupling, out);
  if (ctx->crop_fy > 1 || ctx->crop_fx > 1) return fail(ctx, BIP_ERR_UNSUPPORTED, "bip_map: the crop mask needs a tensor-core precision (FP16X4, FP16X3, BF16X6)");
  if (ctx->assoc == BIP_ASSOC_COUPLING) return fail(ctx, BIP_ERR_UNSUPPORTED, "bip_map: the coupling association needs a tensor-core precision (FP16X4, FP16X3, BF16X6)");
  Planes R1t, R2, Phi;
  BIP_TRY(ensure(ctx, ctx->D1, (size_t)nb * ctx->n_p1 * w2 * sizeof(float2), "D1 (de-tilted S1 windows)"));
  BIP_TRY(ensure(ctx, ctx->D2, (size_t)nb * ctx->n_p2 * w2 * sizeof(float2), "D2 (de-tilted S2 windows)"));
  BIP_TRY(planes_in(ctx, ctx->R1, R1t, w2, ctx->n_ap, nb, "R1 (reconstructed S1 windows)"));
  BIP_TRY(planes_in(ctx, ctx->R2, R2, e.n_det, w2, nb, "R2 (reconstructed S2 windows)"));
  const int64_t rho_rows = ctx->n_rho;
  BIP_TRY(planes_in(ctx, ctx->Phi, Phi, rho_rows * e.n_ch, w2, nb, "Phi (H_n psi)"));

  // a1-a2: S1 windows -> R1^T[s][b]
  BIP_TRY(launch_crop_detilt(ctx, ctx->S1, ctx->p1_h_dev, ctx->n_p1, +1, org, nb, e.w, (float2*)ctx->D1.p));
  BIP_TRY(launch_recon(ctx, (const float2*)ctx->D1.p, ctx->n_p1, ctx->ap_h_dev, ctx->n_ap, ctx->w1_idx_dev, ctx->w1_w_dev,
                       ctx->nn1, +1, recon, org, nb, e.w, /*transpose=*/true, R1t));
  // a3-a5: probe at the atom, times H_n
  Gemm1Args g1;
  g1.A = ctx->A; g1.R1t = R1t; g1.H = e.H_dev; g1.Phi = Phi; g1.phi_ch_stride = rho_rows * Phi.ld;
  g1.n_rho = ctx->n_rho; g1.n_ap = ctx->n_ap; g1.w2 = w2; g1.n_ch = e.n_ch; g1.n_atoms = nb;
  BIP_TRY(precision == BIP_PREC_TF32X3 ? launch_gemm1_tc(ctx, g1) : launch_gemm1_simt(ctx, g1));
  // a6: S2 windows -> R2[d][s]
  BIP_TRY(launch_crop_detilt(ctx, ctx->S2, ctx->p2_h_dev, ctx->n_p2, -1, org, nb, e.w, (float2*)ctx->D2.p));
  BIP_TRY(launch_recon(ctx, (const float2*)ctx->D2.p, ctx->n_p2, e.det_h_dev, e.n_det, e.nn_idx_dev, e.nn_w_dev, e.max_nn, -1,
                       recon, org, nb, e.w, /*transpose=*/false, R2));
  // a7-a8: detector projection and reduction
  Gemm2Args g2;
  g2.Phi = Phi; g2.phi_ch_stride = g1.phi_ch_stride; g2.R2 = R2;
  g2.n_rho = ctx->n_rho; g2.n_det = e.n_det; g2.w2 = w2; g2.n_ch = e.n_ch; g2.n_atoms = nb;
  g2.inv_G = (float)(1.0 / ((double)ctx->g.ny * ctx->g.nx));
  g2.mode = mode;
  g2.bin_of_det = mode == BIP_MODE_QEELS_X ? e.bin_of_det_x_dev : e.bin_of_det_y_dev;
  g2.n_bins = mode == BIP_MODE_QEELS_X ? (int)e.binx.size() : (int)e.biny.size();
  g2.out = out;
  {
    Span s(ctx, sp.pool_map, sp.gemm2);
    BIP_TRY(precision == BIP_PREC_TF32X3 ? launch_gemm2_tc(ctx, g2) : launch_gemm2_simt(ctx, g2));
  }
  ctx->timing.gemm2_launches++;
  ctx->timing.amplitudes += (double)ctx->n_rho * nb * e.n_ch * e.n_det;
  ctx->timing.flops += 8.0 * ctx->n_rho * w2 * ((double)nb * ctx->n_ap + (double)nb * e.n_ch * e.n_det);
  return BIP_OK;
}

static int32_t out_elems(const bip_ctx* ctx, const Edge& e, int mode, int64_t* n, int32_t* nbins, size_t* bytes) {
  int64_t ne = 0; int32_t nb = 0; size_t by = 0;
  switch (mode) {
    case BIP_MODE_MAP: ne = ctx->n_rho; by = ne * sizeof(double); break;
    case BIP_MODE_QEELS_X: nb = (int32_t)e.binx.size(); ne = (int64_t)ctx->n_rho * nb; by = ne * sizeof(float); break;
    case BIP_MODE_QEELS_Y: nb = (int32_t)e.biny.size(); ne = (int64_t)ctx->n_rho * nb; by = ne * sizeof(float); break;
    case BIP_MODE_CUBE: ne = (int64_t)ctx->n_rho * e.n_det; by = ne * sizeof(float); break;
    default: return BIP_ERR_INVALID;
  }
  if (n) *n = ne;
  if (nbins) *nbins = nb;
  if (bytes) *bytes = by;
  return BIP_OK;
}

static int32_t run_edges(bip_ctx* ctx, const std::vector<int32_t>& ids, int mode, int recon, int precision, void* const* outs,
                         const size_t* outs_bytes) {
  if (!ctx->s1_built || !ctx->s2_built) return fail(ctx, BIP_ERR_STATE, "bip_map: call bip_build_S1 and bip_build_S2 first");
  if (ctx->n_rho <= 0) return fail(ctx, BIP_ERR_STATE, "bip_map: call bip_set_scan first");
  if (mode < BIP_MODE_MAP || mode > BIP_MODE_CUBE) return fail(ctx, BIP_ERR_INVALID, "bip_map: unknown mode %d", mode);
  if (recon != BIP_RECON_LINEAR && recon != BIP_RECON_MAGPHASE) return fail(ctx, BIP_ERR_INVALID, "bip_map: unknown recon %d", recon);
  if (precision != BIP_PREC_TF32X3 && precision != BIP_PREC_FP32_SIMT && precision != BIP_PREC_BF16X6 && precision != BIP_PREC_FP16X4 && precision != BIP_PREC_FP16X3) return fail(ctx, BIP_ERR_INVALID, "bip_map: unknown precision %d", precision);
  if (precision == BIP_PREC_FP16X3 && mode == BIP_MODE_CUBE)
    return fail(ctx, BIP_ERR_UNSUPPORTED, "bip_map: FP16X3 drops the x2 y2 products and is offered for the reduced outputs (MAP, QEELS) only; use FP16X4 for the cube");
  if (precision == BIP_PREC_TF32X3 && !ctx->allow_tf32x3)
    return fail(ctx, BIP_ERR_UNSUPPORTED, "bip_map: TF32X3 biases the summed intensity by ~1.25e-8 per accumulating MMA (beyond the 1e-6 bound); "
                "call bip_allow_tf32x3(ctx, 1) to run it as the A/B case, or use FP16X4");
  if (precision != BIP_PREC_FP32_SIMT && !tc_available()) return fail(ctx, BIP_ERR_UNSUPPORTED, "bip_map: the tensor-core path is not built");
  for (size_t k = 0; k < ids.size(); ++k) {
    if (ids[k] < 0 || ids[k] >= (int)ctx->edges.size()) return fail(ctx, BIP_ERR_INVALID, "bip_map: edge %d does not exist", ids[k]);
    size_t need = 0;
    out_elems(ctx, ctx->edges[ids[k]], mode, nullptr, nullptr, &need);
    if (!outs[k]) return fail(ctx, BIP_ERR_INVALID, "bip_map: output %zu is NULL", k);
    if (outs_bytes[k] != need) return fail(ctx, BIP_ERR_INVALID, "bip_map: output %zu has %zu bytes, expected %zu", k, outs_bytes[k], need);
  }
  BIP_TRY(ensure_illumination(ctx, precision));
  auto& sp = ctx->spans;
  sp.adv.clear(); sp.contract.clear(); sp.gemm2.clear();
  sp.pool_map.reset();
  ctx->timing.gemm2_launches = 0; ctx->timing.kernel_launches = 0; ctx->timing.amplitudes = 0; ctx->timing.flops = 0;
  if (ctx->focal && ctx->assoc == BIP_ASSOC_COUPLING) return fail(ctx, BIP_ERR_UNSUPPORTED, "bip_map: focal back-propagation needs the probe-first association");
  if (ctx->focal && sliced_fmt_of(precision) < 0) return fail(ctx, BIP_ERR_UNSUPPORTED, "bip_map: focal back-propagation needs a tensor-core precision (FP16X4, FP16X3, BF16X6)");
  if (!ctx->accumulate)
    for (size_t k = 0; k < ids.size(); ++k) BIP_CUDA(ctx, cudaMemsetAsync(outs[k], 0, outs_bytes[k], ctx->stream));

  std::vector<int32_t> planes;
  for (int32_t id : ids) for (int32_t s : ctx->edges[id].slice) planes.push_back(s);
  std::sort(planes.begin(), planes.end());
  planes.erase(std::unique(planes.begin(), planes.end()), planes.end());
  const size_t budget = ctx->scratch_budget;
  const bool crop = ctx->crop_fy * ctx->crop_fx > 1;
  if (crop && sliced_fmt_of(precision) >= 0)
    for (int32_t id : ids) BIP_TRY(ensure_crop_counts(ctx, ctx->edges[id]));
  for (int32_t plane : planes) {                                         // Alg. 5 line 3
    { Span s(ctx, sp.pool_map, sp.adv); BIP_TRY(seek(ctx, plane)); }                  // line 4: ADVANCETO / PEELTO
    for (size_t k = 0; k < ids.size(); ++k) {
      Edge& e = ctx->edges[ids[k]];
      // atoms are sorted by slice: contiguous range for this plane
      auto lo = std::lower_bound(e.slice.begin(), e.slice.end(), plane) - e.slice.begin();
      auto hi = std::upper_bound(e.slice.begin(), e.slice.end(), plane) - e.slice.begin();
      if (lo == hi) continue;
      const int64_t w2 = (int64_t)e.w * e.w;
      const int64_t el = sliced_fmt_of(precision) == SL_FMT_FP16X4 ? 8 : precision == BIP_PREC_BF16X6 ? 12 : 16;      // operand bytes per complex element
      // scan rows per site of this plane: all of them, or (crop mask) the counted lists -- the association is chosen
      // ONCE per (edge, plane) from the counted rows and the batch is sized for the association that will run
      int64_t rows_max = ctx->n_rho;
      double rows_mean = (double)ctx->n_rho;
      if (crop && sliced_fmt_of(precision) >= 0) {
        rows_max = 1; rows_mean = 0;
        for (auto a = lo; a < hi; ++a) { rows_max = std::max<int64_t>(rows_max, e.crop_counts[a]); rows_mean += e.crop_counts[a]; }
        rows_mean /= (double)(hi - lo);
      }
      const int64_t ely = sliced_fmt_of(precision) >= 0 && sliced_wide(sliced_fmt_of(precision)) ? el * 3 / 2 : el;   // Y operands: + negated imaginary slices
      const size_t per_atom = (size_t)((ctx->n_p1 + ctx->n_p2) * w2 * 8 + rows_max * w2 * 8 +
                                       ely * (round_up(w2, 128) * round_up(ctx->n_ap, 32) + round_up(e.n_det, 128) * round_up(w2, 32)) +
                                       el * (
                                             round_up(rows_max, 256) * (e.n_ch * round_up(w2, 32) + (crop ? round_up(ctx->n_ap, 32) : 0))) +
                                       (crop ? round_up(ctx->n_rho, 256) * 4 : 0));
      const int64_t nd = round_up((int64_t)e.n_ch * e.n_det, 256), Bp = round_up(ctx->n_ap, 128), w2p = round_up(w2, 32);
      const size_t per_atom_coupling = (size_t)((ctx->n_p1 + ctx->n_p2) * w2 * 8 + el * nd * w2p + ely * (Bp * w2p + nd * round_up(ctx->n_ap, 32)) + 8 * nd * Bp +
                                                (crop ? el * round_up(rows_max, 256) * round_up(ctx->n_ap, 32) + round_up(ctx->n_rho, 256) * 4 : 0));
      bool coupling = sliced_fmt_of(precision) >= 0 && use_coupling(ctx, e, rows_mean, budget);
      if (coupling && ctx->assoc == BIP_ASSOC_AUTO && per_atom_coupling > budget) coupling = false;   // does not fit: probe-first does
      const size_t per_atom_use = coupling ? per_atom_coupling : per_atom;
      const int32_t nb_max = (int32_t)std::max<size_t>(1, std::min<size_t>(budget / std::max<size_t>(per_atom_use, 1), 4096));
      Span s(ctx, sp.pool_map, sp.contract);
      for (int32_t a0 = (int32_t)lo; a0 < (int32_t)hi; a0 += nb_max)     // lines 5-8
        BIP_TRY(contract_batch(ctx, e, e.origin_dev, a0, std::min<int32_t>(nb_max, (int32_t)hi - a0), mode, recon, precision, coupling, outs[k]));
    }
  }
  return BIP_OK;
}

// ---- NEXT-3: Algorithm 3 -- S1-partitioned probe, per-scan exit multislice, all G exit beams ----

// fields[(rho, n)][r] = H_n[s] Psi[rho0 + rho][s] on the site's window (r = (origin + s) mod N), zero elsewhere (eq. 3)
__global__ void k_embed_fields(const float2* __restrict__ Psi, int64_t psi_ld, const float2* __restrict__ H, int n_ch, int w, int oy, int ox, int ny,
                               int nx, float2* __restrict__ F) {
  const int rho = blockIdx.y, n = blockIdx.z, w2 = w * w;
  float2* f = F + ((int64_t)rho * n_ch + n) * ny * nx;
  for (int s = blockIdx.x * blockDim.x + threadIdx.x; s < w2; s += gridDim.x * blockDim.x) {
    const int sy = s / w, sx = s - sy * w;
    int ry = oy + sy; if (ry >= ny) ry -= ny;
    int rx = ox + sx; if (rx >= nx) rx -= nx;
    const float2 h = __ldg(H + (int64_t)n * w2 + s), a = Psi[(int64_t)rho * psi_ld + s];
    f[(int64_t)ry * nx + rx] = make_float2(h.x * a.x - h.y * a.y, h.x * a.y + h.y * a.x);
  }
}

static int32_t run_alg3(bip_ctx* ctx, Edge& e, int recon, int precision, float* out) {
  const int fmt = sliced_fmt_of(precision);
  if (fmt < 0 || precision == BIP_PREC_FP16X3) return fail(ctx, BIP_ERR_UNSUPPORTED, "bip_cube_alg3: precision must be FP16X4 or BF16X6");
  if (ctx->crop_fy * ctx->crop_fx > 1) return fail(ctx, BIP_ERR_UNSUPPORTED, "bip_cube_alg3: the crop mask is not applied to the full-grid cube; call bip_set_crop(ctx, 1, 1)");
  BIP_TRY(ensure_illumination(ctx, precision));
  auto& sp = ctx->spans;
  sp.adv.clear(); sp.contract.clear(); sp.gemm2.clear(); sp.pool_map.reset();
  ctx->timing.gemm2_launches = 0; ctx->timing.kernel_launches = 0; ctx->timing.amplitudes = 0; ctx->timing.flops = 0;
  const int ny = ctx->g.ny, nx = ctx->g.nx, nz = ctx->g.nz, w2 = e.w * e.w;
  const int64_t G = (int64_t)ny * nx;
  BIP_CUDA(ctx, cudaMemsetAsync(out, 0, (size_t)ctx->n_rho * G * sizeof(float), ctx->stream));
  // wavefields of one chunk of scan positions: (rho, channel) fields of the whole grid
  const int64_t max_fields = std::max<int64_t>(e.n_ch, (int64_t)(ctx->scratch_budget / 2 / (G * sizeof(float2))));
  const int32_t rho_chunk = (int32_t)std::max<int64_t>(1, std::min<int64_t>(ctx->n_rho, max_fields / e.n_ch));
  BIP_TRY(ensure(ctx, ctx->Fields, (size_t)rho_chunk * e.n_ch * G * sizeof(float2), "exit wavefields (Algorithm 3)"));
  float2* F = reinterpret_cast<float2*>(ctx->Fields.p);
  Sliced R1t;
  BIP_TRY(sliced_in(ctx, ctx->R1s, R1t, fmt, w2, ctx->n_ap, 1, "R1 (reconstructed S1 windows, sliced)", SL_ROWS, true));
  BIP_TRY(ensure(ctx, ctx->Scl, (size_t)R1t.rows_pad * sizeof(float), "row scales"));
  R1t.scale = reinterpret_cast<float*>(ctx->Scl.p); R1t.scale_batch_stride = R1t.rows_pad;
  int32_t a = 0;
  while (a < e.n_atoms) {
    const int32_t plane = e.slice[a];
    { Span s(ctx, sp.pool_map, sp.adv); BIP_TRY(seek_S1(ctx, plane)); }                           // Alg. 3 line 4
    Span sc(ctx, sp.pool_map, sp.contract);
    for (; a < e.n_atoms && e.slice[a] == plane; ++a) {
      Gemm1SlArgs g1;
      BIP_TRY(probe_at_sites(ctx, e, e.origin_dev + 2 * (int64_t)a, 1, recon, false, ctx->A_sl, ctx->n_rho, R1t, &g1));   // lines 5-10 on the window
      for (int32_t r0 = 0; r0 < ctx->n_rho; r0 += rho_chunk) {
        const int32_t nr = std::min(rho_chunk, ctx->n_rho - r0), nf = nr * e.n_ch;
        BIP_CUDA(ctx, cudaMemsetAsync(F, 0, (size_t)nf * G * sizeof(float2), ctx->stream));
        for (int32_t q0 = 0; q0 < nr; q0 += 65535) {
          const int32_t nq = std::min(65535, nr - q0);
          k_embed_fields<<<dim3((unsigned)((w2 + 255) / 256), (unsigned)nq, (unsigned)e.n_ch), 256, 0, ctx->stream>>>(
              g1.Psi + (int64_t)(r0 + q0) * g1.psi_ld, g1.psi_ld, e.H_dev, e.n_ch, e.w, e.origin[2 * a], e.origin[2 * a + 1], ny, nx, F + (int64_t)q0 * e.n_ch * G);
        }
        BIP_CUDA(ctx, cudaGetLastError());
        ctx->timing.kernel_launches++;
        for (int32_t j = plane; j < nz; ++j) BIP_TRY(ms_exit_step(ctx, F, nf, j));               // line 11: to the exit surface
        BIP_TRY(ms_detect(ctx, F, nr, e.n_ch, out + (int64_t)r0 * G));                            // |F psi_n|^2, summed over n
      }
      ctx->timing.amplitudes += (double)ctx->n_rho * e.n_ch * (double)G;
      ctx->timing.flops += 8.0 * ctx->n_rho * w2 * (double)ctx->n_ap;
    }
  }
  return BIP_OK;
}

}  // namespace bip

using namespace bip;

extern "C" {

const char* bip_version(void) {
  static char buf[256];
  static std::once_flag once;
  std::call_once(once, [] {
    int dev = 0, n = 0;
    cudaDeviceProp p{};
    if (cudaGetDeviceCount(&n) == cudaSuccess && n > 0 && cudaGetDevice(&dev) == cudaSuccess && cudaGetDeviceProperties(&p, dev) == cudaSuccess)
      snprintf(buf, sizeof buf, "libbip 0.1 (sm_100a); device %s sm_%d%d; SMs %d; L2 %d MB", p.name, p.major, p.minor, p.multiProcessorCount, p.l2CacheSize >> 20);
    else { cudaGetLastError(); snprintf(buf, sizeof buf, "libbip 0.1 (sm_100a); no CUDA device"); }
  });
  return buf;
}

const char* bip_last_error(const bip_ctx* ctx) { return ctx ? ctx->err.c_str() : g_err.c_str(); }

int32_t bip_create(bip_ctx** out, const bip_grid* g, const void* T, int32_t T_on_device, int32_t n_ap, const int32_t* ap_h,
                   const float* ap_c, int32_t n_p1, const int32_t* p1_h, const bip_weights* w1, int32_t n_p2,
                   const int32_t* p2_h, void* stream) {
  if (!out) return fail(nullptr, BIP_ERR_INVALID, "bip_create: out is NULL");
  *out = nullptr;
  if (!g || g->ny < 8 || g->nx < 8 || g->ny > 8192 || g->nx > 8192 || g->nz < 1 || !(g->ly > 0) || !(g->lx > 0) || !(g->dz > 0) || !(g->lambda > 0))
    return fail(nullptr, BIP_ERR_INVALID, "bip_create: bad grid");
  if (!T) return fail(nullptr, BIP_ERR_INVALID, "bip_create: T is NULL");
  if (!ap_c) return fail(nullptr, BIP_ERR_INVALID, "bip_create: aperture coefficients are NULL");
  BIP_TRY(check_beams(nullptr, *g, n_ap, ap_h, "bip_create: aperture"));
  BIP_TRY(check_beams(nullptr, *g, n_p1, p1_h, "bip_create: S1 parents"));
  BIP_TRY(check_beams(nullptr, *g, n_p2, p2_h, "bip_create: S2 parents"));
  std::vector<int32_t> w1_idx;
  std::vector<float> w1_w;
  int32_t nn1 = 0;
  if (w1) {
    BIP_TRY(check_weights(nullptr, w1, n_ap, n_p1, "bip_create: w1"));
    nn1 = w1->max_nn;
    w1_idx.assign(w1->nn_idx, w1->nn_idx + (size_t)n_ap * nn1);
    w1_w.assign(w1->nn_w, w1->nn_w + (size_t)n_ap * nn1);
  } else {
    BIP_TRY(auto_weights(nullptr, *g, n_ap, ap_h, n_p1, p1_h, w1_idx, w1_w, nn1));
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return fail(nullptr, BIP_ERR_CUDA, "bip_create: no CUDA device (libbip has no CPU path)"); }
  int dev = 0;
  cudaDeviceProp prop{};
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return fail(nullptr, BIP_ERR_CUDA, "bip_create: cannot query the device");
  if (prop.major != 10) return fail(nullptr, BIP_ERR_CUDA, "bip_create: device %s is sm_%d%d; libbip is built for sm_100a only", prop.name, prop.major, prop.minor);

  bip_ctx* ctx = new (std::nothrow) bip_ctx();
  if (!ctx) return fail(nullptr, BIP_ERR_OOM, "bip_create: host allocation failed");
  ctx->g = *g;
  ctx->stream = (cudaStream_t)stream;
  ctx->sm_count = prop.multiProcessorCount;
  ctx->n_ap = n_ap; ctx->n_p1 = n_p1; ctx->n_p2 = n_p2; ctx->nn1 = nn1;
  ctx->w1_idx = w1_idx; ctx->w1_w = w1_w;
  for (int32_t b = 0; b < n_ap; ++b) ctx->ap_c_max = std::max(ctx->ap_c_max, std::hypot(ap_c[2 * b], ap_c[2 * b + 1]));
  ctx->ap_h.assign(ap_h, ap_h + 2 * (size_t)n_ap);
  ctx->p1_h.assign(p1_h, p1_h + 2 * (size_t)n_p1);
  ctx->p2_h.assign(p2_h, p2_h + 2 * (size_t)n_p2);
  const size_t G = (size_t)g->ny * g->nx;
  auto build = [&]() -> int32_t {
    if (T_on_device) ctx->T_dev = (const float2*)T;
    else {
      float2* t = nullptr;
      BIP_TRY(dev_alloc(ctx, (void**)&t, G * g->nz * sizeof(float2), "transmission functions"));
      ctx->T_dev = t; ctx->T_owned = true;
      BIP_CUDA(ctx, cudaMemcpyAsync(t, T, G * g->nz * sizeof(float2), cudaMemcpyHostToDevice, ctx->stream));
    }
    BIP_TRY(upload(ctx, &ctx->ap_h_dev, ap_h, 2 * (size_t)n_ap, "aperture beams"));
    BIP_TRY(upload(ctx, &ctx->p1_h_dev, p1_h, 2 * (size_t)n_p1, "S1 parents"));
    BIP_TRY(upload(ctx, &ctx->p2_h_dev, p2_h, 2 * (size_t)n_p2, "S2 parents"));
    BIP_TRY(upload(ctx, (float**)&ctx->ap_c_dev, ap_c, 2 * (size_t)n_ap, "aperture coefficients"));
    BIP_TRY(upload(ctx, &ctx->w1_idx_dev, ctx->w1_idx.data(), ctx->w1_idx.size(), "w1 indices"));
    BIP_TRY(upload(ctx, &ctx->w1_w_dev, ctx->w1_w.data(), ctx->w1_w.size(), "w1 weights"));
    BIP_TRY(dev_alloc(ctx, (void**)&ctx->S1, (size_t)n_p1 * G * sizeof(float2), "S1 parent columns"));
    BIP_TRY(dev_alloc(ctx, (void**)&ctx->S2, (size_t)n_p2 * G * sizeof(float2), "S2 parent columns"));
    BIP_TRY(ms_init(ctx));
    BIP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    // |T| = 1 (no absorption): the S2 peel and the inverse S1 step undo a slice with conj(T)
    float dev = 0.f;
    BIP_TRY(ms_max_modulus_deviation(ctx, ctx->T_dev, (int64_t)G * g->nz, &dev));
    if (!(dev <= 1e-4f)) return fail(ctx, BIP_ERR_INVALID, "bip_create: transmission functions are not unimodular (max ||T|^2 - 1| = %.3g); "
                                     "absorptive slices are not supported (PAPER.md:372)", dev);
    BIP_TRY(focal_init(ctx));
    return BIP_OK;
  };
  int32_t st = build();
  if (st != BIP_OK) { std::string m = ctx->err; bip_destroy(ctx); g_err = m; return st; }
  *out = ctx;
  return BIP_OK;
}

int32_t bip_clear_edges(bip_ctx* ctx) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  cudaStreamSynchronize(ctx->stream);
  for (Edge& e : ctx->edges) {
    void* blocks[] = {e.H_dev, e.hmax_dev, e.det_h_dev, e.nn_idx_dev, e.nn_w_dev, e.bin_of_det_x_dev, e.bin_of_det_y_dev, e.origin_dev};
    for (void* b : blocks) pool_release(ctx, b);
  }
  ctx->edges.clear();
  return BIP_OK;
}

int32_t bip_destroy(bip_ctx* ctx) {
  if (!ctx) return BIP_OK;
  cudaStreamSynchronize(ctx->stream);
  bip_clear_edges(ctx);
  ms_release(ctx);
  focal_release(ctx);
  ctx->spans.pool_map.destroy(); ctx->spans.pool_b1.destroy(); ctx->spans.pool_b2.destroy();
  if (ctx->T_owned) cudaFree((void*)ctx->T_dev);
  void* ptrs[] = {ctx->ap_h_dev, ctx->p1_h_dev, ctx->p2_h_dev, ctx->ap_c_dev, ctx->w1_idx_dev, ctx->w1_w_dev, ctx->rooty_dev,
                  ctx->rootx_dev, ctx->P_dev, ctx->ms_work, ctx->S1, ctx->S2, ctx->D1.p, ctx->D2.p, ctx->R1.p, ctx->R2.p, ctx->Psi.p,
                  ctx->Phi.p, ctx->R1s.p, ctx->R2s.p, ctx->Phis.p, ctx->Scl.p, ctx->Sync.p, ctx->Fields.p, ctx->D1p.p, ctx->Env.p, ctx->RowIdx.p, ctx->Acrop.p, ctx->Pmax.p, ctx->R1r.p, ctx->HR2.p, ctx->Mc.p, ctx->Ms.p, ctx->rho_dev};
  free_illumination(ctx);
  for (void* p : ptrs) if (p) cudaFree(p);
  for (auto& b : ctx->pool_free) cudaFree(b.first);
  for (auto& b : ctx->pool_size) cudaFree(b.first);
  cudaGetLastError();
  delete ctx;
  return BIP_OK;
}

int32_t bip_build_S1(bip_ctx* ctx) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  auto& sp = ctx->spans;
  sp.build1.clear(); sp.pool_b1.reset();
  { Span s(ctx, sp.pool_b1, sp.build1); BIP_TRY(ms_plane_waves(ctx, ctx->S1, ctx->p1_h_dev, ctx->n_p1, +1)); }
  ctx->plane1 = 0;
  ctx->s1_built = true;
  return BIP_OK;
}

int32_t bip_build_S2(bip_ctx* ctx) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  auto& sp = ctx->spans;
  sp.build2.clear(); sp.pool_b2.reset();
  {
    Span s(ctx, sp.pool_b2, sp.build2);
    BIP_TRY(ms_plane_waves(ctx, ctx->S2, ctx->p2_h_dev, ctx->n_p2, -1));
    ctx->plane2 = ctx->g.nz;
    while (ctx->plane2 > 0) { ctx->plane2--; BIP_TRY(ms_step_S2(ctx, ctx->plane2, -1)); }
    BIP_TRY(ms_flush(ctx));
  }
  ctx->s2_built = true;
  return BIP_OK;
}

int32_t bip_set_scan(bip_ctx* ctx, int32_t n_rho, const double* rho_px) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  if (n_rho <= 0 || !rho_px) return fail(ctx, BIP_ERR_INVALID, "bip_set_scan: empty scan");
  for (int32_t i = 0; i < 2 * n_rho; ++i) if (!std::isfinite(rho_px[i])) return fail(ctx, BIP_ERR_INVALID, "bip_set_scan: non-finite position");
  cudaStreamSynchronize(ctx->stream);
  free_illumination(ctx);
  if (ctx->rho_dev) { cudaFree(ctx->rho_dev); ctx->rho_dev = nullptr; }
  ctx->n_rho = 0;
  BIP_TRY(dev_alloc(ctx, (void**)&ctx->rho_dev, sizeof(double) * 2 * n_rho, "scan positions"));
  BIP_CUDA(ctx, cudaMemcpyAsync(ctx->rho_dev, rho_px, sizeof(double) * 2 * n_rho, cudaMemcpyHostToDevice, ctx->stream));
  BIP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));      // the host array may go away after return
  ctx->n_rho = n_rho;
  ctx->rho_host.assign(rho_px, rho_px + 2 * (size_t)n_rho);
  for (Edge& e : ctx->edges) e.crop_counts_fy = e.crop_counts_fx = 0;      // the per-site scan-row counts depend on the scan
  return BIP_OK;                                           // the illumination matrix (a3) is built on first use
}

int32_t bip_prism_subsample(int32_t n, const int32_t* h, int32_t fy, int32_t fx, int32_t* keep_out, int32_t cap, int32_t* n_keep) {
  if (n < 0 || (n > 0 && !h) || fy < 1 || fx < 1 || !n_keep) return fail(nullptr, BIP_ERR_INVALID, "bip_prism_subsample: bad argument");
  int32_t m = 0;
  for (int32_t b = 0; b < n; ++b)
    if (h[2 * b] % fy == 0 && h[2 * b + 1] % fx == 0) {
      if (keep_out && m < cap) keep_out[m] = b;
      ++m;
    }
  *n_keep = m;
  if (keep_out && m > cap) return fail(nullptr, BIP_ERR_INVALID, "bip_prism_subsample: %d beams retained, capacity %d", m, cap);
  return BIP_OK;
}

int32_t bip_set_association(bip_ctx* ctx, int32_t assoc) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  if (assoc < BIP_ASSOC_PROBE || assoc > BIP_ASSOC_AUTO) return fail(ctx, BIP_ERR_INVALID, "bip_set_association: unknown association %d", assoc);
  ctx->assoc = assoc;
  return BIP_OK;
}

int32_t bip_set_crop(bip_ctx* ctx, int32_t fy, int32_t fx) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  if (fy < 1 || fx < 1 || fy > ctx->g.ny / 2 || fx > ctx->g.nx / 2) return fail(ctx, BIP_ERR_INVALID, "bip_set_crop: factors (%d, %d) outside 1..N/2", fy, fx);
  ctx->crop_fy = fy; ctx->crop_fx = fx;
  return BIP_OK;
}

int32_t bip_add_edge(bip_ctx* ctx, int32_t n_atoms, const int32_t* slice, const int32_t* centre_px, int32_t n_ch, int32_t w,
                     const float* H, int32_t n_det, const int32_t* det_h, const bip_weights* w2, int32_t* edge_id) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  if (n_atoms < 0 || (n_atoms > 0 && (!slice || !centre_px))) return fail(ctx, BIP_ERR_INVALID, "bip_add_edge: bad site list");
  if (n_ch < 1 || n_ch > 1024 || !H) return fail(ctx, BIP_ERR_INVALID, "bip_add_edge: bad channel count or H is NULL");
  if (w < 8 || (w & 1) || w > std::min(ctx->g.ny, ctx->g.nx)) return fail(ctx, BIP_ERR_INVALID, "bip_add_edge: window %d must be even and in 8..min(ny, nx)", w);
  BIP_TRY(check_beams(ctx, ctx->g, n_det, det_h, "bip_add_edge: detector"));
  Edge e;
  if (w2) {
    BIP_TRY(check_weights(ctx, w2, n_det, ctx->n_p2, "bip_add_edge: w2"));
    e.max_nn = w2->max_nn;
    e.w2_idx.assign(w2->nn_idx, w2->nn_idx + (size_t)n_det * w2->max_nn);
    e.w2_w.assign(w2->nn_w, w2->nn_w + (size_t)n_det * w2->max_nn);
  } else {
    // computed once per detector beam list and cached on the context
    const uint64_t key = fnv1a(det_h, sizeof(int32_t) * 2 * (size_t)n_det) ^ (uint64_t)n_det;
    auto it = ctx->auto_w2.find(key);
    if (it == ctx->auto_w2.end() || it->second.det_h.size() != 2 * (size_t)n_det || std::memcmp(it->second.det_h.data(), det_h, sizeof(int32_t) * 2 * (size_t)n_det) != 0) {
      bip::AutoTable t;
      t.det_h.assign(det_h, det_h + 2 * (size_t)n_det);
      BIP_TRY(auto_weights(ctx, ctx->g, n_det, det_h, ctx->n_p2, ctx->p2_h.data(), t.idx, t.w, t.max_nn));
      it = ctx->auto_w2.insert_or_assign(key, std::move(t)).first;
    }
    e.max_nn = it->second.max_nn; e.w2_idx = it->second.idx; e.w2_w = it->second.w;
  }
  e.n_atoms = n_atoms; e.n_ch = n_ch; e.w = w; e.n_det = n_det;
  // sort sites by slice (stable): the plane loop takes contiguous ranges
  std::vector<int32_t> order(n_atoms);
  for (int i = 0; i < n_atoms; ++i) order[i] = i;
  for (int i = 0; i < n_atoms; ++i) {
    if (slice[i] < 0 || slice[i] >= ctx->g.nz) return fail(ctx, BIP_ERR_INVALID, "bip_add_edge: site %d in slice %d outside 0..%d", i, slice[i], ctx->g.nz - 1);
    if (centre_px[2 * i] < 0 || centre_px[2 * i] >= ctx->g.ny || centre_px[2 * i + 1] < 0 || centre_px[2 * i + 1] >= ctx->g.nx)
      return fail(ctx, BIP_ERR_INVALID, "bip_add_edge: site %d centre outside the grid", i);
  }
  std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return slice[a] < slice[b]; });
  e.slice.resize(n_atoms); e.origin.resize(2 * (size_t)n_atoms);
  for (int i = 0; i < n_atoms; ++i) {
    const int a = order[i];
    e.slice[i] = slice[a];
    e.origin[2 * i] = ((centre_px[2 * a] - w / 2) % ctx->g.ny + ctx->g.ny) % ctx->g.ny;
    e.origin[2 * i + 1] = ((centre_px[2 * a + 1] - w / 2) % ctx->g.nx + ctx->g.nx) % ctx->g.nx;
  }
  e.det_h.assign(det_h, det_h + 2 * (size_t)n_det);
  // qEELS bins: distinct signed indices along the resolved axis, ascending
  std::vector<int32_t> bx(n_det), by(n_det);
  for (int d = 0; d < n_det; ++d) { by[d] = det_h[2 * d]; bx[d] = det_h[2 * d + 1]; }
  e.binx = bx; std::sort(e.binx.begin(), e.binx.end()); e.binx.erase(std::unique(e.binx.begin(), e.binx.end()), e.binx.end());
  e.biny = by; std::sort(e.biny.begin(), e.biny.end()); e.biny.erase(std::unique(e.biny.begin(), e.biny.end()), e.biny.end());
  for (int d = 0; d < n_det; ++d) {
    bx[d] = (int32_t)(std::lower_bound(e.binx.begin(), e.binx.end(), bx[d]) - e.binx.begin());
    by[d] = (int32_t)(std::lower_bound(e.biny.begin(), e.biny.end(), by[d]) - e.biny.begin());
  }
  BIP_TRY(upload_pooled(ctx, (float**)&e.H_dev, H, 2 * (size_t)n_ch * w * w, "H windows"));
  std::vector<float> hmax(n_ch, 0.f);
  for (int n = 0; n < n_ch; ++n)
    for (size_t s = 0; s < (size_t)w * w; ++s) {
      const float* h = H + 2 * ((size_t)n * w * w + s);
      hmax[n] = std::max(hmax[n], 1.0001f * std::hypot(h[0], h[1]));
    }
  BIP_TRY(upload_pooled(ctx, &e.hmax_dev, hmax.data(), (size_t)n_ch, "H maxima"));
  BIP_TRY(upload_pooled(ctx, &e.det_h_dev, det_h, 2 * (size_t)n_det, "detector beams"));
  BIP_TRY(upload_pooled(ctx, &e.nn_idx_dev, e.w2_idx.data(), e.w2_idx.size(), "w2 indices"));
  BIP_TRY(upload_pooled(ctx, &e.nn_w_dev, e.w2_w.data(), e.w2_w.size(), "w2 weights"));
  BIP_TRY(upload_pooled(ctx, &e.bin_of_det_x_dev, bx.data(), (size_t)n_det, "qEELS bins"));
  BIP_TRY(upload_pooled(ctx, &e.bin_of_det_y_dev, by.data(), (size_t)n_det, "qEELS bins"));
  BIP_TRY(upload_pooled(ctx, &e.origin_dev, e.origin.data(), 2 * (size_t)n_atoms, "window origins"));
  BIP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));     // host sources may go away after return
  ctx->edges.push_back(std::move(e));
  if (edge_id) *edge_id = (int32_t)ctx->edges.size() - 1;
  return BIP_OK;
}

int32_t bip_output_size(const bip_ctx* ctx, int32_t edge_id, int32_t mode, int64_t* n_elems, int32_t* n_bins) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  if (edge_id < 0 || edge_id >= (int)ctx->edges.size()) return fail(const_cast<bip_ctx*>(ctx), BIP_ERR_INVALID, "edge %d does not exist", edge_id);
  if (ctx->n_rho <= 0) return fail(const_cast<bip_ctx*>(ctx), BIP_ERR_STATE, "bip_output_size: call bip_set_scan first");
  if (out_elems(ctx, ctx->edges[edge_id], mode, n_elems, n_bins, nullptr) != BIP_OK) return fail(const_cast<bip_ctx*>(ctx), BIP_ERR_INVALID, "unknown mode %d", mode);
  return BIP_OK;
}

int32_t bip_map(bip_ctx* ctx, int32_t edge_id, int32_t mode, int32_t recon, int32_t precision, void* out_dev, size_t out_bytes) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  std::vector<int32_t> ids{edge_id};
  void* outs[1] = {out_dev};
  size_t by[1] = {out_bytes};
  return run_edges(ctx, ids, mode, recon, precision, outs, by);
}

int32_t bip_map_all(bip_ctx* ctx, int32_t mode, int32_t recon, int32_t precision, void* const* outs_dev, const size_t* outs_bytes,
                    int32_t n_outs) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  if (n_outs != (int32_t)ctx->edges.size() || !outs_dev || !outs_bytes) return fail(ctx, BIP_ERR_INVALID, "bip_map_all: need one output per edge (%zu)", ctx->edges.size());
  std::vector<int32_t> ids(n_outs);
  for (int i = 0; i < n_outs; ++i) ids[i] = i;
  return run_edges(ctx, ids, mode, recon, precision, outs_dev, outs_bytes);
}

int32_t bip_map_host(bip_ctx* ctx, int32_t edge_id, int32_t mode, int32_t recon, int32_t precision, void* out_host, size_t out_bytes) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  if (!out_host) return fail(ctx, BIP_ERR_INVALID, "bip_map_host: output is NULL");
  void* d = nullptr;
  BIP_TRY(pool_alloc(ctx, &d, out_bytes, "host-call output staging"));
  int32_t st = bip_map(ctx, edge_id, mode, recon, precision, d, out_bytes);
  if (st == BIP_OK) {
    cudaError_t e = cudaMemcpyAsync(out_host, d, out_bytes, cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) st = fail(ctx, BIP_ERR_CUDA, "bip_map_host: %s", cudaGetErrorString(e));
  }
  cudaStreamSynchronize(ctx->stream);
  pool_release(ctx, d);
  return st;
}

int32_t bip_cube_alg3(bip_ctx* ctx, int32_t edge_id, int32_t recon, int32_t precision, float* out_dev, size_t out_bytes) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  if (edge_id < 0 || edge_id >= (int)ctx->edges.size()) return fail(ctx, BIP_ERR_INVALID, "bip_cube_alg3: edge %d does not exist", edge_id);
  if (!ctx->s1_built) return fail(ctx, BIP_ERR_STATE, "bip_cube_alg3: call bip_build_S1 first (S2 is not used by Algorithm 3)");
  if (ctx->n_rho <= 0) return fail(ctx, BIP_ERR_STATE, "bip_cube_alg3: call bip_set_scan first");
  if (recon != BIP_RECON_LINEAR && recon != BIP_RECON_MAGPHASE) return fail(ctx, BIP_ERR_INVALID, "bip_cube_alg3: unknown recon %d", recon);
  const size_t need = (size_t)ctx->n_rho * ctx->g.ny * ctx->g.nx * sizeof(float);
  if (!out_dev || out_bytes != need) return fail(ctx, BIP_ERR_INVALID, "bip_cube_alg3: output has %zu bytes, expected %zu", out_bytes, need);
  if (!tc_available()) return fail(ctx, BIP_ERR_UNSUPPORTED, "bip_cube_alg3: the tensor-core path is not built");
  return run_alg3(ctx, ctx->edges[edge_id], recon, precision, out_dev);
}

int32_t bip_get_windows(const bip_ctx* ctx, int32_t edge_id, int32_t* origin_out) {
  if (!ctx || !origin_out) return fail(nullptr, BIP_ERR_INVALID, "bip_get_windows: NULL argument");
  if (edge_id < 0 || edge_id >= (int)ctx->edges.size()) return fail(const_cast<bip_ctx*>(ctx), BIP_ERR_INVALID, "edge %d does not exist", edge_id);
  const Edge& e = ctx->edges[edge_id];
  std::copy(e.origin.begin(), e.origin.end(), origin_out);
  return BIP_OK;
}

int32_t bip_get_qeels_bins(const bip_ctx* ctx, int32_t edge_id, int32_t mode, int32_t* bins_out) {
  if (!ctx || !bins_out) return fail(nullptr, BIP_ERR_INVALID, "bip_get_qeels_bins: NULL argument");
  if (edge_id < 0 || edge_id >= (int)ctx->edges.size()) return fail(const_cast<bip_ctx*>(ctx), BIP_ERR_INVALID, "edge %d does not exist", edge_id);
  const Edge& e = ctx->edges[edge_id];
  if (mode == BIP_MODE_QEELS_X) std::copy(e.binx.begin(), e.binx.end(), bins_out);
  else if (mode == BIP_MODE_QEELS_Y) std::copy(e.biny.begin(), e.biny.end(), bins_out);
  else return fail(const_cast<bip_ctx*>(ctx), BIP_ERR_INVALID, "mode %d has no bins", mode);
  return BIP_OK;
}

int32_t bip_seek_plane(bip_ctx* ctx, int32_t plane) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  return seek(ctx, plane);
}

int32_t bip_copy_S(bip_ctx* ctx, int32_t which, int32_t p0, int32_t np, void* out_host) {
  if (!ctx || !out_host) return fail(ctx, BIP_ERR_INVALID, "bip_copy_S: NULL argument");
  const int32_t n = which == 1 ? ctx->n_p1 : which == 2 ? ctx->n_p2 : -1;
  if (n < 0) return fail(ctx, BIP_ERR_INVALID, "bip_copy_S: which must be 1 or 2");
  if ((which == 1 && !ctx->s1_built) || (which == 2 && !ctx->s2_built)) return fail(ctx, BIP_ERR_STATE, "bip_copy_S: matrix not built");
  if (p0 < 0 || np < 0 || p0 + np > n) return fail(ctx, BIP_ERR_INVALID, "bip_copy_S: columns %d..%d outside 0..%d", p0, p0 + np, n);
  const size_t G = (size_t)ctx->g.ny * ctx->g.nx;
  const float2* S = which == 1 ? ctx->S1 : ctx->S2;
  BIP_CUDA(ctx, cudaMemcpyAsync(out_host, S + (size_t)p0 * G, (size_t)np * G * sizeof(float2), cudaMemcpyDeviceToHost, ctx->stream));
  BIP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  return BIP_OK;
}

int32_t bip_debug_reconstruct(bip_ctx* ctx, int32_t edge_id, int32_t atom, int32_t which, int32_t recon, void* out_host) {
  if (!ctx || !out_host) return fail(ctx, BIP_ERR_INVALID, "bip_debug_reconstruct: NULL argument");
  if (edge_id < 0 || edge_id >= (int)ctx->edges.size()) return fail(ctx, BIP_ERR_INVALID, "edge %d does not exist", edge_id);
  Edge& e = ctx->edges[edge_id];
  if (atom < 0 || atom >= e.n_atoms) return fail(ctx, BIP_ERR_INVALID, "atom %d does not exist", atom);
  if (which != 1 && which != 2) return fail(ctx, BIP_ERR_INVALID, "which must be 1 or 2");
  if (!ctx->s1_built || !ctx->s2_built) return fail(ctx, BIP_ERR_STATE, "matrices not built");
  const int w2 = e.w * e.w;
  const int32_t* org = e.origin_dev + 2 * (int64_t)atom;
  const int n_par = which == 1 ? ctx->n_p1 : ctx->n_p2;
  const int n_beams = which == 1 ? ctx->n_ap : e.n_det;
  DevBuf& D = which == 1 ? ctx->D1 : ctx->D2;
  BIP_TRY(ensure(ctx, D, (size_t)n_par * w2 * sizeof(float2), "D"));
  float2* R = nullptr;
  BIP_TRY(dev_alloc(ctx, (void**)&R, (size_t)n_beams * w2 * sizeof(float2), "debug reconstruction"));
  int32_t st = launch_crop_detilt(ctx, which == 1 ? ctx->S1 : ctx->S2, which == 1 ? ctx->p1_h_dev : ctx->p2_h_dev, n_par,
                                  which == 1 ? +1 : -1, org, 1, e.w, (float2*)D.p);
  if (st == BIP_OK)
    st = launch_recon_c64(ctx, (const float2*)D.p, n_par, which == 1 ? ctx->ap_h_dev : e.det_h_dev, n_beams,
                          which == 1 ? ctx->w1_idx_dev : e.nn_idx_dev, which == 1 ? ctx->w1_w_dev : e.nn_w_dev,
                          which == 1 ? ctx->nn1 : e.max_nn, which == 1 ? +1 : -1, recon, org, 0, e.w, R);
  if (st == BIP_OK) {
    cudaError_t er = cudaMemcpyAsync(out_host, R, (size_t)n_beams * w2 * sizeof(float2), cudaMemcpyDeviceToHost, ctx->stream);
    if (er == cudaSuccess) er = cudaStreamSynchronize(ctx->stream);
    if (er != cudaSuccess) st = fail(ctx, BIP_ERR_CUDA, "bip_debug_reconstruct: %s", cudaGetErrorString(er));
  }
  cudaStreamSynchronize(ctx->stream);
  cudaFree(R);
  return st;
}

int32_t bip_get_parents(const bip_ctx* ctx, int32_t which, int32_t* h_out, int32_t cap, int32_t* n_out) {
  if (!ctx || !n_out) return fail(nullptr, BIP_ERR_INVALID, "bip_get_parents: NULL argument");
  if (which != 1 && which != 2) return fail(const_cast<bip_ctx*>(ctx), BIP_ERR_INVALID, "bip_get_parents: which must be 1 or 2");
  const std::vector<int32_t>& ph = which == 1 ? ctx->p1_h : ctx->p2_h;
  *n_out = (int32_t)(ph.size() / 2);
  if (h_out) {
    if (cap < *n_out) return fail(const_cast<bip_ctx*>(ctx), BIP_ERR_INVALID, "bip_get_parents: capacity %d < %d parents", cap, *n_out);
    std::copy(ph.begin(), ph.end(), h_out);
  }
  return BIP_OK;
}

int32_t bip_get_weights(const bip_ctx* ctx, int32_t edge_id, int32_t* n_rows, int32_t* max_nn, int32_t* nn_idx_out, float* nn_w_out) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "bip_get_weights: ctx is NULL");
  if (edge_id >= (int)ctx->edges.size()) return fail(const_cast<bip_ctx*>(ctx), BIP_ERR_INVALID, "edge %d does not exist", edge_id);
  const std::vector<int32_t>& idx = edge_id < 0 ? ctx->w1_idx : ctx->edges[edge_id].w2_idx;
  const std::vector<float>& w = edge_id < 0 ? ctx->w1_w : ctx->edges[edge_id].w2_w;
  const int32_t rows = edge_id < 0 ? ctx->n_ap : ctx->edges[edge_id].n_det, nn = edge_id < 0 ? ctx->nn1 : ctx->edges[edge_id].max_nn;
  if (n_rows) *n_rows = rows;
  if (max_nn) *max_nn = nn;
  if (nn_idx_out) std::copy(idx.begin(), idx.end(), nn_idx_out);
  if (nn_w_out) std::copy(w.begin(), w.end(), nn_w_out);
  return BIP_OK;
}

int32_t bip_set_focal(bip_ctx* ctx, int32_t on) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  ctx->focal = on != 0;
  return BIP_OK;
}

int32_t bip_get_focal_distance(const bip_ctx* ctx, int32_t plane, double* d_out) {
  if (!ctx || !d_out) return fail(nullptr, BIP_ERR_INVALID, "bip_get_focal_distance: NULL argument");
  if (plane < 0 || plane > ctx->g.nz) return fail(const_cast<bip_ctx*>(ctx), BIP_ERR_INVALID, "plane %d outside 0..%d", plane, ctx->g.nz);
  *d_out = ctx->focal_d[plane];
  return BIP_OK;
}

int32_t bip_set_accumulate(bip_ctx* ctx, int32_t on) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  ctx->accumulate = on != 0;
  return BIP_OK;
}

int32_t bip_set_transmission(bip_ctx* ctx, const void* T, int32_t T_on_device) {
  if (!ctx || !T) return fail(ctx, BIP_ERR_INVALID, "bip_set_transmission: NULL argument");
  const size_t n = (size_t)ctx->g.ny * ctx->g.nx * ctx->g.nz;
  BIP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  if (T_on_device) {
    if (ctx->T_owned) cudaFree((void*)ctx->T_dev);
    ctx->T_dev = (const float2*)T; ctx->T_owned = false;
  } else {
    if (!ctx->T_owned) { float2* t = nullptr; BIP_TRY(dev_alloc(ctx, (void**)&t, n * sizeof(float2), "transmission functions")); ctx->T_dev = t; ctx->T_owned = true; }
    BIP_CUDA(ctx, cudaMemcpyAsync((void*)ctx->T_dev, T, n * sizeof(float2), cudaMemcpyHostToDevice, ctx->stream));
    BIP_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  }
  ctx->s1_built = ctx->s2_built = false;                       // the scattering matrices belong to the previous configuration
  float dev = 0.f;
  BIP_TRY(ms_max_modulus_deviation(ctx, ctx->T_dev, (int64_t)n, &dev));
  if (!(dev <= 1e-4f)) return fail(ctx, BIP_ERR_INVALID, "bip_set_transmission: transmission functions are not unimodular (max ||T|^2 - 1| = %.3g)", dev);
  return focal_init(ctx);
}

int32_t bip_set_fft_backend(bip_ctx* ctx, int32_t backend) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  if (backend != BIP_FFT_NATIVE && backend != BIP_FFT_CUFFT_F64) return fail(ctx, BIP_ERR_INVALID, "bip_set_fft_backend: unknown backend %d", backend);
  if (backend == BIP_FFT_NATIVE && !fft_supported(ctx))
    return fail(ctx, BIP_ERR_UNSUPPORTED, "bip_set_fft_backend: the native slice step needs a power-of-two grid (8..4096), this one is %d x %d", ctx->g.ny, ctx->g.nx);
  BIP_TRY(ms_flush(ctx));
  ctx->fft_native = backend == BIP_FFT_NATIVE;
  return BIP_OK;
}

int32_t bip_allow_tf32x3(bip_ctx* ctx, int32_t allow) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  ctx->allow_tf32x3 = allow != 0;
  return BIP_OK;
}

int32_t bip_set_scratch_budget(bip_ctx* ctx, size_t bytes) {
  if (!ctx) return fail(nullptr, BIP_ERR_INVALID, "ctx is NULL");
  if (bytes < ((size_t)32 << 20)) return fail(ctx, BIP_ERR_INVALID, "bip_set_scratch_budget: %zu bytes is below the 32 MB minimum", bytes);
  ctx->scratch_budget = bytes;
  return BIP_OK;
}

int32_t bip_get_timing(const bip_ctx* cctx, bip_timing* out) {
  if (!cctx || !out) return fail(nullptr, BIP_ERR_INVALID, "bip_get_timing: NULL argument");
  bip_ctx* ctx = const_cast<bip_ctx*>(cctx);
  cudaStreamSynchronize(ctx->stream);
  auto& sp = ctx->spans;
  ctx->timing.build_s1_ms = sum_ms(sp.build1);
  ctx->timing.build_s2_ms = sum_ms(sp.build2);
  ctx->timing.advance_peel_ms = sum_ms(sp.adv);
  ctx->timing.contract_ms = sum_ms(sp.contract);
  ctx->timing.gemm2_ms = sum_ms(sp.gemm2);
  *out = ctx->timing;
  return BIP_OK;
}

}  // extern "C"
