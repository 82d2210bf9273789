// Internal declarations of libbip (not part of the ABI).
#ifndef BIP_INTERNAL_H_
#define BIP_INTERNAL_H_

#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <map>
#include <string>
#include <utility>
#include <vector>

#include "../../include/bip.h"
#include "bip_sliced.cuh"

namespace bip {

// Records the message on the context (or a thread-local slot when ctx == nullptr) and returns `status`.
int32_t fail(bip_ctx* ctx, int32_t status, const char* fmt, ...) __attribute__((format(printf, 3, 4)));

// Launch-shape experiments (raster group, workers, lag, ...) read BIP_TUNE_* environment variables ONLY in a build
// compiled with -DBIP_TUNING (python -m paper_2607_00756_b200.build --tuning); the shipped library ignores them.
inline int tune_int(const char* name, int dflt) {
#ifdef BIP_TUNING
  if (const char* e = std::getenv(name)) return std::atoi(e);
#else
  (void)name;
#endif
  return dflt;
}

// The N = 256 formulation of the FP16X4 CTA-pair kernel (Y operands with negated imaginary slices, bip_sliced.cuh) is an
// A/B variant: measured 3.4 % (FP16X4) and 5.5 % (FP16X3) SLOWER than the N = 128 formulation on B200
// (profiles/r02_wide_mma.md), so the shipped build never selects it; BIP_TUNE_WIDE=1 in a tuning build does.
inline bool sliced_wide(int fmt) { return fmt == SL_FMT_FP16X4 && tune_int("BIP_TUNE_WIDE", 0) != 0 && tune_int("BIP_TUNE_PAIR", 1) != 0; }

}  // namespace bip

#ifdef __CUDACC__
#include <cuda_runtime.h>
#include <cufft.h>

namespace bip {

// Split-plane operand: a complex matrix [rows][ld] stored as four fp32 planes
//   re_hi, re_lo, im_hi, im_lo  with hi = tf32(x) and lo = tf32(x - hi) (cvt.rna: round-to-nearest, so the tensor
// core's truncation of the low 13 mantissa bits never acts and the split stays unbiased; hi + lo = x to 2^-22).
// The tensor-core kernels feed the planes to tcgen05 kind::tf32 as they are (3xTF32 split); the fp32 SIMT
// reference kernels read hi + lo.  `ld` is a multiple of 32 floats (128 B) and plane bases are 1024 B aligned.
struct Planes {
  float* p[4] = {nullptr, nullptr, nullptr, nullptr};   // re_hi, re_lo, im_hi, im_lo
  int64_t rows = 0;      // rows per batch item (padded to a multiple of 128)
  int64_t ld = 0;        // floats per row
  int64_t batch_stride = 0;   // floats between batch items inside one plane (0 = shared)
};

struct DevBuf {
  void* p = nullptr;
  size_t bytes = 0;
  uint64_t sig = 0;      // layout signature of the planes last carved out of it
};

struct Edge {
  int32_t n_atoms = 0, n_ch = 0, w = 0, n_det = 0, max_nn = 0;
  std::vector<int32_t> slice;          // [n_atoms]
  std::vector<int32_t> origin;         // [n_atoms][2] window origin (centre - w/2) mod N
  std::vector<int32_t> det_h;          // [n_det][2]
  std::vector<int32_t> binx, biny;     // distinct h_x / h_y ascending
  std::vector<int32_t> w2_idx;         // [n_det][max_nn] host copy of the ELL table (bip_get_weights)
  std::vector<float> w2_w;
  std::vector<int32_t> crop_counts;    // [n_atoms] scan rows inside each site's crop window (filled on first use per crop setting)
  int32_t crop_counts_fy = 0, crop_counts_fx = 0;
  int32_t* origin_dev = nullptr;       // [n_atoms][2]
  float2* H_dev = nullptr;             // [n_ch][w*w]
  float* hmax_dev = nullptr;           // [n_ch] max_s |H_n[s]| (row-scale bound of the coupling operands)
  int32_t* det_h_dev = nullptr;        // [n_det][2]
  int32_t* nn_idx_dev = nullptr;       // [n_det][max_nn]
  float* nn_w_dev = nullptr;           // [n_det][max_nn]
  int32_t* bin_of_det_x_dev = nullptr; // [n_det] bin number along x
  int32_t* bin_of_det_y_dev = nullptr;
};

struct EventPool {
  std::vector<cudaEvent_t> all;
  size_t used = 0;
  cudaEvent_t get() {
    if (used == all.size()) { cudaEvent_t e; cudaEventCreate(&e); all.push_back(e); }
    return all[used++];
  }
  void reset() { used = 0; }
  void destroy() { for (auto e : all) cudaEventDestroy(e); all.clear(); used = 0; }
};
typedef std::vector<std::pair<cudaEvent_t, cudaEvent_t>> SpanList;
struct Spans {
  EventPool pool_map, pool_b1, pool_b2;
  SpanList adv, contract, gemm2, build1, build2;
};
struct AutoTable { std::vector<int32_t> det_h, idx; std::vector<float> w; int32_t max_nn = 0; };   // library-computed w2, per detector list
struct KernelInfo { bool attr_set = false; int max_clusters = -1; };   // per (context = device, kernel variant)

}  // namespace bip

// Inverse row pass of a native slice step that has not run yet (bip_fft.cu: consecutive steps on the same columns share it)
struct FftPending { float2* S = nullptr; int n_cols = 0; const float2* T = nullptr; int post = 0; bool active = false; };

struct bip_ctx {
  bip_grid g{};
  cudaStream_t stream = nullptr;
  int sm_count = 0;
  std::string err;

  const float2* T_dev = nullptr;   // [nz][ny][nx]
  bool T_owned = false;

  // aperture / parents
  int32_t n_ap = 0, n_p1 = 0, n_p2 = 0, nn1 = 0;
  std::vector<int32_t> ap_h, p1_h, p2_h;
  int32_t *ap_h_dev = nullptr, *p1_h_dev = nullptr, *p2_h_dev = nullptr;
  float2* ap_c_dev = nullptr;
  float ap_c_max = 0.f;            // max_b |c_b|
  int32_t* w1_idx_dev = nullptr;
  float* w1_w_dev = nullptr;
  std::vector<int32_t> w1_idx;     // host copies (bip_get_weights)
  std::vector<float> w1_w;

  // roots of unity exp(2 pi i k / N), k = 0..N-1 (exact phases for tilt / de-tilt)
  float2 *rooty_dev = nullptr, *rootx_dev = nullptr;
  void* P_dev = nullptr;           // Fresnel propagator / G as double2 [ny][nx]
  void* ms_work = nullptr;         // double2 workspace of the cuFFT slice steps [plan_batch][ny][nx], allocated on first use
  // native fused slice step for power-of-two grids (bip_fft.cu)
  float4 *fft_rooty = nullptr, *fft_rootx = nullptr, *fft_Ey = nullptr, *fft_Ex = nullptr;   // double-float (hi, lo) twiddles and the two 1-D factors of the propagator
  int32_t *fft_permy = nullptr, *fft_permx = nullptr;   // true frequency index of every stored (digit-reversed) position
  int fft_lines = 0, fft_cols = 0;
  // device blocks of per-call objects (edge tables, the staging buffer of bip_map_host), recycled instead of freed: a
  // cudaFree / cudaMalloc pair per bip_add_edge / bip_clear_edges cost up to 0.8 s of driver time in the end-to-end step
  std::vector<std::pair<void*, size_t>> pool_free;
  std::map<void*, size_t> pool_size;
  FftPending fft_pending;          // inverse row pass owed by the last native slice step (fft_flush)
  bool fft_native = false;         // route in use (bip_set_fft_backend)
  float2 *S1 = nullptr, *S2 = nullptr;
  bool s1_built = false, s2_built = false;
  int32_t plane1 = 0, plane2 = 0;  // S1 holds slices 0..plane1-1; S2 holds slices plane2..nz-1
  std::map<int, cufftHandle> plans;   // cuFFT plans by batch size
  int32_t plan_batch = 0;
  bool plan_ok = false;
  size_t scratch_budget = (size_t)12 << 30;   // bip_set_scratch_budget
  bool allow_tf32x3 = false;          // bip_allow_tf32x3
  bool accumulate = false;            // bip_set_accumulate: bip_map adds to the output instead of zeroing it (frozen phonons)
  bool focal = false;                 // bip_set_focal: S1 reconstructed through the scattering-centroid plane (NEXT-4)
  std::vector<double> focal_d;        // [nz + 1] back-propagation distance of every plane (reading c20)
  std::map<int, std::pair<void*, void*>> focal_tables;   // per padded-window size: twiddles, digit-reversal permutation
  bip::DevBuf D1p, Env;               // padded de-tilted parent windows; interpolated beam envelopes (one site)
  bip::Spans spans;                   // CUDA-event spans behind bip_get_timing
  std::map<const void*, bip::KernelInfo> kernel_info;
  std::map<uint64_t, bip::AutoTable> auto_w2;

  // scan
  int32_t n_rho = 0;
  double* rho_dev = nullptr;       // [n_rho][2] scan positions in pixels
  std::vector<double> rho_host;    // the same on the host (crop-mask row lists)
  int32_t crop_fy = 1, crop_fx = 1;  // PRISM crop mask (bip_set_crop); 1 = off
  int32_t assoc = 0;                 // bip_assoc (bip_set_association)
  bip::DevBuf R1r, HR2, Mc, Ms;      // coupling association: R1 rows, H_n R2 rows, M (c64) and M sliced
  bip::DevBuf Pmax;                // max_s |D2[p][s]| per (site, parent): row-scale bound of R2
  bip::DevBuf RowIdx, Acrop;       // per-site scan-row lists and gathered illumination rows (crop mask)
  bip::Planes A;                   // illumination [n_rho][n_ap] split planes (K-major over b); built on first use
  bip::Sliced A_sl;                // the same as a sliced 16-bit operand (format A_sl.fmt); built on first use

  std::vector<bip::Edge> edges;

  // scratch, grown on demand
  bip::DevBuf D1, D2, R1, R2, Psi, Phi;
  bip::DevBuf R1s, R2s, Phis, Scl;  // sliced operands of the tensor-core path and their row scales
  bip::DevBuf Fields;               // wavefields of the per-scan exit multislice (Algorithm 3)
  bip::DevBuf Sync;                 // lockstep counters of the persistent contraction kernel (one per launch slot)
  int sync_slot = 0;

  bip_timing timing{};
  cudaEvent_t ev[8] = {};
};

namespace bip {

#define BIP_CUDA(ctx, call)                                                                          \
  do {                                                                                               \
    cudaError_t e_ = (call);                                                                         \
    if (e_ != cudaSuccess) {                                                                         \
      (void)cudaGetLastError(); /* do not leave it for an unrelated later check */                   \
      return bip::fail((ctx), e_ == cudaErrorMemoryAllocation ? BIP_ERR_OOM : BIP_ERR_CUDA,          \
                       "%s:%d %s: %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_));           \
    }                                                                                                \
  } while (0)

#define BIP_TRY(call)                  \
  do {                                 \
    int32_t s_ = (call);               \
    if (s_ != BIP_OK) return s_;       \
  } while (0)

int32_t dev_alloc(bip_ctx* ctx, void** p, size_t bytes, const char* what);
int32_t ensure(bip_ctx* ctx, DevBuf& b, size_t bytes, const char* what);

// ---- multislice (bip_multislice.cu) ----
int32_t ms_init(bip_ctx* ctx);                       // propagator, roots of unity, cuFFT plan
int32_t ms_plane_waves(bip_ctx* ctx, float2* S, const int32_t* h_dev, int32_t n, int sign);
// max over the n elements of | |T|^2 - 1 | (synchronises the stream)
int32_t ms_max_modulus_deviation(bip_ctx* ctx, const float2* T, int64_t n, float* out);
// forward: S <- P[T_j S] (dir=+1) ; inverse: S <- T_j* P*[S] (dir=-1)               (S1, eq. 6)
int32_t ms_step_S1(bip_ctx* ctx, int32_t j, int dir);
// build/un-peel: S <- T_j P[S] (dir=-1, towards the entrance) ; peel: S <- P*[T_j* S] (dir=+1)   (S2, eq. 12)
int32_t ms_step_S2(bip_ctx* ctx, int32_t j, int dir);
// exit multislice of Algorithm 3 on arbitrary wavefields: F <- P[T_j F] for n fields [n][ny][nx]
int32_t ms_exit_step(bip_ctx* ctx, float2* fields, int n, int32_t j);
// out[rho][ky][kx] += sum_n |F fields[rho][n]|^2 / G (unitary F, corner-origin order); fields are destroyed
int32_t ms_detect(bip_ctx* ctx, float2* fields, int n_rho, int n_ch, float* out);
int32_t pool_alloc(bip_ctx* ctx, void** p, size_t bytes, const char* what);   // recycled device block (bip_api.cu)
void pool_release(bip_ctx* ctx, void* p);
int32_t ms_flush(bip_ctx* ctx);       // end of a sequence of slice steps: every column is complete in memory afterwards

// ---- native fused slice step for power-of-two grids (bip_fft.cu) ----
bool fft_supported(const bip_ctx* ctx);
int32_t fft_init(bip_ctx* ctx);
int32_t fft_slice_op(bip_ctx* ctx, float2* S, int n_cols, const float2* Tj, int pre, int conj_p, int post);
int32_t fft_detect(bip_ctx* ctx, float2* fields, int n_rho, int n_ch, float* out);
int32_t fft_flush(bip_ctx* ctx);      // run the inverse row pass the last fft_slice_op left owing (chained slice steps share row passes)
void fft_release(bip_ctx* ctx);

// ---- S1 focal back-propagation (bip_focal.cu) ----
int32_t focal_padded_window(int32_t w);
int32_t focal_init(bip_ctx* ctx);
int32_t focal_window_fresnel(bip_ctx* ctx, float2* E, int64_t n_win, const int32_t* h_dev, int n_beams, int Wp, double d);
int32_t focal_env_to_r1t(bip_ctx* ctx, const float2* Env, int32_t oy, int32_t ox, int32_t w, int32_t Wp, const Sliced& out, int32_t atom);
void focal_release(bip_ctx* ctx);

// ---- reconstruction (bip_recon.cu) ----
// a1: D[a][p][s] = S_p(r) * exp(-carrier 2 pi i h_p.r/N) on the atoms' windows
int32_t launch_crop_detilt(bip_ctx* ctx, const float2* S, const int32_t* ph_dev, int32_t n_par, int carrier,
                           const int32_t* origin_dev, int32_t n_atoms, int32_t w, float2* D, int32_t origin_shift = 0);
// a2/a6: R[a][beam][s] (or transposed [a][s][beam]) split planes from D with ELL weights, re-tilted
int32_t launch_recon(bip_ctx* ctx, const float2* D, int32_t n_par, const int32_t* bh_dev, int32_t n_beams,
                     const int32_t* nn_idx, const float* nn_w, int32_t max_nn, int carrier, int recon,
                     const int32_t* origin_dev, int32_t n_atoms, int32_t w, bool transpose, Planes out);
int32_t launch_recon_c64(bip_ctx* ctx, const float2* D, int32_t n_par, const int32_t* bh_dev, int32_t n_beams,
                         const int32_t* nn_idx, const float* nn_w, int32_t max_nn, int carrier, int recon,
                         const int32_t* origin_dev, int32_t atom, int32_t w, float2* out, int32_t origin_shift = 0, bool retilt = true);
// a3: illumination planes A[rho][b] = c_b exp(-2 pi i h_b.rho/N)
int32_t launch_illumination(bip_ctx* ctx, const double* rho_dev, int32_t n_rho, Planes out);

// ---- contractions ----
struct Gemm1Args {       // a4 + a5: Psi = A . R1 ; Phi_n = H_n . Psi -> split planes [atom][n][rho][s]
  Planes A;              // [n_rho][n_ap]
  Planes R1t;            // [atom][s][b]   (K-major over b)
  const float2* H;       // [n_ch][w*w]
  Planes Phi;            // [atom][n][n_rho][w*w]: batch_stride per atom, rows = n_ch * rows_per_ch
  int64_t phi_ch_stride; // floats between channels inside one atom
  int32_t n_rho, n_ap, w2, n_ch, n_atoms;
};
struct Gemm2Args {       // a7 + a8: a_n = g Phi_n . R2^T ; |a|^2 reduced per mode
  Planes Phi;
  int64_t phi_ch_stride;
  Planes R2;             // [atom][d][s]
  int32_t n_rho, n_det, w2, n_ch, n_atoms;
  float inv_G;           // 1 / (ny nx): |a|^2 scale of the unitary DFT
  int32_t mode;
  const int32_t* bin_of_det;   // QEELS
  int32_t n_bins;
  void* out;             // MAP double[n_rho]; QEELS float[n_rho][n_bins]; CUBE float[n_rho][n_det]
};
int32_t launch_gemm1_simt(bip_ctx* ctx, const Gemm1Args& a);
int32_t launch_gemm2_simt(bip_ctx* ctx, const Gemm2Args& a);
int32_t launch_gemm1_tc(bip_ctx* ctx, const Gemm1Args& a);
int32_t launch_gemm2_tc(bip_ctx* ctx, const Gemm2Args& a);
bool tc_available();

// ---- contractions on sliced 16-bit operands (bip_gemm_sliced.cu) ----
struct Gemm1SlArgs {     // a4: Psi = A . R1   (c64 [atom][rho][s])
  Sliced A;              // rows rho, k = aperture beams
  Sliced R1t;            // rows s, k = aperture beams, batch = atoms
  float2* Psi;
  int64_t psi_ld, psi_batch_stride;
  int32_t n_rho, w2, n_atoms;
  int32_t drop_tiny = 0; // BIP_PREC_FP16X3
};
struct Gemm2SlArgs {     // a7 + a8
  Sliced Phi;            // rows (n, rho) = n * rows_pad + rho, k = window pixels, batch = atoms
  Sliced R2;             // rows d, k = window pixels, batch = atoms
  int32_t rows_pad;      // padded rho rows per channel
  int32_t n_rho, n_det, n_ch, n_atoms;
  float inv_G;
  int32_t mode;
  const int32_t* bin_of_det;
  int32_t n_bins;
  void* out;
  int32_t drop_tiny = 0; // BIP_PREC_FP16X3
  int32_t n_out_cols = 0;             // 0: = n_det; else column c is detector beam c % n_out_cols (coupling association)
  const int32_t* row_idx = nullptr;   // crop mask: [atom][row_idx_stride] output scan index of each local row, -1 = none
  int64_t row_idx_stride = 0;
};
int32_t launch_crop_rows(bip_ctx* ctx, const int32_t* origin_dev, int32_t n_atoms, int32_t w, int32_t* row_idx, int64_t idx_stride, int32_t* counts);
int32_t launch_gather_rows_sliced(bip_ctx* ctx, const Sliced& src, const int32_t* row_idx, int64_t idx_stride, const Sliced& dst, int32_t n_atoms);
int32_t launch_gemm1_sliced(bip_ctx* ctx, const Gemm1SlArgs& a);
int32_t launch_gemm2_sliced(bip_ctx* ctx, const Gemm2SlArgs& a);
int32_t launch_quantize_phi(bip_ctx* ctx, const float2* Psi, int64_t psi_ld, int64_t psi_batch_stride, const float2* H,
                            const Sliced& Phi, int32_t n_rho, int32_t rows_pad, int32_t w2, int32_t n_ch, int32_t n_atoms);
int32_t launch_recon_t_sliced(bip_ctx* ctx, const float2* D, int32_t n_par, const int32_t* bh_dev, int32_t n_beams,
                              const int32_t* nn_idx, const float* nn_w, int32_t max_nn, int carrier, int recon,
                              const int32_t* origin_dev, int32_t n_atoms, int32_t w, Sliced out);
int32_t launch_recon_rows_sliced(bip_ctx* ctx, const float2* D, int32_t n_par, const int32_t* bh_dev, int32_t n_beams,
                                 const int32_t* nn_idx, const float* nn_w, int32_t max_nn, int carrier, int recon,
                                 const int32_t* origin_dev, int32_t n_atoms, int32_t w, Sliced out, const float2* H = nullptr, int32_t n_ch = 1,
                                 const float* hmax = nullptr);
int32_t launch_illumination_sliced(bip_ctx* ctx, const double* rho_dev, int32_t n_rho, float scale, Sliced out);

}  // namespace bip
#endif  // __CUDACC__
#endif  // BIP_INTERNAL_H_
