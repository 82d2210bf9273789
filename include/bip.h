/*
 * bip.h -- C ABI of libbip: the on-atom contraction of BiP-PRISM (arxiv/paper_2607_00756) on one B200.
 *
 * The library computes Algorithm 5 of the paper ("BiP-PRISM EELS map"): the probe-forming
 * scattering matrix S1 and the adjoint detector matrix S2 are held on sparse parent beams, advanced / peeled
 * plane by plane (eq. 6, eq. 12), and for every ionised atom both are reconstructed on the W x W window
 * Omega_tau by natural-neighbour weights (eq. 15, or the magnitude-preserving eq. 11), combined with the
 * illumination coefficients c_b(rho) into the probe at the atom (eq. 7), multiplied by the transition potentials
 * H_n (eq. 3), projected on S2 (eq. 13) and reduced over detector beams into an elemental map, qEELS bins or the
 * energy-filtered 4D cube (eq. 14, section 2.2.6).
 *
 * Conventions (DESIGN.md section 3 lists every reading of the paper):
 *   - pixel r = (ry, rx), beam h = (hy, hx) signed integer index on the corner-origin DFT grid, |h| < N/2;
 *     h.r/N = hy ry / ny + hx rx / nx.  All [.][2] arrays are (y, x).
 *   - complex data is interleaved (re, im); "c64" = two floats.
 *   - the DFT is unitary: a_d = G^-1/2 sum_r S2^d(r) H psi.
 *   - every function returns a bip_status; nothing throws across the ABI.  Arguments are validated on the host
 *     before any launch.  bip_last_error() returns a NUL-terminated description of the last failure on that
 *     context (or of the last failed bip_create / helper call on this thread when ctx == NULL).
 *   - pointers are HOST pointers unless the name ends in _dev.  The library copies every host array it is
 *     given before returning; device buffers passed in are borrowed (never freed) and must stay valid as stated.
 *   - one context per host thread (a context keeps all of its state -- plans, events, scratch -- in itself; different
 *     contexts may be used from different threads at the same time); all device work is enqueued on the CUDA stream given to bip_create
 *     (a cudaStream_t passed as void*; NULL = the legacy default stream).  Calls return after enqueueing unless
 *     stated otherwise; the caller synchronises the stream before reading device outputs.
 *   - there is NO CPU fallback: every entry point that touches a scattering matrix or an output needs a CUDA
 *     device of compute capability 10.x and fails with BIP_ERR_CUDA otherwise.
 */
#ifndef BIP_H_
#define BIP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define BIP_API __attribute__((visibility("default")))
#else
#define BIP_API
#endif

typedef enum {
  BIP_OK = 0,
  BIP_ERR_INVALID = 1,      /* NULL pointer, bad shape, value out of range                        */
  BIP_ERR_STATE = 2,        /* call order (e.g. bip_map before bip_build_S1 / S2 / bip_set_scan)  */
  BIP_ERR_OOM = 3,          /* device or host allocation failed; message states the bytes asked   */
  BIP_ERR_CUDA = 4,         /* CUDA / cuFFT error, or no sm_100 device                            */
  BIP_ERR_UNSUPPORTED = 5   /* valid request the build cannot serve                               */
} bip_status;

typedef enum { BIP_MODE_MAP = 0, BIP_MODE_QEELS_X = 1, BIP_MODE_QEELS_Y = 2, BIP_MODE_CUBE = 3 } bip_mode;
typedef enum { BIP_RECON_LINEAR = 0, BIP_RECON_MAGPHASE = 1 } bip_recon;
/* Association of the triple product sum_s sum_b S2^d(s) H_n(s) S1^b(s) c_b(rho) (eq. 13):
 * PROBE     probe first: Psi[rho, s] = sum_b c_b(rho) S1^b(s), then a = sum_s S2^d H_n Psi (the paper's contract="probe",
 *           PAPER.md:519); cost per site ~ N_rho W^2 (B + N_ch K).  The default.
 * COUPLING  eq. 13 as printed / Alg. 4 lines 6-8: the scan-independent coupling matrix M^(n,tau)[d, b] = sum_s S2^d H_n S1^b
 *           first, then a = M c(rho) for all scans; cost per site ~ N_ch K B (W^2 + N_rho).  Pays when a site sees few scan
 *           positions (crop mask, small rasters).  Needs N_ch K W^2 operand elements of scratch per site.
 * AUTO      per edge, whichever of the two has the lower cost by these formulas (and fits the scratch budget). */
typedef enum { BIP_ASSOC_PROBE = 0, BIP_ASSOC_COUPLING = 1, BIP_ASSOC_AUTO = 2 } bip_assoc;
/* Arithmetic of the two contractions (all fp32-equivalent).
 * FP16X4 (the one to use): tcgen05 tensor cores on operands split, against a power-of-two row scale, into a 9-bit
 *   fixed-point leading slice and an fp16 residual slice (representation error 2^-21 of the row maximum); a real
 *   product is the four-term sum x1 y1 + (x1 y2 + x2 y1 + x2 y2) -- 2/3 of the tensor time of 3xTF32.  The leading
 *   products x1 y1 are small integers and accumulate EXACTLY in TMEM over chunks of 128 k-elements; chunk sums are
 *   added in fp32 round-to-nearest.  Meets the 1e-6 summed-intensity bound.
 * FP16X3: FP16X4 without the x2 y2 term (each at most 2^-18 of the leading product, zero-mean): three MMAs per real
 *   product, 3/4 of the tensor time of FP16X4.  The analogue of the customary 3xTF32 scheme, which drops lo x lo.
 *   Offered for the detector-reduced outputs (MAP, QEELS_X / _Y), where it is held to the same parity bounds by the
 *   tests (1e-4 per pixel, 1e-6 summed); BIP_MODE_CUBE returns BIP_ERR_UNSUPPORTED (single cube pixels of tiny
 *   windows exceed 1e-4 without the x2 y2 term).
 * BF16X6: the same construction with three bf16 slices per real number (8-bit leading slice, chunks of 256
 *   k-elements) and the six-term product x1 y1 + (x1 y2 + x2 y1) + (x1 y3 + x2 y2 + x3 y1): representation error
 *   2^-24 of the row maximum at the tensor time of 3xTF32.
 * TF32X3: every real product as a_hi b_hi + a_hi b_lo + a_lo b_hi of TF32 operands, accumulated in one TMEM chain.
 *   The tensor core truncates on accumulation (profiles/r01_tcgen05_rounding_probe.txt): per-pixel error within
 *   1e-4 but the summed intensity is biased by ~ -1.25e-8 per accumulating MMA (-2.6e-5 at configs[0]): it does NOT
 *   meet the 1e-6 summed-intensity bound.  Kept as the measured A/B case for that finding; bip_map refuses it with
 *   BIP_ERR_UNSUPPORTED unless bip_allow_tf32x3(ctx, 1) has been called.
 * FP32_SIMT: the same contractions on CUDA cores in fp32 -- the A/B reference for the tensor-core kernels. */
typedef enum { BIP_PREC_TF32X3 = 0, BIP_PREC_FP32_SIMT = 1, BIP_PREC_BF16X6 = 2, BIP_PREC_FP16X4 = 3, BIP_PREC_FP16X3 = 4 } bip_precision;

typedef struct bip_ctx bip_ctx;

/* Real-space grid, cell and slicing. lengths in Angstrom. */
typedef struct {
  int32_t ny, nx;     /* pixels                                     */
  double ly, lx;      /* field of view                              */
  int32_t nz;         /* number of slices                           */
  double dz;          /* slice thickness                            */
  double lambda;      /* electron wavelength                        */
} bip_grid;

/* A natural-neighbour weight table in ELL form (eq. 8): row b lists the parents
 * surrounding beam b. nn_idx[b][j] is a parent NUMBER (position in the parent list) or -1 for padding;
 * nn_w[b][j] >= 0 and each row sums to 1 (+-1e-5, validated). */
typedef struct {
  int32_t n_rows;          /* number of beams being reconstructed            */
  int32_t max_nn;          /* row width, 1..BIP_MAX_NN                       */
  const int32_t* nn_idx;   /* [n_rows][max_nn]                               */
  const float* nn_w;       /* [n_rows][max_nn]                               */
} bip_weights;

#define BIP_MAX_NN 16

/* Event timings of the last bip_map in milliseconds, and of the builds. */
typedef struct {
  float build_s1_ms;       /* bip_build_S1                                              */
  float build_s2_ms;       /* bip_build_S2 (adjoint multislice from the exit surface)   */
  float advance_peel_ms;   /* S1.ADVANCETO + S2.PEELTO inside the last bip_map          */
  float contract_ms;       /* steps a1-a8 (crop .. reduce) inside the last bip_map      */
  float gemm2_ms;          /* the detector projection kernel alone (dominant kernel)    */
  int32_t gemm2_launches;  /* launches of that kernel in the last bip_map               */
  int32_t kernel_launches; /* all of the library's own kernel launches in the last bip_map (cuFFT excluded) */
  double amplitudes;       /* scan x atom x channel x detector-beam amplitudes formed (scans inside the crop mask only) */
  double flops;            /* algorithmic real flops of the association that ran: probe-first 8 rows W^2 (B + N_ch K),
                              coupling 8 N_ch K B (sites W^2 + rows); rows = scan rows contracted (crop mask) */
} bip_timing;

/* ------------------------------------------------------------------------------------------------------------
 * Geometry helpers (host only, no device needed).  They implement the readings of SURVEY.md 8(c) c5-c8.
 * ---------------------------------------------------------------------------------------------------------- */

/* Beams with |h| < N/2 and (hy/ly)^2 + (hx/lx)^2 <= qmax^2 in ascending flat corner-origin index
 * (hy mod ny) * nx + (hx mod nx)  (eq. 5; Alg. 4 line 1).
 * h_out [cap][2]; *n_out receives the count even when cap is too small (then BIP_ERR_INVALID). */
BIP_API int32_t bip_beams_in_disc(const bip_grid* g, double qmax, int32_t* h_out, int32_t cap, int32_t* n_out);

/* Probe coefficients c_b = exp(-i pi lambda defocus |q_b|^2) / sqrt(G n) (eq. 1), c_out [n][2]. */
BIP_API int32_t bip_aperture_coeffs(const bip_grid* g, int32_t n, const int32_t* h, double defocus, float* c_out);

/* Hex-ring parent selection: DC + n_radial rings at |q| = k qmax / n_radial with n_angular k
 * samples from +x, snapped to the nearest beam of h[n][2] (ties: lowest flat index), deduplicated.
 * pos_out [cap] receives ascending positions into h; *n_out the count. */
BIP_API int32_t bip_hexring(const bip_grid* g, int32_t n, const int32_t* h, double qmax, int32_t n_radial,
                    int32_t n_angular, int32_t* pos_out, int32_t cap, int32_t* n_out);

/* n_radial = max(1, round(sqrt(n_beams / pi) / factor)) (parent spacing "factor" in beam pixels). */
BIP_API int32_t bip_n_radial_from_factor(int32_t n_beams, double factor);

/* Parent partition of a beam set by its "parent factor" f (BASELINE.json configs; reading c7) in one call:
 *   f == 1   the exactness limit: parents = all beams, w = identity;
 *   f  > 1   hex-ring parents with n_radial = bip_n_radial_from_factor(n, f), n_angular = 6, and their
 *            Sibson table (eq. 8).
 * pos_out [cap] parent positions into h (ascending), *n_parent their number; nn_idx_out / nn_w_out [n][max_nn]. */
BIP_API int32_t bip_partition(const bip_grid* g, int32_t n, const int32_t* h, double qmax, double factor, int32_t max_nn,
                              int32_t* pos_out, int32_t cap, int32_t* n_parent, int32_t* nn_idx_out, float* nn_w_out);

/* Sibson natural-neighbour weights (eq. 8) of every beam h[n][2] on the parents parent_h[n_parent][2], in
 * physical q coordinates, cells clipped to |q| <= 1024 qmax, delta on a parent, weights < 1e-12 dropped and the
 * row renormalised; row entries in ascending parent number, padded with (-1, 0).
 * nn_idx_out / nn_w_out [n][max_nn].  Fails with BIP_ERR_INVALID if a row needs more than max_nn entries. */
BIP_API int32_t bip_sibson(const bip_grid* g, int32_t n, const int32_t* h, int32_t n_parent, const int32_t* parent_h,
                   double qmax, int32_t max_nn, int32_t* nn_idx_out, float* nn_w_out);

/* ------------------------------------------------------------------------------------------------------------
 * Context
 * ---------------------------------------------------------------------------------------------------------- */

/* Create a context (Alg. 5 "Require").
 *   T          transmission functions T_j = exp(i sigma V_j), c64 [nz][ny][nx].
 *              T_on_device != 0: a device pointer, borrowed for the lifetime of the context.
 *              T_on_device == 0: a host pointer, copied to a device buffer the context owns.
 *   n_ap, ap_h, ap_c   aperture beams h_b [n_ap][2] and coefficients c_b [n_ap][2] (eq. 1).
 *   n_p1, p1_h         S1 parent beams [n_p1][2] (any beams, normally a hex-ring subset of the aperture).
 *   w1                 weights of every aperture beam on the S1 parents (n_rows == n_ap); NULL: the library computes
 *                      the Sibson table itself (bip_sibson with qmax = the largest |q| of the aperture beams).
 *   n_p2, p2_h         S2 parent (detector-side) beams [n_p2][2].
 *   stream             cudaStream_t as void*.
 * T must be unimodular (|T| = 1: phase objects without absorption) -- the S2 peel and the backward S1
 * step undo a slice with conj(T); max ||T|^2 - 1| > 1e-4 is rejected with BIP_ERR_INVALID.
 * The context allocates and owns S1 (n_p1 columns) and S2 (n_p2 columns), c64 [.][ny][nx] each. */
BIP_API int32_t bip_create(bip_ctx** out, const bip_grid* g, const void* T, int32_t T_on_device,
                   int32_t n_ap, const int32_t* ap_h, const float* ap_c,
                   int32_t n_p1, const int32_t* p1_h, const bip_weights* w1,
                   int32_t n_p2, const int32_t* p2_h, void* stream);

BIP_API int32_t bip_destroy(bip_ctx* ctx);

BIP_API const char* bip_last_error(const bip_ctx* ctx);

/* S1 parents <- unit plane waves exp(+2 pi i h_p.r/N) at plane 0 (Alg. 3 line 3). */
BIP_API int32_t bip_build_S1(bip_ctx* ctx);

/* S2 parents <- exp(-2 pi i h_p.r/N) at the exit surface, then u <- T_j . P[u] for j = nz-1 .. 0 (eq. 12,
 * PAPER.md:209-212): the adjoint detector columns at plane 0.  Slice steps by the route of bip_set_fft_backend; timed
 * separately (bip_get_timing). */
BIP_API int32_t bip_build_S2(bip_ctx* ctx);

/* Scan positions rho [n_rho][2] in pixels, any real value.  Builds the illumination matrix
 * c_b(rho) = c_b exp(-2 pi i h_b.rho/N) on the device. */
BIP_API int32_t bip_set_scan(bip_ctx* ctx, int32_t n_rho, const double* rho_px);

/* PRISM beam subsampling (Alg. 2 line 1): positions (ascending) of the beams of h [n][2]
 * with h_y = 0 (mod fy) and h_x = 0 (mod fx) into keep_out [cap]; *n_keep = their number (BIP_ERR_INVALID if cap is too
 * small).  The retained probe coefficients are to be multiplied by fy * fx, "the DFT decimation factor".
 * Host only. */
BIP_API int32_t bip_prism_subsample(int32_t n, const int32_t* h, int32_t fy, int32_t fx, int32_t* keep_out, int32_t cap,
                                    int32_t* n_keep);

/* Probe coefficients of the retained beams, rescaled by fy * fx: c_out[j] = fy fx c_full[keep[j]],
 * c_full [n_full][2] (normalised for the FULL aperture, 1 / sqrt(G n_full)), c_out [n_keep][2].  Host only. */
BIP_API int32_t bip_prism_coeffs(int32_t n_keep, const int32_t* keep, int32_t n_full, const float* c_full, int32_t fy, int32_t fx,
                                 float* c_out);

/* PRISM crop mask: from now on a site contributes only to the scan positions inside its 1/f window,
 * |rho - tau| < N / (2 f) on both axes (periodic distance from the atom's pixel; reading c19).  fy = fx = 1
 * switches the mask off (the default).  The contraction then runs, per site, over that site's scan rows only: the
 * cost per site falls by fy * fx.  Tensor-core precisions only (BIP_PREC_FP16X4 / FP16X3 / BF16X6). */
BIP_API int32_t bip_set_crop(bip_ctx* ctx, int32_t fy, int32_t fx);

/* Choose the association of the on-atom contraction (bip_assoc above) for the following bip_map calls.  Tensor-core
 * precisions only for COUPLING; AUTO falls back to PROBE otherwise. */
BIP_API int32_t bip_set_association(bip_ctx* ctx, int32_t assoc);

/* Register an ionisation edge: its sites, transition-potential windows and detector.
 *   slice [n_atoms]        slice index i(tau) of each site, 0 <= slice < nz
 *   centre_px [n_atoms][2] pixel the atom sits on; the window covers centre - w/2 .. centre + w/2 - 1 (periodic)
 *   H  c64 [n_ch][w][w]    H[n][w/2][w/2] is on the atom's pixel; w even, 8 <= w <= min(ny, nx)
 *   det_h [n_det][2]       detector beams (eq. 5)
 *   w2                     weights of every detector beam on the context's S2 parents (n_rows == n_det); NULL: the
 *                          library computes the Sibson table itself (qmax = the largest |q| of det_h), once per
 *                          detector beam list, and keeps it on the context ("cached")
 * Several edges share S1 / S2 and one plane loop.  *edge_id receives 0, 1, ... */
BIP_API int32_t bip_add_edge(bip_ctx* ctx, int32_t n_atoms, const int32_t* slice, const int32_t* centre_px,
                     int32_t n_ch, int32_t w, const float* H, int32_t n_det, const int32_t* det_h,
                     const bip_weights* w2, int32_t* edge_id);

/* Drop all registered edges (the scattering matrices and scan stay). */
BIP_API int32_t bip_clear_edges(bip_ctx* ctx);

/* Number of output elements of an edge in a mode: MAP n_rho (double), QEELS n_rho * n_bins (float),
 * CUBE n_rho * n_det (float); *n_bins = distinct h_x (QEELS_X) / h_y (QEELS_Y) of the detector, ascending. */
BIP_API int32_t bip_output_size(const bip_ctx* ctx, int32_t edge_id, int32_t mode, int64_t* n_elems, int32_t* n_bins);

/* Run Algorithm 5 for one edge (edge_id >= 0): for every plane holding >= 1 site, in increasing depth,
 * S1.ADVANCETO / S2.PEELTO (the plane cursor is moved from wherever the last call left it; both multislice
 * steps are unitary and are undone exactly when the cursor has to move back) and the on-atom contraction of
 * every site and channel, accumulated into out.
 *   out_dev   MAP: double [n_rho];  QEELS_*: float [n_rho][n_bins];  CUBE: float [n_rho][n_det]
 *             (detector-set order).  Zero-initialised by the call.  out_bytes must match bip_output_size.
 * Returns after enqueueing on the context's stream.  (Under a crop mask the first call after bip_set_crop /
 * bip_set_scan / bip_add_edge counts every site's scan rows on the device and reads the counts back once.) */
BIP_API int32_t bip_map(bip_ctx* ctx, int32_t edge_id, int32_t mode, int32_t recon, int32_t precision,
                void* out_dev, size_t out_bytes);

/* As bip_map with a HOST output buffer: device scratch is allocated, the result copied back and the stream
 * synchronised before returning. */
BIP_API int32_t bip_map_host(bip_ctx* ctx, int32_t edge_id, int32_t mode, int32_t recon, int32_t precision,
                     void* out_host, size_t out_bytes);

/* Run all registered edges in ONE plane loop (multi-edge batching): outs_dev[e] / outs_bytes[e]
 * per edge, same layout as bip_map. */
BIP_API int32_t bip_map_all(bip_ctx* ctx, int32_t mode, int32_t recon, int32_t precision,
                    void* const* outs_dev, const size_t* outs_bytes, int32_t n_outs);

/* Algorithm 3 of the paper (Table 1): the energy-filtered 4D cube on ALL exit beams with
 * only S1 partitioned.  For every ionisation plane S1.ADVANCETO; for every site the partitioned probe on the window
 * (eq. 15 / eq. 11 + eq. 7: steps a1-a4 of the map path), psi_n = H_n psi (eq. 3), carried to the exit surface by
 * conventional multislice for every scan position and channel, |F psi_n|^2 accumulated (Alg. 1 lines 5-8).  S2 is not
 * used (bip_build_S2 need not have run).
 *   out_dev   float [n_rho][ny][nx], exit beam (ky, kx) on the corner-origin DFT grid, unitary F; zero-initialised by the
 *             call; out_bytes = n_rho * ny * nx * 4.
 *   precision BIP_PREC_FP16X4 or BIP_PREC_BF16X6 (arithmetic of the probe contraction a4).
 * The wavefields of a chunk of scan positions live in half of the scratch budget.  Returns after enqueueing. */
BIP_API int32_t bip_cube_alg3(bip_ctx* ctx, int32_t edge_id, int32_t recon, int32_t precision, float* out_dev, size_t out_bytes);

/* Device scratch the plane loop may use for the operands of one batch of sites (default 12 GB, minimum 32 MB): the
 * sites of a plane are contracted in batches that fit. */
BIP_API int32_t bip_set_scratch_budget(bip_ctx* ctx, size_t bytes);

/* Route of the slice steps (bip_build_S2, ADVANCETO, PEELTO; plumbing, timed separately):
 *   BIP_FFT_NATIVE     the library's own fused fp32 slice step, three passes over a column -- two when steps follow one
 *                      another on the same columns (power-of-two grids 8..4096; the default there);
 *   BIP_FFT_CUFFT_F64  cuFFT Z2Z on a double-precision workspace, columns rounded to c64 once per slice (any grid; the
 *                      default for grids that are not powers of two, and the A/B reference of the native route). */
typedef enum { BIP_FFT_NATIVE = 0, BIP_FFT_CUFFT_F64 = 1 } bip_fft_backend;
BIP_API int32_t bip_set_fft_backend(bip_ctx* ctx, int32_t backend);

/* NEXT-4, S1 focal back-propagation (section 2.2.3.1; the paper leaves the plane and the padding open --
 * DESIGN.md reading c20): with on != 0 the S1 side of every site is reconstructed through the scattering-centroid plane of
 * the slices above it.  The de-tilted parent envelopes on the padded window (side 2^ceil(log2(w + 16))) are carried back by
 * d_i = i dz - z_c(i) with the free-space transfer function of their own carrier, interpolated there (eq. 15 / eq. 11),
 * carried forward beam by beam, re-tilted and cropped.  z_c(i) = sum_{j<i} m_j (j + 1/2) dz / sum_{j<i} m_j,
 * m_j = sum_r |T_j(r) - 1|^2.  Exact PRISM in the full-parent limit, identical to the plain reconstruction where d_i = 0.
 * S2 is untouched ("focal back-propagation is applied to S1 alone").  Probe-first association and
 * tensor-core precisions only; one site at a time on the S1 side (1 GB of envelopes per site at configs[1]). */
BIP_API int32_t bip_set_focal(bip_ctx* ctx, int32_t on);

/* d_i of ionisation plane `plane` (0..nz), Angstrom, as the library computed it from T. */
BIP_API int32_t bip_get_focal_distance(const bip_ctx* ctx, int32_t plane, double* d_out);

/* Frozen-phonon averaging re-uses the pipeline once per displaced configuration: replace the
 * transmission functions (same layout and rules as in bip_create; the scattering matrices must be rebuilt:
 * bip_build_S1 / bip_build_S2), and let bip_map ADD to its output (on != 0) instead of zeroing it; the caller divides by
 * the number of configurations. */
BIP_API int32_t bip_set_transmission(bip_ctx* ctx, const void* T, int32_t T_on_device);
BIP_API int32_t bip_set_accumulate(bip_ctx* ctx, int32_t on);

/* Opt in (allow != 0) to BIP_PREC_TF32X3, which misses the 1e-6 summed-intensity bound (see bip_precision). */
BIP_API int32_t bip_allow_tf32x3(bip_ctx* ctx, int32_t allow);

/* Parent beams of S1 (which = 1) or S2 (which = 2) as the context holds them: h_out [cap][2], *n_out their number
 * (h_out may be NULL to query it) -- for the bit-exact index comparison against the oracle. */
BIP_API int32_t bip_get_parents(const bip_ctx* ctx, int32_t which, int32_t* h_out, int32_t cap, int32_t* n_out);

/* The ELL weight table in use: edge_id < 0: w^(1) (aperture beams on S1 parents); else w^(2) of that edge (given by
 * the caller or computed by the library).  *n_rows, *max_nn: its shape; nn_idx_out / nn_w_out [n_rows][max_nn] may be
 * NULL to query the shape only. */
BIP_API int32_t bip_get_weights(const bip_ctx* ctx, int32_t edge_id, int32_t* n_rows, int32_t* max_nn, int32_t* nn_idx_out,
                                float* nn_w_out);

/* Window origins (centre - w/2) mod N of an edge's atoms, int32 [n_atoms][2] -- for bit-exact index checks. */
BIP_API int32_t bip_get_windows(const bip_ctx* ctx, int32_t edge_id, int32_t* origin_out);

/* qEELS bin values (signed beam index along the resolved axis, ascending), int32 [n_bins]. */
BIP_API int32_t bip_get_qeels_bins(const bip_ctx* ctx, int32_t edge_id, int32_t mode, int32_t* bins_out);

/* Move the plane cursor: S1 advanced / S2 peeled so that both sit at ionisation plane `plane` (0..nz): S1 holds
 * slices 0..plane-1, S2 holds slices plane..nz-1.  Moving back applies the inverse steps (|T| = 1, |P| = 1). */
BIP_API int32_t bip_seek_plane(bip_ctx* ctx, int32_t plane);

/* Copy parent columns [p0, p0 + np) of S1 (which = 1) or S2 (which = 2) at the current plane to host,
 * c64 [np][ny][nx]; synchronises the stream. */
BIP_API int32_t bip_copy_S(bip_ctx* ctx, int32_t which, int32_t p0, int32_t np, void* out_host);

/* Reconstructed windows of one atom at the current plane, for parity of steps a1-a2 / a6:
 * which = 1: S1^b|Omega c64 [n_ap][w*w]; which = 2: S2^d|Omega c64 [n_det][w*w].  Host output; synchronises. */
BIP_API int32_t bip_debug_reconstruct(bip_ctx* ctx, int32_t edge_id, int32_t atom, int32_t which, int32_t recon,
                              void* out_host);

/* The ONE entry point that allocates nothing: for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it).  Same result as bip_debug_reconstruct -- the reconstructed windows of one site at
 * the current plane (steps a1-a2 / a6; eq. 15, or eq. 11): which = 1: S1^b|Omega c64
 * [n_ap][w*w]; which = 2: S2^d|Omega c64 [n_det][w*w] -- but written to the caller's DEVICE buffer out_dev (out_bytes =
 * rows * w * w * 8, checked), and with the intermediate de-tilted parent windows D[p][s] in a static device array of
 * BIP_NOALLOC_SCRATCH_BYTES inside the library instead of an allocated buffer.
 *   - n_parent * w * w * 8 bytes must fit the array (n_parent = the S1 / S2 parent count): larger requests fail with
 *     BIP_ERR_UNSUPPORTED and touch nothing.  Every GPU that loads the library holds the array until the process exits.
 *   - The call makes no cudaMalloc / cudaFree and calls no allocating routine; it enqueues two kernels on the context's
 *     stream and returns without synchronising (the caller syncs before reading out_dev).  The first call on a device
 *     resolves the array's address (cudaGetSymbolAddress): make one call before starting a capture.
 *   - Every call on a GPU, from any context or stream, shares the array, which keeps the last call's contents (nothing in it
 *     has to start at zero: each call overwrites what it reads).  Calls that overlap on the GPU race on it: serialise them.
 *   - The plane cursor is not moved (bip_seek_plane first); edge and atom as registered by bip_add_edge. */
#define BIP_NOALLOC_SCRATCH_BYTES (4u << 20)
BIP_API int32_t bip_reconstruct_noalloc(bip_ctx* ctx, int32_t edge_id, int32_t atom, int32_t which, int32_t recon, void* out_dev,
                                        size_t out_bytes);

BIP_API int32_t bip_get_timing(const bip_ctx* ctx, bip_timing* out);

/* Library / device description ("libbip <version>; device <name> sm_XY; SMs n"); never NULL. */
BIP_API const char* bip_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BIP_H_ */
