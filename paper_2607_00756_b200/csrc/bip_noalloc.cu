// bip_reconstruct_noalloc: the one entry point of the library that allocates nothing (include/bip.h), for callers that
// cannot call cudaMalloc -- code under CUDA graph capture, tight serving loops, harnesses that forbid it.
//
// It is the windowed reconstruction of one site (steps a1-a2 / a6 of SURVEY.md 8(a); eq. 15, and eq. 11,
// PAPER.md:183), the same two kernels bip_debug_reconstruct launches: k_crop_detilt writes the de-tilted parent windows
// D[p][s] of the site into scratch, k_recon_c64 reads them back (up to max_nn parents per reconstructed element).  Here that
// scratch is not a cudaMalloc'ed buffer of the context but the file-scope array below, of a fixed, modest size; the output
// goes to a device buffer the caller passes.
//
// The array is a property of the loaded library, not of a context: every GPU that loads libbip holds its
// BIP_NOALLOC_SCRATCH_BYTES until the process exits, and every call on that GPU -- from any context, on any stream --
// shares it.  Calls that overlap on the GPU therefore race on it; serialise them (one stream, or events).  The array keeps
// the contents of the last call; nothing in it has to start at zero, because the first kernel overwrites every element the
// second one reads (n_parent * w * w of them).
#include <mutex>

#include "bip_internal.h"

namespace bip {

namespace {

constexpr size_t NOALLOC_MAX_EL = BIP_NOALLOC_SCRATCH_BYTES / sizeof(float2);

// In host code this name is a host-side stand-in for the array, not a device address: the address the kernels need comes
// from cudaGetSymbolAddress, once per device (scratch_of_current_device).
static __device__ __align__(256) float2 g_noalloc_scratch[NOALLOC_MAX_EL];

constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
float2* g_scratch_addr[MAX_DEVICES] = {};      // device address of g_noalloc_scratch on device i, resolved on first use there

// The array's address on the CURRENT device (the context's: every call of the library runs with it current).  Resolved once
// per device; no allocation (the array is part of the module image).
int32_t scratch_of_current_device(bip_ctx* ctx, float2** out) {
  int dev = -1;
  BIP_CUDA(ctx, cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAX_DEVICES) return fail(ctx, BIP_ERR_UNSUPPORTED, "bip_reconstruct_noalloc: device ordinal %d outside 0..%d", dev, MAX_DEVICES - 1);
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_addr[dev]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      return fail(ctx, BIP_ERR_CUDA, "bip_reconstruct_noalloc: cudaGetSymbolAddress of the static scratch failed on device %d: %s", dev,
                  cudaGetErrorString(e));
    }
    g_scratch_addr[dev] = static_cast<float2*>(p);
  }
  *out = g_scratch_addr[dev];
  return BIP_OK;
}

}  // namespace

}  // namespace bip

using namespace bip;

extern "C" {

int32_t bip_reconstruct_noalloc(bip_ctx* ctx, int32_t edge_id, int32_t atom, int32_t which, int32_t recon, void* out_dev, size_t out_bytes) {
  if (!ctx || !out_dev) return fail(ctx, BIP_ERR_INVALID, "bip_reconstruct_noalloc: NULL argument");
  if (edge_id < 0 || edge_id >= (int)ctx->edges.size()) return fail(ctx, BIP_ERR_INVALID, "bip_reconstruct_noalloc: edge %d does not exist", edge_id);
  Edge& e = ctx->edges[edge_id];
  if (atom < 0 || atom >= e.n_atoms) return fail(ctx, BIP_ERR_INVALID, "bip_reconstruct_noalloc: atom %d does not exist", atom);
  if (which != 1 && which != 2) return fail(ctx, BIP_ERR_INVALID, "bip_reconstruct_noalloc: which must be 1 or 2");
  if (recon != BIP_RECON_LINEAR && recon != BIP_RECON_MAGPHASE) return fail(ctx, BIP_ERR_INVALID, "bip_reconstruct_noalloc: unknown recon %d", recon);
  if (!ctx->s1_built || !ctx->s2_built) return fail(ctx, BIP_ERR_STATE, "bip_reconstruct_noalloc: call bip_build_S1 and bip_build_S2 first");
  const size_t w2 = (size_t)e.w * e.w;
  const int n_par = which == 1 ? ctx->n_p1 : ctx->n_p2;
  const int n_beams = which == 1 ? ctx->n_ap : e.n_det;
  const size_t need_out = (size_t)n_beams * w2 * sizeof(float2);
  if (out_bytes != need_out) return fail(ctx, BIP_ERR_INVALID, "bip_reconstruct_noalloc: output has %zu bytes, expected %zu", out_bytes, need_out);
  const size_t need_el = (size_t)n_par * w2;
  if (need_el > NOALLOC_MAX_EL)
    return fail(ctx, BIP_ERR_UNSUPPORTED,
                "bip_reconstruct_noalloc: %d parent windows of %d x %d need %zu bytes of scratch, the static array holds %zu "
                "(BIP_NOALLOC_SCRATCH_BYTES); use bip_debug_reconstruct or bip_map, which allocate",
                n_par, e.w, e.w, need_el * sizeof(float2), (size_t)BIP_NOALLOC_SCRATCH_BYTES);
  float2* D = nullptr;
  BIP_TRY(scratch_of_current_device(ctx, &D));
  const int32_t* org = e.origin_dev + 2 * (int64_t)atom;
  const int carrier = which == 1 ? +1 : -1;
  // a1 / a6: D[p][s] = S_p(r) exp(-carrier 2 pi i h_p.r / N) on the site's window, into the static scratch
  BIP_TRY(launch_crop_detilt(ctx, which == 1 ? ctx->S1 : ctx->S2, which == 1 ? ctx->p1_h_dev : ctx->p2_h_dev, n_par, carrier, org, 1, e.w, D));
  // a2 / a6: natural-neighbour reconstruction (eq. 15 or eq. 11) + re-tilt, into the caller's buffer
  return launch_recon_c64(ctx, D, n_par, which == 1 ? ctx->ap_h_dev : e.det_h_dev, n_beams, which == 1 ? ctx->w1_idx_dev : e.nn_idx_dev,
                          which == 1 ? ctx->w1_w_dev : e.nn_w_dev, which == 1 ? ctx->nn1 : e.max_nn, carrier, recon, org, 0, e.w,
                          static_cast<float2*>(out_dev));
}

}  // extern "C"
