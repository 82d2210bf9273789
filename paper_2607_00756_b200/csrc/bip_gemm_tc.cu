// tcgen05 / TMEM / TMA versions of the two contractions (steps a4-a5 and a7-a8 of SURVEY.md 8(a)) for sm_100a.
//
// One persistent, warp-specialised kernel computes C[128 x 256] (complex) = X[128 x Kd] . Y[256 x Kd]^T per work
// item from split-plane operands (bip::Planes: re_hi, re_lo, im_hi, im_lo, every value already TF32-representable):
//
//   Cr = Xr Yr - Xi Yi ,  Ci = Xr Yi + Xi Yr ,  each real product = hi.hi + hi.lo + lo.hi      (3xTF32)
//
// i.e. 12 tcgen05.mma.kind::tf32 (M = 128, N = 256, K = 8) per 8 k-elements, fp32 accumulation in TMEM
// (Cr in columns [0, 256), Ci in [256, 512): the whole tensor memory of the SM).  The minus sign of Xi Yi is the
// a_negate bit of the instruction descriptor.  Operand tiles are brought in by TMA (cp.async.bulk.tensor, 64 B
// rows, SWIZZLE_64B) through a 2-stage mbarrier ring; one elected thread issues the MMAs; four epilogue warps read
// the accumulators back with tcgen05.ld and apply the fused epilogue:
//
//   GEMM1 (a4-a5): Phi_n[rho][s] = H_n[s] Psi[rho][s]  -> split planes for every channel n
//   GEMM2 (a7-a8): |a_n[rho][d]|^2 / G summed over channels and reduced per output mode
//
// Warp roles: warp 0 TMA producer, warp 1 TMEM owner + MMA issuer, warps 2-5 epilogue (TMEM lane quarter = warp % 4).
#include <cuda.h>

#include "bip_internal.h"

namespace bip {

namespace {

constexpr int TM = 128;                 // rows per tile  (UMMA M)
constexpr int TN = 256;                 // complex columns per tile (UMMA N)
constexpr int KC = 16;                  // k elements per pipeline stage: 64-byte rows, SWIZZLE_64B
constexpr int UK = 8;                   // k elements per tcgen05.mma.kind::tf32
constexpr int STAGES = 2;
constexpr int A_PLANE = TM * KC * 4;    // 8 KB
constexpr int B_PLANE = TN * KC * 4;    // 16 KB
constexpr int STAGE_BYTES = 4 * A_PLANE + 4 * B_PLANE;   // 96 KB
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*align*/ + 256 /*barriers*/;
constexpr int NUM_THREADS = 192;
constexpr int DGROUP = 9;               // detector tiles per raster group (keeps ~148 concurrent tiles sharing operands in L2)

enum { EPI_GEMM1 = 1, EPI_GEMM2 = 2 };

struct TcParams {
  int epi;
  int n_rt, n_ct;          // row tiles, column tiles per atom
  int n_items;
  int n_ch_loop;           // channels looped inside an item (GEMM2: n_ch, GEMM1: 1)
  int k_chunks;            // ceil(Kd / KC)
  int n_rows, n_cols;      // valid rows (rho) / columns (d or s) per atom
  // GEMM1 epilogue
  const float2* H;
  int n_ch;
  float* phi[4];
  int64_t phi_ld, phi_ch_stride, phi_batch_stride;
  // GEMM2 epilogue
  int mode;
  float inv_G;
  const int32_t* bin_of_det;
  int n_bins;
  void* out;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done = 0;
  while (!done) {
    asm volatile(
        "{\n\t"
        ".reg .pred P1;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2;\n\t"
        "selp.b32 %0, 1, 0, P1;\n\t"
        "}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  }
}

__device__ __forceinline__ void tma_load_5d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2, int c3, int c4) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4)
      : "memory");
}

// K-major, SWIZZLE_64B shared-memory matrix descriptor (cute::UMMA::SmemDescriptor): 8-row x 64-byte swizzle atoms,
// 512 bytes between 8-row groups.
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3FFFF) >> 4);            // start address, bits [0,14)
  d |= (uint64_t)1 << 16;                             // leading byte offset (unused for swizzled K-major), bits [16,30)
  d |= (uint64_t)(512 >> 4) << 32;                    // stride byte offset, bits [32,46)
  d |= (uint64_t)1 << 46;                             // descriptor version (Blackwell)
  d |= (uint64_t)4 << 61;                             // layout type SWIZZLE_64B
  return d;
}

// cute::UMMA::InstrDescriptor for kind::tf32, fp32 accumulate, K-major A and B
__host__ __device__ constexpr uint32_t umma_idesc(bool neg_a) {
  return (1u << 4) | (2u << 7) | (2u << 10) | ((neg_a ? 1u : 0u) << 13) | ((uint32_t)(TN >> 3) << 17) | ((uint32_t)(TM >> 4) << 24);
}

__device__ __forceinline__ void umma_tf32(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t"
      "}" ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
      : "memory");
}

__device__ __forceinline__ void umma_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
        "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
        "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
        "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr));
}

__device__ __forceinline__ float tf32_rna(float x) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return __uint_as_float(r);
}

// item -> (atom, row tile, column tile).  GEMM2 rasterises column tiles in groups of DGROUP so that the ~148
// concurrently running tiles share operand rows in L2.
__device__ __forceinline__ void decode_item(const TcParams& p, int item, int& atom, int& rt, int& ct) {
  const int per_atom = p.n_rt * p.n_ct;
  atom = item / per_atom;
  int idx = item - atom * per_atom;
  const int full = p.n_ct / DGROUP;
  const int blk = p.n_rt * DGROUP;
  if (idx < full * blk) {
    const int g = idx / blk, r = idx - g * blk;
    rt = r / DGROUP;
    ct = g * DGROUP + (r - rt * DGROUP);
  } else {
    idx -= full * blk;
    const int gsz = p.n_ct - full * DGROUP;
    rt = idx / gsz;
    ct = full * DGROUP + (idx - rt * gsz);
  }
}

__global__ void __launch_bounds__(NUM_THREADS, 1)
k_tc_contract(const __grid_constant__ CUtensorMap mapX, const __grid_constant__ CUtensorMap mapY, const TcParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + STAGES * STAGE_BYTES);
  uint64_t* full = bars;                 // [STAGES]
  uint64_t* empty = bars + STAGES;       // [STAGES]
  uint64_t* tmem_full = bars + 2 * STAGES;
  uint64_t* tmem_empty = bars + 2 * STAGES + 1;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * STAGES + 2);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (warp == 0 && lane == 0) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(&mapX) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&mapY) : "memory");
    for (int s = 0; s < STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
    mbar_init(tmem_full, 1);
    mbar_init(tmem_empty, 4);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {   // the whole tensor memory: 512 columns
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ================= TMA producer =================
    if (lane == 0) {
      uint32_t it = 0;
      for (int item = blockIdx.x; item < p.n_items; item += gridDim.x) {
        int atom, rt, ct;
        decode_item(p, item, atom, rt, ct);
        for (int n = 0; n < p.n_ch_loop; ++n) {
          for (int kc = 0; kc < p.k_chunks; ++kc, ++it) {
            const int s = it % STAGES;
            mbar_wait(&empty[s], ((it / STAGES) & 1) ^ 1);
            uint8_t* st = smem + s * STAGE_BYTES;
            mbar_expect_tx(&full[s], STAGE_BYTES);
#pragma unroll
            for (int pl = 0; pl < 4; ++pl) {
              tma_load_5d(st + pl * A_PLANE, &mapX, &full[s], kc * KC, rt * TM, n, p.epi == EPI_GEMM2 ? atom : 0, pl);
              tma_load_5d(st + 4 * A_PLANE + pl * B_PLANE, &mapY, &full[s], kc * KC, ct * TN, 0, atom, pl);
            }
          }
        }
      }
    }
  } else if (warp == 1) {
    // ================= MMA issuer =================
    if (lane == 0) {
      uint32_t it = 0, chan = 0;
      const uint32_t id_pos = umma_idesc(false), id_neg = umma_idesc(true);
      const uint32_t t_cr = tmem_base, t_ci = tmem_base + TN;
      for (int item = blockIdx.x; item < p.n_items; item += gridDim.x) {
        for (int n = 0; n < p.n_ch_loop; ++n, ++chan) {
          mbar_wait(tmem_empty, (chan & 1) ^ 1);        // epilogue has drained the previous accumulators
          asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
          for (int kc = 0; kc < p.k_chunks; ++kc, ++it) {
            const int s = it % STAGES;
            mbar_wait(&full[s], (it / STAGES) & 1);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t a0 = smem_u32(smem + s * STAGE_BYTES), b0 = a0 + 4 * A_PLANE;
#pragma unroll
            for (int ks = 0; ks < KC / UK; ++ks) {
              const uint32_t ko = ks * UK * 4;         // 32 bytes per k-step inside the 64-byte swizzled row
              const uint64_t xrh = umma_desc(a0 + 0 * A_PLANE + ko), xrl = umma_desc(a0 + 1 * A_PLANE + ko);
              const uint64_t xih = umma_desc(a0 + 2 * A_PLANE + ko), xil = umma_desc(a0 + 3 * A_PLANE + ko);
              const uint64_t yrh = umma_desc(b0 + 0 * B_PLANE + ko), yrl = umma_desc(b0 + 1 * B_PLANE + ko);
              const uint64_t yih = umma_desc(b0 + 2 * B_PLANE + ko), yil = umma_desc(b0 + 3 * B_PLANE + ko);
              const uint32_t acc = (kc | ks) ? 1u : 0u;
              // Cr = Xr Yr - Xi Yi   (small cross terms first)
              umma_tf32(t_cr, xrh, yrl, id_pos, acc);
              umma_tf32(t_cr, xrl, yrh, id_pos, 1u);
              umma_tf32(t_cr, xih, yil, id_neg, 1u);
              umma_tf32(t_cr, xil, yih, id_neg, 1u);
              umma_tf32(t_cr, xrh, yrh, id_pos, 1u);
              umma_tf32(t_cr, xih, yih, id_neg, 1u);
              // Ci = Xr Yi + Xi Yr
              umma_tf32(t_ci, xrh, yil, id_pos, acc);
              umma_tf32(t_ci, xrl, yih, id_pos, 1u);
              umma_tf32(t_ci, xih, yrl, id_pos, 1u);
              umma_tf32(t_ci, xil, yrh, id_pos, 1u);
              umma_tf32(t_ci, xrh, yih, id_pos, 1u);
              umma_tf32(t_ci, xih, yrh, id_pos, 1u);
            }
            umma_commit(&empty[s]);                    // stage reusable once these MMAs have read it
          }
          umma_commit(tmem_full);                      // accumulators of this channel complete
        }
      }
    }
  } else {
    // ================= epilogue warps =================
    const int quarter = warp & 3;                      // TMEM lanes [32 q, 32 q + 32) are visible to warps with warp % 4 == q
    const uint32_t t_lane = tmem_base + ((uint32_t)(quarter * 32) << 16);
    uint32_t chan = 0;
    for (int item = blockIdx.x; item < p.n_items; item += gridDim.x) {
      int atom, rt, ct;
      decode_item(p, item, atom, rt, ct);
      const int row = rt * TM + quarter * 32 + lane;   // this thread's rho
      const bool row_ok = row < p.n_rows;
      float rowsum = 0.f;
      for (int n = 0; n < p.n_ch_loop; ++n, ++chan) {
        mbar_wait(tmem_full, chan & 1);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
#pragma unroll 1
        for (int c0 = 0; c0 < TN; c0 += 32) {
          uint32_t cr[32], ci[32];
          tmem_ld32(t_lane + c0, cr);
          tmem_ld32(t_lane + TN + c0, ci);
          asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
          const int col0 = ct * TN + c0;
          if (p.epi == EPI_GEMM2) {
            if (p.mode == BIP_MODE_MAP) {
#pragma unroll
              for (int j = 0; j < 32; ++j) {
                const float re = __uint_as_float(cr[j]), im = __uint_as_float(ci[j]);
                rowsum = fmaf(re, re, fmaf(im, im, rowsum));
              }
            } else if (row_ok) {
              float* out = reinterpret_cast<float*>(p.out);
#pragma unroll 4
              for (int j = 0; j < 32; ++j) {
                const int d = col0 + j;
                if (d < p.n_cols) {
                  const float re = __uint_as_float(cr[j]), im = __uint_as_float(ci[j]);
                  const float v = (re * re + im * im) * p.inv_G;
                  if (p.mode == BIP_MODE_CUBE) atomicAdd(out + (int64_t)row * p.n_cols + d, v);
                  else atomicAdd(out + (int64_t)row * p.n_bins + p.bin_of_det[d], v);
                }
              }
            }
          } else if (row_ok) {
            // GEMM1: Phi_n = H_n Psi for every channel, written as split planes
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              const int s = col0 + j;
              if (s >= p.n_cols) continue;
              const float re = __uint_as_float(cr[j]), im = __uint_as_float(ci[j]);
#pragma unroll 1
              for (int ch = 0; ch < p.n_ch; ++ch) {
                const float2 h = __ldg(&p.H[(int64_t)ch * p.n_cols + s]);
                const float fr = h.x * re - h.y * im, fi = h.x * im + h.y * re;
                const int64_t o = (int64_t)atom * p.phi_batch_stride + (int64_t)ch * p.phi_ch_stride + (int64_t)row * p.phi_ld + s;
                const float rh = tf32_rna(fr), ih = tf32_rna(fi);
                p.phi[0][o] = rh; p.phi[1][o] = tf32_rna(fr - rh);
                p.phi[2][o] = ih; p.phi[3][o] = tf32_rna(fi - ih);
              }
            }
          }
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncwarp();
        if (lane == 0) mbar_arrive(tmem_empty);
      }
      if (p.epi == EPI_GEMM2 && p.mode == BIP_MODE_MAP && row_ok)
        atomicAdd(reinterpret_cast<double*>(p.out) + row, (double)rowsum * (double)p.inv_G);
    }
  }

  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
}

// ---------------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = [] {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) {
      cudaGetLastError();
      f = nullptr;
    }
    return reinterpret_cast<EncodeTiledFn>(f);
  }();
  return fn;
}

// 5-D map over a split-plane operand: (k, row, c2, c3, plane).  Strides in floats (0 for a size-1 dimension).
int32_t make_map(bip_ctx* ctx, CUtensorMap* m, const Planes& P, int64_t k_extent, int64_t rows, int64_t n2, int64_t stride2,
                 int64_t n3, int64_t stride3, int box_rows) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return fail(ctx, BIP_ERR_CUDA, "cuTensorMapEncodeTiled is not available from the driver");
  const int64_t plane_stride = P.p[1] - P.p[0];
  cuuint64_t dims[5] = {(cuuint64_t)k_extent, (cuuint64_t)rows, (cuuint64_t)n2, (cuuint64_t)n3, 4};
  cuuint64_t strides[4] = {(cuuint64_t)P.ld * 4, (cuuint64_t)(n2 > 1 ? stride2 : P.ld) * 4, (cuuint64_t)(n3 > 1 ? stride3 : P.ld) * 4,
                           (cuuint64_t)plane_stride * 4};
  cuuint32_t box[5] = {(cuuint32_t)KC, (cuuint32_t)box_rows, 1, 1, 1};
  cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 5, P.p[0], dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(ctx, BIP_ERR_CUDA, "cuTensorMapEncodeTiled failed: %d (k %lld rows %lld n2 %lld n3 %lld ld %lld)", (int)r,
                                     (long long)k_extent, (long long)rows, (long long)n2, (long long)n3, (long long)P.ld);
  return BIP_OK;
}

int32_t launch(bip_ctx* ctx, const CUtensorMap& mx, const CUtensorMap& my, const TcParams& p) {
  static bool attr_set = false;
  if (!attr_set) {
    BIP_CUDA(ctx, cudaFuncSetAttribute(k_tc_contract, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES));
    attr_set = true;
  }
  const int grid = std::max(1, std::min(p.n_items, ctx->sm_count));
  k_tc_contract<<<grid, NUM_THREADS, SMEM_BYTES, ctx->stream>>>(mx, my, p);
  BIP_CUDA(ctx, cudaGetLastError());
  ctx->timing.kernel_launches++;
  return BIP_OK;
}

}  // namespace

bool tc_available() { return true; }

int32_t launch_gemm1_tc(bip_ctx* ctx, const Gemm1Args& a) {
  CUtensorMap mx, my;
  // X = illumination A[rho][b] (shared by all atoms); Y = R1^T[atom][s][b]
  BIP_TRY(make_map(ctx, &mx, a.A, a.n_ap, a.n_rho, 1, 0, 1, 0, TM));
  BIP_TRY(make_map(ctx, &my, a.R1t, a.n_ap, a.w2, 1, 0, a.n_atoms, a.R1t.batch_stride, TN));
  TcParams p{};
  p.epi = EPI_GEMM1;
  p.n_rt = (a.n_rho + TM - 1) / TM;
  p.n_ct = (a.w2 + TN - 1) / TN;
  p.n_items = a.n_atoms * p.n_rt * p.n_ct;
  p.n_ch_loop = 1;
  p.k_chunks = (a.n_ap + KC - 1) / KC;
  p.n_rows = a.n_rho; p.n_cols = a.w2;
  p.H = a.H; p.n_ch = a.n_ch;
  for (int k = 0; k < 4; ++k) p.phi[k] = a.Phi.p[k];
  p.phi_ld = a.Phi.ld; p.phi_ch_stride = a.phi_ch_stride; p.phi_batch_stride = a.Phi.batch_stride;
  return launch(ctx, mx, my, p);
}

int32_t launch_gemm2_tc(bip_ctx* ctx, const Gemm2Args& a) {
  CUtensorMap mx, my;
  // X = Phi[atom][n][rho][s]; Y = R2[atom][d][s]
  BIP_TRY(make_map(ctx, &mx, a.Phi, a.w2, a.n_rho, a.n_ch, a.phi_ch_stride, a.n_atoms, a.Phi.batch_stride, TM));
  BIP_TRY(make_map(ctx, &my, a.R2, a.w2, a.n_det, 1, 0, a.n_atoms, a.R2.batch_stride, TN));
  TcParams p{};
  p.epi = EPI_GEMM2;
  p.n_rt = (a.n_rho + TM - 1) / TM;
  p.n_ct = (a.n_det + TN - 1) / TN;
  p.n_items = a.n_atoms * p.n_rt * p.n_ct;
  p.n_ch_loop = a.n_ch;
  p.k_chunks = (a.w2 + KC - 1) / KC;
  p.n_rows = a.n_rho; p.n_cols = a.n_det;
  p.mode = a.mode; p.inv_G = a.inv_G; p.bin_of_det = a.bin_of_det; p.n_bins = a.n_bins; p.out = a.out;
  return launch(ctx, mx, my, p);
}

}  // namespace bip
