// tcgen05 / TMEM / bulk-TMA versions of the two contractions (steps a4-a5 and a7-a8 of SURVEY.md 8(a)) on the sliced
// 16-bit operand formats of bip_sliced.cuh (precisions BIP_PREC_FP16X4 and BIP_PREC_BF16X6, both fp32-equivalent).
//
// One persistent, warp-specialised kernel computes C[128 x 128] (complex) = X[128 x Kd] . Y[128 x Kd]^T per work item:
//
//   Cr = Xr Yr - Xi Yi ,  Ci = Xr Yi + Xi Yr
//   real product = x1 y1 + (x1 y2 + x2 y1 + x2 y2)                               FP16X4: 16 MMAs per 16 k-elements
//                = x1 y1 + (x1 y2 + x2 y1) + (x1 y3 + x2 y2 + x3 y1)             BF16X6: 24 MMAs per 16 k-elements
//
// each a tcgen05.mma.kind::f16 (M = 128, N = 128, K = 16).  Four fp32 accumulators live in TMEM (the whole 512
// columns): C0r, C0i take the LEADING products x1 y1 -- small integers, summed EXACTLY over a chunk of 128 (256)
// k-elements -- and C12r, C12i take the small ones over the whole k range.  After every chunk the eight epilogue
// warps read C0 back (tcgen05.ld) and add it to fp32 running sums in registers (round-to-nearest), so the
// truncating accumulation of the tensor core never biases the result (bip_sliced.cuh).  The MMA issuer runs the
// small products LAG k-steps AHEAD of the leading ones, so the tensor pipe keeps working on C12 while the epilogue
// drains C0.  Operand tiles arrive by cp.async.bulk (one contiguous 16 / 24 KB block per operand and k-step)
// through an mbarrier ring; one elected thread issues the MMAs.  Fused epilogues:
//
//   GEMM1 (a4):    Psi[rho][s] = sx[rho] sy[s] C           -> c64, quantised to Phi_n = H_n Psi by k_quantize_phi (a5)
//   GEMM2 (a7-a8): |a_n[rho][d]|^2 / G summed over channels and reduced per output mode
//
// WIDE variant (FP16X4 on CTA pairs; A/B only, tuning builds): the same arithmetic issued as N = 256 MMAs.  With the
// accumulator columns laid out as [Cr | Ci] of the CTA's 64 detector columns, x_re . [y_re ; y_im] and x_im . [-y_im ; y_re]
// give both components in one instruction each, so a k-step takes 8 MMAs of N = 256 instead of 16 of N = 128.  The idea
// was to read every X slice from shared memory half as often (the N = 128 form of FP16X3 saturates the 128 B / clk of
// shared-memory bandwidth).  Measured on B200 it is SLOWER, 3.4 % for FP16X4 and 5.5 % for FP16X3
// (profiles/r02_wide_mma.md): an N = 256 MMA evidently re-reads its A operand per 128 columns, and the Y operand grows
// by the negated imaginary slices (bip_sliced.cuh; per slice the 64-row blocks [-y_im][y_re][y_im] in a stage).  Kept
// as the measured alternative; the shipped build never launches it.
//
// Warp roles: warp 0 bulk-copy producer, warp 1 TMEM owner + MMA issuer, warps 2-9 epilogue (TMEM lane quarter =
// warp % 4, column half = (warp - 2) / 4).
#include <cuda.h>

#include <algorithm>

#include "bip_internal.h"

namespace bip {

namespace {

constexpr int TM = 128, TN = 128;
constexpr int PART_BYTES = SL_TILE_EL * 2;       // 4 KB
constexpr int NUM_EPI_WARPS = 8;
constexpr int NUM_THREADS = 64 + 32 * NUM_EPI_WARPS;
constexpr int DGROUP_DEFAULT = 16;               // column tiles per raster group (concurrent CTAs share operand tiles in L2)

template <int FMT> struct Cfg;
template <> struct Cfg<SL_FMT_FP16X4> {
  static constexpr int PARTS = 4, STAGES = 7, STAGES_PAIR = 9, LAG_MAX = 4;
  static constexpr int CHUNK_STEPS = 8;          // 128 k-elements: 2 * 128 * 2^16 = 2^24, exact
  static constexpr uint32_t AB_FORMAT = 0;       // fp16
};
template <> struct Cfg<SL_FMT_BF16X6> {
  static constexpr int PARTS = 6, STAGES = 4, STAGES_PAIR = 6, LAG_MAX = 2;
  static constexpr int CHUNK_STEPS = 16;         // 256 k-elements: 2 * 256 * 2^14 = 2^23 < 2^24, exact
  static constexpr uint32_t AB_FORMAT = 1;       // bf16
};
template <int FMT> __host__ __device__ constexpr int x_bytes() { return Cfg<FMT>::PARTS * PART_BYTES; }
// bytes of the Y operand per stage and CTA: all of it (single CTA), this CTA's 64-row half of every part (pair), or the
// half with the negated imaginary slices, 3 blocks of 64 rows per slice (WIDE)
template <int FMT, bool PAIR, bool WIDE> __host__ __device__ constexpr int y_bytes() {
  return WIDE ? 6 * (PART_BYTES / 2) : PAIR ? x_bytes<FMT>() / 2 : x_bytes<FMT>();
}
template <int FMT> __host__ __device__ constexpr int stage_bytes() { return 2 * x_bytes<FMT>(); }
// EPI_GEMM2_TILE (CTA pairs, QEELS / CUBE outputs): |a|^2 of the channels of an item is summed in a shared-memory tile
// [column][row] (129-float pitch: conflict-free both when a thread walks its own row and when a warp flushes 32
// consecutive columns of one row), and the tile goes to global memory once per item with coalesced fp32 REDs --
// N_ch times fewer global atomics than reducing per channel.  The tile takes the room of three pipeline stages.
enum { EPI_GEMM1 = 1, EPI_GEMM2 = 2, EPI_GEMM2_TILE = 3 };
constexpr int ACC_LD = TM + 1;
constexpr int ACC_BYTES = TN * ACC_LD * 4;       // 66 048
template <int EPI, int FMT, bool PAIR, bool WIDE> __host__ __device__ constexpr int n_stages() {
  return WIDE ? (EPI == EPI_GEMM2_TILE ? 5 : 8)
              : EPI == EPI_GEMM2_TILE ? (FMT == SL_FMT_FP16X4 ? 6 : 4) : PAIR ? Cfg<FMT>::STAGES_PAIR : Cfg<FMT>::STAGES;
}
template <int EPI, int FMT, bool PAIR, bool WIDE> __host__ __device__ constexpr int smem_bytes() {
  return n_stages<EPI, FMT, PAIR, WIDE>() * (x_bytes<FMT>() + y_bytes<FMT, PAIR, WIDE>()) + 1024 /*align*/ + 512 /*barriers*/ +
         (EPI == EPI_GEMM2_TILE ? ACC_BYTES : 0);
}

struct SlParams {
  const uint16_t* X; const uint16_t* Y;
  const float* sx; const float* sy;
  int64_t x_batch_stride, y_batch_stride, sx_batch_stride, sy_batch_stride;
  int ksteps;
  int n_rt, n_ct, n_items, n_ch_loop;   // row work tiles (pairs of 128-row tiles in pair mode), column tiles per atom
  int n_rt_x;              // 128-row tiles per channel block of X
  int n_rows, n_cols;      // valid rows (rho) / columns (s or d) per atom
  int rows_pad;            // padded rho rows per channel block of X
  int chunk_steps;         // k-steps per exactly accumulated chunk of leading products
  int lag_max;             // the leading products may trail the small ones by up to this many k-steps (< STAGES)
  int dgroup;              // column tiles per raster group
  int drop_tiny;           // FP16X3: the x2 y2 products (<= 2^-18 of the leading ones) are not issued
#ifdef BIP_TUNING
  int probe_x;             // timing probes (wrong results): 1 = X loaded only in the first k-step of a segment, 2 = every worker streams the X of row tile 0
#endif
  unsigned int* sync_counter;   // lockstep of the workers (below); NULL = free-running
  int sync_steps;               // ... every this many k-steps of a segment
  // GEMM1 epilogue
  float2* Psi; int64_t psi_ld, psi_batch_stride;
  // GEMM2 epilogue
  int mode; float inv_G; const int32_t* bin_of_det; int n_bins; void* out;
  int n_out_cols;          // detector beams K of the output: column c of the contraction is beam c % K (the coupling
                           // association runs the channels as extra columns, c = n K + d)
  const int32_t* row_idx; int64_t row_idx_stride;   // crop mask: output scan index of every (site, local row), -1 = none
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
__device__ __forceinline__ bool mbar_test(uint64_t* bar, uint32_t parity) {
  uint32_t done;
  asm volatile(
      "{\n\t"
      ".reg .pred P1;\n\t"
      "mbarrier.test_wait.parity.shared::cta.b64 P1, [%1], %2;\n\t"
      "selp.b32 %0, 1, 0, P1;\n\t"
      "}"
      : "=r"(done)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return done != 0;
}
__device__ __forceinline__ void bulk_load(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// Lockstep of the persistent workers.  Workers that share an operand stream (same row tile, neighbouring column
// tiles) only hit in L2 while they read the same k range at about the same time; free-running they drift apart and
// every worker ends up streaming its operands from HBM (profiles/r01_gemm2_l2_lockstep.md).  The producers of all
// workers therefore meet at a global counter at the start of every (item, channel) segment: one relaxed
// red + acquire-poll per ~150 us.  Lockstep is an L2-locality optimisation only, so the wait is BOUNDED: nothing
// guarantees that every worker of a plain (non-cooperative) launch is resident at once (a second context on another
// stream, an MPS co-tenant), and a worker whose peers have not shown up within LOCKSTEP_BUDGET_NS stops waiting for
// good and runs free -- skipping the meeting is always correct.  Returns false once the budget has expired.
constexpr unsigned long long LOCKSTEP_BUDGET_NS = 2000000ull;   // 2 ms: ~10 segments; a healthy meeting takes microseconds
__device__ __forceinline__ unsigned long long globaltimer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
__device__ __forceinline__ bool lockstep_arrive_wait(unsigned int* counter, unsigned int target) {
  asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(counter) : "memory");
  unsigned int v;
  unsigned long long t0 = 0;
  for (unsigned int spins = 0;; ++spins) {
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(counter) : "memory");
    if ((int)(v - target) >= 0) return true;
    if ((spins & 63u) == 63u) {
      const unsigned long long now = globaltimer_ns();
      if (t0 == 0) t0 = now;
      else if (now - t0 > LOCKSTEP_BUDGET_NS) return false;
    }
  }
}

// K-major, no-swizzle shared-memory matrix descriptor (cute::UMMA::SmemDescriptor, LayoutType::INTERLEAVE):
// core matrices of 8 rows x 16 bytes; LBO = 128 B between the two k halves, SBO = 256 B between 8-row groups.
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3FFFF) >> 4);            // start address, bits [0,14)
  d |= (uint64_t)(128 >> 4) << 16;                    // leading byte offset, bits [16,30)
  d |= (uint64_t)(256 >> 4) << 32;                    // stride byte offset, bits [32,46)
  d |= (uint64_t)1 << 46;                             // descriptor version (Blackwell)
  return d;                                           // layout type 0 = no swizzle
}

// The same descriptor from its low word: within one stage every operand slice differs from the stage base only in the start
// address, so the issuing thread forms  lo = umma_desc_lo(stage base)  once per k-step and each descriptor is lo + (offset >> 4)
// (one uniform add instead of add / shift / mask / or per descriptor: the issue loop, not the tensor pipe, paces FP16X3).
__device__ __forceinline__ uint32_t umma_desc_lo(uint32_t saddr) { return ((saddr & 0x3FFFF) >> 4) | ((uint32_t)(128 >> 4) << 16); }
__device__ __forceinline__ uint64_t umma_desc_at(uint32_t lo, uint32_t byte_off) {
  return ((uint64_t)((256u >> 4) | (1u << 14)) << 32) | (uint64_t)(lo + (byte_off >> 4));
}

// cute::UMMA::InstrDescriptor for kind::f16 (fp16 or bf16 operands), fp32 accumulate, K-major A and B;
// M = 128 (one CTA) or 256 (CTA pair, cta_group::2), N = 128 or 256
__host__ __device__ constexpr uint32_t umma_idesc(uint32_t ab_format, bool neg_a, bool pair, int n = TN) {
  return (1u << 4) | (ab_format << 7) | (ab_format << 10) | ((neg_a ? 1u : 0u) << 13) | ((uint32_t)(n >> 3) << 17) |
         ((uint32_t)((pair ? 2 * TM : TM) >> 4) << 24);
}

template <bool PAIR>
__device__ __forceinline__ void umma_f16(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  if (PAIR)
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
        : "memory");
  else
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
        : "memory");
}

// tcgen05.commit: the mbarrier is arrived on once every MMA issued so far by this thread has completed; for a CTA
// pair the arrival is multicast to the barrier at the same offset in both CTAs.
template <bool PAIR>
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
  if (PAIR)
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 ::"r"(smem_u32(bar)), "h"((uint16_t)3) : "memory");
  else
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// one lane of the (converged) warp: the thread that issues every tcgen05.mma / tcgen05.commit of the CTA
__device__ __forceinline__ uint32_t elect_one() {
  uint32_t pred;
  asm volatile(
      "{\n\t"
      ".reg .pred P1;\n\t"
      "elect.sync _|P1, 0xffffffff;\n\t"
      "selp.b32 %0, 1, 0, P1;\n\t"
      "}"
      : "=r"(pred));
  return pred;
}

// ---- CTA-pair plumbing ----
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// arrive on the barrier at the same shared-memory offset in CTA `rank` of the cluster.  RELAXED: nothing these arrivals
// publish goes through generic-proxy memory (operands land by bulk copy and are read by the tensor core; accumulators are
// read with tcgen05.ld + tcgen05.wait::ld before the arrival), and a release at cluster scope costs a MEMBAR.ALL.GPU per
// arrival -- in the peer's per-k-step "operands landed" forward that fence capped the pair at one k-step per ~1000 clocks
// whatever the number of MMAs (profiles/r02_gemm2_probes.md)
__device__ __forceinline__ void mbar_arrive_cluster(uint64_t* bar, uint32_t rank) {
  asm volatile(
      "{\n\t"
      ".reg .b32 ra;\n\t"
      "mapa.shared::cluster.u32 ra, %0, %1;\n\t"
      "mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [ra];\n\t"
      "}" ::"r"(smem_u32(bar)), "r"(rank)
      : "memory");
}
// Barriers that threads of the peer CTA arrive on (peer_full, c0_empty, c12_empty) are waited on with the plain CTA-scope
// mbar_wait: what those arrivals publish is read by the tensor core or lives in tensor memory and is ordered by
// tcgen05.fence::after_thread_sync; a cluster-scope acquire costs an L1 invalidation (CCTL.IVALL) per wait -- once per k-step
// in the issue loop, its largest single stall (profiles/r02_gemm2_probes.md).

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

// item -> (atom, row tile, column tile); column tiles rasterised in groups of p.dgroup.
__device__ __forceinline__ void decode_item(const SlParams& p, int item, int& atom, int& rt, int& ct) {
  const int DGROUP = p.dgroup;
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

// The small products of one k-step (accumulators C12r, C12i): everything except x1 y1.
template <int FMT, bool PAIR>
__device__ __forceinline__ void issue_small(uint32_t t12r, uint32_t t12i, uint32_t a0, uint32_t b0, uint32_t acc, bool drop_tiny, bool alt_order = false) {
  constexpr uint32_t id_pos = umma_idesc(Cfg<FMT>::AB_FORMAT, false, PAIR), id_neg = umma_idesc(Cfg<FMT>::AB_FORMAT, true, PAIR);
  constexpr int YP = PAIR ? PART_BYTES / 2 : PART_BYTES;      // a CTA of a pair holds 64 of the 128 Y rows of every part
  auto umma = [](uint32_t d, uint64_t da, uint64_t db, uint32_t id, uint32_t ac) { umma_f16<PAIR>(d, da, db, id, ac); };
  if (FMT == SL_FMT_FP16X4) {
    const uint32_t al = umma_desc_lo(a0), bl = umma_desc_lo(b0);
    const uint64_t xr1 = umma_desc_at(al, 0), xr2 = umma_desc_at(al, PART_BYTES), xi1 = umma_desc_at(al, 2 * PART_BYTES), xi2 = umma_desc_at(al, 3 * PART_BYTES);
    const uint64_t yr1 = umma_desc_at(bl, 0), yr2 = umma_desc_at(bl, YP), yi1 = umma_desc_at(bl, 2 * YP), yi2 = umma_desc_at(bl, 3 * YP);
    // tiniest first: x2 y2 (FP16X3 leaves them out), then x1 y2 + x2 y1
    uint32_t acc_r = acc, acc_i = acc;
    if (!drop_tiny) {
      umma(t12r, xr2, yr2, id_pos, acc);
      umma(t12r, xi2, yi2, id_neg, 1u);
      acc_r = 1u;
    }
#ifdef BIP_TUNING
    if (drop_tiny && alt_order) {                     // timing probe: same products, consecutive MMAs share the X slice and alternate the accumulator
      umma(t12r, xr1, yr2, id_pos, acc);
      umma(t12i, xr1, yi2, id_pos, acc);
      umma(t12r, xr2, yr1, id_pos, 1u);
      umma(t12i, xr2, yi1, id_pos, 1u);
      umma(t12r, xi1, yi2, id_neg, 1u);
      umma(t12i, xi1, yr2, id_pos, 1u);
      umma(t12r, xi2, yi1, id_neg, 1u);
      umma(t12i, xi2, yr1, id_pos, 1u);
      return;
    }
#endif
    umma(t12r, xr1, yr2, id_pos, acc_r);
    umma(t12r, xr2, yr1, id_pos, 1u);
    umma(t12r, xi1, yi2, id_neg, 1u);
    umma(t12r, xi2, yi1, id_neg, 1u);
    if (!drop_tiny) {
      umma(t12i, xr2, yi2, id_pos, acc);
      umma(t12i, xi2, yr2, id_pos, 1u);
      acc_i = 1u;
    }
    umma(t12i, xr1, yi2, id_pos, acc_i);
    umma(t12i, xr2, yi1, id_pos, 1u);
    umma(t12i, xi1, yr2, id_pos, 1u);
    umma(t12i, xi2, yr1, id_pos, 1u);
  } else {
    const uint32_t al = umma_desc_lo(a0), bl = umma_desc_lo(b0);
    const uint64_t xr1 = umma_desc_at(al, 0), xr2 = umma_desc_at(al, PART_BYTES), xr3 = umma_desc_at(al, 2 * PART_BYTES);
    const uint64_t xi1 = umma_desc_at(al, 3 * PART_BYTES), xi2 = umma_desc_at(al, 4 * PART_BYTES), xi3 = umma_desc_at(al, 5 * PART_BYTES);
    const uint64_t yr1 = umma_desc_at(bl, 0), yr2 = umma_desc_at(bl, YP), yr3 = umma_desc_at(bl, 2 * YP);
    const uint64_t yi1 = umma_desc_at(bl, 3 * YP), yi2 = umma_desc_at(bl, 4 * YP), yi3 = umma_desc_at(bl, 5 * YP);
    // C12r = sum over (i + j in {3, 4}) of xr_i yr_j - xi_i yi_j
    umma(t12r, xr1, yr3, id_pos, acc);
    umma(t12r, xr2, yr2, id_pos, 1u);
    umma(t12r, xr3, yr1, id_pos, 1u);
    umma(t12r, xi1, yi3, id_neg, 1u);
    umma(t12r, xi2, yi2, id_neg, 1u);
    umma(t12r, xi3, yi1, id_neg, 1u);
    umma(t12r, xr1, yr2, id_pos, 1u);
    umma(t12r, xr2, yr1, id_pos, 1u);
    umma(t12r, xi1, yi2, id_neg, 1u);
    umma(t12r, xi2, yi1, id_neg, 1u);
    // C12i = sum of xr_i yi_j + xi_i yr_j
    umma(t12i, xr1, yi3, id_pos, acc);
    umma(t12i, xr2, yi2, id_pos, 1u);
    umma(t12i, xr3, yi1, id_pos, 1u);
    umma(t12i, xi1, yr3, id_pos, 1u);
    umma(t12i, xi2, yr2, id_pos, 1u);
    umma(t12i, xi3, yr1, id_pos, 1u);
    umma(t12i, xr1, yi2, id_pos, 1u);
    umma(t12i, xr2, yi1, id_pos, 1u);
    umma(t12i, xi1, yr2, id_pos, 1u);
    umma(t12i, xi2, yr1, id_pos, 1u);
  }
}

// The leading products x1 y1 of one k-step (accumulators C0r, C0i): exact.
template <int FMT, bool PAIR>
__device__ __forceinline__ void issue_lead(uint32_t t0r, uint32_t t0i, uint32_t a0, uint32_t b0, uint32_t acc) {
  constexpr uint32_t id_pos = umma_idesc(Cfg<FMT>::AB_FORMAT, false, PAIR), id_neg = umma_idesc(Cfg<FMT>::AB_FORMAT, true, PAIR);
  constexpr int YP = PAIR ? PART_BYTES / 2 : PART_BYTES;
  constexpr int IM = (Cfg<FMT>::PARTS / 2) * PART_BYTES, IMY = (Cfg<FMT>::PARTS / 2) * YP;   // first imaginary slice
  auto umma = [](uint32_t d, uint64_t da, uint64_t db, uint32_t id, uint32_t ac) { umma_f16<PAIR>(d, da, db, id, ac); };
  const uint32_t al = umma_desc_lo(a0), bl = umma_desc_lo(b0);
  const uint64_t xr1 = umma_desc_at(al, 0), xi1 = umma_desc_at(al, IM), yr1 = umma_desc_at(bl, 0), yi1 = umma_desc_at(bl, IMY);
  umma(t0r, xr1, yr1, id_pos, acc);
  umma(t0r, xi1, yi1, id_neg, 1u);
  umma(t0i, xr1, yi1, id_pos, acc);
  umma(t0i, xi1, yr1, id_pos, 1u);
}

// WIDE (FP16X4, CTA pair): N = 256 MMAs on [Cr | Ci].  Stage layout of Y (64-row blocks of 2 KB):
//   slice 1: [-yi1][yr1][yi1]   slice 2: [-yi2][yr2][yi2];  Fr(j) = [yr_j ; yi_j] starts at block 1, Fi(j) = [-yi_j ; yr_j] at block 0.
constexpr int YB = PART_BYTES / 2;               // one 64-row block
__device__ __forceinline__ void issue_small_wide(uint32_t t12, uint32_t a0, uint32_t b0, uint32_t acc, bool drop_tiny) {
  constexpr uint32_t id = umma_idesc(Cfg<SL_FMT_FP16X4>::AB_FORMAT, false, true, 2 * TN);
  const uint64_t xr1 = umma_desc(a0), xr2 = umma_desc(a0 + PART_BYTES), xi1 = umma_desc(a0 + 2 * PART_BYTES), xi2 = umma_desc(a0 + 3 * PART_BYTES);
  const uint64_t fr1 = umma_desc(b0 + YB), fi1 = umma_desc(b0), fr2 = umma_desc(b0 + 4 * YB), fi2 = umma_desc(b0 + 3 * YB);
  uint32_t a = acc;
  if (!drop_tiny) {                              // tiniest first: x2 y2 (FP16X3 leaves them out)
    umma_f16<true>(t12, xr2, fr2, id, a);
    umma_f16<true>(t12, xi2, fi2, id, 1u);
    a = 1u;
  }
  umma_f16<true>(t12, xr1, fr2, id, a);
  umma_f16<true>(t12, xi1, fi2, id, 1u);
  umma_f16<true>(t12, xr2, fr1, id, 1u);
  umma_f16<true>(t12, xi2, fi1, id, 1u);
}
__device__ __forceinline__ void issue_lead_wide(uint32_t t0, uint32_t a0, uint32_t b0, uint32_t acc) {
  constexpr uint32_t id = umma_idesc(Cfg<SL_FMT_FP16X4>::AB_FORMAT, false, true, 2 * TN);
  umma_f16<true>(t0, umma_desc(a0), umma_desc(b0 + YB), id, acc);                      // xr1 . [yr1 ; yi1]
  umma_f16<true>(t0, umma_desc(a0 + 2 * PART_BYTES), umma_desc(b0), id, 1u);           // xi1 . [-yi1 ; yr1]
}

template <int EPI, int FMT, bool PAIR, bool WIDE>
__global__ void __launch_bounds__(NUM_THREADS, 1) k_sliced_contract(const SlParams p) {
  static_assert(!WIDE || (PAIR && FMT == SL_FMT_FP16X4), "the N = 256 formulation is built for FP16X4 on CTA pairs");
  using C = Cfg<FMT>;
  constexpr int STAGES = n_stages<EPI, FMT, PAIR, WIDE>();
  constexpr bool IS_G2 = EPI == EPI_GEMM2 || EPI == EPI_GEMM2_TILE, TILE = EPI == EPI_GEMM2_TILE;
  constexpr int X_BYTES = x_bytes<FMT>(), Y_BYTES = y_bytes<FMT, PAIR, WIDE>(), STAGE_BYTES = X_BYTES + Y_BYTES;
  constexpr int STEP_EL = sl_step_el(FMT);                               // X operand: elements per (row tile, k-step)
  constexpr int STEP_EL_Y = WIDE ? STEP_EL + 2 * SL_TILE_EL : STEP_EL;   // Y operand: + the negated imaginary slices
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + STAGES * STAGE_BYTES);
  uint64_t* full = bars;                       // [STAGES] operands of this CTA have landed
  uint64_t* empty = bars + STAGES;             // [STAGES] every MMA reading the stage has completed
  uint64_t* peer_full = bars + 2 * STAGES;     // [STAGES] (pair leader only) the peer CTA's operands have landed
  uint64_t* c0_full = bars + 3 * STAGES;       // leading accumulators of a chunk complete
  uint64_t* c0_empty = bars + 3 * STAGES + 1;  // ... drained by the epilogue warps (of both CTAs of a pair)
  uint64_t* c12_full = bars + 3 * STAGES + 2;  // small-product accumulators of a (tile, channel) complete
  uint64_t* c12_empty = bars + 3 * STAGES + 3;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 3 * STAGES + 4);
  float* acc_tile = reinterpret_cast<float*>(smem + STAGES * STAGE_BYTES + 512);   // EPI_GEMM2_TILE only

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // a worker is a CTA, or a pair of CTAs (cluster of 2 on one TPC) working on two row tiles of the same column tile
  const uint32_t rank = PAIR ? cluster_ctarank() : 0;
  const int worker = PAIR ? (int)(blockIdx.x >> 1) : (int)blockIdx.x, n_workers = PAIR ? (int)(gridDim.x >> 1) : (int)gridDim.x;
  const int n_my_items = p.n_items > worker ? (p.n_items - 1 - worker) / n_workers + 1 : 0;

  if (warp == 0 && lane == 0) {
    for (int s = 0; s < STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); mbar_init(&peer_full[s], 1); }
    mbar_init(c0_full, 1);
    mbar_init(c0_empty, PAIR ? 2 * NUM_EPI_WARPS : NUM_EPI_WARPS);
    mbar_init(c12_full, 1);
    mbar_init(c12_empty, PAIR ? 2 * NUM_EPI_WARPS : NUM_EPI_WARPS);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {   // the whole tensor memory: 512 columns (of both CTAs of a pair)
    if (PAIR) {
      asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    } else {
      asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(tmem_slot)) : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (PAIR) cluster_sync_all();          // the peer's barriers are initialised before anything arrives on them
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ================= bulk-copy producer =================
    if (lane == 0) {
      uint32_t it = 0;
      unsigned int sync_target = 0;
      bool in_step = p.sync_counter != nullptr;            // false once a meeting has timed out: free-running from then on
      for (int item = worker; item < p.n_items; item += n_workers) {
        int atom, rt, ct;
        decode_item(p, item, atom, rt, ct);
        const unsigned int active = (unsigned int)min(n_workers, p.n_items - (item - worker));   // workers with an item in this wave
        if (PAIR) rt = 2 * rt + (int)rank;
        // a CTA of a pair loads rows [64 rank, 64 rank + 64) of every part of the Y tile
        const uint16_t* ysrc = p.Y + (int64_t)atom * p.y_batch_stride + (int64_t)ct * p.ksteps * STEP_EL_Y + (PAIR ? rank * (SL_TILE_EL / 2) : 0);
        for (int n = 0; n < p.n_ch_loop; ++n) {
          const uint16_t* xsrc = p.X + (int64_t)atom * p.x_batch_stride + ((int64_t)n * p.n_rt_x + rt) * p.ksteps * STEP_EL;
          for (int ks = 0, next_sync = 0; ks < p.ksteps; ++ks, ++it) {
            if (in_step && ks == next_sync) {
              next_sync += p.sync_steps;
              sync_target += active;
              if (rank == 0) in_step = lockstep_arrive_wait(p.sync_counter, sync_target);
            }
            const int s = it % STAGES;
            mbar_wait(&empty[s], ((it / STAGES) & 1) ^ 1);
            uint8_t* st = smem + s * STAGE_BYTES;
#ifdef BIP_TUNING
            if (p.probe_x == 4 && ks > 0) {               // no operand traffic at all: issue + MMA only
              mbar_expect_tx(&full[s], 0);
              continue;
            } else if (p.probe_x == 1 && ks > 0) {
              mbar_expect_tx(&full[s], STAGE_BYTES - X_BYTES);
            } else {
              mbar_expect_tx(&full[s], STAGE_BYTES);
              const uint16_t* xs = p.probe_x == 2 ? p.X + (int64_t)atom * p.x_batch_stride + ((int64_t)n * p.n_rt_x + (PAIR ? (int)rank : 0)) * p.ksteps * STEP_EL : xsrc;
              bulk_load(st, xs + (int64_t)ks * STEP_EL, X_BYTES, &full[s]);
            }
#else
            mbar_expect_tx(&full[s], STAGE_BYTES);
            bulk_load(st, xsrc + (int64_t)ks * STEP_EL, X_BYTES, &full[s]);
#endif
            if (WIDE) {
              // parts in memory: re1 re2 im1 im2 -im1 -im2; blocks in the stage: [-im1][re1][im1][-im2][re2][im2]
              constexpr int dst_block[6] = {1, 4, 2, 5, 0, 3};
#pragma unroll
              for (int part = 0; part < 6; ++part)
                bulk_load(st + X_BYTES + dst_block[part] * YB, ysrc + (int64_t)ks * STEP_EL_Y + part * SL_TILE_EL, YB, &full[s]);
#ifdef BIP_TUNING
            } else if (PAIR && p.probe_x == 3) {          // timing probe (wrong data): the CTA's Y half as ONE copy instead of one per slice
              bulk_load(st + X_BYTES, ysrc + (int64_t)ks * STEP_EL, Y_BYTES, &full[s]);
#endif
            } else if (PAIR) {
#pragma unroll
              for (int part = 0; part < C::PARTS; ++part)
                bulk_load(st + X_BYTES + part * (PART_BYTES / 2), ysrc + (int64_t)ks * STEP_EL + part * SL_TILE_EL, PART_BYTES / 2, &full[s]);
            } else {
              bulk_load(st + X_BYTES, ysrc + (int64_t)ks * STEP_EL, X_BYTES, &full[s]);
            }
          }
        }
      }
      // tail: every tcgen05.commit arrival on the stage barriers has landed before the CTA may exit
      for (int j = 0; j < STAGES; ++j, ++it) mbar_wait(&empty[it % STAGES], ((it / STAGES) & 1) ^ 1);
    }
  } else if (warp == 1) {
    // ================= MMA issuer =================
    // The k-steps of all (tile, channel) segments of this worker form one sequence g = 0 .. total - 1.  The small
    // products of k-step g are issued first; the leading products follow through a second cursor (`pending` k-steps
    // behind).  When the leading cursor reaches a new chunk whose C0 the epilogue has not drained yet, the issuer
    // does not block: it keeps queueing small products (up to lag_max k-steps ahead), so the tensor pipe stays busy
    // during the drain, and the leading products catch up afterwards.  At a segment boundary the leading cursor
    // catches up first: the epilogue cannot release C12 before it has seen every C0 chunk but the last.
    // The whole warp runs the control flow (converged); one elected lane issues the tcgen05 instructions -- a
    // lane-divergent `if (lane == 0)` region makes ptxas wrap every uniform-datapath instruction in an ELECT loop,
    // and the issuing thread, not the tensor pipe, becomes the bottleneck (measured in round 1: the FP16X4 issue loop fell from 1.6 to 1.1 k clk per k-step).
    // In a pair only the leader CTA (rank 0) issues (tcgen05.mma.cta_group::2 drives both tensor cores); the peer's
    // warp 1 forwards "my operands have landed" to the leader's peer_full barriers.
    const uint32_t total = (uint32_t)n_my_items * (uint32_t)p.n_ch_loop * (uint32_t)p.ksteps;
    if (PAIR && rank != 0) {
      uint32_t s = 0, ph = 0;
      for (uint32_t g = 0; g < total; ++g) {
        mbar_wait(&full[s], ph);
        if (elect_one()) mbar_arrive_cluster(&peer_full[s], 0);
        __syncwarp();
        if (++s == STAGES) { s = 0; ph ^= 1; }
      }
    } else {
    const uint32_t t0r = tmem_base, t0i = tmem_base + TN, t12r = tmem_base + 2 * TN, t12i = tmem_base + 3 * TN;
    const uint32_t ksteps = (uint32_t)p.ksteps, chunk = (uint32_t)p.chunk_steps, lag_max = (uint32_t)p.lag_max;
    const uint32_t smem_base = smem_u32(smem);
    const bool drop_tiny = FMT == SL_FMT_FP16X4 && p.drop_tiny != 0;
    uint32_t s_small = 0, ph_small = 0;            // stage and phase of the small-product cursor
    uint32_t ks_s = 0, seg_par = 0;                // its k-step inside the segment; segment parity
    uint32_t s_lead = 0, ks_l = 0, in_chunk = 0, chunk_par = 0, pending = 0;   // leading-product cursor
    auto wait_epi = [&](uint64_t* bar, uint32_t parity) { mbar_wait(bar, parity); };
    auto lead = [&]() {
      if (in_chunk == 0) {
        wait_epi(c0_empty, chunk_par ^ 1);                           // epilogue has drained the previous chunk's C0
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      }
      ++ks_l;
      const bool chunk_end = in_chunk + 1 == chunk || ks_l == ksteps;
      if (elect_one()) {
        const uint32_t a0 = smem_base + s_lead * STAGE_BYTES;
        if (WIDE) issue_lead_wide(t0r, a0, a0 + X_BYTES, in_chunk ? 1u : 0u);
        else issue_lead<FMT, PAIR>(t0r, t0i, a0, a0 + X_BYTES, in_chunk ? 1u : 0u);
        umma_commit<PAIR>(&empty[s_lead]);                           // stage reusable once every MMA so far has read it
        if (chunk_end) umma_commit<PAIR>(c0_full);
      }
      __syncwarp();
      if (chunk_end) { in_chunk = 0; chunk_par ^= 1; } else ++in_chunk;
      if (ks_l == ksteps) ks_l = 0;
      if (++s_lead == STAGES) s_lead = 0;
      --pending;
    };
    for (uint32_t g = 0; g < total; ++g) {
      mbar_wait(&full[s_small], ph_small);
      if (PAIR) mbar_wait(&peer_full[s_small], ph_small);
      if (ks_s == 0) {
        while (pending) lead();
        wait_epi(c12_empty, seg_par ^ 1);                            // epilogue has drained the previous segment's C12
      }
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      const bool seg_end = ks_s + 1 == ksteps;
      if (elect_one()) {
        const uint32_t a0 = smem_base + s_small * STAGE_BYTES;
        if (WIDE) issue_small_wide(t12r, a0, a0 + X_BYTES, ks_s ? 1u : 0u, drop_tiny);
#ifdef BIP_TUNING
        else issue_small<FMT, PAIR>(t12r, t12i, a0, a0 + X_BYTES, ks_s ? 1u : 0u, drop_tiny, p.probe_x == 5);
#else
        else issue_small<FMT, PAIR>(t12r, t12i, a0, a0 + X_BYTES, ks_s ? 1u : 0u, drop_tiny);
#endif
        if (seg_end) umma_commit<PAIR>(c12_full);
      }
      __syncwarp();
      if (seg_end) { ks_s = 0; seg_par ^= 1; } else ++ks_s;
      if (++s_small == STAGES) { s_small = 0; ph_small ^= 1; }
      ++pending;
      while (pending) {
        if (in_chunk == 0 && pending < lag_max && !mbar_test(c0_empty, chunk_par ^ 1)) break;
        lead();
      }
    }
    while (pending) lead();
    }
  } else {
    // ================= epilogue warps =================
    const int quarter = warp & 3;                      // TMEM lanes [32 q, 32 q + 32) are visible to warps with warp % 4 == q
    const int half = (warp - 2) >> 2;                  // columns [64 half, 64 half + 64) of every accumulator
    // accumulator columns: N = 128 form  C0r | C0i | C12r | C12i (128 each, this warp's half at + 64 half);
    //                      WIDE          C0 = [Cr(d 0-63) | Ci(d 0-63) | Cr(d 64-127) | Ci(d 64-127)] | C12 likewise
    constexpr int IM_OFF = WIDE ? 64 : TN;
    const uint32_t t_lane = tmem_base + ((uint32_t)(quarter * 32) << 16) + half * (WIDE ? 128 : 64);
    const int n_chunks = (p.ksteps + p.chunk_steps - 1) / p.chunk_steps;
    uint32_t chunk_id = 0, seg = 0;
    for (int item = worker; item < p.n_items; item += n_workers) {
      int atom, rt, ct;
      decode_item(p, item, atom, rt, ct);
      if (PAIR) rt = 2 * rt + (int)rank;               // the leader's TMEM holds the even row tile, the peer's the odd one
      const int row = rt * TM + quarter * 32 + lane;   // this thread's rho (local row of the site under a crop mask)
      bool row_ok = row < p.n_rows;
      int out_row = row;
      if (IS_G2 && p.row_idx) {
        out_row = row_ok ? __ldg(p.row_idx + (int64_t)atom * p.row_idx_stride + row) : -1;
        row_ok = out_row >= 0;
      }
      const int col0 = ct * TN + half * 64;
      const float* sy = p.sy + (int64_t)atom * p.sy_batch_stride;
      float rowsum = 0.f;
      float* acc_row = acc_tile + (half * 64) * ACC_LD + quarter * 32 + lane;      // this thread's cells: acc_row[j * ACC_LD]
      if (TILE) {
#pragma unroll
        for (int j = 0; j < 64; ++j) acc_row[j * ACC_LD] = 0.f;
      }
      for (int n = 0; n < p.n_ch_loop; ++n, ++seg) {
        float rr[64], ri[64];
#pragma unroll
        for (int j = 0; j < 64; ++j) { rr[j] = 0.f; ri[j] = 0.f; }
#pragma unroll 1
        for (int c = 0; c <= n_chunks; ++c) {
          // n_chunks passes over the exact leading sums C0 and one over the small products C12, which is taken
          // before the last C0 chunk: C12 is complete LAG k-steps earlier, and releasing it first lets the issuer
          // start the next segment's small products while the last chunk drains
          const bool small = c == n_chunks - 1;
          if (small) mbar_wait(c12_full, seg & 1); else mbar_wait(c0_full, chunk_id & 1);
          asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
          const uint32_t tr = t_lane + (small ? 2 * TN : 0), ti = tr + IM_OFF;
#pragma unroll
          for (int g = 0; g < 2; ++g) {
            uint32_t v[32], u[32];
            tmem_ld32(tr + g * 32, v);
            tmem_ld32(ti + g * 32, u);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
            for (int j = 0; j < 32; ++j) { rr[g * 32 + j] += __uint_as_float(v[j]); ri[g * 32 + j] += __uint_as_float(u[j]); }
          }
          asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
          __syncwarp();
          if (lane == 0) {                           // the accumulators may be overwritten: tell the issuing CTA
            uint64_t* bar = small ? c12_empty : c0_empty;
            if (PAIR && rank != 0) mbar_arrive_cluster(bar, 0); else mbar_arrive(bar);
          }
          if (!small) ++chunk_id;
        }
        // ---- end of a (tile, channel): fused epilogue on the running sums ----
        const float sxr = row_ok ? p.sx[(int64_t)atom * p.sx_batch_stride + (int64_t)n * p.rows_pad + row] : 0.f;
        if (TILE) {
          const float sx2 = sxr * sxr;
#pragma unroll
          for (int j = 0; j < 64; ++j) {
            const int d = col0 + j;
            const float s = d < p.n_cols ? __ldg(sy + d) : 0.f;
            acc_row[j * ACC_LD] += fmaf(rr[j], rr[j], ri[j] * ri[j]) * (s * s) * sx2;
          }
        } else if (EPI == EPI_GEMM2) {
          const float sx2 = sxr * sxr;
          if (p.mode == BIP_MODE_MAP) {
            float acc = 0.f;
#pragma unroll
            for (int j = 0; j < 64; ++j) {
              const int d = col0 + j;
              const float s = d < p.n_cols ? __ldg(sy + d) : 0.f;
              acc = fmaf(fmaf(rr[j], rr[j], ri[j] * ri[j]), s * s, acc);
            }
            rowsum = fmaf(acc, sx2, rowsum);
          } else if (row_ok) {
            float* out = reinterpret_cast<float*>(p.out);
            const float f = sx2 * p.inv_G;
#pragma unroll
            for (int j = 0; j < 64; ++j) {
              const int d = col0 + j;
              if (d < p.n_cols) {
                const float s = __ldg(sy + d);
                const float v = fmaf(rr[j], rr[j], ri[j] * ri[j]) * (s * s) * f;
                const int dk = d % p.n_out_cols;
                if (p.mode == BIP_MODE_CUBE) atomicAdd(out + (int64_t)out_row * p.n_out_cols + dk, v);
                else atomicAdd(out + (int64_t)out_row * p.n_bins + __ldg(p.bin_of_det + dk), v);
              }
            }
          }
        } else if (row_ok) {
          // GEMM1: Psi[atom][rho][s], c64
          float2* dst = p.Psi + (int64_t)atom * p.psi_batch_stride + (int64_t)row * p.psi_ld;
#pragma unroll
          for (int j = 0; j < 64; j += 2) {
            const int s0 = col0 + j;
            if (s0 + 1 < p.n_cols) {
              const float a = sxr * __ldg(sy + s0), b = sxr * __ldg(sy + s0 + 1);
              *reinterpret_cast<float4*>(dst + s0) = make_float4(rr[j] * a, ri[j] * a, rr[j + 1] * b, ri[j + 1] * b);
            } else if (s0 < p.n_cols) {
              const float a = sxr * __ldg(sy + s0);
              dst[s0] = make_float2(rr[j] * a, ri[j] * a);
            }
          }
        }
      }
      if (EPI == EPI_GEMM2 && p.mode == BIP_MODE_MAP && row_ok)
        atomicAdd(reinterpret_cast<double*>(p.out) + out_row, (double)rowsum * (double)p.inv_G);
      if (TILE) {
        // flush: the eight epilogue warps take 16 rows each; a warp writes 32 consecutive detector columns per RED
        asm volatile("bar.sync 1, 256;" ::: "memory");
        float* out = reinterpret_cast<float*>(p.out);
        const int ew = warp - 2;
        for (int i = 0; i < 16; ++i) {
          const int rl = ew * 16 + i, grow = rt * TM + rl;
          int orow = grow < p.n_rows ? grow : -1;
          if (orow >= 0 && p.row_idx) orow = __ldg(p.row_idx + (int64_t)atom * p.row_idx_stride + grow);
          if (orow < 0) continue;
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const int c = lane + 32 * k, d = ct * TN + c;
            if (d < p.n_cols) {
              const float v = acc_tile[c * ACC_LD + rl] * p.inv_G;
              const int dk = d % p.n_out_cols;
              if (p.mode == BIP_MODE_CUBE) atomicAdd(out + (int64_t)orow * p.n_out_cols + dk, v);
              else atomicAdd(out + (int64_t)orow * p.n_bins + __ldg(p.bin_of_det + dk), v);
            }
          }
        }
        asm volatile("bar.sync 1, 256;" ::: "memory");
      }
    }
  }

  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (PAIR) {
    cluster_sync_all();                    // neither CTA frees tensor memory or exits while the other still uses its barriers
    if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
  } else {
    if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem_base) : "memory");
  }
}

// a5: Phi_n[rho][s] = H_n[s] Psi[rho][s] as sliced rows (n, rho) with their power-of-two scales.
// One block per (8 consecutive rho, chunk of QCH channels, atom); thread = (row = t & 7, k-group lane = t >> 3) in both
// passes.  Pass 1 sweeps Psi once (64 contiguous bytes per thread and iteration) for the row maxima of all channels of
// the chunk.  Pass 2 keeps 8 Psi values in registers and loops over the channels, so Psi is read twice in all (not
// twice per channel) and the 16-byte
// slice groups of the 8 rows of one k-group land in one contiguous 128-byte line (the blocked layout puts rows r .. r+7
// of a k-group side by side): every store instruction writes whole lines.
constexpr int QCH = 9;
__global__ void __launch_bounds__(256, 4) k_quantize_phi(const float2* __restrict__ Psi, int64_t psi_ld, int64_t psi_batch_stride,
                                                      const float2* __restrict__ H, Sliced Phi, int n_rho, int rows_pad, int w2, int n_ch) {
  __shared__ float inv_s[8][QCH];
  __shared__ int s_max[8][QCH];                      // row maxima as bit patterns (non-negative floats order like ints)
  const int rho0 = blockIdx.x * 8, n0 = blockIdx.y * QCH, atom = blockIdx.z;
  const int nch = min(QCH, n_ch - n0);
  const float2* pbase = Psi + (int64_t)atom * psi_batch_stride;
  const int n_groups = 2 * (int)Phi.ksteps;
  if (threadIdx.x < 8 * QCH) s_max[threadIdx.x / QCH][threadIdx.x % QCH] = 0;
  __syncthreads();
  {
    // sweep 1, same thread layout as the split below (row = t & 7, k-group lane = t >> 3): 64 contiguous bytes of Psi
    // per thread and iteration, independent iterations, the 9 channel maxima in registers
    const int r1 = threadIdx.x & 7, rho1 = rho0 + r1;
    float m[QCH];
#pragma unroll
    for (int c = 0; c < QCH; ++c) m[c] = 0.f;
    if (rho1 < n_rho) {
      const float2* prow1 = pbase + (int64_t)rho1 * psi_ld;
      for (int g = threadIdx.x >> 3; g < n_groups; g += 32) {
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const int s = g * 8 + j;
          if (s < w2) {
            const float2 a = prow1[s];
#pragma unroll
            for (int c = 0; c < QCH; ++c)
              if (c < nch) {
                const float2 h = H ? __ldg(H + (int64_t)(n0 + c) * w2 + s) : make_float2(1.f, 0.f);
                m[c] = fmaxf(m[c], fmaxf(fabsf(h.x * a.x - h.y * a.y), fabsf(h.x * a.y + h.y * a.x)));
              }
          }
        }
      }
#pragma unroll
      for (int c = 0; c < QCH; ++c)
        if (c < nch) atomicMax(&s_max[r1][c], __float_as_int(m[c]));
    }
  }
  __syncthreads();
  if (threadIdx.x < 8 * QCH) {
    const int rr = threadIdx.x / QCH, c = threadIdx.x % QCH, rho_w = rho0 + rr;
    if (c < nch) {
      const float scale = sl_pow2_scale(__int_as_float(s_max[rr][c]));
      inv_s[rr][c] = 1.f / scale;
      if (rho_w < n_rho) Phi.scale[(int64_t)atom * Phi.scale_batch_stride + (int64_t)(n0 + c) * rows_pad + rho_w] = scale;
    }
  }
  __syncthreads();
  const int r = threadIdx.x & 7, rho = rho0 + r;
  if (rho >= n_rho) return;
  const float2* prow = pbase + (int64_t)rho * psi_ld;
  for (int g = threadIdx.x >> 3; g < n_groups; g += 32) {
    float2 a[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const int s = g * 8 + j;
      a[j] = s < w2 ? prow[s] : make_float2(0.f, 0.f);
    }
    for (int c = 0; c < nch; ++c) {
      const float2* hrow = H + (int64_t)(n0 + c) * w2;
      float re[8], im[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const int s = g * 8 + j;
        const float2 h = s < w2 ? (H ? __ldg(hrow + s) : make_float2(1.f, 0.f)) : make_float2(0.f, 0.f);
        re[j] = h.x * a[j].x - h.y * a[j].y;
        im[j] = h.x * a[j].y + h.y * a[j].x;
      }
      sl_store_group(Phi, atom, (int64_t)(n0 + c) * rows_pad + rho, g, re, im, inv_s[r][c]);
    }
  }
}

// Crop mask: the illumination rows of every site's own scan positions, gathered from the shared
// matrix A into a per-site X operand.  One thread per (site, local row, group of 8 beams); rows without a scan are zero.
__global__ void __launch_bounds__(256) k_gather_rows_sliced(Sliced src, const int32_t* __restrict__ row_idx, int64_t idx_stride,
                                                            Sliced dst, int n_groups) {
  const int g = blockIdx.y * blockDim.x + threadIdx.x;   // rows in gridDim.x: a site may keep more than 65535 scan rows
  const int row = blockIdx.x, atom = blockIdx.z;
  if (g >= n_groups) return;
  const int s = row_idx[(int64_t)atom * idx_stride + row];
  const int parts = sl_parts_of(src);
  uint16_t* d = dst.base + (int64_t)atom * dst.batch_stride + sl_group_offset(dst, row, g);
  const uint16_t* q = s >= 0 ? src.base + sl_group_offset(src, s, g) : nullptr;
  for (int part = 0; part < parts; ++part)
    *reinterpret_cast<uint4*>(d + part * SL_TILE_EL) = q ? *reinterpret_cast<const uint4*>(q + part * SL_TILE_EL) : make_uint4(0, 0, 0, 0);
  if (g == 0) dst.scale[(int64_t)atom * dst.scale_batch_stride + row] = s >= 0 ? src.scale[s] : 1.f;
}

constexpr int CROP_THREADS = 1024;
// Crop mask (reading c19): the scan rows of every site, in ascending scan order.  One block of 32 warps per site; warp w owns
// the contiguous scans [w S, (w + 1) S), S = ceil(n_rho / 1024) * 32, and walks them 32 at a time (coalesced reads of the scan
// list): a first sweep counts the scans inside the window, the 32 warp totals give every warp its offset, a second sweep writes
// the rows with ballot-ordered offsets -- no block barrier inside the sweeps (the one-chunk-of-256-at-a-time version needed
// three per chunk; each iteration is one L2 round trip, so the sweeps are latency-bound and want many warps).  fp64, the oracle's expression order:
// d = ((rho - c + N/2) mod N) - N/2, inside iff |d_y| < N_y / (2 f_y) and |d_x| < N_x / (2 f_x).
__global__ void __launch_bounds__(CROP_THREADS) k_crop_rows(const double* __restrict__ rho, int n_rho, const int32_t* __restrict__ origin, int w,
                                                   int ny, int nx, int fy, int fx, int32_t* __restrict__ row_idx, int64_t idx_stride,
                                                   int32_t* __restrict__ counts) {
  __shared__ int warp_tot[CROP_THREADS / 32];
  const int atom = blockIdx.x, t = threadIdx.x, lane = t & 31, wid = t >> 5;
  const double cy = (double)((origin[2 * atom] + w / 2) % ny), cx = (double)((origin[2 * atom + 1] + w / 2) % nx);
  const double hy = ny / (2.0 * fy), hx = nx / (2.0 * fx);
  int32_t* out = row_idx ? row_idx + (int64_t)atom * idx_stride : nullptr;   // NULL: count only
  const int S = ((n_rho + CROP_THREADS - 1) / CROP_THREADS) * 32, r0 = wid * S, r1 = min(n_rho, r0 + S);
  // fmod(a, n) for a power-of-two n: a - n trunc(a (1 / n)), every step exact (a scaling, an integer, a difference whose bits are
  // the low bits of a) and therefore bit-identical to fmod, at a tenth of its cost; any other n takes fmod itself
  const bool pow2 = (ny & (ny - 1)) == 0 && (nx & (nx - 1)) == 0;
  const double inv_ny = 1.0 / ny, inv_nx = 1.0 / nx;      // exact for powers of two: the quotient is a product (fp64 division costs ~30 instructions)
  auto fmod_n = [&](double a, int n, double inv_n) { return pow2 ? a - (double)n * trunc(a * inv_n) : fmod(a, (double)n); };
  auto inside = [&](int r) {
    if (r >= r1) return false;
    const double2 p = *reinterpret_cast<const double2*>(rho + 2 * (int64_t)r);
    double dy = fmod_n(p.x - cy + ny / 2.0, ny, inv_ny);
    double dx = fmod_n(p.y - cx + nx / 2.0, nx, inv_nx);
    if (dy < 0) dy += ny;
    if (dx < 0) dx += nx;
    dy -= ny / 2.0; dx -= nx / 2.0;
    return fabs(dy) < hy && fabs(dx) < hx;
  };
  int n = 0;
  for (int r = r0 + lane; r < r0 + S; r += 32) n += __popc(__ballot_sync(0xffffffffu, inside(r)));
  if (lane == 0) warp_tot[wid] = n;
  __syncthreads();
  int off = 0, total = 0;
  for (int k = 0; k < CROP_THREADS / 32; ++k) { if (k < wid) off += warp_tot[k]; total += warp_tot[k]; }
  if (out) {
    for (int r = r0 + lane; r < r0 + S; r += 32) {
      const bool in = inside(r);
      const unsigned m = __ballot_sync(0xffffffffu, in);
      if (in) out[off + __popc(m & ((1u << lane) - 1u))] = r;
      off += __popc(m);
    }
    for (int64_t i = total + t; i < idx_stride; i += CROP_THREADS) out[i] = -1;
  }
  if (t == 0) counts[atom] = total;
}

template <int EPI, int FMT, bool PAIR, bool WIDE = false>
int32_t launch_fmt(bip_ctx* ctx, const SlParams& p) {
  // per context (= per device): the shared-memory opt-in and the occupancy of this kernel variant
  KernelInfo& ki = ctx->kernel_info[reinterpret_cast<const void*>(&k_sliced_contract<EPI, FMT, PAIR, WIDE>)];
  if (!ki.attr_set) {
    BIP_CUDA(ctx, cudaFuncSetAttribute(k_sliced_contract<EPI, FMT, PAIR, WIDE>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes<EPI, FMT, PAIR, WIDE>()));
    ki.attr_set = true;
  }
  SlParams q = p;
  q.n_rt_x = p.n_rt;
  if (PAIR) {
    if (p.n_rt % 2) return fail(ctx, BIP_ERR_INVALID, "pair kernel: the X operand must be padded to a multiple of 256 rows");
    q.n_rt = p.n_rt / 2;
  }
  q.n_items = p.n_items / p.n_rt * q.n_rt;
  if (q.n_items <= 0) return BIP_OK;
  q.chunk_steps = Cfg<FMT>::CHUNK_STEPS;                 // fixed: the exactness of the leading sums depends on it
#ifdef BIP_TUNING
  q.chunk_steps = std::max(1, tune_int("BIP_TUNE_CHUNK", q.chunk_steps));   // timing probe only: longer chunks are no longer exact
#endif
#ifdef BIP_TUNING
  q.probe_x = tune_int("BIP_TUNE_PROBE_X", 0);
#endif
  q.dgroup = std::max(1, tune_int("BIP_TUNE_DGROUP", DGROUP_DEFAULT));
  q.lag_max = std::min(std::max(1, tune_int("BIP_TUNE_LAG", Cfg<FMT>::LAG_MAX)), n_stages<EPI, FMT, PAIR, WIDE>() - 1);
  int workers = std::max(1, std::min(q.n_items, PAIR ? ctx->sm_count / 2 : ctx->sm_count));
  workers = std::max(1, std::min(workers, tune_int("BIP_TUNE_WORKERS", workers)));
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(PAIR ? 2 * workers : workers);
  cfg.blockDim = dim3(NUM_THREADS);
  cfg.dynamicSmemBytes = smem_bytes<EPI, FMT, PAIR, WIDE>();
  cfg.stream = ctx->stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = PAIR ? 2 : 1; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  // Lockstep pays only when every worker is resident at once: checked against the occupancy the driver reports for
  // this launch configuration (once per context and kernel variant).  The wait itself is bounded (lockstep_arrive_wait).
  if (ki.max_clusters < 0) {
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, k_sliced_contract<EPI, FMT, PAIR, WIDE>, &cfg) != cudaSuccess) { cudaGetLastError(); n = 0; }
    ki.max_clusters = n;
  }
  q.sync_counter = nullptr;
  q.sync_steps = std::max(1, tune_int("BIP_TUNE_SYNCSTEPS", 1 << 30));   // default: once per (item, channel) segment
  if (tune_int("BIP_TUNE_LOCKSTEP", 1) != 0 && workers <= ki.max_clusters) {   // a fresh zeroed counter per launch (64 slots, cleared on the stream)
    BIP_TRY(ensure(ctx, ctx->Sync, 64 * sizeof(unsigned int), "lockstep counters"));
    q.sync_counter = reinterpret_cast<unsigned int*>(ctx->Sync.p) + (ctx->sync_slot++ & 63);
    BIP_CUDA(ctx, cudaMemsetAsync(q.sync_counter, 0, sizeof(unsigned int), ctx->stream));
  }
  BIP_CUDA(ctx, cudaLaunchKernelEx(&cfg, k_sliced_contract<EPI, FMT, PAIR, WIDE>, q));
  ctx->timing.kernel_launches++;
  return BIP_OK;
}

template <int EPI>
int32_t launch(bip_ctx* ctx, const SlParams& p, int fmt, bool y_neg) {
  const bool pair = tune_int("BIP_TUNE_PAIR", 1) != 0, tile = tune_int("BIP_TUNE_TILEACC", 1) != 0;
  if (y_neg) {   // the Y operand carries the negated imaginary slices: the N = 256 formulation (FP16X4 on CTA pairs)
    if (!pair || fmt != SL_FMT_FP16X4) return fail(ctx, BIP_ERR_INVALID, "contraction: a Y operand with negated imaginary slices needs the FP16X4 pair kernel");
    if (tile && EPI == EPI_GEMM2 && p.mode != BIP_MODE_MAP) return launch_fmt<EPI_GEMM2_TILE, SL_FMT_FP16X4, true, true>(ctx, p);
    return launch_fmt<EPI, SL_FMT_FP16X4, true, true>(ctx, p);
  }
  if (pair && tile && EPI == EPI_GEMM2 && p.mode != BIP_MODE_MAP)
    return fmt == SL_FMT_FP16X4 ? launch_fmt<EPI_GEMM2_TILE, SL_FMT_FP16X4, true>(ctx, p) : launch_fmt<EPI_GEMM2_TILE, SL_FMT_BF16X6, true>(ctx, p);
  if (pair) return fmt == SL_FMT_FP16X4 ? launch_fmt<EPI, SL_FMT_FP16X4, true>(ctx, p) : launch_fmt<EPI, SL_FMT_BF16X6, true>(ctx, p);
  return fmt == SL_FMT_FP16X4 ? launch_fmt<EPI, SL_FMT_FP16X4, false>(ctx, p) : launch_fmt<EPI, SL_FMT_BF16X6, false>(ctx, p);
}

}  // namespace

int32_t launch_gemm1_sliced(bip_ctx* ctx, const Gemm1SlArgs& a) {
  if (a.A.fmt != a.R1t.fmt || a.A.neg_im) return fail(ctx, BIP_ERR_INVALID, "gemm1: operand formats differ");
  SlParams p{};
  p.X = a.A.base; p.sx = a.A.scale; p.x_batch_stride = a.A.batch_stride; p.sx_batch_stride = a.A.scale_batch_stride;
  p.Y = a.R1t.base; p.sy = a.R1t.scale; p.y_batch_stride = a.R1t.batch_stride; p.sy_batch_stride = a.R1t.scale_batch_stride;
  p.ksteps = (int)a.A.ksteps;
  p.n_rt = (int)(a.A.rows_pad / TM);
  p.n_ct = (int)(a.R1t.rows_pad / TN);
  p.n_items = a.n_atoms * p.n_rt * p.n_ct;
  p.n_ch_loop = 1;
  p.drop_tiny = a.drop_tiny;
  p.n_rows = a.n_rho; p.n_cols = a.w2; p.rows_pad = (int)a.A.rows_pad;
  p.Psi = a.Psi; p.psi_ld = a.psi_ld; p.psi_batch_stride = a.psi_batch_stride;
  return launch<EPI_GEMM1>(ctx, p, a.A.fmt, a.R1t.neg_im != 0);
}

int32_t launch_crop_rows(bip_ctx* ctx, const int32_t* origin_dev, int32_t n_atoms, int32_t w, int32_t* row_idx, int64_t idx_stride, int32_t* counts) {
  k_crop_rows<<<(unsigned)n_atoms, CROP_THREADS, 0, ctx->stream>>>(ctx->rho_dev, ctx->n_rho, origin_dev, w, ctx->g.ny, ctx->g.nx, ctx->crop_fy,
                                                          ctx->crop_fx, row_idx, idx_stride, counts);
  BIP_CUDA(ctx, cudaGetLastError());
  ctx->timing.kernel_launches++;
  return BIP_OK;
}

int32_t launch_gather_rows_sliced(bip_ctx* ctx, const Sliced& src, const int32_t* row_idx, int64_t idx_stride, const Sliced& dst, int32_t n_atoms) {
  const int n_groups = 2 * (int)src.ksteps;
  dim3 grid((unsigned)dst.rows_pad, (unsigned)((n_groups + 255) / 256), (unsigned)n_atoms);
  k_gather_rows_sliced<<<grid, 256, 0, ctx->stream>>>(src, row_idx, idx_stride, dst, n_groups);
  BIP_CUDA(ctx, cudaGetLastError());
  ctx->timing.kernel_launches++;
  return BIP_OK;
}

int32_t launch_quantize_phi(bip_ctx* ctx, const float2* Psi, int64_t psi_ld, int64_t psi_batch_stride, const float2* H,
                            const Sliced& Phi, int32_t n_rho, int32_t rows_pad, int32_t w2, int32_t n_ch, int32_t n_atoms) {
  dim3 grid((unsigned)((n_rho + 7) / 8), (unsigned)((n_ch + QCH - 1) / QCH), (unsigned)n_atoms);
  k_quantize_phi<<<grid, 256, 0, ctx->stream>>>(Psi, psi_ld, psi_batch_stride, H, Phi, n_rho, rows_pad, w2, n_ch);
  BIP_CUDA(ctx, cudaGetLastError());
  ctx->timing.kernel_launches++;
  return BIP_OK;
}

int32_t launch_gemm2_sliced(bip_ctx* ctx, const Gemm2SlArgs& a) {
  if (a.Phi.fmt != a.R2.fmt || a.Phi.neg_im) return fail(ctx, BIP_ERR_INVALID, "gemm2: operand formats differ");
  SlParams p{};
  p.X = a.Phi.base; p.sx = a.Phi.scale; p.x_batch_stride = a.Phi.batch_stride; p.sx_batch_stride = a.Phi.scale_batch_stride;
  p.Y = a.R2.base; p.sy = a.R2.scale; p.y_batch_stride = a.R2.batch_stride; p.sy_batch_stride = a.R2.scale_batch_stride;
  p.ksteps = (int)a.Phi.ksteps;
  p.rows_pad = a.rows_pad;
  p.n_rt = a.rows_pad / TM;
  p.n_ct = (int)(a.R2.rows_pad / TN);
  p.n_items = a.n_atoms * p.n_rt * p.n_ct;
  p.n_ch_loop = a.n_ch;
  p.drop_tiny = a.drop_tiny;
  p.n_rows = a.n_rho; p.n_cols = a.n_det;
  p.n_out_cols = a.n_out_cols > 0 ? a.n_out_cols : a.n_det;
  p.mode = a.mode; p.inv_G = a.inv_G; p.bin_of_det = a.bin_of_det; p.n_bins = a.n_bins; p.out = a.out;
  p.row_idx = a.row_idx; p.row_idx_stride = a.row_idx_stride;
  return launch<EPI_GEMM2>(ctx, p, a.Phi.fmt, a.R2.neg_im != 0);
}

}  // namespace bip
