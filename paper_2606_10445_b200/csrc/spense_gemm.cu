// Spense hybrid sparse-dense FP8 GEMM for sm_100a (tcgen05 + TMEM + TMA) on CTA PAIRS: one kernel for every token count,
// from decode (M = 1) to prefill-shaped calls.
//
// Three walks, written once as per-role device functions:
//   MODE 0  gate_up : output-split.  Pair tile = 2 operands of 128 rows = the gate and up rows of 128
//                     intermediate indices (interleaved, spense_internal.cuh); tiles below I_s are 2:4 compressed
//                     (tcgen05.mma.sp), the rest dense (tcgen05.mma).  Epilogue: scales -> SiLU(g)*u (Eq. 4) -> E4M3.
//   MODE 1  down    : input-split (also the stand-alone in-split linear).  Pair tile = 2 x 128 rows of the
//                     weight; the K loop runs the sparse stages and then the dense stages INTO THE SAME TMEM ACCUMULATOR.
//   MODE 2          : the stand-alone out-split linear: the tile walk of MODE 0 on 256-row tiles, the plain epilogue of MODE 1.
// spense_gemm_kernel<MODE, DYN>: DYN = gate_up that keeps h in fp32 and tracks max|h| per token (dynamic requant).
//
// Swap-AB: only the A operand of tcgen05.mma.sp can be sparse, so weights are A and tokens are B (MMA-N = padded token
// count); the accumulator holds Y^T [weight rows x tokens].
//
//   * CTA PAIRS (cluster of 2, tcgen05 cta_group::2).  One MMA instruction spans both SMs: M = 256 weight rows = the two
//     operands of a pair stage, ONE PER CTA (the blob stores stages operand-major and every gate_up operand is a
//     self-contained GLU tile), N = 16 .. 256 tokens, of which each CTA stages HALF (the B operand of a cta_group::2 MMA
//     is split across the pair).  Per MMA a CTA fills and reads 128 weight rows + N/2 token rows of shared memory.
//   * One accumulator of up to 240 columns per tile and CTA, DOUBLE BUFFERED (2 x 240 TMEM columns + 16 columns of 2:4
//     metadata = 496 <= 512): the epilogue of a tile overlaps the MMAs of the next one.  241..256 tokens run as one
//     256-column tile with a single buffer.
//   * The grid is a cost-balanced STREAM-K: the linear sequence of stage images (= the byte order of the blob) is cut into
//     n_spans spans, one persistent CTA pair per span (decode is weight-streaming bound: every SM streams an equal share).
//     A tile whose stages fall into several spans is fixed up through an L2-resident fp32 workspace, always adding the
//     partials in span order, so results are bitwise reproducible:
//       2 spans  : the second span finishes its part early (it is its first segment), dumps it and publishes a flag; the
//                  first span (owner) PRELOADS it into its TMEM accumulator before its own MMAs of that tile start;
//       > 2 spans: every span finishes late, so all dump, and the n spans reduce M/n token columns each (reduce-scatter)
//                  through the idle stage ring.
//     Flags hold the epoch of the launch (a device-side counter in the workspace): nothing is reset between launches and
//     CUDA-graph replays see fresh values.  Span i runs on pair n_spans-1-i.  The CTAs of a launch wait for each other, so
//     all of them must be co-resident: 1 CTA/SM by construction (shared memory); the host checks the cluster occupancy the
//     device offers and every wait is bounded (spense_gemm_common.cuh).
//   * More than 240 (256) tokens: token blocks side by side in one launch (grid = blocks x spans x 2 CTAs): the pairs of
//     different blocks walk the same schedule, so a weight stage is read from HBM once and found in L2 by the other blocks.
//   * Weights arrive by TENSOR copies (the blob section seen as rows of 128 bytes, one box = one operand image) because
//     only cp.async.bulk.tensor has the .cta_group::2 form whose completion counts on the LEADER CTA's barrier: the
//     leader's MMA thread waits on one barrier for both CTAs' halves of a stage.
//   * gate_up and down are chained with programmatic dependent launch: the next kernel's CTAs start as this kernel's CTAs
//     exit and fill their rings with weights (which depend on nothing); only activation loads wait.  While a CTA runs its
//     fix-up tail its producer prefetches the first stages of the NEXT kernel's spans into L2 (paced).
//
// Roles per CTA (640 threads): warp 0 weight producer (the CTA's operand), warp 3 activation producer (its half of the
// token tile), warp 1 MMA issuer (leader CTA only), warp 2 TMEM allocator, warps 4-19 epilogue of the CTA's own 128
// accumulator lanes (TMEM lane quadrant = warp & 3, quarter of the token columns = (warp - 4) >> 2).
//
// History (measured on B200, profiles/): a single-CTA-per-span kernel (MMA M = 128 x 2 operands per CTA, bulk copies of
// whole pair stages) served up to 112 tokens until round 2; with the TMEM preload of the partner's partial and without the
// producer's L2 prefetch-ahead the pair kernel is as fast or faster at every token count (M = 1: 50.4 vs 50.6 us/layer,
// 64: 53.8 vs 57.1, 112 all dense: 73.9 vs 82.2), so the other kernel was removed.
#include <mutex>

#include "spense_gemm_common.cuh"

namespace spense {

namespace {

using namespace dev;

__device__ __forceinline__ void epi_sync() { asm volatile("bar.sync 1, 512;" ::: "memory"); }   // the 16 epilogue warps

constexpr int kEpiThreads = 512;
constexpr int kEpiWarps = kEpiThreads / 32;
constexpr int kThreads = 128 + kEpiThreads;
constexpr int kTmemCols = 512;
constexpr int kMetaCol = 480;   // 2 buffers x 8 columns of 2:4 metadata (one operand, K 256)

struct Ctx {
  uint32_t smem_base;          // 1 KB aligned start of the stage ring (shared address)
  uint8_t* smem_gen;           // the same, generic
  int S;                       // ring slots
  uint32_t slot_bytes, ring_bytes, bar_base, b_half_bytes, tmem_base;
  uint32_t rank;               // CTA of the pair: 0 = leader (issues the MMAs), holds operand `rank` and token half `rank`
  int blk;                     // token block of this pair
  int slot0;                   // fix-up slot of span 0 of this block and rank: slot(span) = slot0 + 2 * span
  __device__ __forceinline__ uint32_t full_bar(int s) const { return bar_base + 8u * s; }
  __device__ __forceinline__ uint32_t empty_bar(int s) const { return bar_base + 8u * (8 + s); }
  __device__ __forceinline__ uint32_t accf_bar(int b) const { return bar_base + 8u * (16 + b); }
  __device__ __forceinline__ uint32_t acce_bar(int b) const { return bar_base + 8u * (18 + b); }
  __device__ __forceinline__ uint32_t tmem_slot() const { return bar_base + 8u * 20; }
  __device__ __forceinline__ uint32_t red_bar() const { return bar_base + 8u * 22; }
  __device__ __forceinline__ uint32_t pre_bar() const { return bar_base + 8u * 24; }
  __device__ __forceinline__ volatile uint32_t* tmem_slot_ptr() const { return reinterpret_cast<volatile uint32_t*>(smem_gen + ring_bytes + 8 * 20); }
  __device__ __forceinline__ volatile int* epoch_ptr() const { return reinterpret_cast<volatile int*>(smem_gen + ring_bytes + 8 * 21); }
  __device__ __forceinline__ volatile int* epi_done_ptr() const { return reinterpret_cast<volatile int*>(smem_gen + ring_bytes + 8 * 23); }
  __device__ __forceinline__ float4* sc0() const { return reinterpret_cast<float4*>(smem_gen + ring_bytes + 256); }
  __device__ __forceinline__ float* sc1(int n_pad) const { return reinterpret_cast<float*>(smem_gen + ring_bytes + 256 + 16 * n_pad); }
};

struct Group { int a, b, tile, first; };

// The three roles below run with their WHOLE warp converged and one elected lane issuing: every value they compute is
// warp-uniform (the compiler keeps it in uniform registers, which is where TMA / tcgen05 instructions take their operands
// from), and their loops are a few dozen instructions per stage.  That matters here: a stage is only 4 MMAs of 64-120
// cycles, and a single thread working through ~150 dependent instructions per stage (descriptor construction, cursor
// bookkeeping) was the bottleneck of the first version of this kernel (measured: the MMA thread busy 350 ns per stage
// with the tensor pipe 26 % active).

// Slot image: [operand: values 16 KB | metadata 4 KB] [token half-tile(s): n_pad/2 rows x 128 B, two for a sparse stage].
// Every copy counts on the LEADER's full barrier; the leader's weight producer arms it with the bytes of both CTAs.

// ===================== weight producer (warp 0 of each CTA) =====================
// This CTA's operand of every stage of the span; weights never depend on the previous kernel of the stream.
template <int MODE>
__device__ __forceinline__ void producer_weights(const GemmParams& p, const CUtensorMap* tmap_ws, const CUtensorMap* tmap_wd,
                                                 const Ctx& cx, int span) {
  const bool issuer = elect_one();
  const int S = cx.S;
  const int sb = p.span_begin[span];
  const int n = p.span_begin[span + 1] - sb;
  // one token block: a weight byte is used once (evict first); several: the pairs of the other blocks read the same
  // stage at about the same time and should find it in L2
  const uint64_t pol_w = p.nb == 1 ? policy_evict_first() : policy_evict_normal();
  unsigned long long off;
  Cursor c = cursor_at<MODE>(p, sb, &off);
  uint32_t row = (uint32_t)(off >> 7) + cx.rank * (uint32_t)(c.j < c.ns ? kSparseOperandBytes >> 7 : kOperandBytes >> 7);
  const uint32_t lead_full0 = mapa_shared(cx.full_bar(0), 0);
  const uint32_t tx_s = 2u * ((uint32_t)kSparseOperandBytes + 2u * cx.b_half_bytes), tx_d = 2u * ((uint32_t)kOperandBytes + cx.b_half_bytes);
  int slot = 0;
  uint32_t par = 1;                                        // parity a fresh empty barrier passes
  uint32_t dst = cx.smem_base, fb_lead = lead_full0, fb = cx.full_bar(0), eb = cx.empty_bar(0);
#pragma unroll 1
  for (int w = 0; w < n; ++w) {
    const bool sp = c.j < c.ns;
    const uint32_t rows = sp ? (uint32_t)(kSparseOperandBytes >> 7) : (uint32_t)(kOperandBytes >> 7);
    if (w >= S) wait_bar(p, eb, par);
    if (issuer) {
      if (cx.rank == 0) mbar_expect_tx(fb, sp ? tx_s : tx_d);
      tma_load_2d_pair(dst, sp ? tmap_ws : tmap_wd, 0, (int)row, fb_lead, pol_w);
    }
    row += 2u * rows;
    if (++c.j == c.ns + c.nd) next_tile<MODE>(p, c);
    if ((c.j < c.ns) != sp) row += cx.rank * (uint32_t)(sp ? -32 : 32);   // the other stage kind: operand 1 starts 32 rows earlier / later
    if (++slot == S) { slot = 0; par ^= 1u; dst = cx.smem_base; fb_lead = lead_full0; fb = cx.full_bar(0); eb = cx.empty_bar(0); }
    else { dst += cx.slot_bytes; fb_lead += 8u; fb += 8u; eb += 8u; }
    if (w == 0) trace(p, span, 1);
  }
}

// ===================== activation producer (warp 3 of each CTA) =====================
// This CTA's half of the token tile of every stage; waits for the previous kernel of the stream first.
template <int MODE>
__device__ __forceinline__ void producer_tokens(const GemmParams& p, const CUtensorMap* tmap_b, const Ctx& cx, int span) {
  const bool issuer = elect_one();
  const int S = cx.S;
  const int sb = p.span_begin[span];
  const int n = p.span_begin[span + 1] - sb;
  const uint64_t pol_a = policy_evict_last();
  unsigned long long off;
  Cursor c = cursor_at<MODE>(p, sb, &off);
  const uint32_t lead_full0 = mapa_shared(cx.full_bar(0), 0);
  const int tok0 = cx.blk * p.n_pad + (int)cx.rank * (p.n_pad >> 1);   // first token row of this CTA's half
  pdl_wait();
  int slot = 0;
  uint32_t par = 1;
  uint32_t dst = cx.smem_base + kSparseOperandBytes, fb_lead = lead_full0, eb = cx.empty_bar(0);
#pragma unroll 1
  for (int b = 0; b < n; ++b) {
    const bool sp = c.j < c.ns;
    const int k0 = sp ? c.j * kSparseStageK : p.dense_k0 + (c.j - c.ns) * kDenseStageK;
    if (b >= S) wait_bar(p, eb, par);
    if (issuer) {
      tma_load_2d_pair(dst, tmap_b, k0, tok0, fb_lead, pol_a);
      if (sp) tma_load_2d_pair(dst + cx.b_half_bytes, tmap_b, k0 + 128, tok0, fb_lead, pol_a);
    }
    if (++c.j == c.ns + c.nd) next_tile<MODE>(p, c);
    if (++slot == S) { slot = 0; par ^= 1u; dst = cx.smem_base + kSparseOperandBytes; fb_lead = lead_full0; eb = cx.empty_bar(0); }
    else { dst += cx.slot_bytes; fb_lead += 8u; eb += 8u; }
  }
}

// L2 prefetch of what the NEXT kernel of the stream streams first, issued while this CTA runs its fix-up tail (pairs of the
// launch's first token block; each CTA of the pair takes half of the span's range): one 32 KB chunk per pf_pace_ns so the
// fix-up traffic is not queued behind it; stops with the epilogue.
__device__ __forceinline__ void prefetch_next(const GemmParams& p, const Ctx& cx, int span) {
  if (!p.next_base || cx.blk != p.blk0) return;
  const uint32_t half = (p.next_len[span] >> 1) & ~1023u;
  const uint8_t* nb = p.next_base + (size_t)p.next_off[span] + (size_t)cx.rank * half;
  long long t_next = globaltimer();
#pragma unroll 1
  for (uint32_t o = 0; o < half && *cx.epi_done_ptr() == 0; o += 32768u) {
    const uint32_t chunk = half - o < 32768u ? half - o : 32768u;
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(nb + o), "r"(chunk) : "memory");
    t_next += p.pf_pace_ns;
    while (globaltimer() < t_next && *cx.epi_done_ptr() == 0) __nanosleep(64);
  }
}

// shared-memory matrix descriptors as two words: lo = address >> 4 | LBO >> 4 << 16 (so stepping through a slot or the ring
// is an add on lo), hi = SBO >> 4 | version | layout (constant)
__device__ __forceinline__ uint32_t desc_lo(uint32_t saddr, uint32_t lbo_bytes) { return ((saddr >> 4) & 0x3FFFu) | (((lbo_bytes >> 4) & 0x3FFFu) << 16); }
__device__ __forceinline__ uint32_t desc_hi(uint32_t sbo_bytes, uint32_t layout) { return ((sbo_bytes >> 4) & 0x3FFFu) | (1u << 14) | (layout << 29); }
__device__ __forceinline__ uint64_t desc_of(uint32_t lo, uint32_t hi) { return (uint64_t)lo | ((uint64_t)hi << 32); }

// A span's LAST segment that is the head of a tile shared with exactly one more span (the next one, which dumped the
// tail's partial as its first piece of work, long ago): this span owns the tile.  Instead of adding the partner's partial
// in the final, exposed epilogue (one L2 round trip per 16 token columns: 5 us of tail at 128 tokens, 10 us at 256), each
// CTA's epilogue warps store it into the TMEM accumulator BEFORE the segment's MMAs start, while earlier MMAs run, and the
// MMAs accumulate on top: the final epilogue is the plain one.  (Measured: M = 128 63.9 -> 60.6 us/layer, M = 240
// 96.7 -> 83.5.)
__device__ __forceinline__ bool preloaded_segment(const GemmParams& p, int span, int sb, int se, int tile_first, int tile_end, int seg_end) {
  return seg_end == se && se < tile_end && sb <= tile_first && p.span_begin[span + 2] >= tile_end;
}

// ===================== MMA issuer (warp 1 of the leader CTA) =====================
template <int MODE>
__device__ __forceinline__ void mma_issuer(const GemmParams& p, const Ctx& cx, int span) {
  const bool issuer = elect_one();
  const int S = cx.S;
  const uint32_t idesc_d = (1u << 4) | ((uint32_t)(p.n_pad >> 3) << 17) | ((256u >> 4) << 24);
  const uint32_t idesc_s = idesc_d | (1u << 2);
  const int sb = p.span_begin[span], se = p.span_begin[span + 1];
  unsigned long long off;
  Cursor c = cursor_at<MODE>(p, sb, &off);
  const uint32_t hi_sw = desc_hi(1024, kLayoutSW128), hi_meta = desc_hi(128, kLayoutNone);
  const uint32_t a_lo0 = desc_lo(cx.smem_base, 16), slot16 = cx.slot_bytes >> 4, bh16 = cx.b_half_bytes >> 4;
  uint32_t a_lo = a_lo0;                                    // operand of the current slot; tokens at + kSparseOperandBytes
  int slot = 0, seg = 0;
  uint32_t ph = 0, it = 0;
  uint32_t fb = cx.full_bar(0), eb = cx.empty_bar(0);
  long long t_full = 0, t_acce = 0;
#pragma unroll 1
  for (int s = sb; s < se; ++seg) {
    const int tile_end = c.first + c.ns + c.nd;
    const int seg_end = min(se, tile_end);
    const int buf = p.num_acc_bufs == 2 ? seg & 1 : 0;
    const uint32_t use = (uint32_t)(p.num_acc_bufs == 2 ? seg >> 1 : seg);
    long long tw0 = tracing(p) ? globaltimer() : 0;
    wait_bar(p, cx.acce_bar(buf), (use & 1u) ^ 1u);        // both CTAs' epilogues have drained this accumulator
    const bool pre = preloaded_segment(p, span, sb, se, c.first, tile_end, seg_end);
    if (pre) wait_bar(p, cx.pre_bar(), 0);                 // both CTAs have stored the partner's partial into this accumulator
    if (tracing(p)) t_acce += globaltimer() - tw0;
    tc_fence_after();
    const uint32_t d = cx.tmem_base + (uint32_t)(buf * p.acc_stride);
    uint32_t acc = pre ? 1u : 0u;
#pragma unroll 1
    for (; s < seg_end; ++s, ++it, ++c.j) {
      if (tracing(p)) tw0 = globaltimer();
      wait_bar(p, fb, ph);
      if (tracing(p)) t_full += globaltimer() - tw0;
      tc_fence_after();
      if (s == sb) trace(p, span, 3);
      const uint32_t b_lo = a_lo + (kSparseOperandBytes >> 4);
#ifdef SPENSE_DEBUG_HOOKS
      if (issuer && !(p.dbg & 2)) {              // experiment: stream the stages without issuing the MMAs
#else
      if (issuer) {
#endif
        if (c.j < c.ns) {
          const uint32_t e_base = cx.tmem_base + kMetaCol + (it & 1u) * 8u;
          const uint32_t m_lo = (a_lo & 0x3FFFu) + (kOperandBytes >> 4);     // metadata atoms: LBO 0
          tc_cp_128x128b_pair(e_base, desc_of(m_lo, hi_meta));
          tc_cp_128x128b_pair(e_base + 4u, desc_of(m_lo + (2048u >> 4), hi_meta));
#pragma unroll
          for (uint32_t k = 0; k < 4; ++k) {              // 4 sparse MMAs of K = 64 logical (32 B of A, 64 B of B)
            mma_f8_sparse_pair(d, desc_of(a_lo + 2u * k, hi_sw), desc_of(b_lo + (k >> 1) * bh16 + (k & 1u) * 4u, hi_sw), e_base + 2u * k,
                               idesc_s, acc | k);
          }
        } else {
#pragma unroll
          for (uint32_t k = 0; k < 4; ++k)                // 4 dense MMAs of K = 32
            mma_f8_dense_pair(d, desc_of(a_lo + 2u * k, hi_sw), desc_of(b_lo + 2u * k, hi_sw), idesc_d, acc | k);
        }
      }
      acc = 1;
      if (issuer) tc_commit_pair(eb, 3);                  // both CTAs' slots are free once these MMAs have read them
      if (++slot == S) { slot = 0; ph ^= 1u; a_lo = a_lo0; fb = cx.full_bar(0); eb = cx.empty_bar(0); }
      else { a_lo += slot16; fb += 8u; eb += 8u; }
    }
    if (issuer) tc_commit_pair(cx.accf_bar(buf), 3);      // accumulator complete in both CTAs
    if (s == tile_end) next_tile<MODE>(p, c);
  }
  trace(p, span, 4);
  if (tracing(p) && cx.blk == p.blk0 && issuer) { p.trace[(size_t)span * 16 + 11] = t_full; p.trace[(size_t)span * 16 + 12] = t_acce; }
}

// scale tables of the pair's token block (weight scales come from the blob header, on the device)
__device__ __forceinline__ void epilogue_tables(const GemmParams& p, const Ctx& cx, int et, int m_base, int Mb) {
  if (et < p.n_pad) {
    const int m = m_base + (et < Mb ? et : Mb - 1);
    const float w0 = __ldg(&p.hdr->w_scale[p.scale0]);
    if (p.mode == 0) {
      const float w1 = __ldg(&p.hdr->w_scale[p.scale1]);
      const float sx = __ldg(p.s_act + m);
      const float sh = p.amax_part ? 1.0f : __ldg(p.s_h + (size_t)m * p.sh_stride);
      cx.sc0()[et] = make_float4(sx * w0, sx * w1, p.amax_part ? 0.0f : sh, __frcp_rn(sh));
    } else {
      cx.sc1(p.n_pad)[et] = __ldg(p.s_act + (size_t)m * p.sh_stride) * w0;
    }
  }
}

// ===================== epilogue (16 warps per CTA, the CTA's own 128 lanes) =====================
template <int MODE, bool DYN>
__device__ __forceinline__ void epilogue(const GemmParams& p, const Ctx& cx, int span, int epoch) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int q = warp & 3;
  const int et = threadIdx.x - 128;
  const int m_base = cx.blk * p.n_pad;
  const int Mb = min(p.n_pad, p.M - m_base);
  const int cols_used = min(p.n_pad, (Mb + 7) & ~7);
  const int cols_per = (((p.n_pad + 3) >> 2) + 7) & ~7;
  const int c_begin = ((warp - 4) >> 2) * cols_per;
  const int c_end = min(c_begin + cols_per, cols_used);
  const float* stg = reinterpret_cast<const float*>(cx.smem_gen);   // the idle stage ring stages the reduce-scatter slices
  const size_t part_floats = (size_t)p.n_pad * 128;        // one partial: [col][lane]
  const int sb = p.span_begin[span], se = p.span_begin[span + 1];
  float4* const sc4 = cx.sc0();
  const float* const sc1 = cx.sc1(p.n_pad);
  const uint32_t lead_acce0 = mapa_shared(cx.acce_bar(0), 0);
  const int rank = (int)cx.rank;
  uint32_t red_round = 0;
  auto flag_of = [&](int s, int which) { return p.flags + (cx.slot0 + 2 * s) * 2 + which; };
  auto part_of = [&](int s, int which) { return p.partials + ((size_t)(cx.slot0 + 2 * s) * 2 + which) * part_floats; };

  Group groups[2];
  int n_groups = 0;
  unsigned long long off;
  Cursor cur = cursor_at<MODE>(p, sb, &off);
  // Does the span end with a preloaded segment, and when is its accumulator preloaded?  As early as its buffer is free (after
  // the epilogue of the segment num_acc_bufs before it), but never before this span's own dump (segment 0, if the span
  // starts inside a tile) is published: a span must not make its partner wait for ITS partner.
  int pre_seg = -1, pre_at = -1;
  {
    Cursor w = cur;
    int n_seg = 0, last_first = 0, last_end = 0;
    for (int s = sb; s < se; ++n_seg) {
      last_first = w.first; last_end = w.first + w.ns + w.nd;
      s = min(se, last_end);
      if (s == last_end) next_tile<MODE>(p, w);
    }
    if (preloaded_segment(p, span, sb, se, last_first, last_end, se)) {
      pre_seg = n_seg - 1;
      pre_at = pre_seg >= p.num_acc_bufs ? pre_seg - p.num_acc_bufs + 1 : ((sb > cur.first && pre_seg >= 1) ? 1 : 0);
    }
  }
  int seg = 0;
#pragma unroll 1
  for (int s = sb; s < se; ++seg) {
    const int tile_end = cur.first + cur.ns + cur.nd;
    const int seg_end = min(se, tile_end);
    const int buf = p.num_acc_bufs == 2 ? seg & 1 : 0;
    const uint32_t use = (uint32_t)(p.num_acc_bufs == 2 ? seg >> 1 : seg);
    int a = span, b = span;
    while (p.span_begin[a] > cur.first) --a;
    while (b + 1 < p.n_spans && p.span_begin[b + 1] < tile_end) ++b;

    if (seg == pre_at) {
      // partner's partial [col][lane] of this CTA's operand -> the accumulator of segment pre_seg
      wait_flag(p, flag_of(span + 1, 0), epoch);
      if (et == 0) trace(p, span, 8);
      const float* po = part_of(span + 1, 0) + 32 * q + lane;
      const uint32_t tp = cx.tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)((p.num_acc_bufs == 2 ? pre_seg & 1 : 0) * p.acc_stride);
#pragma unroll 2
      for (int c = c_begin; c < c_end; c += 8) {
        uint32_t v[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] = __float_as_uint(__ldcg(po + (size_t)(c + i) * 128));
        tmem_st8(tp + (uint32_t)c, v);
      }
      tmem_st_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(mapa_shared(cx.pre_bar(), 0));
    }

    wait_bar(p, cx.accf_bar(buf), use & 1u);
    tc_fence_after();
    if (et == 0) trace(p, span, seg == 0 ? 5 : 7);
    const uint32_t t0 = cx.tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * p.acc_stride);

    if (a == b || (b == a + 1 && span == a)) {
      // the whole tile is ours, or we own a tile whose tail the next span has (usually long ago) dumped
      const float* part = nullptr;                         // (a != b: the partner's partial is already in the accumulator)
      int c = c_begin;
      if (part == nullptr) {
#pragma unroll 1
        for (; c + 32 <= c_end; c += 32) tile_block<MODE, DYN, 4>(p, sc4, sc1, t0, part, cur.tile, rank, q, lane, c, Mb, m_base);
      }
#pragma unroll 1
      for (; c + 16 <= c_end; c += 16) tile_block<MODE, DYN, 2>(p, sc4, sc1, t0, part, cur.tile, rank, q, lane, c, Mb, m_base);
      if (c < c_end) tile_block<MODE, DYN, 1>(p, sc4, sc1, t0, part, cur.tile, rank, q, lane, c, Mb, m_base);
    } else {
      // split tile, not (solely) ours to finish: dump the raw fp32 partial [col][lane] and publish it
      const int which = (sb >= cur.first) ? 0 : 1;
      float* slot = part_of(span, which);
#pragma unroll 1
      for (int c = c_begin; c < c_end; c += 8) {
        uint32_t v0[8];
        tmem_ld8(t0 + c, v0);
        tmem_ld_wait();
#pragma unroll
        for (int i = 0; i < 8; ++i) __stcg(slot + (size_t)(c + i) * 128 + 32 * q + lane, __uint_as_float(v0[i]));
      }
      epi_sync();                                          // all partial stores issued (CTA scope) ...
      if (et == 0) st_release(flag_of(span, which), epoch);   // ... one gpu-scope release publishes them (cumulativity)
      if (b > a + 1) {
        groups[n_groups].a = a; groups[n_groups].b = b; groups[n_groups].tile = cur.tile; groups[n_groups].first = cur.first;
        ++n_groups;
      }
    }
    // this CTA's warps are done with the accumulator: one arrival per warp on the LEADER's barrier
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive_cluster(lead_acce0 + 8u * (uint32_t)buf);
    if (et == 0) trace(p, span, 6);
    s = seg_end;
    if (s == tile_end) next_tile<MODE>(p, cur);
  }

  // ---- deferred reduce-scatter of tiles shared by > 2 spans: span j of the group reduces token columns
  // [j*M/n, (j+1)*M/n), adding the n partials in span order, and runs the epilogue on them.  All MMAs of this CTA are
  // complete: the idle stage ring stages the partial slices.
#pragma unroll 1
  for (int gi = 0; gi < n_groups; ++gi) {
    const Group g = groups[gi];
    const int n = g.b - g.a + 1;
    const int j = span - g.a;
    const int m0 = (int)(((long long)j * Mb) / n), m1 = (int)(((long long)(j + 1) * Mb) / n);
    const int rrow = et & 127;
    if (m1 > m0) {
      int cc_max = (int)(cx.ring_bytes / ((uint32_t)n * 512u));
      if (cc_max > m1 - m0) cc_max = m1 - m0;
#pragma unroll 1
      for (int mc = m0; mc < m1; mc += cc_max) {
        const int cc = min(cc_max, m1 - mc);
        if (red_round > 0) {
          fence_proxy_async();
          epi_sync();
        }
        if (et == 0) mbar_expect_tx(cx.red_bar(), (uint32_t)n * (uint32_t)cc * 512u);
#pragma unroll 1
        for (int i = et; i < n; i += kEpiThreads) {
          const int qs = g.a + i;
          const int which = (p.span_begin[qs] >= g.first) ? 0 : 1;
          wait_flag(p, flag_of(qs, which), epoch);
          asm volatile("fence.proxy.async.global;" ::: "memory");
          bulk_g2s(cx.smem_base + (uint32_t)(i * cc) * 512u, part_of(qs, which) + (size_t)mc * 128, (uint32_t)cc * 512u, cx.red_bar(),
                   policy_evict_first());
        }
        wait_bar(p, cx.red_bar(), red_round & 1u);
        ++red_round;
        if (et == 0) trace(p, span, 15);
        if (MODE == 0) {
          // threads 0..63 of each 128-thread column group finish one intermediate index each (gate lane, up lane)
          const int j64 = rrow & 63;
          const int lane_g = glu_gate_lane_of_index(j64);
          const int first = lane_g ^ (lane & 16);
#pragma unroll 1
          for (int c = (et >> 6); c < cc; c += kEpiThreads >> 6) {
            float x = 0.0f, y = 0.0f;
#pragma unroll 4
            for (int qi = 0; qi < n; ++qi) {               // fixed span order: deterministic
              const float* img = stg + ((size_t)qi * cc + c) * 128;
              x += img[first];
              y += img[first ^ 16];
            }
            const float ah = finish_glu<DYN>(p, sc4, g.tile, 64 * rank + j64, mc + c, m_base + mc + c, (lane & 16) ? y : x, (lane & 16) ? x : y);
            if (DYN) {
              const int mx = __reduce_max_sync(0xffffffffu, __float_as_int(ah));
              if (lane == 0) atomicMax(reinterpret_cast<int*>(sc4 + mc + c) + 2, mx);
            }
          }
        } else {
#pragma unroll 1
          for (int c = et >> 7; c < cc; c += kEpiThreads >> 7) {
            float f0 = 0.0f;
#pragma unroll 4
            for (int qi = 0; qi < n; ++qi) f0 += stg[((size_t)qi * cc + c) * 128 + rrow];
            store_y(p, g.tile * 256 + 128 * rank + rrow, m_base + mc + c, f0 * sc1[mc + c]);
          }
        }
      }
    }
    if (et == 0) trace(p, span, 9);
  }
}

}  // namespace

// ------------------------------------------------------------------------------------------ the kernel
template <int MODE, bool DYN>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(kThreads, 1)
spense_gemm_kernel(const __grid_constant__ GemmParams p, const __grid_constant__ CUtensorMap tmap_b,
                        const __grid_constant__ CUtensorMap tmap_ws, const __grid_constant__ CUtensorMap tmap_wd) {
  extern __shared__ uint8_t smem_raw[];
  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  if (warp == 0 && lane == 0) { prefetch_tmap(&tmap_b); prefetch_tmap(&tmap_ws); prefetch_tmap(&tmap_wd); }
  Ctx cx;
  {
    const uint32_t raw = smem_u32(smem_raw);
    cx.smem_base = (raw + 1023u) & ~1023u;
    cx.smem_gen = smem_raw + (cx.smem_base - raw);
    cx.S = p.num_stages;
    cx.slot_bytes = (uint32_t)p.slot_bytes;
    cx.ring_bytes = (uint32_t)cx.S * cx.slot_bytes;
    cx.bar_base = cx.smem_base + cx.ring_bytes;
    cx.b_half_bytes = (uint32_t)(p.n_pad >> 1) * 128u;
    cx.rank = cluster_ctarank();
  }
  // pair b / 2 works on token block blk0 + pair / n_spans, span n_spans - 1 - pair % n_spans of the SAME schedule
  const int pair = (int)blockIdx.x >> 1;
  const int bp = pair / p.n_spans;
  const int span = p.n_spans - 1 - (pair - bp * p.n_spans);
  cx.blk = p.blk0 + bp;
  cx.slot0 = bp * p.n_spans * 2 + (int)cx.rank;
  if (warp == 0 && lane == 0) {
    for (int s = 0; s < cx.S; ++s) { mbar_init(cx.full_bar(s), 1); mbar_init(cx.empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(cx.accf_bar(b), 1); mbar_init(cx.acce_bar(b), 2 * kEpiWarps); }
    mbar_init(cx.red_bar(), 1);
    mbar_init(cx.pre_bar(), 2 * kEpiWarps);
    *cx.epi_done_ptr() = 0;
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc_pair(cx.tmem_slot(), kTmemCols);
  tc_fence_before();
  cluster_sync_all();                                      // barriers and TMEM of BOTH CTAs exist before anyone signals or writes them
  tc_fence_after();
  cx.tmem_base = *cx.tmem_slot_ptr();
  pdl_launch_dependents();
  if (tracing(p) && threadIdx.x == 0 && bp == 0 && cx.rank == 0) {
    uint32_t smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    p.trace[(size_t)span * 16 + 0] = globaltimer(); p.trace[(size_t)span * 16 + 14] = smid;
  }

  if (warp == 0) {
    producer_weights<MODE>(p, &tmap_ws, &tmap_wd, cx, span);
    trace(p, span, 2);
    if (lane == 0) prefetch_next(p, cx, span);
  } else if (warp == 3) {
    producer_tokens<MODE>(p, &tmap_b, cx, span);
  } else if (warp == 1) {
    if (cx.rank == 0) mma_issuer<MODE>(p, cx, span);
  } else if (warp >= 4) {
    const int et = threadIdx.x - 128;
    pdl_wait();
    epilogue_tables(p, cx, et, cx.blk * p.n_pad, min(p.n_pad, p.M - cx.blk * p.n_pad));
    if (et == kEpiThreads - 1) {
      check_header(p);
      take_epoch(p.ws_ctrl, (int)gridDim.x, cx.epoch_ptr());
    }
    epi_sync();
    const int epoch = cx.epoch_ptr()[0];
    epilogue<MODE, DYN>(p, cx, span, epoch);
    if (DYN) {                        // this CTA's max|h| per token column of its block, for the row requant kernel
      epi_sync();
      const int Mb = min(p.n_pad, p.M - cx.blk * p.n_pad);
      if (et < p.n_pad) p.amax_part[(size_t)(cx.slot0 + 2 * span) * p.n_pad + et] = et < Mb ? cx.sc0()[et].z : 0.0f;
    }
    if (et == 0) *cx.epi_done_ptr() = 1;
    if (tracing(p) && et == 0 && bp == 0 && cx.rank == 0) p.trace[(size_t)span * 16 + 10] = globaltimer();
  }

  tc_fence_before();
  cluster_sync_all();                                      // the peer's MMAs read our ring, its epilogue arrives on our barriers
  if (warp == 2) { tc_fence_after(); tmem_dealloc_pair(cx.tmem_base, kTmemCols); }
}

namespace {
size_t smem_bytes_of(const GemmParams& p) { return (size_t)p.num_stages * p.slot_bytes + 1024 + 256 + 20 * (size_t)p.n_pad; }

// per device and kernel instance, once: opt in to the shared memory; how many CTA pairs can be resident at once
template <typename K>
int prepare(K kernel, int which, int dev, int grid) {
  static std::mutex mu;
  static bool ready[4][64] = {};
  static int resident[4][64] = {};
  std::lock_guard<std::mutex> lk(mu);
  if (dev < 0 || dev >= 64) return SPENSE_ERR_CUDA;
  if (!ready[which][dev]) {
    if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemMax) != cudaSuccess) return SPENSE_ERR_CUDA;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(2);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = kSmemMax;
    int clusters = 0;
    if (cudaOccupancyMaxActiveClusters(&clusters, kernel, &cfg) != cudaSuccess) return SPENSE_ERR_CUDA;
    resident[which][dev] = 2 * clusters;
    ready[which][dev] = true;
  }
  return grid <= resident[which][dev] ? SPENSE_OK : SPENSE_ERR_CUDA;
}
}  // namespace

// the once-per-device work of every kernel instance, done ahead of the first launch (spense_workspace_init): the first GEMM
// call then only launches, which is what lets it sit inside a stream capture in a process that never packed a blob
int prepare_gemm_kernels(int dev) {
  int st = prepare(spense_gemm_kernel<0, false>, 0, dev, 0);
  if (!st) st = prepare(spense_gemm_kernel<0, true>, 1, dev, 0);
  if (!st) st = prepare(spense_gemm_kernel<1, false>, 2, dev, 0);
  if (!st) st = prepare(spense_gemm_kernel<2, false>, 3, dev, 0);
  return st;
}

int launch_gemm(const GemmParams& p, const CUtensorMap& tmap_b, const CUtensorMap& tmap_ws, const CUtensorMap& tmap_wd, bool pdl, int dev,
                cudaStream_t stream) {
  const int grid = 2 * p.n_spans * p.nb;
  int st = p.mode == 2     ? prepare(spense_gemm_kernel<2, false>, 3, dev, grid)
           : p.mode == 1   ? prepare(spense_gemm_kernel<1, false>, 2, dev, grid)
           : p.amax_part ? prepare(spense_gemm_kernel<0, true>, 1, dev, grid)
                         : prepare(spense_gemm_kernel<0, false>, 0, dev, grid);
  if (st) return st;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid);
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = smem_bytes_of(p);
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  const cudaError_t e = p.mode == 2     ? cudaLaunchKernelEx(&cfg, spense_gemm_kernel<2, false>, p, tmap_b, tmap_ws, tmap_wd)
                        : p.mode == 1   ? cudaLaunchKernelEx(&cfg, spense_gemm_kernel<1, false>, p, tmap_b, tmap_ws, tmap_wd)
                        : p.amax_part ? cudaLaunchKernelEx(&cfg, spense_gemm_kernel<0, true>, p, tmap_b, tmap_ws, tmap_wd)
                                      : cudaLaunchKernelEx(&cfg, spense_gemm_kernel<0, false>, p, tmap_b, tmap_ws, tmap_wd);
  return e == cudaSuccess ? SPENSE_OK : SPENSE_ERR_CUDA;
}

}  // namespace spense
