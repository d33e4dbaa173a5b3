// Spense hybrid sparse-dense FP8 GEMM for sm_100a (tcgen05 + TMEM + TMA / bulk copy): the DECODE kernel, up to
// kDecodeMaxTokens (112) tokens.  More tokens run on CTA pairs (spense_gemm_wide.cu).
//
// Two GEMMs, written once as per-role device functions:
//   MODE 0  gate_up : output-split.  Pair tile = 2 operands of 128 rows = the gate and up rows of 128
//                     intermediate indices (interleaved, see spense_internal.cuh); tiles below I_s are 2:4 compressed
//                     (tcgen05.mma.sp), the rest dense (tcgen05.mma).  Epilogue: scales -> SiLU(g)*u (Eq. 4,
//                     PAPER.md:141) -> E4M3.
//   MODE 1  down    : input-split.  Pair tile = 2 x 128 rows of W_down; the K loop runs
//                     the sparse stages and then the dense stages INTO THE SAME TMEM ACCUMULATOR.
// spense_gemm_kernel<MODE, DYN>: DYN = gate_up that keeps h in fp32 and tracks max|h| per token (dynamic requant).
//
// Swap-AB: only the A operand of tcgen05.mma.sp can be sparse, so weights are A (MMA-M = 128 weight
// rows) and tokens are B (MMA-N = padded token count); the accumulator holds Y^T [128 rows x tokens].
//
// Decode is weight-streaming bound, so the grid is a cost-balanced stream-K: the linear sequence of
// stage images (= the byte order of the blob) is cut into n_spans spans, one persistent CTA per span.
// A tile whose stages fall into several spans is fixed up through an L2-resident fp32 workspace, always
// adding the partials in span order, so results are bitwise reproducible:
//   * 2 spans  : the second span finishes its part early (it is its first segment), dumps it and
//                publishes a flag; the first span (owner) stages it through its idle ring, adds it to its TMEM
//                accumulator and runs the epilogue;
//   * > 2 spans: every span finishes late, so all dump, and the n spans reduce M/n token columns each
//                (reduce-scatter) instead of one owner reducing n partials serially.
// Flags hold the epoch of the launch (a device-side counter in the workspace), so nothing has to be
// reset between launches and CUDA-graph replays see fresh values.
// Span i runs on CTA n_spans-1-i.  CTAs of one launch wait for each other, so all n_spans <= #SM CTAs
// must be co-resident: 1 CTA/SM by construction (shared memory); the host checks the occupancy the device offers
// and every wait is bounded (spense_gemm_common.cuh).
//
// Warp roles (640 threads): warp 0 producer (bulk copy of the weight stage + TMA of the activation
// tile), warp 1 MMA issuer, warp 2 TMEM allocator, warps 4-19 epilogue (TMEM lane quadrant = warp & 3,
// quarter of the token columns = (warp - 4) >> 2): the last tile's epilogue is exposed at the end of
// every CTA and is instruction-issue bound, so it gets 4 warps per scheduler.  Rarely executed code is
// kept rolled: the kernel is latency-sensitive at its tail and instruction-cache misses on cold paths
// showed up in the timeline.
#include <mutex>

#include "spense_gemm_common.cuh"

namespace spense {

namespace {

using namespace dev;

__device__ __forceinline__ void epi_sync() { asm volatile("bar.sync 1, 512;" ::: "memory"); }   // the 16 epilogue warps

constexpr int kEpiThreads = 512;                 // 16 epilogue warps: 4 per TMEM lane quadrant
constexpr int kThreads = 128 + kEpiThreads;
constexpr int kTmemCols = 512;
constexpr int kMetaCol = 480;   // 2 buffers x 16 columns of 2:4 metadata

// Shared memory after the stage ring: 256 B of barriers and words, then the scale tables of the two modes.
struct Ctx {
  uint32_t smem_base;          // 1 KB aligned start of the stage ring (shared address)
  uint8_t* smem_gen;           // the same, generic
  int S;                       // ring slots
  uint32_t slot_bytes, ring_bytes, bar_base, b_tile_bytes, tmem_base;
  __device__ __forceinline__ uint32_t full_bar(int s) const { return bar_base + 8u * s; }
  __device__ __forceinline__ uint32_t empty_bar(int s) const { return bar_base + 8u * (8 + s); }
  __device__ __forceinline__ uint32_t accf_bar(int b) const { return bar_base + 8u * (16 + b); }
  __device__ __forceinline__ uint32_t acce_bar(int b) const { return bar_base + 8u * (18 + b); }
  __device__ __forceinline__ uint32_t tmem_slot() const { return bar_base + 8u * 20; }
  __device__ __forceinline__ uint32_t red_bar() const { return bar_base + 8u * 22; }
  __device__ __forceinline__ volatile uint32_t* tmem_slot_ptr() const { return reinterpret_cast<volatile uint32_t*>(smem_gen + ring_bytes + 8 * 20); }
  __device__ __forceinline__ volatile int* epoch_ptr() const { return reinterpret_cast<volatile int*>(smem_gen + ring_bytes + 8 * 21); }
  __device__ __forceinline__ volatile int* epi_done_ptr() const { return reinterpret_cast<volatile int*>(smem_gen + ring_bytes + 8 * 23); }
  __device__ __forceinline__ float4* sc0() const { return reinterpret_cast<float4*>(smem_gen + ring_bytes + 256); }
  __device__ __forceinline__ float* sc1(int n_pad) const { return reinterpret_cast<float*>(smem_gen + ring_bytes + 256 + 16 * n_pad); }
};

// A tile shared by more than two spans [a, b]: reduced at the end of the kernel (reduce-scatter).
struct Group { int a, b, tile, first; };

// ===================== producer (one thread) =====================
// Streams the stages of span `span` through the ring.  A weight stage depends on nothing and is issued as soon as its
// slot is free; the activation tiles wait for the previous kernel of the stream (one griddepcontrol.wait, when the ring
// is full of weights).
template <int MODE>
__device__ __forceinline__ void producer(const GemmParams& p, const CUtensorMap* tmap, const Ctx& cx, int span) {
  const int S = cx.S;
  const int sb = p.span_begin[span];
  const int n = p.span_begin[span + 1] - sb;
  const uint64_t pol_w = policy_evict_first();             // a weight byte is used once
  const uint64_t pol_a = policy_evict_last();
  unsigned long long off;
  Cursor c = cursor_at<MODE>(p, sb, &off);
  const uint8_t* src = p.section + off;
  uint32_t info[8];                                        // stages whose weights are in flight: K coordinate | sparse << 31

  auto load_b = [&](int slot, uint32_t inf) {
    const uint32_t b_dst = cx.smem_base + (uint32_t)slot * cx.slot_bytes + kSparseStageBytes;
    const int k0 = (int)(inf & 0x7FFFFFFFu);                // K coordinate | sparse << 31
    tma_load_2d(b_dst, tmap, k0, 0, cx.full_bar(slot), pol_a);
    if (inf >> 31) tma_load_2d(b_dst + cx.b_tile_bytes, tmap, k0 + 128, 0, cx.full_bar(slot), pol_a);
  };

  int w = 0;                                               // weight stages issued
  uint32_t inf_last = 0;                                   // descriptor of the stage issued last (steady state: no table)
  int w_slot = 0, w_round = 0, b_slot = 0;                 // ring positions, kept incrementally (no divisions per stage)
  auto issue_weight = [&](bool blocking) -> bool {
    // everything that does not need the slot is computed before the wait: a freed slot is refilled at once
    const bool sp = c.j < c.ns;
    const uint32_t wb = sp ? (uint32_t)kSparseStageBytes : (uint32_t)kDenseStageBytes;
    const uint32_t inf = (uint32_t)(sp ? c.j * kSparseStageK : p.dense_k0 + (c.j - c.ns) * kDenseStageK) | (sp ? 0x80000000u : 0u);
    const uint32_t tx = wb + (sp ? 2u : 1u) * cx.b_tile_bytes;
    const uint32_t fb = cx.full_bar(w_slot);
    const uint32_t dst = cx.smem_base + (uint32_t)w_slot * cx.slot_bytes;
    if (w_round > 0) {
      const uint32_t par = ((uint32_t)w_round & 1u) ^ 1u;
      if (blocking) wait_bar(p, cx.empty_bar(w_slot), par);
      else if (!mbar_try(cx.empty_bar(w_slot), par)) return false;
    }
    mbar_expect_tx(fb, tx);
    bulk_g2s(dst, src, wb, fb, pol_w);
    inf_last = inf;
    if (!blocking) {                                       // running ahead of the activation tiles: remember it
#pragma unroll
      for (int k = 0; k < 8; ++k)
        if (k == (w & 7)) info[k] = inf;
    }
    src += wb;
    if (++c.j == c.ns + c.nd) next_tile<MODE>(p, c);
    ++w;
    if (++w_slot == S) { w_slot = 0; ++w_round; }
    return true;
  };

  // Weights never depend on the previous kernel of the stream, activations do: fill the whole ring with weight
  // stages, pull a little more of this span into L2, then wait for the previous kernel.
#pragma unroll 1
  while (w < n && w < S && issue_weight(false)) {}
  trace(p, span, 1);
  if (p.self_len[span]) {
    const uint8_t* pf = src + p.self_off[span];
#pragma unroll 1
    for (uint32_t o = 0; o < p.self_len[span]; o += 32768u) {
      const uint32_t chunk = p.self_len[span] - o < 32768u ? p.self_len[span] - o : 32768u;
      asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(pf + o), "r"(chunk) : "memory");
    }
  }
  pdl_wait();
#pragma unroll 1
  for (int b = 0; b < n; ++b) {
    uint32_t inf = 0;
    if (w <= b) {
      issue_weight(true);
      inf = inf_last;
    } else {
#pragma unroll
      for (int k = 0; k < 8; ++k)
        if (k == (b & 7)) inf = info[k];
    }
    load_b(b_slot, inf);
    if (++b_slot == S) b_slot = 0;
  }
}

// L2 prefetch of what the NEXT kernel of the stream streams first, issued while this CTA runs its fix-up tail:
// one 32 KB chunk per pf_pace_ns so the fix-up traffic is not queued behind it; stops with the epilogue.
__device__ __forceinline__ void prefetch_next(const GemmParams& p, const Ctx& cx, int span) {
  if (!p.next_base) return;
  const uint8_t* nb = p.next_base + (size_t)p.next_off[span];
  const uint32_t bytes = p.next_len[span];
  long long t_next = globaltimer();
#pragma unroll 1
  for (uint32_t o = 0; o < bytes && (p.pf_pace_ns == 0 || *cx.epi_done_ptr() == 0); o += 32768u) {
    const uint32_t chunk = bytes - o < 32768u ? bytes - o : 32768u;
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(nb + o), "r"(chunk) : "memory");
    if (p.pf_pace_ns) {
      t_next += p.pf_pace_ns;
      while (globaltimer() < t_next && *cx.epi_done_ptr() == 0) __nanosleep(64);
    }
  }
}

// ===================== MMA issuer (one thread) =====================
template <int MODE>
__device__ __forceinline__ void mma_issuer(const GemmParams& p, const Ctx& cx, int span) {
  const int S = cx.S;
  const uint32_t idesc_d = (1u << 4) | ((uint32_t)(p.n_pad >> 3) << 17) | ((128u >> 4) << 24);
  const uint32_t idesc_s = idesc_d | (1u << 2);
  const int sb = p.span_begin[span], se = p.span_begin[span + 1];
  unsigned long long off;
  Cursor c = cursor_at<MODE>(p, sb, &off);
  int slot = 0, it = 0, seg = 0;
  uint32_t ph = 0;
#pragma unroll 1
  for (int s = sb; s < se; ++seg) {
    const int tile_end = c.first + c.ns + c.nd;
    const int seg_end = min(se, tile_end);
    const int buf = seg % p.num_acc_bufs;
    const uint32_t use = (uint32_t)(seg / p.num_acc_bufs);
    wait_bar(p, cx.acce_bar(buf), (use & 1u) ^ 1u);          // epilogue has drained this accumulator
    tc_fence_after();
    const uint32_t d0 = cx.tmem_base + (uint32_t)(buf * 2 * p.acc_stride);
    const uint32_t d1 = d0 + (uint32_t)p.acc_stride;
    uint32_t acc = 0;
#pragma unroll 1
    for (; s < seg_end; ++s, ++it, ++c.j) {
      wait_bar(p, cx.full_bar(slot), ph);
      tc_fence_after();
      if (s == sb) trace(p, span, 3);
      const uint32_t a0 = cx.smem_base + (uint32_t)slot * cx.slot_bytes;
      const uint32_t b0 = a0 + kSparseStageBytes;
      if (c.j < c.ns) {
        const uint32_t a1 = a0 + kSparseOperandBytes;     // A0 vals | A0 meta | A1 vals | A1 meta
        const uint32_t e_base = cx.tmem_base + kMetaCol + (uint32_t)(it & 1) * 16u;
#pragma unroll
        for (int a = 0; a < 4; ++a)                       // 4 atoms of 2 KB: (A0,k0) (A0,k1) (A1,k0) (A1,k1)
          tc_cp_128x128b(e_base + 4u * a, make_desc((a < 2 ? a0 : a1) + kOperandBytes + 2048u * (a & 1), 0, 128, kLayoutNone));
#pragma unroll
        for (int k = 0; k < 4; ++k) {                     // 4 sparse MMAs of K = 64 logical (32 B of A, 64 B of B)
          const uint64_t bd = make_desc(b0 + (uint32_t)(k >> 1) * cx.b_tile_bytes + (uint32_t)(k & 1) * 64u, 16, 1024, kLayoutSW128);
          mma_f8_sparse(d0, make_desc(a0 + 32u * k, 16, 1024, kLayoutSW128), bd, e_base + 2u * k, idesc_s, acc);
          mma_f8_sparse(d1, make_desc(a1 + 32u * k, 16, 1024, kLayoutSW128), bd, e_base + 8u + 2u * k, idesc_s, acc);
          acc = 1;
        }
      } else {
        const uint32_t a1 = a0 + kOperandBytes;
#pragma unroll
        for (int k = 0; k < 4; ++k) {                     // 4 dense MMAs of K = 32
          const uint64_t bd = make_desc(b0 + 32u * k, 16, 1024, kLayoutSW128);
          mma_f8_dense(d0, make_desc(a0 + 32u * k, 16, 1024, kLayoutSW128), bd, idesc_d, acc);
          mma_f8_dense(d1, make_desc(a1 + 32u * k, 16, 1024, kLayoutSW128), bd, idesc_d, acc);
          acc = 1;
        }
      }
      tc_commit(cx.empty_bar(slot));                      // smem slot free once these MMAs have read it
      if (++slot == S) { slot = 0; ph ^= 1u; }
    }
    tc_commit(cx.accf_bar(buf));                          // accumulator complete for this segment
    if (s == tile_end) next_tile<MODE>(p, c);
  }
  trace(p, span, 4);
}

// scale tables of the launch's tokens (weight scales come from the blob header, on the device)
__device__ __forceinline__ void epilogue_tables(const GemmParams& p, const Ctx& cx, int et) {
  if (et < p.n_pad) {
    const int m = et < p.M ? et : p.M - 1;
    const float w0 = __ldg(&p.hdr->w_scale[p.scale0]);
    if (p.mode == 0) {
      const float w1 = __ldg(&p.hdr->w_scale[p.scale1]);
      const float sx = __ldg(p.s_act + m);
      const float sh = p.amax_part ? 1.0f : __ldg(p.s_h + (size_t)m * p.sh_stride);
      cx.sc0()[et] = make_float4(sx * w0, sx * w1, p.amax_part ? 0.0f : sh, __frcp_rn(sh));   // dynamic: .z = running max|h| bits
    } else {
      cx.sc1(p.n_pad)[et] = __ldg(p.s_act + (size_t)m * p.sh_stride) * w0;
    }
  }
}

// ===================== epilogue (16 warps) =====================
// warp & 3 selects the TMEM lane quadrant, (warp - 4) >> 2 the quarter of the token columns.  Once the CTA's last
// accumulator is complete the stage ring is idle and stages the partials (bulk copies).
template <int MODE, bool DYN>
__device__ __forceinline__ void epilogue(const GemmParams& p, const Ctx& cx, int span, int epoch) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int q = warp & 3;
  const int et = threadIdx.x - 128;                        // 0..511
  const int Mb = p.M;
  const int cols_used = min(p.n_pad, (Mb + 7) & ~7);       // token columns holding real tokens, rounded to the TMEM load width
  const int cols_per = (((p.n_pad + 3) >> 2) + 7) & ~7;    // columns per warp: a quarter, rounded to the TMEM load width
  const int c_begin = ((warp - 4) >> 2) * cols_per;
  const int c_end = min(c_begin + cols_per, cols_used);
  const float* stg = reinterpret_cast<const float*>(cx.smem_gen);   // the stage ring doubles as partial staging
  const size_t part_floats = (size_t)2 * p.n_pad * 128;    // one partial: [operand][col][lane]
  int* const flags = p.flags;
  float* const partials = p.partials;
  const int sb = p.span_begin[span], se = p.span_begin[span + 1];
  float4* const sc4 = cx.sc0();
  const float* const sc1 = cx.sc1(p.n_pad);
  uint32_t red_round = 0;

  Group groups[2];
  int n_groups = 0;
  unsigned long long off;
  Cursor cur = cursor_at<MODE>(p, sb, &off);
  int seg = 0;
#pragma unroll 1
  for (int s = sb; s < se; ++seg) {
    const int tile_end = cur.first + cur.ns + cur.nd;
    const int seg_end = min(se, tile_end);
    const int buf = seg % p.num_acc_bufs;
    const uint32_t use = (uint32_t)(seg / p.num_acc_bufs);
    // spans [a, b] that hold stages of this tile
    int a = span, b = span;
    while (p.span_begin[a] > cur.first) --a;
    while (b + 1 < p.n_spans && p.span_begin[b + 1] < tile_end) ++b;

    wait_bar(p, cx.accf_bar(buf), use & 1u);
    tc_fence_after();
    if (et == 0) trace(p, span, seg == 0 ? 5 : 7);
    const uint32_t t0 = cx.tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * 2 * p.acc_stride);
    const uint32_t t1 = t0 + (uint32_t)p.acc_stride;

    if (a == b || (b == a + 1 && span == a)) {
      // the whole tile is ours, or we own a tile whose tail the next span has (usually long ago) dumped
      const float* part = nullptr;
      if (a != b) {
        wait_flag(p, flags + b * 2, epoch);                // every thread: one ld.acquire when the partner is done (the usual case)
        part = partials + (size_t)b * 2 * part_floats;     // span b starts inside the tile: its first segment
        if (et == 0) trace(p, span, 8);
      }
      if (seg_end == se && n_groups == 0 && et == 0) *cx.epi_done_ptr() = 1;   // last epilogue of this CTA: stop prefetching now
#pragma unroll
      for (int opnd = 0; opnd < 2; ++opnd) {
        const uint32_t t_op = opnd ? t1 : t0;
        const float* part_op = part ? part + (size_t)opnd * p.n_pad * 128 : nullptr;
        int c = c_begin;
#pragma unroll 1
        for (; c + 16 <= c_end; c += 16) tile_block<MODE, DYN, 2>(p, sc4, sc1, t_op, part_op, cur.tile, opnd, q, lane, c, Mb, 0);
        if (c < c_end) tile_block<MODE, DYN, 1>(p, sc4, sc1, t_op, part_op, cur.tile, opnd, q, lane, c, Mb, 0);
      }
      tc_fence_before();
      mbar_arrive(cx.acce_bar(buf));
    } else {
      // split tile, not (solely) ours to finish: dump the raw fp32 partial [operand][col][lane] and publish it
      const int which = (sb >= cur.first) ? 0 : 1;         // our first segment, or our last one
      float* slot = partials + ((size_t)span * 2 + which) * part_floats;
#pragma unroll 1
      for (int c = c_begin; c < c_end; c += 8) {
        uint32_t v0[8], v1[8];
        tmem_ld8(t0 + c, v0);
        tmem_ld8(t1 + c, v1);
        tmem_ld_wait();
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          __stcg(slot + (size_t)(c + i) * 128 + 32 * q + lane, __uint_as_float(v0[i]));
          __stcg(slot + (size_t)(p.n_pad + c + i) * 128 + 32 * q + lane, __uint_as_float(v1[i]));
        }
      }
      tc_fence_before();
      mbar_arrive(cx.acce_bar(buf));
      epi_sync();                                          // all partial stores issued (CTA scope) ...
      if (et == 0) st_release(flags + span * 2 + which, epoch);   // ... one gpu-scope release publishes them (cumulativity)
      if (b > a + 1) {
        groups[n_groups].a = a; groups[n_groups].b = b; groups[n_groups].tile = cur.tile; groups[n_groups].first = cur.first;
        ++n_groups;
      }
    }
    if (et == 0) trace(p, span, 6);
    s = seg_end;
    if (s == tile_end) next_tile<MODE>(p, cur);
  }

  // ---- deferred reduce-scatter of tiles shared by > 2 spans: span j of the group reduces token columns
  // [j*M/n, (j+1)*M/n), adding the n partials in span order, and runs the epilogue on them.  All MMAs of this CTA are
  // complete: the stage ring stages the partial slices.
#pragma unroll 1
  for (int gi = 0; gi < n_groups; ++gi) {
    const Group g = groups[gi];
    const int n = g.b - g.a + 1;
    const int j = span - g.a;
    const int m0 = (int)(((long long)j * Mb) / n), m1 = (int)(((long long)(j + 1) * Mb) / n);
    const int rrow = et & 127;
    if (m1 > m0) {
      int cc_max = (int)(cx.ring_bytes / ((uint32_t)n * 1024u));
      if (cc_max > m1 - m0) cc_max = m1 - m0;
#pragma unroll 1
      for (int mc = m0; mc < m1; mc += cc_max) {
        const int cc = min(cc_max, m1 - mc);
        if (red_round > 0) {                               // staging smem is reused: order our reads before the async writes
          fence_proxy_async();
          epi_sync();
        }
        if (et == 0) mbar_expect_tx(cx.red_bar(), (uint32_t)n * 2u * (uint32_t)cc * 512u);
        // thread i fetches operand (i & 1) of partner (i >> 1) as soon as THAT partner has published
#pragma unroll 1
        for (int i = et; i < 2 * n; i += kEpiThreads) {
          const int qs = g.a + (i >> 1), mat = i & 1;
          const int which = (p.span_begin[qs] >= g.first) ? 0 : 1;
          wait_flag(p, flags + qs * 2 + which, epoch);
          asm volatile("fence.proxy.async.global;" ::: "memory");   // partner's generic-proxy stores -> our async-proxy read
          const float* src = partials + ((size_t)qs * 2 + which) * part_floats + ((size_t)mat * p.n_pad + mc) * 128;
          bulk_g2s(cx.smem_base + (uint32_t)(i * cc) * 512u, src, (uint32_t)cc * 512u, cx.red_bar(), policy_evict_first());
        }
        wait_bar(p, cx.red_bar(), red_round & 1u);
        ++red_round;
        if (et == 0) trace(p, span, 15);
        if (gi == n_groups - 1 && mc + cc_max >= m1 && et == 0) *cx.epi_done_ptr() = 1;
        if (MODE == 0) {
          // thread rrow finishes intermediate index rrow of the tile: operand rrow >> 6, gate lane / up lane = the two
          // halves of a quadrant.  The half-warps read gate and up in opposite order: no bank conflicts.
          const int opnd = rrow >> 6;
          const int lane_g = glu_gate_lane_of_index(rrow & 63);
          const int first = lane_g ^ (lane & 16);
#pragma unroll 1
          for (int c = et >> 7; c < cc; c += kEpiThreads >> 7) {
            float x = 0.0f, y = 0.0f;
#pragma unroll 4
            for (int qi = 0; qi < n; ++qi) {               // fixed span order: deterministic
              const float* img = stg + ((size_t)(2 * qi + opnd) * cc + c) * 128;
              x += img[first];
              y += img[first ^ 16];
            }
            const float ah = finish_glu<DYN>(p, sc4, g.tile, rrow, mc + c, mc + c, (lane & 16) ? y : x, (lane & 16) ? x : y);
            if (DYN) {                                       // the warp's 32 indices share the token column
              const int mx = __reduce_max_sync(0xffffffffu, __float_as_int(ah));
              if (lane == 0) atomicMax(reinterpret_cast<int*>(sc4 + mc + c) + 2, mx);
            }
          }
        } else {
#pragma unroll 1
          for (int c = et >> 7; c < cc; c += kEpiThreads >> 7) {
            float f0 = 0.0f, f1 = 0.0f;
#pragma unroll 4
            for (int qi = 0; qi < n; ++qi) {               // fixed span order: deterministic
              f0 += stg[((size_t)(2 * qi) * cc + c) * 128 + rrow];
              f1 += stg[((size_t)(2 * qi + 1) * cc + c) * 128 + rrow];
            }
            const float kx = sc1[mc + c];
            store_y(p, g.tile * 256 + rrow, mc + c, f0 * kx);
            store_y(p, g.tile * 256 + 128 + rrow, mc + c, f1 * kx);
          }
        }
      }
    }
    if (et == 0) trace(p, span, 9);
  }
}

// barriers, TMEM, the context of the CTA
__device__ __forceinline__ Ctx prologue(const GemmParams& p, uint8_t* smem_raw) {
  Ctx cx;
  const uint32_t raw = smem_u32(smem_raw);
  cx.smem_base = (raw + 1023u) & ~1023u;
  cx.smem_gen = smem_raw + (cx.smem_base - raw);
  cx.S = p.num_stages;
  cx.slot_bytes = (uint32_t)p.slot_bytes;
  cx.ring_bytes = (uint32_t)cx.S * cx.slot_bytes;
  cx.bar_base = cx.smem_base + cx.ring_bytes;
  cx.b_tile_bytes = (uint32_t)p.n_pad * 128u;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (warp == 0 && lane == 0) {
    for (int s = 0; s < cx.S; ++s) { mbar_init(cx.full_bar(s), 1); mbar_init(cx.empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(cx.accf_bar(b), 1); mbar_init(cx.acce_bar(b), kEpiThreads); }
    mbar_init(cx.red_bar(), 1);
    *cx.epi_done_ptr() = 0;
    fence_barrier_init();
  }
  if (warp == 2) tmem_alloc(cx.tmem_slot(), kTmemCols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  cx.tmem_base = *cx.tmem_slot_ptr();
  // let the next kernel of the stream start its own prologue (it waits for us in pdl_wait)
  pdl_launch_dependents();
  return cx;
}

}  // namespace

// ------------------------------------------------------------------------------------------ one GEMM
template <int MODE, bool DYN>
__global__ void __launch_bounds__(kThreads, 1)
spense_gemm_kernel(const __grid_constant__ GemmParams p, const __grid_constant__ CUtensorMap tmap_b) {
  extern __shared__ uint8_t smem_raw[];
  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  if (warp == 0 && lane == 0) prefetch_tmap(&tmap_b);
  Ctx cx = prologue(p, smem_raw);
  const int span = p.n_spans - 1 - (int)blockIdx.x;
  if (p.trace && threadIdx.x == 0) {
    uint32_t smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    p.trace[(size_t)span * 16 + 0] = globaltimer(); p.trace[(size_t)span * 16 + 14] = smid;
  }

  if (warp == 0) {
    if (lane == 0) {
      producer<MODE>(p, &tmap_b, cx, span);
      trace(p, span, 2);
      prefetch_next(p, cx, span);
    }
  } else if (warp == 1) {
    if (lane == 0) mma_issuer<MODE>(p, cx, span);
  } else if (warp >= 4) {
    const int et = threadIdx.x - 128;
    // scales, the workspace and the epoch word may be produced / still in use by the previous kernel
    pdl_wait();
    epilogue_tables(p, cx, et);
    if (et == kEpiThreads - 1) {
      check_header(p);
      take_epoch(p.ws_ctrl, (int)gridDim.x, cx.epoch_ptr());
    }
    epi_sync();
    const int epoch = cx.epoch_ptr()[0];                   // flag value of THIS launch (never equals a stale flag)
    epilogue<MODE, DYN>(p, cx, span, epoch);
    if (DYN) {                        // this CTA's max|h| per token, for the row requant kernel
      epi_sync();
      if (et < p.n_pad) p.amax_part[(size_t)span * p.n_pad + et] = et < p.M ? cx.sc0()[et].z : 0.0f;
    }
    if (et == 0) *cx.epi_done_ptr() = 1;
    if (p.trace && et == 0) p.trace[(size_t)span * 16 + 10] = globaltimer();
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) { tc_fence_after(); tmem_dealloc(cx.tmem_base, kTmemCols); }
}

namespace {
size_t smem_bytes_of(const GemmParams& p) { return (size_t)p.num_stages * p.slot_bytes + 1024 + 256 + 20 * (size_t)p.n_pad; }

// per device and kernel instance, once: opt in to the shared memory, and find out how many CTAs the device can hold
// resident at the same time (the CTAs of a launch wait for each other)
template <typename K>
int prepare(K kernel, int which, int dev, int sms, int grid) {
  static std::mutex mu;
  static bool ready[4][64] = {};
  static int resident[4][64] = {};
  std::lock_guard<std::mutex> lk(mu);
  if (dev < 0 || dev >= 64) return SPENSE_ERR_CUDA;
  if (!ready[which][dev]) {
    if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemMax) != cudaSuccess) return SPENSE_ERR_CUDA;
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kThreads, kSmemMax) != cudaSuccess) return SPENSE_ERR_CUDA;
    resident[which][dev] = per_sm * sms;
    ready[which][dev] = true;
  }
  return grid <= resident[which][dev] ? SPENSE_OK : SPENSE_ERR_CUDA;
}
}  // namespace

int launch_gemm(const GemmParams& p, const CUtensorMap& tmap_b, bool pdl, int dev, int sms, cudaStream_t stream) {
  const int grid = p.n_spans;
  int st = p.mode == 2     ? prepare(spense_gemm_kernel<2, false>, 3, dev, sms, grid)
           : p.mode == 1   ? prepare(spense_gemm_kernel<1, false>, 2, dev, sms, grid)
           : p.amax_part ? prepare(spense_gemm_kernel<0, true>, 1, dev, sms, grid)
                         : prepare(spense_gemm_kernel<0, false>, 0, dev, sms, grid);
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
  const cudaError_t e = p.mode == 2     ? cudaLaunchKernelEx(&cfg, spense_gemm_kernel<2, false>, p, tmap_b)
                        : p.mode == 1   ? cudaLaunchKernelEx(&cfg, spense_gemm_kernel<1, false>, p, tmap_b)
                        : p.amax_part ? cudaLaunchKernelEx(&cfg, spense_gemm_kernel<0, true>, p, tmap_b)
                                      : cudaLaunchKernelEx(&cfg, spense_gemm_kernel<0, false>, p, tmap_b);
  return e == cudaSuccess ? SPENSE_OK : SPENSE_ERR_CUDA;
}

}  // namespace spense
