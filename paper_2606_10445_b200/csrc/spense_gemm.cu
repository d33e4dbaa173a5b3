// Spense hybrid sparse-dense FP8 GEMM for sm_100a (tcgen05 + TMEM + TMA / bulk copy).
//
// Two GEMM "phases", written once as per-role device functions:
//   MODE 0  gate_up : output-split.  Pair tile = 128 rows of W_gate + the same 128 rows
//                     of W_up; tiles below I_s are 2:4 compressed (tcgen05.mma.sp), the rest dense
//                     (tcgen05.mma).  Epilogue: scales -> SiLU(g)*u (Eq. 4) -> E4M3.
//   MODE 1  down    : input-split.  Pair tile = 2 x 128 rows of W_down; the K loop runs
//                     the sparse stages and then the dense stages INTO THE SAME TMEM ACCUMULATOR.
// and the kernels built from them: spense_gemm_kernel<MODE, DYN> (one phase; DYN = gate_up that keeps h in fp32
// and tracks max|h| per token for the dynamic requant) and spense_mlp_kernel (gate_up then down in ONE persistent
// launch, see below).
//
// Swap-AB: only the A operand of tcgen05.mma.sp can be sparse, so weights are A (MMA-M = 128 weight
// rows) and tokens are B (MMA-N = padded token count); the accumulator holds Y^T [128 rows x tokens].
//
// Decode is weight-streaming bound, so the grid is a cost-balanced stream-K: the linear sequence of
// stage images (= the byte order of the blob) is cut into n_spans spans, one persistent CTA per span.
// A tile whose stages fall into several spans is fixed up through an L2-resident fp32 workspace, always
// adding the partials in span order, so results are bitwise reproducible:
//   * 2 spans  : the second span finishes its part early (it is its first segment), dumps it and
//                publishes a flag; the first span (owner) adds it to its TMEM accumulator and runs the
//                epilogue -- nothing but the flag check sits on the owner's critical path;
//   * > 2 spans: every span finishes late, so all dump, and the n spans reduce M/n token columns each
//                (reduce-scatter) instead of one owner reducing n partials serially.
// More than 128 tokens: blocks of 128 tokens SIDE BY SIDE in one launch.  The grid is nb * n_spans CTAs; CTA b works
// on token block b / n_spans and span n_spans-1 - b % n_spans of the same schedule, so the CTAs of different blocks
// read the same weight stage at about the same time: one HBM read, the other blocks hit L2 (measured at M=2048:
// 210 MB of DRAM reads per launch of 4 blocks).  Every block has its own fix-up slots; more blocks than fit run
// as further launches.
// Flags hold the epoch of the launch (a device-side counter in the workspace), so nothing has to be
// reset between launches and CUDA-graph replays see fresh values.
// Span i runs on CTA n_spans-1-i.  CTAs of one launch wait for each other, so all n_spans <= #SM CTAs
// must be co-resident: 1 CTA/SM by construction (shared memory), the device must not be shared.
//
// Fused MLP kernel: on every SM a GEMM CTA spends ~3 us getting started and ~6-8 us in its fix-up tail,
// and with 1 CTA/SM nothing else can stream weights through that SM meanwhile.  spense_mlp_kernel runs both
// phases in one CTA: the producer goes straight on to W_down while the epilogue warps finish gate_up, so
// the ring is full of down stages by the time their Hq tiles exist.  There is no grid-wide barrier: gate_up
// publishes one flag per finished 128-column tile of Hq and down's producer polls exactly the tiles a
// stage reads (the last CTA clears the flags).  gate_up never waits for down, so there is no cycle.
//
// Warp roles (640 threads): warp 0 producer (bulk copy of the weight stage + TMA of the activation
// tile), warp 1 MMA issuer, warp 2 TMEM allocator, warps 4-19 epilogue (TMEM lane quadrant = warp & 3,
// quarter of the token columns = (warp - 4) >> 2): the last tile's epilogue is exposed at the end of
// every CTA and is instruction-issue bound, so it gets 4 warps per scheduler.  Rarely executed code is
// kept rolled: the kernel is latency-sensitive at its tail and instruction-cache misses on cold paths
// showed up in the timeline.
#include <cuda_bf16.h>

#include "spense_internal.cuh"

namespace spense {

namespace {

// Position in the linear stage sequence: pair tile, stage inside the tile, stages of the tile.
struct Cursor {
  int tile, j, ns, nd, first;   // first = linear index of the tile's first stage
};

// byte offset of stage j of pair tile `tile` inside the section (the blob stores every tile once)
template <int MODE>
__device__ __forceinline__ size_t stage_byte_offset(const GemmParams& p, int tile, int j) {
  if (MODE == 0) {
    if (tile < p.tiles_sparse) return ((size_t)tile * p.ns + j) * kSparseStageBytes;
    return (size_t)p.tiles_sparse * p.ns * kSparseStageBytes + ((size_t)(tile - p.tiles_sparse) * p.nd + j) * kDenseStageBytes;
  }
  const size_t base = (size_t)tile * ((size_t)p.ns * kSparseStageBytes + (size_t)p.nd * kDenseStageBytes);
  return base + (j < p.ns ? (size_t)j * kSparseStageBytes
                          : (size_t)p.ns * kSparseStageBytes + (size_t)(j - p.ns) * kDenseStageBytes);
}

// The only place with integer divisions (one copy per mode, called once per role and phase).
template <int MODE>
__device__ __noinline__ Cursor cursor_at(const GemmParams& p, int s, unsigned long long* byte_off) {
  Cursor c;
  if (MODE == 0) {
    const int sparse_total = p.tiles_sparse * p.ns;
    if (s < sparse_total) {
      c.tile = s / p.ns;
      c.first = c.tile * p.ns;
      c.ns = p.ns; c.nd = 0;
    } else {
      const int td = (s - sparse_total) / p.nd;
      c.tile = p.tiles_sparse + td;
      c.first = sparse_total + td * p.nd;
      c.ns = 0; c.nd = p.nd;
    }
  } else {
    const int per = p.ns + p.nd;
    c.tile = s / per;
    c.first = c.tile * per;
    c.ns = p.ns; c.nd = p.nd;
  }
  c.j = s - c.first;
  *byte_off = stage_byte_offset<MODE>(p, c.tile, c.j);
  return c;
}

template <int MODE>
__device__ __forceinline__ void next_tile(const GemmParams& p, Cursor& c) {
  c.first += c.ns + c.nd;
  ++c.tile;
  c.j = 0;
  if (MODE == 0) {
    if (c.tile < p.tiles_sparse) { c.ns = p.ns; c.nd = 0; } else { c.ns = 0; c.nd = p.nd; }
  }
}

// SiLU(g) * u on the hardware exp2 / reciprocal units: branch-free, relative error ~1e-6 (far inside
// the GLU tolerance).  ex2 of a very negative g overflows to +inf -> rcp gives 0 -> h = -0 * u.
__device__ __forceinline__ float silu_mul(float g, float u) {
  float e, r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(-1.4426950408889634f * g));
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(1.0f + e));
  return g * r * u;
}

// a / b from the correctly rounded reciprocal r = RN(1/b) and two FMAs (Markstein): branch-free and
// correctly rounded wherever the quotient is a normal number -- all the E4M3 cast after it can see
// (a zero quotient keeps the sign IEEE division gives it: h = -0 must encode as 0x80 like the oracle's).
__device__ __forceinline__ float div_by(float a, float b, float r) {
  const float q0 = a * r;
  const float rem = fmaf(-q0, b, a);
  const float q = fmaf(rem, r, q0);
  return q == 0.0f ? q0 : q;                               // (+0) + (-0) = +0 would lose the sign of a zero quotient
}

// fp32 -> E4M3 (saturating, round to nearest even); cvt.rn.satfinite.e4m3x2.f32 packs two values
// returns lo in bits 0..7 and hi in bits 8..15
__device__ __forceinline__ uint32_t to_e4m3x2(float lo, float hi) {
  uint16_t r;
  asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(r) : "f"(hi), "f"(lo));
  return r;
}

// optional per-CTA timeline (the harness sets GemmParams::trace through a debug hook; nullptr in production)
__device__ __forceinline__ long long globaltimer() {
  long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
__device__ __forceinline__ void trace(const GemmParams& p, int span, int slot) {
  if (p.trace) p.trace[(size_t)span * 16 + slot] = globaltimer();
}
__device__ __forceinline__ int ld_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release(int* p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void epi_sync() { asm volatile("bar.sync 1, 512;" ::: "memory"); }   // the 16 epilogue warps
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {                        // non-blocking
  uint32_t ok;
  asm volatile("{\n\t.reg .pred p;\n\tmbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
               : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0;
}

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
  int blk;                     // token block of this CTA (0 unless the launch covers several blocks)
  int gbase;                   // first fix-up slot (flags, partials) of this block: block-in-launch * n_spans
  __device__ __forceinline__ uint32_t full_bar(int s) const { return bar_base + 8u * s; }
  __device__ __forceinline__ uint32_t empty_bar(int s) const { return bar_base + 8u * (8 + s); }
  __device__ __forceinline__ uint32_t accf_bar(int b) const { return bar_base + 8u * (16 + b); }
  __device__ __forceinline__ uint32_t acce_bar(int b) const { return bar_base + 8u * (18 + b); }
  __device__ __forceinline__ uint32_t tmem_slot() const { return bar_base + 8u * 20; }
  __device__ __forceinline__ uint32_t red_bar() const { return bar_base + 8u * 22; }
  __device__ __forceinline__ volatile uint32_t* tmem_slot_ptr() const { return reinterpret_cast<volatile uint32_t*>(smem_gen + ring_bytes + 8 * 20); }
  __device__ __forceinline__ volatile int* epoch_ptr() const { return reinterpret_cast<volatile int*>(smem_gen + ring_bytes + 8 * 21); }   // 2 ints
  __device__ __forceinline__ volatile int* epi_done_ptr() const { return reinterpret_cast<volatile int*>(smem_gen + ring_bytes + 8 * 23); }
  __device__ __forceinline__ float4* sc0() const { return reinterpret_cast<float4*>(smem_gen + ring_bytes + 256); }
  __device__ __forceinline__ float* sc1(int n_pad) const { return reinterpret_cast<float*>(smem_gen + ring_bytes + 256 + 16 * n_pad); }
};

// One output element (token m, weight row r of pair tile `tile`): scales, GLU + requant, or the Y store.
// MODE 0: sc = float4 per token column {s_x*s_gate, s_x*s_up, s_h, RN(1/s_h)}; MODE 1: sc = float per token s_h*s_down.
// m = token column inside the block (index of the scale table), m_out = token (output row).
template <int MODE, bool DYN>
__device__ __forceinline__ void finish(const GemmParams& p, const void* sc, int tile, int r, int m, int m_out, float f0, float f1) {
  if (MODE == 0) {
    const float4* sc4 = reinterpret_cast<const float4*>(sc);
    const float4 k = sc4[m];
    const float g = f0 * k.x;
    const float u = f1 * k.y;
    const float h = silu_mul(g, u);
    const size_t o = (size_t)m_out * p.ld_out + tile * 128 + r;
    if (DYN) {
      // dynamic requant: keep h in fp32 and track max|h| per token; the scale does not
      // exist yet, the row requant kernel turns h into Hq once every tile is done.  Called warp-uniformly in m.
      p.h_f32[o] = h;
      const int mx = __reduce_max_sync(0xffffffffu, __float_as_int(fabsf(h)));   // |h| >= 0: int order == float order
      if ((threadIdx.x & 31) == 0) atomicMax(reinterpret_cast<int*>(const_cast<float4*>(sc4) + m) + 2, mx);
      return;
    }
    const float qv = div_by(h, k.z, k.w);
    if (p.h_f32) p.h_f32[o] = h;
    p.hq[o] = (uint8_t)(to_e4m3x2(qv, 0.0f) & 0xFFu);
  } else {
    const float kx = reinterpret_cast<const float*>(sc)[m];
    const int out_row = tile * 256 + r;
    const float y0 = f0 * kx, y1 = f1 * kx;
    const size_t o = (size_t)m_out * p.ld_out + out_row;
    const bool second = out_row + 128 < p.out_rows;
    if (p.y_dtype == SPENSE_F32) {
      float* y = reinterpret_cast<float*>(p.y);
      y[o] = y0;
      if (second) y[o + 128] = y1;
    } else {
      __nv_bfloat16* y = reinterpret_cast<__nv_bfloat16*>(p.y);
      y[o] = __float2bfloat16_rn(y0);
      if (second) y[o + 128] = __float2bfloat16_rn(y1);
    }
  }
}

// A tile shared by more than two spans [a, b]: reduced at the end of the phase (reduce-scatter).
struct Group { int a, b, tile, first; };

// ===================== producer (one thread) =====================
// Streams the stages of span `span` of one phase through the ring.  `it` counts the stages of the whole
// kernel (slot = it % S).  A weight stage depends on nothing and is issued as soon as its slot is free; the
// activation tile of the same stage is issued when its data exists:
//   !gated : after the previous kernel of the stream (one griddepcontrol.wait, when the ring is full of weights);
//   gated  : per stage, when gate_up has published the Hq tiles the stage reads (fused kernel, down phase).
template <int MODE, bool GATED>
__device__ __forceinline__ void producer_phase(const GemmParams& p, const CUtensorMap* tmap, const Ctx& cx, int span,
                                               int& it, bool& pdl_done) {
  const int S = cx.S;
  const int sb = p.span_begin[span];
  const int n = p.span_begin[span + 1] - sb;
  // one token block: a weight byte is used once (evict first); several: the CTAs of the other blocks read the same
  // stage at about the same time and should find it in L2
  const uint64_t pol_w = p.nb == 1 ? policy_evict_first() : policy_evict_normal();
  const uint64_t pol_a = policy_evict_last();
  unsigned long long off;
  Cursor c = cursor_at<MODE>(p, sb, &off);
  const uint8_t* src = p.section + off;
  const int it0 = it;
  uint32_t info[8];                                        // stages whose weights are in flight: K coordinate | sparse << 31
  int dep_lo = 0, dep_hi = 0;                              // Hq tiles [dep_lo, dep_hi) are known to be stored

  auto tiles_ready = [&](uint32_t inf) -> bool {           // at most one poll (16 flags) per call
    const int k0 = (int)(inf & 0x7FFFFFFFu);
    const int t_first = k0 >> 7;
    int t_last = (k0 + ((inf >> 31) ? 255 : 127)) >> 7;
    if (t_last >= p.dep_tiles) t_last = p.dep_tiles - 1;   // a padded K stage reads no further than the last tile
    if (t_first < dep_lo || t_first > dep_hi) dep_lo = dep_hi = t_first;   // the K range restarted (next row tile)
    if (dep_hi > t_last) return true;
    const int4* f = reinterpret_cast<const int4*>(p.dep_flags + (dep_hi & ~3));
    int4 v[4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
      asm volatile("ld.volatile.global.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(v[i].x), "=r"(v[i].y), "=r"(v[i].z), "=r"(v[i].w) : "l"(f + i));
    uint32_t m = 0;
#pragma unroll
    for (int i = 0; i < 4; ++i)
      m |= (uint32_t)((v[i].x != 0) | ((v[i].y != 0) << 1) | ((v[i].z != 0) << 2) | ((v[i].w != 0) << 3)) << (4 * i);
    m >>= dep_hi & 3;
    const int n_ready = __ffs(~m) - 1;                     // consecutive finished tiles from dep_hi on
    if (n_ready > 0) {
      dep_hi += n_ready;
      asm volatile("fence.acq_rel.gpu;" ::: "memory");
      asm volatile("fence.proxy.async.global;" ::: "memory");   // gate_up's generic-proxy stores -> our TMA reads
    }
    return dep_hi > t_last;
  };
  auto load_b = [&](int slot, uint32_t inf) {
    const uint32_t b_dst = cx.smem_base + (uint32_t)slot * cx.slot_bytes + kSparseStageBytes;
    const int k0 = (int)(inf & 0x7FFFFFFFu);                // K coordinate | sparse << 31
    const int row0 = cx.blk * p.n_pad;                      // this CTA's token block
    tma_load_2d(b_dst, tmap, k0, row0, cx.full_bar(slot), pol_a);
    if (inf >> 31) tma_load_2d(b_dst + cx.b_tile_bytes, tmap, k0 + 128, row0, cx.full_bar(slot), pol_a);
  };

  int w = 0;                                               // weight stages issued (of this phase)
  uint32_t pf_off = 0;                                     // gated phase: bytes past `src` already prefetched into L2
  long long pf_next = 0;
  uint32_t inf_last = 0;                                   // descriptor of the stage issued last (steady state: no table)
  // ring position of the next weight stage / the next activation tile, kept incrementally (no divisions per stage)
  int w_slot = it0 % S, w_round = it0 / S;
  int b_slot = w_slot;
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
      if (blocking) mbar_wait(cx.empty_bar(w_slot), par);
      else if (!mbar_test(cx.empty_bar(w_slot), par)) return false;
    }
    mbar_expect_tx(fb, tx);
    bulk_g2s(dst, src, wb, fb, pol_w);
    inf_last = inf;
    if (!blocking) {                                       // running ahead of the activation tiles: remember it
#pragma unroll
      for (int k = 0; k < 8; ++k)
        if (k == ((it0 + w) & 7)) info[k] = inf;
    }
    src += wb;
    if (++c.j == c.ns + c.nd) next_tile<MODE>(p, c);
    ++w;
    if (++w_slot == S) { w_slot = 0; ++w_round; }
    return true;
  };

  if (!GATED && !pdl_done) {
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
    pdl_done = true;
  }
#pragma unroll 1
  for (int b = 0; b < n; ++b) {
    uint32_t inf = 0;
    if (w <= b) {
      issue_weight(true);
      inf = inf_last;
    } else {
#pragma unroll
      for (int k = 0; k < 8; ++k)
        if (k == ((it0 + b) & 7)) inf = info[k];
    }
    if (GATED) {
      // while gate_up has not finished the tiles this stage reads, let the weights run ahead (up to one ring)
#pragma unroll 1
      while (!tiles_ready(inf)) {
        if (w < n && w - b < S && issue_weight(false)) continue;
        // the ring is full and Hq is not there yet: keep HBM busy pulling the following stages into L2 (paced)
        if (p.pf_pace_ns && pf_off < p.gated_pf_bytes && pf_off + 32768u <= (uint32_t)(n - w) * (uint32_t)kDenseStageBytes && globaltimer() >= pf_next) {
          asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src + pf_off), "r"(32768u) : "memory");
          pf_off += 32768u;
          pf_next = globaltimer() + p.pf_pace_ns;
        }
      }
    }
    load_b(b_slot, inf);
    if (++b_slot == S) b_slot = 0;
  }
  it = it0 + n;
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
// it / seg count the stages / accumulator segments of the whole kernel (ring slot, TMEM buffer and parities).
template <int MODE>
__device__ __forceinline__ void mma_phase(const GemmParams& p, const Ctx& cx, int span, int& it, int& seg) {
  const int S = cx.S;
  const uint32_t idesc_d = (1u << 4) | ((uint32_t)(p.n_pad >> 3) << 17) | ((128u >> 4) << 24);
  const uint32_t idesc_s = idesc_d | (1u << 2);
  const int sb = p.span_begin[span], se = p.span_begin[span + 1];
  unsigned long long off;
  Cursor c = cursor_at<MODE>(p, sb, &off);
  int slot = it % S;                                       // ring position, kept incrementally (no divisions per stage)
  uint32_t ph = (uint32_t)(it / S) & 1u;
#pragma unroll 1
  for (int s = sb; s < se; ++seg) {
    const int tile_end = c.first + c.ns + c.nd;
    const int seg_end = min(se, tile_end);
    const int buf = seg % p.num_acc_bufs;
    const uint32_t use = (uint32_t)(seg / p.num_acc_bufs);
    mbar_wait(cx.acce_bar(buf), (use & 1u) ^ 1u);          // epilogue has drained this accumulator
    tc_fence_after();
    const uint32_t d0 = cx.tmem_base + (uint32_t)(buf * 2 * p.acc_stride);
    const uint32_t d1 = d0 + (uint32_t)p.acc_stride;
    uint32_t acc = 0;
#pragma unroll 1
    for (; s < seg_end; ++s, ++it, ++c.j) {
      mbar_wait(cx.full_bar(slot), ph);
      tc_fence_after();
      if (s == sb) trace(p, span, 3);
      const uint32_t a0 = cx.smem_base + (uint32_t)slot * cx.slot_bytes;
      const uint32_t a1 = a0 + kOperandBytes;
      const uint32_t b0 = a0 + kSparseStageBytes;
      if (c.j < c.ns) {
        const uint32_t e_base = cx.tmem_base + kMetaCol + (uint32_t)(it & 1) * 16u;
        const uint32_t m0 = a0 + 2 * kOperandBytes;       // A0 meta: 2 atoms of 2 KB, then A1 meta
#pragma unroll
        for (int a = 0; a < 4; ++a)                       // 4 atoms: (A0,k0) (A0,k1) (A1,k0) (A1,k1)
          tc_cp_128x128b(e_base + 4u * a, make_desc(m0 + 2048u * a, 0, 128, kLayoutNone));
#pragma unroll
        for (int k = 0; k < 4; ++k) {                     // 4 sparse MMAs of K = 64 logical (32 B of A, 64 B of B)
          const uint64_t bd = make_desc(b0 + (uint32_t)(k >> 1) * cx.b_tile_bytes + (uint32_t)(k & 1) * 64u, 16, 1024, kLayoutSW128);
          mma_f8_sparse(d0, make_desc(a0 + 32u * k, 16, 1024, kLayoutSW128), bd, e_base + 2u * k, idesc_s, acc);
          mma_f8_sparse(d1, make_desc(a1 + 32u * k, 16, 1024, kLayoutSW128), bd, e_base + 8u + 2u * k, idesc_s, acc);
          acc = 1;
        }
      } else {
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

// scale tables of the token block that starts at token m_base (Mb tokens)
__device__ __forceinline__ void epilogue_tables(const GemmParams& p, const Ctx& cx, int et, int m_base, int Mb) {
  if (et < p.n_pad) {
    const int m = m_base + (et < Mb ? et : Mb - 1);
    if (p.mode == 0) {
      const float sx = __ldg(p.s_act + m);
      const float sh = p.amax_part ? 1.0f : __ldg(p.s_h + (size_t)m * p.sh_stride);
      cx.sc0()[et] = make_float4(sx * p.w_scale0, sx * p.w_scale1, p.amax_part ? 0.0f : sh, __frcp_rn(sh));   // dynamic: .z = running max|h| bits
    } else {
      cx.sc1(p.n_pad)[et] = __ldg(p.s_act + (size_t)m * p.sh_stride) * p.w_scale0;
    }
  }
}

// ===================== epilogue (16 warps) =====================
// warp & 3 selects the TMEM lane quadrant, (warp - 4) >> 2 the quarter of the token columns.
// ring_free: this is the last phase of the kernel, so once the CTA's last accumulator is complete the stage
// ring is idle and stages the partials (bulk copies); otherwise the producer is already filling the ring with
// the next phase's weights and partials are read straight from L2.
template <int MODE, bool DYN, bool FUSED0>
__device__ __forceinline__ void epilogue_phase(const GemmParams& p, const Ctx& cx, int span, int& seg, uint32_t& red_round,
                                               int epoch, const void* sc) {
  constexpr bool ring_free = !FUSED0;                      // FUSED0: gate_up phase of the fused kernel (publishes tile flags)
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int q = warp & 3;
  const int row = q * 32 + lane;                           // accumulator lane = weight row inside the tile
  const int et = threadIdx.x - 128;                        // 0..511
  const int m_base = cx.blk * p.n_pad;                     // this CTA's token block
  const int Mb = min(p.n_pad, p.M - m_base);
  const int cols_used = min(p.n_pad, (Mb + 7) & ~7);       // token columns holding real tokens, rounded to the TMEM load width
  const int cols_per = (((p.n_pad + 3) >> 2) + 7) & ~7;    // columns per warp: a quarter, rounded to the TMEM load width
  const int c_begin = ((warp - 4) >> 2) * cols_per;
  const int c_end = min(c_begin + cols_per, cols_used);
  const float* stg = reinterpret_cast<const float*>(cx.smem_gen);   // the stage ring doubles as partial staging
  const size_t part_floats = (size_t)2 * p.n_pad * 128;    // one partial: [mat][col][row]
  int* const flags = p.flags + cx.gbase * 2;               // fix-up slots of this token block
  float* const partials = p.partials + (size_t)cx.gbase * 2 * part_floats;
  const int sb = p.span_begin[span], se = p.span_begin[span + 1];

  Group groups[2];
  int n_groups = 0;
  unsigned long long off;
  Cursor cur = cursor_at<MODE>(p, sb, &off);
  int seg_local = 0;
#pragma unroll 1
  for (int s = sb; s < se; ++seg, ++seg_local) {
    const int tile_end = cur.first + cur.ns + cur.nd;
    const int seg_end = min(se, tile_end);
    const int buf = seg % p.num_acc_bufs;
    const uint32_t use = (uint32_t)(seg / p.num_acc_bufs);
    // spans [a, b] that hold stages of this tile
    int a = span, b = span;
    while (p.span_begin[a] > cur.first) --a;
    while (b + 1 < p.n_spans && p.span_begin[b + 1] < tile_end) ++b;

    // staged fix-ups and plain segments wait for the accumulator first; a direct owner-add fetches its partner's
    // partial (dumped long ago) BEFORE that, so the loads are off the critical path
    const bool early_fetch = b == a + 1 && span == a && !ring_free;
    if (!early_fetch) {
      mbar_wait(cx.accf_bar(buf), use & 1u);
      tc_fence_after();
      if (et == 0) trace(p, span, seg_local == 0 ? 5 : 7);
    }
    const uint32_t t0 = cx.tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * 2 * p.acc_stride);
    const uint32_t t1 = t0 + (uint32_t)p.acc_stride;

    if (a == b || (b == a + 1 && span == a)) {
      // the whole tile is ours, or we own a tile whose tail the next span has (usually long ago) dumped
      const bool add = a != b;
      const bool staged = add && ring_free;                // owner = last segment of the span: every MMA is complete
      const float* part = partials + (size_t)b * 2 * part_floats;   // span b starts inside the tile: its first segment
      float a0[8], a1[8];                                  // direct owner-add: the partner's partial, one chunk ahead
      if (add) {
        const int* f = flags + b * 2;
        if (staged) {
          if (et == 0) {
            while (ld_acquire(f) != epoch) {}
            asm volatile("fence.proxy.async.global;" ::: "memory");   // partner's generic-proxy stores -> our async-proxy read
            mbar_expect_tx(cx.red_bar(), 2u * (uint32_t)cols_used * 512u);
            bulk_g2s(cx.smem_base, part, (uint32_t)cols_used * 512u, cx.red_bar(), policy_evict_first());
            bulk_g2s(cx.smem_base + (uint32_t)cols_used * 512u, part + (size_t)p.n_pad * 128, (uint32_t)cols_used * 512u, cx.red_bar(), policy_evict_first());
          }
          mbar_wait(cx.red_bar(), red_round & 1u);
          ++red_round;
        } else {
          while (ld_acquire(f) != epoch) {}                // warp-uniform address: one request per warp
          if (c_begin < c_end) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              a0[i] = __ldcg(part + (size_t)(c_begin + i) * 128 + row);
              a1[i] = __ldcg(part + (size_t)(p.n_pad + c_begin + i) * 128 + row);
            }
          }
        }
        if (et == 0) trace(p, span, 8);
      }
      if (early_fetch) {
        mbar_wait(cx.accf_bar(buf), use & 1u);
        tc_fence_after();
        if (et == 0) trace(p, span, seg_local == 0 ? 5 : 7);
      }
      if (seg_end == se && n_groups == 0 && et == 0 && ring_free) *cx.epi_done_ptr() = 1;   // last epilogue of this CTA: stop prefetching now
#pragma unroll 1
      for (int c = c_begin; c < c_end; c += 8) {
        uint32_t v0[8], v1[8];
        tmem_ld8(t0 + c, v0);
        tmem_ld8(t1 + c, v1);
        tmem_ld_wait();
        float f0[8], f1[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) { f0[i] = __uint_as_float(v0[i]); f1[i] = __uint_as_float(v1[i]); }
        if (staged) {
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            f0[i] += stg[(size_t)(c + i) * 128 + row];
            f1[i] += stg[(size_t)(cols_used + c + i) * 128 + row];
          }
        } else if (add) {
#pragma unroll
          for (int i = 0; i < 8; ++i) { f0[i] += a0[i]; f1[i] += a1[i]; }
          if (c + 8 < c_end) {                             // next chunk's partial loads overlap this chunk's epilogue math
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              a0[i] = __ldcg(part + (size_t)(c + 8 + i) * 128 + row);
              a1[i] = __ldcg(part + (size_t)(p.n_pad + c + 8 + i) * 128 + row);
            }
          }
        }
#pragma unroll
        for (int i = 0; i < 8; ++i)
          if (c + i < Mb) finish<MODE, DYN>(p, sc, cur.tile, row, c + i, m_base + c + i, f0[i], f1[i]);
      }
      tc_fence_before();
      mbar_arrive(cx.acce_bar(buf));
      if (FUSED0) {                                        // Hq[:, tile] complete: all stores issued, one release
        epi_sync();
        if (et == 0) st_release(p.tile_flags + cur.tile, 1);
      }
    } else {
      // split tile, not (solely) ours to finish: dump the raw fp32 partial [mat][col][row] and publish it
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
          __stcg(slot + (size_t)(c + i) * 128 + row, __uint_as_float(v0[i]));
          __stcg(slot + (size_t)(p.n_pad + c + i) * 128 + row, __uint_as_float(v1[i]));
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
  // [j*M/n, (j+1)*M/n), adding the n partials in span order, and runs the epilogue on them.
#pragma unroll 1
  for (int gi = 0; gi < n_groups; ++gi) {
    const Group g = groups[gi];
    const int n = g.b - g.a + 1;
    const int j = span - g.a;
    const int m0 = (int)(((long long)j * Mb) / n), m1 = (int)(((long long)(j + 1) * Mb) / n);
    const int rrow = et & 127;
    if (m1 > m0 && ring_free) {
      // all MMAs of this CTA are complete: the stage ring stages the partial slices
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
        // thread i fetches matrix (i & 1) of partner (i >> 1) as soon as THAT partner has published
#pragma unroll 1
        for (int i = et; i < 2 * n; i += kEpiThreads) {
          const int qs = g.a + (i >> 1), mat = i & 1;
          const int which = (p.span_begin[qs] >= g.first) ? 0 : 1;
          while (ld_acquire(flags + qs * 2 + which) != epoch) {}
          asm volatile("fence.proxy.async.global;" ::: "memory");   // partner's generic-proxy stores -> our async-proxy read
          const float* src = partials + ((size_t)qs * 2 + which) * part_floats + ((size_t)mat * p.n_pad + mc) * 128;
          bulk_g2s(cx.smem_base + (uint32_t)(i * cc) * 512u, src, (uint32_t)cc * 512u, cx.red_bar(), policy_evict_first());
        }
        mbar_wait(cx.red_bar(), red_round & 1u);
        ++red_round;
        if (et == 0) trace(p, span, 15);
        if (gi == n_groups - 1 && mc + cc_max >= m1 && et == 0) *cx.epi_done_ptr() = 1;
#pragma unroll 1
        for (int c = et >> 7; c < cc; c += kEpiThreads >> 7) {
          float f0 = 0.0f, f1 = 0.0f;
#pragma unroll 4
          for (int qi = 0; qi < n; ++qi) {                 // fixed span order: deterministic
            f0 += stg[((size_t)(2 * qi) * cc + c) * 128 + rrow];
            f1 += stg[((size_t)(2 * qi + 1) * cc + c) * 128 + rrow];
          }
          finish<MODE, DYN>(p, sc, g.tile, rrow, mc + c, m_base + mc + c, f0, f1);
        }
      }
    } else if (m1 > m0) {
      // the ring belongs to the next phase already: wait for every partner, then read the slices from L2
      if (et < n) {
        const int qs = g.a + et;
        const int which = (p.span_begin[qs] >= g.first) ? 0 : 1;
        while (ld_acquire(flags + qs * 2 + which) != epoch) {}
      }
      epi_sync();
#pragma unroll 1
      for (int c = m0 + (et >> 7); c < m1; c += kEpiThreads >> 7) {
        float f0 = 0.0f, f1 = 0.0f;
#pragma unroll 1
        for (int q0 = 0; q0 < n; q0 += 4) {                // 8 loads in flight, then added in fixed span order: deterministic
          float v0[4], v1[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const int qs = g.a + min(q0 + k, n - 1);
            const int which = (p.span_begin[qs] >= g.first) ? 0 : 1;
            const float* src = partials + ((size_t)qs * 2 + which) * part_floats;
            v0[k] = __ldcg(src + (size_t)c * 128 + rrow);
            v1[k] = __ldcg(src + (size_t)(p.n_pad + c) * 128 + rrow);
          }
#pragma unroll
          for (int k = 0; k < 4; ++k)
            if (q0 + k < n) { f0 += v0[k]; f1 += v1[k]; }
        }
        finish<MODE, DYN>(p, sc, g.tile, rrow, c, m_base + c, f0, f1);
      }
    }
    if (FUSED0) {                                          // the last of the n reducers publishes the tile
      epi_sync();
      if (et == 0) {
        __threadfence();
        if (atomicAdd(p.tile_cnt + g.tile, 1) == n - 1) {
          p.tile_cnt[g.tile] = 0;
          __threadfence();
          st_release(p.tile_flags + g.tile, 1);
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

// Epoch of a launch = epoch word + 1.  Every CTA reads the word BEFORE it counts itself; the CTA that counts
// last therefore knows all have read it and advances it for the next launch.  (ctrl1: second word pair of a
// fused launch, advanced together with the first.)
__device__ __forceinline__ void take_epoch(int* ctrl0, int* ctrl1, int n_ctas, volatile int* out) {
  const int e0 = ld_acquire(ctrl0);
  const int e1 = ctrl1 ? ld_acquire(ctrl1) : 0;
  out[0] = e0 + 1;
  out[1] = e1 + 1;
  if (atomicAdd(ctrl0 + 1, 1) == n_ctas - 1) {
    ctrl0[1] = 0;
    if (ctrl1) st_release(ctrl1, e1 + 1);
    st_release(ctrl0, e0 + 1);
  }
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
  // a launch covers p.nb token blocks: CTA b works on block blk0 + b / n_spans, span n_spans - 1 - b % n_spans of
  // the SAME stream-K schedule, so the CTAs of different blocks read the same weight stage at about the same time
  // (one HBM read, the rest L2 hits); each block has its own fix-up slots.  A block past the last token idles.
  const int bp = (int)blockIdx.x / p.n_spans;
  const int span = p.n_spans - 1 - ((int)blockIdx.x - bp * p.n_spans);
  cx.blk = p.blk0 + bp;
  cx.gbase = bp * p.n_spans;
  const bool idle = cx.blk * p.n_pad >= p.M;
  if (p.trace && threadIdx.x == 0 && bp == 0) {
    uint32_t smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    p.trace[(size_t)span * 16 + 0] = globaltimer(); p.trace[(size_t)span * 16 + 14] = smid;
  }

  if (idle) {
    // nothing to compute, but the launch counts its CTAs for the epoch
    if (threadIdx.x == 128 + kEpiThreads - 1) {
      pdl_wait();
      take_epoch(p.ws_ctrl, nullptr, (int)gridDim.x, cx.epoch_ptr());
    }
  } else if (warp == 0) {
    if (lane == 0) {
      int it = 0;
      bool pdl_done = false;
      producer_phase<MODE, false>(p, &tmap_b, cx, span, it, pdl_done);
      trace(p, span, 2);
      prefetch_next(p, cx, span);
    }
  } else if (warp == 1) {
    if (lane == 0) {
      int it = 0, seg = 0;
      mma_phase<MODE>(p, cx, span, it, seg);
    }
  } else if (warp >= 4) {
    const int et = threadIdx.x - 128;
    // scales, the workspace and the epoch word may be produced / still in use by the previous kernel
    pdl_wait();
    epilogue_tables(p, cx, et, cx.blk * p.n_pad, min(p.n_pad, p.M - cx.blk * p.n_pad));
    if (et == kEpiThreads - 1) take_epoch(p.ws_ctrl, nullptr, (int)gridDim.x, cx.epoch_ptr());
    epi_sync();
    const int epoch = cx.epoch_ptr()[0];                   // flag value of THIS launch (never equals a stale flag)
    int seg = 0;
    uint32_t red_round = 0;
    const void* sc = MODE == 0 ? (const void*)cx.sc0() : (const void*)cx.sc1(p.n_pad);
    epilogue_phase<MODE, DYN, false>(p, cx, span, seg, red_round, epoch, sc);
    if (DYN) {                        // this CTA's max|h| per token, for the row requant kernel
      epi_sync();
      if (et < p.n_pad) p.amax_part[(size_t)span * p.n_pad + et] = et < p.M ? cx.sc0()[et].z : 0.0f;
    }
    if (et == 0) *cx.epi_done_ptr() = 1;
    if (p.trace && et == 0 && bp == 0) p.trace[(size_t)span * 16 + 10] = globaltimer();
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) { tc_fence_after(); tmem_dealloc(cx.tmem_base, kTmemCols); }
}

// ------------------------------------------------------------------------------------------ the fused layer
// gate_up (pg) then down (pd) in one persistent launch; see the header comment.  Both phases use the same
// token padding, ring geometry and TMEM layout.  CTA b runs span n_spans-1-b of each phase (none if negative).
__global__ void __launch_bounds__(kThreads, 1)
spense_mlp_kernel(const __grid_constant__ GemmParams pg, const __grid_constant__ CUtensorMap tmap_x,
                  const __grid_constant__ GemmParams pd, const __grid_constant__ CUtensorMap tmap_hq) {
  extern __shared__ uint8_t smem_raw[];
  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;
  if (warp == 0 && lane == 0) { prefetch_tmap(&tmap_x); prefetch_tmap(&tmap_hq); }
  Ctx cx = prologue(pg, smem_raw);
  cx.blk = 0;
  cx.gbase = 0;
  const int span_g = pg.n_spans - 1 - (int)blockIdx.x;
  const int span_d = pd.n_spans - 1 - (int)blockIdx.x;
  if (threadIdx.x == 0) {
    uint32_t smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    if (pg.trace && span_g >= 0) { pg.trace[(size_t)span_g * 16 + 0] = globaltimer(); pg.trace[(size_t)span_g * 16 + 14] = smid; }
    if (pd.trace && span_d >= 0) { pd.trace[(size_t)span_d * 16 + 0] = globaltimer(); pd.trace[(size_t)span_d * 16 + 14] = smid; }
  }

  if (warp == 0) {
    if (lane == 0) {
      int it = 0;
      bool pdl_done = false;
      if (span_g >= 0) {
        producer_phase<0, false>(pg, &tmap_x, cx, span_g, it, pdl_done);
        trace(pg, span_g, 2);
      }
      if (span_d >= 0) {
        producer_phase<1, true>(pd, &tmap_hq, cx, span_d, it, pdl_done);   // Hq tiles gated by gate_up's flags
        trace(pd, span_d, 2);
      }
      if (!pdl_done) pdl_wait();                           // "this kernel complete" implies "everything before it complete"
      if (span_d >= 0) prefetch_next(pd, cx, span_d);
    }
  } else if (warp == 1) {
    if (lane == 0) {
      int it = 0, seg = 0;
      if (span_g >= 0) mma_phase<0>(pg, cx, span_g, it, seg);
      if (span_d >= 0) mma_phase<1>(pd, cx, span_d, it, seg);
    }
  } else if (warp >= 4) {
    const int et = threadIdx.x - 128;
    pdl_wait();
    epilogue_tables(pg, cx, et, 0, pg.M);
    epilogue_tables(pd, cx, et, 0, pd.M);
    if (et == kEpiThreads - 1) take_epoch(pg.ws_ctrl, pd.ws_ctrl, (int)gridDim.x, cx.epoch_ptr());
    epi_sync();
    const int epoch_g = cx.epoch_ptr()[0], epoch_d = cx.epoch_ptr()[1];
    int seg = 0;
    uint32_t red_round = 0;
    if (span_g >= 0) {
      epilogue_phase<0, false, true>(pg, cx, span_g, seg, red_round, epoch_g, cx.sc0());
      if (pg.trace && et == 0) pg.trace[(size_t)span_g * 16 + 10] = globaltimer();
    }
    if (span_d >= 0) epilogue_phase<1, false, false>(pd, cx, span_d, seg, red_round, epoch_d, cx.sc1(pd.n_pad));
    if (et == 0) {
      // every Hq load of this CTA has consumed its flags: the last CTA clears them for the next layer
      __threadfence();
      if (atomicAdd(pd.dep_done, 1) == (int)gridDim.x - 1) {
        for (int t = 0; t < pd.dep_tiles; ++t) const_cast<int*>(pd.dep_flags)[t] = 0;
        __threadfence();
        *pd.dep_done = 0;
      }
      *cx.epi_done_ptr() = 1;
      if (pd.trace && span_d >= 0) pd.trace[(size_t)span_d * 16 + 10] = globaltimer();
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) { tc_fence_after(); tmem_dealloc(cx.tmem_base, kTmemCols); }
}

namespace {
size_t smem_bytes_of(const GemmParams& p) { return (size_t)p.num_stages * p.slot_bytes + 1024 + 256 + 20 * (size_t)p.n_pad; }

cudaError_t set_attrs() {
  static bool done = false;
  if (done) return cudaSuccess;
  cudaError_t e = cudaFuncSetAttribute(spense_gemm_kernel<0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemMax);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(spense_gemm_kernel<0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemMax);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(spense_gemm_kernel<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemMax);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(spense_mlp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemMax);
  done = e == cudaSuccess;
  return e;
}
}  // namespace

int launch_gemm(const GemmParams& p, const CUtensorMap& tmap_b, bool pdl, cudaStream_t stream) {
  if (set_attrs() != cudaSuccess) return SPENSE_ERR_CUDA;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(p.n_spans * p.nb));
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = smem_bytes_of(p);
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  const cudaError_t e = p.mode == 1     ? cudaLaunchKernelEx(&cfg, spense_gemm_kernel<1, false>, p, tmap_b)
                        : p.amax_part ? cudaLaunchKernelEx(&cfg, spense_gemm_kernel<0, true>, p, tmap_b)
                                      : cudaLaunchKernelEx(&cfg, spense_gemm_kernel<0, false>, p, tmap_b);
  return e == cudaSuccess ? SPENSE_OK : SPENSE_ERR_CUDA;
}

int launch_mlp(const GemmParams& pg, const CUtensorMap& tmap_x, const GemmParams& pd, const CUtensorMap& tmap_hq,
               cudaStream_t stream) {
  if (set_attrs() != cudaSuccess) return SPENSE_ERR_CUDA;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(pg.n_spans > pd.n_spans ? pg.n_spans : pd.n_spans));
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = smem_bytes_of(pg);
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  const cudaError_t e = cudaLaunchKernelEx(&cfg, spense_mlp_kernel, pg, tmap_x, pd, tmap_hq);
  return e == cudaSuccess ? SPENSE_OK : SPENSE_ERR_CUDA;
}

}  // namespace spense
