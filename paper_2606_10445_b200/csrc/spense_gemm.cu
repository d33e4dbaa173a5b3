// Spense hybrid sparse-dense FP8 GEMM for sm_100a (tcgen05 + TMEM + TMA / bulk copy).
//
// One kernel template, two instances:
//   MODE 0  gate_up : output-split.  Pair tile = 128 rows of W_gate + the same 128 rows
//                     of W_up; tiles below I_s are 2:4 compressed (tcgen05.mma.sp), the rest dense
//                     (tcgen05.mma).  Epilogue: scales -> SiLU(g)*u (Eq. 4) -> E4M3.
//   MODE 1  down    : input-split.  Pair tile = 2 x 128 rows of W_down; the K loop runs
//                     the sparse stages and then the dense stages INTO THE SAME TMEM ACCUMULATOR.
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
// Flags hold the epoch of the launch (a device-side counter in the workspace), so nothing has to be
// reset between launches and CUDA-graph replays see fresh values.
// Span i runs on CTA n_spans-1-i.  CTAs of one launch wait for each other, so all n_spans <= #SM CTAs
// must be co-resident: 1 CTA/SM by construction (shared memory), the device must not be shared.
//
// Warp roles (640 threads): warp 0 producer (bulk copy of the weight stage + TMA of the activation
// tile), warp 1 MMA issuer, warp 2 TMEM allocator, warps 4-19 epilogue (TMEM lane quadrant = warp & 3,
// quarter of the token columns = (warp - 4) >> 2): the last tile's epilogue is exposed at the end of
// every CTA and is instruction-issue bound, so it gets 4 warps per scheduler.  Rarely executed code is kept rolled: the kernel is
// latency-sensitive at its tail and instruction-cache misses on cold paths showed up in the timeline.
#include <cuda_bf16.h>

#include "spense_internal.cuh"

namespace spense {

namespace {

// SiLU(g) * u on the hardware exp2 / reciprocal units: branch-free, relative error ~1e-6 (far inside
// the GLU tolerance).  ex2 of a very negative g overflows to +inf -> rcp gives 0 -> h = -0 * u.
__device__ __forceinline__ float silu_mul(float g, float u) {
  float e, r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(-1.4426950408889634f * g));
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(1.0f + e));
  return g * r * u;
}

// a / b from the correctly rounded reciprocal r = RN(1/b) and two FMAs (Markstein): branch-free and
// correctly rounded wherever the quotient is a normal number -- all the E4M3 cast after it can see.
__device__ __forceinline__ float div_by(float a, float b, float r) {
  const float q0 = a * r;
  const float rem = fmaf(-q0, b, a);
  return fmaf(rem, r, q0);
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

constexpr int kEpiThreads = 512;                 // 16 epilogue warps: 4 per TMEM lane quadrant
constexpr int kThreads = 128 + kEpiThreads;
constexpr int kTmemCols = 512;
constexpr int kMetaCol = 480;   // 2 buffers x 16 columns of 2:4 metadata

// One output element (token m, weight row r of pair tile `tile`): scales, GLU + requant, or the Y store.
// sc holds one float4 per token column: MODE 0 {s_x*s_gate, s_x*s_up, s_h, RN(1/s_h)}, MODE 1 {s_h*s_down, -, -, -}.
template <int MODE>
__device__ __forceinline__ void finish(const GemmParams& p, const float4* sc, int tile, int r, int m, float f0, float f1) {
  const float4 k = sc[m];
  if (MODE == 0) {
    const float g = f0 * k.x;
    const float u = f1 * k.y;
    const float h = silu_mul(g, u);
    const float qv = div_by(h, k.z, k.w);
    const size_t o = (size_t)m * p.ld_out + tile * 128 + r;
    if (p.h_f32) p.h_f32[o] = h;
    p.hq[o] = (uint8_t)(to_e4m3x2(qv, 0.0f) & 0xFFu);
  } else {
    const int out_row = tile * 256 + r;
    const float y0 = f0 * k.x, y1 = f1 * k.x;
    const size_t o = (size_t)m * p.ld_out + out_row;
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


// A segment = consecutive stages of ONE pair tile accumulated into one TMEM buffer.  The producer is the only
// role that walks the schedule (static span, then dynamically claimed tail chunks); it describes every
// segment in a small shared-memory FIFO that the MMA issuer and the epilogue warps follow.
enum { kFixWhole = 0, kFixOwnerAdd = 1, kFixDumpFlag = 2, kFixDumpCount = 3, kFixStop = 4 };
struct Seg {
  int seq;        // entry index + 1, written last (release): the entry is valid once it matches
  int tile;
  int j0, n;      // first stage inside the tile, number of stages
  int ns_tile;    // stages [0, ns_tile) of this tile are 2:4 sparse
  int fix;        // kFix*
  int a;          // OwnerAdd / DumpFlag: flag index; DumpCount: reduced-tile index
  int b;          // partial slot (OwnerAdd: the partner's, Dump*: ours)
};
constexpr int kSegFifo = 16;   // the producer is at most ring + 1 + 2 accumulators (<= 11 segments) ahead of the epilogue
static_assert(256 + kSegFifo * 32 + 64 == kSmemTailBytes, "shared-memory tail layout");

__device__ __forceinline__ int ld_acquire_cta_shared(const int* p) {
  int v;
  asm volatile("ld.acquire.cta.shared::cta.s32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_cta_shared(int* p, int v) {
  asm volatile("st.release.cta.shared::cta.s32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}
__device__ __forceinline__ Seg wait_seg(const Seg* fifo, int idx) {
  const Seg* e = fifo + (idx & (kSegFifo - 1));
  while (ld_acquire_cta_shared(&e->seq) != idx + 1) {}
  return *e;
}

// stages of pair tile t, and the byte offset of its stage j inside the section
template <int MODE>
__device__ __forceinline__ void tile_shape(const GemmParams& p, int t, int& ns, int& nd) {
  if (MODE == 0) {
    if (t < p.tiles_sparse) { ns = p.ns; nd = 0; } else { ns = 0; nd = p.nd; }
  } else {
    ns = p.ns; nd = p.nd;
  }
}
template <int MODE>
__device__ __forceinline__ size_t stage_offset(const GemmParams& p, int t, int j) {
  if (MODE == 0) {
    if (t < p.tiles_sparse) return ((size_t)t * p.ns + j) * kSparseStageBytes;
    return (size_t)p.tiles_sparse * p.ns * kSparseStageBytes + ((size_t)(t - p.tiles_sparse) * p.nd + j) * kDenseStageBytes;
  }
  const size_t base = (size_t)t * ((size_t)p.ns * kSparseStageBytes + (size_t)p.nd * kDenseStageBytes);
  return base + (j < p.ns ? (size_t)j * kSparseStageBytes
                          : (size_t)p.ns * kSparseStageBytes + (size_t)(j - p.ns) * kDenseStageBytes);
}
// linear stage index of the first stage of tile t (the order of span_begin)
template <int MODE>
__device__ __forceinline__ int tile_first(const GemmParams& p, int t) {
  if (MODE == 0) return t < p.tiles_sparse ? t * p.ns : p.tiles_sparse * p.ns + (t - p.tiles_sparse) * p.nd;
  return t * (p.ns + p.nd);
}
// tail chunk q -> (tile, j0, n)
template <int MODE>
__device__ __forceinline__ void tail_chunk(const GemmParams& p, int q, int& tile, int& j0, int& n) {
  int cpt, per, t_off = 0;
  if (MODE == 0) {
    const int qs = p.tail_ts * p.tail_cpt_s;
    if (q < qs) { cpt = p.tail_cpt_s; per = p.ns; }
    else { q -= qs; cpt = p.tail_cpt_d; per = p.nd; t_off = p.tail_ts; }
  } else {
    cpt = p.tail_cpt_s; per = p.ns + p.nd;
  }
  const int tt = q / cpt;
  tile = p.tail_tile0 + t_off + tt;
  j0 = (q - tt * cpt) * p.tail_cs;
  n = min(p.tail_cs, per - j0);
}

}  // namespace

template <int MODE>
__global__ void __launch_bounds__(kThreads, 1)
spense_gemm_kernel(const __grid_constant__ GemmParams p, const __grid_constant__ CUtensorMap tmap_b) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;

  const int S = p.num_stages;
  // after the stage ring: 256 B of barriers | one float4 of scales per token column | segment FIFO | misc
  const uint32_t ring_bytes = (uint32_t)S * p.slot_bytes;
  const uint32_t bar_base = smem_base + ring_bytes;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (8 + s); };
  auto accf_bar = [&](int b) { return bar_base + 8u * (16 + b); };
  auto acce_bar = [&](int b) { return bar_base + 8u * (18 + b); };
  const uint32_t red_bar = bar_base + 8u * 22;   // two barriers: task-reduction double buffer
  const uint32_t tmem_slot = bar_base + 8u * 20;
  uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
  volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(smem_gen + ring_bytes + 8 * 20);
  volatile int* epoch_ptr = reinterpret_cast<volatile int*>(smem_gen + ring_bytes + 8 * 21);
  float4* sc = reinterpret_cast<float4*>(smem_gen + ring_bytes + 256);
  Seg* fifo = reinterpret_cast<Seg*>(smem_gen + ring_bytes + 256 + 16 * p.n_pad);
  volatile int* task_ptr = reinterpret_cast<volatile int*>(fifo + kSegFifo);   // 2 ints: task broadcast (double buffered)

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmap_b);
    for (int s = 0; s < S; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(accf_bar(b), 1); mbar_init(acce_bar(b), kEpiThreads); }
    mbar_init(red_bar, 1);
    mbar_init(red_bar + 8, 1);
    fence_barrier_init();
  }
  if (warp == 3 && lane < kSegFifo) fifo[lane].seq = 0;
  if (warp == 2) tmem_alloc(tmem_slot, kTmemCols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;

  // let the next kernel of the stream start its own prologue (it waits for us in pdl_wait)
  pdl_launch_dependents();

  const int span = p.n_spans - 1 - (int)blockIdx.x;
  const int sb = p.span_begin[span];
  const int se = p.span_begin[span + 1];
  const uint32_t b_tile_bytes = (uint32_t)p.n_pad * 128u;
  if (p.trace && threadIdx.x == 0) {
    uint32_t smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    p.trace[(size_t)span * 16 + 0] = globaltimer(); p.trace[(size_t)span * 16 + 14] = smid;
  }

  if (warp == 0) {
    // ===================== producer =====================
    if (lane == 0) {
      const uint64_t pol_w = policy_evict_first();
      const uint64_t pol_a = policy_evict_last();
      int it = 0, seg_idx = 0, n_issued_static = 0;
      bool pdl_done = false;
      uint32_t info[8];                                    // stages issued before pdl_wait: K coordinate | sparse << 31
      auto load_b = [&](int slot, uint32_t inf) {
        const uint32_t b_dst = smem_base + (uint32_t)slot * p.slot_bytes + kSparseStageBytes;
        const int k0 = (int)(inf & 0x7FFFFFFFu);
        tma_load_2d(b_dst, &tmap_b, k0, 0, full_bar(slot), pol_a);
        if (inf >> 31) tma_load_2d(b_dst + b_tile_bytes, &tmap_b, k0 + 128, 0, full_bar(slot), pol_a);
      };
      // Weights never depend on the previous kernel of the stream, activations do: fill the whole ring with
      // weight stages, then wait for the previous kernel and add the activation tiles.
      auto flush = [&]() {
        trace(p, span, 1);
        pdl_wait();
        pdl_done = true;
#pragma unroll
        for (int k = 0; k < 8; ++k)
          if (k < it) load_b(k, info[k]);
      };
      auto push_seg = [&](int tile, int j0, int n, int ns_tile, int fix, int a, int b) {
        Seg* e = fifo + (seg_idx & (kSegFifo - 1));
        e->tile = tile; e->j0 = j0; e->n = n; e->ns_tile = ns_tile; e->fix = fix; e->a = a; e->b = b;
        st_release_cta_shared(&e->seq, ++seg_idx);
      };
      auto issue = [&](int tile, int j, int ns_tile) {
        if (!pdl_done && it == S) flush();
        const bool sp = j < ns_tile;
        const uint32_t wb = sp ? (uint32_t)kSparseStageBytes : (uint32_t)kDenseStageBytes;
        const uint32_t inf = (uint32_t)(sp ? j * kSparseStageK : p.dense_k0 + (j - ns_tile) * kDenseStageK) | (sp ? 0x80000000u : 0u);
        const int slot = it % S;
        if (it >= S) mbar_wait(empty_bar(slot), ((uint32_t)(it / S) & 1u) ^ 1u);
        mbar_expect_tx(full_bar(slot), wb + (sp ? 2u : 1u) * b_tile_bytes);
        bulk_g2s(smem_base + (uint32_t)slot * p.slot_bytes, p.section + stage_offset<MODE>(p, tile, j), wb, full_bar(slot), pol_w);
        if (pdl_done) {
          load_b(slot, inf);
        } else {
#pragma unroll
          for (int k = 0; k < 8; ++k)
            if (k == it) info[k] = inf;
        }
        ++it;
      };

      // ---- static span: segments per tile
      int tile;
      if (MODE == 0) {
        const int sparse_total = p.tiles_sparse * p.ns;
        tile = sb < sparse_total ? sb / p.ns : p.tiles_sparse + (sb - sparse_total) / p.nd;
      } else {
        tile = sb / (p.ns + p.nd);
      }
      int first = tile_first<MODE>(p, tile);
      const int claim_at = max(sb, se - 2);
      int q_next = p.n_tail_chunks;                        // claimed tail chunk (claimed a little ahead of need)
#pragma unroll 1
      for (int s = sb; s < se;) {
        int ns, nd;
        tile_shape<MODE>(p, tile, ns, nd);
        const int tile_end = first + ns + nd;
        const int seg_end = min(se, tile_end);
        int a = span, b = span;
        while (p.span_begin[a] > first) --a;
        while (b + 1 < p.n_spans && p.span_begin[b + 1] < tile_end) ++b;
        int fix = kFixWhole, fa = 0, fb = 0;
        if (b == a + 1) {
          fix = span == a ? kFixOwnerAdd : kFixDumpFlag;   // span b starts inside the tile: its first segment
          fa = b * 2; fb = b * 2;
        } else if (b > a + 1) {
          fix = kFixDumpCount;
          for (int r = 0; r < p.n_red_static; ++r)
            if (p.red[r].tile == tile) fa = r;
          fb = span * 2 + (sb >= first ? 0 : 1);
        }
        push_seg(tile, s - first, seg_end - s, ns, fix, fa, fb);
#pragma unroll 1
        for (; s < seg_end; ++s) {
          if (s == claim_at && p.n_tail_chunks > 0) {
            if (!pdl_done) flush();                        // the queue counter belongs to the previous kernel until then
            q_next = atomicAdd(p.ws_ctrl + kCtrlChunk, 1);
          }
          issue(tile, s - first, ns);
        }
        ++tile;
        first = tile_end;
      }
      n_issued_static = it;
      if (!pdl_done) flush();
      trace(p, span, 2);
      // ---- dynamic tail: claim chunks until the queue is empty
#pragma unroll 1
      for (int q = q_next; q < p.n_tail_chunks; q = q_next) {
        q_next = atomicAdd(p.ws_ctrl + kCtrlChunk, 1);
        int t, j0, n, ns, nd;
        tail_chunk<MODE>(p, q, t, j0, n);
        tile_shape<MODE>(p, t, ns, nd);
        push_seg(t, j0, n, ns, kFixDumpCount, p.n_red_static + (t - p.tail_tile0), 2 * p.n_spans + q);
#pragma unroll 1
        for (int j = j0; j < j0 + n; ++j) issue(t, j, ns);
      }
      push_seg(0, 0, 0, 0, kFixStop, 0, 0);
      if (p.trace) { p.trace[(size_t)span * 16 + 12] = globaltimer(); p.trace[(size_t)span * 16 + 11] = n_issued_static | ((it - n_issued_static) << 16); }
      // HBM goes idle while the CTAs run their fix-up tails: use that time to pull the first stages of
      // the NEXT kernel's span into L2 (the next GEMM of this layer / the next layer's gate_up).
      if (p.next_base) {
        const uint8_t* nb = p.next_base + (size_t)p.next_off[span];
        const uint32_t bytes = p.next_len[span];
#pragma unroll 1
        for (uint32_t o = 0; o < bytes; o += 32768u) {
          const uint32_t chunk = bytes - o < 32768u ? bytes - o : 32768u;
          asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(nb + o), "r"(chunk) : "memory");
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0) {
      const uint32_t idesc_d = (1u << 4) | ((uint32_t)(p.n_pad >> 3) << 17) | ((128u >> 4) << 24);
      const uint32_t idesc_s = idesc_d | (1u << 2);
      int it = 0;
#pragma unroll 1
      for (int seg = 0;; ++seg) {
        const Seg e = wait_seg(fifo, seg);
        if (e.fix == kFixStop) break;
        const int buf = seg % p.num_acc_bufs;
        const uint32_t use = (uint32_t)(seg / p.num_acc_bufs);
        mbar_wait(acce_bar(buf), (use & 1u) ^ 1u);         // epilogue has drained this accumulator
        tc_fence_after();
        const uint32_t d0 = tmem_base + (uint32_t)(buf * 2 * p.acc_stride);
        const uint32_t d1 = d0 + (uint32_t)p.acc_stride;
        uint32_t acc = 0;
#pragma unroll 1
        for (int j = e.j0; j < e.j0 + e.n; ++j, ++it) {
          const int slot = it % S;
          const uint32_t ph = (uint32_t)(it / S) & 1u;
          mbar_wait(full_bar(slot), ph);
          tc_fence_after();
          if (it == 0) trace(p, span, 3);
          const uint32_t a0 = smem_base + (uint32_t)slot * p.slot_bytes;
          const uint32_t a1 = a0 + kOperandBytes;
          const uint32_t b0 = a0 + kSparseStageBytes;
          if (j < e.ns_tile) {
            const uint32_t e_base = tmem_base + kMetaCol + (uint32_t)(it & 1) * 16u;
            const uint32_t m0 = a0 + 2 * kOperandBytes;   // A0 meta: 2 atoms of 2 KB, then A1 meta
#pragma unroll
            for (int a = 0; a < 4; ++a)                   // 4 atoms: (A0,k0) (A0,k1) (A1,k0) (A1,k1)
              tc_cp_128x128b(e_base + 4u * a, make_desc(m0 + 2048u * a, 0, 128, kLayoutNone));
#pragma unroll
            for (int k = 0; k < 4; ++k) {                 // 4 sparse MMAs of K = 64 logical (32 B of A, 64 B of B)
              const uint64_t bd = make_desc(b0 + (uint32_t)(k >> 1) * b_tile_bytes + (uint32_t)(k & 1) * 64u, 16, 1024, kLayoutSW128);
              mma_f8_sparse(d0, make_desc(a0 + 32u * k, 16, 1024, kLayoutSW128), bd, e_base + 2u * k, idesc_s, acc);
              mma_f8_sparse(d1, make_desc(a1 + 32u * k, 16, 1024, kLayoutSW128), bd, e_base + 8u + 2u * k, idesc_s, acc);
              acc = 1;
            }
          } else {
#pragma unroll
            for (int k = 0; k < 4; ++k) {                 // 4 dense MMAs of K = 32
              const uint64_t bd = make_desc(b0 + 32u * k, 16, 1024, kLayoutSW128);
              mma_f8_dense(d0, make_desc(a0 + 32u * k, 16, 1024, kLayoutSW128), bd, idesc_d, acc);
              mma_f8_dense(d1, make_desc(a1 + 32u * k, 16, 1024, kLayoutSW128), bd, idesc_d, acc);
              acc = 1;
            }
          }
          tc_commit(empty_bar(slot));                     // smem slot free once these MMAs have read it
        }
        tc_commit(accf_bar(buf));                         // accumulator complete for this segment
      }
      trace(p, span, 4);
    }
  }
  else if (warp >= 4) {
    // ===================== epilogue (16 warps) =====================
    // warp & 3 selects the TMEM lane quadrant, (warp - 4) >> 2 the quarter of the token columns.
    const int q = warp & 3;
    const int row = q * 32 + lane;                         // accumulator lane = weight row inside the tile
    const int et = threadIdx.x - 128;                      // 0..511
    const int cols_used = min(p.n_pad, (p.M + 7) & ~7);    // token columns holding real tokens, rounded to the TMEM load width
    const int cols_per = (((p.n_pad + 3) >> 2) + 7) & ~7;  // columns per warp: a quarter, rounded to the TMEM load width
    const int c_begin = ((warp - 4) >> 2) * cols_per;
    const int c_end = min(c_begin + cols_per, cols_used);
    const size_t part_floats = (size_t)2 * p.n_pad * 128;  // one partial: [mat][col][row]

    // scales, the workspace and the epoch word may be produced / still in use by the previous kernel
    pdl_wait();
    if (et < p.n_pad) {
      const int m = et < p.M ? et : p.M - 1;
      float4 k = make_float4(0.f, 0.f, 0.f, 0.f);
      if (MODE == 0) {
        const float sx = __ldg(p.s_act + m);
        const float sh = __ldg(p.s_h + (size_t)m * p.sh_stride);
        k = make_float4(sx * p.w_scale0, sx * p.w_scale1, sh, __frcp_rn(sh));
      } else {
        k.x = __ldg(p.s_act + (size_t)m * p.sh_stride) * p.w_scale0;
      }
      sc[et] = k;
    }
    if (et == kEpiThreads - 1) {
      // Epoch of this launch = epoch word + 1.  Every CTA reads the word BEFORE it counts itself; the CTA
      // that counts last therefore knows all have read it and advances it for the next launch.
      const int e = ld_acquire(p.ws_ctrl + kCtrlEpoch);
      *epoch_ptr = e + 1;
      if (atomicAdd(p.ws_ctrl + kCtrlStarted, 1) == p.n_spans - 1) {
        p.ws_ctrl[kCtrlStarted] = 0;
        st_release(p.ws_ctrl + kCtrlEpoch, e + 1);
      }
    }
    epi_sync();
    const int epoch = *epoch_ptr;                          // flag value of THIS launch (never equals a stale flag)

#pragma unroll 1
    for (int seg = 0;; ++seg) {
      const Seg e = wait_seg(fifo, seg);
      if (e.fix == kFixStop) break;
      const int buf = seg % p.num_acc_bufs;
      const uint32_t use = (uint32_t)(seg / p.num_acc_bufs);
      mbar_wait(accf_bar(buf), use & 1u);
      tc_fence_after();
      if (et == 0) trace(p, span, seg == 0 ? 5 : 7);
      const uint32_t t0 = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * 2 * p.acc_stride);
      const uint32_t t1 = t0 + (uint32_t)p.acc_stride;

      if (e.fix == kFixWhole || e.fix == kFixOwnerAdd) {
        // the whole tile is ours, or we own a tile whose tail the next span has (usually long ago) dumped
        const bool add = e.fix == kFixOwnerAdd;
        const float* part = p.partials + (size_t)e.b * part_floats;
        if (add) {
          while (ld_acquire(p.flags + e.a) != epoch) {}   // warp-uniform address: one request per warp
          if (et == 0) trace(p, span, 8);
        }
#pragma unroll 1
        for (int c = c_begin; c < c_end; c += 8) {
          float a0[8], a1[8];
          if (add) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              a0[i] = __ldcg(part + (size_t)(c + i) * 128 + row);
              a1[i] = __ldcg(part + (size_t)(p.n_pad + c + i) * 128 + row);
            }
          }
          uint32_t v0[8], v1[8];
          tmem_ld8(t0 + c, v0);
          tmem_ld8(t1 + c, v1);
          tmem_ld_wait();
          float f0[8], f1[8];
#pragma unroll
          for (int i = 0; i < 8; ++i) { f0[i] = __uint_as_float(v0[i]); f1[i] = __uint_as_float(v1[i]); }
          if (add) {
#pragma unroll
            for (int i = 0; i < 8; ++i) { f0[i] += a0[i]; f1[i] += a1[i]; }
          }
#pragma unroll
          for (int i = 0; i < 8; ++i)
            if (c + i < p.M) finish<MODE>(p, sc, e.tile, row, c + i, f0[i], f1[i]);
        }
        tc_fence_before();
        mbar_arrive(acce_bar(buf));
      } else {
        // part of a split tile that others finish: dump the raw fp32 partial [mat][col][row] and publish it
        float* slot = p.partials + (size_t)e.b * part_floats;
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
        mbar_arrive(acce_bar(buf));
        epi_sync();                                        // all partial stores issued (CTA scope) ...
        if (et == 0) {                                     // ... one gpu-scope release publishes them (cumulativity)
          if (e.fix == kFixDumpFlag) st_release(p.flags + e.a, epoch);
          else asm volatile("red.release.gpu.global.add.s32 [%0], 1;" ::"l"(p.tile_cnt + e.a) : "memory");
        }
      }
      if (et == 0) trace(p, span, 6);
    }

    // ---- task queue: tiles split into more than two partials (groups of static spans, tail tiles).  A task
    // = (reduced tile, slice of its token columns): wait until all partials of the tile have arrived, add them
    // in partial order (deterministic) and run the epilogue.  Tasks are claimed dynamically; every MMA of this
    // CTA is complete here, so the stage ring is free: its two halves double-buffer the partial slices.
    if (et == 0) trace(p, span, 9);
    const int n_tasks = p.n_red * p.red_slices;
    if (n_tasks > 0) {
      const uint32_t half_bytes = (ring_bytes >> 1) & ~1023u;
      int k = 0;                                           // staged chunks so far (buffer = k & 1)
#pragma unroll 1
      for (int ti = 0;; ++ti) {
        if (et == 0) task_ptr[ti & 1] = atomicAdd(p.ws_ctrl + kCtrlTask, 1);
        epi_sync();
        const int task = task_ptr[ti & 1];
        if (task >= n_tasks) break;
        const int r = task / p.red_slices, sl = task - r * p.red_slices;
        const RedEntry re = p.red[r];
        const int n = re.n_seg;
        const int m0 = (int)(((long long)sl * p.M) / p.red_slices), m1 = (int)(((long long)(sl + 1) * p.M) / p.red_slices);
        if (m0 == m1) continue;
        const bool is_tail = r >= p.n_red_static;
        const int first = tile_first<MODE>(p, re.tile);
        while (ld_acquire(p.tile_cnt + r) < n) {}          // warp-uniform address
        asm volatile("fence.proxy.async.global;" ::: "memory");   // others' generic-proxy stores -> our async-proxy reads
        int ccm = (int)(half_bytes / ((uint32_t)n * 1024u));
        ccm = ccm < 1 ? 1 : ccm;
#pragma unroll 1
        for (int mc = m0; mc < m1; mc += ccm, ++k) {
          const int cc = min(ccm, m1 - mc);
          const uint32_t bar = red_bar + 8u * (uint32_t)(k & 1);
          const uint32_t dst = smem_base + (uint32_t)(k & 1) * half_bytes;
          if (et == 0) mbar_expect_tx(bar, (uint32_t)n * 2u * (uint32_t)cc * 512u);
#pragma unroll 1
          for (int i = et; i < 2 * n; i += kEpiThreads) {
            const int qi = i >> 1, mat = i & 1;
            int slot_idx;
            if (is_tail) {
              slot_idx = 2 * p.n_spans + re.first + qi;
            } else {
              const int qs = re.first + qi;
              slot_idx = qs * 2 + (p.span_begin[qs] >= first ? 0 : 1);
            }
            const float* src = p.partials + (size_t)slot_idx * part_floats + ((size_t)mat * p.n_pad + mc) * 128;
            bulk_g2s(dst + (uint32_t)(i * cc) * 512u, src, (uint32_t)cc * 512u, bar, policy_evict_first());
          }
          mbar_wait(bar, (uint32_t)(k >> 1) & 1u);
          if (et == 0) trace(p, span, 15);
          const float* sl_f = reinterpret_cast<const float*>(smem_gen + (size_t)(k & 1) * half_bytes);
          const int rrow = et & 127;
#pragma unroll 1
          for (int c = et >> 7; c < cc; c += kEpiThreads >> 7) {
            float f0 = 0.0f, f1 = 0.0f;
#pragma unroll 4
            for (int qi = 0; qi < n; ++qi) {               // fixed partial order: deterministic
              f0 += sl_f[((size_t)(2 * qi) * cc + c) * 128 + rrow];
              f1 += sl_f[((size_t)(2 * qi + 1) * cc + c) * 128 + rrow];
            }
            finish<MODE>(p, sc, re.tile, rrow, mc + c, f0, f1);
          }
          // the buffer used now is overwritten two chunks later: order these reads before those async writes
          fence_proxy_async();
          epi_sync();
        }
      }
    }
    // ---- the CTA that finishes last resets the queue counters for the next launch
    if (et == 0) {
      __threadfence();
      if (atomicAdd(p.ws_ctrl + kCtrlDone, 1) == p.n_spans - 1) {
        p.ws_ctrl[kCtrlChunk] = 0;
        p.ws_ctrl[kCtrlTask] = 0;
        for (int r = 0; r < p.n_red; ++r) p.tile_cnt[r] = 0;
        __threadfence();
        p.ws_ctrl[kCtrlDone] = 0;
      }
      if (p.trace) { p.trace[(size_t)span * 16 + 10] = globaltimer(); }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) { tc_fence_after(); tmem_dealloc(tmem_base, kTmemCols); }
}

int launch_gemm(const GemmParams& p, const CUtensorMap& tmap_b, bool pdl, cudaStream_t stream) {
  const size_t smem = (size_t)p.num_stages * p.slot_bytes + 1024 + kSmemTailBytes + 16 * (size_t)p.n_pad;
  static bool attr_set = false;
  if (!attr_set) {
    if (cudaFuncSetAttribute(spense_gemm_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, 232448) != cudaSuccess ||
        cudaFuncSetAttribute(spense_gemm_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 232448) != cudaSuccess)
      return SPENSE_ERR_CUDA;
    attr_set = true;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)p.n_spans);
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  const cudaError_t e = p.mode == 0 ? cudaLaunchKernelEx(&cfg, spense_gemm_kernel<0>, p, tmap_b)
                                    : cudaLaunchKernelEx(&cfg, spense_gemm_kernel<1>, p, tmap_b);
  return e == cudaSuccess ? SPENSE_OK : SPENSE_ERR_CUDA;
}

}  // namespace spense
