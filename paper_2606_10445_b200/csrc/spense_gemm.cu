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

// Position in the linear stage sequence: pair tile, stage inside the tile, stages of the tile.
struct Cursor {
  int tile, j, ns, nd, first;   // first = linear index of the tile's first stage
};

// The only place with integer divisions (one copy, called once per role).
template <int MODE>
__device__ __noinline__ Cursor cursor_at(const GemmParams& p, int s, unsigned long long* byte_off) {
  Cursor c;
  size_t off;
  if (MODE == 0) {
    const int sparse_total = p.tiles_sparse * p.ns;
    if (s < sparse_total) {
      c.tile = s / p.ns;
      c.first = c.tile * p.ns;
      c.ns = p.ns; c.nd = 0;
      off = (size_t)s * kSparseStageBytes;
    } else {
      const int td = (s - sparse_total) / p.nd;
      c.tile = p.tiles_sparse + td;
      c.first = sparse_total + td * p.nd;
      c.ns = 0; c.nd = p.nd;
      off = (size_t)sparse_total * kSparseStageBytes + (size_t)(s - sparse_total) * kDenseStageBytes;
    }
    c.j = s - c.first;
  } else {
    const int per = p.ns + p.nd;
    c.tile = s / per;
    c.first = c.tile * per;
    c.ns = p.ns; c.nd = p.nd;
    c.j = s - c.first;
    off = (size_t)c.tile * ((size_t)p.ns * kSparseStageBytes + (size_t)p.nd * kDenseStageBytes);
    off += c.j < c.ns ? (size_t)c.j * kSparseStageBytes
                      : (size_t)c.ns * kSparseStageBytes + (size_t)(c.j - c.ns) * kDenseStageBytes;
  }
  *byte_off = off;
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
    const size_t o = (size_t)m * p.ld_out + tile * 128 + r;
    if (p.amax_part) {
      // dynamic requant: keep h in fp32 and track max|h| per token; the scale does not
      // exist yet, spense_requant turns h into Hq once every tile is done.  Called warp-uniformly in m.
      p.h_f32[o] = h;
      const int mx = __reduce_max_sync(0xffffffffu, __float_as_int(fabsf(h)));   // |h| >= 0: int order == float order
      if ((threadIdx.x & 31) == 0) atomicMax(reinterpret_cast<int*>(const_cast<float4*>(sc) + m) + 2, mx);
      return;
    }
    const float qv = div_by(h, k.z, k.w);
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

// A tile shared by more than two spans [a, b]: reduced at the end of the span (reduce-scatter).
struct Group { int a, b, tile, first; };

}  // namespace

template <int MODE>
__global__ void __launch_bounds__(kThreads, 1)
spense_gemm_kernel(const __grid_constant__ GemmParams p, const __grid_constant__ CUtensorMap tmap_b) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;

  const int S = p.num_stages;
  // barriers live after the stage ring
  const uint32_t ring_bytes = (uint32_t)S * p.slot_bytes;
  const uint32_t bar_base = smem_base + ring_bytes;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (8 + s); };
  auto accf_bar = [&](int b) { return bar_base + 8u * (16 + b); };
  auto acce_bar = [&](int b) { return bar_base + 8u * (18 + b); };
  const uint32_t red_bar = bar_base + 8u * 22;
  const uint32_t tmem_slot = bar_base + 8u * 20;
  uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
  volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(smem_gen + ring_bytes + 8 * 20);
  volatile int* epoch_ptr = reinterpret_cast<volatile int*>(smem_gen + ring_bytes + 8 * 21);
  volatile int* epi_done_ptr = reinterpret_cast<volatile int*>(smem_gen + ring_bytes + 8 * 23);   // epilogue finished (stops the paced prefetch)

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmap_b);
    for (int s = 0; s < S; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(accf_bar(b), 1); mbar_init(acce_bar(b), kEpiThreads); }
    mbar_init(red_bar, 1);
    *epi_done_ptr = 0;
    fence_barrier_init();
  }
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
    p.trace[(size_t)span * 16 + 0] = globaltimer(); p.trace[(size_t)span * 16 + 12] = globaltimer(); p.trace[(size_t)span * 16 + 14] = smid;
  }

  if (warp == 0) {
    // ===================== producer =====================
    if (lane == 0) {
      const uint64_t pol_w = policy_evict_first();
      const uint64_t pol_a = policy_evict_last();
      unsigned long long off;
      Cursor c = cursor_at<MODE>(p, sb, &off);
      const uint8_t* src = p.section + off;
      const int n = se - sb;
      const int pre = n < S ? n : S;
      uint32_t info[8];                                    // stages issued before pdl_wait: K coordinate | sparse << 31
      // gate_up -> down dependency per Hq tile (spense_mlp): tiles [dep_lo, dep_hi) are known to be stored
      int dep_lo = 0, dep_hi = 0;
      auto need_tile = [&](int t) {
        if (t < dep_lo || t > dep_hi) dep_lo = dep_hi = t;    // the K range restarted (next row tile): verify again
#pragma unroll 1
        while (dep_hi <= t) {
          const int4* f = reinterpret_cast<const int4*>(p.dep_flags + (dep_hi & ~3));
          int4 v[4];
#pragma unroll
          for (int i = 0; i < 4; ++i)
            asm volatile("ld.volatile.global.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(v[i].x), "=r"(v[i].y), "=r"(v[i].z), "=r"(v[i].w) : "l"(f + i));
          uint32_t m = 0;
#pragma unroll
          for (int i = 0; i < 4; ++i)
            m |= ((v[i].x != 0) | ((v[i].y != 0) << 1) | ((v[i].z != 0) << 2) | ((v[i].w != 0) << 3)) << (4 * i);
          m >>= dep_hi & 3;
          const int n_ready = __ffs(~m) - 1;                 // consecutive finished tiles from dep_hi on
          if (n_ready > 0) {
            dep_hi += n_ready;
            asm volatile("fence.acq_rel.gpu;" ::: "memory");
            asm volatile("fence.proxy.async.global;" ::: "memory");   // gate_up's generic-proxy stores -> our TMA reads
          }
        }
      };
      auto load_b = [&](int it, uint32_t inf) {
        const uint32_t b_dst = smem_base + (uint32_t)(it % S) * p.slot_bytes + kSparseStageBytes;
        const int k0 = (int)(inf & 0x7FFFFFFFu);
        if (MODE == 1 && p.dep_flags) {
          const int t_last = (k0 + ((inf >> 31) ? 255 : 127)) >> 7;
          need_tile(k0 >> 7);
          need_tile(t_last < p.dep_tiles ? t_last : p.dep_tiles - 1);
        }
        tma_load_2d(b_dst, &tmap_b, k0, 0, full_bar(it % S), pol_a);
        if (inf >> 31) tma_load_2d(b_dst + b_tile_bytes, &tmap_b, k0 + 128, 0, full_bar(it % S), pol_a);
      };
      // Weights never depend on the previous kernel of the stream, activations do: fill the whole ring with
      // weight stages, then wait for the previous kernel and add the activation tiles.
      auto prefetch_l2 = [&](const uint8_t* base, uint32_t bytes) {
#pragma unroll 1
        for (uint32_t o = 0; o < bytes; o += 32768u) {
          const uint32_t chunk = bytes - o < 32768u ? bytes - o : 32768u;
          asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(base + o), "r"(chunk) : "memory");
        }
      };
      auto flush = [&]() {
        trace(p, span, 1);
        if (p.self_len[span]) prefetch_l2(src + p.self_off[span], p.self_len[span]);
        if (!(MODE == 1 && p.dep_flags)) pdl_wait();
#pragma unroll
        for (int k = 0; k < 8; ++k)
          if (k < pre) load_b(k, info[k]);
      };
#pragma unroll 1
      for (int it = 0; it < n; ++it) {
        if (it == pre) flush();
        const bool sp = c.j < c.ns;
        const uint32_t wb = sp ? (uint32_t)kSparseStageBytes : (uint32_t)kDenseStageBytes;
        const uint32_t inf = (uint32_t)(sp ? c.j * kSparseStageK : p.dense_k0 + (c.j - c.ns) * kDenseStageK) | (sp ? 0x80000000u : 0u);
        const int slot = it % S;
        if (it >= pre) mbar_wait(empty_bar(slot), ((uint32_t)(it / S) & 1u) ^ 1u);
        mbar_expect_tx(full_bar(slot), wb + (sp ? 2u : 1u) * b_tile_bytes);
        bulk_g2s(smem_base + (uint32_t)slot * p.slot_bytes, src, wb, full_bar(slot), pol_w);
        if (it >= pre) {
          load_b(it, inf);
        } else {
#pragma unroll
          for (int k = 0; k < 8; ++k)
            if (k == it) info[k] = inf;
        }
        src += wb;
        if (++c.j == c.ns + c.nd) next_tile<MODE>(p, c);
      }
      if (n <= pre) flush();
      trace(p, span, 2);
      // HBM goes idle while the CTAs run their fix-up tails: use that time to pull the first stages of
      // the NEXT kernel's span into L2 (the next GEMM of this layer / the next layer's gate_up).
      // flag-gated launch: nothing above waited for the previous grid; do it once (it is long done) so that
      // "this kernel complete" still implies "everything before it complete" for the next kernel's PDL wait
      if (MODE == 1 && p.dep_flags) pdl_wait();
      if (p.next_base) {
        const uint8_t* nb = p.next_base + (size_t)p.next_off[span];
        const uint32_t bytes = p.next_len[span];
        if (p.pf_pace_ns == 0) {
          prefetch_l2(nb, bytes);
        } else {
          // paced: one 32 KB chunk per pf_pace_ns, so the queue in front of the fix-up traffic stays shallow;
          // stops when this CTA's epilogue is done (the CTA must not outlive its own work)
          long long t_next = globaltimer();
#pragma unroll 1
          for (uint32_t o = 0; o < bytes && *epi_done_ptr == 0; o += 32768u) {
            const uint32_t chunk = bytes - o < 32768u ? bytes - o : 32768u;
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(nb + o), "r"(chunk) : "memory");
            t_next += p.pf_pace_ns;
            while (globaltimer() < t_next && *epi_done_ptr == 0) __nanosleep(64);
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0) {
      const uint32_t idesc_d = (1u << 4) | ((uint32_t)(p.n_pad >> 3) << 17) | ((128u >> 4) << 24);
      const uint32_t idesc_s = idesc_d | (1u << 2);
      unsigned long long off;
      Cursor c = cursor_at<MODE>(p, sb, &off);
      int it = 0, seg = 0;
#pragma unroll 1
      for (int s = sb; s < se; ++seg) {
        const int tile_end = c.first + c.ns + c.nd;
        const int seg_end = min(se, tile_end);
        const int buf = seg % p.num_acc_bufs;
        const uint32_t use = (uint32_t)(seg / p.num_acc_bufs);
        mbar_wait(acce_bar(buf), (use & 1u) ^ 1u);         // epilogue has drained this accumulator
        tc_fence_after();
        const uint32_t d0 = tmem_base + (uint32_t)(buf * 2 * p.acc_stride);
        const uint32_t d1 = d0 + (uint32_t)p.acc_stride;
        uint32_t acc = 0;
#pragma unroll 1
        for (; s < seg_end; ++s, ++it, ++c.j) {
          const int slot = it % S;
          const uint32_t ph = (uint32_t)(it / S) & 1u;
          mbar_wait(full_bar(slot), ph);
          tc_fence_after();
          if (it == 0) trace(p, span, 3);
          const uint32_t a0 = smem_base + (uint32_t)slot * p.slot_bytes;
          const uint32_t a1 = a0 + kOperandBytes;
          const uint32_t b0 = a0 + kSparseStageBytes;
          if (c.j < c.ns) {
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
        if (s == tile_end) next_tile<MODE>(p, c);
      }
      trace(p, span, 4);
    }
  } else if (warp >= 4) {
    // ===================== epilogue (8 warps) =====================
    // warp & 3 selects the TMEM lane quadrant, (warp - 4) >> 2 the quarter of the token columns.
    const int q = warp & 3;
    const int row = q * 32 + lane;                         // accumulator lane = weight row inside the tile
    const int et = threadIdx.x - 128;                      // 0..511
    const int cols_used = min(p.n_pad, (p.M + 7) & ~7);    // token columns holding real tokens, rounded to the TMEM load width
    const int cols_per = (((p.n_pad + 3) >> 2) + 7) & ~7;  // columns per warp: a quarter, rounded to the TMEM load width
    const int c_begin = ((warp - 4) >> 2) * cols_per;
    const int c_end = min(c_begin + cols_per, cols_used);
    float4* sc = reinterpret_cast<float4*>(smem_gen + ring_bytes + 256);   // one float4 of scales per token column
    const float* stg = reinterpret_cast<const float*>(smem_gen);         // the stage ring doubles as partial staging
    const size_t part_floats = (size_t)2 * p.n_pad * 128;  // one partial: [mat][col][row]

    // scales, the workspace and the epoch word may be produced / still in use by the previous kernel; a
    // flag-gated down has its own workspace half and caller-provided scales: it starts right away
    if (!(MODE == 1 && p.dep_flags)) pdl_wait();
    if (et < p.n_pad) {
      const int m = et < p.M ? et : p.M - 1;
      float4 k = make_float4(0.f, 0.f, 0.f, 0.f);
      if (MODE == 0) {
        const float sx = __ldg(p.s_act + m);
        const float sh = p.amax_part ? 1.0f : __ldg(p.s_h + (size_t)m * p.sh_stride);
        k = make_float4(sx * p.w_scale0, sx * p.w_scale1, p.amax_part ? 0.0f : sh, __frcp_rn(sh));   // dynamic: .z = running max|h| bits
      } else {
        k.x = __ldg(p.s_act + (size_t)m * p.sh_stride) * p.w_scale0;
      }
      sc[et] = k;
    }
    if (et == kEpiThreads - 1) {
      // Epoch of this launch = epoch word + 1.  Every CTA reads the word BEFORE it counts itself; the CTA
      // that counts last therefore knows all have read it and advances it for the next launch.
      const int e = ld_acquire(p.ws_ctrl);
      *epoch_ptr = e + 1;
      if (atomicAdd(p.ws_ctrl + 1, 1) == p.n_spans - 1) {
        p.ws_ctrl[1] = 0;
        st_release(p.ws_ctrl, e + 1);
      }
    }
    epi_sync();
    const int epoch = *epoch_ptr;                          // flag value of THIS launch (never equals a stale flag)

    Group groups[2];
    int n_groups = 0;
    uint32_t red_round = 0;                                // uses of the staging barrier so far
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

      mbar_wait(accf_bar(buf), use & 1u);
      tc_fence_after();
      if (et == 0) trace(p, span, seg == 0 ? 5 : 7);
      const uint32_t t0 = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * 2 * p.acc_stride);
      const uint32_t t1 = t0 + (uint32_t)p.acc_stride;

      if (a == b || (b == a + 1 && span == a)) {
        // the whole tile is ours, or we own a tile whose tail the next span has (usually long ago) dumped
        const bool add = a != b;
        if (add) {
          // Owner of a split tile = last segment of the span: every MMA of this CTA is complete, the ring is free.
          if (et == 0) {
            const int* f = p.flags + b * 2;                // span b starts inside the tile: its first segment
            while (ld_acquire(f) != epoch) {}
            asm volatile("fence.proxy.async.global;" ::: "memory");   // partner's generic-proxy stores -> our async-proxy read
            const float* part = p.partials + (size_t)b * 2 * part_floats;
            mbar_expect_tx(red_bar, 2u * (uint32_t)cols_used * 512u);
            bulk_g2s(smem_base, part, (uint32_t)cols_used * 512u, red_bar, policy_evict_first());
            bulk_g2s(smem_base + (uint32_t)cols_used * 512u, part + (size_t)p.n_pad * 128, (uint32_t)cols_used * 512u, red_bar, policy_evict_first());
          }
          mbar_wait(red_bar, red_round & 1u);
          ++red_round;
          if (et == 0) trace(p, span, 8);
        }
        if (seg_end == se && n_groups == 0 && et == 0) *epi_done_ptr = 1;   // last epilogue of this CTA: stop prefetching now
#pragma unroll 1
        for (int c = c_begin; c < c_end; c += 8) {
          uint32_t v0[8], v1[8];
          tmem_ld8(t0 + c, v0);
          tmem_ld8(t1 + c, v1);
          tmem_ld_wait();
          float f0[8], f1[8];
#pragma unroll
          for (int i = 0; i < 8; ++i) { f0[i] = __uint_as_float(v0[i]); f1[i] = __uint_as_float(v1[i]); }
          if (add) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              f0[i] += stg[(size_t)(c + i) * 128 + row];
              f1[i] += stg[(size_t)(cols_used + c + i) * 128 + row];
            }
          }
#pragma unroll
          for (int i = 0; i < 8; ++i)
            if (c + i < p.M) finish<MODE>(p, sc, cur.tile, row, c + i, f0[i], f1[i]);
        }
        tc_fence_before();
        mbar_arrive(acce_bar(buf));
        if (MODE == 0 && p.tile_flags) {                     // Hq[:, tile] complete: all stores issued, one release
          epi_sync();
          if (et == 0) st_release(p.tile_flags + cur.tile, 1);
        }
      } else {
        // split tile, not (solely) ours to finish: dump the raw fp32 partial [mat][col][row] and publish it
        const int which = (sb >= cur.first) ? 0 : 1;       // our first segment, or our last one
        float* slot = p.partials + ((size_t)span * 2 + which) * part_floats;
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
        if (et == 0) st_release(p.flags + span * 2 + which, epoch);   // ... one gpu-scope release publishes them (cumulativity)
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
    // All MMAs of this CTA are complete here, so the stage ring is free to stage the partial slices.
#pragma unroll 1
    for (int gi = 0; gi < n_groups; ++gi) {
      const Group g = groups[gi];
      const int n = g.b - g.a + 1;
      const int j = span - g.a;
      const int m0 = (int)(((long long)j * p.M) / n), m1 = (int)(((long long)(j + 1) * p.M) / n);
      if (m1 > m0) {
        int cc_max = (int)(ring_bytes / ((uint32_t)n * 1024u));
        if (cc_max > m1 - m0) cc_max = m1 - m0;
#pragma unroll 1
        for (int mc = m0; mc < m1; mc += cc_max) {
          const int cc = min(cc_max, m1 - mc);
          if (red_round > 0) {                             // staging smem is reused: order our reads before the async writes
            fence_proxy_async();
            epi_sync();
          }
          if (et == 0) mbar_expect_tx(red_bar, (uint32_t)n * 2u * (uint32_t)cc * 512u);
          // thread i fetches matrix (i & 1) of partner (i >> 1) as soon as THAT partner has published
#pragma unroll 1
          for (int i = et; i < 2 * n; i += kEpiThreads) {
            const int qs = g.a + (i >> 1), mat = i & 1;
            const int which = (p.span_begin[qs] >= g.first) ? 0 : 1;
            while (ld_acquire(p.flags + qs * 2 + which) != epoch) {}
            asm volatile("fence.proxy.async.global;" ::: "memory");   // partner's generic-proxy stores -> our async-proxy read
            const float* src = p.partials + ((size_t)qs * 2 + which) * part_floats + ((size_t)mat * p.n_pad + mc) * 128;
            bulk_g2s(smem_base + (uint32_t)(i * cc) * 512u, src, (uint32_t)cc * 512u, red_bar, policy_evict_first());
          }
          mbar_wait(red_bar, red_round & 1u);
          ++red_round;
          if (et == 0) trace(p, span, 15);
          if (gi == n_groups - 1 && mc + cc_max >= m1 && et == 0) *epi_done_ptr = 1;
          const int rrow = et & 127;
#pragma unroll 1
          for (int c = et >> 7; c < cc; c += kEpiThreads >> 7) {
            float f0 = 0.0f, f1 = 0.0f;
#pragma unroll 4
            for (int qi = 0; qi < n; ++qi) {               // fixed span order: deterministic
              f0 += stg[((size_t)(2 * qi) * cc + c) * 128 + rrow];
              f1 += stg[((size_t)(2 * qi + 1) * cc + c) * 128 + rrow];
            }
            finish<MODE>(p, sc, g.tile, rrow, mc + c, f0, f1);
          }
        }
      }
      if (MODE == 0 && p.tile_flags) {                       // the last of the n reducers publishes the tile
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
    if (MODE == 0 && p.amax_part) {                          // this CTA's max|h| per token, for spense_requant
      epi_sync();
      if (et < p.n_pad) p.amax_part[(size_t)span * p.n_pad + et] = et < p.M ? sc[et].z : 0.0f;
    }
    if (MODE == 1 && p.dep_flags && et == 0) {             // every load of this CTA has consumed its flags
      __threadfence();
      if (atomicAdd(p.dep_done, 1) == p.n_spans - 1) {
        for (int t = 0; t < p.dep_tiles; ++t) const_cast<int*>(p.dep_flags)[t] = 0;
        __threadfence();
        *p.dep_done = 0;
      }
    }
    if (et == 0) *epi_done_ptr = 1;
    if (p.trace && et == 0) { p.trace[(size_t)span * 16 + 10] = globaltimer(); p.trace[(size_t)span * 16 + 11] = (se - sb) | (seg << 16); p.trace[(size_t)span * 16 + 13] = globaltimer(); }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) { tc_fence_after(); tmem_dealloc(tmem_base, kTmemCols); }
}

int launch_gemm(const GemmParams& p, const CUtensorMap& tmap_b, bool pdl, cudaStream_t stream) {
  const size_t smem = (size_t)p.num_stages * p.slot_bytes + 1024 + 256 + 4 * 4 * (size_t)p.n_pad;
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
