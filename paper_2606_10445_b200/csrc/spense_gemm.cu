// Spense hybrid sparse-dense FP8 GEMM for sm_100a (tcgen05 + TMEM + TMA / bulk copy).
//
// One kernel, two modes:
//   mode 0  gate_up : output-split.  Pair tile = 128 rows of W_gate + the same 128 rows
//                     of W_up; tiles below I_s are 2:4 compressed (tcgen05.mma.sp), the rest dense
//                     (tcgen05.mma).  Epilogue: scales -> SiLU(g)*u (Eq. 4) -> E4M3.
//   mode 1  down    : input-split.  Pair tile = 2 x 128 rows of W_down; the K loop runs
//                     the sparse stages and then the dense stages INTO THE SAME TMEM ACCUMULATOR.
//
// Swap-AB: only the A operand of tcgen05.mma.sp can be sparse, so weights are A (MMA-M = 128 weight
// rows) and tokens are B (MMA-N = padded token count); the accumulator holds Y^T [128 rows x tokens].
//
// Decode is weight-streaming bound, so the grid is a byte-balanced stream-K: the linear sequence of
// stage images is cut into n_spans equal-byte spans, one persistent CTA per span.  A CTA whose span
// starts inside a tile contributes an fp32 partial through an L2-resident workspace; the CTA that
// holds the tile's first stage owns the epilogue and adds the partials in fixed span order, so
// results are bitwise reproducible.  Span i runs on CTA n_spans-1-i: an owner only ever waits for
// higher-numbered spans = lower-numbered CTAs, which the hardware schedules first.
//
// Warp roles (384 threads): warp 0 producer (bulk copy of the weight stage + TMA of the activation
// tile), warp 1 MMA issuer, warp 2 TMEM allocator, warps 4-11 epilogue (TMEM lane quadrant = warp & 3,
// half of the token columns = (warp - 4) >> 2).
#include <cuda_bf16.h>

#include "spense_internal.cuh"

namespace spense {

namespace {

struct TileInfo {
  int tile;        // pair-tile index
  int first;       // linear stage index of the tile's first stage
  int ns, nd;      // sparse / dense stages of this tile
  size_t offset;   // byte offset of the tile's first stage image in the section
};

__device__ __forceinline__ TileInfo tile_of_stage(const GemmParams& p, int s) {
  TileInfo t;
  if (p.mode == 0) {
    const int sparse_total = p.tiles_sparse * p.ns;
    if (s < sparse_total) {
      t.tile = s / p.ns;
      t.first = t.tile * p.ns;
      t.ns = p.ns; t.nd = 0;
      t.offset = (size_t)t.first * kSparseStageBytes;
    } else {
      const int td = (s - sparse_total) / p.nd;
      t.tile = p.tiles_sparse + td;
      t.first = sparse_total + td * p.nd;
      t.ns = 0; t.nd = p.nd;
      t.offset = (size_t)sparse_total * kSparseStageBytes + (size_t)td * p.nd * kDenseStageBytes;
    }
  } else {
    const int per = p.ns + p.nd;
    t.tile = s / per;
    t.first = t.tile * per;
    t.ns = p.ns; t.nd = p.nd;
    t.offset = (size_t)t.tile * ((size_t)p.ns * kSparseStageBytes + (size_t)p.nd * kDenseStageBytes);
  }
  return t;
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

// optional per-CTA timeline (debug builds of the harness set GemmParams::trace; nullptr in production)
__device__ __forceinline__ void trace(const GemmParams& p, int span, int slot) {
  if (p.trace) p.trace[(size_t)span * 16 + slot] = clock64();
}
__device__ __forceinline__ long long globaltimer() {
  long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}

constexpr int kThreads = 384;
constexpr int kTmemCols = 512;
constexpr int kMetaCol = 480;   // 2 buffers x 16 columns of 2:4 metadata

}  // namespace

__global__ void __launch_bounds__(kThreads, 1)
spense_gemm_kernel(const __grid_constant__ GemmParams p, const __grid_constant__ CUtensorMap tmap_b) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const int warp = threadIdx.x >> 5;
  const int lane = threadIdx.x & 31;

  const int S = p.num_stages;
  // barriers live after the stage ring
  const uint32_t bar_base = smem_base + (uint32_t)S * p.slot_bytes;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (8 + s); };
  auto accf_bar = [&](int b) { return bar_base + 8u * (16 + b); };
  auto acce_bar = [&](int b) { return bar_base + 8u * (18 + b); };
  auto part_bar = [&](int r) { return bar_base + 8u * (22 + r); };
  const uint32_t tmem_slot = bar_base + 8u * 20;
  uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
  volatile uint32_t* tmem_slot_ptr = reinterpret_cast<volatile uint32_t*>(smem_gen + (size_t)S * p.slot_bytes + 8 * 20);

  if (warp == 0 && lane == 0) {
    prefetch_tmap(&tmap_b);
    for (int s = 0; s < S; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(accf_bar(b), 1); mbar_init(acce_bar(b), 256); }
    for (int r = 0; r < 8; ++r) mbar_init(part_bar(r), 1);
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
  if (p.trace && threadIdx.x == 0) { p.trace[(size_t)span * 16 + 0] = clock64(); p.trace[(size_t)span * 16 + 12] = globaltimer(); }

  if (warp == 0) {
    // ===================== producer =====================
    if (lane == 0) {
      const uint64_t pol_w = policy_evict_first();
      const uint64_t pol_a = policy_evict_last();
      bool waited = false;
      int it = 0;
      for (int s = sb; s < se;) {
        const TileInfo t = tile_of_stage(p, s);
        const int seg_end = min(se, t.first + t.ns + t.nd);
        for (; s < seg_end; ++s, ++it) {
          const int j = s - t.first;
          const int slot = it % S;
          const uint32_t ph = (uint32_t)(it / S) & 1u;
          mbar_wait(empty_bar(slot), ph ^ 1u);
          if (it == 0) trace(p, span, 1);
          const uint32_t a_dst = smem_base + (uint32_t)slot * p.slot_bytes;
          const uint32_t b_dst = a_dst + kSparseStageBytes;
          if (j < t.ns) {
            mbar_expect_tx(full_bar(slot), kSparseStageBytes + 2 * b_tile_bytes);
            bulk_g2s(a_dst, p.section + t.offset + (size_t)j * kSparseStageBytes, kSparseStageBytes, full_bar(slot), pol_w);
            if (!waited) { pdl_wait(); waited = true; }   // weights never depend on the previous kernel; activations do
            tma_load_2d(b_dst, &tmap_b, j * kSparseStageK, 0, full_bar(slot), pol_a);
            tma_load_2d(b_dst + b_tile_bytes, &tmap_b, j * kSparseStageK + 128, 0, full_bar(slot), pol_a);
          } else {
            const int jd = j - t.ns;
            mbar_expect_tx(full_bar(slot), kDenseStageBytes + b_tile_bytes);
            bulk_g2s(a_dst, p.section + t.offset + (size_t)t.ns * kSparseStageBytes + (size_t)jd * kDenseStageBytes,
                     kDenseStageBytes, full_bar(slot), pol_w);
            if (!waited) { pdl_wait(); waited = true; }
            tma_load_2d(b_dst, &tmap_b, p.dense_k0 + jd * kDenseStageK, 0, full_bar(slot), pol_a);
          }
        }
      }
      trace(p, span, 2);
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0) {
      const uint32_t idesc_d = (1u << 4) | ((uint32_t)(p.n_pad >> 3) << 17) | ((128u >> 4) << 24);
      const uint32_t idesc_s = idesc_d | (1u << 2);
      int it = 0, seg = 0;
      for (int s = sb; s < se; ++seg) {
        const TileInfo t = tile_of_stage(p, s);
        const int seg_end = min(se, t.first + t.ns + t.nd);
        const int buf = seg % p.num_acc_bufs;
        const uint32_t use = (uint32_t)(seg / p.num_acc_bufs);
        mbar_wait(acce_bar(buf), (use & 1u) ^ 1u);         // epilogue has drained this accumulator
        tc_fence_after();
        const uint32_t d0 = tmem_base + (uint32_t)(buf * 2 * p.acc_stride);
        const uint32_t d1 = d0 + (uint32_t)p.acc_stride;
        uint32_t acc = 0;
        for (; s < seg_end; ++s, ++it) {
          const int j = s - t.first;
          const int slot = it % S;
          const uint32_t ph = (uint32_t)(it / S) & 1u;
          mbar_wait(full_bar(slot), ph);
          tc_fence_after();
          if (it == 0) trace(p, span, 3);
          const uint32_t a0 = smem_base + (uint32_t)slot * p.slot_bytes;
          const uint32_t a1 = a0 + kOperandBytes;
          const uint32_t b0 = a0 + kSparseStageBytes;
          if (j < t.ns) {
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
  } else if (warp >= 4) {
    // ===================== epilogue (8 warps) =====================
    // warp & 3 selects the TMEM lane quadrant, (warp - 4) >> 2 the half of the token columns.
    const int q = warp & 3;
    const int half = (warp - 4) >> 2;
    const int row = q * 32 + lane;                         // accumulator lane = weight row inside the tile
    const int et = threadIdx.x - 128;                      // 0..255
    const int cols_half = p.n_pad >> 1;                    // multiple of 8
    const int c_begin = half * cols_half;
    float* sc = reinterpret_cast<float*>(smem_gen + (size_t)S * p.slot_bytes + 256);   // [4][n_pad] per-token scales
    int seg = 0;
    bool waited = false;
    uint32_t stage_round = 0;                              // parity of the partial-staging barriers
    for (int s = sb; s < se; ++seg) {
      const TileInfo t = tile_of_stage(p, s);
      const int tile_end = t.first + t.ns + t.nd;
      const int seg_end = min(se, tile_end);
      const bool owner = (s == t.first);
      const int buf = seg % p.num_acc_bufs;
      const uint32_t use = (uint32_t)(seg / p.num_acc_bufs);
      if (!waited) {
        // scales and the workspace may be produced / still in use by the previous kernel of the stream
        pdl_wait();
        waited = true;
        if (et < p.n_pad) {
          const int m = et < p.M ? et : p.M - 1;
          if (p.mode == 0) {
            const float sx = __ldg(p.s_act + m);
            sc[et] = sx * p.w_scale0;
            sc[p.n_pad + et] = sx * p.w_scale1;
            const float sh = __ldg(p.s_h + (size_t)m * p.sh_stride);
            sc[2 * p.n_pad + et] = sh;
            sc[3 * p.n_pad + et] = __frcp_rn(sh);
          } else {
            sc[et] = __ldg(p.s_act + (size_t)m * p.sh_stride) * p.w_scale0;
          }
        }
        asm volatile("bar.sync 1, 256;" ::: "memory");
      }
      mbar_wait(accf_bar(buf), use & 1u);
      tc_fence_after();
      if (et == 0) trace(p, span, seg == 0 ? 5 : 7);
      const uint32_t t0 = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(buf * 2 * p.acc_stride);
      const uint32_t t1 = t0 + (uint32_t)p.acc_stride;

      if (!owner) {
        // contributor: dump the raw fp32 partial [mat][col][row], then publish
        float* slot = p.partials + (size_t)span * (2 * p.n_pad * 128);
        for (int c = c_begin; c < c_begin + cols_half; c += 8) {
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
        asm volatile("bar.sync 1, 256;" ::: "memory");     // all partial stores issued (CTA scope) ...
        if (et == 0) {                                     // ... one gpu-scope release publishes them (cumulativity)
          __threadfence();
          asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p.flags + span), "r"(1) : "memory");
        }
      } else {
        // owner.  Contributors are the following spans that start inside this tile; that can only
        // happen on the CTA's last segment, when the whole stage ring is free: stage their partials
        // into shared memory with bulk copies (one L2 round trip for all of them), then add in span order.
        int n_contrib = 0;
        while (span + 1 + n_contrib < p.n_spans && p.span_begin[span + 1 + n_contrib] < tile_end) ++n_contrib;
        const uint32_t region_bytes = (uint32_t)p.n_pad * 1024u;
        int n_regions = (int)(((uint32_t)S * p.slot_bytes) / region_bytes);
        n_regions = n_regions > 8 ? 8 : n_regions;
        const int out_row = (p.mode == 0) ? (t.tile * 128 + row) : (t.tile * 256 + row);
        int base = 0;
        do {
          const int cnt = min(n_regions, n_contrib - base);
          if (cnt > 0) {
            if (base > 0) {                                // regions are being reused: order our reads before the new async writes
              fence_proxy_async();
              asm volatile("bar.sync 1, 256;" ::: "memory");
            }
            if (et < cnt) {
              const int* f = p.flags + span + 1 + base + et;
              int v;
              do {
                asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(f) : "memory");
              } while (v == 0);
              asm volatile("st.relaxed.gpu.global.s32 [%0], %1;" ::"l"(f), "r"(0) : "memory");   // leave the workspace clean
              mbar_expect_tx(part_bar(et), region_bytes);
              bulk_g2s(smem_base + (uint32_t)et * region_bytes, p.partials + (size_t)(span + 1 + base + et) * (2 * p.n_pad * 128),
                       region_bytes, part_bar(et), policy_evict_first());
            }
            for (int r = 0; r < cnt; ++r) mbar_wait(part_bar(r), stage_round & 1u);
            ++stage_round;
            if (et == 0 && base == 0) trace(p, span, 8);
          }
          const bool last_round = base + cnt >= n_contrib;
          for (int c = c_begin; c < c_begin + cols_half; c += 8) {
            uint32_t v0[8], v1[8];
            tmem_ld8(t0 + c, v0);
            tmem_ld8(t1 + c, v1);
            tmem_ld_wait();
            float f0[8], f1[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) { f0[i] = __uint_as_float(v0[i]); f1[i] = __uint_as_float(v1[i]); }
            for (int r = 0; r < cnt; ++r) {                // fixed span order: deterministic
              const float* reg = reinterpret_cast<const float*>(smem_gen + (size_t)r * region_bytes);
#pragma unroll
              for (int i = 0; i < 8; ++i) {
                f0[i] += reg[(size_t)(c + i) * 128 + row];
                f1[i] += reg[(size_t)(p.n_pad + c + i) * 128 + row];
              }
            }
            if (!last_round) {                             // more contributors than staging regions: park the sum in TMEM
#pragma unroll
              for (int i = 0; i < 8; ++i) { v0[i] = __float_as_uint(f0[i]); v1[i] = __float_as_uint(f1[i]); }
              tmem_st8(t0 + c, v0);
              tmem_st8(t1 + c, v1);
              continue;
            }
            if (p.mode == 0) {
#pragma unroll
              for (int i = 0; i < 8; i += 2) {
                float h[2], qv[2];
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                  const int m = c + i + e;
                  const float g = f0[i + e] * sc[m];
                  const float u = f1[i + e] * sc[p.n_pad + m];
                  h[e] = silu_mul(g, u);
                  qv[e] = div_by(h[e], sc[2 * p.n_pad + m], sc[3 * p.n_pad + m]);
                }
                const uint32_t qb = to_e4m3x2(qv[0], qv[1]);
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                  const int m = c + i + e;
                  if (m < p.M) {
                    const size_t o = (size_t)m * p.ld_out + out_row;
                    if (p.h_f32) p.h_f32[o] = h[e];
                    p.hq[o] = (uint8_t)(qb >> (8 * e));
                  }
                }
              }
            } else {
#pragma unroll
              for (int i = 0; i < 8; ++i) {
                const int m = c + i;
                if (m < p.M) {
                  const float scl = sc[m];
                  const float y0 = f0[i] * scl, y1 = f1[i] * scl;
                  const size_t o = (size_t)m * p.ld_out + out_row;
                  if (p.y_dtype == SPENSE_F32) {
                    float* y = reinterpret_cast<float*>(p.y);
                    y[o] = y0;
                    if (out_row + 128 < p.out_rows) y[o + 128] = y1;
                  } else {
                    __nv_bfloat16* y = reinterpret_cast<__nv_bfloat16*>(p.y);
                    y[o] = __float2bfloat16_rn(y0);
                    if (out_row + 128 < p.out_rows) y[o + 128] = __float2bfloat16_rn(y1);
                  }
                }
              }
            }
          }
          if (!last_round) tmem_st_wait();
          base += cnt;
        } while (base < n_contrib);
        tc_fence_before();
        mbar_arrive(acce_bar(buf));
      }
      if (et == 0) trace(p, span, seg == 0 ? 6 : 9);
      s = seg_end;
    }
    if (p.trace && et == 0) { p.trace[(size_t)span * 16 + 10] = seg; p.trace[(size_t)span * 16 + 11] = se - sb; p.trace[(size_t)span * 16 + 13] = globaltimer(); }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) { tc_fence_after(); tmem_dealloc(tmem_base, kTmemCols); }
}

int launch_gemm(const GemmParams& p, const CUtensorMap& tmap_b, bool pdl, cudaStream_t stream) {
  const size_t smem = (size_t)p.num_stages * p.slot_bytes + 1024 + 256 + 4 * 4 * (size_t)p.n_pad;
  static bool attr_set = false;
  if (!attr_set) {
    if (cudaFuncSetAttribute(spense_gemm_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 232448) != cudaSuccess)
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
  if (cudaLaunchKernelEx(&cfg, spense_gemm_kernel, p, tmap_b) != cudaSuccess) return SPENSE_ERR_CUDA;
  return SPENSE_OK;
}

}  // namespace spense
