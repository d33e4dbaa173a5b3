// Device helpers of the Spense GEMM kernel (spense_gemm.cu): the walk over the linear stage sequence, the element-wise
// epilogue (scales -> SiLU*up -> E4M3, Eq. 4) and the bounded waits.  Nothing here is shared with oracle/.
#pragma once

#include <cuda_bf16.h>

#include "spense_internal.cuh"

namespace spense {
namespace dev {

// Position in the linear stage sequence: pair tile, stage inside the tile, stages of the tile.
struct Cursor {
  int tile, j, ns, nd, first;   // first = linear index of the tile's first stage
};

// MODE 0 (gate_up) and MODE 2 (out-split linear) walk whole-K tiles, the sparse tiles first; MODE 1 (down, in-split linear)
// walks tiles whose K loop is sparse stages followed by dense stages
__host__ __device__ constexpr bool out_split(int mode) { return mode != 1; }

// byte offset of stage j of pair tile `tile` inside the section (the blob stores every tile once)
template <int MODE>
__device__ __forceinline__ size_t stage_byte_offset(const GemmParams& p, int tile, int j) {
  if (out_split(MODE)) {
    if (tile < p.tiles_sparse) return ((size_t)tile * p.ns + j) * kSparseStageBytes;
    return (size_t)p.tiles_sparse * p.ns * kSparseStageBytes + ((size_t)(tile - p.tiles_sparse) * p.nd + j) * kDenseStageBytes;
  }
  const size_t base = (size_t)tile * ((size_t)p.ns * kSparseStageBytes + (size_t)p.nd * kDenseStageBytes);
  return base + (j < p.ns ? (size_t)j * kSparseStageBytes
                          : (size_t)p.ns * kSparseStageBytes + (size_t)(j - p.ns) * kDenseStageBytes);
}

// The only place with integer divisions (one copy per mode, called once per role).
template <int MODE>
static __device__ __noinline__ Cursor cursor_at(const GemmParams& p, int s, unsigned long long* byte_off) {
  Cursor c;
  if (out_split(MODE)) {
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
  if (out_split(MODE)) {
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
// A divisor below 2^-128 (a caller's tiny s_h) has no finite fp32 reciprocal: those take the IEEE division.
__device__ __forceinline__ float div_by(float a, float b, float r) {
  if (__builtin_expect(!(fabsf(r) <= 3.402823466e+38f), 0)) return __fdiv_rn(a, b);
  const float q0 = a * r;
  const float rem = fmaf(-q0, b, a);
  const float q = fmaf(rem, r, q0);
  return q == 0.0f ? q0 : q;                               // (+0) + (-0) = +0 would lose the sign of a zero quotient
}

// fp32 -> E4M3 (saturating, round to nearest even); cvt.rn.satfinite.e4m3x2.f32 packs two values:
// lo in bits 0..7, hi in bits 8..15
__device__ __forceinline__ uint32_t to_e4m3x2(float lo, float hi) {
  uint16_t r;
  asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(r) : "f"(hi), "f"(lo));
  return r;
}

__device__ __forceinline__ long long globaltimer() {
  long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
// optional per-CTA timeline: SPENSE_DEBUG_HOOKS builds set GemmParams::trace; the shipped library compiles none of it
__device__ __forceinline__ bool tracing(const GemmParams& p) {
#ifdef SPENSE_DEBUG_HOOKS
  return p.trace != nullptr;
#else
  return false;
#endif
}
__device__ __forceinline__ void trace(const GemmParams& p, int span, int slot) {
  if (tracing(p)) p.trace[(size_t)span * 16 + slot] = globaltimer();
}
__device__ __forceinline__ int ld_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release(int* p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// ---- bounded waits.  The CTAs of a launch wait for each other (split-K fix-up), so all of them must be resident at
// the same time; the host checks that against the occupancy the device offers before launching, and every wait here
// gives up after kWaitBudgetNs: the CTA records SPENSE_ERR_TIMEOUT in the mapped host status word and traps, so a launch
// whose peers never show up (device shared with work that pins SMs) fails with a CUDA error instead of hanging for ever;
// spense_device_status() then says why.  The trap is deliberate and documented as fatal to the context (spense.h): a
// cooperative exit would have to unwind four warp roles, the pair's cluster barrier and the TMEM allocation of CTAs whose
// peers are not coming, and a launch in that state has no result worth keeping.
// A launch that works never reads the timer: the first try succeeds.
static __device__ __noinline__ void give_up(int* status, int code) {
  atomicCAS_system(status, 0, code);
  __threadfence_system();
  __trap();
}
__device__ __forceinline__ void wait_bar(const GemmParams& p, uint32_t bar, uint32_t parity) {
  if (mbar_try(bar, parity)) return;
  const long long t0 = globaltimer();
#pragma unroll 1
  for (;;) {
#pragma unroll 1
    for (int i = 0; i < 32; ++i) {
      if (mbar_try(bar, parity)) return;
#ifdef SPENSE_DEBUG_HOOKS
      if ((p.dbg & 4) && threadIdx.x >= 128) __nanosleep(200);
#endif
    }
    if (globaltimer() - t0 > kWaitBudgetNs) give_up(p.status, SPENSE_ERR_TIMEOUT);
  }
}
__device__ __forceinline__ void wait_flag(const GemmParams& p, const int* flag, int epoch) {
  if (ld_acquire(flag) == epoch) return;
  const long long t0 = globaltimer();
#pragma unroll 1
  for (;;) {
#pragma unroll 1
    for (int i = 0; i < 256; ++i)
      if (ld_acquire(flag) == epoch) return;
    if (globaltimer() - t0 > kWaitBudgetNs) give_up(p.status, SPENSE_ERR_TIMEOUT);
  }
}

// Epoch of a launch = epoch word + 1.  Every CTA reads the word BEFORE it counts itself; the CTA that counts
// last therefore knows all have read it and advances it for the next launch.
__device__ __forceinline__ void take_epoch(int* ctrl, int n_ctas, volatile int* out) {
  const int e0 = ld_acquire(ctrl);
  out[0] = e0 + 1;
  if (atomicAdd(ctrl + 1, 1) == n_ctas - 1) {
    ctrl[1] = 0;
    st_release(ctrl, e0 + 1);
  }
}

// the blob header against the shape the caller stated: a mismatch is reported, the launch runs on (garbage out)
__device__ __forceinline__ void check_header(const GemmParams& p) {
  const BlobHeader* h = p.hdr;
  if (__ldg(&h->magic) != kBlobMagic || __ldg(&h->version) != kBlobVersion || __ldg(&h->H) != p.H || __ldg(&h->I) != p.I ||
      __ldg(&h->I_dense) != p.I_d || __ldg(&h->kind) != p.kind) {
    atomicCAS_system(p.status, 0, SPENSE_ERR_BAD_BLOB);
    __threadfence_system();
  }
}

// One GLU output (token column m of the block, intermediate index j of pair tile `tile`): scales, SiLU(g) * u, then
// (static scale) the IEEE division by s_h and the E4M3 cast, or (DYN: the scale does not exist yet) h kept in fp32;
// returns |h| for the running maximum.  sc4 = float4 per token column {s_x*s_gate, s_x*s_up, s_h, RN(1/s_h)};
// m_out = token (output row).
template <bool DYN>
__device__ __forceinline__ float finish_glu(const GemmParams& p, const float4* sc4, int tile, int j, int m, int m_out, float acc_g, float acc_u) {
  const float4 k = sc4[m];
  const float g = acc_g * k.x;
  const float u = acc_u * k.y;
  const float h = silu_mul(g, u);
  const size_t o = (size_t)m_out * p.ld_out + tile * 128 + j;
  if (DYN) {
    p.h_f32[o] = h;
    return fabsf(h);
  }
  const float qv = div_by(h, k.z, k.w);
  if (p.h_f32) p.h_f32[o] = h;
  p.hq[o] = (uint8_t)(to_e4m3x2(qv, 0.0f) & 0xFFu);
  return 0.0f;
}

// NG groups of 8 token columns of ONE gate_up operand, read with two tcgen05.ld.16x256b.xNG (gate half, up half of the
// warp's lane quadrant): thread t holds, for group j, lanes t/4 (k = 4 j + 0, 1) and t/4 + 8 (k = 4 j + 2, 3), columns
// c + 8 j + 2 (t % 4) + (k & 1).
template <int NG>
__device__ __forceinline__ void load_glu(uint32_t t_gate, int c, float (&g)[4 * NG], float (&u)[4 * NG]) {
  uint32_t rg[4 * NG], ru[4 * NG];
  if (NG == 1) {
    tmem_ld_16x256b(t_gate + c, reinterpret_cast<uint32_t(&)[4]>(rg[0]));
    tmem_ld_16x256b(t_gate + (16u << 16) + c, reinterpret_cast<uint32_t(&)[4]>(ru[0]));
  } else if (NG == 2) {
    tmem_ld_16x256b_x2(t_gate + c, reinterpret_cast<uint32_t(&)[8]>(rg[0]));
    tmem_ld_16x256b_x2(t_gate + (16u << 16) + c, reinterpret_cast<uint32_t(&)[8]>(ru[0]));
  } else {
    tmem_ld_16x256b_x4(t_gate + c, reinterpret_cast<uint32_t(&)[16]>(rg[0]));
    tmem_ld_16x256b_x4(t_gate + (16u << 16) + c, reinterpret_cast<uint32_t(&)[16]>(ru[0]));
  }
  tmem_ld_wait();
#pragma unroll
  for (int i = 0; i < 4 * NG; ++i) { g[i] = __uint_as_float(rg[i]); u[i] = __uint_as_float(ru[i]); }
}
// index of element k of load_glu (gu = 0 gate, 1 up) inside a [col][128 lanes] partial image; q = lane quadrant
__device__ __forceinline__ int glu_part_index(int k, int gu, int q, int t, int c) {
  return (c + 8 * (k >> 2) + 2 * (t & 3) + (k & 1)) * 128 + 32 * q + 16 * gu + (t >> 2) + 8 * ((k >> 1) & 1);
}
// their epilogue.  j0 = index inside the pair tile of the quadrant's first lane (64 a + 16 q); sc4 = float4 per token column
// {s_x*s_gate, s_x*s_up, s_h, RN(1/s_h)}.  Called by all 32 lanes.
template <bool DYN, int NG>
__device__ __forceinline__ void glu_block(const GemmParams& p, float4* sc4, int tile, int j0, int c, int Mb, int m_base,
                                          const float (&g)[4 * NG], const float (&u)[4 * NG]) {
  const int t = threadIdx.x & 31;
  const int jr = tile * 128 + j0 + (t >> 2);
#pragma unroll
  for (int j = 0; j < NG; ++j) {
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const int col = c + 8 * j + 2 * (t & 3) + e;
      float mx = 0.0f;
      if (col < Mb) {
        const float4 k = sc4[col];
        const size_t o = (size_t)(m_base + col) * p.ld_out + jr;
#pragma unroll
        for (int li = 0; li < 2; ++li) {
          const int i = 4 * j + 2 * li + e;
          const float h = silu_mul(g[i] * k.x, u[i] * k.y);
          if (DYN) {
            p.h_f32[o + 8 * li] = h;
            mx = fmaxf(mx, fabsf(h));
          } else {
            if (p.h_f32) p.h_f32[o + 8 * li] = h;
            p.hq[o + 8 * li] = (uint8_t)(to_e4m3x2(div_by(h, k.z, k.w), 0.0f) & 0xFFu);
          }
        }
      }
      if (DYN) {
        // max|h| of the 16 indices per token column: over the 8 threads that share t % 4, then one shared atomic each
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 4));
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 8));
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 16));
        if (t < 4 && col < Mb) atomicMax(reinterpret_cast<int*>(sc4 + col) + 2, __float_as_int(mx));   // |h| >= 0: int order == float order
      }
    }
  }
}

// One Y element: y = acc * s_h[m] * s_down
__device__ __forceinline__ void store_y(const GemmParams& p, int out_row, int m_out, float y) {
  if (out_row >= p.out_rows) return;
  const size_t o = (size_t)m_out * p.ld_out + out_row;
  if (p.y_dtype == SPENSE_F32) reinterpret_cast<float*>(p.y)[o] = y;
  else reinterpret_cast<__nv_bfloat16*>(p.y)[o] = __float2bfloat16_rn(y);
}

// Epilogue of NG groups of 8 token columns of ONE accumulator (operand `opnd` of the pair tile; one lane quadrant per
// warp); `part` = the partner's partial [col][lane] of that operand to add first (owner of a tile split over two spans),
// read straight from L2, or nullptr.
template <int MODE, bool DYN, int NG>
__device__ __forceinline__ void tile_block(const GemmParams& p, float4* sc4, const float* sc1, uint32_t t0, const float* part, int tile,
                                           int opnd, int q, int lane, int c, int Mb, int m_base) {
  if (MODE == 0) {
    float g[4 * NG], u[4 * NG], pg[4 * NG], pu[4 * NG];
    if (part) {
#pragma unroll
      for (int i = 0; i < 4 * NG; ++i) {
        pg[i] = __ldcg(part + glu_part_index(i, 0, q, lane, c));
        pu[i] = __ldcg(part + glu_part_index(i, 1, q, lane, c));
      }
    }
    load_glu<NG>(t0, c, g, u);
    if (part) {
#pragma unroll
      for (int i = 0; i < 4 * NG; ++i) { g[i] += pg[i]; u[i] += pu[i]; }
    }
    glu_block<DYN, NG>(p, sc4, tile, 64 * opnd + 16 * q, c, Mb, m_base, g, u);
  } else {
    uint32_t r[8 * NG];
    float pv[8 * NG];
    if (part) {
#pragma unroll
      for (int i = 0; i < 8 * NG; ++i) pv[i] = __ldcg(part + (size_t)(c + i) * 128 + 32 * q + lane);
    }
    if (NG == 1) tmem_ld8(t0 + c, reinterpret_cast<uint32_t(&)[8]>(r[0]));
    else if (NG == 2) tmem_ld16(t0 + c, reinterpret_cast<uint32_t(&)[16]>(r[0]));
    else tmem_ld32(t0 + c, reinterpret_cast<uint32_t(&)[32]>(r[0]));
    tmem_ld_wait();
    const int row = tile * 256 + 128 * opnd + 32 * q + lane;
#pragma unroll
    for (int i = 0; i < 8 * NG; ++i)
      if (c + i < Mb) store_y(p, row, m_base + c + i, (__uint_as_float(r[i]) + (part ? pv[i] : 0.0f)) * sc1[c + i]);
  }
}

// where operand row `lane` of a gate_up operand comes from (blob layout, spense_internal.cuh): index inside the operand's
// 64 intermediate indices and whether it is an up row
__device__ __forceinline__ int glu_index_of_lane(int lane) { return ((lane >> 5) << 4) | (lane & 15); }
__device__ __forceinline__ int glu_gate_lane_of_index(int j64) { return ((j64 >> 4) << 5) | (j64 & 15); }

}  // namespace dev
}  // namespace spense
