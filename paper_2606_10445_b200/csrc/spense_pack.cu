// spense_pack kernels: P1 permute, P2 validate + 2:4 compress, P3 re-tile into stage images.
// Integer / byte work only: results are bit-exact by construction (Eq. 1 PAPER.md:69, PAPER.md:74,
// Fig. 4).  Also the E4M3 quantise helper (reading Q5).
#include <mutex>

#include "spense_internal.cuh"

namespace spense {

namespace {

// error words in the pack workspace
struct PackErr {
  unsigned long long nan_key, nan_cnt, n24_key, n24_cnt;
  int perm_bad;
  int pad[7];
};

__device__ __forceinline__ unsigned long long err_key(int matrix, int row, int group) {
  return ((unsigned long long)matrix << 56) | ((unsigned long long)(unsigned)row << 28) | (unsigned long long)(unsigned)group;
}

// One group of 4 bytes (little endian in `w`) -> 2 value bytes (low 16 bits) + nibble (bits 16..19).
// Rule (readings Q6/Q7): kept = non-zero positions, filled up with the smallest positions not
// yet kept; nibble = i0 | i1 << 2; zero bytes (+-0) are stored as 0x00.  status: bit0 NaN byte, bit1 > 2 non-zero.
__device__ __forceinline__ uint32_t compress_group(uint32_t w, int& status) {
  int nzmask = 0;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const uint32_t b = (w >> (8 * i)) & 0x7Fu;
    if (b == 0x7Fu) status |= 1;
    if (b != 0) nzmask |= 1 << i;
  }
  const int cnt = __popc(nzmask);
  if (cnt > 2) { status |= 2; return 0x40000u; }
  int i0, i1;
  if (cnt == 2) {
    i0 = __ffs(nzmask) - 1;
    i1 = 31 - __clz(nzmask);
  } else if (cnt == 1) {
    const int k = __ffs(nzmask) - 1;
    if (k == 0) { i0 = 0; i1 = 1; } else { i0 = 0; i1 = k; }
  } else {
    i0 = 0; i1 = 1;
  }
  uint32_t v0 = (w >> (8 * i0)) & 0xFFu, v1 = (w >> (8 * i1)) & 0xFFu;
  if ((v0 & 0x7Fu) == 0) v0 = 0;
  if ((v1 & 0x7Fu) == 0) v1 = 0;
  return v0 | (v1 << 8) | ((uint32_t)(i0 | (i1 << 2)) << 16);
}

__device__ __forceinline__ void report(PackErr* err, int status, int matrix, int row, int group) {
  if (status & 1) { atomicMin(&err->nan_key, err_key(matrix, row, group)); atomicAdd(&err->nan_cnt, 1ull); }
  if (status & 2) { atomicMin(&err->n24_key, err_key(matrix, row, group)); atomicAdd(&err->n24_cnt, 1ull); }
}

__global__ void pack_init_kernel(PackErr* err, int* marks, int I) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) {
    err->nan_key = ~0ull; err->n24_key = ~0ull; err->nan_cnt = 0; err->n24_cnt = 0; err->perm_bad = 0;
  }
  if (i < I) marks[i] = 0;
}

__global__ void perm_mark_kernel(const int32_t* perm, int* marks, PackErr* err, int I) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= I) return;
  const int o = perm[i];
  if (o < 0 || o >= I) { atomicAdd(&err->perm_bad, 1); return; }
  if (atomicAdd(&marks[o], 1) != 0) atomicAdd(&err->perm_bad, 1);
}

__global__ void write_header_kernel(BlobHeader* h, BlobHeader v) { if (threadIdx.x == 0 && blockIdx.x == 0) *h = v; }

// gate / up: blockIdx.y = matrix (0 gate, 1 up), blockIdx.x = new (permuted) row.  Each thread handles
// 8 consecutive K bytes (2 groups) per step.
__global__ void pack_gate_up_kernel(Geometry g, const uint8_t* __restrict__ wgate, const uint8_t* __restrict__ wup,
                                    const int32_t* __restrict__ perm, uint8_t* __restrict__ blob, spense_canon_t canon,
                                    PackErr* err) {
  const int matrix = blockIdx.y;
  const int r = blockIdx.x;
  const int src_row = perm ? perm[r] : r;
  const uint8_t* src = (matrix == 0 ? wgate : wup) + (size_t)src_row * g.H;
  // pair tile r / 128; inside it operand (r % 128) / 64 holds the gate and the up row of an index in the two 16-lane
  // halves of one lane quadrant (layout: spense_internal.cuh)
  const int tile = r >> 7, opnd = (r >> 6) & 1;
  const int rr = (((r >> 4) & 3) << 5) | (matrix << 4) | (r & 15);
  uint8_t* sec = blob + g.gate_up_off;
  if (matrix == 0 && canon.perm && threadIdx.x == 0) canon.perm[r] = src_row;
  if (r < g.I_s) {
    uint8_t* tile_base = sec + (size_t)tile * g.gu_ns * kSparseStageBytes;
    uint8_t* cval = matrix == 0 ? canon.gate_sp_val : canon.up_sp_val;
    uint8_t* cmeta = matrix == 0 ? canon.gate_sp_meta : canon.up_sp_meta;
    const int steps = g.gu_ns * (kSparseStageK / 8);       // padded K / 8
    for (int t = threadIdx.x; t < steps; t += blockDim.x) {
      uint32_t vals = 0, meta = 0x44;
      if (8 * t < g.H) {
        const uint2 w = *reinterpret_cast<const uint2*>(src + 8 * t);
        int st0 = 0, st1 = 0;
        const uint32_t c0 = compress_group(w.x, st0);
        const uint32_t c1 = compress_group(w.y, st1);
        if (st0) report(err, st0, matrix, r, 2 * t);
        if (st1) report(err, st1, matrix, r, 2 * t + 1);
        vals = (c0 & 0xFFFFu) | (c1 << 16);
        meta = ((c0 >> 16) & 0xFu) | (((c1 >> 16) & 0xFu) << 4);
        if (cval) *reinterpret_cast<uint32_t*>(cval + (size_t)r * (g.H / 2) + 4 * t) = vals;
        if (cmeta) cmeta[(size_t)r * (g.H / 8) + t] = (uint8_t)meta;
      }
      const int js = t >> 5;                                // 32 meta bytes (= 128 value bytes) per stage and row
      const int tb = t & 31;
      uint8_t* stage = tile_base + (size_t)js * kSparseStageBytes;
      *reinterpret_cast<uint32_t*>(stage + opnd * kSparseOperandBytes + sw128_offset(rr, 4 * tb)) = vals;
      stage[opnd * kSparseOperandBytes + kOperandBytes + (tb >> 4) * 2048 + rr * 16 + (tb & 15)] = (uint8_t)meta;
    }
  } else {
    const int td = tile - g.gu_tiles_sparse;
    uint8_t* tile_base = sec + (size_t)g.gu_tiles_sparse * g.gu_ns * kSparseStageBytes + (size_t)td * g.gu_nd * kDenseStageBytes;
    uint8_t* cdn = matrix == 0 ? canon.gate_dn : canon.up_dn;
    for (int t = threadIdx.x; t < g.H / 8; t += blockDim.x) {
      const uint2 w = *reinterpret_cast<const uint2*>(src + 8 * t);
      int st = 0;
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        if (((w.x >> (8 * i)) & 0x7Fu) == 0x7Fu) st |= 1;
        if (((w.y >> (8 * i)) & 0x7Fu) == 0x7Fu) st |= 4;
      }
      if (st & 1) report(err, 1, matrix, r, 2 * t);
      if (st & 4) report(err, 1, matrix, r, 2 * t + 1);
      if (cdn) *reinterpret_cast<uint2*>(cdn + (size_t)(r - g.I_s) * g.H + 8 * t) = w;
      const int jd = (8 * t) >> 7, b = (8 * t) & 127;
      *reinterpret_cast<uint2*>(tile_base + (size_t)jd * kDenseStageBytes + opnd * kOperandBytes + sw128_offset(rr, b)) = w;
    }
  }
}

// down: blockIdx.x = output row n (padded to 256 * dn_tiles).  Columns are gathered through perm.
__global__ void pack_down_kernel(Geometry g, const uint8_t* __restrict__ wdown, const int32_t* __restrict__ perm,
                                 uint8_t* __restrict__ blob, spense_canon_t canon, PackErr* err, int matrix_id) {
  const int n = blockIdx.x;
  const bool real_row = n < g.H;
  const uint8_t* src = wdown + (size_t)(real_row ? n : 0) * g.I;
  const int tile = n >> 8, sub = (n >> 7) & 1, rr = n & 127;
  uint8_t* tile_base = blob + g.down_off + (size_t)tile * ((size_t)g.dn_ns * kSparseStageBytes + (size_t)g.dn_nd * kDenseStageBytes);
  // sparse K range (padded to 256)
  const int steps = g.dn_ns * (kSparseStageK / 8);
  for (int t = threadIdx.x; t < steps; t += blockDim.x) {
    uint32_t vals = 0, meta = 0x44;
    if (real_row && 8 * t < g.I_s) {
      uint32_t wx = 0, wy = 0;
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const int k0 = 8 * t + i, k1 = 8 * t + 4 + i;
        wx |= (uint32_t)src[perm ? perm[k0] : k0] << (8 * i);
        wy |= (uint32_t)src[perm ? perm[k1] : k1] << (8 * i);
      }
      int st0 = 0, st1 = 0;
      const uint32_t c0 = compress_group(wx, st0);
      const uint32_t c1 = compress_group(wy, st1);
      if (st0) report(err, st0, matrix_id, n, 2 * t);
      if (st1) report(err, st1, matrix_id, n, 2 * t + 1);
      vals = (c0 & 0xFFFFu) | (c1 << 16);
      meta = ((c0 >> 16) & 0xFu) | (((c1 >> 16) & 0xFu) << 4);
      if (canon.down_sp_val) *reinterpret_cast<uint32_t*>(canon.down_sp_val + (size_t)n * (g.I_s / 2) + 4 * t) = vals;
      if (canon.down_sp_meta) canon.down_sp_meta[(size_t)n * (g.I_s / 8) + t] = (uint8_t)meta;
    }
    const int js = t >> 5, tb = t & 31;
    uint8_t* stage = tile_base + (size_t)js * kSparseStageBytes;
    *reinterpret_cast<uint32_t*>(stage + sub * kSparseOperandBytes + sw128_offset(rr, 4 * tb)) = vals;
    stage[sub * kSparseOperandBytes + kOperandBytes + (tb >> 4) * 2048 + rr * 16 + (tb & 15)] = (uint8_t)meta;
  }
  // dense K range
  uint8_t* dense_base = tile_base + (size_t)g.dn_ns * kSparseStageBytes;
  for (int t = threadIdx.x; t < g.I_d / 8; t += blockDim.x) {
    uint2 w = make_uint2(0, 0);
    if (real_row) {
      int st = 0;
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const int k0 = g.I_s + 8 * t + i, k1 = k0 + 4;
        const uint32_t b0 = src[perm ? perm[k0] : k0], b1 = src[perm ? perm[k1] : k1];
        if ((b0 & 0x7Fu) == 0x7Fu) st |= 1;
        if ((b1 & 0x7Fu) == 0x7Fu) st |= 4;
        w.x |= b0 << (8 * i);
        w.y |= b1 << (8 * i);
      }
      if (st & 1) report(err, 1, matrix_id, n, (g.I_s + 8 * t) / 4);
      if (st & 4) report(err, 1, matrix_id, n, (g.I_s + 8 * t) / 4 + 1);
      if (canon.down_dn) *reinterpret_cast<uint2*>(canon.down_dn + (size_t)n * g.I_d + 8 * t) = w;
    }
    const int jd = (8 * t) >> 7, b = (8 * t) & 127;
    *reinterpret_cast<uint2*>(dense_base + (size_t)jd * kDenseStageBytes + sub * kOperandBytes + sw128_offset(rr, b)) = w;
  }
}

// out-split linear: blockIdx.x = new (permuted) row, padded to whole 256-row tiles.  Geometry from make_geometry_linear:
// g.H = K, g.I = N, g.I_s = sparse rows (a multiple of 256).  Operand rows are in natural order.
__global__ void pack_rows_kernel(Geometry g, const uint8_t* __restrict__ w, const int32_t* __restrict__ perm, uint8_t* __restrict__ blob,
                                 spense_linear_canon_t canon, PackErr* err) {
  const int r = blockIdx.x;
  const bool real_row = r < g.I;
  const int src_row = real_row ? (perm ? perm[r] : r) : 0;
  const uint8_t* src = w + (size_t)src_row * g.H;
  const int tile = r >> 8, opnd = (r >> 7) & 1, rr = r & 127;
  uint8_t* sec = blob + g.gate_up_off;
  if (real_row && canon.perm && threadIdx.x == 0) canon.perm[r] = src_row;
  if (r < g.I_s) {
    uint8_t* tile_base = sec + (size_t)tile * g.gu_ns * kSparseStageBytes;
    const int steps = g.gu_ns * (kSparseStageK / 8);
    for (int t = threadIdx.x; t < steps; t += blockDim.x) {
      uint32_t vals = 0, meta = 0x44;
      if (8 * t < g.H) {
        const uint2 v = *reinterpret_cast<const uint2*>(src + 8 * t);
        int st0 = 0, st1 = 0;
        const uint32_t c0 = compress_group(v.x, st0);
        const uint32_t c1 = compress_group(v.y, st1);
        if (st0) report(err, st0, 0, r, 2 * t);
        if (st1) report(err, st1, 0, r, 2 * t + 1);
        vals = (c0 & 0xFFFFu) | (c1 << 16);
        meta = ((c0 >> 16) & 0xFu) | (((c1 >> 16) & 0xFu) << 4);
        if (canon.sp_val) *reinterpret_cast<uint32_t*>(canon.sp_val + (size_t)r * (g.H / 2) + 4 * t) = vals;
        if (canon.sp_meta) canon.sp_meta[(size_t)r * (g.H / 8) + t] = (uint8_t)meta;
      }
      const int js = t >> 5, tb = t & 31;
      uint8_t* stage = tile_base + (size_t)js * kSparseStageBytes;
      *reinterpret_cast<uint32_t*>(stage + opnd * kSparseOperandBytes + sw128_offset(rr, 4 * tb)) = vals;
      stage[opnd * kSparseOperandBytes + kOperandBytes + (tb >> 4) * 2048 + rr * 16 + (tb & 15)] = (uint8_t)meta;
    }
  } else {
    const int td = tile - g.gu_tiles_sparse;
    uint8_t* tile_base = sec + (size_t)g.gu_tiles_sparse * g.gu_ns * kSparseStageBytes + (size_t)td * g.gu_nd * kDenseStageBytes;
    for (int t = threadIdx.x; t < g.H / 8; t += blockDim.x) {
      uint2 v = make_uint2(0, 0);
      if (real_row) {
        v = *reinterpret_cast<const uint2*>(src + 8 * t);
        int st = 0;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          if (((v.x >> (8 * i)) & 0x7Fu) == 0x7Fu) st |= 1;
          if (((v.y >> (8 * i)) & 0x7Fu) == 0x7Fu) st |= 4;
        }
        if (st & 1) report(err, 1, 0, r, 2 * t);
        if (st & 4) report(err, 1, 0, r, 2 * t + 1);
        if (canon.dn) *reinterpret_cast<uint2*>(canon.dn + (size_t)(r - g.I_s) * g.H + 8 * t) = v;
      }
      const int jd = (8 * t) >> 7, b = (8 * t) & 127;
      *reinterpret_cast<uint2*>(tile_base + (size_t)jd * kDenseStageBytes + opnd * kOperandBytes + sw128_offset(rr, b)) = v;
    }
  }
}

__global__ void copy_perm_kernel(const int32_t* perm, int32_t* out, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = perm ? perm[i] : i;
}

// ---------------------------------------------------------------- quantise helper
__device__ __forceinline__ float block_max(float v) {
  __shared__ float red[32];
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x < 32) {
    v = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : 0.0f;
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    if (threadIdx.x == 0) red[0] = v;
  }
  __syncthreads();
  return red[0];
}

__global__ void row_amax_kernel(const float* __restrict__ in, int64_t cols, float* __restrict__ amax) {
  const float* row = in + (size_t)blockIdx.x * cols;
  float m = 0.0f;
  for (int64_t c = threadIdx.x; c < cols; c += blockDim.x) m = fmaxf(m, fabsf(row[c]));
  m = block_max(m);
  if (threadIdx.x == 0) amax[blockIdx.x] = m;
}

__global__ void tensor_amax_kernel(const float* __restrict__ row_amax, int64_t rows, float* __restrict__ out) {
  float m = 0.0f;
  for (int64_t r = threadIdx.x; r < rows; r += blockDim.x) m = fmaxf(m, row_amax[r]);
  m = block_max(m);
  if (threadIdx.x == 0) out[0] = m;
}

__global__ void quantize_kernel(const float* __restrict__ in, int64_t cols, const float* __restrict__ amax, int per_row,
                                uint8_t* __restrict__ out, float* __restrict__ scales) {
  const float a = per_row ? amax[blockIdx.x] : amax[0];
  const float s = a > 0.0f ? __fdiv_rn(a, 448.0f) : 1.0f;
  if (threadIdx.x == 0 && (per_row || blockIdx.x == 0)) scales[per_row ? blockIdx.x : 0] = s;
  const float* row = in + (size_t)blockIdx.x * cols;
  uint8_t* orow = out + (size_t)blockIdx.x * cols;
  for (int64_t c = threadIdx.x; c < cols; c += blockDim.x) {
    uint16_t r;
    asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(r) : "f"(0.0f), "f"(__fdiv_rn(row[c], s)));
    orow[c] = (uint8_t)(r & 0xFF);
  }
}

// ---------------------------------------------------------------- dynamic per-token requant
// h [rows, cols] fp32 (written by gate_up in dynamic mode) -> s_h[m] = max_j|h[m,j]| / 448 (1 if zero),
// Hq[m,j] = E4M3_rne_sat(h[m,j] / s_h[m]).  The row maximum comes from the per-CTA maxima gate_up left in amax_part:
// row m belongs to token block m / block_rows whose CTAs own the slots [blk * n_part, (blk + 1) * n_part), each
// [part_stride] floats indexed by the token column m % block_rows (no atomics, nothing to reset).
// grid = (column chunks of chunk_cols, rows), about two 256-thread CTAs per SM (launch_requant_rows): the kernel sits on the
// critical path between gate_up and down, few rows must still fill the machine, and many small CTAs per SM keep the
// next kernel's CTAs (which want to fill their weight rings meanwhile) out of the register file for longer.
__global__ void __launch_bounds__(256) requant_rows_kernel(const float* __restrict__ h, int cols, int chunk_cols, const float* __restrict__ amax_part,
                                                           int n_part, int part_stride, int block_rows, uint8_t* __restrict__ hq,
                                                           float* __restrict__ s_h) {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // down may become resident and stream its weights now
  asm volatile("griddepcontrol.wait;" ::: "memory");                // h and amax_part come from the previous kernel
  const int row = blockIdx.y;
  const int blk = row / block_rows, col = row - blk * block_rows;
  const float* part = amax_part + (size_t)blk * n_part * part_stride + col;
  float m = 0.0f;
  for (int i = threadIdx.x; i < n_part; i += blockDim.x) m = fmaxf(m, __ldcg(part + (size_t)i * part_stride));
  m = block_max(m);
  const float s = m > 0.0f ? __fdiv_rn(m, 448.0f) : 1.0f;
  if (blockIdx.x == 0 && threadIdx.x == 0) s_h[row] = s;
  const int c0 = blockIdx.x * chunk_cols;
  const float4* src = reinterpret_cast<const float4*>(h + (size_t)row * cols + c0);
  uint32_t* dst = reinterpret_cast<uint32_t*>(hq + (size_t)row * cols + c0);
  const int n4 = min(chunk_cols, cols - c0) >> 2;                // cols, chunk_cols % 128 == 0
  // four loads in flight per thread: a couple of CTAs per SM have few warps to hide the L2 latency with
  const float r = __frcp_rn(s);
  const bool r_finite = r <= 3.402823466e+38f;   // a row maximum below 448 * 2^-128 gives s without a finite fp32 reciprocal
  auto quant2 = [&](float a, float b) {
    // a / s, b / s correctly rounded (Markstein, as in the GEMM epilogue; a zero quotient keeps its sign)
    const float qa0 = a * r, qb0 = b * r;
    float qa = fmaf(fmaf(-qa0, s, a), r, qa0), qb = fmaf(fmaf(-qb0, s, b), r, qb0);
    qa = qa == 0.0f ? qa0 : qa;
    qb = qb == 0.0f ? qb0 : qb;
    if (!r_finite) { qa = __fdiv_rn(a, s); qb = __fdiv_rn(b, s); }   // uniform over the CTA (one row): IEEE division
    uint16_t o;
    asm("cvt.rn.satfinite.e4m3x2.f32 %0, %1, %2;" : "=h"(o) : "f"(qb), "f"(qa));
    return (uint32_t)o;
  };
#pragma unroll 1
  for (int i0 = threadIdx.x; i0 < n4; i0 += 4 * blockDim.x) {
    float4 v[4];
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if (i0 + k * blockDim.x < n4) v[k] = __ldcg(src + i0 + k * blockDim.x);
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if (i0 + k * blockDim.x < n4) dst[i0 + k * blockDim.x] = quant2(v[k].x, v[k].y) | (quant2(v[k].z, v[k].w) << 16);
  }
}

}  // namespace

int launch_requant_rows(const float* d_h, int rows, int cols, const float* d_amax_part, int n_part, int part_stride,
                        int block_rows, uint8_t* d_hq, float* d_sh, int sms, cudaStream_t stream) {
  cudaLaunchConfig_t cfg = {};
  int per_row = (2 * sms + rows - 1) / rows;                     // chunks per row: about two CTAs per SM in all
  per_row = per_row < 2 ? 2 : per_row;
  int chunk_cols = ((cols + per_row - 1) / per_row + 127) / 128 * 128;
  chunk_cols = chunk_cols < 1024 ? 1024 : chunk_cols;
  cfg.gridDim = dim3((unsigned)((cols + chunk_cols - 1) / chunk_cols), (unsigned)rows);
  cfg.blockDim = dim3(256);
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  const cudaError_t e = cudaLaunchKernelEx(&cfg, requant_rows_kernel, d_h, cols, chunk_cols, d_amax_part, n_part, part_stride, block_rows, d_hq, d_sh);
  return e == cudaSuccess ? SPENSE_OK : SPENSE_ERR_CUDA;
}

int launch_quantize(const float* d_in, int64_t rows, int64_t cols, int32_t mode, uint8_t* d_out, float* d_scales,
                    void* d_ws, cudaStream_t stream) {
  float* amax = reinterpret_cast<float*>(d_ws);
  row_amax_kernel<<<(unsigned)rows, 256, 0, stream>>>(d_in, cols, amax);
  const float* src = amax;
  if (mode == SPENSE_PER_TENSOR) {
    tensor_amax_kernel<<<1, 256, 0, stream>>>(amax, rows, amax + rows);
    src = amax + rows;
  }
  quantize_kernel<<<(unsigned)rows, 256, 0, stream>>>(d_in, cols, src, mode == SPENSE_PER_ROW, d_out, d_scales);
  return cudaGetLastError() == cudaSuccess ? SPENSE_OK : SPENSE_ERR_CUDA;
}

int launch_pack(const spense_shape_t* shape, const uint8_t* d_wgate, const uint8_t* d_wup, const uint8_t* d_wdown,
                const float* h_w_scale, const int32_t* d_perm, void* d_blob, const spense_canon_t* canon, void* d_ws,
                int64_t* h_err_where, cudaStream_t stream) {
  const Geometry g = make_geometry(shape->H, shape->I, shape->I_dense);
  PackErr* err = reinterpret_cast<PackErr*>(d_ws);
  int* marks = reinterpret_cast<int*>(reinterpret_cast<uint8_t*>(d_ws) + 128);
  spense_canon_t c = {};
  if (canon) c = *canon;
  pack_init_kernel<<<(g.I + 255) / 256, 256, 0, stream>>>(err, marks, g.I);
  PackErr herr;
  if (d_perm) {
    perm_mark_kernel<<<(g.I + 255) / 256, 256, 0, stream>>>(d_perm, marks, err, g.I);
    if (cudaMemcpyAsync(&herr, err, sizeof(herr), cudaMemcpyDeviceToHost, stream) != cudaSuccess) return SPENSE_ERR_CUDA;
    if (cudaStreamSynchronize(stream) != cudaSuccess) return SPENSE_ERR_CUDA;
    if (herr.perm_bad) return SPENSE_ERR_BAD_PERM;
  }
  BlobHeader hdr = {};
  hdr.magic = kBlobMagic; hdr.version = kBlobVersion;
  hdr.H = g.H; hdr.I = g.I; hdr.I_dense = g.I_d;
  hdr.w_scale[0] = h_w_scale[0]; hdr.w_scale[1] = h_w_scale[1]; hdr.w_scale[2] = h_w_scale[2];
  hdr.gate_up_off = g.gate_up_off; hdr.down_off = g.down_off; hdr.total_bytes = g.total_bytes;
  if (cudaMemsetAsync(d_blob, 0, kBlobHeaderBytes, stream) != cudaSuccess) return SPENSE_ERR_CUDA;
  write_header_kernel<<<1, 32, 0, stream>>>(reinterpret_cast<BlobHeader*>(d_blob), hdr);
  uint8_t* blob = reinterpret_cast<uint8_t*>(d_blob);
  pack_gate_up_kernel<<<dim3(g.I, 2), 256, 0, stream>>>(g, d_wgate, d_wup, d_perm, blob, c, err);
  pack_down_kernel<<<g.dn_tiles * 256, 256, 0, stream>>>(g, d_wdown, d_perm, blob, c, err, 2);
  if (cudaGetLastError() != cudaSuccess) return SPENSE_ERR_CUDA;
  if (cudaMemcpyAsync(&herr, err, sizeof(herr), cudaMemcpyDeviceToHost, stream) != cudaSuccess) return SPENSE_ERR_CUDA;
  if (cudaStreamSynchronize(stream) != cudaSuccess) return SPENSE_ERR_CUDA;
  auto fill = [&](unsigned long long key, unsigned long long cnt) {
    if (!h_err_where) return;
    h_err_where[0] = (int64_t)(key >> 56);
    h_err_where[1] = (int64_t)((key >> 28) & 0xFFFFFFFull);
    h_err_where[2] = (int64_t)(key & 0xFFFFFFFull);
    h_err_where[3] = (int64_t)cnt;
  };
  if (herr.nan_cnt) { fill(herr.nan_key, herr.nan_cnt); return SPENSE_ERR_NAN_WEIGHT; }
  if (herr.n24_cnt) { fill(herr.n24_key, herr.n24_cnt); return SPENSE_ERR_NOT_2_4; }
  return SPENSE_OK;
}

int launch_pack_linear(const spense_linear_shape_t* shape, const uint8_t* d_w, float w_scale, const int32_t* d_perm, void* d_blob,
                       const spense_linear_canon_t* canon, void* d_ws, int64_t* h_err_where, cudaStream_t stream) {
  const bool in_split = shape->split == SPENSE_SPLIT_IN;
  const Geometry g = make_geometry_linear(shape->N, shape->K, shape->n_dense, in_split);
  const int n_perm = in_split ? shape->K : shape->N;
  PackErr* err = reinterpret_cast<PackErr*>(d_ws);
  int* marks = reinterpret_cast<int*>(reinterpret_cast<uint8_t*>(d_ws) + 128);
  spense_linear_canon_t c = {};
  if (canon) c = *canon;
  pack_init_kernel<<<(n_perm + 255) / 256, 256, 0, stream>>>(err, marks, n_perm);
  PackErr herr;
  if (d_perm) {
    perm_mark_kernel<<<(n_perm + 255) / 256, 256, 0, stream>>>(d_perm, marks, err, n_perm);
    if (cudaMemcpyAsync(&herr, err, sizeof(herr), cudaMemcpyDeviceToHost, stream) != cudaSuccess) return SPENSE_ERR_CUDA;
    if (cudaStreamSynchronize(stream) != cudaSuccess) return SPENSE_ERR_CUDA;
    if (herr.perm_bad) return SPENSE_ERR_BAD_PERM;
  }
  BlobHeader hdr = {};
  hdr.magic = kBlobMagic; hdr.version = kBlobVersion;
  hdr.H = g.H; hdr.I = g.I; hdr.I_dense = g.I_d;
  hdr.w_scale[0] = hdr.w_scale[1] = hdr.w_scale[2] = w_scale;
  hdr.gate_up_off = kBlobHeaderBytes; hdr.down_off = kBlobHeaderBytes; hdr.total_bytes = g.total_bytes;
  hdr.kind = in_split ? kBlobLinearIn : kBlobLinearOut;
  if (cudaMemsetAsync(d_blob, 0, kBlobHeaderBytes, stream) != cudaSuccess) return SPENSE_ERR_CUDA;
  write_header_kernel<<<1, 32, 0, stream>>>(reinterpret_cast<BlobHeader*>(d_blob), hdr);
  uint8_t* blob = reinterpret_cast<uint8_t*>(d_blob);
  if (in_split) {
    spense_canon_t cc = {};
    cc.down_sp_val = c.sp_val; cc.down_sp_meta = c.sp_meta; cc.down_dn = c.dn;
    if (c.perm) copy_perm_kernel<<<(n_perm + 255) / 256, 256, 0, stream>>>(d_perm, c.perm, n_perm);
    pack_down_kernel<<<g.dn_tiles * 256, 256, 0, stream>>>(g, d_w, d_perm, blob, cc, err, 0);
  } else {
    pack_rows_kernel<<<g.gu_tiles * 256, 256, 0, stream>>>(g, d_w, d_perm, blob, c, err);
  }
  if (cudaGetLastError() != cudaSuccess) return SPENSE_ERR_CUDA;
  if (cudaMemcpyAsync(&herr, err, sizeof(herr), cudaMemcpyDeviceToHost, stream) != cudaSuccess) return SPENSE_ERR_CUDA;
  if (cudaStreamSynchronize(stream) != cudaSuccess) return SPENSE_ERR_CUDA;
  auto fill = [&](unsigned long long key, unsigned long long cnt) {
    if (!h_err_where) return;
    h_err_where[0] = (int64_t)(key >> 56);
    h_err_where[1] = (int64_t)((key >> 28) & 0xFFFFFFFull);
    h_err_where[2] = (int64_t)(key & 0xFFFFFFFull);
    h_err_where[3] = (int64_t)cnt;
  };
  if (herr.nan_cnt) { fill(herr.nan_key, herr.nan_cnt); return SPENSE_ERR_NAN_WEIGHT; }
  if (herr.n24_cnt) { fill(herr.n24_key, herr.n24_cnt); return SPENSE_ERR_NOT_2_4; }
  return SPENSE_OK;
}

}  // namespace spense

// ---------------------------------------------------------------- spense_quantize_e4m3_static (include/spense.h)
// The quantise helper for callers that have no device allocator to ask for the (rows + 1)-float scratch: the row maxima
// and the tensor maximum live in an array that is part of the library image.  Same three kernels as launch_quantize.
namespace spense {
namespace {

// Resident on every GPU that loads libspense.so, from load to process exit: 4 * (65536 + 64) bytes = 256.25 KB.
// Layout as in launch_quantize: [0, rows) row maxima, [rows] the tensor maximum.  Nothing in it has to start at zero
// (row_amax_kernel writes every slot the later kernels read), so calls do not clear it; it keeps the last call's values.
static __device__ __align__(256) float g_quant_scratch[SPENSE_QUANTIZE_STATIC_MAX_ROWS + 64];

std::mutex g_quant_mu;
float* g_quant_ptr[64];   // per device ordinal: the DEVICE address of g_quant_scratch on that device (null = not set up yet)

// In host code `g_quant_scratch` names a host-side shadow of the symbol, not memory a kernel can use: the address the
// kernels get is looked up once per device, with that device current.  Allocates nothing.
int quant_scratch_of_current_device(float** out) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return SPENSE_ERR_CUDA;
  std::lock_guard<std::mutex> lk(g_quant_mu);
  if (!g_quant_ptr[dev]) {
    int major = 0, minor = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev) != cudaSuccess)
      return SPENSE_ERR_CUDA;
    if (major != 10 || minor != 0) return SPENSE_ERR_ARCH;
    float* p = nullptr;
    if (cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_quant_scratch) != cudaSuccess || !p) return SPENSE_ERR_CUDA;
    g_quant_ptr[dev] = p;
  }
  *out = g_quant_ptr[dev];
  return SPENSE_OK;
}

}  // namespace
}  // namespace spense

extern "C" int spense_quantize_e4m3_static(const float* d_in, int64_t rows, int64_t cols, int32_t mode, uint8_t* d_out,
                                           float* d_scales, spense_stream_t stream) {
  if (!d_in || !d_out || !d_scales || rows < 1 || cols < 1 || (mode != SPENSE_PER_TENSOR && mode != SPENSE_PER_ROW))
    return SPENSE_ERR_ARG;
  if (rows > SPENSE_QUANTIZE_STATIC_MAX_ROWS) return SPENSE_ERR_STATIC_SCRATCH;
  float* scratch = nullptr;
  const int st = spense::quant_scratch_of_current_device(&scratch);
  if (st) return st;
  return spense::launch_quantize(d_in, rows, cols, mode, d_out, d_scales, scratch, reinterpret_cast<cudaStream_t>(stream));
}
