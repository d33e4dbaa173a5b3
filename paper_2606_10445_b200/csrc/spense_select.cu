// SpenseGPT+ dense-index selection on the GPU (Eqs. 8-12):
//   s^gate_i = 1/H sum_j |Wg[i,j]| sqrt(Hx[j]),  s^up likewise,  s^down_i = sqrt(Hh[i]) / H sum_n |Wd[n,i]|   (Eq. 9)
//   s_i = sum over the three of s^mlp_i / (mean(s^mlp) + eps)                                                (Eqs. 10-11)
//   D = the I_dense indices of largest s (ties to the lower index), ascending; perm = stable partition         (Eq. 12, Q9)
// All three passes are HBM-bound reads of the fp32 weights (3 * I * H * 4 bytes, once).  Every reduction runs in
// a fixed order, so the scores and the selection are bitwise reproducible.
// Also the first slice of the pruning front-end (NEXT-4): magnitude 2:4 pruning of the sparse region in permuted order.
#include "spense_internal.cuh"

namespace spense {
namespace {

__device__ __forceinline__ float block_sum(float v, float* red) {      // fixed tree: deterministic
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x < 32) {
    v = threadIdx.x < (blockDim.x >> 5) ? red[threadIdx.x] : 0.0f;
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (threadIdx.x == 0) red[0] = v;
  }
  __syncthreads();
  const float r = red[0];
  __syncthreads();
  return r;
}

// one block per row i of W [I, H]: out[i] = 1/H sum_j |W[i,j]| * sqrt(hx[j])
__global__ void __launch_bounds__(256) row_score_kernel(const float* __restrict__ w, const float* __restrict__ hx, int H,
                                                        float* __restrict__ out) {
  __shared__ float red[32];
  const float4* row = reinterpret_cast<const float4*>(w + (size_t)blockIdx.x * H);
  const float4* h4 = reinterpret_cast<const float4*>(hx);
  float acc = 0.0f;
  for (int j = threadIdx.x; j < (H >> 2); j += blockDim.x) {            // H % 128 == 0
    const float4 a = __ldcs(row + j);
    const float4 b = __ldg(h4 + j);
    acc += fabsf(a.x) * sqrtf(b.x) + fabsf(a.y) * sqrtf(b.y) + fabsf(a.z) * sqrtf(b.z) + fabsf(a.w) * sqrtf(b.w);
  }
  acc = block_sum(acc, red);
  if (threadIdx.x == 0) out[blockIdx.x] = acc / (float)H;
}

// W [H, I] column sums in two fixed-order steps: block (c, r) adds |W| over 64 rows for 1024 columns (whole 4 KB row
// segments: sequential DRAM pages), then one thread per column adds the H/64 partial sums in row order.
constexpr int kColRows = 64;
__global__ void __launch_bounds__(256) col_partial_kernel(const float* __restrict__ w, int H, int I, float* __restrict__ part) {
  const int c4 = blockIdx.x * 256 + threadIdx.x;                        // float4 column group
  if (c4 * 4 >= I) return;
  const int n0 = blockIdx.y * kColRows, n1 = min(H, n0 + kColRows);
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  for (int n = n0; n < n1; ++n) {
    const float4 v = __ldcs(reinterpret_cast<const float4*>(w + (size_t)n * I) + c4);
    acc.x += fabsf(v.x); acc.y += fabsf(v.y); acc.z += fabsf(v.z); acc.w += fabsf(v.w);
  }
  reinterpret_cast<float4*>(part + (size_t)blockIdx.y * I)[c4] = acc;
}
__global__ void __launch_bounds__(256) col_final_kernel(const float* __restrict__ part, const float* __restrict__ hh, int H, int I,
                                                        int n_chunks, float* __restrict__ out) {
  const int col = blockIdx.x * 256 + threadIdx.x;
  if (col >= I) return;
  float s = 0.0f;
  for (int k = 0; k < n_chunks; ++k) s += part[(size_t)k * I + col];
  out[col] = s * sqrtf(hh[col]) / (float)H;
}

// one block: the three means (Eq. 10), then s_i (Eq. 11)
__global__ void __launch_bounds__(1024) combine_kernel(const float* __restrict__ sg, const float* __restrict__ su,
                                                       const float* __restrict__ sd, int I, float eps, float* __restrict__ score) {
  __shared__ float red[32];
  float a = 0.0f, b = 0.0f, c = 0.0f;
  for (int i = threadIdx.x; i < I; i += blockDim.x) { a += sg[i]; b += su[i]; c += sd[i]; }
  const float mg = block_sum(a, red) / (float)I + eps;
  const float mu = block_sum(b, red) / (float)I + eps;
  const float md = block_sum(c, red) / (float)I + eps;
  for (int i = threadIdx.x; i < I; i += blockDim.x) score[i] = sg[i] / mg + su[i] / mu + sd[i] / md;
}

// Radix select (one block): T = bits of the I_dense-th largest score (scores are >= 0, so the bit pattern orders
// like the value) and how many indices with score == T belong to the set (the lowest ones: ties to the lower index).
__global__ void __launch_bounds__(1024) threshold_kernel(const float* __restrict__ score, int I, int K, uint32_t* __restrict__ out) {
  __shared__ int hist[256];
  __shared__ uint32_t prefix, mask;
  __shared__ int k_rem;
  if (threadIdx.x == 0) { prefix = 0; mask = 0; k_rem = K; }
  __syncthreads();
  if (K <= 0) {                                                         // nothing is dense: threshold above every key
    if (threadIdx.x == 0) { out[0] = 0xFFFFFFFFu; out[1] = 0; }
    return;
  }
  for (int shift = 24; shift >= 0; shift -= 8) {
    if (threadIdx.x < 256) hist[threadIdx.x] = 0;
    __syncthreads();
    for (int i = threadIdx.x; i < I; i += blockDim.x) {
      const uint32_t key = __float_as_uint(score[i]);
      if ((key & mask) == prefix) atomicAdd(&hist[(key >> shift) & 255u], 1);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      int d = 255;
      while (d > 0 && hist[d] < k_rem) { k_rem -= hist[d]; --d; }
      prefix |= (uint32_t)d << shift;
      mask |= 255u << shift;
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) { out[0] = prefix; out[1] = (uint32_t)k_rem; }
}

// one block: stable partition -> dense_idx ascending, perm = [sparse ascending | dense ascending].
// dense(i) = key_i > T, or key_i == T and fewer than `need` equal keys lie below i.
__global__ void __launch_bounds__(1024) partition_kernel(const float* __restrict__ score, const uint32_t* __restrict__ thr, int I,
                                                         int I_dense, int* __restrict__ dense_idx, int* __restrict__ perm) {
  __shared__ int warp_eq[32], warp_d[32];
  __shared__ int base_eq, base_d;
  const uint32_t T = thr[0];
  const int need = (int)thr[1];
  if (threadIdx.x == 0) { base_eq = 0; base_d = 0; }
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int i0 = 0; i0 < I; i0 += 1024) {
    const int i = i0 + threadIdx.x;
    const uint32_t key = i < I ? __float_as_uint(score[i]) : 0u;
    const int eq = (i < I && key == T) ? 1 : 0;
    int eq_incl = eq;                                                   // inclusive scan of the equal-key flags
    for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, eq_incl, o); if (lane >= o) eq_incl += t; }
    if (lane == 31) warp_eq[wid] = eq_incl;
    __syncthreads();
    int eq_off = 0;
    for (int k = 0; k < wid; ++k) eq_off += warp_eq[k];
    const int eq_before = base_eq + eq_off + eq_incl - eq;
    const int f = (i < I && (key > T || (eq && eq_before < need))) ? 1 : 0;
    int incl = f;                                                       // inclusive scan of the dense flags
    for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += t; }
    if (lane == 31) warp_d[wid] = incl;
    __syncthreads();
    int d_off = 0;
    for (int k = 0; k < wid; ++k) d_off += warp_d[k];
    const int d_before = base_d + d_off + incl - f;                     // dense indices below i
    if (i < I) {
      if (f) { dense_idx[d_before] = i; perm[(I - I_dense) + d_before] = i; }
      else perm[i - d_before] = i;
    }
    __syncthreads();
    if (threadIdx.x == 1023) { base_eq += eq_off + eq_incl; base_d += d_off + incl; }
    __syncthreads();
  }
}

// ---------------------------------------------------------------- magnitude 2:4 pruning (first slice)
// keep mask of one group of 4: the 2 entries of largest |w|, ties to the lower index
__device__ __forceinline__ int keep_mask_2of4(float a0, float a1, float a2, float a3) {
  const float m[4] = {fabsf(a0), fabsf(a1), fabsf(a2), fabsf(a3)};
  int mask = 0;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    int beats = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j)
      if (j != i) beats += (m[j] > m[i] || (m[j] == m[i] && j < i)) ? 1 : 0;
    if (beats < 2) mask |= 1 << i;
  }
  return mask;
}

// rows [0, I_s) of P^T W (gate or up), groups of 4 along H: one thread per group, in place
__global__ void __launch_bounds__(256) prune_rows_kernel(float* __restrict__ w, const int32_t* __restrict__ perm, int H, int I_s) {
  const int groups = H >> 2;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (long long)I_s * groups) return;
  const int r = (int)(i / groups), g = (int)(i - (long long)r * groups);
  float4* ptr = reinterpret_cast<float4*>(w + (size_t)(perm ? perm[r] : r) * H) + g;
  float4 v = *ptr;
  const int k = keep_mask_2of4(v.x, v.y, v.z, v.w);
  if (!(k & 1)) v.x = 0.0f;
  if (!(k & 2)) v.y = 0.0f;
  if (!(k & 4)) v.z = 0.0f;
  if (!(k & 8)) v.w = 0.0f;
  *ptr = v;
}

// columns [0, I_s) of W_down P, groups of 4 along the PERMUTED intermediate dimension: one thread per (row, group)
__global__ void __launch_bounds__(256) prune_cols_kernel(float* __restrict__ w, const int32_t* __restrict__ perm, int I, int I_s, int H) {
  const int groups = I_s >> 2;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (long long)H * groups) return;
  const int n = (int)(i / groups), g = (int)(i - (long long)n * groups);
  float* row = w + (size_t)n * I;
  int c[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) c[k] = perm ? perm[4 * g + k] : 4 * g + k;
  const int keep = keep_mask_2of4(row[c[0]], row[c[1]], row[c[2]], row[c[3]]);
#pragma unroll
  for (int k = 0; k < 4; ++k)
    if (!(keep & (1 << k))) row[c[k]] = 0.0f;
}

}  // namespace

int launch_prune(const spense_shape_t* shape, float* d_wgate, float* d_wup, float* d_wdown, const int32_t* d_perm, cudaStream_t stream) {
  const int H = shape->H, I = shape->I, I_s = shape->I - shape->I_dense;
  if (I_s == 0) return SPENSE_OK;
  const long long n_rows = (long long)I_s * (H >> 2), n_cols = (long long)H * (I_s >> 2);
  prune_rows_kernel<<<(unsigned)((n_rows + 255) / 256), 256, 0, stream>>>(d_wgate, d_perm, H, I_s);
  prune_rows_kernel<<<(unsigned)((n_rows + 255) / 256), 256, 0, stream>>>(d_wup, d_perm, H, I_s);
  prune_cols_kernel<<<(unsigned)((n_cols + 255) / 256), 256, 0, stream>>>(d_wdown, d_perm, I, I_s, H);
  return cudaGetLastError() == cudaSuccess ? SPENSE_OK : SPENSE_ERR_CUDA;
}

int launch_select(const spense_shape_t* shape, const float* d_wgate, const float* d_wup, const float* d_wdown,
                  const float* d_hdiag_x, const float* d_hdiag_h, float eps, float* d_score, int32_t* d_dense_idx,
                  int32_t* d_perm, void* d_ws, cudaStream_t stream) {
  const int H = shape->H, I = shape->I;
  float* sg = reinterpret_cast<float*>(d_ws);
  float* su = sg + I;
  float* sd = su + I;
  float* score = d_score ? d_score : sd + I;
  uint32_t* thr = reinterpret_cast<uint32_t*>(sd + 2 * (size_t)I);
  float* part = reinterpret_cast<float*>(thr + I);
  const int n_chunks = (H + kColRows - 1) / kColRows;
  row_score_kernel<<<I, 256, 0, stream>>>(d_wgate, d_hdiag_x, H, sg);
  row_score_kernel<<<I, 256, 0, stream>>>(d_wup, d_hdiag_x, H, su);
  col_partial_kernel<<<dim3((I / 4 + 255) / 256, n_chunks), 256, 0, stream>>>(d_wdown, H, I, part);
  col_final_kernel<<<(I + 255) / 256, 256, 0, stream>>>(part, d_hdiag_h, H, I, n_chunks, sd);
  combine_kernel<<<1, 1024, 0, stream>>>(sg, su, sd, I, eps, score);
  threshold_kernel<<<1, 1024, 0, stream>>>(score, I, shape->I_dense, thr);
  partition_kernel<<<1, 1024, 0, stream>>>(score, thr, I, shape->I_dense, d_dense_idx, d_perm);
  return cudaGetLastError() == cudaSuccess ? SPENSE_OK : SPENSE_ERR_CUDA;
}

}  // namespace spense
