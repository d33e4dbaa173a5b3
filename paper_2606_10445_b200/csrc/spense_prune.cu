// SparseGPT's 2:4 column sweep with the dense columns on the right as compensation buffer (PAPER.md:98-111
// Eqs. 2-3).  Offline, fp32, plain CUDA cores: the sweep is sequential along K, parallel over rows.
//
// W [N, K] row-major, columns in PERMUTED order (sparse columns [0, K_s) first), pruned and compensated IN PLACE.
// U [K, K] upper triangular with H^-1 = U^T U (the caller factorises the damped Hessian with a library routine): row j of
// the inverse Hessian of the not yet processed columns is U[j][j] * U[j][j:], so Eq. 3 for a pruned weight w_j reads
//     e = w_j / U[j][j],   w[c] -= e * U[j][c]  for the unprocessed columns c > j,   w_j = 0,
// and its error eps_j = w_j^2 / U[j][j]^2.  Columns are taken in blocks of 128: obs_block_kernel sweeps a block (one thread
// per row, the block of W and the diagonal block of U in shared memory) and leaves the e of every (row, column) in Err;
// obs_trailing_kernel applies them to all columns right of the block at once, W[:, j1:] -= Err @ U[j0:j1, j1:].
#include "spense_internal.cuh"

namespace spense {

namespace {

constexpr int kObsBlock = 128;      // columns per block
constexpr int kObsRows = 128;       // rows per CTA of the block sweep (one thread each)
constexpr int kObsLd = kObsBlock + 1;   // padded row stride of the W tile: thread r, column c -> bank (r + c) % 32

// One block of columns [j0, j0 + cols): cols <= 128, cols % 4 == 0.  Dynamic smem: W tile [128][129] + U block [128][128].
__global__ void __launch_bounds__(kObsRows) obs_block_kernel(float* __restrict__ w, const float* __restrict__ u, int N, int K, int j0, int cols,
                                                             float* __restrict__ err) {
  extern __shared__ float sm[];
  float* wt = sm;                                  // [kObsRows][kObsLd]
  float* ub = sm + kObsRows * kObsLd;              // [kObsBlock][kObsBlock]: U[j0 + a][j0 + b]
  const int r0 = blockIdx.x * kObsRows;
  const int t = threadIdx.x;
  // coalesced loads: consecutive threads read consecutive columns
  for (int i = t; i < kObsRows * cols; i += kObsRows) {
    const int r = i / cols, c = i - r * cols;
    wt[r * kObsLd + c] = r0 + r < N ? w[(size_t)(r0 + r) * K + j0 + c] : 0.0f;
  }
  for (int i = t; i < cols * cols; i += kObsRows) {
    const int a = i / cols, b = i - a * cols;
    ub[a * kObsBlock + b] = u[(size_t)(j0 + a) * K + j0 + b];
  }
  __syncthreads();
  float* row = wt + t * kObsLd;
  unsigned prune4 = 0;                             // bit c: column j + c of the current group is to be pruned
  for (int j = 0; j < cols; ++j) {
    if ((j & 3) == 0) {
      // "within each group, SparseGPT selects the weights to prune using the OBS-based error criterion":
      // eps_c = w_c^2 / U_cc^2 with the current w; the 2 smallest go, ties to the lower column
      float eps[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const float d = ub[(j + c) * kObsBlock + j + c];
        eps[c] = __fdiv_rn(row[j + c] * row[j + c], d * d);
      }
      prune4 = 0;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        int rank = 0;
#pragma unroll
        for (int o = 0; o < 4; ++o) rank += (eps[o] < eps[c]) || (eps[o] == eps[c] && o < c);
        if (rank < 2) prune4 |= 1u << c;
      }
    }
    float e = 0.0f;
    if ((prune4 >> (j & 3)) & 1u) {
      e = __fdiv_rn(row[j], ub[j * kObsBlock + j]);
      row[j] = 0.0f;
      const float* uj = ub + j * kObsBlock;
      for (int c = j + 1; c < cols; ++c) row[c] = fmaf(-e, uj[c], row[c]);
    }
    if (r0 + t < N) err[(size_t)(r0 + t) * kObsBlock + j] = e;
  }
  __syncthreads();
  for (int i = t; i < kObsRows * cols; i += kObsRows) {
    const int r = i / cols, c = i - r * cols;
    if (r0 + r < N) w[(size_t)(r0 + r) * K + j0 + c] = wt[r * kObsLd + c];
  }
}

// W[:, j1:K] -= Err[N, cols] @ U[j0:j0+cols, j1:K].  64 x 64 output tile per CTA, 256 threads x (4 x 4), the whole
// reduction dimension (cols <= 128) staged in two halves.
constexpr int kTile = 64;
__global__ void __launch_bounds__(256) obs_trailing_kernel(float* __restrict__ w, const float* __restrict__ u, const float* __restrict__ err, int N, int K,
                                                           int j0, int cols, int j1) {
  constexpr int kChunk = 64;                       // reduction columns staged at a time
  __shared__ float se[kChunk][kTile + 1];          // Err^T tile: [k][row]
  __shared__ float su[kChunk][kTile];              // U tile:     [k][col]
  const int r0 = blockIdx.y * kTile, c0 = j1 + blockIdx.x * kTile;
  const int t = threadIdx.x;
  const int tr = (t / 16) * 4, tc = (t % 16) * 4;
  float acc[4][4] = {};
  for (int k0 = 0; k0 < cols; k0 += kChunk) {
    const int kc = cols - k0 < kChunk ? cols - k0 : kChunk;
    __syncthreads();
    for (int i = t; i < kTile * kc; i += 256) {
      const int r = i / kc, k = i - r * kc;        // consecutive threads: consecutive k of one row (contiguous in Err)
      se[k][r] = r0 + r < N ? err[(size_t)(r0 + r) * kObsBlock + k0 + k] : 0.0f;
    }
    for (int i = t; i < kc * kTile; i += 256) {
      const int k = i / kTile, c = i - k * kTile;
      su[k][c] = c0 + c < K ? u[(size_t)(j0 + k0 + k) * K + c0 + c] : 0.0f;
    }
    __syncthreads();
    for (int k = 0; k < kc; ++k) {
      float a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) { a[i] = se[k][tr + i]; b[i] = su[k][tc + i]; }
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int jx = 0; jx < 4; ++jx) acc[i][jx] = fmaf(a[i], b[jx], acc[i][jx]);
    }
  }
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int jx = 0; jx < 4; ++jx) {
      const int r = r0 + tr + i, c = c0 + tc + jx;
      if (r < N && c < K) w[(size_t)r * K + c] -= acc[i][jx];
    }
}

}  // namespace

int launch_prune_obs(int N, int K, int K_sparse, float* d_w, const float* d_u, void* d_ws, cudaStream_t stream) {
  float* err = reinterpret_cast<float*>(d_ws);
  const size_t smem = (size_t)(kObsRows * kObsLd + kObsBlock * kObsBlock) * sizeof(float);
  if (cudaFuncSetAttribute(obs_block_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return SPENSE_ERR_CUDA;
  for (int j0 = 0; j0 < K_sparse; j0 += kObsBlock) {
    const int cols = K_sparse - j0 < kObsBlock ? K_sparse - j0 : kObsBlock;
    // W is swept in place: a launch that is refused is reported at once, before the next block builds on a matrix
    // that is only partly processed (the caller must then treat d_w as undefined)
    obs_block_kernel<<<(N + kObsRows - 1) / kObsRows, kObsRows, smem, stream>>>(d_w, d_u, N, K, j0, cols, err);
    if (cudaGetLastError() != cudaSuccess) return SPENSE_ERR_CUDA;
    const int j1 = j0 + cols;
    if (j1 < K) {
      obs_trailing_kernel<<<dim3((K - j1 + kTile - 1) / kTile, (N + kTile - 1) / kTile), 256, 0, stream>>>(d_w, d_u, err, N, K, j0, cols, j1);
      if (cudaGetLastError() != cudaSuccess) return SPENSE_ERR_CUDA;
    }
  }
  return SPENSE_OK;
}

}  // namespace spense
