/*
 * spense.h -- C ABI of the B200-native Spense hybrid sparse-dense FP8 GLU-MLP library.
 *
 * Method: arxiv/paper_2606_10445 (SpenseGPT).  Citations are lines of the paper text.
 *   - 2:4 semi-structured sparsity along K, ||W[i,4j:4j+4]||_0 <= 2          Eq. 1
 *   - compressed storage = non-zero values + a few position bits per group
 *   - Spense format: one contiguous 2:4 region + one contiguous dense region   Sec. 3.2
 *   - output-split (W_gate, W_up) and input-split (W_down, sparse then dense
 *     accumulated into the same output)                                        Sec. 3.2
 *   - intermediate-index permutation P, MLP(X) unchanged                       Eq. 4
 *   - dense indices placed last
 *
 * Conventions
 *   - Layout is PyTorch's: Y = X W^T, W in R^{N x K} row-major, X in R^{M x K}.
 *     H = hidden size, I = intermediate size, I_dense = number of dense intermediate indices,
 *     I_s = I - I_dense.  In PERMUTED intermediate order the sparse region is [0, I_s) and the dense
 *     region is [I_s, I).  W_gate, W_up are [I, H]; W_down is [H, I].
 *   - FP8 is E4M3 (FN: bias 7, no inf, NaN = 0x7F/0xFF, max 448), stored as uint8_t.
 *     Weights carry one fp32 scale per matrix, activations one fp32 scale per token.
 *   - Pointers prefixed d_ are DEVICE pointers, h_ are HOST pointers.  The library allocates no
 *     device memory: the caller owns every buffer; size queries say how large they must be.
 *     Device pointers must be 128-byte aligned.
 *   - Every call returns a status (0 = SPENSE_OK, negative = error).  Nothing throws, aborts or
 *     prints.  Argument errors are detected on the host before any launch.
 *   - All GPU work is enqueued on the caller's stream.  GEMM calls never synchronise and never read device
 *     memory on the host: the first call on a fresh blob may be issued inside a CUDA stream capture.  The library's
 *     one-time set-up per process and device (a pinned host status word, a driver entry point, per-kernel attributes)
 *     is done by spense_workspace_init, which every GEMM caller has to call anyway and which must NOT be captured.
 *     spense_pack synchronises the stream once to read back its validation word.
 *   - What only the device can see is reported through a pinned host status word (spense_device_status):
 *     the blob header (magic, version, shape) is checked by the kernels that read the weight scales from it
 *     (SPENSE_ERR_BAD_BLOB), and a CTA that waits more than 2 s for the other CTAs of its launch records
 *     SPENSE_ERR_TIMEOUT and traps instead of hanging.  A recorded error is returned by every later GEMM call
 *     until it is cleared.  The two differ in what survives them: after SPENSE_ERR_BAD_BLOB the launch has ended
 *     normally (nothing stored) and clearing the word is all it takes to go on.  SPENSE_ERR_TIMEOUT is FATAL to the
 *     process's CUDA context: the trap is a sticky launch failure, every later CUDA call of the process (the
 *     caller's own included) fails, device memory of the context is lost, and clearing the word recovers nothing --
 *     the word, which lives in host memory, is there so that the process can still say WHY before it exits.
 *   - There is NO CPU fallback: on a device that is not sm_100 the calls return SPENSE_ERR_ARCH.
 */
#ifndef SPENSE_H_
#define SPENSE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct CUstream_st* spense_stream_t; /* == cudaStream_t */

enum {
  SPENSE_OK = 0,
  SPENSE_ERR_ARG = -1,              /* null pointer, M < 1 or M > 2^20, bad enum */
  SPENSE_ERR_ALIGN = -2,            /* pointer not aligned as required */
  SPENSE_ERR_SHAPE = -3,            /* H, I, I_dense not multiples of 128, I_dense > I, too large */
  SPENSE_ERR_BUFFER_TOO_SMALL = -4, /* blob_bytes / ws_bytes below the size query */
  SPENSE_ERR_NOT_2_4 = -5,          /* a sparse-region group of 4 has > 2 non-zero bytes */
  SPENSE_ERR_NAN_WEIGHT = -6,       /* a weight byte is 0x7F / 0xFF */
  SPENSE_ERR_BAD_PERM = -7,         /* perm is not a bijection of [0, I) */
  SPENSE_ERR_ARCH = -8,             /* current device is not sm_100 */
  SPENSE_ERR_CUDA = -9,             /* a CUDA call failed; cudaGetLastError is preserved */
  SPENSE_ERR_BAD_BLOB = -10,        /* blob header does not match the shape / version (detected on the device) */
  SPENSE_ERR_TIMEOUT = -11,         /* a CTA gave up waiting for the other CTAs of its launch (detected on the device);
                                       the kernel trapped: the CUDA context is lost, restart the process */
  SPENSE_ERR_STATIC_SCRATCH = -12   /* the request does not fit the built-in scratch of an allocation-free entry point */
};

enum { SPENSE_F32 = 0, SPENSE_BF16 = 1 };          /* y_dtype */
enum { SPENSE_PER_TENSOR = 0, SPENSE_PER_ROW = 1 }; /* quantise mode */

typedef struct {
  int32_t H;       /* hidden size,        multiple of 128 */
  int32_t I;       /* intermediate size,  multiple of 128 */
  int32_t I_dense; /* dense intermediate indices (last block after permutation), multiple of 128, 0..I */
} spense_shape_t;

/* Canonical (layout-independent) result of the pack, DEVICE arrays owned by the caller; any member
 * may be NULL (not written).  Encoding (readings Q6/Q7):
 *   vals[r, 2g], vals[r, 2g+1] = the bytes at positions i0 < i1 of group g of row r;
 *   nibble(g) = i0 | i1 << 2;  meta byte b of a row = nibble(2b) | nibble(2b+1) << 4.            */
typedef struct {
  int32_t* perm;         /* [I]         new -> old (as used)                                  */
  uint8_t* gate_sp_val;  /* [I_s, H/2]                                                         */
  uint8_t* up_sp_val;    /* [I_s, H/2]                                                         */
  uint8_t* gate_sp_meta; /* [I_s, H/8]                                                         */
  uint8_t* up_sp_meta;   /* [I_s, H/8]                                                         */
  uint8_t* gate_dn;      /* [I_dense, H]                                                       */
  uint8_t* up_dn;        /* [I_dense, H]                                                       */
  uint8_t* down_sp_val;  /* [H, I_s/2]                                                         */
  uint8_t* down_sp_meta; /* [H, I_s/8]                                                         */
  uint8_t* down_dn;      /* [H, I_dense]                                                       */
} spense_canon_t;

int spense_version(void);
const char* spense_strerror(int status);

/* The first error a kernel of an earlier launch recorded (SPENSE_OK if none): SPENSE_ERR_BAD_BLOB or
 * SPENSE_ERR_TIMEOUT.  Host only; meaningful once the launches in question have completed (synchronise the
 * stream first -- after a time-out that synchronise itself returns a CUDA error, the word is still readable).
 * clear != 0 resets the word (enough to continue after BAD_BLOB; after TIMEOUT the context is gone, see above).                                                            */
int spense_device_status(int clear);

/* Host helper (Sec. 3.3.1; reading Q9): the permutation that moves the chosen dense
 * indices to the back, keeping ascending original order inside both regions.  h_perm[new] = old. */
int spense_perm_from_dense_idx(int32_t I, const int32_t* h_dense_idx, int32_t n_dense, int32_t* h_perm);

/* Host helper: the SpenseGPT choice of dense indices (Eq. 5, reading Q1): the LAST n_dense of the
 * I intermediate indices, ascending.  (SpenseGPT+'s choice is spense_select_dense.)                          */
int spense_dense_idx_last(int32_t I, int32_t n_dense, int32_t* h_dense_idx);

/* Bytes of the packed blob and of the pack workspace for a shape. */
int spense_pack_sizes(const spense_shape_t* shape, size_t* blob_bytes, size_t* workspace_bytes);

/* spense_pack -- "When deploying, we rearrange the indices for kernel efficiency" (Fig. 4,
 * PAPER.md:137): P1 permute the intermediate indices (rows of W_gate / W_up, columns of W_down),
 * P2 validate Eq. 1 on the sparse region and compress it to values + 2-bit position metadata
 * (PAPER.md:74), P3 re-tile everything into the opaque device blob the GEMM kernels stream.
 *   d_wgate, d_wup [I, H], d_wdown [H, I]: E4M3 bytes in ORIGINAL index order (read only).
 *   h_w_scale[3]: per-tensor fp32 scales of gate, up, down (host), stored in the blob header.
 *   d_perm [I] (device) new -> old, or NULL for the identity.
 *   d_blob / blob_bytes: output; canon: optional canonical outputs (NULL or members NULL).
 *   d_ws / ws_bytes: scratch.  h_err_where[4] (nullable, host): on NOT_2_4 / NAN_WEIGHT receives
 *   {matrix (0 gate, 1 up, 2 down), row, group, number of offending groups}; first offender in
 *   (matrix, row, group) order.  On error the blob contents are undefined.                       */
int spense_pack(const spense_shape_t* shape, const uint8_t* d_wgate, const uint8_t* d_wup,
                const uint8_t* d_wdown, const float* h_w_scale, const int32_t* d_perm, void* d_blob,
                size_t blob_bytes, const spense_canon_t* canon, void* d_ws, size_t ws_bytes,
                int64_t* h_err_where, spense_stream_t stream);

/* Workspace for the GEMM calls at up to M tokens (split-K partial tiles, flags, a launch-epoch word).
 * The workspace must be initialised ONCE with spense_workspace_init before its first use (outside stream capture: the
 * call also performs the library's one-time set-up for the current device, which allocates a few pinned host bytes); every
 * launch advances the epoch word, so nothing needs resetting between calls or CUDA-graph replays.
 * One workspace must not be used by two streams concurrently.  The CTAs of one GEMM launch wait
 * for each other (split-K fix-up): the calls refuse (SPENSE_ERR_CUDA) a grid the device cannot hold resident at
 * once, and a launch starved of SMs by other work ends with SPENSE_ERR_TIMEOUT (a trap: fatal to the CUDA context,
 * but reported) instead of hanging.                                                                         */
int spense_workspace_size(const spense_shape_t* shape, int32_t M, size_t* bytes);
int spense_workspace_init(void* d_ws, size_t ws_bytes, spense_stream_t stream);

/* Launch geometry the library uses for (shape, M tokens, mode 0 = gate_up / 1 = down) on a device with `sms` SMs
 * (host only, no device needed): the stream-K schedule cuts the linear sequence of weight stages (the byte order of
 * the blob) into spans of equal cost, one persistent CTA pair per span.  Writes
 * n_spans + 1 span boundaries (linear stage indices) into span_begin (room for 161 ints) and returns n_spans, or a
 * negative status.  info (nullable, 6 ints) = {stages, token blocks per launch, token columns per block, ring
 * slots, token blocks, CTAs per span}.  Every CTA of a launch must be resident at the same time: the grid is
 * info[1] * n_spans * info[5] CTAs at one CTA per SM.                                                       */
int spense_schedule(const spense_shape_t* shape, int32_t M, int32_t mode, int32_t sms, int32_t* span_begin, int32_t* info);

/* spense_gate_up -- output-split Spense GEMM for W_gate and W_up fused with the GLU
 * (Eq. 4, sigma = SiLU) and FP8 re-quantisation for the down projection:
 *   g = (X Wg^T) * s_x[m] * s_gate,  u = (X Wu^T) * s_x[m] * s_up,  h = g / (1 + exp(-g)) * u,
 *   hq[m, j] = E4M3_rne_sat(h[m, j] / s_h[m])          (j in PERMUTED intermediate order)
 * Row tiles j < I_s run on 2:4 sparse tensor-core MMAs, the others on dense MMAs.
 *   d_x [M, H] E4M3, d_sx [M] fp32; d_sh: requant scale, sh_stride 0 = one scalar, 1 = per token.
 *   d_hq [M, I] E4M3 out; d_h_f32 nullable [M, I] fp32 out (h before re-quantisation, for parity). */
int spense_gate_up(const spense_shape_t* shape, const void* d_blob, const uint8_t* d_x,
                   const float* d_sx, int32_t M, const float* d_sh, int32_t sh_stride, uint8_t* d_hq,
                   float* d_h_f32, void* d_ws, size_t ws_bytes, spense_stream_t stream);

/* spense_down -- input-split Spense GEMM: the K loop runs the sparse K range
 * [0, I_s) on sparse MMAs and continues with the dense range [I_s, I) into the SAME accumulator:
 *   y[m, n] = (sum_k hq[m, k] * Wd[n, k]) * s_h[m] * s_down.
 *   d_hq [M, I] E4M3 (permuted order); d_y [M, H] fp32 (SPENSE_F32) or bf16 (SPENSE_BF16).
 *   d_next_blob (nullable): packed blob of the layer that runs NEXT on this stream, same shape; while
 *   this launch drains, the first stages that layer's gate_up will stream are prefetched into L2
 *   (a performance hint only: results never depend on it).                                         */
int spense_down(const spense_shape_t* shape, const void* d_blob, const uint8_t* d_hq, const float* d_sh,
                int32_t sh_stride, int32_t M, void* d_y, int32_t y_dtype, void* d_ws, size_t ws_bytes,
                const void* d_next_blob, spense_stream_t stream);

/* spense_mlp -- the whole layer: gate_up then down on one stream (programmatic dependent launch).
 *   d_hq_scratch [M, I] E4M3 scratch; d_h_f32 nullable as in spense_gate_up; d_next_blob nullable as
 *   in spense_down.                                                                               */
int spense_mlp(const spense_shape_t* shape, const void* d_blob, const uint8_t* d_x, const float* d_sx,
               int32_t M, const float* d_sh, int32_t sh_stride, uint8_t* d_hq_scratch, float* d_h_f32,
               void* d_y, int32_t y_dtype, void* d_ws, size_t ws_bytes, const void* d_next_blob,
               spense_stream_t stream);

/* spense_mlp_dyn -- the whole layer with DYNAMIC per-token re-quantisation of h (the
 * paper's FP8 serving runs quantise activations dynamically): the scale is not an input,
 *   s_h[m] = max_j |h[m, j]| / 448   (fp32 division; 1 if the row is all zero),
 *   Hq[m, j] = E4M3_rne_sat(h[m, j] / s_h[m]),   y as in spense_down with that s_h.
 * Three stream-ordered steps (programmatic dependent launch): gate_up leaves h in fp32 in d_h_scratch and
 * the per-CTA maxima of |h| in the workspace, a row kernel forms s_h and Hq, down consumes them.
 *   d_sh_out [M] fp32 (written); d_hq_scratch [M, I] bytes (written); d_h_scratch [M, I] fp32 (written);
 *   other arguments as in spense_mlp.  Same status codes.                                            */
int spense_mlp_dyn(const spense_shape_t* shape, const void* d_blob, const uint8_t* d_x, const float* d_sx,
                   int32_t M, float* d_sh_out, uint8_t* d_hq_scratch, float* d_h_scratch, void* d_y,
                   int32_t y_dtype, void* d_ws, size_t ws_bytes, const void* d_next_blob,
                   spense_stream_t stream);

/* spense_mlp_host -- same, with HOST activations and results: copies h_x [M, H], h_sx [M], h_sh
 * (1 or M floats) to the device staging buffers, runs spense_mlp, copies y back to h_y and
 * synchronises the stream.  Staging (device): d_x [M, H], d_scales [2*M] fp32, d_hq_scratch [M, I],
 * d_y [M, H] of y_dtype.  Host buffers should be pinned for full copy bandwidth.                 */
int spense_mlp_host(const spense_shape_t* shape, const void* d_blob, const uint8_t* h_x, const float* h_sx,
                    int32_t M, const float* h_sh, int32_t sh_stride, void* h_y, int32_t y_dtype,
                    uint8_t* d_x, float* d_scales, uint8_t* d_hq_scratch, void* d_y, void* d_ws,
                    size_t ws_bytes, const void* d_next_blob, spense_stream_t stream);

/* spense_mlp_stack_host -- the same HOST activations through n_layers packed layers of one shape, one after the other
 * on the stream (every layer reads x, the last one's y is returned): ONE host-to-device copy of the inputs, n_layers x
 * spense_mlp (each naming the next blob as L2 prefetch hint), ONE device-to-host copy of y, ONE synchronise.  This is
 * the unit bench.py times end to end (a decode step of several layers whose inputs arrive from the host); a real model
 * chains its layers on the device with spense_mlp.  d_blobs: HOST array of n_layers DEVICE blob pointers.  Staging
 * buffers and the other arguments as in spense_mlp_host.                                                      */
int spense_mlp_stack_host(const spense_shape_t* shape, const void* const* d_blobs, int32_t n_layers, const uint8_t* h_x,
                          const float* h_sx, int32_t M, const float* h_sh, int32_t sh_stride, void* h_y, int32_t y_dtype,
                          uint8_t* d_x, float* d_scales, uint8_t* d_hq_scratch, void* d_y, void* d_ws, size_t ws_bytes,
                          spense_stream_t stream);

/* spense_select_dense -- SpenseGPT+ dense-index selection (Eqs. 8-12):
 *   s^gate_i = 1/H sum_j |Wg[i,j]| sqrt(Hx[j]),  s^up likewise,  s^down_i = sqrt(Hh[i]) / H sum_n |Wd[n,i]|   (Eq. 9)
 *   s_i = sum over the three projections of s^mlp_i / (mean(s^mlp) + eps)                            (Eqs. 10, 11)
 *   D = the shape->I_dense indices of largest s_i, ties to the lower index                           (Eq. 12)
 * Inputs (device, fp32, original index order): d_wgate, d_wup [I, H]; d_wdown [H, I]; d_hdiag_x [H] = diag(X^T X)
 * of the MLP input; d_hdiag_h [I] = diag of the Hessian of down's input.  eps >= 0 (the paper gives no value).
 * Outputs (device): d_score [I] (nullable); d_dense_idx [I_dense] ascending; d_perm [I] new -> old, the stable
 * partition spense_pack expects (sparse indices ascending, then D ascending).
 * Every reduction runs in a fixed order: scores and selection are bitwise reproducible.  No synchronisation.
 * Workspace: spense_select_workspace_size bytes, 16-byte aligned.                                         */
int spense_select_workspace_size(const spense_shape_t* shape, size_t* bytes);
int spense_select_dense(const spense_shape_t* shape, const float* d_wgate, const float* d_wup, const float* d_wdown,
                        const float* d_hdiag_x, const float* d_hdiag_h, float eps, float* d_score,
                        int32_t* d_dense_idx, int32_t* d_perm, void* d_ws, size_t ws_bytes, spense_stream_t stream);

/* spense_prune_2to4_magnitude -- pruning front-end, first slice: magnitude 2:4 pruning of the
 * SPARSE region in PERMUTED intermediate order ("permute ... then apply [the pruner] while protecting the selected dense
 * indices"; Eq. 1): of every 4 consecutive weights along K the 2 of largest |w| are kept
 * (ties to the lower index), the others become +0.  K is H for rows [0, I_s) of P^T W_gate / P^T W_up and the permuted
 * intermediate dimension for columns [0, I_s) of W_down P (reading Q9b).  Magnitude stands in for SparseGPT's OBS mask
 * and weight update (Eqs. 2-3), which need calibration activations.
 * In place on DEVICE fp32 matrices in ORIGINAL index order: d_wgate, d_wup [I, H], d_wdown [H, I]; d_perm [I] new -> old
 * or NULL (identity).  Integer / comparison work only: bit-exact against the oracle.  No synchronisation.        */
int spense_prune_2to4_magnitude(const spense_shape_t* shape, float* d_wgate, float* d_wup, float* d_wdown,
                                const int32_t* d_perm, spense_stream_t stream);

/* spense_prune_obs_2to4 -- pruning front-end: SparseGPT's 2:4 column sweep on ONE matrix with the
 * dense columns on the right as compensation buffer (Eqs. 2-3; "placing dense columns on the right
 * keeps them available as a compensation buffer"; "apply SparseGPT ... to the sparse regions while
 * protecting the selected dense indices").
 *   d_w [N, K] fp32 row-major, columns in PERMUTED order: the sparse columns [0, K_sparse) first (K_sparse % 4 == 0),
 *   the dense columns last; pruned and compensated IN PLACE.  d_u [K, K] fp32 row-major: the upper triangular factor U of
 *   the inverse of the (damped) input Hessian, H^-1 = U^T U, which the caller computes with a library routine.
 * Columns are processed left to right and frozen once processed; when the sweep reaches a group of 4 it marks, per row,
 * the 2 weights of smallest eps_m = w_m^2 / [H^-1]_mm (Eq. 3, with the inverse Hessian of the not yet processed columns;
 * ties to the lower column); a marked weight is removed with delta_m = -w_m / [H^-1]_mm * H^-1[m, :] over the columns
 * not yet processed.  Columns >= K_sparse are never pruned.  For a layer: W_down P with K_sparse = I_s; the rows
 * [0, I_s) of P^T W_gate / P^T W_up with K_sparse = K = H (their dense rows are left alone, Q9b).
 * fp32 arithmetic; floating point decides the masks, so results are compared with the oracle on loss and on the rows
 * whose masks agree.  Workspace: spense_prune_obs_workspace_size bytes.  No synchronisation.              */
int spense_prune_obs_workspace_size(int32_t N, int32_t K, size_t* bytes);
int spense_prune_obs_2to4(int32_t N, int32_t K, int32_t K_sparse, float* d_w, const float* d_u, void* d_ws, size_t ws_bytes,
                          spense_stream_t stream);

/* spense_quantize_e4m3 -- helper (reading Q5): scale = amax / 448 (1 if amax == 0), per tensor or
 * per row; out = E4M3_rne_sat(in / scale) with an IEEE fp32 division.  d_scales: 1 or rows floats.
 * d_ws needs 4 bytes * (rows + 1). Bit-exact against the oracle.                                  */
int spense_quantize_e4m3(const float* d_in, int64_t rows, int64_t cols, int32_t mode, uint8_t* d_out,
                         float* d_scales, void* d_ws, size_t ws_bytes, spense_stream_t stream);

/* spense_probe_read -- measurement helper ("time floors"): stream `bytes` of device memory through the SMs
 * exactly as the GEMM kernels stream their weights (one cp.async.bulk of 32 KB after the other into a 192 KB shared-memory
 * ring per SM, chunks dealt round robin over one CTA per SM) and discard them.  The rate of this call, timed by the caller
 * with events around it, is the read-only HBM ceiling of the box for this access pattern: bench.py reports the GEMM's
 * achieved GB/s against it next to the copy rate of MEASURED_PEAKS.json.  Not part of the Spense path.
 *   d_buf: DEVICE, 128-byte aligned, bytes a multiple of 32768 (use more than the 126 MB L2, e.g. >= 2 GB).
 *   d_sink: DEVICE, 256 uint32 (one XOR word per CTA, proof that the bytes arrived).  No synchronisation.             */
int spense_probe_read(const void* d_buf, size_t bytes, uint32_t* d_sink, spense_stream_t stream);

/* spense_quantize_e4m3_static -- spense_quantize_e4m3 for callers that cannot provide the d_ws scratch because they cannot
 * allocate device memory at the point of the call: code running inside a serving engine after it has handed the whole
 * HBM budget to its KV-cache pool, a plug-in invoked from a host callback or from inside a framework's own allocator
 * hook (where cudaMalloc would re-enter or deadlock), a real-time loop that must not hit the implicit device
 * synchronisation of cudaMalloc / cudaFree.  Same arithmetic, same kernels and bit-identical results as
 * spense_quantize_e4m3; only the home of the (rows + 1) floats of scratch differs: a fixed array inside the library image
 * (256.25 KB, held by every GPU that loads libspense.so until the process exits) instead of a caller buffer.
 *   d_in [rows, cols] fp32, d_out [rows, cols] E4M3 bytes, d_scales [1] or [rows] fp32: DEVICE, caller-owned, as in
 *   spense_quantize_e4m3.  rows <= SPENSE_QUANTIZE_STATIC_MAX_ROWS, else SPENSE_ERR_STATIC_SCRATCH and nothing is launched
 *   (cols is not limited by the scratch).
 * The call itself allocates nothing, on the host or on the device: no cudaMalloc / cudaFree / cudaHostAlloc and no
 * library routine that allocates.  The first call on each device looks up the device address of the array (the device
 * must be current, as for every call here); make that first call outside any stream capture.  Later calls only
 * enqueue the three kernels on `stream`; no synchronisation.
 * ALL calls on one device share the one array: two calls whose kernels can overlap on the GPU (different streams without
 * an ordering between them, or different host threads doing so) race on it and give wrong scales -- order them on one
 * stream or with events.  Nothing in the array needs to start at zero, it simply holds the last call's maxima.          */
#define SPENSE_QUANTIZE_STATIC_MAX_ROWS 65536
int spense_quantize_e4m3_static(const float* d_in, int64_t rows, int64_t cols, int32_t mode, uint8_t* d_out,
                                float* d_scales, spense_stream_t stream);

/* ---- Stand-alone Spense linears: the format is defined per weight matrix -- "Spense splits the
 * weight matrix into two parts: the semi-structured sparse part and the dense part" (Sec. 3.2) -- and comes
 * in two orientations: OUTPUT-split (the rows of W in R^{N x K} are split: "the input is multiplied
 * separately by the semi-structured sparse and dense weights, and the outputs are concatenated") and INPUT-split (the
 * reduction dimension is split: "a sparse matrix multiplication is performed first ... followed by a dense matrix
 * multiplication that accumulates into the same output").  No GLU, no re-quantisation: y = (x W^T) * s_x[m] * s_w.
 *   N, K multiples of 128.  n_dense = dense rows (out-split) or dense columns (in-split), a multiple of 128; for the
 *   out-split the sparse row count N - n_dense must be a multiple of 256 (sparse and dense rows never share a 256-row
 *   MMA tile).  In PERMUTED order the sparse region comes first, the dense region last.             */
enum { SPENSE_SPLIT_OUT = 0, SPENSE_SPLIT_IN = 1 };
typedef struct {
  int32_t N;       /* output features (rows of W)                                      */
  int32_t K;       /* input features  (columns of W, the reduction dimension)          */
  int32_t n_dense; /* dense rows (SPENSE_SPLIT_OUT) / dense columns (SPENSE_SPLIT_IN)  */
  int32_t split;   /* SPENSE_SPLIT_OUT | SPENSE_SPLIT_IN                               */
} spense_linear_shape_t;

/* Canonical result of spense_pack_linear (DEVICE, caller-owned, members nullable); encoding as in spense_canon_t.
 *   out-split: perm [N]; sp_val [N_s, K/2]; sp_meta [N_s, K/8]; dn [n_dense, K]       (N_s = N - n_dense)
 *   in-split : perm [K]; sp_val [N, K_s/2]; sp_meta [N, K_s/8]; dn [N, n_dense]       (K_s = K - n_dense)            */
typedef struct {
  int32_t* perm;
  uint8_t* sp_val;
  uint8_t* sp_meta;
  uint8_t* dn;
} spense_linear_canon_t;

/* Bytes of the packed blob and of the pack workspace of one linear. */
int spense_linear_pack_sizes(const spense_linear_shape_t* shape, size_t* blob_bytes, size_t* workspace_bytes);

/* spense_pack_linear -- spense_pack for ONE matrix: P1 permute (rows of W for the out-split, columns for the in-split;
 * d_perm new -> old over N resp. K, or NULL), P2 validate Eq. 1 on the sparse region -- 2:4 along K, for the
 * in-split along the PERMUTED K -- and compress it, P3 re-tile into the stage images the GEMM streams.
 *   d_w [N, K] E4M3 bytes in ORIGINAL order; w_scale: the per-tensor fp32 scale, stored in the blob header.
 *   h_err_where[4] as in spense_pack with matrix = 0.  Synchronises the stream once.  Other arguments as in spense_pack. */
int spense_pack_linear(const spense_linear_shape_t* shape, const uint8_t* d_w, float w_scale, const int32_t* d_perm,
                       void* d_blob, size_t blob_bytes, const spense_linear_canon_t* canon, void* d_ws, size_t ws_bytes,
                       int64_t* h_err_where, spense_stream_t stream);

/* Workspace of the linear GEMM calls at up to M tokens: same rules as spense_workspace_size / spense_workspace_init. */
int spense_linear_workspace_size(const spense_linear_shape_t* shape, int32_t M, size_t* bytes);

/* spense_linear_out_split -- y[m, n] = (sum_k x[m, k] W'[n, k]) * s_x[m * sx_stride] * s_w with W' = the row-permuted
 * weight: 256-row tiles below N_s run on 2:4 sparse MMAs, the others on dense MMAs (output-split).
 * y is in PERMUTED row order: y[:, new] belongs to original output feature perm[new].
 * spense_linear_in_split -- the same sum with the K loop running the sparse range [0, K_s) on sparse MMAs and continuing
 * with the dense range into the same accumulator (input-split); x is in PERMUTED column order.
 *   d_x [M, K] E4M3; d_sx fp32, sx_stride 0 = one scalar, 1 = per token; d_y [M, N] fp32 or bf16.  The blob must come from
 *   spense_pack_linear with the same shape (checked on the device: SPENSE_ERR_BAD_BLOB).  No synchronisation.          */
int spense_linear_out_split(const spense_linear_shape_t* shape, const void* d_blob, const uint8_t* d_x, const float* d_sx,
                            int32_t sx_stride, int32_t M, void* d_y, int32_t y_dtype, void* d_ws, size_t ws_bytes,
                            spense_stream_t stream);
int spense_linear_in_split(const spense_linear_shape_t* shape, const void* d_blob, const uint8_t* d_x, const float* d_sx,
                           int32_t sx_stride, int32_t M, void* d_y, int32_t y_dtype, void* d_ws, size_t ws_bytes,
                           spense_stream_t stream);

#ifdef __cplusplus
}
#endif
#endif /* SPENSE_H_ */
