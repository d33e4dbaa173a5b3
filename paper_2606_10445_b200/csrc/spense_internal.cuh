// Internal definitions shared by the CUDA translation units of libspense (never installed).
// Blob geometry, kernel parameter blocks and the sm_100a PTX wrappers (mbarrier, TMA / bulk copy,
// tcgen05 MMA / TMEM).  Nothing here is shared with oracle/.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "spense.h"

namespace spense {

// ------------------------------------------------------------------------------------------
// Blob geometry.  The blob is a sequence of pipeline-stage images: each stage is EXACTLY the bytes
// one cp.async.bulk drops into shared memory (128B-swizzle pre-applied), so the producer streams
// perfectly sequential DRAM pages with one bulk copy per stage and needs no tensor map for weights.
//
//   "pair tile" = two 128-row A operands (MMA-M = 128 each) that share one B (activation) tile:
//       gate_up : rows [128t, 128t+128) of W_gate and of W_up       (tile t < I_s/128 sparse, else dense)
//       down    : rows [256t, 256t+128) and [256t+128, 256t+256) of W_down (sparse K range, then dense)
//   sparse stage (K = 256 logical): A0 vals 16 KB | A0 meta 4 KB | A1 vals 16 KB | A1 meta 4 KB
//   dense  stage (K = 128)        : A0 16 KB | A1 16 KB
//   (operand-major, so that each CTA of a pair loads one operand: 20 KB / 16 KB contiguous)
//   vals / dense images: 128 rows x 128 B, canonical K-major SWIZZLE_128B (8-row x 128 B atoms,
//       16-byte chunk index XOR (row & 7)).  meta image: 2 atoms of 128 rows x 16 B, row-major
//       (one atom = K 128 logical = what one tcgen05.cp.128x128b moves to TMEM).
//   gate_up operand rows: operand a of pair tile t holds the gate AND the up rows of the 64 intermediate indices
//       128 t + 64 a + [0, 64): operand row 32 q + i = gate row of index 16 q + i, operand row 32 q + 16 + i = up row of
//       the same index (q < 4, i < 16).  g and u of one index then sit in the two 16-lane halves of ONE TMEM lane
//       quadrant of ONE accumulator, so a warp reads both with two tcgen05.ld.16x256b and every operand is a
//       self-contained GLU tile (what lets the kernel give each CTA of a pair one operand).
// ------------------------------------------------------------------------------------------
constexpr int kTileRows = 128;
constexpr int kSparseStageK = 256;           // logical K per sparse stage
constexpr int kDenseStageK = 128;            // K per dense stage
constexpr int kOperandBytes = 128 * 128;     // one 128 x 128 B operand image
constexpr int kMetaBytes = 128 * 32;         // one operand's metadata per sparse stage
constexpr int kSparseOperandBytes = kOperandBytes + kMetaBytes;         // 20480: values + metadata of one operand
constexpr int kSparseStageBytes = 2 * kSparseOperandBytes;              // 40960
constexpr int kDenseStageBytes = 2 * kOperandBytes;                    // 32768
constexpr int kBlobHeaderBytes = 1024;
constexpr uint32_t kBlobMagic = 0x53504E53u;  // "SNPS"
constexpr int kBlobVersion = 2;
constexpr int kMaxSpans = 160;               // fix-up slots of a launch (one per CTA)
constexpr int kMaxTokens = 1 << 20;           // tokens per call (the activation tensor map is built over all of them)
constexpr int kSmemMax = 232448;             // opt-in dynamic shared memory per CTA
constexpr int kWideMaxTokens = 240;          // token columns of one CTA pair (2 accumulator buffers x 240 + 16 metadata columns of TMEM)
constexpr int kWideMaxTokens1 = 256;         // 241..256 tokens: ONE block of 256 columns with a single accumulator buffer (the largest MMA-N), so
                                             // the weights cross the L2 -> SM path once instead of once per 128-token block
constexpr int kFlagBytes = 4096;             // control words (128 B) + 2 flags per slot
constexpr int kAmaxBytes = kMaxSpans * 256 * 4;   // dynamic requant: max|h| per slot and token column (follows the flags)
constexpr int kWsFixedBytes = kFlagBytes + kAmaxBytes;   // zeroed by spense_workspace_init; partials follow
constexpr long long kWaitBudgetNs = 2000000000ll;   // a CTA gives up waiting for a peer after 2 s (a launch takes < 10 ms)

struct BlobHeader {
  uint32_t magic;
  int32_t version;
  int32_t H, I, I_dense;
  float w_scale[3];
  uint64_t gate_up_off, down_off, total_bytes;
  int32_t kind;               // 0: GLU MLP layer (spense_pack); 1: in-split linear, 2: out-split linear (spense_pack_linear)
};
constexpr int kBlobMlp = 0, kBlobLinearIn = 1, kBlobLinearOut = 2;

struct Geometry {
  int H, I, I_d, I_s;
  // gate_up
  int gu_tiles, gu_tiles_sparse;   // I/128, I_s/128
  int gu_ns, gu_nd;                // stages per sparse tile: ceil(H/256); per dense tile: H/128
  // down
  int dn_tiles;                    // ceil(H/256)
  int dn_ns, dn_nd;                // ceil(I_s/256), I_d/128
  size_t gate_up_off, down_off, total_bytes;
};

__host__ __device__ inline Geometry make_geometry(int H, int I, int I_d) {
  Geometry g;
  g.H = H; g.I = I; g.I_d = I_d; g.I_s = I - I_d;
  g.gu_tiles = I / 128;
  g.gu_tiles_sparse = g.I_s / 128;
  g.gu_ns = (H + 255) / 256;
  g.gu_nd = H / 128;
  g.dn_tiles = (H + 255) / 256;
  g.dn_ns = (g.I_s + 255) / 256;
  g.dn_nd = I_d / 128;
  g.gate_up_off = kBlobHeaderBytes;
  size_t gu = (size_t)g.gu_tiles_sparse * g.gu_ns * kSparseStageBytes +
              (size_t)(g.gu_tiles - g.gu_tiles_sparse) * g.gu_nd * kDenseStageBytes;
  g.down_off = g.gate_up_off + gu;
  size_t dn = (size_t)g.dn_tiles * ((size_t)g.dn_ns * kSparseStageBytes + (size_t)g.dn_nd * kDenseStageBytes);
  g.total_bytes = g.down_off + dn;
  return g;
}

// One linear W [N, K] (spense_pack_linear): the blob is the header followed by ONE section.
//   in-split : the down section of a layer with H = N, I = K, I_d = n_dense (pair tile = 256 rows, sparse K stages then dense).
//   out-split: pair tile t = rows [256 t, 256 t + 256) of the row-permuted W, operand a = rows 256 t + 128 a + [0, 128) in
//              natural order; the N_s / 256 sparse tiles first (ceil(K / 256) sparse stages each), then the dense tiles
//              (K / 128 dense stages each; a last half tile is zero padded).  Held in the gate_up fields of Geometry.
__host__ __device__ inline Geometry make_geometry_linear(int N, int K, int n_dense, bool in_split) {
  Geometry g;
  if (in_split) {
    g = make_geometry(N, K, n_dense);
    g.gu_tiles = 0; g.gu_tiles_sparse = 0;
    g.down_off = kBlobHeaderBytes;
    g.total_bytes = g.down_off + (size_t)g.dn_tiles * ((size_t)g.dn_ns * kSparseStageBytes + (size_t)g.dn_nd * kDenseStageBytes);
    return g;
  }
  g.H = K; g.I = N; g.I_d = n_dense; g.I_s = N - n_dense;
  g.gu_tiles_sparse = g.I_s / 256;
  g.gu_tiles = g.gu_tiles_sparse + (n_dense + 255) / 256;
  g.gu_ns = (K + 255) / 256;
  g.gu_nd = K / 128;
  g.dn_tiles = 0; g.dn_ns = 0; g.dn_nd = 0;
  g.gate_up_off = kBlobHeaderBytes;
  g.down_off = g.gate_up_off + (size_t)g.gu_tiles_sparse * g.gu_ns * kSparseStageBytes +
               (size_t)(g.gu_tiles - g.gu_tiles_sparse) * g.gu_nd * kDenseStageBytes;
  g.total_bytes = g.down_off;
  return g;
}

// byte offset of element (row r, byte column b) inside one 128 x 128 B SWIZZLE_128B operand image
__host__ __device__ inline int sw128_offset(int r, int b) {
  return (r >> 3) * 1024 + (r & 7) * 128 + ((((b >> 4) ^ (r & 7)) & 7) << 4) + (b & 15);
}

// ------------------------------------------------------------------------------------------
// GEMM kernel parameters.  One kernel serves gate_up (mode 0), down / the in-split linear (mode 1) and the out-split
// linear (mode 2: the tile walk of mode 0 with 256-row tiles, the plain epilogue of mode 1): a byte-balanced
// stream-K walk over the linear sequence of stages; span i = stages [span_begin[i], span_begin[i+1]).
// ------------------------------------------------------------------------------------------
struct GemmParams {
  const uint8_t* section;   // first stage image of this matrix family
  const BlobHeader* hdr;    // the blob header (device): weight scales are READ ON THE DEVICE from it, magic / shape are checked there
  int H, I, I_d;            // the shape the caller states (compared with the header on the device)
  int mode;                 // 0 gate_up, 1 down / in-split linear, 2 out-split linear
  int kind;                 // what the blob must be (BlobHeader::kind)
  int num_tiles, tiles_sparse;
  int ns, nd;               // mode 0: stages of a sparse tile / of a dense tile; mode 1: per tile both
  int dense_k0;             // K byte offset of the first dense stage in the B operand (mode 1: I_s)
  int n_spans;              // stream-K spans of the schedule (= CTAs, or CTA pairs, per token block)
  int M, n_pad;             // tokens in this call; token columns of one MMA (a token block, padded to 16)
  int nb, blk0;             // token blocks covered by this launch and the first of them: the CTAs of the nb blocks walk the
                            // same schedule side by side, so a weight stage is read from HBM once and found in L2 by the others
  int num_stages, slot_bytes, acc_stride, num_acc_bufs;
  // epilogue
  const float* s_act;       // mode 0: s_x [M]; mode 1: s_h (stride sh_stride)
  const float* s_h;         // mode 0: requant scale
  int sh_stride;
  int scale0, scale1;       // indices into hdr->w_scale: mode 0: gate, up; mode 1: down, down
  uint8_t* hq;              // mode 0 out [M, ld_out]
  float* h_f32;             // mode 0 optional out
  float* amax_part;         // mode 0, dynamic requant: per-slot per-token max|h| [slots][n_pad] (then hq is not written)
  void* y;                  // mode 1 out [M, ld_out]
  int y_dtype;
  int ld_out;               // I (mode 0) or H (mode 1)
  int out_rows;             // valid output columns (I or H) for masking padded tiles
  int* ws_ctrl;             // workspace control words: [0] epoch of the last launch, [1] started-CTA count
  int* flags;               // workspace: 2 ints per slot (first / last segment), hold the epoch of the dump
  float* partials;          // workspace: 2 partial tiles per slot
  int* status;              // mapped pinned host word: first device-side error (bad blob header, a peer CTA never showed up)
  int pf_pace_ns;           // next-kernel L2 prefetch: nanoseconds per 32 KB chunk (0 = all at once)
  long long* trace;         // debug timeline (16 slots per span; SPENSE_DEBUG_HOOKS builds) or nullptr
  int dbg;                  // debug experiments (SPENSE_DEBUG_HOOKS builds; 0 in production)
  const uint8_t* next_base; // section the NEXT kernel of the stream will stream (L2 prefetch during our tail) or nullptr
  int span_begin[kMaxSpans + 1];
  uint32_t next_off[kMaxSpans];   // byte offset of span i's first stage in next_base ...
  uint32_t next_len[kMaxSpans];   // ... and how many bytes of it to prefetch
};

// ------------------------------------------------------------------------------------------
// PTX wrappers
// ------------------------------------------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// one try (the hardware suspends the thread up to an implementation-defined time): true once the phase is complete
__device__ __forceinline__ bool mbar_try(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
               : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0;
}
// arrive on a barrier of another CTA of the cluster (address from mapa)
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_bar) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_bar) : "memory");
}
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t mapa_shared(uint32_t addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void fence_barrier_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ uint64_t policy_evict_first() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ uint64_t policy_evict_normal() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  return p;
}
// 1-D bulk copy global -> shared, completion on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t pol) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
      ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
}
// 2-D tiled TMA load (SASS: UTMALDG) issued by either CTA of a pair: the bytes land in the issuing CTA, the transaction count goes to `cluster_bar`
// (the LEADER CTA's barrier, a shared::cluster address), so the leader's MMA thread sees both halves of a stage
__device__ __forceinline__ void tma_load_2d_pair(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t cluster_bar, uint64_t pol) {
  asm volatile(
      "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint "
      "[%0], [%1, {%2, %3}], [%4], %5;"
      ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(cluster_bar), "l"(pol) : "memory");
}
__device__ __forceinline__ void prefetch_tmap(const CUtensorMap* map) {
  asm volatile("prefetch.tensormap [%0];" ::"l"(map) : "memory");
}

// TMEM
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// ---- CTA-pair (cta_group::2) forms: one thread of the leader CTA issues for both CTAs; A = 128 rows from each CTA
// (same smem offset), B = N/2 rows from each, D = 128 lanes x N columns in each CTA's TMEM, metadata per CTA
__device__ __forceinline__ void tmem_alloc_pair(uint32_t smem_dst, uint32_t ncols) {   // one warp of EACH CTA, same smem offset
  asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_pair(uint32_t taddr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tc_commit_pair(uint32_t bar, uint16_t cta_mask) {   // arrives on `bar` (same offset) in every CTA of the mask
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
               ::"r"(bar), "h"(cta_mask) : "memory");
}
__device__ __forceinline__ void mma_f8_dense_pair(uint32_t d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::f8f6f4 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void mma_f8_sparse_pair(uint32_t d, uint64_t adesc, uint64_t bdesc, uint32_t e, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %5, 0;\n\t"
      "tcgen05.mma.sp.cta_group::2.kind::f8f6f4 [%0], %1, %2, [%3], %4, p;\n\t}"
      ::"r"(d), "l"(adesc), "l"(bdesc), "r"(e), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void tc_cp_128x128b_pair(uint32_t taddr, uint64_t sdesc) {
  asm volatile("tcgen05.cp.cta_group::2.128x128b [%0], %1;" ::"r"(taddr), "l"(sdesc) : "memory");
}
// 16 lanes x 8 columns: thread t gets lanes t/4 (v[0], v[1]) and t/4 + 8 (v[2], v[3]) of the 16 lanes that start at the
// address's lane (a multiple of 16 inside the warp's quadrant), columns 2 (t % 4) and 2 (t % 4) + 1
__device__ __forceinline__ void tmem_ld_16x256b(uint32_t taddr, uint32_t (&v)[4]) {
  asm volatile("tcgen05.ld.sync.aligned.16x256b.x1.b32 {%0,%1,%2,%3}, [%4];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]) : "r"(taddr) : "memory");
}
// .x2 / .x4: the same for 2 / 4 groups of 8 columns; group j lands in v[4 j .. 4 j + 3]
__device__ __forceinline__ void tmem_ld_16x256b_x2(uint32_t taddr, uint32_t (&v)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.16x256b.x2.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld_16x256b_x4(uint32_t taddr, uint32_t (&v)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.16x256b.x4.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
        "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
      : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,"
      "%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
        "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
        "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
        "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
        "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
      : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&v)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
               : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t (&v)[8]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
               ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]) : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// shared-memory matrix descriptor (sm_100 "version 1")
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes, uint32_t layout) {
  return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16) |
         ((uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32) | (1ull << 46) | ((uint64_t)layout << 61);
}
constexpr uint32_t kLayoutSW128 = 2, kLayoutNone = 0;

__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile(
      "{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.u32 %0, 1, 0, P;\n\t}" : "=r"(pred));
  return pred != 0;
}
#endif  // __CUDACC__

// host-side entry points implemented in the .cu files
int launch_pack(const spense_shape_t* shape, const uint8_t* d_wgate, const uint8_t* d_wup, const uint8_t* d_wdown,
                const float* h_w_scale, const int32_t* d_perm, void* d_blob, const spense_canon_t* canon, void* d_ws,
                int64_t* h_err_where, cudaStream_t stream);
int launch_pack_linear(const spense_linear_shape_t* shape, const uint8_t* d_w, float w_scale, const int32_t* d_perm, void* d_blob,
                       const spense_linear_canon_t* canon, void* d_ws, int64_t* h_err_where, cudaStream_t stream);
int prepare_gemm_kernels(int dev);
int launch_gemm(const GemmParams& p, const CUtensorMap& tmap_b, const CUtensorMap& tmap_ws, const CUtensorMap& tmap_wd, bool pdl, int dev,
                cudaStream_t stream);
int launch_requant_rows(const float* d_h, int rows, int cols, const float* d_amax_part, int n_part, int part_stride,
                        int block_rows, uint8_t* d_hq, float* d_sh, int sms, cudaStream_t stream);
int launch_select(const spense_shape_t* shape, const float* d_wgate, const float* d_wup, const float* d_wdown,
                  const float* d_hdiag_x, const float* d_hdiag_h, float eps, float* d_score, int32_t* d_dense_idx,
                  int32_t* d_perm, void* d_ws, cudaStream_t stream);
int launch_prune(const spense_shape_t* shape, float* d_wgate, float* d_wup, float* d_wdown, const int32_t* d_perm, cudaStream_t stream);
int launch_prune_obs(int N, int K, int K_sparse, float* d_w, const float* d_u, void* d_ws, cudaStream_t stream);
int launch_read_probe(const void* d_buf, size_t bytes, uint32_t* d_sink, int sms, cudaStream_t stream);
int launch_quantize(const float* d_in, int64_t rows, int64_t cols, int32_t mode, uint8_t* d_out, float* d_scales,
                    void* d_ws, cudaStream_t stream);

}  // namespace spense
