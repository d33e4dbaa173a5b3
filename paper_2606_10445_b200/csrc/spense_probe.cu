// Read-only HBM stream probe (SURVEY.md 8d "time floors": the read ceiling of the box, measured in the bench run).
// The GEMM kernels are read streams: one thread per CTA drops contiguous stage images into a shared-memory ring with
// cp.async.bulk.  This kernel is that producer with nothing behind it -- same instruction, same 32 KB granule, same ring
// depth per SM, the bytes discarded -- so its rate is what a weight stream of this design can reach at best.
#include "spense_internal.cuh"

namespace spense {
namespace {

constexpr int kProbeChunk = 32768;   // one bulk copy; the GEMM's stage halves are 16-20 KB, the ring 6-7 stages deep
constexpr int kProbeSlots = 6;       // 192 KB in flight per SM

__global__ void __launch_bounds__(32) read_probe_kernel(const uint8_t* __restrict__ buf, long long n_chunks, uint32_t* __restrict__ sink) {
  extern __shared__ __align__(128) uint8_t ring[];
  __shared__ __align__(8) uint64_t bars[kProbeSlots];
  if (threadIdx.x != 0) return;
  for (int s = 0; s < kProbeSlots; ++s) mbar_init(smem_u32(&bars[s]), 1);
  fence_barrier_init();
  const uint64_t pol = policy_evict_first();
  const uint32_t ring0 = smem_u32(ring);
  // chunks are dealt round robin: at any moment the CTAs together read one contiguous window of DRAM pages
  long long next = blockIdx.x;
  auto issue = [&](int s) {
    const uint32_t bar = smem_u32(&bars[s]);
    mbar_expect_tx(bar, kProbeChunk);
    bulk_g2s(ring0 + (uint32_t)s * kProbeChunk, buf + (size_t)next * kProbeChunk, kProbeChunk, bar, pol);
    next += gridDim.x;
  };
  for (int s = 0; s < kProbeSlots && next < n_chunks; ++s) issue(s);
  uint32_t acc = 0;
  long long k = 0;
  for (long long c = blockIdx.x; c < n_chunks; c += gridDim.x, ++k) {
    const int s = (int)(k % kProbeSlots);
    const uint32_t parity = (uint32_t)((k / kProbeSlots) & 1);
    while (!mbar_try(smem_u32(&bars[s]), parity)) {}
    acc ^= *reinterpret_cast<volatile uint32_t*>(ring + (size_t)s * kProbeChunk + ((c * 4) & (kProbeChunk - 4)));   // the bytes did arrive
    fence_proxy_async();               // that read is ordered before the slot is overwritten by the next bulk copy
    if (next < n_chunks) issue(s);
  }
  sink[blockIdx.x] = acc;
}

}  // namespace

int launch_read_probe(const void* d_buf, size_t bytes, uint32_t* d_sink, int sms, cudaStream_t stream) {
  static bool ready[64] = {};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return SPENSE_ERR_CUDA;
  const int smem = kProbeSlots * kProbeChunk;
  if (!ready[dev]) {
    if (cudaFuncSetAttribute(read_probe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem) != cudaSuccess) return SPENSE_ERR_CUDA;
    ready[dev] = true;
  }
  const long long n_chunks = (long long)(bytes / kProbeChunk);
  const int grid = n_chunks < sms ? (int)n_chunks : sms;
  read_probe_kernel<<<grid, 32, smem, stream>>>(reinterpret_cast<const uint8_t*>(d_buf), n_chunks, d_sink);
  return cudaGetLastError() == cudaSuccess ? SPENSE_OK : SPENSE_ERR_CUDA;
}

}  // namespace spense
