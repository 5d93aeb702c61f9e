// Measurement aid, not part of the C ABI (not declared in include/delta.h): what the path between the SMs and L2 sustains.
//
// The intermediates of the hot path (X, S, the 1/sqrt rows) never reach HBM at config 2, but they cross the SM <-> L2
// crossbar twice, and the outputs cross it once: per chunk about 2.3 x the algorithmic bytes.  ncu
// (l1tex__m_xbar2l1tex_read_bytes, l1tex__m_l1tex2xbar_write_bytes) counts those bytes per kernel; this probe gives
// the rate to hold them against: persistent CTAs, one per SM, whose first warp streams a source that fits L2 into
// shared memory with cp.async.bulk (the pair kernel's way of reading S) while the other 24 warps write a destination
// with plain 16-byte streaming stores in full 512-byte runs (the best pattern the path has).  `bench.py --probe-fabric`
// times it with CUDA events and prints read-only, write-only and combined figures.
#include "delta_internal.h"

namespace delta {
namespace {

constexpr int kProbePiece = 32768, kProbeSlots = 4, kProbeThreads = 800;

__device__ __forceinline__ uint32_t su32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void wait_parity(uint64_t *bar, uint32_t par) {
  uint32_t ok = 0;
  while (!ok)
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(su32(bar)), "r"(par) : "memory");
}

__global__ void __launch_bounds__(kProbeThreads, 1)
probe_fabric_kernel(const char *__restrict__ src, size_t read_bytes, char *__restrict__ dst, size_t write_bytes) {
  extern __shared__ __align__(128) unsigned char sm[];
  __shared__ uint64_t bar[kProbeSlots];
  const int tid = threadIdx.x;
  if (tid == 0) {
    for (int s = 0; s < kProbeSlots; ++s) asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(su32(bar + s)));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid < 32) {
    if (tid == 0 && read_bytes) {
      const size_t np = read_bytes / kProbePiece;
      int n = 0;
      for (size_t i = blockIdx.x; i < np; i += gridDim.x, ++n) {
        const int s = n % kProbeSlots;
        if (n >= kProbeSlots) wait_parity(bar + s, ((n / kProbeSlots) - 1) & 1);  // the slot's previous copy has landed
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(su32(bar + s)), "r"(kProbePiece) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                         su32(sm + (size_t)s * kProbePiece)),
                     "l"(src + i * kProbePiece), "r"(kProbePiece), "r"(su32(bar + s))
                     : "memory");
      }
      for (int m = (n > kProbeSlots ? n - kProbeSlots : 0); m < n; ++m) wait_parity(bar + m % kProbeSlots, (m / kProbeSlots) & 1);
    }
    return;
  }
  const int t = tid - 32, nt = kProbeThreads - 32;
  const size_t n4 = write_bytes / 16;
  for (size_t i = (size_t)blockIdx.x * nt + t; i < n4; i += (size_t)gridDim.x * nt)
    __stcs(reinterpret_cast<float4 *>(dst) + i, make_float4(1.f, 2.f, 3.f, 4.f));
}

}  // namespace
}  // namespace delta

// One launch: read `read_bytes` of d_src (a multiple of 32 KiB is used) into shared memory and write `write_bytes` of
// d_dst (a multiple of 16).  Either may be 0.  Device pointers, 16-byte aligned; asynchronous on `stream`.
extern "C" int delta_internal_probe_fabric(const void *d_src, size_t read_bytes, void *d_dst, size_t write_bytes, void *stream) {
  using namespace delta;
  if ((read_bytes && !d_src) || (write_bytes && !d_dst)) return DELTA_ERR_INVALID_ARG;
  int dev = 0, sms = 0;
  DELTA_CUDA_CHECK(cudaGetDevice(&dev));
  DELTA_CUDA_CHECK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const size_t smem = (size_t)kProbeSlots * kProbePiece;
  int rc = opt_in_smem(probe_fabric_kernel, smem);
  if (rc) return rc;
  probe_fabric_kernel<<<sms, kProbeThreads, smem, reinterpret_cast<cudaStream_t>(stream)>>>(
      reinterpret_cast<const char *>(d_src), read_bytes, reinterpret_cast<char *>(d_dst), write_bytes);
  DELTA_CUDA_CHECK(cudaGetLastError());
  return DELTA_OK;
}
