// delta_coherence_static (include/delta.h): Eq. (1b), for callers that cannot let scratch be allocated.
//
// The coherence stage needs scratch: the four shifted copies of 1/sqrt(S_cc[f]) (store_rsq4 in delta_internal.h) and
// 1/sqrt(L R_cc[0]) per channel, written by auto_prep_kernel from the caller's autospectra and read by pair_kernel.
// delta_coherence keeps them in the plan's workspace; here they live in a file-scope device array of
// DELTA_STATIC_SCRATCH_BYTES that every GPU loading the library holds until exit.  The kernels are the ones of the
// existing path (launch_auto_prep, launch_pair): only where the scratch lives differs.
//
// g_static_scratch names the array in DEVICE code.  In host code the same name is a host-side stand-in, not a device
// address, so the launchers are never given it: the device address comes from cudaGetSymbolAddress, asked once per
// device with that device current, in this translation unit (the one that defines the array).
#include <mutex>

#include "delta_internal.h"

namespace delta {
namespace {

static __device__ __align__(256) unsigned char g_static_scratch[DELTA_STATIC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
void *g_scratch_addr[kMaxDevices] = {};  // device address of g_static_scratch on device d (0: not asked yet)

// the array's address on the current device; `dev` = cudaGetDevice()
int static_scratch_addr(int dev, unsigned char **out) {
  if (dev < 0 || dev >= kMaxDevices) return DELTA_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_addr[dev]) {
    void *q = nullptr;
    DELTA_CUDA_CHECK(cudaGetSymbolAddress(&q, g_static_scratch));
    if (!q) return DELTA_ERR_CUDA;
    g_scratch_addr[dev] = q;
  }
  *out = reinterpret_cast<unsigned char *>(g_scratch_addr[dev]);
  return DELTA_OK;
}

inline size_t round256(size_t v) { return (v + 255) & ~(size_t)255; }

}  // namespace
}  // namespace delta

extern "C" int delta_coherence_static(delta_plan *p, const float *d_S, const float *d_Sauto, float *d_G, void *stream) {
  using namespace delta;
  if (!p || !d_S || !d_Sauto || !d_G) return DELTA_ERR_INVALID_ARG;
  const Layout &l = p->lay;
  // scratch: float rsq4[4][C][Fp], then (256-byte aligned) float rnorm[C]
  const size_t rsq_bytes = round256((size_t)4 * l.C * l.Fp * sizeof(float));
  const size_t need = rsq_bytes + round256((size_t)l.C * sizeof(float));
  if (need > (size_t)DELTA_STATIC_SCRATCH_BYTES) return DELTA_ERR_TOO_LARGE;
  if (!p->ws) return DELTA_ERR_NO_WORKSPACE;  // the plan's constant tables (twiddles, pair list) are read from it
  if ((reinterpret_cast<uintptr_t>(d_S) & 15) != 0) return DELTA_ERR_ALIGNMENT;
  int dev = -1;
  DELTA_CUDA_CHECK(cudaGetDevice(&dev));
  if (dev != p->device) return DELTA_ERR_INVALID_ARG;  // the plan's device must be the current one
  unsigned char *scratch = nullptr;
  int rc = static_scratch_addr(dev, &scratch);
  if (rc) return rc;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  // The array keeps the last call's contents.  auto_prep_kernel writes every element the pair kernel computes with,
  // but the row copies of the pair kernel carry the rows' padding along, so the part in use is cleared first.
  DELTA_CUDA_CHECK(cudaMemsetAsync(scratch, 0, need, st));
  float *rsq = reinterpret_cast<float *>(scratch);
  float *rnorm = reinterpret_cast<float *>(scratch + rsq_bytes);
  rc = launch_auto_prep(p, d_Sauto, rsq, rnorm, st);
  if (rc) return rc;
  return launch_pair(p, d_S, rsq, rnorm, d_G, nullptr, nullptr, nullptr, st);
}
