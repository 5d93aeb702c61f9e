// Write-out of one (channel, bin) of the STFT for the 8 segments of a segment block into the frequency-major X layout
// (delta_internal.h), shared by the FFT-based STFT kernel (stft.cu) and the direct-DFT kernel for transform lengths that
// are not powers of two (dft_generic.cu).  Holds the f1/f2 options that act on X: band-pass mask (R19), per-segment
// normalisation (phase-lock estimator, R21) and, in tensor-core mode, the split into fp16 hi + lo.
#pragma once
#include <cuda_fp16.h>

#include "delta_internal.h"

namespace delta {

// re, im: X[c, 8 kb + q, f], q < 8.  sc: the channel's power-of-two fp16 scale (tensor-core mode only).
template <bool TC>
__device__ __forceinline__ void store_x_bin(void *__restrict__ Xout, const Layout &lay, int kb, int c, int f, float sc,
                                            const float *re, const float *im) {
  const int64_t plane = (int64_t)lay.Kc * lay.Cp * kSegBlock;  // one [kc][c][8] block
  const int64_t within = ((int64_t)kb * lay.Cp + c) * kSegBlock;
  const int64_t base = (int64_t)f * lay.x_elems_per_f + within;
  const float keep = (f >= lay.f_lo && f <= lay.f_hi) ? 1.f : 0.f;  // band-pass mask (R19)
  float nre[kSegBlock], nim[kSegBlock];
  if (lay.estimator == DELTA_EST_PHASE_LOCK) {  // per-segment-normalised estimator (f2): X -> X / |X|, 0 where X = 0
#pragma unroll
    for (int q = 0; q < kSegBlock; ++q) {
      const float m2 = fmaf(re[q], re[q], im[q] * im[q]);
      const float r = m2 > 0.f ? rsqrtf(m2) : 0.f;
      nre[q] = re[q] * r;
      nim[q] = im[q] * r;
    }
    re = nre;
    im = nim;
  }
  if (TC) {
    // split fp16: v * scale = hi + lo
    __half *X = reinterpret_cast<__half *>(Xout);
    const float s = keep * sc;
    __align__(16) __half2 hr[4], hi_[4], lr[4], li[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const float r0 = re[2 * q] * s, r1 = re[2 * q + 1] * s, i0 = im[2 * q] * s, i1 = im[2 * q + 1] * s;
      hr[q] = __floats2half2_rn(r0, r1);
      hi_[q] = __floats2half2_rn(i0, i1);
      const float2 hrf = __half22float2(hr[q]), hif = __half22float2(hi_[q]);
      lr[q] = __floats2half2_rn(r0 - hrf.x, r1 - hrf.y);
      li[q] = __floats2half2_rn(i0 - hif.x, i1 - hif.y);
    }
    *reinterpret_cast<uint4 *>(X + base + 0 * plane) = *reinterpret_cast<const uint4 *>(hr);
    *reinterpret_cast<uint4 *>(X + base + 1 * plane) = *reinterpret_cast<const uint4 *>(hi_);
    *reinterpret_cast<uint4 *>(X + base + 2 * plane) = *reinterpret_cast<const uint4 *>(lr);
    *reinterpret_cast<uint4 *>(X + base + 3 * plane) = *reinterpret_cast<const uint4 *>(li);
  } else {
    float *X = reinterpret_cast<float *>(Xout);
    *reinterpret_cast<float4 *>(X + base) = make_float4(keep * re[0], keep * re[1], keep * re[2], keep * re[3]);
    *reinterpret_cast<float4 *>(X + base + 4) = make_float4(keep * re[4], keep * re[5], keep * re[6], keep * re[7]);
    *reinterpret_cast<float4 *>(X + base + plane) = make_float4(keep * im[0], keep * im[1], keep * im[2], keep * im[3]);
    *reinterpret_cast<float4 *>(X + base + plane + 4) = make_float4(keep * im[4], keep * im[5], keep * im[6], keep * im[7]);
  }
}

}  // namespace delta
