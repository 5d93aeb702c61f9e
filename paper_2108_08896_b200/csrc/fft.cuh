// Shared-memory radix-4 Stockham FFT (autosort, decimation in frequency) for a group of GROUP
// threads, plus the split/merge steps that turn an N = L/2 point complex transform into the
// L-point real transform (STFT) and its inverse (Eq. 1d).
// No cuFFT anywhere: every butterfly is here.
#pragma once
#include <cuda_runtime.h>

namespace delta {

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }

template <int GROUP>
__device__ __forceinline__ void group_sync() {
  if (GROUP <= 32) __syncwarp(); else __syncthreads();
}

// tw[f] = exp(-2 pi i f / L), f = 0..L-1, L = 2N (device global, read through the read-only path).
// The N-point twiddle exp(-+2 pi i j / N) is tw[2j] (conjugated for the inverse).
template <bool INVERSE>
__device__ __forceinline__ float2 twiddle(const float2 *__restrict__ tw, int idx) {
  float2 w = __ldg(tw + idx);
  if (INVERSE) w.y = -w.y;
  return w;
}

// One radix-4 pass: current sub-transform length n, stride s (n * s == N).
template <int N, int GROUP, bool INVERSE>
__device__ __forceinline__ void radix4_pass(const float2 *x, float2 *y, const float2 *__restrict__ tw,
                                            int tid, int n, int s) {
  const int n1s = N / 4;  // s * (n/4)
  for (int t = tid; t < N / 4; t += GROUP) {
    const int q = t & (s - 1);
    const int ps = t - q;  // p * s
    const float2 a = x[t], b = x[t + n1s], c = x[t + 2 * n1s], d = x[t + 3 * n1s];
    const float2 apc = cadd(a, c), amc = csub(a, c), bpd = cadd(b, d), bmd = csub(b, d);
    // forward: -i (b - d); inverse: +i (b - d)
    const float2 jbmd = INVERSE ? make_float2(-bmd.y, bmd.x) : make_float2(bmd.y, -bmd.x);
    const float2 w1 = twiddle<INVERSE>(tw, 2 * ps);
    const float2 w2 = twiddle<INVERSE>(tw, 4 * ps);
    const float2 w3 = twiddle<INVERSE>(tw, 6 * ps);
    float2 *o = y + q + 4 * ps;  // q + s * 4p
    o[0] = cadd(apc, bpd);
    o[s] = cmul(w1, cadd(amc, jbmd));
    o[2 * s] = cmul(w2, csub(apc, bpd));
    o[3 * s] = cmul(w3, csub(amc, jbmd));
  }
}

// In: x (N complex).  Scratch: y.  Returns the buffer holding the (unnormalised) transform.
// All GROUP threads of the group must call it; buffers are shared memory.
template <int N, int GROUP, bool INVERSE>
__device__ __forceinline__ float2 *fft_stockham(float2 *x, float2 *y, const float2 *__restrict__ tw, int tid) {
  int n = N, s = 1;
#pragma unroll
  for (; n >= 4; n >>= 2, s <<= 2) {
    radix4_pass<N, GROUP, INVERSE>(x, y, tw, tid, n, s);
    group_sync<GROUP>();
    float2 *t = x; x = y; y = t;
  }
  if (n == 2) {  // final radix-2 pass: p = 0, stride s = N/2, twiddle 1
    for (int t = tid; t < N / 2; t += GROUP) {
      const float2 a = x[t], b = x[t + N / 2];
      y[t] = cadd(a, b);
      y[t + N / 2] = csub(a, b);
    }
    group_sync<GROUP>();
    float2 *t = x; x = y; y = t;
  }
  return x;
}

// Real forward transform, split step: Z = FFT_N(z), z[n] = x[2n] + i x[2n+1]  ->
//   X[f] = (Z[f] + conj Z[N-f])/2 - (i/2) e^{-2 pi i f/L} (Z[f] - conj Z[N-f]),  f = 0..N, Z[N] = Z[0].
template <int N>
__device__ __forceinline__ float2 rfft_split(const float2 *Z, const float2 *__restrict__ tw, int f) {
  const float2 zf = Z[f & (N - 1)];
  const float2 zr = Z[(N - f) & (N - 1)];
  const float2 e = make_float2(0.5f * (zf.x + zr.x), 0.5f * (zf.y - zr.y));   // (Z[f] + conj Zr)/2
  const float2 d = make_float2(0.5f * (zf.x - zr.x), 0.5f * (zf.y + zr.y));   // (Z[f] - conj Zr)/2
  const float2 w = __ldg(tw + f);                                             // e^{-2 pi i f/L}
  const float2 wd = cmul(w, d);
  return make_float2(e.x + wd.y, e.y - wd.x);  // e - i * (w d)
}

// Real inverse transform, merge step: given Hermitian half spectrum S[0..N] (Im S[0], Im S[N] ignored)
//   Zin[f] = (S[f] + conj S[N-f])/2 + i e^{+2 pi i f/L} (S[f] - conj S[N-f])/2,   f = 0..N-1
// then z = IFFT_N(Zin) (unnormalised) gives x[2n] = Re z[n]/N, x[2n+1] = Im z[n]/N  where
// x[m] = (1/L) sum_{f<L} S_full[f] e^{+2 pi i f m/L}.
__device__ __forceinline__ float2 irfft_merge(float2 sf, float2 sr, float2 w_conj) {
  const float2 e = make_float2(0.5f * (sf.x + sr.x), 0.5f * (sf.y - sr.y));
  const float2 d = make_float2(0.5f * (sf.x - sr.x), 0.5f * (sf.y + sr.y));
  const float2 wd = cmul(w_conj, d);
  return make_float2(e.x - wd.y, e.y + wd.x);  // e + i * (w d)
}

}  // namespace delta
