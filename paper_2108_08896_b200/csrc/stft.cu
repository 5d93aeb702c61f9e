// a0 + a1 of the hot path:
//   offsets_kernel   a0  per-shot channel offsets o_c = mean of the first n_first samples   (R1)
//   chscale_kernel       per-channel power-of-two scale of the split-fp16 operands (tensor-core mode)
//   stft_kernel      a0+a1  normalise + periodic Hann + L-point real FFT of every segment
//   stft_unpack_kernel   test accessor: X layout -> complex64 [C][K][F]
//
// The real transform of a segment is an N = L/2 point complex FFT of z[n] = x[2n] + i x[2n+1] held in
// registers (fft_reg.cuh) followed by the split step; the split is fused into the transposed write-out.
#include <cooperative_groups.h>
#include <cuda_fp16.h>

#include "delta_internal.h"
#include "fft_reg.cuh"
#include "x_store.cuh"

namespace cg = cooperative_groups;

namespace delta {

// ------------------------------------------------------------------------------------------
// a0: o_c = mean of the first n_first samples (integer-exact sum for int16)
__global__ void __launch_bounds__(256) offsets_kernel(const void *__restrict__ x, int64_t ld, int in_dtype, int n_first,
                                                      double *__restrict__ offs, long long *__restrict__ isum) {
  const int c = blockIdx.x;
  __shared__ double red_d[8];
  __shared__ long long red_i[8];
  double sd = 0.0;
  long long si = 0;
  if (in_dtype == DELTA_I16) {
    const short *row = reinterpret_cast<const short *>(x) + (int64_t)c * ld;
    for (int t = threadIdx.x; t < n_first; t += 256) si += row[t];
  } else {
    const float *row = reinterpret_cast<const float *>(x) + (int64_t)c * ld;
    for (int t = threadIdx.x; t < n_first; t += 256) sd += (double)row[t];
  }
  for (int o = 16; o > 0; o >>= 1) {
    sd += __shfl_xor_sync(0xffffffffu, sd, o);
    si += __shfl_xor_sync(0xffffffffu, si, o);
  }
  if ((threadIdx.x & 31) == 0) {
    red_d[threadIdx.x >> 5] = sd;
    red_i[threadIdx.x >> 5] = si;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double td = 0.0;
    long long ti = 0;
    for (int w = 0; w < 8; ++w) {
      td += red_d[w];
      ti += red_i[w];
    }
    if (in_dtype == DELTA_I16) {
      isum[c] = ti;
      offs[c] = (double)ti / (double)n_first;
    } else {
      isum[c] = 0;
      offs[c] = td / (double)n_first;
    }
  }
}

// ------------------------------------------------------------------------------------------
// Sample access with the offset normalisation of reading R1 fused into the load.
struct SampleLoader {
  const void *x;
  int in_dtype, norm_mode;
  float o, inv_o;         // float input: offset and 1/offset
  long long isum;         // int16 input: integer sum over n_first samples
  float inv_isum, inv_n;  // 1/isum, 1/n_first
  int n_first;
  long long i_mul, i_sub;  // int16: numerator = x * i_mul - i_sub
  float i_scale, f_sub, f_scale;

  __device__ __forceinline__ void init(const void *x_, int in_dtype_, int norm_mode_, int n_first_,
                                       const double *__restrict__ offs, const long long *__restrict__ isums, int c) {
    x = x_; in_dtype = in_dtype_; norm_mode = norm_mode_; n_first = n_first_;
    o = 0.f; inv_o = 0.f; isum = 0; inv_isum = 0.f; inv_n = 0.f;
    i_mul = 1; i_sub = 0; i_scale = 1.f; f_sub = 0.f; f_scale = 1.f;
    if (norm_mode != DELTA_NORM_NONE) {
      const double od = offs[c];
      o = (float)od;
      inv_o = (float)(1.0 / od);
      isum = isums[c];
      inv_isum = (float)(1.0 / (double)isum);
      inv_n = (float)(1.0 / (double)n_first);
      i_mul = n_first; i_sub = isum; i_scale = norm_mode == DELTA_NORM_RELATIVE ? inv_isum : inv_n;
      f_sub = o; f_scale = norm_mode == DELTA_NORM_RELATIVE ? inv_o : 1.f;
    }
  }
  // branch-free forms (NONE: multiplier 1, subtrahend 0, scale 1: bit-identical to the plain conversion)
  __device__ __forceinline__ float conv_i16(int v) const {
    // (x - o) = (x n - sum)/n exactly in integers; one rounding at the conversion
    return __ll2float_rn((long long)v * i_mul - i_sub) * i_scale;
  }
  __device__ __forceinline__ float conv_f32(float v) const { return (v - f_sub) * f_scale; }
  __device__ __forceinline__ float operator()(int64_t idx) const {
    if (in_dtype == DELTA_I16) return conv_i16(reinterpret_cast<const short *>(x)[idx]);
    return conv_f32(reinterpret_cast<const float *>(x)[idx]);
  }
  // samples idx, idx+1; `pair_ok`: the element pair is naturally aligned (one vector load)
  __device__ __forceinline__ float2 two(int64_t idx, bool pair_ok) const {
    if (in_dtype == DELTA_I16) {
      if (pair_ok) {
        const short2 v = *reinterpret_cast<const short2 *>(reinterpret_cast<const short *>(x) + idx);
        return make_float2(conv_i16(v.x), conv_i16(v.y));
      }
      const short *p = reinterpret_cast<const short *>(x) + idx;
      return make_float2(conv_i16(p[0]), conv_i16(p[1]));
    }
    if (pair_ok) {
      const float2 v = *reinterpret_cast<const float2 *>(reinterpret_cast<const float *>(x) + idx);
      return make_float2(conv_f32(v.x), conv_f32(v.y));
    }
    const float *p = reinterpret_cast<const float *>(x) + idx;
    return make_float2(conv_f32(p[0]), conv_f32(p[1]));
  }
};

// per-channel power-of-two scale for the split-fp16 operands: |X| <= (L/2) max|y|  =>  scale * |X| <= 2^14.
__device__ __forceinline__ float scale_from_max(float m, float wsum) {
  const float bound = m * wsum;  // |X| <= sum_n w[n] |y| <= wsum max|y|   (Hann: wsum = L/2)
  float sc = 1.f;
  if (bound > 0.f && isfinite(bound)) {
    int e;
    frexpf(bound, &e);         // bound = mant * 2^e, mant in [0.5, 1)  =>  bound < 2^e
    sc = ldexpf(1.f, 14 - e);  // scale * bound < 2^14
  }
  return sc;
}

// One pass over the chunk for chunks too long for the cluster variant of stft_kernel.  grid = (C, NS): every block
// takes a slice of one channel (16-byte loads), the blocks of a channel combine their maxima with atomicMax on the
// float bits (all values are >= 0) and the last one to arrive writes the scale and re-arms the two words.
__global__ void __launch_bounds__(256)
chscale_kernel(const void *__restrict__ x, int64_t ld, int in_dtype, int norm_mode, int n_first,
               const double *__restrict__ offs, const long long *__restrict__ isum, int T, float wsum,
               float *__restrict__ chscale, unsigned *__restrict__ chmax, unsigned *__restrict__ chcnt) {
  const int c = blockIdx.x, NS = gridDim.y, tid = threadIdx.x;
  SampleLoader ldr;
  ldr.init(x, in_dtype, norm_mode, n_first, offs, isum, c);
  const int64_t row0 = (int64_t)c * ld;
  const int per = (((T + NS - 1) / NS) + 7) & ~7;
  const int s0 = blockIdx.y * per, s1 = min(T, s0 + per);
  float m = 0.f;
  if (in_dtype == DELTA_I16) {
    const short *r = reinterpret_cast<const short *>(x) + row0;
    int t = s0 + tid;
    if ((reinterpret_cast<uintptr_t>(r + s0) & 15) == 0) {
      const int nv = (s1 - s0) >> 3;
#pragma unroll 4
      for (int q = tid; q < nv; q += 256) {
        const uint4 v = *reinterpret_cast<const uint4 *>(r + s0 + 8 * q);
        const unsigned wv[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          m = fmaxf(m, fabsf(ldr.conv_i16((short)(wv[k] & 0xffffu))));
          m = fmaxf(m, fabsf(ldr.conv_i16((short)(wv[k] >> 16))));
        }
      }
      t = s0 + 8 * nv + tid;
    }
    for (; t < s1; t += 256) m = fmaxf(m, fabsf(ldr.conv_i16(r[t])));
  } else {
    const float *r = reinterpret_cast<const float *>(x) + row0;
    int t = s0 + tid;
    if ((reinterpret_cast<uintptr_t>(r + s0) & 15) == 0) {
      const int nv = (s1 - s0) >> 2;
#pragma unroll 4
      for (int q = tid; q < nv; q += 256) {
        const float4 v = *reinterpret_cast<const float4 *>(r + s0 + 4 * q);
        m = fmaxf(fmaxf(m, fabsf(ldr.conv_f32(v.x))), fabsf(ldr.conv_f32(v.y)));
        m = fmaxf(fmaxf(m, fabsf(ldr.conv_f32(v.z))), fabsf(ldr.conv_f32(v.w)));
      }
      t = s0 + 4 * nv + tid;
    }
    for (; t < s1; t += 256) m = fmaxf(m, fabsf(ldr.conv_f32(r[t])));
  }
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  __shared__ float red[8];
  if ((tid & 31) == 0) red[tid >> 5] = m;
  __syncthreads();
  if (tid == 0) {
#pragma unroll
    for (int w = 1; w < 8; ++w) m = fmaxf(m, red[w]);
    if (!(m == m)) m = __int_as_float(0x7f800000);  // NaN input: treat as +inf (scale 1)
    atomicMax(chmax + c, __float_as_uint(m));
    __threadfence();
    if (atomicAdd(chcnt + c, 1u) == (unsigned)(NS - 1)) {
      __threadfence();
      const float mm = __uint_as_float(atomicExch(chmax + c, 0u));
      chcnt[c] = 0u;
      chscale[c] = scale_from_max(mm, wsum);
    }
  }
}

// Predicated loads of int16 samples (0 where the predicate is off).  Written as PTX because the compiler turns the
// conditional loads of the int16 path into a branch around every element, and each load is then consumed before the next is
// issued: sixteen dependent memory latencies per thread instead of one (4 us of the config-4 STFT).
__device__ __forceinline__ uint32_t ldg_s16x2_if(const short *p, bool pred) {
  uint32_t v;
  asm("{\n\t.reg .pred q;\n\tsetp.ne.b32 q, %2, 0;\n\tmov.b32 %0, 0;\n\t@q ld.global.nc.b32 %0, [%1];\n\t}" : "=r"(v) : "l"(p), "r"((int)pred));
  return v;
}
__device__ __forceinline__ uint32_t ldg_s16_if(const short *p, bool pred) {  // zero-extended 16 bits
  uint32_t v;
  asm("{\n\t.reg .pred q;\n\tsetp.ne.b32 q, %2, 0;\n\tmov.b32 %0, 0;\n\t@q ld.global.nc.u16 %0, [%1];\n\t}" : "=r"(v) : "l"(p), "r"((int)pred));
  return v;
}

// ------------------------------------------------------------------------------------------
template <int L>
struct StftCfg {
  static constexpr int N = L / 2;
  using G = FftGeom<N>;
  static constexpr int T = G::T;
  // channels per CTA: two adjacent channels make the 16-byte pieces of the write-out whole 32-byte sectors (one channel per
  // CTA at nfft 2048 cost 25 % of the kernel: half-written sectors, twice the SM -> L2 bytes); nfft 4096 has room for one
  static constexpr int CH = N <= 1024 ? 2 : 1;
  static constexpr int NFFT = CH * kSegBlock;                      // transforms per CTA
  static constexpr int THREADS = NFFT * T;
  static constexpr int CHPAD = CH > 1 ? 16 / CH : 0;                 // float2 skew between channels (bank spread)
  static constexpr int SMEM_F2 = NFFT * G::BUF + CH * CHPAD;
};

// Sum of v over the T threads of a transform group (threads g*T .. g*T+T-1 of the CTA).  Groups wider than a warp go
// through shared memory with CTA barriers, so for T > 32 EVERY thread of the CTA must call it.
template <int T>
__device__ __forceinline__ float group_sum(float v, float *wsums, int tid) {
  constexpr int W = T < 32 ? T : 32;
#pragma unroll
  for (int o = W / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o, W);
  if (T > 32) {
    __syncthreads();
    if ((tid & 31) == 0) wsums[tid >> 5] = v;
    __syncthreads();
    constexpr int WPG = T / 32 > 0 ? T / 32 : 1;
    const int w0 = (tid / T) * WPG;
    v = 0.f;
#pragma unroll
    for (int w = 0; w < WPG; ++w) v += wsums[w0 + w];
  }
  return v;
}

// Real forward transform, split step: Z = FFT_N(z), z[n] = x[2n] + i x[2n+1]  ->
//   X[f] = (Z[f] + conj Z[N-f])/2 - (i/2) e^{-2 pi i f/L} (Z[f] - conj Z[N-f]),  f = 0..N, Z[N] = Z[0].
__device__ __forceinline__ float2 rfft_split(float2 zf, float2 zr, float2 w) {
  const float2 e = make_float2(0.5f * (zf.x + zr.x), 0.5f * (zf.y - zr.y));  // (Z[f] + conj Zr)/2
  const float2 d = make_float2(0.5f * (zf.x - zr.x), 0.5f * (zf.y + zr.y));  // (Z[f] - conj Zr)/2
  const float2 wd = cmul(w, d);
  return make_float2(e.x + wd.y, e.y - wd.x);  // e - i * (w d)
}

// CLUSTER (tensor-core mode, at most 8 segment blocks): the CTAs of one channel group form a thread-block cluster
// and agree on the per-channel fp16 scale through distributed shared memory, so no separate pass over the chunk
// (chscale_kernel) is needed.
// grid = (ceil(K/8), ceil(C/CH)).  Phase 1: one group of T threads per (channel, segment) transform.
// Phase 2: one thread per (channel, bin) gathers the 8 segments of the CTA and writes one 16-byte
// (fp16) or 32-byte (fp32) piece per operand plane of the frequency-major X layout.
template <int L, bool TC, bool CLUSTER, bool DETREND>
__global__ void __launch_bounds__(StftCfg<L>::THREADS, 1024 / StftCfg<L>::THREADS)
stft_kernel(const void *__restrict__ x, int64_t ld, int in_dtype, int norm_mode, int n_first,
            const double *__restrict__ offs, const long long *__restrict__ isum, const float2 *__restrict__ tw,
            const float *__restrict__ win, const float2 *__restrict__ ftab, Layout lay, void *__restrict__ Xout,
            float *__restrict__ wpart) {
  using Cfg = StftCfg<L>;
  using G = typename Cfg::G;
  constexpr int N = Cfg::N, T = Cfg::T, E = G::E, CH = Cfg::CH;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2 *zb = reinterpret_cast<float2 *>(smem_raw);
  __shared__ float wred[Cfg::THREADS / 32];  // per-warp energy of the windowed samples
  __shared__ float gsum[Cfg::THREADS / 32];  // per-warp sample sums (detrend, transforms wider than a warp)
  __shared__ float wmax[Cfg::THREADS / 32];  // per-warp max |y|
  __shared__ float cmax[CH];                 // per-channel max |y| over this CTA's segments (read by the cluster)
  __shared__ float csc[CH];                  // per-channel fp16 scale

  // tensor-core mode: the per-channel fp16 scales travel with the operands (C floats behind the planes of the X buffer)
  float *chscale = reinterpret_cast<float *>(reinterpret_cast<char *>(Xout) + lay.x_scale_off);
  pdl_launch_dependents();
  {
    // L2 prefetch of the CTA's samples, one request per 128-byte line.  It is a hint without a data dependence, so it
    // is issued before pdl_wait (while the predecessor drains) and with far more lines in flight than demand loads get:
    // the loads after the wait then find the chunk in L2 instead of paying the DRAM latency with 16 loads per thread.
    const size_t esz = in_dtype == DELTA_I16 ? 2 : 4;
    const int64_t s0 = (int64_t)blockIdx.x * kSegBlock * lay.H;
    const int64_t cnt = min((int64_t)(kSegBlock - 1) * lay.H + lay.Ls, (int64_t)lay.T - s0);
    const int nl = (int)((cnt * (int64_t)esz + 127) / 128) + 1;
    for (int i = threadIdx.x; i < CH * nl; i += Cfg::THREADS) {
      const int ch = blockIdx.y * CH + i / nl;
      if (ch < lay.C) {
        const char *a = reinterpret_cast<const char *>(x) + ((int64_t)ch * ld + s0) * esz + (int64_t)(i % nl) * 128;
        const char *end = reinterpret_cast<const char *>(x) + ((int64_t)ch * ld + s0 + cnt) * esz;
        if (a < end) asm volatile("prefetch.global.L2 [%0];" ::"l"(a));
      }
    }
  }
  pdl_wait();  // the chunk may come from the caller's previous kernel; X, wpart and the scales are read by ours
  if (lay.jitter_mask & kJitStftStart) __nanosleep((unsigned)(((blockIdx.x * 7 + blockIdx.y * 3) % 5) * lay.jitter_ns));  // (test hook)

  const int tid = threadIdx.x, g = tid / T, gt = tid % T;
  const int cl = g / kSegBlock, kk = g % kSegBlock;
  const int kb = blockIdx.x, c0 = blockIdx.y * CH;
  float2 *buf = zb + g * G::BUF + cl * Cfg::CHPAD;

  {
    const int c = c0 + cl, k = kb * kSegBlock + kk;
    float2 v[E], wv[E];
    float amax = 0.f;
    if (c < lay.C && k < lay.K) {
      SampleLoader ldr;
      ldr.init(x, in_dtype, norm_mode, n_first, offs, isum, c);
      const int64_t t0 = (int64_t)c * ld + (int64_t)k * lay.H;
      const size_t esz = in_dtype == DELTA_I16 ? 2 : 4;
      const bool pair_ok = ((t0 & 1) == 0) && ((reinterpret_cast<uintptr_t>(x) & (2 * esz - 1)) == 0);
      // all loads of the segment are issued before the first use (one DRAM latency per thread, not E);
      // samples beyond the segment length Ls <= L (zero-padded transforms, R22) are not read
      const int nfull = lay.Ls >> 1;
      const bool odd = lay.Ls & 1;
      float2 smp[E];
      if (in_dtype == DELTA_I16) {
        const short *xs = reinterpret_cast<const short *>(x) + t0;
        uint32_t raw[E];  // low half = sample 2n, high half = sample 2n + 1 (0 beyond the segment)
        if (pair_ok) {
#pragma unroll
          for (int u = 0; u < E; ++u) {
            const int n = gt + T * u;
            raw[u] = ldg_s16x2_if(xs + 2 * n, n < nfull) | ldg_s16_if(xs + 2 * n, n == nfull && odd);
          }
        } else {
#pragma unroll
          for (int u = 0; u < E; ++u) {
            const int n = gt + T * u;
            raw[u] = ldg_s16_if(xs + 2 * n, n < nfull || (n == nfull && odd)) | (ldg_s16_if(xs + 2 * n + 1, n < nfull) << 16);
          }
        }
#pragma unroll
        for (int u = 0; u < E; ++u)
          smp[u] = make_float2(ldr.conv_i16((short)(raw[u] & 0xffffu)), ldr.conv_i16((short)(raw[u] >> 16)));
      } else {
        const float *xf = reinterpret_cast<const float *>(x) + t0;
        float2 raw[E];
        if (pair_ok) {
#pragma unroll
          for (int u = 0; u < E; ++u) {
            const int n = gt + T * u;
            raw[u] = n < nfull ? *reinterpret_cast<const float2 *>(xf + 2 * n)
                               : make_float2((n == nfull && odd) ? xf[2 * n] : 0.f, 0.f);
          }
        } else {
#pragma unroll
          for (int u = 0; u < E; ++u) {
            const int n = gt + T * u;
            raw[u] = n < nfull ? make_float2(xf[2 * n], xf[2 * n + 1]) : make_float2((n == nfull && odd) ? xf[2 * n] : 0.f, 0.f);
          }
        }
#pragma unroll
        for (int u = 0; u < E; ++u) smp[u] = make_float2(ldr.conv_f32(raw[u].x), ldr.conv_f32(raw[u].y));
      }
      if (lay.Ls < L) {  // the padding is zero whatever the normalisation made of the unread samples
#pragma unroll
        for (int u = 0; u < E; ++u) {
          const int n = gt + T * u;
          if (n >= nfull) smp[u] = make_float2((n == nfull && odd) ? smp[u].x : 0.f, 0.f);
        }
      }
#pragma unroll
      for (int u = 0; u < E; ++u) wv[u] = __ldg(reinterpret_cast<const float2 *>(win) + gt + T * u);
      if (!DETREND) {
#pragma unroll
        for (int u = 0; u < E; ++u) {
          if (CLUSTER) amax = fmaxf(amax, fmaxf(fabsf(smp[u].x), fabsf(smp[u].y)));
          v[u] = make_float2(smp[u].x * wv[u].x, smp[u].y * wv[u].y);
        }
      } else {
#pragma unroll
        for (int u = 0; u < E; ++u) v[u] = smp[u];
      }
    } else {
#pragma unroll
      for (int u = 0; u < E; ++u) {
        v[u] = make_float2(0.f, 0.f);
        if (DETREND) wv[u] = make_float2(0.f, 0.f);
      }
    }
    if (DETREND) {  // subtract the mean of the segment's L samples (f1 variant), then the window;
      float sm = 0.f;  // every thread of the CTA takes part (group_sum may use CTA barriers)
#pragma unroll
      for (int u = 0; u < E; ++u) sm += v[u].x + v[u].y;
      sm = group_sum<T>(sm, gsum, tid);
      const float mean = sm / (float)lay.Ls;
#pragma unroll
      for (int u = 0; u < E; ++u) {
        v[u] = make_float2(v[u].x - mean, v[u].y - mean);
        if (CLUSTER) amax = fmaxf(amax, fmaxf(fabsf(v[u].x), fabsf(v[u].y)));
        v[u] = make_float2(v[u].x * wv[u].x, v[u].y * wv[u].y);
      }
    }
    {  // energy of the windowed segment (zero-lag autocorrelation of Eq. 1d by Parseval), fixed summation order
      float ss = 0.f;
#pragma unroll
      for (int u = 0; u < E; ++u) ss = fmaf(v[u].x, v[u].x, fmaf(v[u].y, v[u].y, ss));
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
      if (CLUSTER) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
      }
      if ((tid & 31) == 0) {
        wred[tid >> 5] = ss;
        if (CLUSTER) wmax[tid >> 5] = amax;
      }
    }
    if (CLUSTER) {
      // publish this CTA's per-channel max |y| to the cluster now; the matching wait comes after the FFT, so the
      // cluster barrier's latency is hidden behind the transform
      __syncthreads();
      if (tid < CH) {
        constexpr int WPC = kSegBlock * T / 32;
        float m = 0.f;
#pragma unroll
        for (int w = 0; w < WPC; ++w) m = fmaxf(m, wmax[tid * WPC + w]);
        cmax[tid] = m;
      }
      cg::this_cluster().barrier_arrive();
    }
    fft_inplace<N, false>(v, FftPadMap{buf}, ftab, gt);
    fft_group_sync<T>();  // every read-back of the group is done before Z overwrites the buffer
#pragma unroll
    for (int u = 0; u < E; ++u) buf[fft_pad(gt + T * u)] = v[u];
  }
  __syncthreads();
  if (tid < CH && c0 + tid < lay.C) {  // the 8 T threads of a channel are 8 T / 32 consecutive warps
    constexpr int WPC = kSegBlock * T / 32;
    float e = 0.f;
#pragma unroll
    for (int w = 0; w < WPC; ++w) e += wred[tid * WPC + w];
    wpart[(int64_t)(c0 + tid) * lay.nkb + kb] = e;
    if (TC && !CLUSTER && kb == 0 && lay.estimator == DELTA_EST_PHASE_LOCK) chscale[c0 + tid] = 8192.f;  // unit phasors
  }
  if (CLUSTER) {
    // per-channel power-of-two scale: sum_n w[n] |y| <= (L/2) max|y|  =>  scale * |X| < 2^14 (same rule as chscale_kernel)
    cg::cluster_group cluster = cg::this_cluster();
    cluster.barrier_wait();  // every CTA of the channel group has published cmax
    if (tid < CH) {
      float m = 0.f;
      const unsigned nb = cluster.num_blocks();
      for (unsigned r = 0; r < nb; ++r) m = fmaxf(m, *cluster.map_shared_rank(&cmax[tid], r));
      const float sc = scale_from_max(m, lay.wsum);
      csc[tid] = sc;
      if (kb == 0 && c0 + tid < lay.C) chscale[c0 + tid] = lay.estimator == DELTA_EST_PHASE_LOCK ? 8192.f : sc;
    }
    cluster.barrier_arrive();  // remote reads of cmax are done; waited for just before the CTA exits
    __syncthreads();           // csc is visible to the CTA
  }

  if (lay.jitter_mask & kJitStftMid) __nanosleep((unsigned)(((blockIdx.x * 3 + blockIdx.y + 1) % 4) * lay.jitter_ns));  // (test hook)
  // Phase 2.  Bins f and N - f come from the same pair Z[f], Z[N-f]:  with e = (Z[f] + conj Z[N-f])/2,
  // d = (Z[f] - conj Z[N-f])/2 and (a, b) = e^{-2 pi i f/L} d:  X[f] = (e.x + b, e.y - a),  X[N-f] = (e.x - b, -e.y - a).
  // One thread does both for the 8 segments of the CTA; bin N/2 (its own partner) is done once.
  auto store_bin = [&](int c, int pcl, int f, const float *re, const float *im) {
    // split fp16 scale of the channel (2^13 for unit phasors); unused in FP32 mode
    const float sc = !TC ? 1.f : (lay.estimator == DELTA_EST_PHASE_LOCK ? 8192.f : (CLUSTER ? csc[pcl] : chscale[c]));
    store_x_bin<TC>(Xout, lay, kb, c, f, sc, re, im);
  };
  // Work items: (channel, f0) with f0 = 0 .. N/2 - 1, i.e. CH N/2 of them; with 16 points per thread that is exactly the
  // number of threads, so the loop runs once.  Bin N/2, its own partner, is a second turn of the item of f0 = 0 (as a 129th
  // item per channel it sent two threads of the CTA through the whole loop again while all the others waited; as a third
  // inline store of every thread it cost registers: spills at nfft 1024).
  constexpr int HB = N / 2;
  for (int idx = tid; idx < CH * HB; idx += Cfg::THREADS) {
    const int pcl = idx % CH, f0 = idx / CH;
    const int c = c0 + pcl;
    if (c >= lay.C) continue;
    const float2 *zc = zb + pcl * (kSegBlock * G::BUF + Cfg::CHPAD);
    for (int f = f0; f <= N / 2; f += (f0 == 0 ? N / 2 : N)) {  // f0 = 0: f = 0, N/2;  else: f = f0
      const float2 w = __ldg(tw + f);  // e^{-2 pi i f/L}
      const int i_f = fft_pad(f), i_r = fft_pad((N - f) & (N - 1));
      float re[kSegBlock], im[kSegBlock], re2[kSegBlock], im2[kSegBlock];
#pragma unroll
      for (int s = 0; s < kSegBlock; ++s) {
        const float2 zf = zc[s * G::BUF + i_f], zr = zc[s * G::BUF + i_r];
        const float2 e = make_float2(0.5f * (zf.x + zr.x), 0.5f * (zf.y - zr.y));
        const float2 d = make_float2(0.5f * (zf.x - zr.x), 0.5f * (zf.y + zr.y));
        const float2 wd = cmul(w, d);
        re[s] = e.x + wd.y;
        im[s] = e.y - wd.x;
        re2[s] = e.x - wd.y;
        im2[s] = -e.y - wd.x;
      }
      store_bin(c, pcl, f, re, im);
      if (2 * f != N) store_bin(c, pcl, N - f, re2, im2);
    }
  }
  if (CLUSTER) cg::this_cluster().barrier_wait();  // no CTA exits while its cmax may still be read
}

// test accessor: X layout -> complex64 [C][K][F]
__global__ void __launch_bounds__(256)
stft_unpack_kernel(const void *__restrict__ Xin, Layout lay, int tc_mode, float2 *__restrict__ out) {
  const float *chscale = reinterpret_cast<const float *>(reinterpret_cast<const char *>(Xin) + lay.x_scale_off);
  const int64_t total = (int64_t)lay.C * lay.K * lay.F;
  for (int64_t idx = (int64_t)blockIdx.x * 256 + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * 256) {
    const int f = (int)(idx % lay.F);
    const int64_t ck = idx / lay.F;
    const int k = (int)(ck % lay.K), c = (int)(ck / lay.K);
    const int kc = k / kSegBlock, kk = k % kSegBlock;
    const int64_t plane = (int64_t)lay.Kc * lay.Cp * kSegBlock;
    const int64_t within = ((int64_t)kc * lay.Cp + c) * kSegBlock + kk;
    const int64_t base = (int64_t)f * lay.x_elems_per_f;
    float2 v;
    if (!tc_mode) {
      const float *X = reinterpret_cast<const float *>(Xin);
      v = make_float2(X[base + within], X[base + plane + within]);
    } else {
      const __half *X = reinterpret_cast<const __half *>(Xin);
      const float inv = 1.f / chscale[c];
      v.x = (__half2float(X[base + 0 * plane + within]) + __half2float(X[base + 2 * plane + within])) * inv;
      v.y = (__half2float(X[base + 1 * plane + within]) + __half2float(X[base + 3 * plane + within])) * inv;
    }
    out[idx] = v;
  }
}

// ------------------------------------------------------------------------------------------
// launchers
int launch_offsets(delta_plan *p, const void *d_x, int64_t ld, int n_first, cudaStream_t st) {
  offsets_kernel<<<p->lay.C, 256, 0, st>>>(d_x, ld, p->cfg.in_dtype, n_first, p->d_offs(), p->d_isum());
  p->launches++;
  DELTA_CUDA_CHECK(cudaGetLastError());
  return DELTA_OK;
}

template <int L, bool TC, bool CLUSTER, bool DETREND>
static int launch_stft_LTD(delta_plan *p, const void *d_x, int64_t ld, void *d_X, cudaStream_t st) {
  using Cfg = StftCfg<L>;
  const Layout &lay = p->lay;
  const size_t smem = (size_t)Cfg::SMEM_F2 * sizeof(float2);
  int rc = opt_in_smem(stft_kernel<L, TC, CLUSTER, DETREND>, smem);
  if (rc) return rc;
  // the segment blocks of one channel group are one cluster
  LaunchCfg lc(dim3(lay.nkb, (lay.C + Cfg::CH - 1) / Cfg::CH), dim3(Cfg::THREADS), smem, st, p->use_pdl, CLUSTER ? lay.nkb : 0);
  DELTA_CUDA_CHECK(cudaLaunchKernelEx(&lc.cfg, stft_kernel<L, TC, CLUSTER, DETREND>, d_x, ld, p->cfg.in_dtype, p->cfg.norm_mode, p->n_first,
                                      (const double *)p->d_offs(), (const long long *)p->d_isum(), p->d_tw(), p->d_win(),
                                      p->d_ftab(), lay, d_X, p->d_wpart()));
  p->launches++;
  DELTA_CUDA_CHECK(cudaGetLastError());
  return DELTA_OK;
}

template <int L, bool TC, bool CLUSTER>
static int launch_stft_LT(delta_plan *p, const void *d_x, int64_t ld, void *d_X, cudaStream_t st) {
  return p->lay.detrend == DELTA_DETREND_CONSTANT ? launch_stft_LTD<L, TC, CLUSTER, true>(p, d_x, ld, d_X, st)
                                                  : launch_stft_LTD<L, TC, CLUSTER, false>(p, d_x, ld, d_X, st);
}

template <int L>
static int launch_stft_L(delta_plan *p, const void *d_x, int64_t ld, void *d_X, cudaStream_t st) {
  const Layout &lay = p->lay;
  if (p->contraction == DELTA_CONTRACT_TC) {
    if (lay.nkb <= 8) return launch_stft_LT<L, true, true>(p, d_x, ld, d_X, st);  // scale agreed inside the cluster
    if (lay.estimator == DELTA_EST_PHASE_LOCK) return launch_stft_LT<L, true, false>(p, d_x, ld, d_X, st);  // fixed scale
    int ns = (8 * p->num_sms + lay.C - 1) / lay.C;  // about 8 blocks per SM
    ns = ns < 1 ? 1 : (ns > 64 ? 64 : ns);
    chscale_kernel<<<dim3(lay.C, ns), 256, 0, st>>>(d_x, ld, p->cfg.in_dtype, p->cfg.norm_mode, p->n_first, p->d_offs(),
                                                    p->d_isum(), lay.T,
                                                    lay.wsum * (lay.detrend ? 2.f : 1.f),  // |y - mean| <= 2 max|y|
                                                    reinterpret_cast<float *>(reinterpret_cast<char *>(d_X) + lay.x_scale_off),
                                                    p->d_chmax(), p->d_chcnt());
    p->launches++;
    DELTA_CUDA_CHECK(cudaGetLastError());
    return launch_stft_LT<L, true, false>(p, d_x, ld, d_X, st);
  }
  return launch_stft_LT<L, false, false>(p, d_x, ld, d_X, st);
}

// ------------------------------------------------------------------------------------------
// Transform lengths that are not powers of two (the paper fixes no segment length, L107): the
// definition itself,  X[k, f] = sum_n w[n] y[kH + n] e^{-2 pi i f n / L},  as a direct sum over the windowed samples of a
// segment block held in shared memory (the phase index f n mod L is advanced by additions).  O(L^2) per segment: a
// correct, unhurried path for the odd case (a 500-point transform costs about 0.1 ms per 192-channel chunk); the
// register FFT serves the powers of two.  grid = (ceil(K/8), C), 256 threads; shared memory: float [8][L].
template <bool TC, bool DETREND>
__global__ void __launch_bounds__(256)
stft_dft_kernel(const void *__restrict__ x, int64_t ld, int in_dtype, int norm_mode, int n_first,
                const double *__restrict__ offs, const long long *__restrict__ isum, const float2 *__restrict__ tw,
                const float *__restrict__ win, Layout lay, void *__restrict__ Xout, float *__restrict__ wpart) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float *seg = reinterpret_cast<float *>(smem_raw);  // [8][L]
  __shared__ float red[8];
  const float *chscale = reinterpret_cast<const float *>(reinterpret_cast<const char *>(Xout) + lay.x_scale_off);
  pdl_launch_dependents();
  pdl_wait();
  const int tid = threadIdx.x, kb = blockIdx.x, c = blockIdx.y, L = lay.L;
  SampleLoader ldr;
  ldr.init(x, in_dtype, norm_mode, n_first, offs, isum, c);
  for (int idx = tid; idx < kSegBlock * L; idx += 256) {
    const int k8 = idx / L, n = idx - k8 * L, k = kb * kSegBlock + k8;
    seg[idx] = (k < lay.K && n < lay.Ls) ? ldr((int64_t)c * ld + (int64_t)k * lay.H + n) : 0.f;
  }
  __syncthreads();
  {  // warp k8 owns segment k8: optional detrend (mean of the Ls samples), window, energy of the windowed samples
    const int k8 = tid >> 5, lane = tid & 31;
    float *sk = seg + k8 * L;
    float mean = 0.f;
    if (DETREND) {
      float sm = 0.f;
      for (int n = lane; n < lay.Ls; n += 32) sm += sk[n];
      for (int o = 16; o > 0; o >>= 1) sm += __shfl_xor_sync(0xffffffffu, sm, o);
      mean = kb * kSegBlock + k8 < lay.K ? sm / (float)lay.Ls : 0.f;
    }
    float ss = 0.f;
    for (int n = lane; n < L; n += 32) {
      const float v = (sk[n] - mean) * __ldg(win + n);  // the window is zero beyond Ls
      sk[n] = v;
      ss = fmaf(v, v, ss);
    }
    for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
    if (lane == 0) red[k8] = ss;
  }
  __syncthreads();
  if (tid == 0) {
    float e = 0.f;
    for (int w = 0; w < 8; ++w) e += red[w];
    wpart[(int64_t)c * lay.nkb + kb] = e;
  }
  const float sc = !TC ? 1.f : (lay.estimator == DELTA_EST_PHASE_LOCK ? 8192.f : chscale[c]);
  for (int f = tid; f < lay.F; f += 256) {
    float re[kSegBlock], im[kSegBlock];
#pragma unroll
    for (int q = 0; q < kSegBlock; ++q) re[q] = im[q] = 0.f;
    int idx = 0;  // f n mod L
    for (int n = 0; n < L; ++n) {
      const float2 w = __ldg(tw + idx);  // e^{-2 pi i (f n mod L) / L}
#pragma unroll
      for (int q = 0; q < kSegBlock; ++q) {
        const float sv = seg[q * L + n];
        re[q] = fmaf(sv, w.x, re[q]);
        im[q] = fmaf(sv, w.y, im[q]);
      }
      idx += f;
      if (idx >= L) idx -= L;
    }
    store_x_bin<TC>(Xout, lay, kb, c, f, sc, re, im);
  }
}

static int launch_stft_dft(delta_plan *p, const void *d_x, int64_t ld, void *d_X, cudaStream_t st) {
  const Layout &lay = p->lay;
  const bool tc = p->contraction == DELTA_CONTRACT_TC, det = lay.detrend == DELTA_DETREND_CONSTANT;
  if (tc && lay.estimator != DELTA_EST_PHASE_LOCK) {  // per-channel fp16 scales: one pass over the chunk
    int ns = (8 * p->num_sms + lay.C - 1) / lay.C;
    ns = ns < 1 ? 1 : (ns > 64 ? 64 : ns);
    chscale_kernel<<<dim3(lay.C, ns), 256, 0, st>>>(d_x, ld, p->cfg.in_dtype, p->cfg.norm_mode, p->n_first, p->d_offs(),
                                                    p->d_isum(), lay.T, lay.wsum * (det ? 2.f : 1.f),
                                                    reinterpret_cast<float *>(reinterpret_cast<char *>(d_X) + lay.x_scale_off),
                                                    p->d_chmax(), p->d_chcnt());
    p->launches++;
    DELTA_CUDA_CHECK(cudaGetLastError());
  }
  const size_t smem = (size_t)kSegBlock * lay.L * sizeof(float);
  LaunchCfg lc(dim3(lay.nkb, lay.C), dim3(256), smem, st, p->use_pdl);
#define DELTA_DFT_LAUNCH(TC_, DET_)                                                                                        \
  do {                                                                                                                     \
    int rc = opt_in_smem(stft_dft_kernel<TC_, DET_>, smem);                                                                \
    if (rc) return rc;                                                                                                     \
    DELTA_CUDA_CHECK(cudaLaunchKernelEx(&lc.cfg, stft_dft_kernel<TC_, DET_>, d_x, ld, p->cfg.in_dtype, p->cfg.norm_mode,   \
                                        p->n_first, (const double *)p->d_offs(), (const long long *)p->d_isum(), p->d_tw(), \
                                        p->d_win(), lay, d_X, p->d_wpart()));                                              \
  } while (0)
  if (tc && det) DELTA_DFT_LAUNCH(true, true);
  else if (tc) DELTA_DFT_LAUNCH(true, false);
  else if (det) DELTA_DFT_LAUNCH(false, true);
  else DELTA_DFT_LAUNCH(false, false);
#undef DELTA_DFT_LAUNCH
  p->launches++;
  DELTA_CUDA_CHECK(cudaGetLastError());
  return DELTA_OK;
}

int launch_stft(delta_plan *p, const void *d_x, int64_t ld, void *d_X, cudaStream_t st) {
  if (!has_fft_path(p->lay.L)) return launch_stft_dft(p, d_x, ld, d_X, st);
#define CALL(LL) launch_stft_L<LL>(p, d_x, ld, d_X, st)
  DELTA_SWITCH_L(p->lay.L, CALL)
#undef CALL
}

// The padding of the X layout (rows C..Cp-1 of every [kc] block, and the blocks kc >= ceil(K/8)) is read by both
// contractions and written by no kernel: the workspace X is zeroed once, a caller-supplied X here.  One thread per
// 8-segment run (16 bytes of fp16 or 32 bytes of fp32).
__global__ void __launch_bounds__(256) stft_pad_zero_kernel(void *__restrict__ Xout, Layout lay, int planes, int elem_bytes) {
  const int64_t total = (int64_t)lay.F * planes * lay.Kc * lay.Cp;
  for (int64_t idx = (int64_t)blockIdx.x * 256 + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * 256) {
    const int c = (int)(idx % lay.Cp);
    const int kc = (int)((idx / lay.Cp) % lay.Kc);
    if (c < lay.C && kc < lay.nkb) continue;
    uint4 *q = reinterpret_cast<uint4 *>(reinterpret_cast<char *>(Xout) + idx * kSegBlock * elem_bytes);
    q[0] = make_uint4(0u, 0u, 0u, 0u);
    if (elem_bytes == 4) q[1] = make_uint4(0u, 0u, 0u, 0u);
  }
}

int launch_stft_pad_zero(delta_plan *p, void *d_X, cudaStream_t st) {
  const Layout &lay = p->lay;
  if (lay.Cp == lay.C && lay.Kc == lay.nkb) return DELTA_OK;
  const bool tc = p->contraction == DELTA_CONTRACT_TC;
  const int64_t total = (int64_t)lay.F * (tc ? 4 : 2) * lay.Kc * lay.Cp;
  const int64_t want = (total + 255) / 256;
  stft_pad_zero_kernel<<<(unsigned)(want < 148 * 16 ? want : 148 * 16), 256, 0, st>>>(d_X, lay, tc ? 4 : 2, tc ? 2 : 4);
  p->launches++;
  DELTA_CUDA_CHECK(cudaGetLastError());
  return DELTA_OK;
}

int launch_stft_unpack(delta_plan *p, const void *d_X, float *d_out, cudaStream_t st) {
  const int64_t total = (int64_t)p->lay.C * p->lay.K * p->lay.F;
  const int64_t want = (total + 255) / 256;
  const int blocks = (int)(want < 148 * 16 ? want : 148 * 16);
  stft_unpack_kernel<<<blocks, 256, 0, st>>>(d_X, p->lay, p->contraction == DELTA_CONTRACT_TC, reinterpret_cast<float2 *>(d_out));
  p->launches++;
  DELTA_CUDA_CHECK(cudaGetLastError());
  return DELTA_OK;
}

}  // namespace delta
