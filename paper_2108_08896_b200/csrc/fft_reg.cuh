// Register-resident mixed-radix FFT for a group of T = N/E threads (N = L/2 complex points).
//
// Every thread keeps E points in registers; a pass is a radix-R butterfly done entirely in registers
// (R in {4, 8, 16}); between passes the group transposes through shared memory, addressed through an
// index map `m(e)` (any bijection of 0..N-1 onto distinct float2 slots that the group owns): FftPadMap is
// a private buffer padded by one slot per 16, the pair kernel maps onto the slots of its S tile.  Used for the forward transform of the STFT and for the inverse
// transform of the cross-correlation (Eq. 1d).  No cuFFT: every butterfly is here.
//
// Register/array correspondence, before AND after fft_inplace():   v[u]  <->  x[tid + T*u],  u < E,
// so global loads and stores with consecutive `tid` are coalesced and the result is in natural order.
//
// Decimation in frequency, Stockham ordering.  Pass p (radix R, stride S = product of the earlier
// radices) takes butterfly b = tid + T*i (i < E/R), q = b mod S, r = b / S:
//     y[q + S*(R*r + k)] = W_N^{S*r*k} * DFT_R( x[b + t*N/R], t < R )[k]
// The twiddles W_N^{S*r*k} come from per-pass tables built in float64 on the host (fft_twiddle_table):
//     table[off_p + (k-1)*(N/(R*S)) + r],  k = 1..R-1.
#pragma once
#include <cuda_runtime.h>
#include <math.h>

#ifdef __CUDACC__
#define DELTA_HD __host__ __device__ __forceinline__
#else
#define DELTA_HD inline
#endif

namespace delta {

DELTA_HD float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
DELTA_HD float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
DELTA_HD float2 cmul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
// multiply by the forward constant (wr, wi); the inverse transform uses its conjugate
template <bool INV>
DELTA_HD float2 cmul_c(float2 a, float wr, float wi) {
  return cmul(a, make_float2(wr, INV ? -wi : wi));
}
// forward: * (-i);  inverse: * (+i)
template <bool INV>
DELTA_HD float2 mul_w4(float2 a) {
  return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
}

template <bool INV>
DELTA_HD void dft4(float2 &a0, float2 &a1, float2 &a2, float2 &a3) {
  const float2 t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), t3 = mul_w4<INV>(csub(a1, a3));
  a0 = cadd(t0, t2);
  a2 = csub(t0, t2);
  a1 = cadd(t1, t3);
  a3 = csub(t1, t3);
}

template <int R, bool INV>
struct Dft;

template <bool INV>
struct Dft<4, INV> {
  static DELTA_HD void run(float2 *a) { dft4<INV>(a[0], a[1], a[2], a[3]); }
};

// n = 2 n1 + n2, k = k1 + 4 k2:  X[k1 + 4 k2] = E[k1] + (-1)^k2 W8^k1 O[k1]
template <bool INV>
struct Dft<8, INV> {
  static DELTA_HD void run(float2 *a) {
    constexpr float h = 0.70710678118654752440f;
    dft4<INV>(a[0], a[2], a[4], a[6]);
    dft4<INV>(a[1], a[3], a[5], a[7]);
    const float2 o0 = a[1];
    const float2 o1 = cmul_c<INV>(a[3], h, -h);
    const float2 o2 = mul_w4<INV>(a[5]);
    const float2 o3 = cmul_c<INV>(a[7], -h, -h);
    const float2 e0 = a[0], e1 = a[2], e2 = a[4], e3 = a[6];
    a[0] = cadd(e0, o0); a[4] = csub(e0, o0);
    a[1] = cadd(e1, o1); a[5] = csub(e1, o1);
    a[2] = cadd(e2, o2); a[6] = csub(e2, o2);
    a[3] = cadd(e3, o3); a[7] = csub(e3, o3);
  }
};

// n = 4 n1 + n2, k = k1 + 4 k2:  A[n2][k1] = DFT4_{n1} a[4 n1 + n2];  A *= W16^{n2 k1};  X[k1 + 4 k2] = DFT4_{n2} A[n2][k1]
template <bool INV>
struct Dft<16, INV> {
  static DELTA_HD void run(float2 *a) {
    constexpr float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f, h = 0.70710678118654752440f;
#pragma unroll
    for (int n2 = 0; n2 < 4; ++n2) dft4<INV>(a[n2], a[4 + n2], a[8 + n2], a[12 + n2]);
    // a[4 k1 + n2] now holds A[n2][k1]
    a[4 + 1] = cmul_c<INV>(a[4 + 1], c1, -s1);   // W16^1
    a[4 + 2] = cmul_c<INV>(a[4 + 2], h, -h);     // W16^2
    a[4 + 3] = cmul_c<INV>(a[4 + 3], s1, -c1);   // W16^3
    a[8 + 1] = cmul_c<INV>(a[8 + 1], h, -h);     // W16^2
    a[8 + 2] = mul_w4<INV>(a[8 + 2]);            // W16^4
    a[8 + 3] = cmul_c<INV>(a[8 + 3], -h, -h);    // W16^6
    a[12 + 1] = cmul_c<INV>(a[12 + 1], s1, -c1); // W16^3
    a[12 + 2] = cmul_c<INV>(a[12 + 2], -h, -h);  // W16^6
    a[12 + 3] = cmul_c<INV>(a[12 + 3], -c1, s1); // W16^9
#pragma unroll
    for (int k1 = 0; k1 < 4; ++k1) dft4<INV>(a[4 * k1], a[4 * k1 + 1], a[4 * k1 + 2], a[4 * k1 + 3]);
    // a[4 k1 + k2] = X[k1 + 4 k2]  ->  natural order
    float2 t;
    t = a[1]; a[1] = a[4]; a[4] = t;
    t = a[2]; a[2] = a[8]; a[8] = t;
    t = a[3]; a[3] = a[12]; a[12] = t;
    t = a[6]; a[6] = a[9]; a[9] = t;
    t = a[7]; a[7] = a[13]; a[13] = t;
    t = a[11]; a[11] = a[14]; a[14] = t;
  }
};

// ---------------------------------------------------------------------------------------------
// Geometry of a transform: E points per thread, NP passes of radices R0, R1, R2.  Variant V = 0 is the default
// (E = 16 where possible: fewest exchanges, used by the STFT); V = 1 is the narrow variant (E = 8: half the registers per
// thread and a whole warp per 256-point transform, used by the pair kernel where occupancy matters more).
template <int N, int V = 0>
struct FftGeom;
#define DELTA_FFT_GEOM(N_, V_, E_, NP_, R0_, R1_, R2_)                                      \
  template <>                                                                               \
  struct FftGeom<N_, V_> {                                                                  \
    static constexpr int N = N_, E = E_, NP = NP_, R0 = R0_, R1 = R1_, R2 = R2_, T = N_ / E_; \
    static constexpr int BUF = N_ + N_ / 16;                      /* padded exchange buffer */ \
    static constexpr int OFF1 = (R0_ - 1) * (N_ / R0_);           /* table offset of pass 1 */ \
    static constexpr int TABLE = OFF1 + (NP_ == 3 ? (R1_ - 1) * (N_ / (R0_ * R1_)) : 0);      \
  };
DELTA_FFT_GEOM(32, 0, 8, 2, 8, 4, 1)
DELTA_FFT_GEOM(64, 0, 8, 2, 8, 8, 1)
DELTA_FFT_GEOM(128, 0, 16, 2, 16, 8, 1)
DELTA_FFT_GEOM(256, 0, 16, 2, 16, 16, 1)
DELTA_FFT_GEOM(512, 0, 16, 3, 8, 8, 8)
DELTA_FFT_GEOM(1024, 0, 16, 3, 16, 8, 8)
DELTA_FFT_GEOM(2048, 0, 16, 3, 16, 16, 8)
DELTA_FFT_GEOM(256, 1, 8, 3, 8, 8, 4)
#undef DELTA_FFT_GEOM

DELTA_HD int fft_pad(int i) { return i + (i >> 4); }
// Exchange maps.  An element index always splits into a thread-dependent part e_t and a compile-time part e_c that occupy
// disjoint bits (e = e_t + e_c = e_t | e_c); a map turns e_t into a handle once (`pre`) and then addresses element
// e_t + e_c from the handle and e_c (`at`), so that the compile-time part folds into an immediate.
struct FftPadMap {
  float2 *buf;  // FftGeom<N>::BUF entries, private to the group
  typedef int Handle;
  DELTA_HD Handle pre(int e_t) const { return e_t; }
  DELTA_HD float2 &at(Handle h, int e_c) const { return buf[fft_pad(h + e_c)]; }
};

DELTA_HD float2 fft_ld_tw(const float2 *p) {
#ifdef __CUDA_ARCH__
  return *p;  // shared memory or global memory; the callers keep the tables in shared memory
#else
  return *p;
#endif
}

// One pass.  LAST: results stay in registers (natural order, see header); otherwise they go through the map.
// Butterfly b = tid + T i: with S | T the thread part of its output index is  (tid mod S) + S R (tid / S)  and the
// compile-time part  R T i + S k.
template <class G, int R, int S, bool LAST, bool INV, class Map>
DELTA_HD void fft_pass(float2 *v, const Map &m, const float2 *tp, int tid) {
  constexpr int N = G::N;
  constexpr int NB = G::E / R, CNT = N / (R * S);
  static_assert(LAST || G::T % S == 0, "the stride of a pass must divide the group size");
  const int r_t = tid / S;
  const typename Map::Handle h = m.pre((tid & (S - 1)) + S * R * r_t);
#pragma unroll
  for (int i = 0; i < NB; ++i) {
    float2 a[R];
#pragma unroll
    for (int t = 0; t < R; ++t) a[t] = v[i + NB * t];
    Dft<R, INV>::run(a);
    if constexpr (LAST) {
#pragma unroll
      for (int k = 0; k < R; ++k) v[i + NB * k] = a[k];
    } else {
      const int r = r_t + (G::T / S) * i;
#pragma unroll
      for (int k = 1; k < R; ++k) {
        float2 w = fft_ld_tw(tp + (k - 1) * CNT + r);
        if (INV) w.y = -w.y;
        a[k] = cmul(a[k], w);
      }
#pragma unroll
      for (int k = 0; k < R; ++k) m.at(h, R * G::T * i + S * k) = a[k];
    }
  }
}

template <class G, class Map>
DELTA_HD void fft_readback(float2 *v, const Map &m, int tid) {
  const typename Map::Handle h = m.pre(tid);
#pragma unroll
  for (int u = 0; u < G::E; ++u) v[u] = m.at(h, G::T * u);
}

#ifdef __CUDACC__
// Group barrier: groups of T <= 32 threads live inside one warp (all 32 lanes execute the same pass
// sequence), larger groups use the CTA barrier (every thread of the CTA must take part).
template <int T>
__device__ __forceinline__ void fft_group_sync() {
  if (T <= 32) __syncwarp(); else __syncthreads();
}
template <int T>
struct FftCtaSync {
  static __device__ __forceinline__ void sync() { fft_group_sync<T>(); }
};
// The same for a kernel whose CTA also holds warps that do not take part (a producer warp): groups wider than a warp
// meet at named barrier ID with NT participating threads (all the transform threads of the CTA).
template <int T, int ID, int NT>
struct FftNamedSync {
  static __device__ __forceinline__ void sync() {
    if (T <= 32) __syncwarp(); else asm volatile("bar.sync %0, %1;" ::"n"(ID), "n"(NT) : "memory");
  }
};

// The same with one named barrier per group: group g of the CTA (threads g T .. g T + T - 1, T a multiple of 32) meets at
// barrier 1 + g, so the groups of a CTA run free of each other.  At most 15 groups wider than a warp per CTA.
template <int T>
struct FftGroupBarSync {
  static __device__ __forceinline__ void sync() {
    if (T <= 32) __syncwarp(); else asm volatile("bar.sync %0, %1;" ::"r"(1 + (int)threadIdx.x / T), "n"(T) : "memory");
  }
};

// v[u] <-> x[tid + T*u] in, X[tid + T*u] out (unnormalised).  The slots behind `m` are shared memory owned
// by the group; other threads of the group may still be reading them when the call returns, so the group
// must pass another Sync::sync() before it writes them again.
template <class G, bool INV, class Sync, class Map>
__device__ __forceinline__ void fft_inplace_g(float2 *v, const Map &m, const float2 *__restrict__ tp, int tid) {
  fft_pass<G, G::R0, 1, false, INV>(v, m, tp, tid);
  Sync::sync();
  fft_readback<G>(v, m, tid);
  if constexpr (G::NP == 2) {
    fft_pass<G, G::R1, G::R0, true, INV>(v, m, tp, tid);
  } else {
    Sync::sync();
    fft_pass<G, G::R1, G::R0, false, INV>(v, m, tp + G::OFF1, tid);
    Sync::sync();
    fft_readback<G>(v, m, tid);
    fft_pass<G, G::R2, G::R0 * G::R1, true, INV>(v, m, tp, tid);
  }
}
template <int N, bool INV, class Map>
__device__ __forceinline__ void fft_inplace(float2 *v, const Map &m, const float2 *__restrict__ tp, int tid) {
  fft_inplace_g<FftGeom<N, 0>, INV, FftCtaSync<FftGeom<N, 0>::T>>(v, m, tp, tid);
}
#endif

// Host: the per-pass twiddle tables of FftGeom<N> (forward sign), float64 -> float32.
// `out` must hold fft_table_size(N) entries.  Returns the entry count, 0 for an unsupported N.
inline void fft_radices(int N, int V, int *np, int *r) {
  *np = 0;
  r[0] = r[1] = r[2] = 1;
#define DELTA_FFT_CASE(N_, V_) \
  if (N == N_ && V == V_) { *np = FftGeom<N_, V_>::NP; r[0] = FftGeom<N_, V_>::R0; r[1] = FftGeom<N_, V_>::R1; r[2] = FftGeom<N_, V_>::R2; }
  DELTA_FFT_CASE(32, 0) DELTA_FFT_CASE(64, 0) DELTA_FFT_CASE(128, 0) DELTA_FFT_CASE(256, 0)
  DELTA_FFT_CASE(512, 0) DELTA_FFT_CASE(1024, 0) DELTA_FFT_CASE(2048, 0) DELTA_FFT_CASE(256, 1)
#undef DELTA_FFT_CASE
}

inline int fft_table_size(int N, int V = 0) {
  int np, r[3];
  fft_radices(N, V, &np, r);
  if (np == 0) return 0;
  int n = (r[0] - 1) * (N / r[0]);
  if (np == 3) n += (r[1] - 1) * (N / (r[0] * r[1]));
  return n;
}

inline int fft_twiddle_table(int N, float2 *out, int V = 0) {
  int np, r[3];
  fft_radices(N, V, &np, r);
  if (np == 0) return 0;
  int o = 0, S = 1;
  for (int p = 0; p + 1 < np; ++p) {
    const int R = r[p], cnt = N / (R * S);
    for (int k = 1; k < R; ++k)
      for (int i = 0; i < cnt; ++i) {
        // W_N^{S*i*k}, exponent reduced in integers before the call to cos/sin
        const long long e = ((long long)S * i * k) % N;
        const double ang = -2.0 * 3.14159265358979323846 * (double)e / (double)N;
        out[o++] = make_float2((float)cos(ang), (float)sin(ang));
      }
    S *= R;
  }
  return o;
}

}  // namespace delta
