// a4 + a5 of the hot path: everything that is per channel pair.
//   pair_kernel       Eq. (1b) coherence, Eq. (1c) cross-phase, |Eq. (1a)| cross-power
//                     Eq. (1d) cross-correlation = inverse real FFT of S_ij, normalised   (R12)
//   auto_prep_kernel  1/sqrt(S_cc[f]) from caller-supplied autospectra (staged calls only)
//   s_unpack_kernel   test accessor: S layout -> complex64 [P][F]
//
// One CTA owns one block of PB consecutive (lexicographic) pairs, i.e. one contiguous [F][PB] tile of S and one
// contiguous run of rows in each output array.  The tile arrives with a single cp.async.bulk copy.  Phase A
// sweeps it with lanes along frequency (coalesced 128-byte stores of G, A, P).  Phase B gives every pair a
// group of T = N/E threads which form the half-length complex input of the inverse real transform in
// registers, run the register FFT of fft_reg.cuh using the pair's own (now dead) tile slots as exchange
// space, leave the 2N real lags there and sweep them out with lanes along the lag (coalesced stores of rho).
#include "delta_internal.h"
#include "fft_reg.cuh"

namespace delta {

namespace {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

template <int L>
struct PairCfg {
  static constexpr int N = L / 2, F = N + 1;
  using G = FftGeom<N>;
  static constexpr int T = G::T, E = G::E;
  static constexpr int PB = pair_block(L);
  static constexpr int THREADS = PB * T;
  static constexpr int SW = T < 32 ? 32 : T;  // threads that sweep one pair's row together
  static constexpr int PU = SW / T;           // pairs per sweep unit
  static constexpr size_t TILE_BYTES = (size_t)F * PB * sizeof(float2);
  static constexpr size_t SMEM = TILE_BYTES + 2 * PB * sizeof(float) + PB * sizeof(ushort2) + 16;
  static_assert(THREADS % 32 == 0 && THREADS <= 1024, "block shape");
  static_assert(TILE_BYTES % 16 == 0, "bulk copy size");
};

// exchange space of the register FFT = the tile slots of pair `pl` (one per row), rows permuted so that the
// strided accesses of the passes spread over the banks
template <int PB>
struct TileMap {
  float2 *tile;
  int pl;
  __device__ __forceinline__ float2 &operator()(int e) const {
    const int r = e ^ ((e >> 4) & 15);
    return tile[r * PB + ((pl ^ r) & (PB - 1))];
  }
};

// atan2 from a degree-13 odd minimax polynomial on [0, 1] (max error 3.2e-7 rad), octant folding
__device__ __forceinline__ float atan2_poly(float y, float x) {
  const float ax = fabsf(x), ay = fabsf(y);
  const float mx = fmaxf(ax, ay), mn = fminf(ax, ay);
  const float t = __fdividef(mn, fmaxf(mx, 1e-37f));
  const float u = t * t;
  float p = 0.006811792496591806f;
  p = fmaf(p, u, -0.0336042195558548f);
  p = fmaf(p, u, 0.07962366938591003f);
  p = fmaf(p, u, -0.1323334276676178f);
  p = fmaf(p, u, 0.19807815551757812f);
  p = fmaf(p, u, -0.3331736922264099f);
  p = fmaf(p, u, 0.9999961256980896f);
  float a = p * t;
  a = ay > ax ? 1.5707963267948966f - a : a;
  a = x < 0.f ? 3.14159265358979323846f - a : a;
  return copysignf(a, y);
}

__device__ __forceinline__ float sqrt_approx(float v) {
  float r;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
  return r;
}

// Real inverse transform, merge step: given the Hermitian half spectrum S[0..N] (Im S[0], Im S[N] ignored)
//   Zin[f] = (S[f] + conj S[N-f])/2 + i e^{+2 pi i f/L} (S[f] - conj S[N-f])/2,   f = 0..N-1
// then z = IFFT_N(Zin) (unnormalised) gives x[2n] = Re z[n]/N, x[2n+1] = Im z[n]/N  where
// x[m] = (1/L) sum_{f<L} S_full[f] e^{+2 pi i f m/L}.
__device__ __forceinline__ float2 irfft_merge(float2 sf, float2 sr, float2 w_conj) {
  const float2 e = make_float2(0.5f * (sf.x + sr.x), 0.5f * (sf.y - sr.y));
  const float2 d = make_float2(0.5f * (sf.x - sr.x), 0.5f * (sf.y + sr.y));
  const float2 wd = cmul(w_conj, d);
  return make_float2(e.x - wd.y, e.y + wd.x);  // e + i * (w d)
}

template <int W>
__device__ __forceinline__ void unit_sync() {
  if (W <= 32) __syncwarp(); else __syncthreads();
}

}  // namespace

template <int L>
__global__ void __launch_bounds__(PairCfg<L>::THREADS)
pair_kernel(const float2 *__restrict__ S, const float *__restrict__ Sauto, const float *__restrict__ Srsq,
            const ushort2 *__restrict__ pairs, const float2 *__restrict__ tw, const float2 *__restrict__ ftab,
            Layout lay, float *__restrict__ G, float *__restrict__ A, float *__restrict__ Pw, float *__restrict__ R) {
  using Cfg = PairCfg<L>;
  constexpr int N = Cfg::N, F = Cfg::F, T = Cfg::T, E = Cfg::E, PB = Cfg::PB, SW = Cfg::SW, PU = Cfg::PU;
  constexpr int THREADS = Cfg::THREADS, NW = THREADS / 32;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float2 *tile = reinterpret_cast<float2 *>(smem_raw);                        // [F][PB], slot = (pl ^ f) & (PB-1)
  float *rs = reinterpret_cast<float *>(smem_raw + Cfg::TILE_BYTES);          // [PB][2]: 1/sqrt(L R_cc[0]) of i, j
  ushort2 *ij_s = reinterpret_cast<ushort2 *>(rs + 2 * PB);                   // [PB]
  uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw + ((Cfg::TILE_BYTES + 2 * PB * sizeof(float) + PB * sizeof(ushort2) + 7) & ~(size_t)7));

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t p0 = (int64_t)blockIdx.x * PB;

  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(1));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"((uint32_t)Cfg::TILE_BYTES) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(tile)),
                 "l"(S + (int64_t)blockIdx.x * F * PB), "r"((uint32_t)Cfg::TILE_BYTES), "r"(smem_u32(bar))
                 : "memory");
  }
  if (tid < PB) ij_s[tid] = (p0 + tid < lay.P) ? pairs[p0 + tid] : make_ushort2(0, 0);
  __syncthreads();

  // R_cc[0] = (1/L) sum over all L bins of S_cc = (1/L) (S_cc[0] + 2 sum_{0<f<N} S_cc[f] + S_cc[N])
  if (R) {
    for (int idx = warp; idx < 2 * PB; idx += NW) {
      const ushort2 ij = ij_s[idx >> 1];
      const float *a = Sauto + (int64_t)((idx & 1) ? ij.y : ij.x) * F;
      float sum = 0.f;
      for (int f = lane; f < F; f += 32) sum = fmaf((f == 0 || f == N) ? 1.f : 2.f, __ldg(a + f), sum);
      for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
      if (lane == 0) rs[idx] = sum > 0.f ? rsqrtf(sum) : 0.f;
    }
  }
  __syncthreads();

  {  // the tile has landed?
    uint32_t ok = 0;
    while (!ok)
      asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                   : "=r"(ok) : "r"(smem_u32(bar)), "r"(0) : "memory");
  }

  const int unit = tid / SW, lu = tid % SW;

  // ---- phase A: G, A, P for bins 0..N-1, lanes along frequency --------------------------------
  if (G || A || Pw) {
#pragma unroll 1
    for (int pi = 0; pi < PU; ++pi) {
      const int pl = unit * PU + pi;
      const int64_t p = p0 + pl;
      if (p >= lay.P) continue;
      const ushort2 ij = ij_s[pl];
      const float *ri = Srsq + (int64_t)ij.x * F, *rj = Srsq + (int64_t)ij.y * F;
      const int64_t o = p * F;
#pragma unroll 4
      for (int f = lu; f < N; f += SW) {
        const float2 s = tile[f * PB + ((pl ^ f) & (PB - 1))];
        const float mag = sqrt_approx(fmaf(s.x, s.x, s.y * s.y));
        if (Pw) Pw[o + f] = mag;
        if (G) G[o + f] = mag * __ldg(ri + f) * __ldg(rj + f);
        if (A) A[o + f] = atan2_poly(s.y, s.x);
      }
    }
  }
  // Nyquist bin (row N is never used as exchange space, so it can be done by one thread per pair)
  if (tid < PB && p0 + tid < lay.P && (G || A || Pw)) {
    const int pl = tid;
    const ushort2 ij = ij_s[pl];
    const float2 s = tile[N * PB + ((pl ^ N) & (PB - 1))];
    const float mag = sqrt_approx(fmaf(s.x, s.x, s.y * s.y));
    const int64_t o = (p0 + pl) * F + N;
    if (Pw) Pw[o] = mag;
    if (G) G[o] = mag * __ldg(Srsq + (int64_t)ij.x * F + N) * __ldg(Srsq + (int64_t)ij.y * F + N);
    if (A) A[o] = atan2_poly(s.y, s.x);
  }
  if (!R) return;
  unit_sync<SW>();

  // ---- phase B: rho = irfft(S) / sqrt(R_ii[0] R_jj[0]) -------------------------------------------
  {
    const int pl = tid / T, gt = tid % T;
    const TileMap<PB> map{tile, pl};
    float2 v[E];
#pragma unroll
    for (int u = 0; u < E; ++u) {
      const int f = gt + T * u;
      float2 sf = tile[f * PB + ((pl ^ f) & (PB - 1))];
      float2 sr = tile[(N - f) * PB + ((pl ^ (N - f)) & (PB - 1))];
      if (f == 0) { sf.y = 0.f; sr.y = 0.f; }
      float2 w = __ldg(tw + f);
      w.y = -w.y;  // e^{+2 pi i f / L}
      v[u] = irfft_merge(sf, sr, w);
    }
    fft_group_sync<T>();  // every S value of the pair is in registers before its slots become exchange space
    fft_inplace<N, true>(v, map, ftab, gt);
    fft_group_sync<T>();
#pragma unroll
    for (int u = 0; u < E; ++u) map(gt + T * u) = v[u];  // z[n] = (x[2n], x[2n+1]) * N, natural order
  }
  unit_sync<SW>();
#pragma unroll 1
  for (int pi = 0; pi < PU; ++pi) {
    const int pl = unit * PU + pi;
    const int64_t p = p0 + pl;
    if (p >= lay.P) continue;
    const TileMap<PB> map{tile, pl};
    // rho = x / sqrt(R_ii[0] R_jj[0]),  x = z/N,  R_cc[0] = (sum over all L bins of S_cc)/L
    const float norm = 2.f * rs[2 * pl] * rs[2 * pl + 1];
    float *Rp = R + p * lay.nlags;
    for (int q = lu; q < lay.nlags; q += SW) {
      const int xi = (q - lay.M) & (L - 1);
      Rp[q] = reinterpret_cast<const float *>(&map(xi >> 1))[xi & 1] * norm;
    }
  }
}

// rsq[c][f] = 1/sqrt(S_cc[f]) (0 where S_cc[f] <= 0, reading R16)
__global__ void __launch_bounds__(256) auto_prep_kernel(const float *__restrict__ Sauto, float *__restrict__ rsq, int64_t n) {
  const int64_t idx = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (idx < n) {
    const float a = Sauto[idx];
    rsq[idx] = a > 0.f ? rsqrtf(a) : 0.f;
  }
}

// test accessor: S layout -> complex64 [P][F], lexicographic pairs
__global__ void __launch_bounds__(256) s_unpack_kernel(const float2 *__restrict__ S, Layout lay, float2 *__restrict__ out) {
  const int64_t total = lay.P * lay.F;
  for (int64_t idx = (int64_t)blockIdx.x * 256 + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * 256) {
    const int f = (int)(idx % lay.F);
    const int64_t p = idx / lay.F;
    out[idx] = S[((p >> lay.pb_shift) * lay.F + f) * lay.PB + ((p ^ f) & (lay.PB - 1))];
  }
}

// ------------------------------------------------------------------------------------------
template <int L>
static int launch_pair_L(delta_plan *p, const float *d_S, const float *d_auto, const float *d_rsq, float *d_G, float *d_A,
                         float *d_P, float *d_R, cudaStream_t st) {
  using Cfg = PairCfg<L>;
  const Layout &lay = p->lay;
  if (lay.Pblk == 0 || lay.P == 0) return DELTA_OK;
  int rc = opt_in_smem(pair_kernel<L>, Cfg::SMEM);
  if (rc) return rc;
  pair_kernel<L><<<(unsigned)lay.Pblk, Cfg::THREADS, Cfg::SMEM, st>>>(reinterpret_cast<const float2 *>(d_S), d_auto, d_rsq,
                                                                    p->d_pairs(), p->d_tw(), p->d_ftab(), lay, d_G, d_A, d_P,
                                                                    d_R);
  p->launches++;
  DELTA_CUDA_CHECK(cudaGetLastError());
  return DELTA_OK;
}

int launch_pair(delta_plan *p, const float *d_S, const float *d_auto, const float *d_rsq, float *d_G, float *d_A, float *d_P,
                float *d_R, cudaStream_t st) {
#define CALL(LL) launch_pair_L<LL>(p, d_S, d_auto, d_rsq, d_G, d_A, d_P, d_R, st)
  DELTA_SWITCH_L(p->lay.L, CALL)
#undef CALL
}

int launch_auto_prep(delta_plan *p, const float *d_auto, float *d_rsq, cudaStream_t st) {
  const int64_t n = (int64_t)p->lay.C * p->lay.F;
  auto_prep_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d_auto, d_rsq, n);
  p->launches++;
  DELTA_CUDA_CHECK(cudaGetLastError());
  return DELTA_OK;
}

int launch_s_unpack(delta_plan *p, const float *d_S, float *d_out, cudaStream_t st) {
  const int64_t total = p->lay.P * p->lay.F;
  if (total == 0) return DELTA_OK;
  const int64_t want = (total + 255) / 256;
  s_unpack_kernel<<<(unsigned)(want < 148 * 16 ? want : 148 * 16), 256, 0, st>>>(reinterpret_cast<const float2 *>(d_S), p->lay,
                                                                                 reinterpret_cast<float2 *>(d_out));
  p->launches++;
  DELTA_CUDA_CHECK(cudaGetLastError());
  return DELTA_OK;
}

}  // namespace delta
