// a4 + a5 of the hot path: everything that is per channel pair.
//   pair_kernel       Eq. (1b) coherence, Eq. (1c) cross-phase, |Eq. (1a)| cross-power
//                     Eq. (1d) cross-correlation = inverse real FFT of S_ij, normalised   (R12)
//   auto_prep_kernel  1/sqrt(S_cc[f]) from caller-supplied autospectra (staged calls only)
//   s_unpack_kernel   test accessor: S layout -> complex64 [P][F]
//
// One CTA owns one block of PB consecutive (lexicographic) pairs, i.e. one contiguous [F][PB] tile of S and one
// contiguous run of rows in each output array.  The tile arrives with a single cp.async.bulk copy.  Every pair
// has a group of T = N/E threads; thread gt of the group owns the bins f = gt + T u (u < E), which is exactly the
// register layout the inverse FFT of fft_reg.cuh starts from.  Each S value is therefore read from shared memory
// once for G, A, P (stored straight away, 16 lanes = 64 contiguous bytes per row) and for the merge step of the
// inverse real transform; the transform exchanges through a private padded buffer that aliases the (by then
// dead) tile, ends in registers in natural order, and rho is stored from registers as float2.
#include "delta_internal.h"
#include "fft_reg.cuh"

namespace delta {

namespace {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

struct PairConsts {
  float2 wstep[16];  // e^{-2 pi i T u / L}
};

template <int L>
struct PairCfg {
  static constexpr int N = L / 2, F = N + 1;
  using G = FftGeom<N, pair_fft_variant(N)>;
  static constexpr int T = G::T, E = G::E;
  static constexpr int PB = pair_block(L);
  static constexpr int THREADS = PB * T;
  // resident warps per SM the register budget is sized for: 48 (40 registers) with 8 points per thread, else 32 (64)
#ifndef DELTA_PAIR_WARPS
#define DELTA_PAIR_WARPS 32
#endif
  static constexpr int WARPS = E <= 8 ? 48 : DELTA_PAIR_WARPS;
  static constexpr int MIN_CTAS = (WARPS * 32) / THREADS > 0 ? (WARPS * 32) / THREADS : 1;
  static constexpr size_t TILE_BYTES = (size_t)F * PB * sizeof(float2);
  static constexpr size_t EXCH_BYTES = (size_t)PB * G::BUF * sizeof(float2);
  static constexpr size_t BUF_BYTES = ((TILE_BYTES > EXCH_BYTES ? TILE_BYTES : EXCH_BYTES) + 15) & ~(size_t)15;
  static constexpr int FP = (F + 3) & ~3;                                   // pitch of the rsq table
  static constexpr size_t ROWS_BYTES = (size_t)PB * FP * sizeof(float);     // 1/sqrt(S_jj) row of every pair's j
  static constexpr size_t OFF_RS = BUF_BYTES + ROWS_BYTES;                    // float [2][PB]
  static constexpr size_t OFF_IJ = OFF_RS + 2 * PB * sizeof(float);           // ushort2 [PB]
  static constexpr size_t OFF_PG = OFF_IJ + PB * sizeof(ushort2);             // int [PB]: lexicographic index (pair lists)
  static constexpr size_t OFF_BAR = (OFF_PG + PB * sizeof(int) + 7) & ~(size_t)7;
  static constexpr size_t SMEM = OFF_BAR + 16;
  static_assert(THREADS % 32 == 0 && THREADS <= 1024, "block shape");
  static_assert(TILE_BYTES % 16 == 0, "bulk copy size");
  static_assert((T & (T - 1)) == 0 && (PB & (PB - 1)) == 0, "powers of two");
};

// atan2 from a degree-13 odd minimax polynomial on [0, 1] (max error 3.2e-7 rad), octant folding
__device__ __forceinline__ float atan2_poly(float y, float x) {
  const float ax = fabsf(x), ay = fabsf(y);
  const float mx = fmaxf(ax, ay), mn = fminf(ax, ay);
  float rc;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rc) : "f"(fmaxf(mx, 1e-37f)));
  const float t = mn * rc;
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
// irfft_merge2 returns twice that Zin (the halvings are left to the caller's normalisation).
__device__ __forceinline__ float2 irfft_merge2(float2 sf, float2 sr, float2 w_conj) {
  const float2 e = make_float2(sf.x + sr.x, sf.y - sr.y);
  const float2 d = make_float2(sf.x - sr.x, sf.y + sr.y);
  const float2 wd = cmul(w_conj, d);
  return make_float2(e.x - wd.y, e.y + wd.x);  // e + i * (w d)
}

// (i, j) of lexicographic pair p: row i holds the pairs [start(i), start(i+1)), start(i) = i C - i (i + 1) / 2.
// Float estimate of the root, then exact integer correction.
__device__ __forceinline__ ushort2 pair_of(int64_t p, int C) {
  const float b = 2.f * (float)C - 1.f;
  int i = (int)((b - sqrtf(fmaxf(b * b - 8.f * (float)p, 0.f))) * 0.5f);
  i = i < 0 ? 0 : (i > C - 2 ? C - 2 : i);
  auto start = [C](int r) { return (int64_t)r * C - ((int64_t)r * (r + 1)) / 2; };
  while (i < C - 2 && start(i + 1) <= p) ++i;
  while (i > 0 && start(i) > p) --i;
  return make_ushort2((unsigned short)i, (unsigned short)(p - start(i) + i + 1));
}

// Output stores: the results are written once and never read by this library, so they are marked streaming
// (evict-first) to keep S and X, which the next kernels re-read, in L2.
#ifdef DELTA_PLAIN_STORES
#define ST4(p, v) (*reinterpret_cast<float4 *>(p) = (v))
#define ST2(p, v) (*reinterpret_cast<float2 *>(p) = (v))
#define ST1(p, v) (*(p) = (v))
#else
#define ST4(p, v) __stcs(reinterpret_cast<float4 *>(p), (v))
#define ST2(p, v) __stcs(reinterpret_cast<float2 *>(p), (v))
#define ST1(p, v) __stcs((p), (v))
#endif

}  // namespace

// GAPALL: G, A and Pw are all requested (no per-element pointer tests)
// FULL: max_lag == L/2 (every lag of the circular correlation is stored; the two end points are the same sample)
// Zero-lag autocorrelations (R12): sum over all L bins of S_cc = rscale * sum_{k<nrp} rpart[c rp_stride + k].
template <int L, bool FULL, bool GAPALL>
__global__ void __launch_bounds__(PairCfg<L>::THREADS, PairCfg<L>::MIN_CTAS)
pair_kernel(const float2 *__restrict__ S, const float *__restrict__ Srsq, const float *__restrict__ rpart, int nrp,
            int rp_stride, float rscale, const ushort2 *__restrict__ list, const float2 *__restrict__ tw,
            const float2 *__restrict__ ftab, Layout lay, PairConsts pc, float *__restrict__ G_, float *__restrict__ A_,
            float *__restrict__ Pw_, float *__restrict__ R_, long long *trace) {
  using Cfg = PairCfg<L>;
  using Geo = typename Cfg::G;
  constexpr int N = Cfg::N, F = Cfg::F, T = Cfg::T, E = Cfg::E, PB = Cfg::PB;
  constexpr int THREADS = Cfg::THREADS;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float2 *tile = reinterpret_cast<float2 *>(smem_raw);                     // [F][PB], slot = (pl ^ s_swz(f)) & (PB-1)
  float2 *exch = reinterpret_cast<float2 *>(smem_raw);                     // [PB][BUF] once the tile is dead
  float *rowj = reinterpret_cast<float *>(smem_raw + Cfg::BUF_BYTES);      // [PB][FP]: 1/sqrt(S_jj[f]) of pair pl's j
  float *rs = reinterpret_cast<float *>(smem_raw + Cfg::OFF_RS);           // [2][PB]: 1/sqrt(L R_cc[0]) of i, j
  ushort2 *ij_s = reinterpret_cast<ushort2 *>(smem_raw + Cfg::OFF_IJ);     // [PB]
  int *pg_s = reinterpret_cast<int *>(smem_raw + Cfg::OFF_PG);             // [PB]
  uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw + Cfg::OFF_BAR);

  float *const G = G_, *const A = A_, *const Pw = Pw_, *const R = R_;
  const bool wantG = G, wantR = R;
  const int tid = threadIdx.x;
  const int64_t p0 = (int64_t)blockIdx.x * PB;

  // debug: globaltimer stamps of the CTA's phases (delta_debug_set_trace): trace[8192 + 8 blockIdx + k]
  auto stamp = [&](int k) {
    if (trace && tid == 0) {
      long long g;
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g));
      trace[8192 + 8 * (int64_t)blockIdx.x + k] = g;
    }
  };
  stamp(0);
  pdl_launch_dependents();
  if (tid < PB) {
    // all pairs: (i, j) of lexicographic pair p0 + tid;  pair list (f2): entry p0 + tid of the list, whose S values sit
    // at lexicographic index pg in the S layout
    ushort2 ij = make_ushort2(0, 1);
    if (p0 + tid < lay.Po) ij = list ? list[p0 + tid] : pair_of(p0 + tid, lay.C);
    ij_s[tid] = ij;
    pg_s[tid] = (int)ij.x * lay.C - ((int)ij.x * ((int)ij.x + 1)) / 2 + (int)ij.y - (int)ij.x - 1;
  }
  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(1));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  pdl_wait();  // S, rsq and the energy partials come from the preceding kernels; the outputs may still be read by a consumer
  stamp(1);
  __syncthreads();
  if (tid == 0) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"((uint32_t)((list ? 0 : Cfg::TILE_BYTES) + (wantG ? Cfg::ROWS_BYTES : 0))) : "memory");
    if (!list)
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(tile)),
                   "l"(S + (int64_t)blockIdx.x * F * PB), "r"((uint32_t)Cfg::TILE_BYTES), "r"(smem_u32(bar))
                   : "memory");
  }
  if (list) {  // gather the tile: slot sl of row f belongs to the CTA's pair pl = (sl ^ s_swz(f)) mod PB
    for (int idx = tid; idx < F * PB; idx += THREADS) {
      const int f = idx / PB, sw = s_swz(f);
      const int pg = pg_s[((idx % PB) ^ sw) & (PB - 1)];
      tile[idx] = __ldg(S + ((int64_t)(pg >> lay.pb_shift) * F + f) * PB + ((pg ^ sw) & (PB - 1)));
    }
  }
  if (tid < PB && wantG) {  // this pair's 1/sqrt(S_jj) row; a lane's complete_tx may precede lane 0's expect_tx: the
                            // transaction count is signed and the phase cannot complete before lane 0's arrival
    const ushort2 ij = ij_s[tid];
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(rowj + tid * Cfg::FP)),
                 "l"(Srsq + (int64_t)ij.y * Cfg::FP), "r"((uint32_t)(Cfg::FP * sizeof(float))), "r"(smem_u32(bar))
                 : "memory");
  }

  // rs[role][pl] = 1/sqrt(sum over all L bins of S_cc) = 1/sqrt(L R_cc[0]),  c = i (role 0) or j (role 1) of pair pl
  if (R && tid < 2 * PB) {
    const ushort2 ij = ij_s[tid % PB];
    const float *a = rpart + (int64_t)(tid / PB ? ij.y : ij.x) * rp_stride;
    float sum = 0.f;
    for (int k = 0; k < nrp; ++k) sum += __ldg(a + k);
    sum *= rscale;
    rs[tid] = sum > 0.f ? rsqrtf(sum) : 0.f;
  }
  __syncthreads();

  {  // the tile has landed?  (bounded: a faulted copy must trap, not hang the GPU)
    uint32_t ok = 0;
    long long t0 = 0;
    for (uint32_t spins = 0; !ok; ++spins) {
      asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                   : "=r"(ok) : "r"(smem_u32(bar)), "r"(0) : "memory");
      if (spins == 64) t0 = clock64();
      if (spins > 64 && (spins & 1023) == 0 && clock64() - t0 > 4000000000LL) __trap();
    }
  }

  stamp(2);  // tile landed
  const int pl = tid / T, gt = tid % T;
  const int64_t p = p0 + pl;
  const bool valid = p < lay.Po;
  const float2 wg = __ldg(tw + gt);  // e^{-2 pi i gt / L}

  // ---- pass 1: G, A, P ------------------------------------------------------------------------------------------
  // The store path is what binds this kernel (without its stores it runs in half the time), so pass 1 has its own
  // thread mapping: a thread owns 4 consecutive bins of one pair and stores float4; a warp covers 512 contiguous
  // bytes of one row.  Rows have F = N + 1 floats (F mod 4 = 1), so element (p, f) is 16-byte aligned iff
  // (p + f) mod 4 = 0: the groups of pair p start at f0 = (-p) mod 4; the f0 head and the 0..3 tail bins go scalar.
  if ((G || A || Pw) && p0 < lay.Po) {
    auto value = [&](float2 s, float g2, float &mag, float &coh, float &ang) {
      mag = sqrt_approx(fmaf(s.x, s.x, s.y * s.y));
      coh = mag * g2;
      ang = atan2_poly(s.y, s.x);
    };
    constexpr int NG = N / 4;  // group slots per pair
    const bool vec4 = (((reinterpret_cast<uintptr_t>(G) | reinterpret_cast<uintptr_t>(A) | reinterpret_cast<uintptr_t>(Pw)) & 15) == 0);
    if (vec4) {
      // R pairs are in flight per iteration; a thread keeps its group g and its pair slot qa, so with R a multiple of 4
      // the bins f, the tile rows and the alignment shift f0 do not depend on the iteration (p0 is a multiple of 4)
      constexpr int R = THREADS / NG, NIT = PB / R;
      static_assert(R >= 1 && (R & (R - 1)) == 0 && PB % R == 0, "pairs per iteration");
      const int g = tid % NG, qa = tid / NG;
      if constexpr (R % 4 == 0) {
        // Everything but the pair is the same in every iteration, so the bins, the four tile addresses (the pair offset
        // it R only flips slot bits: one XOR) and the base pointers are hoisted.  The G/A/P pass is bound by the
        // load/store unit's wavefronts, so the two 1/sqrt rows are read as aligned float4 (two loads cover the four
        // bins f0 + 4g .. + 3 of a group that starts f0 floats past a 16-byte boundary; f0 is warp-uniform), and the
        // row of channel i, shared by consecutive lexicographic pairs, is re-read only when i changes.
        const int f0 = (-qa) & 3, ng = (F - f0) >> 2, f = f0 + 4 * g;
        if (g < ng) {
          int tb[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) tb[k] = (f + k) * PB + ((qa ^ s_swz(f + k)) & (PB - 1));
          const int64_t at0 = (p0 + qa) * F + f;
          float *Pw0 = Pw ? Pw + at0 : nullptr, *G0 = G ? G + at0 : nullptr, *A0 = A ? A + at0 : nullptr;
          auto quad = [&](const float4 a, const float4 bq, float *r) {  // elements f0 .. f0 + 3 of (a, bq)
            switch (f0) {
              case 0: r[0] = a.x; r[1] = a.y; r[2] = a.z; r[3] = a.w; break;
              case 1: r[0] = a.y; r[1] = a.z; r[2] = a.w; r[3] = bq.x; break;
              case 2: r[0] = a.z; r[1] = a.w; r[2] = bq.x; r[3] = bq.y; break;
              default: r[0] = a.w; r[1] = bq.x; r[2] = bq.y; r[3] = bq.z; break;
            }
          };
          int icur = -1;
          float gi[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
          for (int it = 0; it < NIT; ++it) {
            const int ql = it * R + qa;
            if (p0 + ql >= lay.Po) continue;
            float g2[4] = {0.f, 0.f, 0.f, 0.f};
            if (wantG) {
              const int i = ij_s[ql].x;
              if (i != icur) {  // warp-uniform
                const float4 *src = reinterpret_cast<const float4 *>(Srsq + (int64_t)i * Cfg::FP + 4 * g);
                quad(__ldg(src), __ldg(src + 1), gi);
                icur = i;
              }
              const float4 *rowq = reinterpret_cast<const float4 *>(rowj + ql * Cfg::FP + 4 * g);
              float gj[4];
              quad(rowq[0], rowq[1], gj);
#pragma unroll
              for (int k = 0; k < 4; ++k) g2[k] = gi[k] * gj[k];
            }
            float2 sv[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) sv[k] = tile[tb[k] ^ (it * R)];
            float m[4], c[4], an[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) value(sv[k], g2[k], m[k], c[k], an[k]);
            if (GAPALL || Pw) ST4(Pw0 + it * R * F, make_float4(m[0], m[1], m[2], m[3]));
            if (GAPALL || G) ST4(G0 + it * R * F, make_float4(c[0], c[1], c[2], c[3]));
            if (GAPALL || A) ST4(A0 + it * R * F, make_float4(an[0], an[1], an[2], an[3]));
          }
        }
      } else {
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
          const int ql = (it * R) ^ qa;  // = it R + qa (qa < R, R a power of two)
          const int64_t q = p0 + ql;
          const int f0 = (-(qa + ((it * R) & 3))) & 3, ng = (F - f0) >> 2;
          if (q >= lay.Po || g >= ng) continue;
          const int f = f0 + 4 * g;
          const ushort2 qij = ij_s[ql];
          const float *qi = Srsq + (int64_t)qij.x * Cfg::FP + f, *qj = rowj + ql * Cfg::FP + f;
          float2 sv[4];
          float g2[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            sv[k] = tile[(f + k) * PB + (((qa ^ s_swz(f + k)) ^ (it * R)) & (PB - 1))];
            g2[k] = wantG ? __ldg(qi + k) * qj[k] : 0.f;
          }
          float m[4], c[4], an[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) value(sv[k], g2[k], m[k], c[k], an[k]);
          const int64_t at = q * F + f;
          if (GAPALL || Pw) ST4(Pw + at, make_float4(m[0], m[1], m[2], m[3]));
          if (GAPALL || G) ST4(G + at, make_float4(c[0], c[1], c[2], c[3]));
          if (GAPALL || A) ST4(A + at, make_float4(an[0], an[1], an[2], an[3]));
        }
      }
    }
    // scalar bins: the edges of the vector path (at most 6 per pair), or everything if the arrays are not 16-byte aligned
    const int per = vec4 ? 8 : F;
    for (int item = tid; item < PB * per; item += THREADS) {
      const int ql = item / per, e = item % per;
      const int64_t q = p0 + ql;
      if (q >= lay.Po) continue;
      int f = e;
      if (vec4) {
        const int f0 = (int)((-q) & 3), ng = (F - f0) >> 2;
        f = e < f0 ? e : f0 + 4 * ng + (e - f0);
        if (f >= F) continue;
      }
      const ushort2 qij = ij_s[ql];
      const float g2 = wantG ? __ldg(Srsq + (int64_t)qij.x * Cfg::FP + f) * rowj[ql * Cfg::FP + f] : 0.f;
      float m, c, an;
      value(tile[f * PB + ((ql ^ s_swz(f)) & (PB - 1))], g2, m, c, an);
      if (GAPALL || Pw) ST1(Pw + q * F + f, m);
      if (GAPALL || G) ST1(G + q * F + f, c);
      if (GAPALL || A) ST1(A + q * F + f, an);
    }
  }
  stamp(3);  // pass 1 done (thread 0's share)
  if (!wantR) return;

  // ---- pass 2: merge step of the inverse real transform (S read again from the tile; twice the merge of
  // irfft_merge, the factor 1/2 goes into the normalisation) ------------------------------------------------
  float2 v[E];
  const int pg = pl ^ s_swz(gt);
#pragma unroll
  for (int u = 0; u < E; ++u) {
    const int f = gt + T * u;
    const int fr = N - f;
    float2 sf = tile[f * PB + ((pg ^ s_swz(T * u)) & (PB - 1))];  // s_swz(gt | T u) = s_swz(gt) ^ s_swz(T u)
    float2 sr = tile[fr * PB + ((pl ^ s_swz(fr)) & (PB - 1))];
    if (u == 0 && gt == 0) { sf.y = 0.f; sr.y = 0.f; }  // Im S[0], Im S[N] do not enter the real transform
    const float2 w = cmul(wg, pc.wstep[u]);               // e^{-2 pi i f / L}; the inverse uses its conjugate
    v[u] = irfft_merge2(sf, sr, make_float2(w.x, -w.y));
  }
  stamp(4);
  __syncthreads();  // every S value is in registers: the tile becomes exchange space

  // ---- rho = irfft(S) / sqrt(R_ii[0] R_jj[0]) ----------------------------------------------------------------
  fft_inplace_g<Geo, true>(v, FftPadMap{exch + pl * Geo::BUF}, ftab, gt);  // z[n] = (x[2n], x[2n+1]) * N, n = gt + T u
  stamp(5);  // FFT done
  if (!valid) return;
  // rho = x / sqrt(R_ii[0] R_jj[0]),  x = z/N,  R_cc[0] = (sum over all L bins of S_cc)/L
  const float norm = rs[pl] * rs[PB + pl];  // 2 (L/N) x 1/2 (irfft_merge2)
  float *Rp = R + p * lay.nlags;
  if (FULL) {
    // lag m = xi for xi <= L/2 and xi - L for xi >= L/2; row position q = m + L/2
    const bool vec = (reinterpret_cast<uintptr_t>(Rp) & 7) == 0;  // q is even: float2 stores iff the row is 8-byte aligned
#pragma unroll
    for (int u = 0; u < E; ++u) {
      const int n = gt + T * u;
      const float a = v[u].x * norm, b = v[u].y * norm;
      const int q = (u < E / 2) ? 2 * n + N : 2 * n - N;
#ifdef DELTA_DBG_NOSTORE_R
      if (lay.Po < 0)
#endif
      if (vec) {
        ST2(Rp + q, make_float2(a, b));
      } else {
        ST1(Rp + q, a);
        ST1(Rp + q + 1, b);
      }
      if (u == E / 2 && gt == 0) ST1(Rp + L, a);  // xi = L/2 is lag -L/2 and lag +L/2
    }
  } else {
    const int M = lay.M;
#pragma unroll
    for (int u = 0; u < E; ++u) {
      const int n = gt + T * u;
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const int xi = 2 * n + h;
        const float val = (h ? v[u].y : v[u].x) * norm;
        if (xi <= M) Rp[xi + M] = val;
        if (xi >= L - M) Rp[xi - L + M] = val;
      }
    }
  }
  stamp(6);
}

// rsq[c][f] = 1/sqrt(S_cc[f]) (0 where S_cc[f] <= 0, reading R16) and
// rsum[c] = S_cc[0] + 2 sum_{0<f<N} S_cc[f] + S_cc[N] = sum over all L bins = L R_cc[0].  One warp per channel.
__global__ void __launch_bounds__(32) auto_prep_kernel(const float *__restrict__ Sauto, float *__restrict__ rsq,
                                                       float *__restrict__ rsum, int F, int Fp) {
  const int c = blockIdx.x, lane = threadIdx.x;
  float sum = 0.f;
  for (int f = lane; f < F; f += 32) {
    const float a = Sauto[(int64_t)c * F + f];
    rsq[(int64_t)c * Fp + f] = a > 0.f ? rsqrtf(a) : 0.f;
    sum = fmaf((f == 0 || f == F - 1) ? 1.f : 2.f, a, sum);
  }
  for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
  if (lane == 0) rsum[c] = sum;
}

// acc = wa acc + wn x (f2: accumulation of spectra over chunks); wa == 0 does not read acc
__global__ void __launch_bounds__(256) axpby_kernel(float *__restrict__ acc, const float *__restrict__ x, int64_t n, float wa,
                                                    float wn, int vec) {
  const int64_t stride = (int64_t)gridDim.x * 256;
  if (vec) {
    const int64_t n4 = n >> 2;
    float4 *a4 = reinterpret_cast<float4 *>(acc);
    const float4 *x4 = reinterpret_cast<const float4 *>(x);
    for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n4; i += stride) {
      const float4 v = x4[i];
      float4 o = make_float4(wn * v.x, wn * v.y, wn * v.z, wn * v.w);
      if (wa != 0.f) {
        const float4 a = a4[i];
        o = make_float4(fmaf(wa, a.x, o.x), fmaf(wa, a.y, o.y), fmaf(wa, a.z, o.z), fmaf(wa, a.w, o.w));
      }
      a4[i] = o;
    }
    for (int64_t i = (n4 << 2) + (int64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += stride)
      acc[i] = (wa != 0.f ? wa * acc[i] : 0.f) + wn * x[i];
  } else {
    for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < n; i += stride)
      acc[i] = (wa != 0.f ? wa * acc[i] : 0.f) + wn * x[i];
  }
}

// test accessor: S layout -> complex64 [P][F], lexicographic pairs
__global__ void __launch_bounds__(256) s_unpack_kernel(const float2 *__restrict__ S, Layout lay, float2 *__restrict__ out) {
  const int64_t total = lay.P * lay.F;
  for (int64_t idx = (int64_t)blockIdx.x * 256 + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * 256) {
    const int f = (int)(idx % lay.F);
    const int64_t p = idx / lay.F;
    out[idx] = S[((p >> lay.pb_shift) * lay.F + f) * lay.PB + ((p ^ s_swz(f)) & (lay.PB - 1))];
  }
}

// ------------------------------------------------------------------------------------------
template <int L>
static int launch_pair_L(delta_plan *p, const float *d_S, const float *d_rsq, const float *rpart, int nrp, int rp_stride,
                         float rscale, float *d_G, float *d_A, float *d_P, float *d_R, cudaStream_t st) {
  using Cfg = PairCfg<L>;
  const Layout &lay = p->lay;
  if (lay.Poblk == 0 || lay.Po == 0) return DELTA_OK;
  const ushort2 *list = p->cfg.n_pairs > 0 ? p->d_pairs() : nullptr;
  PairConsts pc;
  for (int u = 0; u < 16; ++u) pc.wstep[u] = p->h_wstep[u];
  const bool full = lay.M == L / 2;
#define DELTA_PAIR_LAUNCH(FULL_, GAPALL_)                                                                           \
  do {                                                                                                              \
    int rc = opt_in_smem(pair_kernel<L, FULL_, GAPALL_>, Cfg::SMEM);                                                \
    if (rc) return rc;                                                                                              \
    LaunchCfg lc(dim3((unsigned)lay.Poblk), dim3(Cfg::THREADS), Cfg::SMEM, st, p->use_pdl);                          \
    DELTA_CUDA_CHECK(cudaLaunchKernelEx(&lc.cfg, pair_kernel<L, FULL_, GAPALL_>, reinterpret_cast<const float2 *>(d_S), \
                                        d_rsq, rpart, nrp, rp_stride, rscale, list, p->d_tw(), p->d_ftab2(), lay, pc, \
                                        d_G, d_A, d_P, d_R, p->d_trace));                                                       \
  } while (0)
  const bool gapall = d_G && d_A && d_P;
  if (full && gapall) DELTA_PAIR_LAUNCH(true, true);
  else if (full) DELTA_PAIR_LAUNCH(true, false);
  else if (gapall) DELTA_PAIR_LAUNCH(false, true);
  else DELTA_PAIR_LAUNCH(false, false);
#undef DELTA_PAIR_LAUNCH
  p->launches++;
  DELTA_CUDA_CHECK(cudaGetLastError());
  return DELTA_OK;
}

int launch_pair(delta_plan *p, const float *d_S, const float *d_rsq, const float *rpart, int nrp, int rp_stride, float rscale,
                float *d_G, float *d_A, float *d_P, float *d_R, cudaStream_t st) {
#define CALL(LL) launch_pair_L<LL>(p, d_S, d_rsq, rpart, nrp, rp_stride, rscale, d_G, d_A, d_P, d_R, st)
  DELTA_SWITCH_L(p->lay.L, CALL)
#undef CALL
}

int launch_auto_prep(delta_plan *p, const float *d_auto, float *d_rsq, float *d_rsum, cudaStream_t st) {
  auto_prep_kernel<<<(unsigned)p->lay.C, 32, 0, st>>>(d_auto, d_rsq, d_rsum, p->lay.F, p->lay.Fp);
  p->launches++;
  DELTA_CUDA_CHECK(cudaGetLastError());
  return DELTA_OK;
}

int launch_axpby(delta_plan *p, float *acc, const float *x, int64_t n, float wa, float wn, cudaStream_t st) {
  if (n <= 0) return DELTA_OK;
  const int vec = ((reinterpret_cast<uintptr_t>(acc) | reinterpret_cast<uintptr_t>(x)) & 15) == 0;
  const int64_t want = ((vec ? n / 4 : n) + 255) / 256;
  const int64_t cap = (int64_t)p->num_sms * 16;
  axpby_kernel<<<(unsigned)(want < 1 ? 1 : (want < cap ? want : cap)), 256, 0, st>>>(acc, x, n, wa, wn, vec);
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
