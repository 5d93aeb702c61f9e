// CUDA-core kernels of libdelta_b200 (sm_100a):
//   contract_fp32_kernel  a2+a3 Eq. (1a) on the FP32 FMA pipe
//   pair_epilogue_kernel  a4+a5 Eq. (1b), (1c), |1a|, (1d) per pair
#include <cuda_fp16.h>

#include "delta_internal.h"
#include "fft.cuh"

namespace delta {

// ------------------------------------------------------------------------------------------
template <int L>
struct FftCfg {
  static constexpr int N = L / 2;
  static constexpr int GROUP = (N / 8 < 32) ? 32 : ((N / 8 > kThreads) ? kThreads : N / 8);
  static constexpr int CONC = kThreads / GROUP;  // transforms in flight per CTA
  static constexpr int FS = N + 4;               // staging row stride (floats); == 4 mod 8
};

// ------------------------------------------------------------------------------------------
// a2+a3, Eq. (1a) on the FP32 pipe.  grid = (upper-triangular 64x64 channel tiles, F).
// S_ij = scale * sum_k (a_i + i b_i)(a_j - i b_j) = scale * [ (a_i a_j + b_i b_j) + i (b_i a_j - a_i b_j) ]
__global__ void __launch_bounds__(kThreads)
contract_fp32_kernel(const float *__restrict__ X, Layout lay, float scale, float2 *__restrict__ S,
                     float *__restrict__ Sauto) {
  constexpr int KT = 32;  // segments per shared-memory stage
  __shared__ __align__(16) float As[2][KT][kPairTile];
  __shared__ __align__(16) float Bs[2][KT][kPairTile];
  const int f = blockIdx.y;
  int bi = 0, rem = blockIdx.x;
  const int nb = (lay.C + kPairTile - 1) / kPairTile;
  while (rem >= nb - bi) { rem -= nb - bi; ++bi; }
  const int bj = bi + rem;
  const int tid = threadIdx.x, ty = tid >> 4, tx = tid & 15;
  const float *Xf = X + (int64_t)f * lay.x_elems_per_f;

  float acc_re[4][4], acc_im[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) acc_re[a][b] = acc_im[a][b] = 0.f;

  for (int k0 = 0; k0 < lay.Kp; k0 += KT) {
    for (int idx = tid; idx < 1024; idx += kThreads) {
      const int h = idx & 1, row = (idx >> 1) & 63, kcl = (idx >> 7) & 3, part = idx >> 9;
      const int kc = k0 / kSegBlock + kcl;
      float4 va = make_float4(0.f, 0.f, 0.f, 0.f), vb = va;
      if (kc < lay.Kc) {
        const int64_t o = ((int64_t)part * lay.Kc + kc) * lay.Cp;
        va = __ldg(reinterpret_cast<const float4 *>(Xf + (o + bi * kPairTile + row) * kSegBlock + 4 * h));
        vb = __ldg(reinterpret_cast<const float4 *>(Xf + (o + bj * kPairTile + row) * kSegBlock + 4 * h));
      }
      const int kl = kcl * kSegBlock + 4 * h;
      As[part][kl + 0][row] = va.x; As[part][kl + 1][row] = va.y; As[part][kl + 2][row] = va.z; As[part][kl + 3][row] = va.w;
      Bs[part][kl + 0][row] = vb.x; Bs[part][kl + 1][row] = vb.y; Bs[part][kl + 2][row] = vb.z; Bs[part][kl + 3][row] = vb.w;
    }
    __syncthreads();
#pragma unroll 8
    for (int kk = 0; kk < KT; ++kk) {
      const float4 ar4 = *reinterpret_cast<const float4 *>(&As[0][kk][4 * ty]);
      const float4 ai4 = *reinterpret_cast<const float4 *>(&As[1][kk][4 * ty]);
      const float4 br4 = *reinterpret_cast<const float4 *>(&Bs[0][kk][4 * tx]);
      const float4 bi4 = *reinterpret_cast<const float4 *>(&Bs[1][kk][4 * tx]);
      const float ar[4] = {ar4.x, ar4.y, ar4.z, ar4.w}, ai[4] = {ai4.x, ai4.y, ai4.z, ai4.w};
      const float br[4] = {br4.x, br4.y, br4.z, br4.w}, bim[4] = {bi4.x, bi4.y, bi4.z, bi4.w};
#pragma unroll
      for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
          acc_re[a][b] = fmaf(ar[a], br[b], acc_re[a][b]);
          acc_re[a][b] = fmaf(ai[a], bim[b], acc_re[a][b]);
          acc_im[a][b] = fmaf(ai[a], br[b], acc_im[a][b]);
          acc_im[a][b] = fmaf(-ar[a], bim[b], acc_im[a][b]);
        }
    }
    __syncthreads();
  }

  const int C = lay.C;
#pragma unroll
  for (int a = 0; a < 4; ++a) {
    const int i = bi * kPairTile + 4 * ty + a;
    if (i >= C) continue;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      const int j = bj * kPairTile + 4 * tx + b;
      if (j >= C) continue;
      if (i < j) {
        if (S) S[(int64_t)f * lay.Ppad + (j * (j - 1)) / 2 + i] = make_float2(acc_re[a][b] * scale, acc_im[a][b] * scale);
      } else if (i == j) {
        if (Sauto) Sauto[(int64_t)i * lay.F + f] = acc_re[a][b] * scale;
      }
    }
  }
}

// ------------------------------------------------------------------------------------------
// a4+a5: all per-pair quantities from S[f][p].  One CTA owns PB consecutive pairs for all bins,
// so each output array receives one contiguous run per CTA.
template <int L>
struct PairCfg {
  static constexpr int PB = (L <= 512) ? 32 : 16384 / L;
};

template <int GROUP>
__device__ __forceinline__ void group_reduce2(float &a, float &b, float *red, int g, int gt) {
  for (int o = 16; o > 0; o >>= 1) {
    a += __shfl_xor_sync(0xffffffffu, a, o);
    b += __shfl_xor_sync(0xffffffffu, b, o);
  }
  if (GROUP > 32) {
    constexpr int W = GROUP / 32;
    const int w = gt >> 5;
    __syncthreads();
    if ((gt & 31) == 0) {
      red[(g * W + w) * 2 + 0] = a;
      red[(g * W + w) * 2 + 1] = b;
    }
    __syncthreads();
    a = 0.f; b = 0.f;
    for (int q = 0; q < W; ++q) {
      a += red[(g * W + q) * 2 + 0];
      b += red[(g * W + q) * 2 + 1];
    }
  }
}

template <int L>
__global__ void __launch_bounds__(kThreads)
pair_epilogue_kernel(const float2 *__restrict__ S, const float *__restrict__ Sauto,
                     const ushort2 *__restrict__ pairs, const float2 *__restrict__ tw, Layout lay,
                     float *__restrict__ G, float *__restrict__ A, float *__restrict__ Pw, float *__restrict__ R) {
  using Cfg = FftCfg<L>;
  constexpr int N = Cfg::N, F = N + 1, GROUP = Cfg::GROUP, CONC = Cfg::CONC;
  constexpr int PB = PairCfg<L>::PB, ROUNDS = PB / CONC, TS = PB + 1;
  static_assert(PB % CONC == 0, "pair block must be a multiple of the concurrent transforms");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2 *tile = reinterpret_cast<float2 *>(smem_raw);  // [F][TS]
  float2 *bufA = tile + F * TS;
  float2 *bufB = bufA + CONC * N;
  float *red = reinterpret_cast<float *>(bufB + CONC * N);  // [8][2]

  const int tid = threadIdx.x, g = tid / GROUP, gt = tid % GROUP;
  const int64_t p0 = (int64_t)blockIdx.x * PB;
  for (int idx = tid; idx < F * PB; idx += kThreads) {
    const int f = idx / PB, pl = idx - f * PB;
    tile[f * TS + pl] = __ldg(S + (int64_t)f * lay.Ppad + p0 + pl);
  }
  __syncthreads();

#pragma unroll 1
  for (int r = 0; r < ROUNDS; ++r) {
    const int pl = r * CONC + g;
    const int64_t ps = p0 + pl;  // position in S order (column-major upper triangle)
    const bool valid = ps < lay.P;
    const ushort2 ij = pairs[valid ? ps : 0];
    // output row: lexicographic pair index (reading R9)
    const int64_t p = (int64_t)ij.x * lay.C - ((int64_t)ij.x * (ij.x + 1)) / 2 + (ij.y - ij.x - 1);
    const float *ai = Sauto + (int64_t)ij.x * F, *aj = Sauto + (int64_t)ij.y * F;
    float si = 0.f, sj = 0.f;
    for (int f = gt; f < F; f += GROUP) {
      const float2 s = tile[f * TS + pl];
      const float a_i = __ldg(ai + f), a_j = __ldg(aj + f);
      const float wt = (f == 0 || f == N) ? 1.f : 2.f;
      si = fmaf(wt, a_i, si);
      sj = fmaf(wt, a_j, sj);
      if (valid) {
        const float mag = sqrtf(fmaf(s.x, s.x, s.y * s.y));
        const int64_t o = p * F + f;
        if (Pw) Pw[o] = mag;
        if (G) G[o] = (a_i > 0.f && a_j > 0.f) ? mag * rsqrtf(a_i) * rsqrtf(a_j) : 0.f;
        if (A) A[o] = atan2f(s.y, s.x);
      }
    }
    if (R) {
      group_reduce2<GROUP>(si, sj, red, g, gt);
      float2 *a = bufA + g * N, *b = bufB + g * N;
      for (int f = gt; f < N; f += GROUP) {
        float2 sf = tile[f * TS + pl], sr = tile[(N - f) * TS + pl];
        if (f == 0) { sf.y = 0.f; sr.y = 0.f; }
        float2 w = __ldg(tw + f);
        w.y = -w.y;  // e^{+2 pi i f / L}
        a[f] = irfft_merge(sf, sr, w);
      }
      group_sync<GROUP>();
      const float *xs = reinterpret_cast<const float *>(fft_stockham<N, GROUP, true>(a, b, tw, gt));
      // rho = x / sqrt(R_ii[0] R_jj[0]),  x = z/N,  R_cc[0] = (sum over all L bins of S_cc)/L
      const float norm = (si > 0.f && sj > 0.f) ? 2.f * rsqrtf(si) * rsqrtf(sj) : 0.f;
      if (valid) {
        float *Rp = R + p * lay.nlags;
        for (int q = gt; q < lay.nlags; q += GROUP) Rp[q] = xs[(q - lay.M) & (L - 1)] * norm;
      }
      group_sync<GROUP>();
    }
  }
}

// ------------------------------------------------------------------------------------------
// launchers
int launch_contract_fp32(delta_plan *p, const void *d_X, float *d_S, float *d_auto, cudaStream_t st) {
  const Layout &lay = p->lay;
  const int nb = (lay.C + kPairTile - 1) / kPairTile;
  dim3 grid(nb * (nb + 1) / 2, lay.F);
  contract_fp32_kernel<<<grid, kThreads, 0, st>>>(reinterpret_cast<const float *>(d_X), lay, p->s2 / (float)lay.K,
                                                  reinterpret_cast<float2 *>(d_S), d_auto);
  p->launches++;
  DELTA_CUDA_CHECK(cudaGetLastError());
  return DELTA_OK;
}

template <int L>
static int launch_pair_epilogue_L(delta_plan *p, const float *d_S, const float *d_auto, float *d_G, float *d_A,
                                  float *d_P, float *d_R, cudaStream_t st) {
  using Cfg = FftCfg<L>;
  constexpr int PB = PairCfg<L>::PB;
  const Layout &lay = p->lay;
  const size_t smem = (size_t)(Cfg::N + 1) * (PB + 1) * sizeof(float2) + (size_t)2 * Cfg::CONC * Cfg::N * sizeof(float2) +
                      64 * sizeof(float);
  int rc = opt_in_smem(pair_epilogue_kernel<L>, smem);
  if (rc) return rc;
  const int blocks = (int)((lay.P + PB - 1) / PB);
  if (blocks == 0) return DELTA_OK;
  pair_epilogue_kernel<L><<<blocks, kThreads, smem, st>>>(reinterpret_cast<const float2 *>(d_S), d_auto, p->d_pairs(),
                                                          p->d_tw(), lay, d_G, d_A, d_P, d_R);
  p->launches++;
  DELTA_CUDA_CHECK(cudaGetLastError());
  return DELTA_OK;
}

int launch_pair_epilogue(delta_plan *p, const float *d_S, const float *d_auto, float *d_G, float *d_A, float *d_P,
                         float *d_R, cudaStream_t st) {
#define CALL(LL) launch_pair_epilogue_L<LL>(p, d_S, d_auto, d_G, d_A, d_P, d_R, st)
  DELTA_SWITCH_L(p->lay.L, CALL)
#undef CALL
}

}  // namespace delta
