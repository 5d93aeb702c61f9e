// a2+a3 on the FP32 FMA pipe: Eq. (1a).  The CUDA-core version of the contraction, kept
// selectable (DELTA_CONTRACT_FP32) as the A/B partner of the tensor-core kernel and for shapes the
// tensor-core tile plan does not cover.
#include "delta_internal.h"

namespace delta {

// grid = (upper-triangular 64x64 channel tiles, F).
// S_ij = scale * sum_k (a_i + i b_i)(a_j - i b_j) = scale * [ (a_i a_j + b_i b_j) + i (b_i a_j - a_i b_j) ]
__global__ void __launch_bounds__(kThreads)
contract_fp32_kernel(const float *__restrict__ X, Layout lay, float scale, float2 *__restrict__ S,
                     float *__restrict__ Sauto, float *__restrict__ Srsq, const float *__restrict__ wpart, float rscale,
                     float *__restrict__ rnorm) {
  constexpr int KT = 32;  // segments per shared-memory stage
  __shared__ __align__(16) float As[2][KT][kPairTile];
  __shared__ __align__(16) float Bs[2][KT][kPairTile];
  const int f = blockIdx.y;
  if (rnorm && blockIdx.x == 0 && blockIdx.y == 0) {
    // 1/sqrt(L R_cc[0]) for the normalisation of rho, from the windowed signal energy (Parseval, pin P4): fixed order
    for (int c = threadIdx.x; c < lay.C; c += kThreads) {
      float sum = 0.f;
      for (int k = 0; k < lay.nkb; ++k) sum += wpart[(int64_t)c * lay.nkb + k];
      sum *= rscale;
      rnorm[c] = sum > 0.f ? rsqrtf(sum) : 0.f;
    }
  }
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

  const int C = lay.C, pb_mask = lay.PB - 1;
#pragma unroll
  for (int a = 0; a < 4; ++a) {
    const int i = bi * kPairTile + 4 * ty + a;
    if (i >= C) continue;
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      const int j = bj * kPairTile + 4 * tx + b;
      if (j >= C) continue;
      if (i < j) {
        if (S) {
          // lexicographic pair index, block-major, slot swizzled by bin (Layout in delta_internal.h)
          const int64_t p = (int64_t)i * C - ((int64_t)i * (i + 1)) / 2 + (j - i - 1);
          S[((p >> lay.pb_shift) * lay.F + f) * lay.PB + ((p ^ s_swz(f)) & pb_mask)] =
              make_float2(acc_re[a][b] * scale, acc_im[a][b] * scale);
        }
      } else if (i == j) {
        const float v = acc_re[a][b] * scale;
        if (Sauto) Sauto[(int64_t)i * lay.F + f] = v;
        if (Srsq) store_rsq4(Srsq, lay, i, f, v > 0.f ? rsqrtf(v) : 0.f);
      }
    }
  }
}

int launch_contract_fp32(delta_plan *p, const void *d_X, float *d_S, float *d_auto, float *d_rsq, float *d_rnorm, float rscale,
                         cudaStream_t st) {
  const Layout &lay = p->lay;
  const int nb = (lay.C + kPairTile - 1) / kPairTile;
  dim3 grid(nb * (nb + 1) / 2, lay.F);
  contract_fp32_kernel<<<grid, kThreads, 0, st>>>(reinterpret_cast<const float *>(d_X), lay, p->s2 / (float)lay.K,
                                                  reinterpret_cast<float2 *>(d_S), d_auto, d_rsq, (const float *)p->d_wpart(), rscale,
                                                  d_rnorm);
  p->launches++;
  DELTA_CUDA_CHECK(cudaGetLastError());
  return DELTA_OK;
}

}  // namespace delta
