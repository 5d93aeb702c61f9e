// a2+a3 on the 5th-generation tensor cores: Eq. (1a), as a batched Hermitian rank-K
// contraction  S_f = s^2/K * X_f X_f^H  with tcgen05.mma (kind::f16) and TMEM accumulators.
//
//   X_f = A + iB (C x K, A = Re, B = Im).   Re S = A A^T + B B^T,   Im S = B A^T - A B^T.
//   Operands are split fp16:  x * s_c = hi + lo  (s_c a per-channel power of two, |x s_c| <= 2^14), and every
//   real product is formed as hi*hi + hi*lo + lo*hi (the dropped lo*lo term is 2^-22 relative): 3 MMAs.
//   The -A B^T term uses the negate-A bit of the instruction descriptor, so one copy of the operands in
//   shared memory serves all twelve MMAs of a K=16 step.
//
// Operand layout (written by stft_kernel, see delta_internal.h): half X[f][plane][kc][Cp][8], plane = hi_re,
// hi_im, lo_re, lo_im.  For one K=16 step a plane's [2][Cp][8] block is exactly the canonical K-major
// SWIZZLE_NONE shared-memory image of a Cp x 16 operand (core matrix = 8 rows x 16 B, SBO = 128 B between
// 8-row groups, LBO = Cp*16 B between the two 8-wide K halves), so it is brought in with plain
// cp.async.bulk copies (no tensor map) and any 8-aligned row range is addressed by moving the descriptor's
// start address.
//
// Roles (one CTA per SM, persistent over (bin, group) items): warp 8 lane 0 = bulk-copy producer,
// warp 9 lane 0 = MMA issuer, warps 0-7 = epilogue (TMEM -> registers -> scale -> coalesced S stores).
#include <cuda_fp16.h>

#include "delta_internal.h"

namespace delta {

namespace {

constexpr int kTcThreads = 320;
constexpr int kEpiWarps = 8;

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *b, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t *b) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *b, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
// Bounded wait: a pipeline bug must not hang the GPU; after ~2 s the kernel traps.
__device__ __forceinline__ void mbar_wait(uint64_t *b, uint32_t parity) {
  const uint32_t addr = smem_u32(b);
  long long t0 = 0;
  for (uint32_t spins = 0;; ++spins) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(addr), "r"(parity)
        : "memory");
    if (ok) return;
    if (spins == 64) t0 = clock64();
    if (spins > 64 && (spins & 1023) == 0 && clock64() - t0 > 4000000000LL) __trap();
  }
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ uint64_t make_sdesc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFF) << 16) |
         ((uint64_t)((sbo_bytes >> 4) & 0x3FFF) << 32) | ((uint64_t)1 << 46);
}
// kind::f16 instruction descriptor: D = F32, A = B = F16, both K-major, M = 128.
__device__ __forceinline__ uint32_t make_idesc(int N, int neg_a) {
  return (1u << 4) | ((uint32_t)neg_a << 13) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
}
__device__ __forceinline__ void mma_f16(uint32_t taddr, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(taddr),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void mma_commit(uint64_t *bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float *v) {
  uint32_t r[16];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
        "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr));
#pragma unroll
  for (int q = 0; q < 16; ++q) v[q] = __uint_as_float(r[q]);
}

}  // namespace

struct TcTile {
  int row0;     // first channel of the 128-row A operand (multiple of 64)
  int col0;     // first channel of the N-row B operand
  int N;        // multiple of 16, <= 256
  int lane_lo;  // rows below row0 + lane_lo are owned by another tile (0 or 64)
  int tm_re, tm_im;  // TMEM column offsets of the two accumulators
};
struct TcParams {
  int ngroups;
  int ntiles[kTcMaxGroups];
  TcTile tiles[kTcMaxGroups][kTcMaxTiles];
  int nstage, ksteps;
  uint32_t stage_bytes, plane_bytes;  // per stage: 4 planes of 2*Cp*16 bytes
  int64_t plane_elems;                // halves between planes in global memory: Kc*Cp*8
  int64_t kstep_elems;                // halves per K=16 step inside a plane: 2*Cp*8
};

__global__ void __launch_bounds__(kTcThreads, 1)
contract_tc_kernel(const __half *__restrict__ X, Layout lay, TcParams prm, float scale, const float *__restrict__ chscale,
                   float2 *__restrict__ S, float *__restrict__ Sauto) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  unsigned char *stages = smem_raw;
  float *inv_scale = reinterpret_cast<float *>(stages + (size_t)prm.nstage * prm.stage_bytes);  // [Cp]
  uint64_t *full_bar = reinterpret_cast<uint64_t *>(inv_scale + lay.Cp);
  uint64_t *empty_bar = full_bar + prm.nstage;
  uint64_t *tmem_full = empty_bar + prm.nstage;
  uint64_t *tmem_empty = tmem_full + 1;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tmem_empty + 1);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nitems = lay.F * prm.ngroups;

  for (int c = tid; c < lay.Cp; c += kTcThreads) inv_scale[c] = (c < lay.C) ? 1.f / chscale[c] : 0.f;
  if (tid == 0) {
    for (int s = 0; s < prm.nstage; ++s) {
      mbar_init(full_bar + s, 1);
      mbar_init(empty_bar + s, 1);
    }
    mbar_init(tmem_full, 1);
    mbar_init(tmem_empty, kEpiWarps);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem_base = *tmem_slot;

  if (warp == kEpiWarps) {
    // ===== producer: stream the four operand planes of every K=16 step =====
    if (lane == 0) {
      uint32_t step = 0;
      for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
        const int f = item / prm.ngroups;
        const __half *Xf = X + (int64_t)f * lay.x_elems_per_f;
        for (int ks = 0; ks < prm.ksteps; ++ks, ++step) {
          const int s = step % prm.nstage;
          const uint32_t use = step / prm.nstage;
          if (use > 0) mbar_wait(empty_bar + s, (use - 1) & 1);
          mbar_expect_tx(full_bar + s, prm.stage_bytes);
          unsigned char *dst = stages + (size_t)s * prm.stage_bytes;
#pragma unroll
          for (int pl = 0; pl < 4; ++pl)
            bulk_g2s(dst + (size_t)pl * prm.plane_bytes, Xf + pl * prm.plane_elems + ks * prm.kstep_elems, prm.plane_bytes,
                     full_bar + s);
        }
      }
    }
  } else if (warp == kEpiWarps + 1) {
    // ===== MMA issuer =====
    if (lane == 0) {
      const uint32_t lbo = (uint32_t)lay.Cp * 16u, sbo = 128u;
      uint32_t step = 0, it = 0;
      for (int item = blockIdx.x; item < nitems; item += gridDim.x, ++it) {
        const int g = item % prm.ngroups;
        if (it > 0) mbar_wait(tmem_empty, (it - 1) & 1);  // epilogue has drained the accumulators
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        for (int ks = 0; ks < prm.ksteps; ++ks, ++step) {
          const int s = step % prm.nstage;
          mbar_wait(full_bar + s, (step / prm.nstage) & 1);
          asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
          const uint32_t sb = smem_u32(stages + (size_t)s * prm.stage_bytes);
          const uint32_t p_hr = sb, p_hi = sb + prm.plane_bytes, p_lr = sb + 2 * prm.plane_bytes, p_li = sb + 3 * prm.plane_bytes;
          for (int t = 0; t < prm.ntiles[g]; ++t) {
            const TcTile tl = prm.tiles[g][t];
            const uint32_t ao = (uint32_t)(tl.row0 / 8) * 128u, bo = (uint32_t)(tl.col0 / 8) * 128u;
            const uint32_t id = make_idesc(tl.N, 0), idn = make_idesc(tl.N, 1);
            const uint32_t acc = ks > 0 ? 1u : 0u;
            const uint32_t d_re = tmem_base + (uint32_t)tl.tm_re, d_im = tmem_base + (uint32_t)tl.tm_im;
#define SD(plane, off) make_sdesc((plane) + (off), lbo, sbo)
            // Re S += A A^T + B B^T
            mma_f16(d_re, SD(p_hr, ao), SD(p_hr, bo), id, acc);
            mma_f16(d_re, SD(p_hr, ao), SD(p_lr, bo), id, 1u);
            mma_f16(d_re, SD(p_lr, ao), SD(p_hr, bo), id, 1u);
            mma_f16(d_re, SD(p_hi, ao), SD(p_hi, bo), id, 1u);
            mma_f16(d_re, SD(p_hi, ao), SD(p_li, bo), id, 1u);
            mma_f16(d_re, SD(p_li, ao), SD(p_hi, bo), id, 1u);
            // Im S += B A^T - A B^T
            mma_f16(d_im, SD(p_hi, ao), SD(p_hr, bo), id, acc);
            mma_f16(d_im, SD(p_hi, ao), SD(p_lr, bo), id, 1u);
            mma_f16(d_im, SD(p_li, ao), SD(p_hr, bo), id, 1u);
            mma_f16(d_im, SD(p_hr, ao), SD(p_hi, bo), idn, 1u);
            mma_f16(d_im, SD(p_hr, ao), SD(p_li, bo), idn, 1u);
            mma_f16(d_im, SD(p_lr, ao), SD(p_hi, bo), idn, 1u);
#undef SD
          }
          mma_commit(empty_bar + s);  // stage reusable once these MMAs have read it
        }
        mma_commit(tmem_full);  // accumulators of this item complete
      }
    }
  } else {
    // ===== epilogue warps: warp = quadrant (lanes of TMEM) + 4 * column half =====
    const int q = warp & 3, h = warp >> 2;
    const int C = lay.C;
    uint32_t it = 0;
    for (int item = blockIdx.x; item < nitems; item += gridDim.x, ++it) {
      const int f = item / prm.ngroups, g = item % prm.ngroups;
      mbar_wait(tmem_full, it & 1);
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      float2 *Sf = S ? S + (int64_t)f * lay.Ppad : nullptr;
      for (int t = 0; t < prm.ntiles[g]; ++t) {
        const TcTile tl = prm.tiles[g][t];
        if (32 * q < tl.lane_lo) continue;
        const int i = tl.row0 + 32 * q + lane;
        const float si = scale * inv_scale[i];
        const int nhalf = tl.N / 2;
        const uint32_t lane_addr = (uint32_t)(32 * q) << 16;
        for (int c0 = h * nhalf; c0 < (h + 1) * nhalf; c0 += 16) {
          float re[16], im[16];
          tmem_ld16(tmem_base + lane_addr + (uint32_t)(tl.tm_re + c0), re);
          tmem_ld16(tmem_base + lane_addr + (uint32_t)(tl.tm_im + c0), im);
          asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
          const int jbase = tl.col0 + c0;
          if (jbase + 15 < i || i >= C) continue;   // whole chunk below the diagonal for this lane
#pragma unroll
          for (int u = 0; u < 16; ++u) {
            const int j = jbase + u;
            if (j >= C) break;
            if (i < j) {
              if (Sf) {
                const float sc = si * inv_scale[j];
                Sf[(j * (j - 1)) / 2 + i] = make_float2(re[u] * sc, im[u] * sc);
              }
            } else if (i == j && Sauto) {
              Sauto[(int64_t)i * lay.F + f] = re[u] * si * inv_scale[j];
            }
          }
        }
      }
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      __syncwarp();
      if (lane == 0) mbar_arrive(tmem_empty);
    }
  }

  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512));
}

// ------------------------------------------------------------------------------------------
bool tc_plan_tiles(int Cp, TcHostPlan *out) {
  // rows are covered by M = 128 tiles over pairs of 64-channel blocks; each tile's columns start at its
  // own first row (upper triangle) and are cut into slabs of <= 256; tiles are packed into groups whose
  // accumulators (Re + Im = 2N columns) fit the 512 TMEM columns.
  struct T { int row0, col0, N, lane_lo; };
  T list[64];
  int n = 0;
  const int nb = Cp / 64;
  for (int m = 0; 2 * m + 1 < nb; ++m)
    for (int c = 128 * m; c < Cp; c += 256) {
      if (n >= 64) return false;
      list[n++] = {128 * m, c, (Cp - c) < 256 ? (Cp - c) : 256, 0};
    }
  if (nb & 1) {
    if (n >= 64) return false;
    list[n++] = {64 * (nb - 2), 64 * (nb - 1), 64, 64};
  }
  // first-fit decreasing by N
  for (int a = 0; a < n; ++a)
    for (int b = a + 1; b < n; ++b)
      if (list[b].N > list[a].N) { T t = list[a]; list[a] = list[b]; list[b] = t; }
  int used[kTcMaxGroups];
  out->ngroups = 0;
  for (int g = 0; g < kTcMaxGroups; ++g) { used[g] = 0; out->ntiles[g] = 0; }
  for (int a = 0; a < n; ++a) {
    int g = 0;
    for (; g < kTcMaxGroups; ++g)
      if (used[g] + 2 * list[a].N <= 512 && out->ntiles[g] < kTcMaxTiles) break;
    if (g == kTcMaxGroups) return false;
    int *slot = &out->ntiles[g];
    out->tiles[g][*slot][0] = list[a].row0;
    out->tiles[g][*slot][1] = list[a].col0;
    out->tiles[g][*slot][2] = list[a].N;
    out->tiles[g][*slot][3] = list[a].lane_lo;
    out->tiles[g][*slot][4] = used[g];
    out->tiles[g][*slot][5] = used[g] + list[a].N;
    used[g] += 2 * list[a].N;
    ++*slot;
    if (g + 1 > out->ngroups) out->ngroups = g + 1;
  }
  return true;
}

int launch_contract_tc(delta_plan *p, const void *d_X, float *d_S, float *d_auto, cudaStream_t st) {
  const Layout &lay = p->lay;
  TcParams prm;
  memset(&prm, 0, sizeof(prm));
  prm.ngroups = p->tc.ngroups;
  for (int g = 0; g < kTcMaxGroups; ++g) {
    prm.ntiles[g] = p->tc.ntiles[g];
    for (int t = 0; t < kTcMaxTiles; ++t) {
      const int *s = p->tc.tiles[g][t];
      prm.tiles[g][t] = {s[0], s[1], s[2], s[3], s[4], s[5]};
    }
  }
  prm.ksteps = lay.Kp / 16;
  prm.plane_bytes = (uint32_t)lay.Cp * 32u;  // [2][Cp][8] halves
  prm.stage_bytes = 4u * prm.plane_bytes;
  prm.plane_elems = (int64_t)lay.Kc * lay.Cp * kSegBlock;
  prm.kstep_elems = (int64_t)2 * lay.Cp * kSegBlock;
  const size_t fixed = (size_t)lay.Cp * sizeof(float) + 64 * sizeof(uint64_t) + 64;
  int nstage = (int)((200 * 1024 - fixed) / prm.stage_bytes);
  if (nstage > 8) nstage = 8;
  if (nstage < 2) return DELTA_ERR_UNSUPPORTED;
  prm.nstage = nstage;
  size_t smem = (size_t)nstage * prm.stage_bytes + fixed;
  if (smem < 120 * 1024) smem = 120 * 1024;  // one CTA per SM: each CTA allocates all 512 TMEM columns
  cudaError_t e = cudaFuncSetAttribute(contract_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) { set_cuda_error(e); return DELTA_ERR_CUDA; }
  const int nitems = lay.F * prm.ngroups;
  const int grid = nitems < p->num_sms ? nitems : p->num_sms;
  contract_tc_kernel<<<grid, kTcThreads, smem, st>>>(reinterpret_cast<const __half *>(d_X), lay, prm, p->s2 / (float)lay.K,
                                                      p->d_chscale(), reinterpret_cast<float2 *>(d_S), d_auto);
  p->launches++;
  DELTA_CUDA_CHECK(cudaGetLastError());
  return DELTA_OK;
}

}  // namespace delta
