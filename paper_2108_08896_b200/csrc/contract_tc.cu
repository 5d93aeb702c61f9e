// a2+a3 on the 5th-generation tensor cores: Eq. (1a), as a batched Hermitian rank-K
// contraction  S_f = s^2/K * X_f X_f^H  with tcgen05.mma (kind::f16) and TMEM accumulators.
//
//   X_f = A + iB (C x K, A = Re, B = Im).   Re S = A A^T + B B^T,   Im S_ij = B_i A_j - A_i B_j.
//   Operands are split fp16:  x * s_c = hi + lo  (s_c a per-channel power of two, |x s_c| <= 2^14), and every
//   real product is formed as hi*hi + hi*lo + lo*hi (the dropped lo*lo term is 2^-22 relative): 3 MMAs.
//   The subtracted term uses the negate-A bit of the instruction descriptor, so one copy of the operands in
//   shared memory serves all twelve MMAs of a K=16 step.
//
// Operand layout (written by stft_kernel, see delta_internal.h): half X[f][plane][kc][Cp][8], plane = hi_re,
// hi_im, lo_re, lo_im.  For one K=16 step a plane's [2][Cp][8] block is exactly the canonical K-major
// SWIZZLE_NONE shared-memory image of a Cp x 16 operand (core matrix = 8 rows x 16 B, SBO = 128 B between
// 8-row groups, LBO = Cp*16 B between the two 8-wide K halves), so it is brought in with plain
// cp.async.bulk copies (no tensor map) and any 8-aligned row range is addressed by moving the descriptor's
// start address.
//
// Accumulator tiles ("units"): TMEM lanes = channel j (128 rows of the A operand), TMEM columns = channel i
// (N <= 128 rows of the B operand), Re in columns [tm, tm+N), Im in [tm+N, tm+2N).  Only i < j is kept, so the
// units cover the lower triangle; a lane (fixed j) then walks consecutive lexicographic pairs when the
// epilogue fixes i and lets the 32 lanes of a warp store: S leaves the SM in 256-byte runs.
//
// Roles (one CTA per SM, persistent over (bin, group) items): warps 0-15 = epilogue (4 TMEM lane quadrants x 4 column
// slices: TMEM -> registers -> scale -> S stores), warp 16 = bulk-copy producer, warp 17 = MMA issuer (both loops are
// warp-uniform, one elected lane issues).  Every unit has
// its own TMEM region and full/empty mbarrier pair, so the epilogue of unit u overlaps the MMAs of the
// following units (and, when all K steps of a bin fit in the operand ring, of the next bin: "unit-major").
#include <cuda_fp16.h>

#include "delta_internal.h"

namespace delta {

namespace {

constexpr int kColSplit = 4;              // column slices of a unit, one per epilogue warp of a lane quadrant
constexpr int kEpiWarps = 4 * kColSplit;
constexpr int kTcThreads = 32 * (kEpiWarps + 2);

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
// predicated 8-byte global store (no branch: see the epilogue)
__device__ __forceinline__ void st_pred_f2(float2 *p, float a, float b, bool pred) {
  asm volatile("{\n\t.reg .pred q;\n\tsetp.ne.b32 q, %3, 0;\n\t@q st.global.v2.f32 [%0], {%1, %2};\n\t}" ::"l"(p), "f"(a), "f"(b),
               "r"((int)pred)
               : "memory");
}
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
  return pred != 0;
}
__device__ __forceinline__ void fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }

}  // namespace

struct TcUnit {
  int row0;              // first channel of the 128-row A operand = channel of TMEM lane 0 (multiple of 8)
  int lane_lo, lane_hi;  // lanes [lane_lo, lane_hi) are owned by this unit (multiples of 32)
  int col0, N;           // B operand rows = channels [col0, col0 + N), N a multiple of 64 up to 256
  int tm;                // TMEM column of Re; Im follows at tm + N
};
struct TcParams {
  int ngroups;
  int nunits[kTcMaxGroups];
  TcUnit units[kTcMaxGroups][kTcMaxUnits];
  int nstage, ksteps, unit_major;
  uint32_t stage_bytes, plane_bytes;  // per stage: 4 planes of 2*Cp*16 bytes
  int64_t plane_elems;                // halves between planes in global memory: Kc*Cp*8
  int64_t kstep_elems;                // halves per K=16 step inside a plane: 2*Cp*8
};

// trace[role * 512 + n] = clock64 stamps of CTA 0 (role 0 producer, 1 MMA issuer, 2 epilogue warp 0)
#define TC_TRACE(role, slot)                                                        \
  do {                                                                              \
    if (TRACE && blockIdx.x == 0 && (slot) < 512) trace[(role) * 512 + (slot)] = clock64(); \
  } while (0)

template <bool TRACE>
__global__ void __launch_bounds__(kTcThreads, 1)
contract_tc_kernel(const __half *__restrict__ X, Layout lay, TcParams prm, float scale, float2 *__restrict__ S,
                   float *__restrict__ Sauto, float *__restrict__ Srsq, const float *__restrict__ wpart, float rscale,
                   float *__restrict__ rnorm, long long *trace) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  unsigned char *stages = smem_raw;
  // itab[c] = {rowbase(c) = c C - c(c+1)/2 - c - 1 (int bits), 1/chscale[c]}: pair index p(i, j) = rowbase(i) + j
  float2 *itab = reinterpret_cast<float2 *>(stages + (size_t)prm.nstage * prm.stage_bytes);  // [Cp]
  uint64_t *full_bar = reinterpret_cast<uint64_t *>(itab + lay.Cp);
  uint64_t *empty_bar = full_bar + prm.nstage;
  uint64_t *tfull = empty_bar + prm.nstage;  // [kTcMaxUnits]
  uint64_t *tempty = tfull + kTcMaxUnits;    // [kTcMaxUnits]
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(tempty + kTcMaxUnits);

  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);  // provably warp-uniform
  const int nitems = lay.F * prm.ngroups;
  if (tid == 0) TC_TRACE(3, 0);
  if (TRACE && tid == 0) { long long g; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g)); trace[5 * 512 + 2 * blockIdx.x] = g; }

  if (tid == 0) {
    for (int s = 0; s < prm.nstage; ++s) {
      mbar_init(full_bar + s, 1);
      mbar_init(empty_bar + s, 1);
    }
    for (int u = 0; u < kTcMaxUnits; ++u) {
      mbar_init(tfull + u, 1);
      mbar_init(tempty + u, kEpiWarps);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  pdl_launch_dependents();
  pdl_wait();  // X (with its scales) comes from the STFT kernel; S, Sauto, Srsq of the previous chunk are still being read
  // the per-channel fp16 scales travel with the operands: C floats behind the planes of the X buffer
  const float *chscale = reinterpret_cast<const float *>(reinterpret_cast<const char *>(X) + lay.x_scale_off);
  if (rnorm && blockIdx.x == gridDim.x - 1) {
    // 1/sqrt(L R_cc[0]) for the normalisation of rho, from the windowed signal energy (Parseval, pin P4): fixed order
    for (int c = tid; c < lay.C; c += kTcThreads) {
      float sum = 0.f;
      for (int k = 0; k < lay.nkb; ++k) sum += wpart[(int64_t)c * lay.nkb + k];
      sum *= rscale;
      rnorm[c] = sum > 0.f ? rsqrtf(sum) : 0.f;
    }
  }
  for (int c = tid; c < lay.Cp; c += kTcThreads)
    itab[c] = make_float2(__int_as_float(c * lay.C - (c * (c + 1)) / 2 - c - 1), (c < lay.C) ? 1.f / chscale[c] : 0.f);
  fence_before();
  __syncthreads();
  fence_after();
  const uint32_t tmem_base = *tmem_slot;
  if (tid == 0) TC_TRACE(3, 1);

  if (warp == kEpiWarps) {
    // ===== producer: stream the four operand planes of every K=16 step =====
    // The whole warp walks the loop (warp-uniform values live in uniform registers, which is what the bulk-copy
    // and MMA instructions take); one elected lane issues.
    // stage index and use count advance incrementally: no division by the (run-time) stage count in the loop
    uint32_t s = 0, pass = 0, kidx = 0;  // pass = completed trips around the stage ring
    int f = blockIdx.x / prm.ngroups, g = blockIdx.x % prm.ngroups;
    const int fstep = gridDim.x / prm.ngroups, gstep = gridDim.x % prm.ngroups;
    for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
      const __half *Xf = X + (int64_t)f * lay.x_elems_per_f;
      if (prm.unit_major == 3) {
        // mode 3 (the K steps of a bin do not fit in the ring, many channels): every unit streams its own operands, and only those: per
        // plane and K half the 128 rows of A (channels row0 ..) and the N rows of B (channels col0 ..), packed as
        // [plane][K half][128 + N rows][8].  (Whole-Cp stages made every unit pull all channels through the crossbar.)
        for (int u = 0; u < prm.nunits[g]; ++u) {
          const TcUnit un = prm.units[g][u];
          const uint32_t R = 128u + (uint32_t)un.N;
          for (int ks = 0; ks < prm.ksteps; ++ks, ++kidx) {
            if (lay.jitter_mask & kJitTcProducer) __nanosleep((unsigned)lay.jitter_ns);  // (test hook)
            if (pass) mbar_wait(empty_bar + s, (pass - 1) & 1u);
            if (elect_one()) {
              mbar_expect_tx(full_bar + s, 8u * R * 16u);
              unsigned char *dst = stages + (size_t)s * prm.stage_bytes;
#pragma unroll
              for (int pk = 0; pk < 8; ++pk) {  // plane pk / 2, K half pk % 2
                const __half *src = Xf + (pk >> 1) * prm.plane_elems + ks * prm.kstep_elems + (int64_t)(pk & 1) * lay.Cp * kSegBlock;
                bulk_g2s(dst + (size_t)pk * R * 16u, src + (int64_t)un.row0 * kSegBlock, 128u * 16u, full_bar + s);
                bulk_g2s(dst + (size_t)pk * R * 16u + 128u * 16u, src + (int64_t)un.col0 * kSegBlock, (uint32_t)un.N * 16u, full_bar + s);
              }
            }
            __syncwarp();
            if (++s == (uint32_t)prm.nstage) { s = 0; ++pass; }
          }
        }
      } else {
        // mode 2 (the K steps do not fit in the ring, few channels): every unit streams the bin's operands again (L2 hits)
        const int reps = prm.unit_major == 2 ? prm.nunits[g] : 1;
        for (int kk = 0; kk < reps * prm.ksteps; ++kk, ++kidx) {
          const int ks = kk % prm.ksteps;
          if (lay.jitter_mask & kJitTcProducer) __nanosleep((unsigned)lay.jitter_ns);  // (test hook)
          if (pass) mbar_wait(empty_bar + s, (pass - 1) & 1u);
          if (elect_one()) {
            mbar_expect_tx(full_bar + s, prm.stage_bytes);
            unsigned char *dst = stages + (size_t)s * prm.stage_bytes;
#pragma unroll
            for (int pl = 0; pl < 4; ++pl)
              bulk_g2s(dst + (size_t)pl * prm.plane_bytes, Xf + pl * prm.plane_elems + ks * prm.kstep_elems, prm.plane_bytes,
                       full_bar + s);
            TC_TRACE(0, kidx);
          }
          __syncwarp();
          if (++s == (uint32_t)prm.nstage) { s = 0; ++pass; }
        }
      }
      f += fstep; g += gstep;
      if (g >= prm.ngroups) { g -= prm.ngroups; ++f; }
    }
  } else if (warp == kEpiWarps + 1) {
    // ===== MMA issuer =====
    const uint32_t lbo = (uint32_t)lay.Cp * 16u, sbo = 128u;
    uint32_t tr = 0;
    uint32_t used = 0, par = 0;  // per-unit bits: unit has been used; parity of its use count
    // descriptor = dbase + (shared address >> 4): all addresses are 16-byte aligned and below 256 KB
    const uint64_t dbase = make_sdesc(0, lbo, sbo);
    const uint32_t st16 = smem_u32(stages) >> 4, stage16 = prm.stage_bytes >> 4, plane16 = prm.plane_bytes >> 4;

    // the twelve MMAs of one (unit, K step): Re += A_j A_i + B_j B_i;  Im += A_j B_i - B_j A_i  (rows j, cols i)
    auto issue = [&](uint64_t dbase, uint32_t plane16, uint32_t ao16, uint32_t bo16, uint32_t id, uint32_t idn, uint32_t d_re,
                     uint32_t d_im, uint32_t s, uint32_t acc) {
      const uint64_t sb = dbase + (st16 + s * stage16);
      const uint64_t a_hr = sb + ao16, a_hi = a_hr + plane16, a_lr = a_hi + plane16, a_li = a_lr + plane16;
      const uint64_t b_hr = sb + bo16, b_hi = b_hr + plane16, b_lr = b_hi + plane16, b_li = b_lr + plane16;
      if (elect_one()) {
        mma_f16(d_re, a_hr, b_hr, id, acc);
        mma_f16(d_im, a_hr, b_hi, id, acc);
        mma_f16(d_re, a_hr, b_lr, id, 1u);
        mma_f16(d_im, a_hr, b_li, id, 1u);
        mma_f16(d_re, a_lr, b_hr, id, 1u);
        mma_f16(d_im, a_lr, b_hi, id, 1u);
        mma_f16(d_re, a_hi, b_hi, id, 1u);
        mma_f16(d_im, a_hi, b_hr, idn, 1u);
        mma_f16(d_re, a_hi, b_li, id, 1u);
        mma_f16(d_im, a_hi, b_lr, idn, 1u);
        mma_f16(d_re, a_li, b_hi, id, 1u);
        mma_f16(d_im, a_li, b_hr, idn, 1u);
      }
      __syncwarp();
    };
    // Before the first MMA of a unit its TMEM columns must have been read out.  tempty[u] says that for the last unit of
    // index u.  But groups lay their units out differently (a 64-wide unit takes 128 columns, a 128-wide one 256), so the
    // columns of unit u may also belong to a unit of HIGHER index of the CTA's previous item, which nothing above waits
    // for: then the highest such index is awaited too.  That is enough: every epilogue warp reads the units in order, so
    // a completed phase of tempty[m] means that all units before it (of that item and of the items before) are read out;
    // indices below u have been awaited by this item's earlier units, and an index above u has not been used again yet,
    // so its parity bit still stands for the previous item's phase.  (Found in round 2: 576 channels have such
    // transitions, e.g. (64, 128, 64) -> (128, 128); it is also why 256-wide units "failed parity" on config 5 in round 1.)
    int g = blockIdx.x % prm.ngroups, gp = -1;  // group of this item, of the previous item
    auto wait_unit_free = [&](int u, const TcUnit &un) {
      if (lay.jitter_mask & kJitTcMma) __nanosleep((unsigned)lay.jitter_ns);  // (test hook)
      if ((used >> u) & 1u) {  // epilogue has drained the previous use
        mbar_wait(tempty + u, ((par >> u) & 1u) ^ 1u);
        fence_after();
      }
      if (gp >= 0 && gp != g) {
        int need = -1;
        for (int up = u + 1; up < prm.nunits[gp]; ++up) {
          const int otm = prm.units[gp][up].tm, oend = otm + 2 * prm.units[gp][up].N;
          if (otm < un.tm + 2 * un.N && oend > un.tm) need = up;
        }
        if (need >= 0) {
          mbar_wait(tempty + need, ((par >> need) & 1u) ^ 1u);
          fence_after();
        }
      }
    };
    auto unit_done = [&](int u) {
      if (elect_one()) mma_commit(tfull + u);
      __syncwarp();
      used |= 1u << u;
      par ^= 1u << u;
    };

    uint32_t s0 = 0, pass0 = 0;  // stage and ring pass of the item's first K step
    const int gstep = gridDim.x % prm.ngroups;
    for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
      const int nu = prm.nunits[g];
      if (prm.unit_major >= 2) {
        // unit after unit, each with its own pass over the K steps: the epilogue of unit u overlaps the MMAs of unit u+1
        uint32_t s = s0, pass = pass0;
        for (int u = 0; u < nu; ++u) {
          const TcUnit un = prm.units[g][u];
          // mode 3, packed stage of this unit: A rows at 0, B rows at 128, R = 128 + N rows per K half
          const bool packed = prm.unit_major == 3;
          const uint32_t R = 128u + (uint32_t)un.N;
          const uint64_t dbase_u = packed ? make_sdesc(0, R * 16u, sbo) : dbase;
          const uint32_t plane16_u = packed ? 2u * R : plane16;
          const uint32_t ao16 = packed ? 0u : (uint32_t)(un.row0 / 8) * 8u, bo16 = packed ? 128u : (uint32_t)(un.col0 / 8) * 8u;
          const uint32_t id = make_idesc(un.N, 0), idn = make_idesc(un.N, 1);
          const uint32_t d_re = tmem_base + (uint32_t)un.tm, d_im = d_re + (uint32_t)un.N;
          wait_unit_free(u, un);
          for (int ks = 0; ks < prm.ksteps; ++ks) {
            mbar_wait(full_bar + s, pass & 1u);
            fence_after();
            issue(dbase_u, plane16_u, ao16, bo16, id, idn, d_re, d_im, s, ks > 0 ? 1u : 0u);
            if (elect_one()) mma_commit(empty_bar + s);
            __syncwarp();
            if (++s == (uint32_t)prm.nstage) { s = 0; ++pass; }
          }
          unit_done(u);
        }
        s0 = s; pass0 = pass;
      } else {
        for (int u = 0; u < nu; ++u) {
          const TcUnit un = prm.units[g][u];
          const uint32_t ao16 = (uint32_t)(un.row0 / 8) * 8u, bo16 = (uint32_t)(un.col0 / 8) * 8u;
          const uint32_t id = make_idesc(un.N, 0), idn = make_idesc(un.N, 1);
          const uint32_t d_re = tmem_base + (uint32_t)un.tm, d_im = d_re + (uint32_t)un.N;
          wait_unit_free(u, un);
          uint32_t s = s0, pass = pass0;
          for (int ks = 0; ks < prm.ksteps; ++ks) {
            if (u == 0) {
              mbar_wait(full_bar + s, pass & 1u);
              fence_after();
              if (lane == 0) TC_TRACE(4, tr);
            }
            issue(dbase, plane16, ao16, bo16, id, idn, d_re, d_im, s, ks > 0 ? 1u : 0u);
            if (u == nu - 1) {  // stage reusable once every unit has read it
              if (elect_one()) mma_commit(empty_bar + s);
              __syncwarp();
            }
            if (++s == (uint32_t)prm.nstage) { s = 0; ++pass; }
          }
          unit_done(u);
          if (lane == 0) { TC_TRACE(1, tr); } ++tr;
          if (u == nu - 1) { s0 = s; pass0 = pass; }
        }
      }
      gp = g;
      g += gstep;
      if (g >= prm.ngroups) g -= prm.ngroups;
    }
  } else {
    // ===== epilogue warps: warp = lane quadrant of TMEM + 4 * column slice =====
    // Lane = channel j, TMEM column = channel i.  For a fixed i the 32 lanes of a warp hold 32 consecutive
    // lexicographic pairs p = rowbase(i) + j, so every store instruction writes two or three full 128-byte
    // lines of S.  The loop body is branch-free (predicated store) so the 16 elements of a chunk interleave.
    const int q = warp & 3, h = warp >> 2;
    const int C = lay.C, F = lay.F;
    const int pb_mask = lay.PB - 1;
    const int blk_stride = F * lay.PB;  // float2 elements between pair blocks
    uint32_t par = 0, tr = 0;  // per-unit parity of the use count
    int f = blockIdx.x / prm.ngroups, g = blockIdx.x % prm.ngroups;
    const int fstep = gridDim.x / prm.ngroups, gstep = gridDim.x % prm.ngroups;
    for (int item = blockIdx.x; item < nitems; item += gridDim.x, f += fstep + (g + gstep >= prm.ngroups), g = (g + gstep) % prm.ngroups) {
      const int nu = prm.nunits[g];
      const int fx = s_swz(f) & pb_mask;
      float2 *Sf = S + (int64_t)f * lay.PB;
      for (int u = 0; u < nu; ++u) {
        const TcUnit un = prm.units[g][u];
        mbar_wait(tfull + u, (par >> u) & 1u);
        par ^= 1u << u;
        fence_after();
        if (warp == 0) { TC_TRACE(2, tr); ++tr; }
        // (test hook: a slow epilogue makes a too-early reuse of its TMEM columns by the next item show every time)
        if (((lay.jitter_mask & kJitTcEpiLate) && u > 0) || ((lay.jitter_mask & kJitTcEpiSkew) && (warp & 1)))
          __nanosleep((unsigned)lay.jitter_ns);
        if (32 * q >= un.lane_lo && 32 * q < un.lane_hi) {
          const int jw0 = un.row0 + 32 * q, j = jw0 + lane;
          const bool jok = j < C;
          const float sj = scale * itab[j].y;
          const int ncols = un.N / kColSplit;
          const uint32_t lane_addr = (uint32_t)(32 * q) << 16;
          for (int c0 = h * ncols; c0 < (h + 1) * ncols; c0 += 16) {
            const int ibase = un.col0 + c0;
            if (ibase > jw0 + 31) continue;  // i > j for every lane of this warp
            float re[16], im[16];
            tmem_ld16(tmem_base + lane_addr + (uint32_t)(un.tm + c0), re);
            tmem_ld16(tmem_base + lane_addr + (uint32_t)(un.tm + un.N + c0), im);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (S) {
              // All 16 table reads, then all 16 addresses, then 16 predicated stores: the stores are inline PTX so
              // that the compiler cannot turn the predicate into a branch around each element (it did, and every
              // element then waited for its own shared-memory read: 2,000 cycles per 16 columns).
              float2 t[16];
#pragma unroll
              for (int e = 0; e < 16; ++e) t[e] = itab[ibase + e];  // {rowbase(i) as int bits, 1/scale_i}
#pragma unroll
              for (int e = 0; e < 16; ++e) {
                const int p = __float_as_int(t[e].x) + j;  // lexicographic pair index of (i, j)
                const float sc = sj * t[e].y;
                const int off = (p >> lay.pb_shift) * blk_stride + ((p ^ fx) & pb_mask);
                st_pred_f2(Sf + off, re[e] * sc, im[e] * sc, (ibase + e < j) && jok);
              }
            }
            if (ibase + 15 >= jw0) {  // this chunk crosses the diagonal: autospectrum of channel j
              float a = 0.f;
#pragma unroll
              for (int e = 0; e < 16; ++e) a = (ibase + e == j) ? re[e] : a;
              if (j >= ibase && j < ibase + 16 && jok) {
                a *= sj * itab[j].y;
                if (Sauto) Sauto[(int64_t)j * F + f] = a;
                if (Srsq) store_rsq4(Srsq, lay, j, f, a > 0.f ? rsqrtf(a) : 0.f);
              }
            }
          }
        }
        fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(tempty + u);
        if (warp == 0) { TC_TRACE(2, tr); ++tr; }
      }
    }
  }

  fence_before();
  __syncthreads();
  if (tid == 0) TC_TRACE(3, 2);
  if (TRACE && tid == 0) { long long g; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g)); trace[5 * 512 + 2 * blockIdx.x + 1] = g; }
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512));
}

// ------------------------------------------------------------------------------------------
// Host: cover the lower triangle (i < j) and the diagonal with units of 128 lanes (j) x N <= 128 columns (i),
// then pack the units into groups whose accumulators (Re + Im = 2N columns each) fit the 512 TMEM columns.
bool tc_plan_tiles(int Cp, TcHostPlan *out) {
  struct U { int row0, lane_lo, lane_hi, col0, N; };
  U list[kTcMaxGroups * kTcMaxUnits];
  int n = 0;
  auto add_row_tile = [&](int r0, int lane_hi, int col_end) {
    constexpr int kMaxN = 128;  // widest accumulator unit (wider units: less tensor time, but their epilogue overlaps less)
    for (int c = 0, N = 0; c < col_end; c += N) {
      if (n >= kTcMaxGroups * kTcMaxUnits) return false;
      N = (col_end - c) < kMaxN ? (col_end - c) : kMaxN;
      int lane_lo = c > r0 ? ((c - r0) & ~31) : 0;  // lanes below have j < col0: nothing to keep
      list[n++] = {r0, lane_lo, lane_hi, c, N};
    }
    return true;
  };
  if (Cp < 128 || (Cp & 63) != 0) return false;
  for (int r0 = Cp - 128; r0 >= 0; r0 -= 128)
    if (!add_row_tile(r0, 128, r0 + 128)) return false;
  if ((Cp & 127) == 64 && !add_row_tile(0, 64, 64)) return false;

  int used[kTcMaxGroups];
  out->ngroups = 0;
  for (int g = 0; g < kTcMaxGroups; ++g) { used[g] = 0; out->nunits[g] = 0; }
  for (int a = 0; a < n; ++a) {
    int g = 0;
    for (; g < kTcMaxGroups; ++g)
      if (used[g] + 2 * list[a].N <= 512 && out->nunits[g] < kTcMaxUnits) break;
    if (g == kTcMaxGroups) return false;
    int *u = out->units[g][out->nunits[g]++];
    u[0] = list[a].row0; u[1] = list[a].lane_lo; u[2] = list[a].lane_hi;
    u[3] = list[a].col0; u[4] = list[a].N; u[5] = used[g];
    used[g] += 2 * list[a].N;
    if (g + 1 > out->ngroups) out->ngroups = g + 1;
  }
  return true;
}

int launch_contract_tc(delta_plan *p, const void *d_X, float *d_S, float *d_auto, float *d_rsq, float *d_rnorm, float rscale,
                       cudaStream_t st) {
  const Layout &lay = p->lay;
  TcParams prm;
  memset(&prm, 0, sizeof(prm));
  prm.ngroups = p->tc.ngroups;
  for (int g = 0; g < kTcMaxGroups; ++g) {
    prm.nunits[g] = p->tc.nunits[g];
    for (int u = 0; u < kTcMaxUnits; ++u) {
      const int *s = p->tc.units[g][u];
      prm.units[g][u] = {s[0], s[1], s[2], s[3], s[4], s[5]};
    }
  }
  prm.ksteps = lay.Kp / 16;
  prm.plane_bytes = (uint32_t)lay.Cp * 32u;  // [2][Cp][8] halves
  prm.stage_bytes = 4u * prm.plane_bytes;
  prm.plane_elems = (int64_t)lay.Kc * lay.Cp * kSegBlock;
  prm.kstep_elems = (int64_t)2 * lay.Cp * kSegBlock;
  const size_t fixed = (size_t)lay.Cp * sizeof(float2) + 64 * sizeof(uint64_t) + 64;
  int nstage = (int)((200 * 1024 - fixed) / prm.stage_bytes);
  if (nstage > 8) nstage = 8;
  // 1: all K steps of a bin stay in the ring and are shared by its units;  2: every unit streams the bin's operands again;
  // 3: every unit streams its own 128 + N <= 256 operand rows, packed (less than all channels from 320 channels on: at 192
  //    the packed stages carry MORE rows, 84.9 vs 82.9 us at config 3; at 384 / 576 channels 222 vs 261 and 115 vs 125 us)
  // (K-step-major order, all units advancing together, was measured slower: their epilogues cannot overlap the MMAs)
  prm.unit_major = (nstage >= 2 && 2 * prm.ksteps <= nstage) ? 1 : (lay.Cp > 256 ? 3 : 2);
  if (prm.unit_major == 3) {  // [4 planes][2 K halves][256 rows][8 halves]
    prm.stage_bytes = 8u * 256u * 16u;
    nstage = (int)((200 * 1024 - fixed) / prm.stage_bytes);
    if (nstage > 6) nstage = 6;
  }
  if (nstage < 2) return DELTA_ERR_UNSUPPORTED;
  prm.nstage = nstage;
  size_t smem = (size_t)nstage * prm.stage_bytes + fixed;
  if (smem < 120 * 1024) smem = 120 * 1024;  // one CTA per SM: each CTA allocates all 512 TMEM columns
  const int nitems = lay.F * prm.ngroups;
  const int grid = nitems < p->num_sms ? nitems : p->num_sms;
  const float scale = p->s2 / (float)lay.K;
  if (p->d_trace) {
    int rc = opt_in_smem(contract_tc_kernel<true>, smem);
    if (rc) return rc;
    LaunchCfg lc(dim3(grid), dim3(kTcThreads), smem, st, p->use_pdl);
    DELTA_CUDA_CHECK(cudaLaunchKernelEx(&lc.cfg, contract_tc_kernel<true>, reinterpret_cast<const __half *>(d_X), lay, prm, scale,
                                        reinterpret_cast<float2 *>(d_S), d_auto, d_rsq, (const float *)p->d_wpart(), rscale,
                                        d_rnorm, p->d_trace));
  } else {
    int rc = opt_in_smem(contract_tc_kernel<false>, smem);
    if (rc) return rc;
    LaunchCfg lc(dim3(grid), dim3(kTcThreads), smem, st, p->use_pdl);
    DELTA_CUDA_CHECK(cudaLaunchKernelEx(&lc.cfg, contract_tc_kernel<false>, reinterpret_cast<const __half *>(d_X), lay, prm, scale,
                                        reinterpret_cast<float2 *>(d_S), d_auto, d_rsq, (const float *)p->d_wpart(), rscale,
                                        d_rnorm, (long long *)nullptr));
  }
  p->launches++;
  DELTA_CUDA_CHECK(cudaGetLastError());
  return DELTA_OK;
}

}  // namespace delta
