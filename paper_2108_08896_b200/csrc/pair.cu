// a4 + a5 of the hot path: everything that is per channel pair.
//   pair_kernel       Eq. (1b) coherence, Eq. (1c) cross-phase, |Eq. (1a)| cross-power
//                     Eq. (1d) cross-correlation = inverse real FFT of S_ij, normalised   (R12)
//   auto_prep_kernel  1/sqrt(S_cc[f]) from caller-supplied autospectra (staged calls only)
//   s_unpack_kernel   test accessor: S layout -> complex64 [P][F]
//
// pair_kernel is persistent, one CTA per SM.  A tile = PB consecutive (lexicographic) pairs = one contiguous [F][PB] block
// of S and one contiguous run of rows in each output array.  A producer warp keeps a ring of NSLOT tile slots full (one
// cp.async.bulk copy per tile, one per 1/sqrt(S_jj) row, and the pairs' channels and rho normalisations) while NTEAM
// teams of PB x T threads work on NTEAM tiles; the only CTA-wide synchronisation is the full / empty mbarrier pair of
// each slot.  Every pair has a group of T = N/E threads (for L <= 1024 inside one warp, so warps run free of each other
// and their store-bound and arithmetic-bound phases overlap on the SM):
//   pass 1  a thread owns 4 consecutive bins per step: |S| (cross-power), |S|/sqrt(S_ii S_jj), atan2; float4 stores
//   pass 2  thread gt owns bins f = gt + T u (u < E), the register layout the inverse FFT of fft_reg.cuh starts from:
//           merge step of the inverse real transform, register FFT exchanging through the pair's own column of the
//           tile (private padded buffers for the long transforms), rho stored from registers as float2.
#include "delta_internal.h"
#include "fft_reg.cuh"

namespace delta {

namespace {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

struct PairConsts {
  float2 wstep[16];  // e^{-2 pi i T u / L}
};

constexpr size_t kSmemPerSm = 227 * 1024;

template <int L>
struct PairCfg {
  static constexpr int N = L / 2, F = N + 1;
  using G = FftGeom<N, 0>;
  static constexpr int T = G::T, E = G::E;
  static constexpr int PB = pair_block(L);
  static constexpr int FP = (F + 3) & ~3;  // pitch of the rsq table
  static constexpr int TTHREADS = PB * T;  // threads of a team: one group of T per pair of a tile
  static constexpr int TW = TTHREADS / 32; // warps of a team
  // The inverse transform of a pair exchanges through the pair's own (by then dead) column of the tile where the tile has
  // 16 pairs per row (FftTileMap); the narrower tiles of the long transforms use private padded buffers, and their
  // 1/sqrt(S_jj) rows come from global memory instead of the slot.
  static constexpr bool IN_TILE = PB == 16;
  static constexpr bool ROWS = IN_TILE;
  static constexpr size_t TILE_BYTES = (size_t)F * PB * sizeof(float2);
  // per slot, behind the tile: [rows: float [PB][FP]]  ij ushort2[PB], pg int[PB] (lexicographic index), rs float[2][PB]
  static constexpr size_t OFF_ROWS = TILE_BYTES;
  static constexpr size_t ROW_BYTES = (size_t)FP * sizeof(float);
  static constexpr size_t OFF_IJ = OFF_ROWS + (ROWS ? PB * ROW_BYTES : 0), OFF_PG = OFF_IJ + PB * 4, OFF_RS = OFF_PG + PB * 4;
  static constexpr size_t SLOT_BYTES = (OFF_RS + 2 * PB * 4 + 127) & ~(size_t)127;
  static constexpr size_t FTAB_BYTES = (((size_t)(G::TABLE > 0 ? G::TABLE : 1) * sizeof(float2)) + 15) & ~(size_t)15;
  static constexpr size_t EXCH_BYTES = IN_TILE ? 0 : (size_t)PB * G::BUF * sizeof(float2);  // per team
  // One CTA per SM: NTEAM teams work on NTEAM tiles while a producer warp fills the remaining slot(s) of the ring.
  static constexpr size_t FIXED = FTAB_BYTES + 256;
  static constexpr int MAX_TEAMS = 768 / TTHREADS < 8 ? (768 / TTHREADS < 1 ? 1 : 768 / TTHREADS) : 8;  // 24 warps: 80 registers each
  static constexpr int FIT = (int)((kSmemPerSm - FIXED - EXCH_BYTES) / SLOT_BYTES);  // slots if there is one team
  static constexpr int NTEAM = IN_TILE ? (FIT - 1 < 1 ? 1 : (FIT - 1 > MAX_TEAMS ? MAX_TEAMS : FIT - 1)) : 1;
  static constexpr int NSLOT = IN_TILE ? (FIT > NTEAM + 2 ? NTEAM + 2 : FIT) : 2;
  static constexpr int CTHREADS = NTEAM * TTHREADS;
  static constexpr int THREADS = CTHREADS + 32;  // + the producer warp
  static constexpr size_t OFF_EXCH = NSLOT * SLOT_BYTES;
  static constexpr size_t OFF_FTAB = (OFF_EXCH + NTEAM * EXCH_BYTES + 15) & ~(size_t)15;  // the transform's twiddle tables
  // Tile n is announced on full[n mod 2 NSLOT]: two "full" barriers per slot, used in turn.  A parity wait is right only if
  // the waiter is less than one phase ahead of the barrier, and with one barrier per slot a team could be: the copies of
  // tiles n and n + 1 may land out of order, and the team done with n + 1 would then take the still pending phase of
  // tile n for the completed phase of tile n + NSLOT.  With two barriers the phase in doubt belongs to tile n - NSLOT,
  // which was consumed before the producer could issue tile n, and that was before the tile this team worked on last
  // (n + NSLOT - NTEAM >= n).
  static constexpr int NFULL = 2 * NSLOT;
  static constexpr size_t OFF_BAR = (OFF_FTAB + FTAB_BYTES + 7) & ~(size_t)7;              // full[NFULL], empty[NSLOT]
  static constexpr size_t SMEM = OFF_BAR + (NFULL + NSLOT) * 8;
  static_assert(TTHREADS % 32 == 0 && THREADS <= 1024 && NTEAM >= 1, "block shape");
  static_assert(T <= 32 || CTHREADS / T <= 15, "one named barrier per group wider than a warp");
  static_assert(TILE_BYTES % 16 == 0 && ROW_BYTES % 16 == 0 && PB % 4 == 0 && 2 * PB <= 32, "tile shape");
  static_assert((T & (T - 1)) == 0 && (PB & (PB - 1)) == 0 && E % 4 == 0, "powers of two");
  static_assert(NSLOT >= 2 && NSLOT >= NTEAM && SMEM <= kSmemPerSm, "shared memory");
};

// Exchange map of the register FFT onto a pair's own column of a 16-pairs-per-row tile (float2 slots, 128 bytes per row,
// pair pl in slot (pl ^ s_swz(row)) & 15 of a row).  Element e = 16 a + b goes to row 16 a + phi(b ^ a ^ 4 (a & 3)),
// phi(x) = x ^ (x >> 2): its slot is then (pl ^ b ^ a) & 15, which makes the transposing writes (a = thread) and the
// read-back (b = thread) of every geometry bank-conflict free (brute-force checked).  Everything is linear over XOR,
// so the compile-time part of an index folds into one immediate: one LOP3 per access.
__host__ __device__ constexpr uint32_t tile_phi(uint32_t x) { return (x ^ (x >> 2)) & 15u; }
__host__ __device__ constexpr uint32_t tile_lin(uint32_t e) {  // byte offset of element e in the column of pair 0
  return ((e >> 4) << 11) | (tile_phi((e & 15u) ^ ((e >> 4) & 15u) ^ (((e >> 4) & 3u) << 2)) << 7) | ((((e & 15u) ^ (e >> 4)) & 15u) << 3);
}
struct FftTileMap {
  unsigned char *tile;
  uint32_t plx;  // pl << 3
  typedef uint32_t Handle;
  __device__ __forceinline__ Handle pre(int e_t) const { return tile_lin((uint32_t)e_t) ^ plx; }
  __device__ __forceinline__ float2 &at(Handle h, int e_c) const {
    return *reinterpret_cast<float2 *>(tile + (h ^ tile_lin((uint32_t)e_c)));
  }
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
#define ST4(p, v) __stcs(reinterpret_cast<float4 *>(p), (v))
#define ST2(p, v) __stcs(reinterpret_cast<float2 *>(p), (v))
#define ST1(p, v) __stcs((p), (v))

__device__ __forceinline__ void mbar_init(uint64_t *b, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t *b) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *b, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
// Bounded wait: a faulted copy or a pipeline bug must trap after ~2 s, not hang the GPU.
__device__ __forceinline__ void mbar_wait(uint64_t *b, uint32_t parity) {
  const uint32_t addr = smem_u32(b);
  long long t0 = 0;
  for (uint32_t spins = 0;; ++spins) {
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(addr), "r"(parity) : "memory");
    if (ok) return;
    // a waiting warp must not take issue slots from the working ones: back off after a few quick polls
    if (spins >= 4) __nanosleep(spins < 16 ? 100 : 400);
    if (spins == 64) t0 = clock64();
    if (spins > 64 && (spins & 255) == 0 && clock64() - t0 > 4000000000LL) __trap();
  }
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

}  // namespace

// GAPALL: G, A and Pw are all requested (no per-element pointer tests)
// FULL: max_lag == L/2 (every lag of the circular correlation is stored; the two end points are the same sample)
// rnorm[c] = 1/sqrt(sum over all L bins of S_cc) = 1/sqrt(L R_cc[0]) (0 where that sum is 0; reading R16).
// Srsq: the four shifted copies of 1/sqrt(S_cc[f]) (store_rsq4 in delta_internal.h).
template <int L, bool FULL, bool GAPALL>
__global__ void __launch_bounds__(PairCfg<L>::THREADS, 1)
pair_kernel(const float2 *__restrict__ S, const float *__restrict__ Srsq, const float *__restrict__ rnorm,
            const ushort2 *__restrict__ list, const float2 *__restrict__ tw, const float2 *__restrict__ ftab, Layout lay,
            PairConsts pc, float *__restrict__ G_, float *__restrict__ A_, float *__restrict__ Pw_, float *__restrict__ R_) {
  using Cfg = PairCfg<L>;
  using Geo = typename Cfg::G;
  constexpr int N = Cfg::N, F = Cfg::F, T = Cfg::T, E = Cfg::E, PB = Cfg::PB, NSLOT = Cfg::NSLOT, NTEAM = Cfg::NTEAM;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float2 *ftab_s = reinterpret_cast<float2 *>(smem_raw + Cfg::OFF_FTAB);
  uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + Cfg::OFF_BAR), *empty = full + Cfg::NFULL;

  float *const G = G_, *const A = A_, *const Pw = Pw_, *const R = R_;
  const bool wantG = G != nullptr, wantGAP = G || A || Pw;
  const int tid = threadIdx.x;
  // the CTA's tiles: blockIdx.x + n gridDim.x, n = 0 .. ncta-1; tile n goes through slot n mod NSLOT and is worked on
  // by team n mod NTEAM
  const int ntiles = (int)lay.Poblk;
  const int ncta = ((int)blockIdx.x < ntiles) ? (ntiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;

  pdl_launch_dependents();
  if (tid == 0) {
    for (int s = 0; s < Cfg::NFULL; ++s) mbar_init(full + s, 1);
    for (int s = 0; s < NSLOT; ++s) mbar_init(empty + s, Cfg::TW);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  for (int i = tid; i < Geo::TABLE; i += Cfg::THREADS) ftab_s[i] = __ldg(ftab + i);  // a constant table of the plan
  __syncthreads();
  pdl_wait();  // S, rsq and rnorm come from the preceding kernels; the outputs may still be read by a consumer
  if (tid >= Cfg::CTHREADS) {
    // ===== producer warp: fills slot n mod NSLOT with tile n of this CTA: the pairs' channels, the rho normalisation
    // and the bulk copies.  The tables of tile n + 1 are worked out (global loads and all) before the wait for its slot.
    const int lane = tid - Cfg::CTHREADS, pl = lane % PB;
    const bool rows = Cfg::ROWS && wantG;
    ushort2 ij = make_ushort2(0, 1);
    float rs = 0.f;
    auto tables = [&](int n) {
      const int64_t p = ((int64_t)blockIdx.x + (int64_t)n * gridDim.x) * PB + pl;
      // all pairs: (i, j) of lexicographic pair p;  pair list (f2): entry p of the list, whose S values sit at
      // lexicographic index pg in the S layout
      ij = make_ushort2(0, 1);
      if (p < lay.Po) ij = list ? list[p] : pair_of(p, lay.C);
      if (R) rs = __ldg(rnorm + (lane < PB ? ij.x : ij.y));
    };
    if (ncta > 0) tables(0);
    for (int n = 0; n < ncta; ++n) {
      const int tile = blockIdx.x + n * gridDim.x;
      const int s = n % NSLOT;
      uint64_t *fullb = full + n % Cfg::NFULL;
      unsigned char *st = smem_raw + (size_t)s * Cfg::SLOT_BYTES;
      if (lay.jitter_mask & kJitPairProducer) __nanosleep((unsigned)lay.jitter_ns);  // (test hook)
      if (n >= NSLOT) mbar_wait(empty + s, (n / NSLOT - 1) & 1);
      if (lane < PB) {
        reinterpret_cast<ushort2 *>(st + Cfg::OFF_IJ)[lane] = ij;
        reinterpret_cast<int *>(st + Cfg::OFF_PG)[lane] = (int)ij.x * lay.C - ((int)ij.x * ((int)ij.x + 1)) / 2 + (int)ij.y - (int)ij.x - 1;
      }
      if (R && lane < 2 * PB) reinterpret_cast<float *>(st + Cfg::OFF_RS)[lane] = rs;
      __syncwarp();
      if (lane == 0) {
        const uint32_t bytes = (list ? 0u : (uint32_t)Cfg::TILE_BYTES) + (rows ? (uint32_t)(PB * Cfg::ROW_BYTES) : 0u);
        if (bytes) mbar_expect_tx(fullb, bytes); else mbar_arrive(fullb);
        // (test hook kJitPairReorder: the copy of an even tile waits until the next tile's copy is on its way)
        const bool defer = (lay.jitter_mask & kJitPairReorder) && !(n & 1) && n + 1 < ncta;
        if (!list && !defer) bulk_g2s(st, S + (int64_t)tile * F * PB, (uint32_t)Cfg::TILE_BYTES, fullb);  // else: the groups gather
        if ((lay.jitter_mask & kJitPairReorder) && (n & 1) && !list) {
          __nanosleep((unsigned)lay.jitter_ns);
          const int m = n - 1;
          bulk_g2s(smem_raw + (size_t)(m % NSLOT) * Cfg::SLOT_BYTES, S + (int64_t)(blockIdx.x + m * gridDim.x) * F * PB,
                   (uint32_t)Cfg::TILE_BYTES, full + m % Cfg::NFULL);
        }
      }
      __syncwarp();
      // 1/sqrt(S_jj) row of every pair, from the copy of the table that is aligned for the pair's float4 groups
      if (rows && lane < PB)
        bulk_g2s(st + Cfg::OFF_ROWS + lane * Cfg::ROW_BYTES, Srsq + ((int64_t)((-pl) & 3) * lay.C + ij.y) * Cfg::FP,
                 (uint32_t)Cfg::ROW_BYTES, fullb);
      if (n + 1 < ncta) tables(n + 1);
    }
    return;
  }
  // ===== compute warps =====
  const int team = tid / Cfg::TTHREADS, tt = tid % Cfg::TTHREADS;

  using Sync = FftGroupBarSync<T>;  // groups wider than a warp meet at a named barrier of their own
  float2 *exch = reinterpret_cast<float2 *>(smem_raw + Cfg::OFF_EXCH);  // [PB][BUF] (narrow tiles only)
  const int pl = tt / T, gt = tt % T;
  float2 wg = __ldg(tw + gt);  // e^{-2 pi i gt / L}
  // Output rows have F = N + 1 floats (F mod 4 = 1), so element (p, f) is 16-byte aligned iff (p + f) mod 4 = 0: the
  // float4 groups of pair p start at f0 = (-p) mod 4 = (-pl) mod 4 (tiles start at multiples of 4); the f0 head bins and
  // the tail bins go scalar.  Copy f0 of the rsq table holds bin f at index f - f0, so its float4 reads are aligned too.
  const bool vec4 = (((reinterpret_cast<uintptr_t>(G) | reinterpret_cast<uintptr_t>(A) | reinterpret_cast<uintptr_t>(Pw)) & 15) == 0);
  const int f0 = (-pl) & 3, ng = (F - f0) >> 2;
  const float *rsq_f0 = Srsq + (int64_t)f0 * lay.C * Cfg::FP;
  auto value = [&](float2 s, float g2, float &mag, float &coh, float &ang) {
    mag = sqrt_approx(fmaf(s.x, s.x, s.y * s.y));
    coh = mag * g2;
    ang = atan2_poly(s.y, s.x);
  };

  for (int n = team; n < ncta; n += NTEAM) {
    const int tile = blockIdx.x + n * gridDim.x;
    const int s = n % NSLOT;
    unsigned char *st = smem_raw + (size_t)s * Cfg::SLOT_BYTES;
    float2 *tl = reinterpret_cast<float2 *>(st);  // [F][PB], slot = (pl ^ s_swz(f)) & (PB-1)
    if (lay.jitter_mask & kJitPairTeams) __nanosleep((unsigned)(team * lay.jitter_ns));  // (test hook)
    mbar_wait(full + n % Cfg::NFULL, (n / Cfg::NFULL) & 1);
    const ushort2 ij = reinterpret_cast<const ushort2 *>(st + Cfg::OFF_IJ)[pl];
    const int64_t p = (int64_t)tile * PB + pl;
    const bool valid = p < lay.Po;
    if (list) {  // gather this pair's column: slot (pl ^ s_swz(f)) of row f holds S[pg][f]
      const int pg = reinterpret_cast<const int *>(st + Cfg::OFF_PG)[pl];
      const float2 *src = S + (int64_t)(pg >> lay.pb_shift) * F * PB;
      for (int f = gt; f < F; f += T) {
        const int sw = s_swz(f);
        tl[f * PB + ((pl ^ sw) & (PB - 1))] = __ldg(src + f * PB + ((pg ^ sw) & (PB - 1)));
      }
      Sync::sync();
    }

    // ---- pass 1: G, A, P ----------------------------------------------------------------------------------------
    if (wantGAP && valid) {
      const float *ri = rsq_f0 + (int64_t)ij.x * Cfg::FP;
      if (vec4 && gt < ng) {
        // Step q covers the bins f0 + 4 (gt + T q) .. + 3.  A step moves 4 T rows down the tile, which changes neither
        // the slot (it depends on bits 0..5 of the row, and 4 T is a multiple of 64 or the only step) nor anything
        // else but a constant offset: tile addresses, table rows and output pointers are set up once per tile.
        // (The two shortest transforms have 4 T < 64: their slots are worked out per step.)
        constexpr int NQ = E / 4;
        constexpr bool HOIST = (4 * T) % 64 == 0;
        const int fb = f0 + 4 * gt;
        const float2 *tb[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) tb[k] = tl + (fb + k) * PB + ((pl ^ s_swz(fb + k)) & (PB - 1));
        const float4 *gi4 = reinterpret_cast<const float4 *>(ri) + gt;
        const float4 *gj4 = Cfg::ROWS ? reinterpret_cast<const float4 *>(st + Cfg::OFF_ROWS + pl * Cfg::ROW_BYTES) + gt
                                      : reinterpret_cast<const float4 *>(rsq_f0 + (int64_t)ij.y * Cfg::FP) + gt;
        if (wantG) {  // the later steps' pieces of the row of channel i: into L1 now, so that only the first step can miss
#pragma unroll
          for (int q = 1; q < NQ; ++q)
            if (gt + T * q < ng) asm volatile("prefetch.global.L1 [%0];" ::"l"(gi4 + T * q));
        }
        const int64_t at = p * F + fb;
        float *Pw0 = Pw ? Pw + at : nullptr, *G0 = G ? G + at : nullptr, *A0 = A ? A + at : nullptr;
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
          if (gt + T * q >= ng) continue;
          float2 sv[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const int f = fb + k + 4 * T * q;
            sv[k] = HOIST ? tb[k][q * 4 * T * PB] : tl[f * PB + ((pl ^ s_swz(f)) & (PB - 1))];
          }
          float g2[4] = {0.f, 0.f, 0.f, 0.f};
          if (wantG) {
            // the row of channel i comes through L1 (every pair of the tile reads the same one or two rows)
            const float4 gi = __ldg(gi4 + T * q), gj = Cfg::ROWS ? gj4[T * q] : __ldg(gj4 + T * q);
            g2[0] = gi.x * gj.x; g2[1] = gi.y * gj.y; g2[2] = gi.z * gj.z; g2[3] = gi.w * gj.w;
          }
          float m[4], c[4], an[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) value(sv[k], g2[k], m[k], c[k], an[k]);
          if (GAPALL || Pw) ST4(Pw0 + q * 4 * T, make_float4(m[0], m[1], m[2], m[3]));
          if (GAPALL || G) ST4(G0 + q * 4 * T, make_float4(c[0], c[1], c[2], c[3]));
          if (GAPALL || A) ST4(A0 + q * 4 * T, make_float4(an[0], an[1], an[2], an[3]));
        }
      }
      // scalar bins: the edges of the vector path (the f0 head bins and the bins from f0 + 4 ng on: at most 5), or every
      // bin if the arrays are not 16-byte aligned.  Copy 0 of the rsq table holds bin f at index f.
      const int ntail = vec4 ? F - (f0 + 4 * ng) : F - f0;
      for (int e = gt; e < f0 + ntail; e += T) {
        const int f = e < f0 ? e : (vec4 ? f0 + 4 * ng : f0) + (e - f0);
        const float g2 = wantG ? __ldg(Srsq + (int64_t)ij.x * Cfg::FP + f) * __ldg(Srsq + (int64_t)ij.y * Cfg::FP + f) : 0.f;
        float m, c, an;
        value(tl[f * PB + ((pl ^ s_swz(f)) & (PB - 1))], g2, m, c, an);
        if (GAPALL || Pw) ST1(Pw + p * F + f, m);
        if (GAPALL || G) ST1(G + p * F + f, c);
        if (GAPALL || A) ST1(A + p * F + f, an);
      }
    }
    if (lay.jitter_mask & kJitPairWarps) __nanosleep((unsigned)(((tid >> 5) & 3) * lay.jitter_ns));  // (test hook)
    if (!R) {  // the slot is free once every group of this warp has read it
      __syncwarp();
      if ((tid & 31) == 0) mbar_arrive(empty + s);
      continue;
    }

    // ---- pass 2: merge step of the inverse real transform (S read again from the tile; twice the merge of
    // irfft_merge, the factor 1/2 goes into the normalisation) ------------------------------------------------
    float2 v[E];
    // (the products wg * wstep[u] below are the same for every tile; the compiler would keep all E of them alive across
    // the tile loop, in local memory: make wg opaque per tile instead)
    asm volatile("" : "+f"(wg.x), "+f"(wg.y));
    const int pg = pl ^ s_swz(gt);
#pragma unroll
    for (int u = 0; u < E; ++u) {
      const int f = gt + T * u;
      const int fr = N - f;
      float2 sf = tl[f * PB + ((pg ^ s_swz(T * u)) & (PB - 1))];  // s_swz(gt | T u) = s_swz(gt) ^ s_swz(T u)
      float2 sr = tl[fr * PB + ((pl ^ s_swz(fr)) & (PB - 1))];
      if (u == 0 && gt == 0) { sf.y = 0.f; sr.y = 0.f; }  // Im S[0], Im S[N] do not enter the real transform
      const float2 w = cmul(wg, pc.wstep[u]);               // e^{-2 pi i f / L}; the inverse uses its conjugate
      v[u] = irfft_merge2(sf, sr, make_float2(w.x, -w.y));
    }
    const float norm = reinterpret_cast<const float *>(st + Cfg::OFF_RS)[pl] * reinterpret_cast<const float *>(st + Cfg::OFF_RS)[PB + pl];

    // ---- rho = irfft(S) / sqrt(R_ii[0] R_jj[0]) ----------------------------------------------------------------
    // x = z/N with z[n] = (x[2n], x[2n+1]) N, n = gt + T u; norm = 1/(L sqrt(R_ii[0] R_jj[0])) carries 2 (L/N) x 1/2.
    Sync::sync();  // every S value of the group's pairs is in registers (and the last transform's read-back is done)
    if constexpr (Cfg::IN_TILE) {
      fft_inplace_g<Geo, true, Sync>(v, FftTileMap{st, (uint32_t)pl << 3}, ftab_s, gt);
      Sync::sync();  // the group's read-back is done: the slot can be refilled
      if ((tid & 31) == 0) mbar_arrive(empty + s);
    } else {
      if ((tid & 31) == 0) mbar_arrive(empty + s);  // this warp's S values are in registers (the slot counts every warp)
      fft_inplace_g<Geo, true, Sync>(v, FftPadMap{exch + pl * Geo::BUF}, ftab_s, gt);
    }
    float *Rp = R + p * lay.nlags;
    if (FULL && T <= 32) {
      // lag m = xi for xi <= L/2 and xi - L for xi >= L/2; row position q = m + L/2.  Element nn holds xi = 2 nn, 2 nn + 1
      // at the even position q: a float2 store if the row is 8-byte aligned.  Rows have 2 M + 1 floats, so every other
      // row is not: there the pairs are taken one sample later, (x[2 nn + 1], x[2 nn + 2]) at q + 1, with x[2 nn + 2] from
      // the next thread of the group (from the next element of thread 0 for the last thread).  That covers the
      // positions 1 .. L (xi = L/2 at position L included); position 0, also xi = L/2, is stored on its own.  (Scalar
      // stores for those rows, 64-byte pieces and twice the instructions, cost 3 us in a store-only replica.)
      // (every thread of the warp takes part in the shuffles; the pairs beyond the last one of a ragged tile do not store)
      const bool odd = (reinterpret_cast<uintptr_t>(Rp) & 7) != 0;
#pragma unroll
      for (int u = 0; u < E; ++u) {
        const int nn = gt + T * u;
        const float a = v[u].x * norm, b = v[u].y * norm;
        const int q = (u < E / 2) ? 2 * nn + N : 2 * nn - N;
        const float nxt = __shfl_sync(0xffffffffu, gt == 0 ? v[(u + 1) % E].x : v[u].x, (gt + 1) & (T - 1), T < 32 ? T : 32) * norm;
        if (valid) {
          ST2(Rp + q + (odd ? 1 : 0), odd ? make_float2(b, nxt) : make_float2(a, b));
          if (u == E / 2 && gt == 0) ST1(Rp + (odd ? 0 : L), a);  // xi = L/2 is lag -L/2 and lag +L/2
        }
      }
    } else if (!valid) {
    } else if (FULL) {  // groups wider than a warp
      const bool vec = (reinterpret_cast<uintptr_t>(Rp) & 7) == 0;
#pragma unroll
      for (int u = 0; u < E; ++u) {
        const int nn = gt + T * u;
        const float a = v[u].x * norm, b = v[u].y * norm;
        const int q = (u < E / 2) ? 2 * nn + N : 2 * nn - N;
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
        const int nn = gt + T * u;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int xi = 2 * nn + h;
          const float val = (h ? v[u].y : v[u].x) * norm;
          if (xi <= M) Rp[xi + M] = val;
          if (xi >= L - M) Rp[xi - L + M] = val;
        }
      }
    }
  }
}

// rsq4 = the four shifted copies of 1/sqrt(S_cc[f]) (0 where S_cc[f] <= 0, reading R16) and
// rnorm[c] = 1/sqrt(S_cc[0] + 2 sum_{0<f<N} S_cc[f] + S_cc[N]) = 1/sqrt(sum over all L bins) = 1/sqrt(L R_cc[0]).
// One warp per channel.
__global__ void __launch_bounds__(32) auto_prep_kernel(const float *__restrict__ Sauto, float *__restrict__ rsq4,
                                                       float *__restrict__ rnorm, Layout lay) {
  const int c = blockIdx.x, lane = threadIdx.x, F = lay.F;
  float sum = 0.f;
  for (int f = lane; f < F; f += 32) {
    const float a = Sauto[(int64_t)c * F + f];
    store_rsq4(rsq4, lay, c, f, a > 0.f ? rsqrtf(a) : 0.f);
    sum = fmaf((f == 0 || f == F - 1) ? 1.f : 2.f, a, sum);
  }
  for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
  if (lane == 0) rnorm[c] = sum > 0.f ? rsqrtf(sum) : 0.f;
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
static int launch_pair_L(delta_plan *p, const float *d_S, const float *d_rsq, const float *d_rnorm, float *d_G, float *d_A,
                         float *d_P, float *d_R, cudaStream_t st) {
  using Cfg = PairCfg<L>;
  const Layout &lay = p->lay;
  if (lay.Poblk == 0 || lay.Po == 0) return DELTA_OK;
  const ushort2 *list = p->cfg.n_pairs > 0 ? p->d_pairs() : nullptr;
  PairConsts pc;
  for (int u = 0; u < 16; ++u) pc.wstep[u] = p->h_wstep[u];
  const bool full = lay.M == L / 2;
  // persistent: one CTA per SM (or fewer if there are not that many tiles), NTEAM tiles in work on each
  const int64_t want = (lay.Poblk + Cfg::NTEAM - 1) / Cfg::NTEAM;
  const unsigned grid = (unsigned)(want < p->num_sms ? want : p->num_sms);
#define DELTA_PAIR_LAUNCH(FULL_, GAPALL_)                                                                           \
  do {                                                                                                              \
    int rc = opt_in_smem(pair_kernel<L, FULL_, GAPALL_>, Cfg::SMEM);                                                \
    if (rc) return rc;                                                                                              \
    LaunchCfg lc(dim3(grid), dim3(Cfg::THREADS), Cfg::SMEM, st, p->use_pdl);                                        \
    DELTA_CUDA_CHECK(cudaLaunchKernelEx(&lc.cfg, pair_kernel<L, FULL_, GAPALL_>, reinterpret_cast<const float2 *>(d_S), \
                                        d_rsq, d_rnorm, list, p->d_tw(), p->d_ftab(), lay, pc, d_G, d_A, d_P, d_R)); \
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

// ------------------------------------------------------------------------------------------
// Transform lengths that are not powers of two: the per-pair quantities from the definitions,
// with Eq. (1d) as the direct inverse sum  R[m] = (1/L) (S[0] + (-1)^m S[L/2] + 2 sum_{0<f<L/2} Re(S[f] e^{+2 pi i f m/L}))
// over the Hermitian half spectrum (L even; Im S[0], Im S[L/2] ignored).  One CTA per tile of PB pairs; O(L^2) per pair.
__global__ void __launch_bounds__(256)
pair_dft_kernel(const float2 *__restrict__ S, const float *__restrict__ Srsq, const float *__restrict__ rnorm,
                const ushort2 *__restrict__ list, const float2 *__restrict__ tw, Layout lay, float *__restrict__ G,
                float *__restrict__ A, float *__restrict__ Pw, float *__restrict__ R) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2 *tl = reinterpret_cast<float2 *>(smem_raw);  // [F][PB], slot = (pl ^ s_swz(f)) & (PB-1)
  __shared__ ushort2 ij_s[16];
  __shared__ int pg_s[16];
  const int tid = threadIdx.x, PB = lay.PB, F = lay.F, L = lay.L, Fp = lay.Fp;
  const int64_t p0 = (int64_t)blockIdx.x * PB;
  pdl_launch_dependents();
  if (tid < PB) {
    ushort2 ij = make_ushort2(0, 1);
    if (p0 + tid < lay.Po) ij = list ? list[p0 + tid] : pair_of(p0 + tid, lay.C);
    ij_s[tid] = ij;
    pg_s[tid] = (int)ij.x * lay.C - ((int)ij.x * ((int)ij.x + 1)) / 2 + (int)ij.y - (int)ij.x - 1;
  }
  pdl_wait();
  __syncthreads();
  for (int idx = tid; idx < F * PB; idx += 256) {
    const int f = idx / PB, sw = s_swz(f);
    const int pg = pg_s[((idx % PB) ^ sw) & (PB - 1)];  // the pair whose slot this is
    tl[idx] = __ldg(S + ((int64_t)(pg >> lay.pb_shift) * F + f) * PB + ((pg ^ sw) & (PB - 1)));
  }
  __syncthreads();
  const int nv = (int)(lay.Po - p0 < PB ? lay.Po - p0 : PB);
  if (G || A || Pw) {
    for (int e = tid; e < nv * F; e += 256) {
      const int pl = e / F, f = e - pl * F;
      const ushort2 ij = ij_s[pl];
      const float2 s = tl[f * PB + ((pl ^ s_swz(f)) & (PB - 1))];
      const float mag = sqrt_approx(fmaf(s.x, s.x, s.y * s.y));
      const int64_t at = (p0 + pl) * F + f;
      if (Pw) Pw[at] = mag;
      if (G) G[at] = mag * __ldg(Srsq + (int64_t)ij.x * Fp + f) * __ldg(Srsq + (int64_t)ij.y * Fp + f);
      if (A) A[at] = atan2_poly(s.y, s.x);
    }
  }
  if (R) {
    const int nl = lay.nlags, M = lay.M, half = L / 2;
    for (int e = tid; e < nv * nl; e += 256) {
      const int pl = e / nl, q = e - pl * nl;
      const int m = q - M, mm = m < 0 ? m + L : m;  // lag mod L
      const int slot = pl, sgn = (m & 1) ? -1 : 1;
      float acc = 0.f;
      int idx = 0;  // f mm mod L
      for (int f = 1; f < half; ++f) {
        idx += mm;
        if (idx >= L) idx -= L;
        const float2 w = __ldg(tw + idx);  // e^{-2 pi i idx / L}: cos = w.x, sin = -w.y
        const float2 s = tl[f * PB + ((slot ^ s_swz(f)) & (PB - 1))];
        acc = fmaf(s.x, w.x, fmaf(s.y, w.y, acc));  // Re(S e^{+i theta}) = S.x cos - S.y sin
      }
      const float s0 = tl[(pl ^ s_swz(0)) & (PB - 1)].x, sh = tl[half * PB + ((pl ^ s_swz(half)) & (PB - 1))].x;
      const ushort2 ij = ij_s[pl];
      R[(p0 + pl) * nl + q] = (2.f * acc + s0 + (float)sgn * sh) * __ldg(rnorm + ij.x) * __ldg(rnorm + ij.y);
    }
  }
}

static int launch_pair_dft(delta_plan *p, const float *d_S, const float *d_rsq, const float *d_rnorm, float *d_G, float *d_A,
                           float *d_P, float *d_R, cudaStream_t st) {
  const Layout &lay = p->lay;
  if (lay.Poblk == 0 || lay.Po == 0) return DELTA_OK;
  const ushort2 *list = p->cfg.n_pairs > 0 ? p->d_pairs() : nullptr;
  const size_t smem = (size_t)lay.F * lay.PB * sizeof(float2);
  int rc = opt_in_smem(pair_dft_kernel, smem);
  if (rc) return rc;
  LaunchCfg lc(dim3((unsigned)lay.Poblk), dim3(256), smem, st, p->use_pdl);
  DELTA_CUDA_CHECK(cudaLaunchKernelEx(&lc.cfg, pair_dft_kernel, reinterpret_cast<const float2 *>(d_S), d_rsq, d_rnorm, list,
                                      p->d_tw(), lay, d_G, d_A, d_P, d_R));
  p->launches++;
  DELTA_CUDA_CHECK(cudaGetLastError());
  return DELTA_OK;
}

int launch_pair(delta_plan *p, const float *d_S, const float *d_rsq, const float *d_rnorm, float *d_G, float *d_A, float *d_P,
                float *d_R, cudaStream_t st) {
  if (!has_fft_path(p->lay.L)) return launch_pair_dft(p, d_S, d_rsq, d_rnorm, d_G, d_A, d_P, d_R, st);
#define CALL(LL) launch_pair_L<LL>(p, d_S, d_rsq, d_rnorm, d_G, d_A, d_P, d_R, st)
  DELTA_SWITCH_L(p->lay.L, CALL)
#undef CALL
}

int launch_auto_prep(delta_plan *p, const float *d_auto, float *d_rsq, float *d_rnorm, cudaStream_t st) {
  auto_prep_kernel<<<(unsigned)p->lay.C, 32, 0, st>>>(d_auto, d_rsq, d_rnorm, p->lay);
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
