// Internal declarations of libdelta_b200 (not part of the C ABI; see include/delta.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>
#include <vector>

#include "delta.h"

namespace delta {

constexpr int kPairTile = 64;     // channel block of the FP32 contraction tiles
constexpr int kSegBlock = 8;      // segments per K-chunk ("kc") of the X layout
constexpr int kThreads = 256;
constexpr int kTcMaxGroups = 16;  // TMEM-sized groups of accumulator units per frequency bin
constexpr int kTcMaxUnits = 4;    // units per group

// unit plan of the tensor-core contraction (host side; see contract_tc.cu)
struct TcHostPlan {
  int ngroups;
  int nunits[kTcMaxGroups];
  int units[kTcMaxGroups][kTcMaxUnits][6];  // row0, lane_lo, lane_hi, col0, N, tmem column of Re
};
bool tc_plan_tiles(int Cp, TcHostPlan *out);

// pairs per block of the S layout = pairs per tile of the pair kernel (two tiles and the exchange buffers must fit
// shared memory).  8 or 32 pairs per tile instead of 16 were measured slower at nfft 512 (round 1).
constexpr int pair_block(int L) { return L <= 1024 ? 16 : (L == 2048 ? 8 : 4); }
constexpr int pair_fft_points(int N) { return N <= 64 ? 8 : 16; }  // E of FftGeom<N> (fft_reg.cuh)

// transform lengths served by the register FFT (fft_reg.cuh); every other even length in [16, 4096] takes the direct-DFT
// kernels (stft_dft_kernel, pair_dft_kernel)
constexpr bool has_fft_path(int L) { return (L & (L - 1)) == 0 && L >= 64 && L <= 4096; }

struct Layout {
  // X (STFT) buffer, frequency-major so that one bin's C x K matrix is one contiguous block:
  //   FP32 mode : float  X[f][part][kc][c][8]                 part 0 = Re, 1 = Im
  //   TC   mode : __half X[f][prec][part][kc][c][8]           prec 0 = hi, 1 = lo (split fp16)
  // k = 8*kc + kk, c < Cp (rows C..Cp-1 are zero), kc < Kc = Kp/8, Kp = K rounded up to 16.
  int C, Cp, T, L, N, H, K, Kp, Kc, F, M, nlags;
  int Ls;   // samples per segment (nperseg <= L; the rest of the transform's input is zero)
  int Fp;   // row pitch of the rsq table: F rounded up to 4 floats
  int64_t x_scale_off;  // TC mode: byte offset of the C per-channel fp16 scales (float) behind the operand planes of an X buffer
  float wsum;      // sum_n |w[n]|: |X| <= wsum max|y| bounds the split-fp16 operands
  int detrend;     // DELTA_DETREND_*
  int estimator;   // DELTA_EST_*
  int f_lo, f_hi;  // pass band of the optional band-pass filter, in bins (0 .. F-1 when it is off)
  int nkb;  // segment blocks per channel = ceil(K / 8): one partial of the windowed signal energy each (wpart)
  // S (cross-spectra) is complex64 [Pblk][F][PB]: pairs in lexicographic order p = iC - i(i+1)/2 + (j-i-1),
  // block = p / PB, and inside row f of a block pair p sits in slot (p ^ s_swz(f)) & (PB-1), s_swz(f) = f ^ (f >> 2).
  // One block is one
  // contiguous tile for the pair kernel; the XOR makes its column (fixed pair) reads bank-conflict free.
  int PB, pb_shift;
  int64_t P, Pblk;    // all pairs i < j: the S layout
  int64_t Po, Poblk;  // output rows: P, or the length of the explicit pair list (f2)
  int64_t x_elems_per_f;  // elements (float or half) per frequency
  // Test hook (delta_internal_set_jitter, api.cu; both 0 in normal use): the roles of the kernels sleep jitter_ns nanoseconds
  // at the places the bits of jitter_mask name, so that a protocol that only holds for the usual relative speeds of
  // producer, consumer and neighbours fails every time instead of once in a long while.
  int jitter_mask, jitter_ns;
};
enum : int {
  kJitTcEpiLate = 1,     // contraction: epilogue warps sleep before every accumulator unit but the first of an item
  kJitTcEpiSkew = 2,     //              odd epilogue warps sleep before every unit
  kJitTcProducer = 4,    //              the operand producer sleeps before every stage
  kJitTcMma = 8,         //              the MMA issuer sleeps before every unit
  kJitPairProducer = 16, // pair kernel: the producer sleeps before every tile
  kJitPairTeams = 32,    //              team t sleeps t x ns before every tile
  kJitPairWarps = 64,    //              warp w sleeps (w mod 4) x ns between the two passes
  kJitStftStart = 128,   // STFT: CTAs start skewed
  kJitStftMid = 256,     //       CTAs are skewed again before the write-out
  kJitPairReorder = 512  // pair kernel: the copy of every even tile of a CTA is issued after the next tile's copy and a pause
                         //              (concurrent bulk copies may complete in any order; this makes them)
};

// Row swizzle of the S layout.  It is XOR-linear (s_swz(a ^ b) = s_swz(a) ^ s_swz(b)), and makes the three column
// access patterns of the pair kernel bank-conflict free: 4 consecutive bins per lane with lanes 4 bins apart (G/A/P pass),
// bins gt + T u over lanes gt (merge), and at most 2-way for the mirrored bins N - f.
#if defined(__CUDACC__)
__host__ __device__
#endif
constexpr int s_swz(int f) { return f ^ (f >> 2); }

struct Workspace {
  size_t off_tw, off_win, off_ftab, off_pairs, off_offs, off_isum, off_chmax, off_chcnt, off_X, off_S, off_auto, off_rsq, off_wpart, off_rnorm, total;
};

// The table of 1/sqrt(S_cc[f]) is kept as four shifted copies, float rsq4[4][C][Fp]: copy s holds bin f at index f - s
// (f >= s).  The float4 groups of an output row start at bin f0 = (-p) mod 4 (pair.cu), and copy f0 makes the matching
// float4 reads of the table 16-byte aligned.  Copy 0 is the plain table.
#if defined(__CUDACC__)
__device__ __forceinline__ void store_rsq4(float *rsq4, const Layout &lay, int c, int f, float v) {
#pragma unroll
  for (int s = 0; s < 4; ++s)
    if (f >= s) rsq4[((int64_t)s * lay.C + c) * lay.Fp + (f - s)] = v;
}
#endif

}  // namespace delta

struct delta_plan {
  delta_config cfg;
  delta::Layout lay;
  delta::Workspace wsl;
  int contraction;   // resolved mode
  float s2;          // spectral scaling s^2 (reading R6)
  // host tables (uploaded by delta_plan_set_workspace)
  std::vector<float2> h_tw;      // e^{-2 pi i f / L}, f = 0..L-1
  std::vector<float> h_win;      // periodic Hann
  float2 h_wstep[16];            // e^{-2 pi i T u / L}, u < E: bin f = gt + T u of a thread has twiddle tw[gt] * wstep[u]
  std::vector<float2> h_ftab;    // per-pass twiddles of the register FFT (fft_reg.cuh), N = L/2
  std::vector<ushort2> h_pairs;  // the explicit pair list (empty: all pairs)
  delta::TcHostPlan tc;
  int num_sms = 148;
  // device state
  char *ws = nullptr;
  size_t ws_bytes = 0;
  int device = -1;
  bool offsets_set = false;
  int n_first = 0;
  int launches = 0;
  long long *d_trace = nullptr;  // debug: clock stamps of the tensor-core contraction (delta_debug_set_trace)
  bool band_on = false;  // band-pass filter or phase-lock estimator: rho is normalised from the autospectra, not from
                         // the windowed signal energy (Parseval does not apply to the modified spectra)
  bool use_pdl = true;  // programmatic dependent launch between the hot-path kernels (DELTA_NO_PDL=1 switches it off)
  bool stage_events_on = false;
  cudaEvent_t stage_ev[4] = {nullptr, nullptr, nullptr, nullptr};
  // delta_analyze_shot_host: host -> device copies on copy_stream, device -> host copies on d2h_stream
  cudaStream_t copy_stream = nullptr, d2h_stream = nullptr;
  cudaEvent_t ev_copied[2] = {nullptr, nullptr};    // input slot s holds its chunk
  cudaEvent_t ev_consumed[2] = {nullptr, nullptr};  // the kernels have read input slot s
  cudaEvent_t ev_start = nullptr;
  std::vector<cudaEvent_t> ev_out, ev_back;         // per output set: computed / copied back

  const float2 *d_tw() const { return reinterpret_cast<const float2 *>(ws + wsl.off_tw); }
  const float *d_win() const { return reinterpret_cast<const float *>(ws + wsl.off_win); }
  const float2 *d_ftab() const { return reinterpret_cast<const float2 *>(ws + wsl.off_ftab); }
  const ushort2 *d_pairs() const { return reinterpret_cast<const ushort2 *>(ws + wsl.off_pairs); }
  double *d_offs() const { return reinterpret_cast<double *>(ws + wsl.off_offs); }
  long long *d_isum() const { return reinterpret_cast<long long *>(ws + wsl.off_isum); }
  unsigned *d_chmax() const { return reinterpret_cast<unsigned *>(ws + wsl.off_chmax); }  // zero between launches
  unsigned *d_chcnt() const { return reinterpret_cast<unsigned *>(ws + wsl.off_chcnt); }  // zero between launches
  void *d_X() const { return ws + wsl.off_X; }
  float *d_S() const { return reinterpret_cast<float *>(ws + wsl.off_S); }
  float *d_auto() const { return reinterpret_cast<float *>(ws + wsl.off_auto); }
  float *d_rsq() const { return reinterpret_cast<float *>(ws + wsl.off_rsq); }
  // wpart[c][kb] = sum over the 8 segments of block kb of sum_n (w[n] y_c[kH+n])^2  (written by stft_kernel);
  // by Parseval  sum over all L bins of S_cc = L s^2/K * sum_kb wpart[c][kb] = L R_cc[0]   (pin P4)
  float *d_wpart() const { return reinterpret_cast<float *>(ws + wsl.off_wpart); }
  // rnorm[c] = 1/sqrt(sum over all L bins of S_cc) = 1/sqrt(L R_cc[0]): from wpart (contraction kernels, fused call) or
  // from caller-supplied autospectra (auto_prep_kernel, staged calls)
  float *d_rnorm() const { return reinterpret_cast<float *>(ws + wsl.off_rnorm); }
};

namespace delta {

void set_cuda_error(cudaError_t e);
#define DELTA_CUDA_CHECK(expr)                 \
  do {                                         \
    cudaError_t _e = (expr);                   \
    if (_e != cudaSuccess) {                   \
      ::delta::set_cuda_error(_e);             \
      return DELTA_ERR_CUDA;                   \
    }                                          \
  } while (0)

// Programmatic dependent launch: a kernel launched with the attribute may become resident while its predecessor in
// the stream is still running; it must call pdl_wait() before it reads anything the predecessor wrote or writes
// anything the predecessor reads.  pdl_launch_dependents() lets the successor start its own prologue early.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
#endif
struct LaunchCfg {
  cudaLaunchConfig_t cfg;
  cudaLaunchAttribute attr[2];
  LaunchCfg(dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl, unsigned cluster_x = 0) {
    cfg = cudaLaunchConfig_t{};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    unsigned n = 0;
    if (pdl) {
      attr[n].id = cudaLaunchAttributeProgrammaticStreamSerialization;
      attr[n].val.programmaticStreamSerializationAllowed = 1;
      ++n;
    }
    if (cluster_x > 1) {
      attr[n].id = cudaLaunchAttributeClusterDimension;
      attr[n].val.clusterDim.x = cluster_x;
      attr[n].val.clusterDim.y = 1;
      attr[n].val.clusterDim.z = 1;
      ++n;
    }
    cfg.attrs = attr;
    cfg.numAttrs = n;
  }
};

// Opt in to more than 48 KB of dynamic shared memory.  The attribute belongs to the (kernel, device) pair and is a
// maximum, so it is set once per pair and raised only when a launch needs more (the launchers call this every time).
// Fixed-size table, no heap: the launch path allocates nothing.
struct SmemOptIn {
  const void *kern;
  int dev;
  size_t bytes;
};
template <typename Kern>
static inline int opt_in_smem(Kern kern, size_t bytes) {
  if (bytes <= 48 * 1024) return DELTA_OK;
  constexpr int kSlots = 256;
  static std::mutex mu;  // one table per translation unit and kernel signature
  static SmemOptIn seen[kSlots];
  static int nseen = 0;
  int dev = 0;
  DELTA_CUDA_CHECK(cudaGetDevice(&dev));
  const void *key = reinterpret_cast<const void *>(kern);
  std::lock_guard<std::mutex> lock(mu);
  SmemOptIn *slot = nullptr;
  for (int i = 0; i < nseen; ++i)
    if (seen[i].kern == key && seen[i].dev == dev) slot = &seen[i];
  if (slot && slot->bytes >= bytes) return DELTA_OK;
  DELTA_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
  if (slot) slot->bytes = bytes;
  else if (nseen < kSlots) seen[nseen++] = {key, dev, bytes};  // (a full table only costs the call again next time)
  return DELTA_OK;
}

// dispatch on the transform length (validate() admits powers of two in [64, 4096])
#define DELTA_SWITCH_L(L_, CALL)           \
  switch (L_) {                            \
    case 64: return CALL(64);              \
    case 128: return CALL(128);            \
    case 256: return CALL(256);            \
    case 512: return CALL(512);            \
    case 1024: return CALL(1024);          \
    case 2048: return CALL(2048);          \
    case 4096: return CALL(4096);          \
    default: return DELTA_ERR_UNSUPPORTED; \
  }

// launchers (each returns a delta_status and counts its launches into plan->launches)
int launch_offsets(delta_plan *p, const void *d_x, int64_t ld, int n_first, cudaStream_t st);
int launch_stft(delta_plan *p, const void *d_x, int64_t ld, void *d_X, cudaStream_t st);
int launch_stft_pad_zero(delta_plan *p, void *d_X, cudaStream_t st);  // zero padding of a caller-supplied X buffer
int launch_stft_unpack(delta_plan *p, const void *d_X, float *d_out, cudaStream_t st);
// Both contractions write S (may be null), the autospectra and the rsq4 table (either may be null), and, if d_rnorm is
// not null, rnorm[c] = 1/sqrt(rscale * sum_k wpart[c][k]) from the STFT kernel's energy partials.
int launch_contract_fp32(delta_plan *p, const void *d_X, float *d_S, float *d_auto, float *d_rsq, float *d_rnorm, float rscale,
                         cudaStream_t st);
int launch_contract_tc(delta_plan *p, const void *d_X, float *d_S, float *d_auto, float *d_rsq, float *d_rnorm, float rscale,
                       cudaStream_t st);
int launch_auto_prep(delta_plan *p, const float *d_auto, float *d_rsq, float *d_rnorm, cudaStream_t st);
int launch_pair(delta_plan *p, const float *d_S, const float *d_rsq, const float *d_rnorm, float *d_G, float *d_A, float *d_P,
                float *d_R, cudaStream_t st);
int launch_axpby(delta_plan *p, float *acc, const float *x, int64_t n, float wa, float wn, cudaStream_t st);
int launch_s_unpack(delta_plan *p, const float *d_S, float *d_out, cudaStream_t st);

}  // namespace delta
