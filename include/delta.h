/* delta.h -- C ABI of libdelta_b200: the all-channel-pairs spectral path of the Delta framework
 * (arxiv 2108.08896, "Near real-time streaming analysis of big fusion data"), hand-written CUDA
 * for NVIDIA B200 (sm_100a).
 *
 * What the library computes, per streamed channel-by-time chunk (citations are line numbers of
 * the paper text, /root/reference/PAPER.md; DESIGN.md section 3 lists the readings R1..R22 taken
 * where the paper is silent or garbled):
 *
 *   normalisation   y_c[t] = (x_c[t] - o_c)/o_c               "After normalizing each chunk" L107, L89
 *   STFT            X_c[k,f] = sum_n w[n] y_c[kH+n] e^{-2 pi i f n/L}        L107, L169 (Hann, R2-R5)
 *   Eq. (1a) L95    S_ij[f]  = s^2 (1/K) sum_k X_i[k,f] conj(X_j[k,f])       (E[.] = mean over segments)
 *                   P_ij[f]  = |S_ij[f]|                                     cross-power
 *   Eq. (1b) L97    G_ij[f]  = |S_ij[f]| / sqrt(S_ii[f] S_jj[f])             coherence
 *   Eq. (1c) L100   A_ij[f]  = atan2(Im S_ij[f], Re S_ij[f])                 cross-phase
 *   Eq. (1d) L102   rho_ij[m] = IFFT_L(S_ij)[m] / sqrt(R_ii[0] R_jj[0])      cross-correlation, m = -M..M
 *   for all C(C-1)/2 channel pairs i < j, lexicographic ("18336 ... channel pair combinations" L107), or for an
 *   explicit pair list.  Variants next to the path (delta_config): band-pass filter, other windows, detrend,
 *   zero-padded segments, per-segment-normalised coherence; delta_accumulate averages spectra over chunks.
 *
 * Conventions
 *   - Pointers named d_* are DEVICE pointers, h_* are HOST pointers; all are owned by the caller.
 *     The library never allocates device memory: scratch comes from delta_plan_set_workspace().
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Every call
 *     that takes a stream is asynchronous on it and never synchronises, unless stated otherwise.
 *   - Every function returns DELTA_OK (0) or a negative delta_status; nothing is printed.
 *   - A plan is bound to the device that is current when delta_plan_set_workspace() is called and
 *     must not be used from two streams at the same time (it owns the scratch buffers).
 *   - There is no CPU fallback: without a CUDA device every compute call returns DELTA_ERR_CUDA.
 *
 * Symbols: C channels, T samples per chunk, L = nfft, H = hop, K = (T-L)/H + 1 segments (no
 * padding, tail dropped; (T - nperseg)/H + 1 with zero-padded segments), F = L/2+1 one-sided bins,
 * P = C(C-1)/2 pairs (or the length of the pair list), M = max_lag.
 */
#ifndef DELTA_B200_H
#define DELTA_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DELTA_VERSION 201 /* 0.2.1: delta_coherence_static, DELTA_ERR_TOO_LARGE (0.2.0: out_ring in
                             delta_analyze_shot_host; scales inside X buffers; DELTA_ERR_NO_MEMORY) */

typedef enum {
  DELTA_OK = 0,
  DELTA_ERR_INVALID_ARG = -1, /* NULL pointer, non-positive size, unknown enum value               */
  DELTA_ERR_UNSUPPORTED = -2, /* nfft odd or outside [16,4096], T < segment length, hop larger
                                 than the segment, max_lag > L/2, C > 4096                         */
  DELTA_ERR_ALIGNMENT = -3,   /* a device pointer is not 16-byte aligned                            */
  DELTA_ERR_NO_WORKSPACE = -4,/* compute call before delta_plan_set_workspace(), or it is too small */
  DELTA_ERR_CUDA = -5,        /* a CUDA runtime call failed; see delta_last_cuda_error()            */
  DELTA_ERR_STATE = -6,       /* e.g. norm_mode needs offsets and delta_set_offsets() was not called */
  DELTA_ERR_NO_MEMORY = -7,   /* host allocation of the plan failed                                 */
  DELTA_ERR_TOO_LARGE = -8    /* delta_coherence_static: the plan needs more than DELTA_STATIC_SCRATCH_BYTES */
} delta_status;

/* periodic (DFT-even) windows, x = 2 pi n/L: Hann 1/2 - 1/2 cos x (R4, the default); the others are the f1 variants:
 * Hamming 0.54 - 0.46 cos x, rectangular 1, Blackman 0.42 - 0.5 cos x + 0.08 cos 2x */
enum { DELTA_WIN_HANN_PERIODIC = 0, DELTA_WIN_HAMMING_PERIODIC = 1, DELTA_WIN_RECT = 2, DELTA_WIN_BLACKMAN_PERIODIC = 3 };
/* Eq. (1b) estimator: from the segment-averaged spectra (R10, the default), or the per-segment-normalised variant (f2):
 * every X[c,k,f] is replaced by X/|X| before Eq. (1a), so S is a mean of unit phasors, S_cc = s^2, G = |mean phasor| */
enum { DELTA_EST_AVERAGED = 0, DELTA_EST_PHASE_LOCK = 1 };
/* per-segment detrend before the window: none (R5, the default) or the mean of the segment's samples */
enum { DELTA_DETREND_NONE = 0, DELTA_DETREND_CONSTANT = 1 };
enum { DELTA_SCALE_WINPOW = 0,                       /* s^2 = 1/sum w^2 (default; white noise of
                                                        variance v has E S_ii = v)                    */
       DELTA_SCALE_NONE = 1,                         /* s^2 = 1                                       */
       DELTA_SCALE_DENSITY = 2,                      /* s^2 = 1/(fs sum w^2)                          */
       DELTA_SCALE_SPECTRUM = 3 };                   /* s^2 = 1/(sum w)^2                             */
enum { DELTA_F32 = 0, DELTA_I16 = 1 };               /* element type of the input chunk               */
enum { DELTA_NORM_NONE = 0,                          /* y = x                                         */
       DELTA_NORM_SUBTRACT = 1,                      /* y = x - o_c                                   */
       DELTA_NORM_RELATIVE = 2 };                    /* y = (x - o_c)/o_c   (delta T_e/<T_e>, L89)    */
enum { DELTA_CONTRACT_AUTO = 0,                      /* library picks: tensor cores up to 960 channels */
       DELTA_CONTRACT_FP32 = 1,                      /* Eq. (1a) on the FP32 FMA pipe                 */
       DELTA_CONTRACT_TC = 2 };                      /* Eq. (1a) on tcgen05 tensor cores, split fp16;
                                                        more than 960 channels: DELTA_ERR_UNSUPPORTED */

typedef struct {
  int32_t n_channels;   /* C >= 1                                                                     */
  int32_t n_samples;    /* T >= nfft, samples per channel per chunk                                   */
  int32_t nfft;         /* L, transform length: even, 16..4096.  Powers of two from 64 up run on the register
                         * FFT; any other even length on direct-DFT kernels (O(L^2), correct, not tuned)        */
  int32_t hop;          /* H in [1, L]; overlap = L - H                                               */
  int32_t window;       /* DELTA_WIN_*                                                                */
  int32_t scaling;      /* DELTA_SCALE_*                                                              */
  float   fs;           /* sampling rate in Hz; only DELTA_SCALE_DENSITY uses it                      */
  int32_t in_dtype;     /* DELTA_F32 | DELTA_I16                                                      */
  int32_t norm_mode;    /* DELTA_NORM_*; SUBTRACT and RELATIVE need delta_set_offsets() once per shot */
  int32_t max_lag;      /* M in [0, L/2]; cross-correlation lags -M..M                                */
  int32_t n_pairs;      /* 0 => all i < j in lexicographic order ("channel pair combinations") */
  const int32_t *h_pairs; /* host [n_pairs][2] or NULL: explicit pair list (f2), every entry 0 <= i < j < C (else
                           * DELTA_ERR_INVALID_ARG), copied by delta_plan_create; the per-pair outputs then have
                           * n_pairs rows in list order (S_ji = conj S_ij gives the swapped pair: G, P equal, A
                           * negated, rho with the lags reversed); d_S still holds all pairs */
  int32_t contraction;  /* DELTA_CONTRACT_*                                                           */
  /* Optional band-pass pre-processing filter ("pre-processing filters", L231: the demo's 5-9 kHz pass
   * band), reading R19: an ideal mask on the bins of every segment's transform; bin f is kept iff
   * bp_lo_hz <= f fs / nfft <= bp_hi_hz.  Both 0 => no filter.  Needs fs > 0 and 0 <= bp_lo_hz <= bp_hi_hz, else
   * DELTA_ERR_INVALID_ARG.  Outside the band S = 0, hence P = G = A = 0; rho is normalised with the filtered
   * zero-lag autocorrelations. */
  float   bp_lo_hz, bp_hi_hz;
  int32_t detrend;      /* DELTA_DETREND_*                                                            */
  int32_t estimator;    /* DELTA_EST_*                                                                */
  int32_t nperseg;      /* 0 => nfft.  Otherwise segments of nperseg <= nfft samples (window of that length),
                         * zero-padded to nfft (f2, R22): the correlation of Eq. (1d) is then the linear one for
                         * |lag| <= nfft - nperseg.  Needs hop <= nperseg <= n_samples; K = (T - nperseg)/hop + 1 */
} delta_config;

typedef struct {
  int32_t n_segments;      /* K */
  int32_t n_bins;          /* F = L/2 + 1 */
  int32_t n_lags;          /* 2M + 1 */
  int32_t contraction;     /* the mode the plan resolved DELTA_CONTRACT_AUTO to */
  int64_t n_pairs;         /* P: rows of the per-pair outputs (all pairs, or the length of the explicit list) */
  int64_t workspace_bytes; /* minimum size for delta_plan_set_workspace() */
  int64_t x_bytes;         /* size of a d_X buffer  (delta_stft output, opaque layout) */
  int64_t s_bytes;         /* size of a d_S buffer (delta_cross_spectra output, opaque layout) */
  int64_t s_block_pairs;   /* pairs per block of the d_S layout (see delta_cross_spectra) */
} delta_sizes;

typedef struct delta_plan delta_plan; /* opaque; owned by the library */

/* Validates the configuration, copies it, builds host-side tables.  Makes no CUDA call, so it
 * also works on a machine without a GPU.  *out is set to NULL on failure. */
int delta_plan_create(const delta_config *cfg, delta_plan **out);
int delta_plan_destroy(delta_plan *plan);
int delta_plan_sizes(const delta_plan *plan, delta_sizes *out);

/* Hands the plan its scratch memory (>= workspace_bytes, 256-byte aligned, device memory that
 * stays valid while the plan is used) and uploads the twiddle / window / pair tables into it on
 * `stream`.  Binds the plan to the current device. */
int delta_plan_set_workspace(delta_plan *plan, void *d_workspace, size_t bytes, void *stream);

/* Per-shot offsets for DELTA_NORM_SUBTRACT / RELATIVE (reading R1): o_c = mean of the first
 * n_first samples of channel c of d_x (the first chunk of the shot), element type = in_dtype,
 * `ld` = elements between consecutive channels.  For int16 input the sum is exact (integer). */
int delta_set_offsets(delta_plan *plan, const void *d_x, int64_t ld, int32_t n_first, void *stream);
/* Copies the C offsets (as float64: integer sum / n_first for int16) to h_out.  Synchronises stream. */
int delta_get_offsets(delta_plan *plan, double *h_out, void *stream);

/* a0 + a1.  Normalise, window and Fourier-transform every segment of every channel.
 * d_x: [C][ld] of in_dtype, ld >= T.  d_X: x_bytes, layout opaque (see delta_stft_unpack). */
int delta_stft(delta_plan *plan, const void *d_x, int64_t ld, void *d_X, void *stream);
/* Test accessor: expands d_X to complex64 [C][K][F] (interleaved re, im), unscaled as in the
 * definition above. */
int delta_stft_unpack(delta_plan *plan, const void *d_X, float *d_out, void *stream);

/* a2 + a3, Eq. (1a).  d_S: s_bytes of complex64 in the library's pair-block layout
 * [ceil(P/B)][F][B], B = s_block_pairs: lexicographic pair p is in block p / B, and inside row f of
 * the block in slot (p ^ f ^ (f >> 2)) mod B (use delta_cross_spectra_unpack to read it); d_Sauto: float [C][F]
 * autospectra S_cc[f].  Either may be NULL. */
int delta_cross_spectra(delta_plan *plan, const void *d_X, float *d_S, float *d_Sauto, void *stream);
/* Test accessor: expands d_S to complex64 [P][F] (interleaved re, im), pairs lexicographic. */
int delta_cross_spectra_unpack(delta_plan *plan, const float *d_S, float *d_out, void *stream);

/* a4, Eq. (1b): d_G float [P][F].  0 where S_ii S_jj = 0 (R16). */
int delta_coherence(delta_plan *plan, const float *d_S, const float *d_Sauto, float *d_G, void *stream);
/* a4, Eq. (1b) again, for callers that cannot let scratch be allocated or handed over: code under
 * CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  Same arguments, same kernels and same
 * result as delta_coherence, but the stage's scratch -- the table of 1/sqrt(S_cc[f]) in four shifted copies and
 * 1/sqrt(L R_cc[0]), 4 C ceil4(F) + C floats, each part rounded up to 256 bytes -- lives in a device array of
 * DELTA_STATIC_SCRATCH_BYTES inside the library (held by every GPU that loads the library, until the process exits)
 * instead of the plan's workspace.  The call allocates nothing (no cudaMalloc, cudaFree or allocating library routine); the
 * plan's workspace must still be set: the constant tables of the plan are read from it.
 *   - A plan that needs more scratch than the array holds is refused with DELTA_ERR_TOO_LARGE (8 MiB covers every
 *     BASELINE config: 0.8 MB at config 2, 6.3 MB at config 5; 576 channels at nfft 512 need 2.4 MB).
 *   - The plan's device must be the current device (else DELTA_ERR_INVALID_ARG).
 *   - ALL calls on a device, from any plan, share the one array.  Calls that overlap on the GPU (different streams
 *     without an ordering between them) race on it: order them, or use delta_coherence, whose scratch is per plan.  The
 *     array keeps the last call's contents; every call clears the part it uses before writing it. */
#define DELTA_STATIC_SCRATCH_BYTES (8u << 20)
int delta_coherence_static(delta_plan *plan, const float *d_S, const float *d_Sauto, float *d_G, void *stream);
/* a4, Eq. (1c): d_A float [P][F], radians in [-pi, pi]. */
int delta_crossphase(delta_plan *plan, const float *d_S, float *d_A, void *stream);
/* a4, |Eq. (1a)|: d_P float [P][F]. */
int delta_crosspower(delta_plan *plan, const float *d_S, float *d_P, void *stream);
/* a5, Eq. (1d): d_R float [P][2M+1], lags -M..M increasing, normalised by sqrt(R_ii[0] R_jj[0]),
 * circular in the lag (R12).  0 where the denominator is 0. */
int delta_crosscorr(delta_plan *plan, const float *d_S, const float *d_Sauto, float *d_R, void *stream);

/* f2 (shot-level accumulation): the expectation of Eq. (1a), over the segments of several chunks.
 * d_S_acc = w_acc d_S_acc + w_new d_S (s_bytes each, the library's layout) and the same for the autospectra
 * (float [C][F]); either pair of pointers may be NULL.  w_acc = 0 initialises (the old contents are not read).
 * Every chunk has the same number of segments, so n calls with (n-1)/n, 1/n weights -- or weights 1 and any common
 * factor: G, A and rho do not depend on it -- give the average over all segments.  The staged calls
 * (delta_coherence, ...) then work on the accumulated spectra. */
int delta_accumulate(delta_plan *plan, float *d_S_acc, float *d_Sauto_acc, const float *d_S, const float *d_Sauto,
                     float w_acc, float w_new, void *stream);

/* The whole path a0..a5 for one chunk resident in device memory, using the plan's workspace for
 * X and S.  Any output pointer may be NULL (that quantity is then not computed / stored).
 * Outputs as in the staged calls: d_G, d_A, d_P [P][F]; d_R [P][2M+1]; d_Sauto [C][F]. */
int delta_analyze_chunk(delta_plan *plan, const void *d_x, int64_t ld,
                        float *d_G, float *d_A, float *d_P, float *d_R, float *d_Sauto, void *stream);

/* a6: a whole shot from HOST memory ("streamed as chunks of 10,000 samples"; ~500 MB/s stream, L201).
 * h_x: [n_chunks][C][T] of in_dtype (pinned memory for true overlap).  Chunk n+1 is copied host->device on an
 * internal side stream while chunk n is analysed on `stream` (two device input slots taken from d_slots,
 * >= 2*C*T*sizeof(in_dtype) bytes, 256-byte aligned).  If set_offsets != 0 the offsets are taken from the first
 * n_first samples of chunk 0.
 * Device outputs (NULL pointer = that quantity is skipped): chunk n goes to output set  n mod out_ring  (out_ring = 0:
 * every chunk its own set, n), set s starting s*stride_X elements into d_X (a stride of 0 makes all sets one).
 * Host outputs (any may be NULL): chunk n's result is copied device->host to h_X + n*(its full size) on a second
 * internal stream, under the kernels of the following chunks; an output set is not overwritten before its
 * copy-back is over (out_ring <= 64 when host outputs are requested and sets are reused, else
 * DELTA_ERR_UNSUPPORTED).  Returns after enqueuing; `stream` ends after the last copy-back, so the caller
 * synchronises that one stream. */
int delta_analyze_shot_host(delta_plan *plan, const void *h_x, int32_t n_chunks, void *d_slots,
                            int32_t set_offsets, int32_t n_first,
                            float *d_G, float *d_A, float *d_P, float *d_R, float *d_Sauto,
                            int64_t stride_GAP, int64_t stride_R, int64_t stride_auto, int32_t out_ring,
                            float *h_G, float *h_A, float *h_P, float *h_R, float *h_Sauto,
                            void *stream);

/* Profiling hook.  `events` = 4 cudaEvent_t handles (passed as void*) owned by the caller, or NULL to
 * switch the hook off.  While set, every delta_analyze_chunk() records events[0] before the STFT
 * stage, events[1] after it, events[2] after the contraction and events[3] after the pair stage, on
 * the launching stream (so the caller can time each stage with cudaEventElapsedTime). */
int delta_plan_set_stage_events(delta_plan *plan, void *const *events);

/* Number of kernels the last delta_analyze_chunk() on this plan launched (for bench accounting). */
int delta_last_launch_count(const delta_plan *plan);

const char *delta_strerror(int status);
/* cudaError_t of the last failing CUDA call made by this library in the calling thread (0 if none). */
int delta_last_cuda_error(void);
int delta_version(void);

#ifdef __cplusplus
}
#endif
#endif /* DELTA_B200_H */
