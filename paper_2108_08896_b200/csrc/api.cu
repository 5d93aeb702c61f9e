// C-ABI entry points of libdelta_b200 (include/delta.h): argument validation, plan and workspace
// management, and the launch sequences.  All arithmetic of the path lives in the kernels.
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>

#include "delta_internal.h"
#include "fft_reg.cuh"

namespace delta {

static thread_local int g_last_cuda_error = 0;
void set_cuda_error(cudaError_t e) { g_last_cuda_error = (int)e; }

static inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }
static inline bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

static int validate(const delta_config *c) {
  if (!c) return DELTA_ERR_INVALID_ARG;
  if (c->n_channels < 1 || c->n_samples < 1 || c->nfft < 1 || c->hop < 1 || c->max_lag < 0) return DELTA_ERR_INVALID_ARG;
  if (c->window < DELTA_WIN_HANN_PERIODIC || c->window > DELTA_WIN_BLACKMAN_PERIODIC) return DELTA_ERR_INVALID_ARG;
  if (c->detrend < DELTA_DETREND_NONE || c->detrend > DELTA_DETREND_CONSTANT) return DELTA_ERR_INVALID_ARG;
  if (c->estimator < DELTA_EST_AVERAGED || c->estimator > DELTA_EST_PHASE_LOCK) return DELTA_ERR_INVALID_ARG;
  if (c->scaling < DELTA_SCALE_WINPOW || c->scaling > DELTA_SCALE_SPECTRUM) return DELTA_ERR_INVALID_ARG;
  if (c->in_dtype != DELTA_F32 && c->in_dtype != DELTA_I16) return DELTA_ERR_INVALID_ARG;
  if (c->norm_mode < DELTA_NORM_NONE || c->norm_mode > DELTA_NORM_RELATIVE) return DELTA_ERR_INVALID_ARG;
  if (c->contraction < DELTA_CONTRACT_AUTO || c->contraction > DELTA_CONTRACT_TC) return DELTA_ERR_INVALID_ARG;
  if (c->scaling == DELTA_SCALE_DENSITY && !(c->fs > 0.f)) return DELTA_ERR_INVALID_ARG;
  if (c->n_pairs < 0 || (c->n_pairs > 0 && !c->h_pairs)) return DELTA_ERR_INVALID_ARG;
  if (c->bp_lo_hz != 0.f || c->bp_hi_hz != 0.f) {
    if (!(c->fs > 0.f) || !(c->bp_lo_hz >= 0.f) || !(c->bp_hi_hz >= c->bp_lo_hz)) return DELTA_ERR_INVALID_ARG;
  }
  const int L = c->nfft;
  if (L < 16 || L > 4096 || (L & 1) != 0) return DELTA_ERR_UNSUPPORTED;  // even lengths; see has_fft_path()
  if (c->nperseg < 0 || c->nperseg > L) return DELTA_ERR_INVALID_ARG;
  const int Ls = c->nperseg > 0 ? c->nperseg : L;
  if (c->hop > Ls) return DELTA_ERR_UNSUPPORTED;
  if (c->n_samples < Ls) return DELTA_ERR_UNSUPPORTED;
  if (c->max_lag > L / 2) return DELTA_ERR_UNSUPPORTED;
  if (c->n_channels > 4096) return DELTA_ERR_UNSUPPORTED;
  for (int k = 0; k < c->n_pairs; ++k) {  // explicit pair list (f2): 0 <= i < j < C
    const int i = c->h_pairs[2 * k], j = c->h_pairs[2 * k + 1];
    if (i < 0 || j <= i || j >= c->n_channels) return DELTA_ERR_INVALID_ARG;
  }
  return DELTA_OK;
}

// bytes of an X buffer: the operand planes, then (tensor-core mode) the C per-channel scales
static size_t x_buffer_bytes(const delta_plan *p) {
  const size_t planes = (size_t)p->lay.x_scale_off;
  return p->contraction == DELTA_CONTRACT_TC ? align_up(planes + (size_t)p->lay.C * sizeof(float), 16) : planes;
}

static bool tc_supported(const delta_config *c) {
  // the tile plan must exist (up to 16 groups of accumulator units per bin: 960 channels); the operand stages of many
  // channels are packed per unit (contract_tc.cu, mode 3), so shared memory does not limit the channel count
  size_t Cp = align_up((size_t)c->n_channels, 64);
  if (Cp < 128) Cp = 128;
  TcHostPlan tmp;
  return tc_plan_tiles((int)Cp, &tmp);
}

}  // namespace delta

using namespace delta;

extern "C" {

int delta_plan_create(const delta_config *cfg, delta_plan **out) {
  if (!out) return DELTA_ERR_INVALID_ARG;
  *out = nullptr;
  int rc = validate(cfg);
  if (rc) return rc;
  if (cfg->contraction == DELTA_CONTRACT_TC && !tc_supported(cfg)) return DELTA_ERR_UNSUPPORTED;
  delta_plan *p = new (std::nothrow) delta_plan();
  if (!p) return DELTA_ERR_NO_MEMORY;
  p->cfg = *cfg;
  p->use_pdl = std::getenv("DELTA_NO_PDL") == nullptr;
  p->cfg.h_pairs = nullptr;
  p->contraction = (cfg->contraction == DELTA_CONTRACT_AUTO) ? (tc_supported(cfg) ? DELTA_CONTRACT_TC : DELTA_CONTRACT_FP32)
                                                             : cfg->contraction;
  Layout &l = p->lay;
  l.C = cfg->n_channels;
  l.Cp = (int)align_up((size_t)l.C, 64);
  if (l.Cp < 128) l.Cp = 128;
  l.T = cfg->n_samples;
  l.L = cfg->nfft;
  l.N = l.L / 2;
  l.H = cfg->hop;
  l.Ls = cfg->nperseg > 0 ? cfg->nperseg : l.L;
  l.K = (l.T - l.Ls) / l.H + 1;
  l.Kp = (int)align_up((size_t)l.K, 16);
  l.Kc = l.Kp / kSegBlock;
  l.nkb = (l.K + kSegBlock - 1) / kSegBlock;
  l.F = l.L / 2 + 1;
  l.Fp = (l.F + 3) & ~3;
  l.f_lo = 0;
  l.f_hi = l.F - 1;
  l.estimator = cfg->estimator;
  const bool band = cfg->bp_lo_hz != 0.f || cfg->bp_hi_hz != 0.f;
  p->band_on = band || cfg->estimator == DELTA_EST_PHASE_LOCK;
  if (band) {  // bin f is kept iff lo L <= f fs <= hi L (float64); the kept bins are one contiguous range
    const double lo = (double)cfg->bp_lo_hz * l.L, hi = (double)cfg->bp_hi_hz * l.L, fs = (double)cfg->fs;
    l.f_lo = l.F;
    l.f_hi = -1;
    for (int f = 0; f < l.F; ++f)
      if (lo <= f * fs && f * fs <= hi) {
        if (f < l.f_lo) l.f_lo = f;
        l.f_hi = f;
      }
  }
  l.M = cfg->max_lag;
  l.nlags = 2 * l.M + 1;
  l.P = (int64_t)l.C * (l.C - 1) / 2;
  l.PB = pair_block(l.L);
  l.pb_shift = l.PB == 32 ? 5 : (l.PB == 16 ? 4 : (l.PB == 8 ? 3 : 2));
  l.Pblk = (l.P + l.PB - 1) / l.PB;
  l.Po = cfg->n_pairs > 0 ? cfg->n_pairs : l.P;
  l.Poblk = (l.Po + l.PB - 1) / l.PB;
  // floats (2 parts) or halves (2 precisions x 2 parts) per frequency
  l.x_elems_per_f = (int64_t)(p->contraction == DELTA_CONTRACT_TC ? 4 : 2) * l.Kc * l.Cp * kSegBlock;
  // TC mode: the C per-channel fp16 scales follow the operand planes inside the X buffer (a multiple of 16 bytes in)
  l.x_scale_off = (int64_t)l.F * l.x_elems_per_f * (p->contraction == DELTA_CONTRACT_TC ? 2 : 4);

  // host tables in float64, rounded once
  const int L = l.L;
  p->h_tw.resize(L);
  p->h_win.resize(L);
  double sw = 0.0, sw2 = 0.0;
  for (int n = 0; n < L; ++n) {
    const double ang = -2.0 * M_PI * (double)n / (double)L;
    p->h_tw[n] = make_float2((float)std::cos(ang), (float)std::sin(ang));
    const double xw = 2.0 * M_PI * (double)n / (double)l.Ls;  // the window spans the segment; zero over the padding
    double w;
    switch (cfg->window) {
      case DELTA_WIN_HAMMING_PERIODIC: w = 0.54 - 0.46 * std::cos(xw); break;
      case DELTA_WIN_RECT: w = 1.0; break;
      case DELTA_WIN_BLACKMAN_PERIODIC: w = 0.42 - 0.5 * std::cos(xw) + 0.08 * std::cos(2.0 * xw); break;
      default: w = 0.5 - 0.5 * std::cos(xw); break;
    }
    if (n >= l.Ls) w = 0.0;
    p->h_win[n] = (float)w;
    sw += w;
    sw2 += w * w;
  }
  l.wsum = (float)(sw * (1.0 + 1e-6));  // all four windows are non-negative
  l.detrend = cfg->detrend;
  p->h_ftab.resize((size_t)fft_table_size(l.N) + 1);
  fft_twiddle_table(l.N, p->h_ftab.data());
  {
    const int E = pair_fft_points(l.N);  // E of the pair kernel's FFT geometry
    const int Tg = l.N / E;
    for (int u = 0; u < 16; ++u) {
      const long long e = ((long long)Tg * u) % L;
      const double ang = -2.0 * M_PI * (double)e / (double)L;
      p->h_wstep[u] = make_float2((float)std::cos(ang), (float)std::sin(ang));
    }
  }
  switch (cfg->scaling) {
    case DELTA_SCALE_WINPOW: p->s2 = (float)(1.0 / sw2); break;
    case DELTA_SCALE_NONE: p->s2 = 1.f; break;
    case DELTA_SCALE_DENSITY: p->s2 = (float)(1.0 / ((double)cfg->fs * sw2)); break;
    default: p->s2 = (float)(1.0 / (sw * sw)); break;
  }
  for (int k = 0; k < cfg->n_pairs; ++k)
    p->h_pairs.push_back(make_ushort2((unsigned short)cfg->h_pairs[2 * k], (unsigned short)cfg->h_pairs[2 * k + 1]));
  memset(&p->tc, 0, sizeof(p->tc));
  if (p->contraction == DELTA_CONTRACT_TC && !tc_plan_tiles(l.Cp, &p->tc)) { delete p; return DELTA_ERR_UNSUPPORTED; }

  Workspace &w = p->wsl;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes, 256); return at; };
  w.off_tw = take((size_t)L * sizeof(float2));
  w.off_win = take((size_t)L * sizeof(float));
  w.off_ftab = take(p->h_ftab.size() * sizeof(float2));
  w.off_pairs = take((p->h_pairs.size() + 1) * sizeof(ushort2));
  w.off_offs = take((size_t)l.C * sizeof(double));
  w.off_isum = take((size_t)l.C * sizeof(long long));
  w.off_chmax = take((size_t)l.C * sizeof(unsigned));
  w.off_chcnt = take((size_t)l.C * sizeof(unsigned));
  w.off_X = take(x_buffer_bytes(p));
  w.off_S = take((size_t)(l.Pblk > 0 ? l.Pblk : 1) * l.F * l.PB * sizeof(float2));
  w.off_auto = take((size_t)l.C * l.F * sizeof(float));
  w.off_rsq = take((size_t)4 * l.C * l.Fp * sizeof(float));  // four shifted copies (store_rsq4)
  w.off_wpart = take((size_t)l.C * l.nkb * sizeof(float));
  w.off_rnorm = take((size_t)l.C * sizeof(float));
  w.total = o;
  *out = p;
  return DELTA_OK;
}

int delta_plan_destroy(delta_plan *p) {
  if (!p) return DELTA_ERR_INVALID_ARG;
  if (p->copy_stream) cudaStreamDestroy(p->copy_stream);
  if (p->d2h_stream) cudaStreamDestroy(p->d2h_stream);
  for (int s = 0; s < 2; ++s) {
    if (p->ev_copied[s]) cudaEventDestroy(p->ev_copied[s]);
    if (p->ev_consumed[s]) cudaEventDestroy(p->ev_consumed[s]);
  }
  if (p->ev_start) cudaEventDestroy(p->ev_start);
  for (cudaEvent_t e : p->ev_out) cudaEventDestroy(e);
  for (cudaEvent_t e : p->ev_back) cudaEventDestroy(e);
  delete p;
  return DELTA_OK;
}

int delta_plan_sizes(const delta_plan *p, delta_sizes *out) {
  if (!p || !out) return DELTA_ERR_INVALID_ARG;
  const Layout &l = p->lay;
  out->n_segments = l.K;
  out->n_bins = l.F;
  out->n_lags = l.nlags;
  out->contraction = p->contraction;
  out->n_pairs = l.Po;
  out->workspace_bytes = (int64_t)p->wsl.total;
  out->x_bytes = (int64_t)x_buffer_bytes(p);
  out->s_bytes = (int64_t)(l.Pblk > 0 ? l.Pblk : 1) * l.F * l.PB * (int64_t)sizeof(float2);
  out->s_block_pairs = l.PB;
  return DELTA_OK;
}

int delta_plan_set_workspace(delta_plan *p, void *d_ws, size_t bytes, void *stream) {
  if (!p || !d_ws) return DELTA_ERR_INVALID_ARG;
  if ((reinterpret_cast<uintptr_t>(d_ws) & 255u) != 0) return DELTA_ERR_ALIGNMENT;
  if (bytes < p->wsl.total) return DELTA_ERR_NO_WORKSPACE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  DELTA_CUDA_CHECK(cudaGetDevice(&p->device));
  DELTA_CUDA_CHECK(cudaDeviceGetAttribute(&p->num_sms, cudaDevAttrMultiProcessorCount, p->device));
  p->ws = reinterpret_cast<char *>(d_ws);
  p->ws_bytes = bytes;
  p->offsets_set = false;
  const Layout &l = p->lay;
  DELTA_CUDA_CHECK(cudaMemcpyAsync(p->ws + p->wsl.off_tw, p->h_tw.data(), (size_t)l.L * sizeof(float2), cudaMemcpyHostToDevice, st));
  DELTA_CUDA_CHECK(cudaMemcpyAsync(p->ws + p->wsl.off_win, p->h_win.data(), (size_t)l.L * sizeof(float), cudaMemcpyHostToDevice, st));
  DELTA_CUDA_CHECK(cudaMemcpyAsync(p->ws + p->wsl.off_ftab, p->h_ftab.data(), p->h_ftab.size() * sizeof(float2), cudaMemcpyHostToDevice, st));
  if (!p->h_pairs.empty())
    DELTA_CUDA_CHECK(cudaMemcpyAsync(p->ws + p->wsl.off_pairs, p->h_pairs.data(), p->h_pairs.size() * sizeof(ushort2), cudaMemcpyHostToDevice, st));
  // zero rows C..Cp-1 of the workspace X once (kernels never write them)
  DELTA_CUDA_CHECK(cudaMemsetAsync(p->ws + p->wsl.off_X, 0, p->wsl.off_S - p->wsl.off_X, st));
  DELTA_CUDA_CHECK(cudaMemsetAsync(p->ws + p->wsl.off_offs, 0, p->wsl.off_X - p->wsl.off_offs, st));
  return DELTA_OK;
}

static int need_ws(const delta_plan *p) {
  if (!p) return DELTA_ERR_INVALID_ARG;
  if (!p->ws) return DELTA_ERR_NO_WORKSPACE;
  return DELTA_OK;
}

int delta_set_offsets(delta_plan *p, const void *d_x, int64_t ld, int32_t n_first, void *stream) {
  int rc = need_ws(p);
  if (rc) return rc;
  if (!d_x || n_first < 1 || ld < n_first) return DELTA_ERR_INVALID_ARG;
  p->n_first = n_first;
  rc = launch_offsets(p, d_x, ld, n_first, reinterpret_cast<cudaStream_t>(stream));
  if (rc == DELTA_OK) p->offsets_set = true;
  return rc;
}

int delta_get_offsets(delta_plan *p, double *h_out, void *stream) {
  int rc = need_ws(p);
  if (rc) return rc;
  if (!h_out) return DELTA_ERR_INVALID_ARG;
  if (!p->offsets_set) return DELTA_ERR_STATE;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  DELTA_CUDA_CHECK(cudaMemcpyAsync(h_out, p->d_offs(), (size_t)p->lay.C * sizeof(double), cudaMemcpyDeviceToHost, st));
  DELTA_CUDA_CHECK(cudaStreamSynchronize(st));
  return DELTA_OK;
}

static int check_input(const delta_plan *p, const void *d_x, int64_t ld) {
  if (!d_x || ld < p->lay.T) return DELTA_ERR_INVALID_ARG;
  if (p->cfg.norm_mode != DELTA_NORM_NONE && !p->offsets_set) return DELTA_ERR_STATE;
  return DELTA_OK;
}

int delta_stft(delta_plan *p, const void *d_x, int64_t ld, void *d_X, void *stream) {
  int rc = need_ws(p);
  if (rc) return rc;
  if (!d_X) return DELTA_ERR_INVALID_ARG;
  rc = check_input(p, d_x, ld);
  if (rc) return rc;
  if (!aligned16(d_X)) return DELTA_ERR_ALIGNMENT;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  if (d_X != p->d_X()) {  // the padding of the layout is read by the contraction: zero it in a caller's buffer
    rc = launch_stft_pad_zero(p, d_X, st);
    if (rc) return rc;
  }
  return launch_stft(p, d_x, ld, d_X, st);
}

int delta_cross_spectra_unpack(delta_plan *p, const float *d_S, float *d_out, void *stream) {
  int rc = need_ws(p);
  if (rc) return rc;
  if (!d_S || !d_out) return DELTA_ERR_INVALID_ARG;
  return launch_s_unpack(p, d_S, d_out, reinterpret_cast<cudaStream_t>(stream));
}

// Development hook, not part of the C ABI (not declared in include/delta.h): while d_trace (>= 8192 int64) is set, CTA 0 of
// the tensor-core contraction writes SM clock stamps of its producer / MMA / epilogue roles and every CTA its start and
// end time (contract_tc.cu).
int delta_internal_set_trace(delta_plan *p, void *d_trace) {
  if (!p) return DELTA_ERR_INVALID_ARG;
  p->d_trace = reinterpret_cast<long long *>(d_trace);
  return DELTA_OK;
}

// Test hook, not part of the C ABI: the producer / consumer / neighbour roles of the kernels sleep `ns` nanoseconds at the
// places the bits of `mask` name (kJit* in delta_internal.h).  Results must not depend on it: a wait that is missing in a
// pipeline corrupts them every time under the right skew instead of once in a long while (tests/test_parity_gpu.py).
int delta_internal_set_jitter(delta_plan *p, int mask, int ns) {
  if (!p || mask < 0 || ns < 0 || ns > 1000000) return DELTA_ERR_INVALID_ARG;
  p->lay.jitter_mask = ns ? mask : 0;
  p->lay.jitter_ns = mask ? ns : 0;
  return DELTA_OK;
}

int delta_stft_unpack(delta_plan *p, const void *d_X, float *d_out, void *stream) {
  int rc = need_ws(p);
  if (rc) return rc;
  if (!d_X || !d_out) return DELTA_ERR_INVALID_ARG;
  return launch_stft_unpack(p, d_X, d_out, reinterpret_cast<cudaStream_t>(stream));
}

// d_rsq / d_rnorm: the plan's tables for the pair stage of the fused call; null for the staged delta_cross_spectra,
// which is a function of its arguments only
static int contract(delta_plan *p, const void *d_X, float *d_S, float *d_auto, float *d_rsq, float *d_rnorm, cudaStream_t st) {
  const float rscale = (float)p->lay.L * p->s2 / (float)p->lay.K;  // sum over all L bins of S_cc = rscale * sum_k wpart[c][k]
  return p->contraction == DELTA_CONTRACT_TC ? launch_contract_tc(p, d_X, d_S, d_auto, d_rsq, d_rnorm, rscale, st)
                                             : launch_contract_fp32(p, d_X, d_S, d_auto, d_rsq, d_rnorm, rscale, st);
}

int delta_cross_spectra(delta_plan *p, const void *d_X, float *d_S, float *d_Sauto, void *stream) {
  int rc = need_ws(p);
  if (rc) return rc;
  if (!d_X) return DELTA_ERR_INVALID_ARG;
  if (!aligned16(d_X) || (d_S && !aligned16(d_S))) return DELTA_ERR_ALIGNMENT;
  if (!d_S && !d_Sauto) return DELTA_OK;
  return contract(p, d_X, d_S, d_Sauto, nullptr, nullptr, reinterpret_cast<cudaStream_t>(stream));
}

static int pair_stage(delta_plan *p, const float *d_S, const float *d_Sauto, float *G, float *A, float *P, float *R,
                      void *stream, bool need_auto) {
  int rc = need_ws(p);
  if (rc) return rc;
  if (!d_S || (need_auto && !d_Sauto)) return DELTA_ERR_INVALID_ARG;
  if (!G && !A && !P && !R) return DELTA_ERR_INVALID_ARG;
  if (!aligned16(d_S)) return DELTA_ERR_ALIGNMENT;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  if (need_auto) {  // coherence and rho need 1/sqrt(S_cc[f]) and 1/sqrt(R_cc[0]) of the caller's autospectra (plan scratch)
    rc = launch_auto_prep(p, d_Sauto, p->d_rsq(), p->d_rnorm(), st);
    if (rc) return rc;
  }
  return launch_pair(p, d_S, p->d_rsq(), p->d_rnorm(), G, A, P, R, st);
}

int delta_coherence(delta_plan *p, const float *d_S, const float *d_Sauto, float *d_G, void *stream) {
  if (!d_G) return DELTA_ERR_INVALID_ARG;
  return pair_stage(p, d_S, d_Sauto, d_G, nullptr, nullptr, nullptr, stream, true);
}
int delta_crossphase(delta_plan *p, const float *d_S, float *d_A, void *stream) {
  if (!d_A) return DELTA_ERR_INVALID_ARG;
  return pair_stage(p, d_S, nullptr, nullptr, d_A, nullptr, nullptr, stream, false);
}
int delta_crosspower(delta_plan *p, const float *d_S, float *d_P, void *stream) {
  if (!d_P) return DELTA_ERR_INVALID_ARG;
  return pair_stage(p, d_S, nullptr, nullptr, nullptr, d_P, nullptr, stream, false);
}
int delta_crosscorr(delta_plan *p, const float *d_S, const float *d_Sauto, float *d_R, void *stream) {
  if (!d_R) return DELTA_ERR_INVALID_ARG;
  return pair_stage(p, d_S, d_Sauto, nullptr, nullptr, nullptr, d_R, stream, true);
}

int delta_accumulate(delta_plan *p, float *d_S_acc, float *d_Sauto_acc, const float *d_S, const float *d_Sauto, float w_acc,
                     float w_new, void *stream) {
  int rc = need_ws(p);
  if (rc) return rc;
  if ((d_S_acc == nullptr) != (d_S == nullptr) || (d_Sauto_acc == nullptr) != (d_Sauto == nullptr)) return DELTA_ERR_INVALID_ARG;
  if (!d_S_acc && !d_Sauto_acc) return DELTA_ERR_INVALID_ARG;
  if ((d_S_acc && (!aligned16(d_S_acc) || !aligned16(d_S)))) return DELTA_ERR_ALIGNMENT;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const Layout &l = p->lay;
  if (d_S_acc) {
    rc = launch_axpby(p, d_S_acc, d_S, (int64_t)(l.Pblk > 0 ? l.Pblk : 1) * l.F * l.PB * 2, w_acc, w_new, st);
    if (rc) return rc;
  }
  if (d_Sauto_acc) rc = launch_axpby(p, d_Sauto_acc, d_Sauto, (int64_t)l.C * l.F, w_acc, w_new, st);
  return rc;
}

int delta_analyze_chunk(delta_plan *p, const void *d_x, int64_t ld, float *d_G, float *d_A, float *d_P, float *d_R,
                        float *d_Sauto, void *stream) {
  int rc = need_ws(p);
  if (rc) return rc;
  rc = check_input(p, d_x, ld);
  if (rc) return rc;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  p->launches = 0;
  const bool ev = p->stage_events_on;
  if (ev) DELTA_CUDA_CHECK(cudaEventRecord(p->stage_ev[0], st));
  rc = launch_stft(p, d_x, ld, p->d_X(), st);
  if (rc) return rc;
  if (ev) DELTA_CUDA_CHECK(cudaEventRecord(p->stage_ev[1], st));
  float *au = d_Sauto ? d_Sauto : p->d_auto();
  const bool pairs_wanted = (d_G || d_A || d_P || d_R) && p->lay.Po > 0;
  rc = contract(p, p->d_X(), pairs_wanted ? p->d_S() : nullptr, au, p->d_rsq(), (pairs_wanted && !p->band_on) ? p->d_rnorm() : nullptr, st);
  if (rc) return rc;
  if (ev) DELTA_CUDA_CHECK(cudaEventRecord(p->stage_ev[2], st));
  // zero-lag autocorrelations for rho come from the windowed signal energy the STFT kernel left in wpart (Parseval);
  // with the band-pass filter on, from the filtered autospectra
  if (pairs_wanted && p->band_on) {
    rc = launch_auto_prep(p, au, p->d_rsq(), p->d_rnorm(), st);
    if (rc) return rc;
  }
  if (pairs_wanted) rc = launch_pair(p, p->d_S(), p->d_rsq(), p->d_rnorm(), d_G, d_A, d_P, d_R, st);
  if (rc) return rc;
  if (ev) DELTA_CUDA_CHECK(cudaEventRecord(p->stage_ev[3], st));
  return rc;
}

int delta_plan_set_stage_events(delta_plan *p, void *const *events) {
  if (!p) return DELTA_ERR_INVALID_ARG;
  p->stage_events_on = events != nullptr;
  for (int s = 0; s < 4; ++s) {
    p->stage_ev[s] = events ? reinterpret_cast<cudaEvent_t>(events[s]) : nullptr;
    if (events && !events[s]) { p->stage_events_on = false; return DELTA_ERR_INVALID_ARG; }
  }
  return DELTA_OK;
}

int delta_analyze_shot_host(delta_plan *p, const void *h_x, int32_t n_chunks, void *d_slots, int32_t set_offsets,
                            int32_t n_first, float *d_G, float *d_A, float *d_P, float *d_R, float *d_Sauto,
                            int64_t stride_GAP, int64_t stride_R, int64_t stride_auto, int32_t out_ring, float *h_G,
                            float *h_A, float *h_P, float *h_R, float *h_Sauto, void *stream) {
  int rc = need_ws(p);
  if (rc) return rc;
  if (!h_x || !d_slots || n_chunks < 1 || out_ring < 0) return DELTA_ERR_INVALID_ARG;
  if ((reinterpret_cast<uintptr_t>(d_slots) & 255u) != 0) return DELTA_ERR_ALIGNMENT;
  if ((h_G && !d_G) || (h_A && !d_A) || (h_P && !d_P) || (h_R && !d_R) || (h_Sauto && !d_Sauto)) return DELTA_ERR_INVALID_ARG;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  const Layout &l = p->lay;
  const size_t esz = p->cfg.in_dtype == DELTA_I16 ? 2 : 4;
  const size_t chunk_bytes = (size_t)l.C * l.T * esz;
  const size_t slot_bytes = align_up(chunk_bytes, 256);
  const bool any_host = h_G || h_A || h_P || h_R || h_Sauto;
  // device output set of chunk n: n mod out_ring (out_ring = 0: every chunk its own set, n)
  int nsets = out_ring > 0 ? (out_ring < n_chunks ? out_ring : n_chunks) : n_chunks;
  // a zero stride of a requested output makes all sets one
  if (((d_G || d_A || d_P) && stride_GAP == 0) || (d_R && stride_R == 0) || (d_Sauto && stride_auto == 0)) nsets = 1;
  if (!p->copy_stream) {
    DELTA_CUDA_CHECK(cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking));
    DELTA_CUDA_CHECK(cudaStreamCreateWithFlags(&p->d2h_stream, cudaStreamNonBlocking));
    for (int s = 0; s < 2; ++s) {
      DELTA_CUDA_CHECK(cudaEventCreateWithFlags(&p->ev_copied[s], cudaEventDisableTiming));
      DELTA_CUDA_CHECK(cudaEventCreateWithFlags(&p->ev_consumed[s], cudaEventDisableTiming));
    }
    DELTA_CUDA_CHECK(cudaEventCreateWithFlags(&p->ev_start, cudaEventDisableTiming));
  }
  // one "computed" / "copied back" event pair per output set that is reused (bounded: sets beyond 64 are never reused
  // before the shot ends unless the ring is shorter, and a ring is at most a handful of sets)
  const bool reuse = any_host && nsets < n_chunks;
  if (reuse && nsets > 64) return DELTA_ERR_UNSUPPORTED;
  const int nev = any_host ? (reuse ? nsets : 1) : 0;
  while ((int)p->ev_out.size() < nev) {
    cudaEvent_t a = nullptr, b = nullptr;
    DELTA_CUDA_CHECK(cudaEventCreateWithFlags(&a, cudaEventDisableTiming));
    DELTA_CUDA_CHECK(cudaEventCreateWithFlags(&b, cudaEventDisableTiming));
    p->ev_out.push_back(a);
    p->ev_back.push_back(b);
  }
  // the copy streams must not start before work already queued on `stream` (e.g. a previous shot still reading the
  // slots or the output sets) has finished
  DELTA_CUDA_CHECK(cudaEventRecord(p->ev_start, st));
  DELTA_CUDA_CHECK(cudaStreamWaitEvent(p->copy_stream, p->ev_start, 0));
  if (any_host) DELTA_CUDA_CHECK(cudaStreamWaitEvent(p->d2h_stream, p->ev_start, 0));
  const size_t gap_bytes = (size_t)l.Po * l.F * sizeof(float), r_bytes = (size_t)l.Po * l.nlags * sizeof(float);
  const size_t au_bytes = (size_t)l.C * l.F * sizeof(float);
  int total_launches = 0;
  for (int n = 0; n < n_chunks; ++n) {
    const int s = n & 1;
    char *slot = reinterpret_cast<char *>(d_slots) + (size_t)s * slot_bytes;
    if (n >= 2) DELTA_CUDA_CHECK(cudaStreamWaitEvent(p->copy_stream, p->ev_consumed[s], 0));
    DELTA_CUDA_CHECK(cudaMemcpyAsync(slot, reinterpret_cast<const char *>(h_x) + (size_t)n * chunk_bytes, chunk_bytes,
                                     cudaMemcpyHostToDevice, p->copy_stream));
    DELTA_CUDA_CHECK(cudaEventRecord(p->ev_copied[s], p->copy_stream));
    DELTA_CUDA_CHECK(cudaStreamWaitEvent(st, p->ev_copied[s], 0));
    if (n == 0 && set_offsets) {
      rc = delta_set_offsets(p, slot, l.T, n_first, stream);
      if (rc) return rc;
    }
    const int set = n % nsets;
    // the copy-back of the chunk that used this output set before must be over before the kernels overwrite it
    if (reuse && n >= nsets) DELTA_CUDA_CHECK(cudaStreamWaitEvent(st, p->ev_back[set], 0));
    float *g = d_G ? d_G + (size_t)set * stride_GAP : nullptr, *a = d_A ? d_A + (size_t)set * stride_GAP : nullptr;
    float *pw = d_P ? d_P + (size_t)set * stride_GAP : nullptr, *r = d_R ? d_R + (size_t)set * stride_R : nullptr;
    float *au = d_Sauto ? d_Sauto + (size_t)set * stride_auto : nullptr;
    rc = delta_analyze_chunk(p, slot, l.T, g, a, pw, r, au, stream);
    if (rc) return rc;
    total_launches += p->launches;
    DELTA_CUDA_CHECK(cudaEventRecord(p->ev_consumed[s], st));
    if (any_host) {
      // device -> host on its own stream, so that it runs under the kernels (and the host -> device copy) of the next chunks
      const int e = reuse ? set : 0;
      DELTA_CUDA_CHECK(cudaEventRecord(p->ev_out[e], st));
      DELTA_CUDA_CHECK(cudaStreamWaitEvent(p->d2h_stream, p->ev_out[e], 0));
      cudaStream_t dh = p->d2h_stream;
      if (h_G) DELTA_CUDA_CHECK(cudaMemcpyAsync(h_G + (size_t)n * l.Po * l.F, g, gap_bytes, cudaMemcpyDeviceToHost, dh));
      if (h_A) DELTA_CUDA_CHECK(cudaMemcpyAsync(h_A + (size_t)n * l.Po * l.F, a, gap_bytes, cudaMemcpyDeviceToHost, dh));
      if (h_P) DELTA_CUDA_CHECK(cudaMemcpyAsync(h_P + (size_t)n * l.Po * l.F, pw, gap_bytes, cudaMemcpyDeviceToHost, dh));
      if (h_R) DELTA_CUDA_CHECK(cudaMemcpyAsync(h_R + (size_t)n * l.Po * l.nlags, r, r_bytes, cudaMemcpyDeviceToHost, dh));
      if (h_Sauto) DELTA_CUDA_CHECK(cudaMemcpyAsync(h_Sauto + (size_t)n * l.C * l.F, au, au_bytes, cudaMemcpyDeviceToHost, dh));
      DELTA_CUDA_CHECK(cudaEventRecord(p->ev_back[e], dh));
    }
  }
  if (any_host) {  // `stream` ends after the last copy-back: the caller synchronises one stream
    DELTA_CUDA_CHECK(cudaEventRecord(p->ev_back[0], p->d2h_stream));
    DELTA_CUDA_CHECK(cudaStreamWaitEvent(st, p->ev_back[0], 0));
  }
  p->launches = total_launches;
  return DELTA_OK;
}

int delta_last_launch_count(const delta_plan *p) { return p ? p->launches : 0; }

const char *delta_strerror(int status) {
  switch (status) {
    case DELTA_OK: return "ok";
    case DELTA_ERR_INVALID_ARG: return "invalid argument";
    case DELTA_ERR_UNSUPPORTED: return "unsupported configuration";
    case DELTA_ERR_ALIGNMENT: return "pointer not sufficiently aligned";
    case DELTA_ERR_NO_WORKSPACE: return "workspace missing or too small";
    case DELTA_ERR_CUDA: return "CUDA runtime error (see delta_last_cuda_error)";
    case DELTA_ERR_STATE: return "call sequence error (offsets not set)";
    case DELTA_ERR_NO_MEMORY: return "host memory allocation failed";
    case DELTA_ERR_TOO_LARGE: return "plan needs more scratch than DELTA_STATIC_SCRATCH_BYTES (use delta_coherence)";
    default: return "unknown status";
  }
}

int delta_last_cuda_error(void) { return g_last_cuda_error; }
int delta_version(void) { return DELTA_VERSION; }

}  // extern "C"
