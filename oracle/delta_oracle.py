"""Float64 CPU oracle for the all-channel-pairs spectral path of the Delta framework.

TEST INFRASTRUCTURE ONLY.  Nothing on the product path may import, call or execute this
module: only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs do.  It shares no code, table, constant generator, pre- or
post-processing with the CUDA path under ``paper_2108_08896_b200/`` and imports nothing from
it.  It is deliberately plain and slow: float64 throughout, a *direct* DFT through explicit
DFT matrices (no FFT routine), no blocking / fusion / reordering beyond what the definitions
state, so that a reader can check every function against the paper by eye.

What it computes (citations are /root/reference/PAPER.md line numbers):

  * chunk normalisation "After normalizing each chunk, the chunks are streamed" (L107), in the
    reading delta T_e / <T_e> of L89:  y = (x - o_c) / o_c                        -> offsets(), normalise()
  * "short-time Fourier Transformation of each data chunk" (L107, L169)          -> stft()
  * Eq. (1a):  P_XY(w) = E[ X(w) Y^dagger(w) ]   (E = mean over segments)   -> cross_spectra(), auto_spectra(), crosspower()
  * Eq. (1b):  G_XY(w) = |S_XY| / sqrt(S_XX S_YY)                           -> coherence()
  * Eq. (1c): A_XY(w) = arctan(Im S_XY / Re S_XY)  (four-quadrant)         -> crossphase()
  * Eq. (1d): R_XY = IFFT(S_XY)  (normalised, lags -M..M)                  -> crosscorr()
  * "(192 choose 2) = 18336 possible channel pair combinations" (L107)           -> all_pairs(), pair_index()
  * optional band-pass pre-processing filter (L67, L231), reading R19              -> band_mask(), bandpass()

Where the paper is silent the readings of DESIGN.md section 3 (R1..R16) apply; each function
names the reading it uses.  Every convention that affects an output is pinned by
tests/test_oracle_pins.py (closed forms, Parseval, brute-force time-domain correlation,
library special cases, white-noise statistics); no function here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np

# ----------------------------------------------------------------------------------------------
# enumerations mirrored (by value, not by import) from include/delta.h
SCALE_WINPOW, SCALE_NONE, SCALE_DENSITY, SCALE_SPECTRUM = 0, 1, 2, 3
NORM_NONE, NORM_SUBTRACT, NORM_RELATIVE = 0, 1, 2
WIN_HANN, WIN_HAMMING, WIN_RECT, WIN_BLACKMAN = 0, 1, 2, 3
DETREND_NONE, DETREND_CONSTANT = 0, 1


# ----------------------------------------------------------------------------------------------
# channel pairs
def all_pairs(C: int) -> np.ndarray:
    """All (i, j) with i < j in lexicographic order, shape [C(C-1)/2][2]  (reading R9)."""
    return np.array([(i, j) for i in range(C) for j in range(i + 1, C)], dtype=np.int32).reshape(-1, 2)


def pair_index(i: int, j: int, C: int) -> int:
    """Position of (i, j), i < j, in all_pairs(C):  p = i*C - i(i+1)/2 + (j - i - 1)."""
    assert 0 <= i < j < C
    return i * C - (i * (i + 1)) // 2 + (j - i - 1)


# ----------------------------------------------------------------------------------------------
# step 2: offset normalisation (reading R1)
def offsets(x_first: np.ndarray) -> np.ndarray:
    """o_c = mean over the given samples (the first n samples of the SHOT), per channel."""
    x_first = np.asarray(x_first)
    if np.issubdtype(x_first.dtype, np.integer):
        return x_first.astype(np.int64).sum(axis=1).astype(np.float64) / x_first.shape[1]
    return x_first.astype(np.float64).mean(axis=1)


def normalise(x: np.ndarray, o: np.ndarray | None, mode: int) -> np.ndarray:
    """NONE: y = x;  SUBTRACT: y = x - o_c;  RELATIVE: y = (x - o_c)/o_c   (float64)."""
    y = np.asarray(x).astype(np.float64)
    if mode == NORM_NONE:
        return y
    o = np.asarray(o, dtype=np.float64)[:, None]
    if mode == NORM_SUBTRACT:
        return y - o
    if mode == NORM_RELATIVE:
        return (y - o) / o
    raise ValueError("bad norm mode")


# ----------------------------------------------------------------------------------------------
# steps 3-5: segmentation, window, transform (readings R2-R5)
def n_segments(T: int, L: int, H: int) -> int:
    """K = floor((T - L)/H) + 1: no padding, tail dropped (reading R3)."""
    return (T - L) // H + 1


def hann_periodic(L: int) -> np.ndarray:
    """w[n] = 1/2 - 1/2 cos(2 pi n / L), n = 0..L-1  (periodic / DFT-even Hann, reading R4)."""
    n = np.arange(L, dtype=np.float64)
    return 0.5 - 0.5 * np.cos(2.0 * np.pi * n / L)


def window(L: int, kind: int = WIN_HANN) -> np.ndarray:
    """Periodic (DFT-even) windows, n = 0..L-1, x = 2 pi n / L  (the paper names none: R4 default Hann; the others are
    the f1 variants of SURVEY.md section 8f):  Hann 0.5 - 0.5 cos x;  Hamming 0.54 - 0.46 cos x;  rectangular 1;
    Blackman 0.42 - 0.5 cos x + 0.08 cos 2x."""
    x = 2.0 * np.pi * np.arange(L, dtype=np.float64) / L
    if kind == WIN_HANN:
        return hann_periodic(L)
    if kind == WIN_HAMMING:
        return 0.54 - 0.46 * np.cos(x)
    if kind == WIN_RECT:
        return np.ones(L)
    if kind == WIN_BLACKMAN:
        return 0.42 - 0.5 * np.cos(x) + 0.08 * np.cos(2.0 * x)
    raise ValueError("bad window")


def dft_matrix(L: int, nbins: int) -> np.ndarray:
    """W[n, f] = exp(-2 pi i (n f mod L)/L), n < L, f < nbins; phase reduced in integers."""
    n = np.arange(L, dtype=np.int64)[:, None]
    f = np.arange(nbins, dtype=np.int64)[None, :]
    return np.exp(-2j * np.pi * ((n * f) % L).astype(np.float64) / L)


def stft(y: np.ndarray, L: int, H: int, win: int = WIN_HANN, detrend: int = DETREND_NONE,
         nperseg: int | None = None) -> np.ndarray:
    """X[c, k, f] = sum_n w[n] y[c, kH + n] exp(-2 pi i f n / L),  f = 0..L/2, unscaled.

    Default: no detrend (R5); nperseg == nfft (R2), segments never leave the chunk (L107).
    detrend = CONSTANT (f1 variant): the mean of the samples of a segment is subtracted before the window.
    nperseg = Ls < L (f2 variant, R22): segments of Ls samples (window of length Ls), zero-padded to the transform
    length L, so that the circular correlation of Eq. (1d) is the LINEAR one for lags |m| <= L - Ls."""
    y = np.asarray(y, dtype=np.float64)
    C, T = y.shape
    Ls = L if nperseg is None else nperseg
    K = n_segments(T, Ls, H)
    F = L // 2 + 1
    w = window(Ls, win)
    W = dft_matrix(L, F)[:Ls]          # the padded samples are zero: only the first Ls rows of the DFT matrix act
    X = np.empty((C, K, F), dtype=np.complex128)
    for c in range(C):
        seg = np.stack([y[c, k * H:k * H + Ls] for k in range(K)])
        if detrend == DETREND_CONSTANT:
            seg = seg - seg.mean(axis=1, keepdims=True)
        X[c] = (seg * w[None, :]) @ W
    return X


def band_mask(L: int, fs: float, lo_hz: float, hi_hz: float) -> np.ndarray:
    """Pre-processing band-pass of PAPER.md L67 ("optional pre-processing filters"), L231 (the demo's 5-9 kHz pass
    band), in reading R19: an ideal (brick-wall) mask on the bins of every segment's transform.  Bin f (frequency
    f fs / L) is kept iff lo_hz <= f fs / L <= hi_hz, tested as lo_hz L <= f fs <= hi_hz L in float64.
    Returns a boolean [L/2+1] array."""
    f = np.arange(L // 2 + 1, dtype=np.float64)
    return (np.float64(lo_hz) * L <= f * np.float64(fs)) & (f * np.float64(fs) <= np.float64(hi_hz) * L)


def bandpass(X: np.ndarray, mask: np.ndarray) -> np.ndarray:
    """X[c, k, f] with the bins outside the pass band set to zero (R19)."""
    return np.where(mask[None, None, :], X, 0.0)


def scale_factor(L: int, scaling: int = SCALE_WINPOW, fs: float = 1.0, win: int = WIN_HANN,
                 nperseg: int | None = None) -> float:
    """s^2 of step 6 (reading R6): WINPOW 1/sum w^2 (default), NONE 1, DENSITY 1/(fs sum w^2),
    SPECTRUM 1/(sum w)^2.  Two-sided values: no one-sided doubling (R7)."""
    w = window(L if nperseg is None else nperseg, win)
    if scaling == SCALE_WINPOW:
        return 1.0 / float(np.sum(w * w))
    if scaling == SCALE_NONE:
        return 1.0
    if scaling == SCALE_DENSITY:
        return 1.0 / (fs * float(np.sum(w * w)))
    if scaling == SCALE_SPECTRUM:
        return 1.0 / float(np.sum(w)) ** 2
    raise ValueError("bad scaling")


# ----------------------------------------------------------------------------------------------
# step 6: Eq. (1a):  P_XY = E[X Y^dagger], E = mean over the K segments (R8, R10)
def cross_spectra(X: np.ndarray, pairs: np.ndarray, s2: float) -> np.ndarray:
    """S[p, f] = s2 * (1/K) sum_k X[i_p, k, f] * conj(X[j_p, k, f])   (complex128 [P][F])."""
    pairs = np.asarray(pairs).reshape(-1, 2)
    K = X.shape[1]
    S = np.empty((pairs.shape[0], X.shape[2]), dtype=np.complex128)
    for p, (i, j) in enumerate(pairs):
        S[p] = s2 * (X[i] * np.conj(X[j])).sum(axis=0) / K
    return S


def auto_spectra(X: np.ndarray, s2: float) -> np.ndarray:
    """S_cc[f] = s2 * (1/K) sum_k |X[c, k, f]|^2   (float64 [C][F]); denominators of Eq. (1b)."""
    K = X.shape[1]
    return s2 * (X.real ** 2 + X.imag ** 2).sum(axis=1) / K


# step 7: cross-power (north_star: |S_ij|; Eq. 1a gives the complex S)
def crosspower(S: np.ndarray) -> np.ndarray:
    return np.abs(S)


# step 8: Eq. (1b)
def coherence(S: np.ndarray, Sauto: np.ndarray, pairs: np.ndarray) -> np.ndarray:
    """G[p, f] = |S[p, f]| / sqrt(S_ii[f] S_jj[f]); 0 where the denominator is 0 (R16)."""
    pairs = np.asarray(pairs).reshape(-1, 2)
    den = np.sqrt(Sauto[pairs[:, 0]] * Sauto[pairs[:, 1]])
    G = np.zeros_like(den)
    np.divide(np.abs(S), den, out=G, where=den > 0)
    return G


# step 9: Eq. (1c), PAPER.md L100 (garbled in the source; reading R11: four-quadrant arg S)
def crossphase(S: np.ndarray) -> np.ndarray:
    return np.arctan2(S.imag, S.real)


# step 10: Eq. (1d), PAPER.md L102 (reading R12)
def hermitian_extend(S_half: np.ndarray, L: int) -> np.ndarray:
    """[.., L/2+1] one-sided bins -> [.., L] bins with S[L - f] = conj(S[f]), f = 1..L/2-1."""
    full = np.empty(S_half.shape[:-1] + (L,), dtype=np.complex128)
    full[..., :L // 2 + 1] = S_half
    for f in range(1, L // 2):
        full[..., L - f] = np.conj(S_half[..., f])
    return full


def idft_lag_matrix(L: int, M: int) -> np.ndarray:
    """V[f, q] = (1/L) exp(+2 pi i (f m_q mod L)/L), m_q = -M..M (increasing), f = 0..L-1."""
    f = np.arange(L, dtype=np.int64)[:, None]
    m = np.arange(-M, M + 1, dtype=np.int64)[None, :]
    return np.exp(2j * np.pi * ((f * m) % L).astype(np.float64) / L) / L


def crosscorr(S: np.ndarray, Sauto: np.ndarray, pairs: np.ndarray, L: int, M: int) -> np.ndarray:
    """rho[p, q] = R_p[m_q] / sqrt(R_ii[0] R_jj[0]),  m_q = -M..M,
    R_p[m] = (1/L) sum_{f=0}^{L-1} S_p[f] exp(+2 pi i f m / L)  (real part; circular in m),
    R_cc[0] = (1/L) sum_{f=0}^{L-1} S_cc[f];  0 where the denominator is 0."""
    pairs = np.asarray(pairs).reshape(-1, 2)
    V = idft_lag_matrix(L, M)
    R = (hermitian_extend(S, L) @ V).real
    R0 = hermitian_extend(Sauto.astype(np.complex128), L).real.sum(axis=-1) / L
    den = np.sqrt(R0[pairs[:, 0]] * R0[pairs[:, 1]])[:, None]
    rho = np.zeros_like(R)
    np.divide(R, den, out=rho, where=den > 0)
    return rho


# f2 variant: per-segment-normalised coherence.  Eq. (1b), forms the coherence from
# the segment-AVERAGED spectra (reading R10).  The variant used in the field for phase locking normalises every segment
# first: X[c, k, f] -> X / |X| (0 where X = 0), so that S_ij[f] = s2 (1/K) sum_k exp(i (phi_i - phi_j)) is a mean of unit
# phasors, S_cc = s2, and Eq. (1b) gives |mean phasor|: 1 for a phase difference that is the same in every segment, whatever
# the amplitudes do; about sqrt(pi / 4K) for independent segments.
def unit_phasors(X: np.ndarray) -> np.ndarray:
    mag = np.abs(X)
    out = np.zeros_like(X)
    np.divide(X, mag, out=out, where=mag > 0)
    return out


# f2 variant: shot-level accumulation.  The expectation E[.] of Eq. (1a), taken
# over the segments of SEVERAL chunks instead of one: since every chunk has the same K, that is the plain mean of the
# per-chunk spectra.  Coherence, phase and correlation are then formed from the accumulated spectra (R10).
def accumulate(spectra: list) -> np.ndarray:
    """Mean over chunks of per-chunk cross- or auto-spectra (all of one shape)."""
    acc = np.zeros_like(spectra[0])
    for sp in spectra:
        acc = acc + sp
    return acc / len(spectra)


# ----------------------------------------------------------------------------------------------
# the whole path for one chunk, in the paper's order (L107: normalise -> STFT -> Eqs. 1)
def analyze_chunk(x, L, H, M, pairs=None, scaling=SCALE_WINPOW, fs=1.0,
                  norm_mode=NORM_NONE, offs=None, want_S=False, band=None, win=WIN_HANN, detrend=DETREND_NONE,
                  phase_lock=False, nperseg=None):
    """Returns dict(G, A, P, R, Sauto[, S]) for one channel-by-time chunk x[C][T].
    band = (lo_hz, hi_hz): band-pass pre-processing (R19) between the transform and Eq. (1); needs fs."""
    x = np.asarray(x)
    C = x.shape[0]
    if pairs is None:
        pairs = all_pairs(C)
    y = normalise(x, offs, norm_mode)
    X = stft(y, L, H, win, detrend, nperseg)
    if band is not None:
        X = bandpass(X, band_mask(L, fs, band[0], band[1]))
    if phase_lock:
        X = unit_phasors(X)
    s2 = scale_factor(L, scaling, fs, win, nperseg)
    Sauto = auto_spectra(X, s2)
    S = cross_spectra(X, pairs, s2)
    out = dict(G=coherence(S, Sauto, pairs), A=crossphase(S), P=crosspower(S),
               R=crosscorr(S, Sauto, pairs, L, M), Sauto=Sauto)
    if want_S:
        out["S"] = S
        out["X"] = X
    return out
