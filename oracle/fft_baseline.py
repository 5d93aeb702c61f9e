"""Second CPU arm: the float64 pipeline of the oracle with numpy's FFT in place of the direct DFT.

TEST / BASELINE INFRASTRUCTURE ONLY (same rule as delta_oracle.py: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import it; it shares no code with the CUDA path).

It is NOT the oracle: the oracle is delta_oracle.py (direct DFT, definitions written out).  This module exists because
(a) BASELINE.md section 3 asks for an honest CPU figure next to the deliberately slow oracle ("CPU, library FFT"), and
(b) the full-size parity tests need every output row in float64, which the oracle's Python loop over pairs cannot
deliver in minutes.  Every user first checks it against the oracle (tests/test_oracle_pins.py::test_fft_baseline_*,
and each full-size test on sampled channels of its own input).  Default readings only: periodic
Hann, no detrend, WINPOW scaling, no normalisation, all pairs i < j in lexicographic order.
"""
from __future__ import annotations

import numpy as np


def hann(L: int) -> np.ndarray:
    return 0.5 - 0.5 * np.cos(2.0 * np.pi * np.arange(L) / L)


def stft(x: np.ndarray, L: int, H: int) -> np.ndarray:
    """X[c, k, f] = rfft(hann_periodic * x[c, kH : kH+L]), complex128 [C][K][F]."""
    x = np.asarray(x, dtype=np.float64)
    C, T = x.shape
    K = (T - L) // H + 1
    w = hann(L)
    idx = (np.arange(K) * H)[:, None] + np.arange(L)[None, :]
    X = np.empty((C, K, L // 2 + 1), dtype=np.complex128)
    for c in range(C):
        X[c] = np.fft.rfft(x[c][idx] * w[None, :], axis=1)
    return X


def row_start(i: int, C: int) -> int:
    """Lexicographic index of pair (i, i+1)."""
    return i * C - (i * (i + 1)) // 2


class Spectra:
    """Autospectra of a chunk and, row by row (all pairs (i, j > i) of one i), Eq. (1a)-(1d) of PAPER.md L95-103."""

    def __init__(self, x: np.ndarray, L: int, H: int, M: int):
        X = stft(x, L, H)
        self.C, self.K, self.F = X.shape
        self.L, self.M = L, M
        self.s2 = 1.0 / float(np.sum(hann(L) ** 2))
        self.Sauto = self.s2 * (X.real ** 2 + X.imag ** 2).sum(axis=1) / self.K          # [C][F]
        # zero-lag autocorrelation: (1/L) sum over all L bins of the Hermitian extension
        self.R0 = np.concatenate([self.Sauto, self.Sauto[:, -2:0:-1]], axis=1).sum(axis=1) / L
        self.Xf = np.ascontiguousarray(X.transpose(2, 0, 1))                              # [F][C][K]
        self.lag_idx = np.arange(-M, M + 1) % L

    def row(self, i: int):
        """(G, A, P, rho) for the pairs (i, j), j = i+1 .. C-1: float64 [C-1-i][F] x 3 and [C-1-i][2M+1]."""
        L = self.L
        # S[j, f] = s2/K sum_k X[i,k,f] conj X[j,k,f]   (batched matrix-vector products over the bins)
        S = (self.s2 / self.K) * np.matmul(np.conj(self.Xf[:, i + 1:, :]), self.Xf[:, i, :, None])[..., 0].T
        den = np.sqrt(self.Sauto[i][None, :] * self.Sauto[i + 1:])
        ok = den > 0
        P = np.abs(S)
        G = np.where(ok, P / np.where(ok, den, 1.0), 0.0)
        A = np.arctan2(S.imag, S.real)
        Sfull = np.concatenate([S, np.conj(S[:, -2:0:-1])], axis=1)
        Sfull[:, 0] = Sfull[:, 0].real
        Sfull[:, L // 2] = Sfull[:, L // 2].real
        Rfull = np.fft.ifft(Sfull, axis=1).real
        dR = np.sqrt(self.R0[i] * self.R0[i + 1:])[:, None]
        rho = np.where(dR > 0, Rfull[:, self.lag_idx] / np.where(dR > 0, dR, 1.0), 0.0)
        return G, A, P, rho


def analyze_chunk(x: np.ndarray, L: int, H: int, M: int) -> dict:
    """dict(G, A, P, R, Sauto) for all pairs of x (use on small channel counts, or for timing)."""
    sp = Spectra(x, L, H, M)
    rows = [sp.row(i) for i in range(sp.C - 1)]
    cat = lambda k, width: np.concatenate([r[k] for r in rows]) if rows else np.zeros((0, width))
    return dict(G=cat(0, sp.F), A=cat(1, sp.F), P=cat(2, sp.F), R=cat(3, 2 * M + 1), Sauto=sp.Sauto)
