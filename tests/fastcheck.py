"""Float64 checker for FULL-SIZE outputs (test infrastructure, CPU, numpy only).

The oracle (oracle/delta_oracle.py) is a direct DFT with explicit matrices and a Python loop over pairs: at the full
sizes of BASELINE configs 3 and 5 and of the 576-channel workload it would take hours.  This module computes the same
definitions (default readings only: Hann, no detrend, WINPOW scaling, no normalisation) through
numpy's rfft / irfft and matrix products, block by block over the pairs, in float64.  It is NOT a second oracle: every
test that uses it first asserts that it agrees with the oracle to 1e-9 on sampled channels of the same input (the
library FFT is also one of the oracle's own pins, P6), and only then uses it to check every output row.

It shares no code with the CUDA path and imports nothing from it.
"""
from __future__ import annotations

import numpy as np


def stft(x: np.ndarray, L: int, H: int) -> np.ndarray:
    """X[c, k, f] = rfft(hann_periodic * x[c, kH : kH+L]), float64 / complex128, [C][K][F]."""
    x = np.asarray(x, dtype=np.float64)
    C, T = x.shape
    K = (T - L) // H + 1
    w = 0.5 - 0.5 * np.cos(2.0 * np.pi * np.arange(L) / L)
    idx = (np.arange(K) * H)[:, None] + np.arange(L)[None, :]
    X = np.empty((C, K, L // 2 + 1), dtype=np.complex128)
    for c in range(C):
        X[c] = np.fft.rfft(x[c][idx] * w[None, :], axis=1)
    return X


def row_start(i: int, C: int) -> int:
    return i * C - (i * (i + 1)) // 2


def check_all_pairs(x: np.ndarray, L: int, H: int, M: int, outs: dict, tol: dict, label: str = "") -> dict:
    """outs: {name: dict(G, A, P, R, Sauto)} -- numpy float32 outputs (all pairs i < j, lexicographic) of one or more runs on
    the same input.  Compares EVERY element of every run with the float64 values, asserts north_star's tolerances and
    returns the maxima per run.  Works row block by row block (all pairs (i, j > i) of one i at a time), so memory
    stays at a few hundred MB, and the float64 values are formed once for all runs."""
    C = x.shape[0]
    X = stft(x, L, H)                      # [C][K][F]
    K = X.shape[1]
    w = 0.5 - 0.5 * np.cos(2.0 * np.pi * np.arange(L) / L)
    s2 = 1.0 / np.sum(w * w)
    Sauto = s2 * (X.real ** 2 + X.imag ** 2).sum(axis=1) / K          # [C][F]
    R0 = np.concatenate([Sauto, Sauto[:, -2:0:-1]], axis=1).sum(axis=1) / L   # Hermitian extension of the autospectra
    stats = {name: dict(auto_rel=0.0, P_rel_gated=0.0, P_abs_norm=0.0, G_abs=0.0, A_gated=0.0, R_abs=0.0, rows=0) for name in outs}
    for name, out in outs.items():
        sa = np.asarray(out["Sauto"], dtype=np.float64)
        stats[name]["auto_rel"] = float(np.max(np.abs(sa - Sauto) / np.maximum(Sauto, 1e-300)))
    Xf = np.ascontiguousarray(X.transpose(2, 0, 1))                     # [F][C][K]
    del X
    lag_idx = (np.arange(-M, M + 1) % L)
    for i in range(C - 1):
        p0, n = row_start(i, C), C - 1 - i
        # S[j, f] = s2/K sum_k X[i,k,f] conj X[j,k,f], j = i+1 .. C-1   (batched matrix-vector products over the bins)
        S = (s2 / K) * np.matmul(np.conj(Xf[:, i + 1:, :]), Xf[:, i, :, None])[..., 0].T
        den = np.sqrt(Sauto[i][None, :] * Sauto[i + 1:])
        ok = den > 0
        sden = np.where(ok, den, 1.0)
        P = np.abs(S)
        G = np.where(ok, P / sden, 0.0)
        A = np.arctan2(S.imag, S.real)
        Sfull = np.concatenate([S, np.conj(S[:, -2:0:-1])], axis=1)
        Sfull[:, 0] = Sfull[:, 0].real
        Sfull[:, L // 2] = Sfull[:, L // 2].real
        Rfull = np.fft.ifft(Sfull, axis=1).real
        dR = np.sqrt(R0[i] * R0[i + 1:])[:, None]
        rho = np.where(dR > 0, Rfull[:, lag_idx] / np.where(dR > 0, dR, 1.0), 0.0)
        sl = slice(p0, p0 + n)
        gate = G > 0.1
        for name, out in outs.items():
            st = stats[name]
            dP = np.abs(np.asarray(out["P"][sl], dtype=np.float64) - P)
            st["P_rel_gated"] = max(st["P_rel_gated"], float(np.max(np.where(gate, dP / np.maximum(P, 1e-300), 0.0))))
            st["P_abs_norm"] = max(st["P_abs_norm"], float(np.max(np.where(ok, dP / sden, 0.0))))
            st["G_abs"] = max(st["G_abs"], float(np.max(np.abs(np.asarray(out["G"][sl], dtype=np.float64) - G))))
            dA = np.abs(np.angle(np.exp(1j * (np.asarray(out["A"][sl], dtype=np.float64) - A))))
            st["A_gated"] = max(st["A_gated"], float(np.max(np.where(gate, dA, 0.0))))
            st["R_abs"] = max(st["R_abs"], float(np.max(np.abs(np.asarray(out["R"][sl], dtype=np.float64) - rho))))
            st["rows"] += n
    for name, st in stats.items():
        lab = f"{label} [{name}]"
        assert st["rows"] == C * (C - 1) // 2
        assert st["auto_rel"] <= tol["P_rel"], f"{lab}: autospectra rel err {st['auto_rel']:.3g}"
        assert st["P_rel_gated"] <= tol["P_rel"], f"{lab}: cross-power rel err (G>0.1) {st['P_rel_gated']:.3g}"
        assert st["P_abs_norm"] <= tol["P_abs"], f"{lab}: cross-power abs err / sqrt(SiiSjj) {st['P_abs_norm']:.3g}"
        assert st["G_abs"] <= tol["G"], f"{lab}: coherence abs err {st['G_abs']:.3g}"
        assert st["A_gated"] <= tol["A"], f"{lab}: cross-phase err (G>0.1) {st['A_gated']:.3g}"
        assert st["R_abs"] <= tol["R"], f"{lab}: cross-correlation abs err {st['R_abs']:.3g}"
    return stats


def analyze_sampled(x: np.ndarray, L: int, H: int, M: int) -> dict:
    """The same quantities for ALL pairs of a (small) channel subset, as plain arrays -- for the comparison with the
    oracle that every test makes before it trusts check_all_pairs."""
    C = x.shape[0]
    X = stft(x, L, H)
    K = X.shape[1]
    w = 0.5 - 0.5 * np.cos(2.0 * np.pi * np.arange(L) / L)
    s2 = 1.0 / np.sum(w * w)
    Sauto = s2 * (X.real ** 2 + X.imag ** 2).sum(axis=1) / K
    R0 = np.concatenate([Sauto, Sauto[:, -2:0:-1]], axis=1).sum(axis=1) / L
    G, A, P, R = [], [], [], []
    lag_idx = (np.arange(-M, M + 1) % L)
    for i in range(C - 1):
        S = s2 / K * np.einsum("kf,jkf->jf", X[i], np.conj(X[i + 1:]))
        den = np.sqrt(Sauto[i][None, :] * Sauto[i + 1:])
        P.append(np.abs(S)); G.append(np.abs(S) / den); A.append(np.arctan2(S.imag, S.real))
        Sfull = np.concatenate([S, np.conj(S[:, -2:0:-1])], axis=1)
        Sfull[:, 0] = Sfull[:, 0].real
        Sfull[:, L // 2] = Sfull[:, L // 2].real
        R.append(np.fft.ifft(Sfull, axis=1).real[:, lag_idx] / np.sqrt(R0[i] * R0[i + 1:])[:, None])
    return dict(G=np.concatenate(G), A=np.concatenate(A), P=np.concatenate(P), R=np.concatenate(R), Sauto=Sauto)
