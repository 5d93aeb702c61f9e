"""Float64 checker for FULL-SIZE outputs (test infrastructure, CPU, numpy only).

The oracle (oracle/delta_oracle.py) is a direct DFT with explicit matrices and a Python loop over pairs: at the full
sizes of BASELINE configs 3 and 5 and of the 576-channel workload it would take hours.  oracle/fft_baseline.py computes
the same definitions (default readings only) through numpy's rfft / irfft and matrix products, row block by row block, in
float64.  It is NOT a second oracle: every test that uses this checker first asserts that it agrees with the oracle to
1e-9 on sampled channels of the same input (the library FFT is also one of the oracle's own pins, P6), and only then
uses it to check every output row.  Nothing here imports or shares code with the CUDA path.
"""
from __future__ import annotations

import numpy as np

from oracle import fft_baseline as fb


def check_all_pairs(x: np.ndarray, L: int, H: int, M: int, outs: dict, tol: dict, label: str = "") -> dict:
    """outs: {name: dict(G, A, P, R, Sauto)} -- numpy float32 outputs (all pairs i < j, lexicographic) of one or more runs on
    the same input.  Compares EVERY element of every run with the float64 values, asserts north_star's tolerances and
    returns the maxima per run.  Works row block by row block (all pairs (i, j > i) of one i at a time), so memory
    stays at a few hundred MB, and the float64 values are formed once for all runs."""
    sp = fb.Spectra(x, L, H, M)
    C = sp.C
    stats = {name: dict(auto_rel=0.0, P_rel_gated=0.0, P_abs_norm=0.0, G_abs=0.0, A_gated=0.0, R_abs=0.0, rows=0) for name in outs}
    for name, out in outs.items():
        sa = np.asarray(out["Sauto"], dtype=np.float64)
        stats[name]["auto_rel"] = float(np.max(np.abs(sa - sp.Sauto) / np.maximum(sp.Sauto, 1e-300)))
    for i in range(C - 1):
        p0, n = fb.row_start(i, C), C - 1 - i
        G, A, P, rho = sp.row(i)
        den = np.sqrt(sp.Sauto[i][None, :] * sp.Sauto[i + 1:])
        ok = den > 0
        sden = np.where(ok, den, 1.0)
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
    """All pairs of a (small) channel subset -- for the comparison with the oracle that every test makes first."""
    return fb.analyze_chunk(x, L, H, M)
