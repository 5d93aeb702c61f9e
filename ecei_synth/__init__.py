"""Seeded synthetic ECEi-shaped inputs for the five BASELINE.json configurations.

These are stand-ins for KSTAR ECEi shot data, which is not available:
same shapes (24 x 8 = 192 channels, 10,000-sample chunks, 500 kHz), same kind of content
(broadband 1/f^2-type turbulence, spatially correlated over ~2 channels, plus a coherent mode
advected poloidally), generated from numpy's PCG64 with fixed seeds.  The recipe is stated
in DESIGN.md section 4.

This module serves BOTH the oracle-side tests and the CUDA-side tests / bench.  It holds none of
the method's arithmetic (no STFT, no cross-spectra, no coherence ...): it only makes input
arrays.  numpy's FFT is used here purely as a colouring / delay filter for noise synthesis.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

FS = 500e3  # Hz, BASELINE.json configs


@dataclass(frozen=True)
class Workload:
    """Shape parameters of one BASELINE.json configuration."""
    name: str
    C: int
    T: int
    nfft: int
    hop: int
    max_lag: int
    dtype: str  # "f32" | "i16"
    n_chunks: int = 1
    n_first: int = 0  # samples used for the per-shot offsets (config 4)

    @property
    def K(self) -> int:
        return (self.T - self.nfft) // self.hop + 1

    @property
    def F(self) -> int:
        return self.nfft // 2 + 1

    @property
    def P(self) -> int:
        return self.C * (self.C - 1) // 2


WORKLOADS = {
    "tiny": Workload("tiny", 8, 2048, 256, 128, 128, "f32"),
    "single": Workload("single", 192, 10_000, 512, 256, 256, "f32"),
    "long": Workload("long", 192, 100_000, 1024, 512, 512, "f32"),
    "streamed": Workload("streamed", 192, 10_000, 512, 256, 256, "i16", n_chunks=250, n_first=5000),
    "wide": Workload("wide", 384, 50_000, 2048, 512, 1024, "f32"),
}


# ------------------------------------------------------------------------------------------
def tiny(seed: int = 1) -> np.ndarray:
    """Config 1: 8 x 2048 float32, three unit sinusoids (5, 20, 60 kHz) with per-channel phase
    offset 0.3*i rad, plus N(0, sigma = 0.1) noise."""
    w = WORKLOADS["tiny"]
    rng = np.random.Generator(np.random.PCG64(seed))
    t = np.arange(w.T, dtype=np.float64) / FS
    x = np.zeros((w.C, w.T))
    for i in range(w.C):
        for f in (5e3, 20e3, 60e3):
            x[i] += np.sin(2 * np.pi * f * t + 0.3 * i)
    x += 0.1 * rng.standard_normal((w.C, w.T))
    return x.astype(np.float32)


def _grid_cholesky(rows: int = 24, cols: int = 8, corr_len: float = 2.0) -> np.ndarray:
    r = np.repeat(np.arange(rows), cols).astype(np.float64)
    c = np.tile(np.arange(cols), rows).astype(np.float64)
    d2 = (r[:, None] - r[None, :]) ** 2 + (c[:, None] - c[None, :]) ** 2
    sigma = np.exp(-d2 / (2.0 * corr_len ** 2))
    return np.linalg.cholesky(sigma + 1e-6 * np.eye(rows * cols))


def turbulence(T: int, seed: int, rows: int = 24, cols: int = 8, f_knee: float = 1e3,
               mode_f: float = 20e3, mode_bw: float = 1e3, mode_amp: float = 0.5,
               v_pol: float = 5e3, dtype=np.float32) -> np.ndarray:
    """One 24 x 8 array of unit-variance 'turbulence' plus an advected coherent mode.

    white noise -> Lorentzian colouring 1/sqrt(1 + (f/f_knee)^2) with DC removed (PSD ~ 1/f^2
    above the knee) -> Cholesky mixing with Gaussian spatial correlation (length 2 channels)
    -> unit variance per channel; + mode_amp * (white noise band-passed to mode_f +- mode_bw,
    unit variance, delayed per poloidal row by row * (0.40 m / 24) / v_pol).  Returns [192][T].
    """
    C = rows * cols
    rng = np.random.Generator(np.random.PCG64(seed))
    freqs = np.fft.rfftfreq(T, d=1.0 / FS)
    colour = 1.0 / np.sqrt(1.0 + (freqs / f_knee) ** 2)
    colour[0] = 0.0
    g = np.empty((C, T), dtype=np.float32)
    for c in range(C):
        white = rng.standard_normal(T)
        g[c] = np.fft.irfft(np.fft.rfft(white) * colour, n=T)
    Lch = _grid_cholesky(rows, cols).astype(np.float32)
    x = np.empty((C, T), dtype=np.float32)
    blk = 1 << 18
    for t0 in range(0, T, blk):
        x[:, t0:t0 + blk] = Lch @ g[:, t0:t0 + blk]
    del g
    x /= x.std(axis=1, dtype=np.float64)[:, None].astype(np.float32)

    mode_spec = np.fft.rfft(rng.standard_normal(T))
    mode_spec[np.abs(freqs - mode_f) > mode_bw] = 0.0
    base = np.fft.irfft(mode_spec, n=T)
    mode_spec /= base.std()
    tau_row = (0.40 / rows) / v_pol  # seconds per poloidal row
    for r in range(rows):
        delayed = np.fft.irfft(mode_spec * np.exp(-2j * np.pi * freqs * (r * tau_row)), n=T)
        x[r * cols:(r + 1) * cols] += (mode_amp * delayed).astype(np.float32)[None, :]
    return x.astype(dtype, copy=False)


def single(seed: int = 2) -> np.ndarray:
    """Config 2: 192 x 10,000 float32."""
    return turbulence(WORKLOADS["single"].T, seed)


def long(seed: int = 3) -> np.ndarray:
    """Config 3: 192 x 100,000 float32."""
    return turbulence(WORKLOADS["long"].T, seed)


def wide(seed_a: int = 5, seed_b: int = 6) -> np.ndarray:
    """Config 5: 384 x 50,000 float32; array B = 0.3 A + sqrt(0.91) B' (pixel-wise corr. 0.3)."""
    T = WORKLOADS["wide"].T
    a = turbulence(T, seed_a)
    b = turbulence(T, seed_b)
    return np.concatenate([a, (0.3 * a + np.sqrt(0.91) * b).astype(np.float32)], axis=0)


def streamed(seed: int = 4, n_chunks: int = 250) -> tuple[np.ndarray, np.ndarray]:
    """Config 4: int16 digitizer counts, host layout [n_chunks][192][10000] (each chunk one
    contiguous 3.84 MB block), counts = round(o_c + 200 x_c[t]), o_c ~ U(2000, 3000).
    Returns (counts, o_true)."""
    w = WORKLOADS["streamed"]
    T = n_chunks * w.T
    x = turbulence(T, seed)
    rng = np.random.Generator(np.random.PCG64(seed + 1000))
    o = rng.uniform(2000.0, 3000.0, size=w.C)
    counts = np.empty((n_chunks, w.C, w.T), dtype=np.int16)
    for n in range(n_chunks):
        seg = x[:, n * w.T:(n + 1) * w.T].astype(np.float64)
        counts[n] = np.rint(o[:, None] + 200.0 * seg).astype(np.int16)
    return counts, o


def white(C: int, T: int, seed: int, sigma: float = 1.0) -> np.ndarray:
    """Independent white Gaussian channels (for the white-noise coherence pin)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    return (sigma * rng.standard_normal((C, T))).astype(np.float32)


def make(name: str) -> np.ndarray:
    """Input of a named workload (for 'streamed' the first element of streamed())."""
    if name == "tiny":
        return tiny()
    if name == "single":
        return single()
    if name == "long":
        return long()
    if name == "wide":
        return wide()
    if name == "streamed":
        return streamed()[0]
    raise KeyError(name)


# ------------------------------------------------------------------------------------------
# High-dynamic-range stress inputs ("literal 1/f^2 stress case"): they attack the per-channel scale of
# the split-fp16 operands of the tensor-core contraction, whose bins far below a channel's strongest component
# have the fewest significant bits.
def tone_over_floor(C: int, T: int, floor: float, seed: int, f_tone: float = 31.25e3, shared: float = 0.7) -> np.ndarray:
    """Unit-amplitude tone (the same frequency in every channel, phase 0.2 c rad) over a white floor of standard
    deviation `floor`; a fraction `shared` of the floor's amplitude is common to all channels, so that the floor bins
    are coherent (G > 0.1) and their cross-power counts at the relative tolerance."""
    rng = np.random.Generator(np.random.PCG64(seed))
    t = np.arange(T, dtype=np.float64) / FS
    common = rng.standard_normal(T)
    x = np.empty((C, T))
    for c in range(C):
        own = rng.standard_normal(T)
        x[c] = np.sin(2 * np.pi * f_tone * t + 0.2 * c) + floor * (shared * common + np.sqrt(1.0 - shared ** 2) * own)
    return x.astype(np.float32)


def power_law(C: int, T: int, seed: int, exponent: float = 2.0, shared: float = 0.7) -> np.ndarray:
    """Gaussian noise with PSD ~ 1/f^exponent down to the lowest non-zero frequency of the record (no knee, DC
    removed), unit variance; a common component of amplitude fraction `shared` makes all bins coherent."""
    rng = np.random.Generator(np.random.PCG64(seed))
    freqs = np.fft.rfftfreq(T, d=1.0 / FS)
    colour = np.zeros_like(freqs)
    colour[1:] = freqs[1:] ** (-exponent / 2.0)

    def coloured():
        g = np.fft.irfft(np.fft.rfft(rng.standard_normal(T)) * colour, n=T)
        return g / g.std()

    common = coloured()
    x = np.empty((C, T))
    for c in range(C):
        x[c] = shared * common + np.sqrt(1.0 - shared ** 2) * coloured()
    return x.astype(np.float32)
