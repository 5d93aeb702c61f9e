"""Pins for the float64 oracle (oracle/delta_oracle.py) against things other than itself.

The paper prints no spectral values (PAPER.md gives only Eq. 1a-1d, and structural
constants, L107), so the oracle is pinned by closed forms, invariants, brute-force time-domain
restatements, independent library routines (numpy.fft / scipy.signal, which are neither the
oracle nor the CUDA path) and white-noise statistics.  Each pin names the mistake it would catch.
Pin numbers P1..P10 follow DESIGN.md section 5.
"""
import os

import numpy as np
import pytest
import scipy.signal as sps

import ecei_synth as es
from oracle import delta_oracle as o

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def read_constants():
    out = {}
    with open(os.path.join(GOLDEN, "paper_constants.txt")) as fh:
        for line in fh:
            line = line.split("#")[0].split()
            if len(line) == 2:
                out[line[0]] = int(line[1])
    return out


# ---------------------------------------------------------------------------- paper constants
def test_paper_structural_constants():
    c = read_constants()
    assert c["grid_rows"] * c["grid_cols"] == c["n_channels"]
    assert len(o.all_pairs(c["n_channels"])) == c["n_pairs"]
    assert c["shot_samples"] // c["chunk_samples"] == c["shot_chunks"]
    # segmentation rule (no padding, tail dropped) is the only one that gives BASELINE's counts
    assert o.n_segments(2048, 256, 128) == c["tiny_segments"]
    assert o.n_segments(100_000, 1024, 512) == c["long_segments"]
    assert len(o.all_pairs(384)) == c["wide_pairs"]
    assert len(o.all_pairs(8)) == c["tiny_pairs"]
    # the workload table of the input module agrees
    assert es.WORKLOADS["single"].P == c["n_pairs"] and es.WORKLOADS["single"].K == 38
    assert es.WORKLOADS["wide"].K == 94 and es.WORKLOADS["long"].K == c["long_segments"]


def test_pair_index_is_lexicographic():
    for C in (2, 3, 8, 17):
        pairs = o.all_pairs(C)
        for p, (i, j) in enumerate(pairs):
            assert i < j and o.pair_index(int(i), int(j), C) == p
        assert len(pairs) == C * (C - 1) // 2


# ---------------------------------------------------------------------------- window
@pytest.mark.parametrize("L", [64, 256, 512, 2048])
def test_hann_closed_forms(L):
    w = o.hann_periodic(L)
    assert abs(w.sum() - L / 2) < 1e-9 * L          # sum w   = L/2
    assert abs((w * w).sum() - 3 * L / 8) < 1e-9 * L  # sum w^2 = 3L/8
    assert w[0] == 0.0 and abs(w[L // 2] - 1.0) < 1e-15
    assert np.allclose(w[1:], w[1:][::-1], atol=1e-15)  # periodic: symmetric about L/2, w[L]=w[0]
    assert abs(o.scale_factor(L) - 8.0 / (3 * L)) < 1e-15
    # overlap correlation at 50 %: sum_n w[n] w[n+L/2] = L/16  ->  r_1 = 1/6
    assert abs((w[:L // 2] * w[L // 2:]).sum() / (w * w).sum() - 1.0 / 6.0) < 1e-12


# ---------------------------------------------------------------------------- P1: closed form
@pytest.mark.parametrize("L,H,q", [(256, 128, 10), (256, 64, 37), (512, 256, 5), (128, 100, 20)])
def test_P1_bin_centred_tone_closed_form(L, H, q):
    """x_i[t] = cos(2 pi q t / L + phi_i): |X[q]| = L/4, |X[q+-1]| = L/8, all other bins 0;
    S_ij[q] = s2 (L/4)^2 e^{i(phi_i - phi_j)}, G = 1, A = phi_i - phi_j.
    Catches: symmetric instead of periodic Hann, wrong DFT sign, conj on the wrong operand,
    wrong scaling, averaging mistakes, wrong hop handling."""
    T = 4 * L + 3 * H + 7
    t = np.arange(T)
    phi = np.array([0.4, -0.7, 2.9])
    x = np.stack([np.cos(2 * np.pi * q * t / L + p) for p in phi])
    X = o.stft(x, L, H)
    K = o.n_segments(T, L, H)
    assert X.shape == (3, K, L // 2 + 1)
    mag = np.abs(X)
    assert np.allclose(mag[:, :, q], L / 4, atol=1e-9)
    assert np.allclose(mag[:, :, q - 1], L / 8, atol=1e-9)
    assert np.allclose(mag[:, :, q + 1], L / 8, atol=1e-9)
    rest = np.delete(mag, [q - 1, q, q + 1], axis=2)
    assert rest.max() < 1e-10
    # phase of X at segment k: phi + 2 pi q k H / L
    for k in range(K):
        d = np.angle(X[:, k, q] * np.exp(-1j * (phi + 2 * np.pi * q * k * H / L)))
        assert np.abs(d).max() < 1e-10
    s2 = o.scale_factor(L)
    pairs = o.all_pairs(3)
    S = o.cross_spectra(X, pairs, s2)
    Sa = o.auto_spectra(X, s2)
    for p, (i, j) in enumerate(pairs):
        expect = s2 * (L / 4) ** 2 * np.exp(1j * (phi[i] - phi[j]))
        assert abs(S[p, q] - expect) < 1e-9 * abs(expect)
    G = o.coherence(S, Sa, pairs)
    A = o.crossphase(S)
    assert np.allclose(G[:, q], 1.0, atol=1e-12)
    dphi = np.array([phi[i] - phi[j] for i, j in pairs])
    assert np.abs(np.angle(np.exp(1j * (A[:, q] - dphi)))).max() < 1e-10
    assert np.allclose(Sa[:, q], s2 * (L / 4) ** 2, rtol=1e-10)
    assert np.allclose(o.crosspower(S)[:, q], s2 * (L / 4) ** 2, rtol=1e-10)


# ---------------------------------------------------------------------------- P2, P3
def _rand_chunk(C=5, T=1500, seed=11):
    return np.random.default_rng(seed).standard_normal((C, T))


def test_P2_self_coherence_and_P3_hermitian_symmetry():
    """G_ii = 1, rho_ii[0] = 1, A_ii = 0;  S_ji = conj S_ij => P, G symmetric, A_ji = -A_ij,
    rho_ji[m] = rho_ij[-m].  Catches pair-handling and lag-ordering mistakes."""
    L, H, M = 128, 64, 64
    x = _rand_chunk()
    X = o.stft(x, L, H)
    s2 = o.scale_factor(L)
    Sa = o.auto_spectra(X, s2)
    self_pairs = np.array([(c, c) for c in range(5)])
    S = o.cross_spectra(X, self_pairs, s2)
    assert np.allclose(S.real, Sa, rtol=1e-12) and np.abs(S.imag).max() < 1e-12
    assert np.allclose(o.coherence(S, Sa, self_pairs), 1.0, atol=1e-12)
    assert np.abs(o.crossphase(S)).max() < 1e-12
    rho = o.crosscorr(S, Sa, self_pairs, L, M)
    assert np.allclose(rho[:, M], 1.0, atol=1e-12)
    assert np.abs(rho).max() <= 1.0 + 1e-12
    fwd = np.array([(0, 3), (1, 4), (2, 3)])
    rev = fwd[:, ::-1]
    Sf, Sr = o.cross_spectra(X, fwd, s2), o.cross_spectra(X, rev, s2)
    assert np.allclose(Sr, np.conj(Sf), rtol=1e-13)
    assert np.allclose(o.coherence(Sf, Sa, fwd), o.coherence(Sr, Sa, rev))
    assert np.allclose(o.crossphase(Sr)[:, 1:-1], -o.crossphase(Sf)[:, 1:-1])
    rf, rr = o.crosscorr(Sf, Sa, fwd, L, M), o.crosscorr(Sr, Sa, rev, L, M)
    assert np.allclose(rr, rf[:, ::-1], atol=1e-13)
    assert np.abs(rf).max() <= 1.0 + 1e-12  # Cauchy-Schwarz


# ---------------------------------------------------------------------------- P4: Parseval
def test_P4_parseval_per_segment_and_lag0():
    """|X0|^2 + 2 sum |Xf|^2 + |X_{L/2}|^2 = L sum (w y)^2 for every segment, and
    R_ii[0] = s2 (1/K) sum_k sum_n (w y)^2.  Catches a wrong DFT kernel / dropped bins /
    one-sided doubling / wrong 1/L in the inverse."""
    L, H = 256, 96
    x = _rand_chunk(3, 2000, 5)
    X = o.stft(x, L, H)
    w = o.hann_periodic(L)
    K = X.shape[1]
    e_seg = np.empty((3, K))
    for c in range(3):
        for k in range(K):
            e_seg[c, k] = ((w * x[c, k * H:k * H + L]) ** 2).sum()
    p = np.abs(X) ** 2
    lhs = p[:, :, 0] + 2 * p[:, :, 1:L // 2].sum(axis=2) + p[:, :, L // 2]
    assert np.allclose(lhs, L * e_seg, rtol=1e-12)
    s2 = o.scale_factor(L)
    Sa = o.auto_spectra(X, s2)
    R0 = o.hermitian_extend(Sa.astype(complex), L).real.sum(axis=1) / L
    assert np.allclose(R0, s2 * e_seg.mean(axis=1), rtol=1e-12)
    # un-normalised R_ii[0] through crosscorr's own path: rho * R0
    sp = np.array([(0, 0), (0, 1)])
    S = o.cross_spectra(X, sp, s2)
    rho = o.crosscorr(S, Sa, sp, L, 4)
    assert abs(rho[0, 4] - 1.0) < 1e-12


# ---------------------------------------------------------------------------- P5: brute force
def test_P5_time_domain_circular_correlation_and_lag_sign():
    """R_ij[m] = s2 (1/K) sum_k sum_n yh_i,k[(n+m) mod L] yh_j,k[n], yh = windowed segment.
    And: if channel j is channel i delayed by d samples, rho_ij peaks at m = -d and
    A_ij[f] = +2 pi f d / L.  Catches a wrong sign/conjugate in Eq. 1a or 1d, wrong lag order,
    missing Hermitian half, wrong 1/L."""
    L, H, M = 64, 32, 32
    x = _rand_chunk(3, 400, 2)
    K = o.n_segments(400, L, H)
    w = o.hann_periodic(L)
    s2 = o.scale_factor(L)
    pairs = np.array([(0, 1), (1, 2), (0, 2), (0, 0), (1, 1), (2, 2)])
    X = o.stft(x, L, H)
    S = o.cross_spectra(X, pairs, s2)
    Sa = o.auto_spectra(X, s2)
    rho = o.crosscorr(S, Sa, pairs, L, M)
    Rb = np.zeros((len(pairs), 2 * M + 1))
    for p, (i, j) in enumerate(pairs):
        for q, m in enumerate(range(-M, M + 1)):
            acc = 0.0
            for k in range(K):
                yi = w * x[i, k * H:k * H + L]
                yj = w * x[j, k * H:k * H + L]
                for n in range(L):
                    acc += yi[(n + m) % L] * yj[n]
            Rb[p, q] = s2 * acc / K
    r0 = {c: Rb[3 + c, M] for c in range(3)}
    for p, (i, j) in enumerate(pairs):
        assert np.allclose(rho[p], Rb[p] / np.sqrt(r0[i] * r0[j]), atol=1e-12)
    # delayed copy
    d = 5
    T = 4000
    base = np.random.default_rng(9).standard_normal(T + d)
    xi, xj = base[d:], base[:T]          # x_j[t] = x_i[t - d]
    xx = np.stack([xi, xj])
    L, H, M = 128, 64, 64
    r = o.analyze_chunk(xx, L, H, M)
    assert np.argmax(r["R"][0]) - M == -d
    f = np.arange(1, L // 2)
    sel = r["G"][0, 1:L // 2] > 0.8
    err = np.angle(np.exp(1j * (r["A"][0, 1:L // 2] - 2 * np.pi * f * d / L)))
    assert sel.sum() > 10 and np.abs(err[sel]).max() < 0.2


# ---------------------------------------------------------------------------- P6: library
@pytest.mark.parametrize("L,H", [(256, 128), (512, 128), (128, 96)])
def test_P6_library_special_cases(L, H):
    """numpy rfft / scipy Welch routines are independent code.  Oracle X == rfft(w * segment);
    scipy csd(x_i, x_j) (density, fs = 1, two-sided, no detrend) == conj(S_ij) [scipy conjugates
    its FIRST argument]; 'spectrum' scaling == conj(S_ij) sum w^2/(sum w)^2; scipy coherence
    == G^2.  Catches any deviation of the oracle from the standard Welch estimator."""
    x = _rand_chunk(4, 3000, 21)
    C, T = x.shape
    K = o.n_segments(T, L, H)
    X = o.stft(x, L, H)
    w = o.hann_periodic(L)
    assert np.allclose(w, sps.get_window("hann", L, fftbins=True), atol=1e-15)
    for c in range(C):
        for k in (0, K // 2, K - 1):
            ref = np.fft.rfft(w * x[c, k * H:k * H + L])
            assert np.allclose(X[c, k], ref, rtol=1e-10, atol=1e-10)
    pairs = o.all_pairs(C)
    s2 = o.scale_factor(L)
    S = o.cross_spectra(X, pairs, s2)
    Sa = o.auto_spectra(X, s2)
    G = o.coherence(S, Sa, pairs)
    kw = dict(fs=1.0, window="hann", nperseg=L, noverlap=L - H, nfft=L, detrend=False,
              return_onesided=False)
    F = L // 2 + 1
    for p, (i, j) in enumerate(pairs):
        _, Pd = sps.csd(x[i], x[j], scaling="density", **kw)
        assert np.allclose(np.conj(Pd[:F]), S[p], rtol=1e-9, atol=1e-12)
        _, Ps = sps.csd(x[i], x[j], scaling="spectrum", **kw)
        assert np.allclose(np.conj(Ps[:F]), S[p] * (w * w).sum() / w.sum() ** 2, rtol=1e-9, atol=1e-12)
        _, Coh = sps.coherence(x[i], x[j], fs=1.0, window="hann", nperseg=L, noverlap=L - H,
                               nfft=L, detrend=False)
        assert np.allclose(Coh, G[p] ** 2, rtol=1e-9, atol=1e-12)
    # scaling options against scipy's definitions
    Ssp = o.cross_spectra(X, pairs[:1], o.scale_factor(L, o.SCALE_SPECTRUM))
    _, Ps = sps.csd(x[0], x[1], scaling="spectrum", **kw)
    assert np.allclose(np.conj(Ps[:F]), Ssp[0], rtol=1e-9, atol=1e-12)
    fs = 500e3
    Sd = o.cross_spectra(X, pairs[:1], o.scale_factor(L, o.SCALE_DENSITY, fs))
    kw2 = dict(kw, fs=fs)
    _, Pd = sps.csd(x[0], x[1], scaling="density", **kw2)
    assert np.allclose(np.conj(Pd[:F]), Sd[0], rtol=1e-9, atol=1e-18)
    # inverse transform against numpy irfft (circular lags)
    M = L // 2
    rho = o.crosscorr(S, Sa, pairs, L, M)
    R0 = np.fft.irfft(Sa, n=L)[:, 0]
    for p, (i, j) in enumerate(pairs):
        Sp = S[p].copy()
        r = np.fft.irfft(Sp, n=L)
        lag = np.array([r[m % L] for m in range(-M, M + 1)]) / np.sqrt(R0[i] * R0[j])
        assert np.allclose(rho[p], lag, atol=1e-12)


# ---------------------------------------------------------------------------- P7: config 1
def test_P7_injected_phase_offsets_tiny_config():
    """BASELINE config 1: A_ij = 0.3 (i - j) at the tone bins; coherence there >= 0.999."""
    wl = es.WORKLOADS["tiny"]
    x = es.tiny()
    assert x.shape == (8, 2048) and x.dtype == np.float32
    r = o.analyze_chunk(x, wl.nfft, wl.hop, wl.max_lag)
    assert r["G"].shape == (28, 129) and r["R"].shape == (28, 257) and r["Sauto"].shape == (8, 129)
    pairs = o.all_pairs(8)
    expect = np.array([0.3 * (i - j) for i, j in pairs])
    for b in (10, 31):   # 20 kHz -> bin 10.24, 60 kHz -> bin 30.72 (nearest bins)
        assert np.abs(np.angle(np.exp(1j * (r["A"][:, b] - expect)))).max() < 2e-2
        assert r["G"][:, b].min() > 0.999
    # noise-free version: tight
    t = np.arange(2048) / es.FS
    xn = np.stack([sum(np.sin(2 * np.pi * f * t + 0.3 * i) for f in (5e3, 20e3, 60e3)) for i in range(8)])
    rn = o.analyze_chunk(xn, 256, 128, 128)
    for b, tol in ((3, 1e-3), (10, 1e-5), (31, 1e-5)):
        assert np.abs(np.angle(np.exp(1j * (rn["A"][:, b] - expect)))).max() < tol


# ---------------------------------------------------------------------------- P8: white noise
def _welch_phi(L, H, K):
    w = o.hann_periodic(L)
    phi = 1.0
    s = 1
    while s * H < L and s < K:
        r = (w[:L - s * H] * w[s * H:]).sum() / (w * w).sum()
        phi += 2 * (1 - s / K) * r * r
        s += 1
    return phi


@pytest.mark.parametrize("L,H,T,expect", [(256, 128, 2048, 0.235), (512, 256, 10_000, 0.148),
                                          (2048, 512, 50_000, 0.1265)])
def test_P8_independent_white_noise(L, H, T, expect):
    """E S_ii = sigma^2 under WINPOW scaling; mean coherence of independent channels
    = sqrt(pi phi / 4K) with Welch's overlap factor phi (about 1/sqrt(K_segments)).
    Catches wrong averaging (sum vs mean), wrong scaling, coherence formed before averaging."""
    sigma = 0.7
    C = 24
    x = es.white(C, T, seed=77, sigma=sigma)
    K = o.n_segments(T, L, H)
    X = o.stft(x, L, H)
    s2 = o.scale_factor(L)
    Sa = o.auto_spectra(X, s2)
    assert abs(Sa[:, 2:-2].mean() / sigma ** 2 - 1.0) < 0.02
    pairs = o.all_pairs(C)
    G = o.coherence(o.cross_spectra(X, pairs, s2), Sa, pairs)[:, 2:-2]
    theory = np.sqrt(np.pi * _welch_phi(L, H, K) / (4 * K))
    assert abs(theory - expect) < 2e-3            # closed form reproduces DESIGN.md's numbers
    assert abs(G.mean() / theory - 1.0) < 0.03
    assert 0.6 / np.sqrt(K) < G.mean() < 1.4 / np.sqrt(K)   # north_star: "near 1/sqrt(K_segments)"


# ---------------------------------------------------------------------------- P10: scale laws
def test_P10_scale_laws():
    L, H, M = 128, 64, 64
    x = _rand_chunk(3, 1200, 3)
    a = -2.5
    x2 = x.copy()
    x2[1] *= a
    r1, r2 = o.analyze_chunk(x, L, H, M), o.analyze_chunk(x2, L, H, M)
    pairs = o.all_pairs(3)
    for p, (i, j) in enumerate(pairs):
        touched = 1 in (i, j)
        assert np.allclose(r2["G"][p], r1["G"][p], atol=1e-12)
        assert np.allclose(r2["P"][p], r1["P"][p] * (abs(a) if touched else 1.0), rtol=1e-12)
        if touched:   # negative scale: phase shifts by pi, correlation flips
            d = np.angle(np.exp(1j * (r2["A"][p] - r1["A"][p] - np.pi)))
            assert np.abs(d[1:-1]).max() < 1e-9
            assert np.allclose(r2["R"][p], -r1["R"][p], atol=1e-12)
        else:
            assert np.allclose(r2["A"][p], r1["A"][p]) and np.allclose(r2["R"][p], r1["R"][p])


# ---------------------------------------------------------------------------- normalisation (step 2)
def test_offset_normalisation_int16():
    """y = (x - o_c)/o_c with o_c = mean of the first n samples (reading R1)."""
    rng = np.random.default_rng(4)
    o_true = np.array([2100.0, 2950.0])
    sig = rng.standard_normal((2, 6000))
    counts = np.rint(o_true[:, None] + 200 * sig).astype(np.int16)
    offs = o.offsets(counts[:, :5000])
    # integer-exact mean
    for c in range(2):
        assert offs[c] == sum(int(v) for v in counts[c, :5000]) / 5000
    y = o.normalise(counts, offs, o.NORM_RELATIVE)
    assert np.allclose(y, (counts.astype(float) - offs[:, None]) / offs[:, None])
    assert abs(y[:, :5000].mean(axis=1)).max() < 1e-12
    assert np.allclose(o.normalise(counts, offs, o.NORM_SUBTRACT), counts - offs[:, None])
    assert np.array_equal(o.normalise(counts, None, o.NORM_NONE), counts.astype(float))
    # a per-channel scale cancels in G, A, rho and scales P by 1/(o_i o_j)
    L, H, M = 128, 64, 16
    r_rel = o.analyze_chunk(counts, L, H, M, norm_mode=o.NORM_RELATIVE, offs=offs)
    r_sub = o.analyze_chunk(counts, L, H, M, norm_mode=o.NORM_SUBTRACT, offs=offs)
    assert np.allclose(r_rel["G"], r_sub["G"], atol=1e-12)
    assert np.allclose(r_rel["R"], r_sub["R"], atol=1e-12)
    assert np.allclose(r_rel["P"] * offs[0] * offs[1], r_sub["P"], rtol=1e-12)


# ---------------------------------------------------------------------------- P9: chunk independence
def test_P9_chunks_are_independent():
    """"any calculation is performed individually on each time-chunk"."""
    x = _rand_chunk(3, 3000, 8)
    a = o.analyze_chunk(x[:, :1000], 128, 64, 64)
    b = o.analyze_chunk(x[:, 1000:2000], 128, 64, 64)
    x2 = x.copy()
    x2[:, 1000:] += 5.0
    a2 = o.analyze_chunk(x2[:, :1000], 128, 64, 64)
    for k in a:
        assert np.array_equal(a[k], a2[k])
    assert not np.allclose(a["G"], b["G"])


# ---------------------------------------------------------------------------- workload generators
def test_single_config_signature():
    """The config-2 stand-in has the structure DESIGN.md section 4 states: a 20 kHz mode (bin 20
    of 257) coherent over the whole array, advected poloidally: A_ij = +2 pi f (tau_j - tau_i)."""
    wl = es.WORKLOADS["single"]
    x = es.single()
    assert x.shape == (192, 10_000) and x.dtype == np.float32
    rows = [0, 3, 6, 12]
    sel = np.array([r * 8 for r in rows])
    pairs = o.all_pairs(len(sel))
    r = o.analyze_chunk(x[sel], wl.nfft, wl.hop, wl.max_lag)
    tau = (0.40 / 24) / 5e3 * es.FS   # samples per row
    b = 20
    assert r["G"][:, b].min() > 0.9
    for p, (i, j) in enumerate(pairs):
        expect = 2 * np.pi * b / wl.nfft * tau * (rows[j] - rows[i])
        assert abs(np.angle(np.exp(1j * (r["A"][p, b] - expect)))) < 0.1


def test_golden_oracle_regression():
    """tests/golden/tiny_oracle.txt is written by tests/golden/make_golden.py, which calls only
    oracle/ and ecei_synth; it guards the oracle against accidental change."""
    path = os.path.join(GOLDEN, "tiny_oracle.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    wl = es.WORKLOADS["tiny"]
    r = o.analyze_chunk(es.tiny(), wl.nfft, wl.hop, wl.max_lag)
    assert len(rows) > 20
    for name, p, q, val in rows:
        assert abs(r[name][int(p), int(q)] - float(val)) < 1e-12 * max(1.0, abs(float(val)))


# ---------------------------------------------------------------------------- f1: band-pass pre-processing (R19)
def test_P11_bandpass_kept_bins_of_the_papers_demo_band():
    """the demo uses a 5-9 kHz pass band.  At BASELINE config 2 (nfft 512, fs 500 kHz) the bin
    spacing is 976.5625 Hz, so the kept bins are 6..9 (5859.4 .. 8789.1 Hz): hand-computed, not from the oracle."""
    m = o.band_mask(512, 500e3, 5e3, 9e3)
    assert m.shape == (257,) and np.flatnonzero(m).tolist() == [6, 7, 8, 9]
    assert o.band_mask(256, 500e3, 0.0, 250e3).all()                       # the whole band: nothing removed
    assert np.flatnonzero(o.band_mask(256, 500e3, 0.0, 0.0)).tolist() == [0]   # DC only
    # a band edge exactly on a bin keeps the bin (closed interval): bin 16 of 256 at fs = 512 Hz is 32 Hz
    assert np.flatnonzero(o.band_mask(256, 512.0, 32.0, 34.0)).tolist() == [16, 17]


def test_P12_bandpass_is_a_per_segment_circular_filter():
    """Masking the bins of a segment's transform = filtering the windowed segment with the ideal circular filter.
    So the band-passed cross-correlation must equal the brute-force circular correlation (P5's form) of the
    FILTERED windowed segments, the filtered segments coming from numpy's rfft/irfft (independent library code),
    and a tone outside the band must vanish from every output.  Catches: mask applied to the wrong side of the
    spectrum, normalisation of rho taken from unfiltered autospectra, mask edges off by one."""
    L, H, M, fs = 64, 32, 32, 6400.0       # bin spacing 100 Hz
    lo, hi = 450.0, 1250.0                 # keeps bins 5..12
    T = 400
    t = np.arange(T)
    rng = np.random.default_rng(12)
    x = 0.05 * rng.standard_normal((3, T))
    x += np.sin(2 * np.pi * 8 * t / L + np.array([[0.0], [0.4], [0.9]]))      # bin 8: in the band
    x += 2.0 * np.sin(2 * np.pi * 20 * t / L + np.array([[0.1], [0.2], [0.3]]))  # bin 20: outside
    K = o.n_segments(T, L, H)
    w = o.hann_periodic(L)
    s2 = o.scale_factor(L)
    mask = o.band_mask(L, fs, lo, hi)
    assert np.flatnonzero(mask).tolist() == list(range(5, 13))
    r = o.analyze_chunk(x, L, H, M, fs=fs, band=(lo, hi))
    full = o.analyze_chunk(x, L, H, M, fs=fs)
    # in the band nothing changes, outside everything is exactly zero (G = 0 by R16, A = atan2(0, 0) = 0)
    for k in ("G", "A", "P"):
        assert np.array_equal(r[k][:, mask], full[k][:, mask])
        assert np.all(r[k][:, ~mask] == 0.0)
    assert np.all(r["Sauto"][:, ~mask] == 0.0) and np.array_equal(r["Sauto"][:, mask], full["Sauto"][:, mask])
    assert full["P"][:, 20].min() > 1e-3           # the out-of-band tone was really there
    # brute force in the time domain on filtered segments
    def filt(seg):
        Z = np.fft.rfft(seg)
        Z[~mask] = 0.0
        return np.fft.irfft(Z, L)
    pairs = o.all_pairs(3)
    yf = [[filt(w * x[c, k * H:k * H + L]) for k in range(K)] for c in range(3)]
    def corr(i, j, m):
        return s2 * sum(np.dot(np.roll(yf[i][k], -m), yf[j][k]) for k in range(K)) / K
    r0 = [corr(c, c, 0) for c in range(3)]
    for p, (i, j) in enumerate(pairs):
        for q, m in enumerate(range(-M, M + 1)):
            assert abs(r["R"][p, q] - corr(i, j, m) / np.sqrt(r0[i] * r0[j])) < 1e-12
    # phases of the in-band tone survive: A_01 = -0.4, A_12 = -0.5 at bin 8 (x_i ahead of x_j => negative, R8)
    assert abs(r["A"][0, 8] + 0.4) < 0.05 and abs(r["A"][2, 8] + 0.5) < 0.05


# ---------------------------------------------------------------------------- f1: other windows, constant detrend
@pytest.mark.parametrize("kind,name", [(o.WIN_HANN, "hann"), (o.WIN_HAMMING, "hamming"), (o.WIN_RECT, "boxcar"),
                                       (o.WIN_BLACKMAN, "blackman")])
@pytest.mark.parametrize("detrend", [o.DETREND_NONE, o.DETREND_CONSTANT])
def test_P13_windows_and_detrend_against_scipy(kind, name, detrend):
    """The window variants equal scipy's periodic (fftbins) windows, and the whole estimator with a window and the
    constant detrend equals scipy's Welch cross-spectral density (independent library code; scipy conjugates its
    first argument, P6).  Closed form for the rectangular window: a bin-centred unit cosine has |X[q]| = L/2 and
    nothing anywhere else.  Catches: symmetric instead of periodic window, mean taken over the chunk instead of the
    segment, detrend after the window, s^2 taken from the wrong window."""
    L, H = 128, 64
    w = o.window(L, kind)
    assert np.allclose(w, sps.get_window(name, L, fftbins=True), atol=1e-15)
    x = _rand_chunk(3, 1500, 31) + np.array([[3.0], [-2.0], [0.5]])    # offsets make the detrend matter
    X = o.stft(x, L, H, kind, detrend)
    pairs = o.all_pairs(3)
    s2 = o.scale_factor(L, o.SCALE_WINPOW, 1.0, kind)
    assert abs(s2 - 1.0 / np.sum(w * w)) < 1e-15
    S = o.cross_spectra(X, pairs, s2)
    kw = dict(fs=1.0, window=name, nperseg=L, noverlap=L - H, nfft=L,
              detrend="constant" if detrend == o.DETREND_CONSTANT else False, return_onesided=False, scaling="density")
    for p, (i, j) in enumerate(pairs):
        _, Pd = sps.csd(x[i], x[j], **kw)
        assert np.allclose(np.conj(Pd[:L // 2 + 1]), S[p], rtol=1e-9, atol=1e-12)
    if detrend == o.DETREND_CONSTANT:      # the DC bin of a detrended rectangular-window segment is exactly empty
        Xr = o.stft(x, L, H, o.WIN_RECT, detrend)
        assert np.abs(Xr[:, :, 0]).max() < 1e-10
    if kind == o.WIN_RECT:
        q = 9
        t = np.arange(600)
        Xc = o.stft(np.cos(2 * np.pi * q * t / L + 0.7)[None, :], L, H, kind, o.DETREND_NONE)
        assert np.allclose(np.abs(Xc[0, :, q]), L / 2, atol=1e-9)
        others = np.delete(np.abs(Xc[0]), q, axis=1)
        assert others.max() < 1e-9


# ---------------------------------------------------------------------------- f2: accumulation over chunks
def test_P14_accumulation_over_chunks_is_the_mean_over_all_segments():
    """Accumulating per-chunk spectra = Eq. (1a) with E[.] over the segments of all the chunks: compare with the
    cross-spectrum computed in one go from the stacked segments.  And the point of it: for independent noise the
    coherence floor drops like 1/sqrt(number of chunks) (P8's law with K -> n K)."""
    L, H, T, n = 64, 32, 640, 6
    rng = np.random.default_rng(14)
    chunks = [rng.standard_normal((3, T)) for _ in range(n)]
    pairs = o.all_pairs(3)
    s2 = o.scale_factor(L)
    Xs = [o.stft(c, L, H) for c in chunks]
    S_acc = o.accumulate([o.cross_spectra(X, pairs, s2) for X in Xs])
    Sa_acc = o.accumulate([o.auto_spectra(X, s2) for X in Xs])
    X_all = np.concatenate(Xs, axis=1)                      # all segments of all chunks
    assert np.allclose(S_acc, o.cross_spectra(X_all, pairs, s2), rtol=1e-12, atol=1e-14)
    assert np.allclose(Sa_acc, o.auto_spectra(X_all, s2), rtol=1e-12, atol=1e-14)
    G1 = o.coherence(o.cross_spectra(Xs[0], pairs, s2), o.auto_spectra(Xs[0], s2), pairs)
    Gn = o.coherence(S_acc, Sa_acc, pairs)
    assert 0.30 < Gn[:, 2:-2].mean() / G1[:, 2:-2].mean() < 0.55      # 1/sqrt(6) = 0.41


# ---------------------------------------------------------------------------- f2: per-segment-normalised coherence
def test_P15_phase_lock_estimator():
    """Unit phasors per segment: (1) two tones with a fixed phase difference but amplitudes that jump from segment to
    segment (one channel's amplitude independent of the other's): the ordinary coherence is well below 1, the
    phase-lock value is 1 and the cross-phase is the injected one; (2) autospectra are exactly s2 everywhere;
    (3) independent white noise without overlap: the mean of |mean of K random unit phasors| is the Rayleigh mean
    sqrt(pi / (4 K)) (closed form), e.g. 0.221 for K = 16."""
    L, H, q = 64, 64, 9                       # no overlap: segments are independent
    K = 16
    T = K * L
    rng = np.random.default_rng(15)
    a1 = np.repeat(rng.uniform(0.2, 3.0, K), L)
    a2 = np.repeat(rng.uniform(0.2, 3.0, K), L)
    t = np.arange(T)
    x = np.stack([a1 * np.cos(2 * np.pi * q * t / L + 0.9), a2 * np.cos(2 * np.pi * q * t / L + 0.2)])
    plain = o.analyze_chunk(x, L, H, L // 2)
    lock = o.analyze_chunk(x, L, H, L // 2, phase_lock=True)
    assert plain["G"][0, q] < 0.93
    assert abs(lock["G"][0, q] - 1.0) < 1e-12 and abs(lock["A"][0, q] - 0.7) < 1e-9
    assert np.allclose(lock["Sauto"], o.scale_factor(L), rtol=1e-12)
    n = rng.standard_normal((24, T))
    g = o.analyze_chunk(n, L, H, L // 2, phase_lock=True)["G"][:, 1:-1]
    assert abs(g.mean() - np.sqrt(np.pi / (4 * K))) < 0.01


# ---------------------------------------------------------------------------- f2: zero-padded segments (R22)
def test_P16_zero_padded_segments_give_the_linear_correlation():
    """nperseg = L/2 samples zero-padded to L: (1) equals scipy's Welch CSD with nperseg < nfft; (2) the correlation
    of Eq. (1d) is then the LINEAR (no wrap-around) windowed correlation for every lag |m| <= L - nperseg: brute force
    over plain sums; (3) a copy delayed by d = 40 samples (more than half the un-padded transform) is found at m = -40."""
    L, Ls, H = 128, 64, 32
    x = _rand_chunk(3, 1200, 16)
    X = o.stft(x, L, H, nperseg=Ls)
    K = o.n_segments(1200, Ls, H)
    assert X.shape == (3, K, L // 2 + 1)
    pairs = o.all_pairs(3)
    s2 = o.scale_factor(L, nperseg=Ls)
    w = o.hann_periodic(Ls)
    assert abs(s2 - 1.0 / np.sum(w * w)) < 1e-15
    S = o.cross_spectra(X, pairs, s2)
    kw = dict(fs=1.0, window="hann", nperseg=Ls, noverlap=Ls - H, nfft=L, detrend=False, return_onesided=False,
              scaling="density")
    for p, (i, j) in enumerate(pairs):
        _, Pd = sps.csd(x[i], x[j], **kw)
        assert np.allclose(np.conj(Pd[:L // 2 + 1]), S[p], rtol=1e-9, atol=1e-12)
    M = L - Ls
    r = o.analyze_chunk(x, L, H, M, nperseg=Ls)
    def lin(i, j, m):     # sum_n yh_i[n + m] yh_j[n], indices outside 0..Ls-1 contribute nothing
        acc = 0.0
        for k in range(K):
            yi, yj = w * x[i, k * H:k * H + Ls], w * x[j, k * H:k * H + Ls]
            for n in range(Ls):
                if 0 <= n + m < Ls:
                    acc += yi[n + m] * yj[n]
        return s2 * acc / K
    r0 = [lin(c, c, 0) for c in range(3)]
    for p, (i, j) in enumerate(pairs):
        for q, m in enumerate(range(-M, M + 1)):
            assert abs(r["R"][p, q] - lin(i, j, m) / np.sqrt(r0[i] * r0[j])) < 1e-12
    d = 40                                            # a delay beyond L/2 of the un-padded transform (32)
    base = np.random.default_rng(3).standard_normal(3000 + d)
    xx = np.stack([base[d:], base[:3000]])            # x_1[t] = x_0[t - d]
    padded = o.analyze_chunk(xx, 128, 32, 64, nperseg=64)["R"][0]
    assert np.argmax(padded) - 64 == -d               # found at its true lag, no wrap-around image


# ----------------------------------------------------------------------------------------------
# oracle/fft_baseline.py is the "CPU, library FFT" arm of BASELINE.md section 3 and the float64 checker of the full-size
# GPU tests.  It is not the oracle; it is pinned TO the oracle here (the library FFT itself is pin P6).
@pytest.mark.parametrize("C,T,L,H,M", [(8, 2048, 256, 128, 128), (5, 3000, 128, 100, 40), (12, 10_000, 512, 256, 256)])
def test_fft_baseline_equals_oracle(C, T, L, H, M):
    from oracle import fft_baseline as fb
    x = np.random.default_rng(C * 31 + L).standard_normal((C, T))
    x[1] += 0.6 * x[0]
    ref = o.analyze_chunk(x, L, H, M)
    got = fb.analyze_chunk(x, L, H, M)
    for k in ("G", "P", "R", "Sauto"):
        assert got[k].shape == ref[k].shape, k
        assert np.max(np.abs(got[k] - ref[k])) <= 1e-10 * max(1.0, float(np.abs(ref[k]).max())), k
    assert np.max(np.abs(np.angle(np.exp(1j * (got["A"] - ref["A"]))))) <= 1e-8


# ----------------------------------------------------------------------------------------------
# f1: transform lengths that are not powers of two.  The oracle is a direct DFT and takes any even L; what pins it
# there is again independent library code (scipy's Welch CSD / coherence and numpy's irfft run at L = 500, 768, 1000).
@pytest.mark.parametrize("L,H", [(500, 250), (768, 192), (1000, 400)])
def test_non_power_of_two_lengths_against_scipy(L, H):
    rng = np.random.default_rng(L)
    T = 12 * L
    x = rng.standard_normal((3, T))
    x[1] = 0.8 * np.roll(x[0], 3) + 0.4 * x[1]
    out = o.analyze_chunk(x, L, H, L // 2, want_S=True)
    K = o.n_segments(T, L, H)
    pairs = o.all_pairs(3)
    for p, (i, j) in enumerate(pairs):
        f, Pxy = sps.csd(x[i, :(K - 1) * H + L], x[j, :(K - 1) * H + L], fs=1.0, window=sps.get_window("hann", L, fftbins=True),
                         nperseg=L, noverlap=L - H, nfft=L, detrend=False, return_onesided=False, scaling="spectrum")
        w = o.hann_periodic(L)
        s_spec = 1.0 / np.sum(w) ** 2
        S_sc = np.conj(Pxy[:L // 2 + 1]) / s_spec * o.scale_factor(L)     # scipy: conj(X_i) X_j, 'spectrum' scaling
        assert np.max(np.abs(out["S"][p] - S_sc)) <= 1e-10 * np.max(np.abs(S_sc))
        _, Cxy = sps.coherence(x[i, :(K - 1) * H + L], x[j, :(K - 1) * H + L], window=sps.get_window("hann", L, fftbins=True),
                               nperseg=L, noverlap=L - H, nfft=L, detrend=False)
        assert np.max(np.abs(out["G"][p] ** 2 - Cxy)) <= 1e-10
        # Eq. (1d): numpy's inverse real FFT of the half spectrum (Im of DC and Nyquist dropped, as irfft does)
        R = np.fft.irfft(out["S"][p], n=L)
        R0 = np.array([np.fft.irfft(out["Sauto"][c], n=L)[0] for c in (i, j)])
        rho = np.concatenate([R[L - L // 2:], R[:L // 2 + 1]]) / np.sqrt(R0[0] * R0[1])
        assert np.max(np.abs(out["R"][p] - rho)) <= 1e-12
