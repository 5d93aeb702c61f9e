"""GPU parity: the CUDA path (through the C ABI, via the ctypes binding) against the float64 oracle,
element by element on the same seeded inputs.

Tolerances are BASELINE.json north_star's:
  cross-power  1e-4 relative      (reading R13: where G_oracle > 0.1 and on autospectra; elsewhere
                                    |dP| <= 1e-5 sqrt(S_ii S_jj), which is tighter than the coherence bound)
  coherence    1e-4 absolute
  cross-phase  1e-3 rad where G_oracle > 0.1, compared modulo 2 pi (R15)
  cross-corr   1e-4 absolute on the normalised rho
"""
import numpy as np
import pytest
import torch

import ecei_synth as es
from oracle import delta_oracle as o

pytestmark = pytest.mark.gpu

TOL_P_REL, TOL_G, TOL_A, TOL_R = 1e-4, 1e-4, 1e-3, 1e-4


def binding():
    from paper_2108_08896_b200 import binding as b
    return b


def dev(x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def compare(out, ref, pairs, label="", p_abs_tol=1e-5):
    """out: dict of numpy float32 arrays for `pairs`; ref: oracle dict for the same pairs."""
    G, A, P, R, Sa = (np.asarray(out[k], dtype=np.float64) for k in ("G", "A", "P", "R", "Sauto"))
    for k in ("G", "A", "P", "R", "Sauto"):
        assert np.isfinite(out[k]).all(), f"{label}: non-finite {k}"
    pairs = np.asarray(pairs).reshape(-1, 2)
    den = np.sqrt(ref["Sauto"][pairs[:, 0]] * ref["Sauto"][pairs[:, 1]]) if len(pairs) else np.zeros((0, 1))
    gate = ref["G"] > 0.1
    stats = {}
    stats["auto_rel"] = float(np.max(np.abs(Sa - ref["Sauto"]) / np.maximum(ref["Sauto"], 1e-300))) if Sa.size else 0.0
    assert stats["auto_rel"] <= TOL_P_REL, f"{label}: autospectra rel err {stats['auto_rel']:.3g}"
    if len(pairs) == 0:
        return stats
    dP = np.abs(P - ref["P"])
    stats["P_rel_gated"] = float(np.max(np.where(gate, dP / np.maximum(ref["P"], 1e-300), 0.0)))
    stats["P_abs_norm"] = float(np.max(np.where(den > 0, dP / np.where(den > 0, den, 1.0), 0.0)))
    stats["G_abs"] = float(np.max(np.abs(G - ref["G"])))
    dA = np.abs(np.angle(np.exp(1j * (A - ref["A"]))))
    stats["A_gated"] = float(np.max(np.where(gate, dA, 0.0)))
    stats["R_abs"] = float(np.max(np.abs(R - ref["R"])))
    assert stats["P_rel_gated"] <= TOL_P_REL, f"{label}: cross-power rel err (G>0.1) {stats['P_rel_gated']:.3g}"
    assert stats["P_abs_norm"] <= p_abs_tol, f"{label}: cross-power abs err / sqrt(SiiSjj) {stats['P_abs_norm']:.3g}"
    assert stats["G_abs"] <= TOL_G, f"{label}: coherence abs err {stats['G_abs']:.3g}"
    assert stats["A_gated"] <= TOL_A, f"{label}: cross-phase err (G>0.1) {stats['A_gated']:.3g}"
    assert stats["R_abs"] <= TOL_R, f"{label}: cross-correlation abs err {stats['R_abs']:.3g}"
    return stats


@pytest.fixture(params=["fp32", "tc"])
def mode(request):
    """Both contraction back ends: FP32 FMA pipe and tcgen05 tensor cores (split fp16)."""
    b = binding()
    return b.CONTRACT_FP32 if request.param == "fp32" else b.CONTRACT_TC


def gpu_analyze(x, L, H, M, in_dtype=None, norm_mode=0, n_first=0, contraction=0, scaling=0, fs=500e3, ld_pad=0, band=None,
                window=0, detrend=0):
    b = binding()
    C, T = x.shape
    in_dtype = (b.I16 if x.dtype == np.int16 else b.F32) if in_dtype is None else in_dtype
    plan = b.Plan(C, T, L, H, M, in_dtype=in_dtype, norm_mode=norm_mode, contraction=contraction, scaling=scaling, fs=fs,
                  band=band, window=window, detrend=detrend)
    if ld_pad:
        buf = torch.zeros((C, T + ld_pad), dtype=dev(x[:1, :1]).dtype, device="cuda")
        buf[:, :T] = dev(x)
        xd = buf[:, :T]
    else:
        xd = dev(x)
    if norm_mode != 0:
        plan.set_offsets(xd, n_first)
    out = plan.analyze_chunk(xd)
    torch.cuda.synchronize()
    return plan, {k: v.cpu().numpy() for k, v in out.items()}


def oracle_for(x, L, H, M, pairs=None, norm_mode=0, offs=None, scaling=0, fs=500e3, band=None, win=0, detrend=0):
    return o.analyze_chunk(x, L, H, M, pairs=pairs, norm_mode=norm_mode, offs=offs, scaling=scaling, fs=fs, band=band,
                           win=win, detrend=detrend)


# ------------------------------------------------------------------------------------------
def test_library_is_the_cuda_path():
    b = binding()
    import os
    assert os.path.exists(b.LIB_PATH)
    plan = b.Plan(8, 2048, 256, 128)
    assert plan.sizes.contraction in (b.CONTRACT_FP32, b.CONTRACT_TC)


def test_config1_tiny_full(mode):
    w = es.WORKLOADS["tiny"]
    x = es.tiny()
    _, out = gpu_analyze(x, w.nfft, w.hop, w.max_lag, contraction=mode)
    ref = oracle_for(x, w.nfft, w.hop, w.max_lag)
    st = compare(out, ref, o.all_pairs(w.C), "tiny")
    print("tiny", st)
    # P7: injected phases recovered by the CUDA path itself
    expect = np.array([0.3 * (i - j) for i, j in o.all_pairs(8)])
    assert np.abs(np.angle(np.exp(1j * (out["A"][:, 10] - expect)))).max() < 2e-2


def test_config2_single_chunk_full(mode):
    w = es.WORKLOADS["single"]
    x = es.single()
    _, out = gpu_analyze(x, w.nfft, w.hop, w.max_lag, contraction=mode)
    ref = oracle_for(x, w.nfft, w.hop, w.max_lag)
    st = compare(out, ref, o.all_pairs(w.C), "single")
    print("single", st)


def test_stft_stage_against_oracle(mode):
    b = binding()
    w = es.WORKLOADS["tiny"]
    x = es.tiny()
    plan = b.Plan(w.C, w.T, w.nfft, w.hop, w.max_lag, contraction=mode)
    X = plan.stft_unpack(plan.stft(dev(x))).cpu().numpy()
    Xo = o.stft(x, w.nfft, w.hop)
    assert X.shape == Xo.shape
    scale = np.abs(Xo).max()
    assert np.abs(X - Xo).max() <= 2e-6 * scale


def test_staged_calls_equal_fused_call(mode):
    b = binding()
    w = es.WORKLOADS["single"]
    x = es.single()[:40]
    plan = b.Plan(40, w.T, w.nfft, w.hop, w.max_lag, contraction=mode)
    xd = dev(x)
    fused = plan.analyze_chunk(xd)
    X = plan.stft(xd)
    S, Sa = plan.cross_spectra(X)
    G, A, P, R = plan.coherence(S, Sa), plan.crossphase(S), plan.crosspower(S), plan.crosscorr(S, Sa)
    torch.cuda.synchronize()
    for name, t in (("G", G), ("A", A), ("P", P), ("Sauto", Sa)):
        assert torch.equal(t, fused[name]), name
    # rho: the fused call takes the zero-lag autocorrelations R_cc[0] from the windowed signal energy (time domain),
    # the staged call from the caller's autospectra (sum over bins); Parseval makes them equal up to float32 rounding
    assert torch.max(torch.abs(R - fused["R"])).item() < 5e-6
    # S itself against the oracle (through the unpack accessor: [P][F], lexicographic pairs)
    Xo = o.stft(x, w.nfft, w.hop)
    pairs = o.all_pairs(40)
    s2 = o.scale_factor(w.nfft)
    So = o.cross_spectra(Xo, pairs, s2)
    Sg = plan.cross_spectra_unpack(S).cpu().numpy()
    Sa_o = o.auto_spectra(Xo, s2)
    den = np.sqrt(Sa_o[pairs[:, 0]] * Sa_o[pairs[:, 1]])
    assert np.max(np.abs(Sg - So) / den) < 1e-5


@pytest.mark.parametrize("C,T,L,H,M", [
    (5, 3000, 128, 100, 40),    # ragged everything: odd C, hop not dividing L, short lags
    (2, 64, 64, 64, 32),        # T == L: a single segment; smallest transform
    (3, 700, 64, 1, 0),         # hop 1 (K = 637 segments), lag 0 only
    (1, 1000, 256, 128, 128),   # a single channel: no pairs, autospectra only
    (70, 1200, 256, 256, 128),  # no overlap; more than one 64-channel tile with a ragged one
    (4, 9000, 4096, 2048, 2048),  # largest transform
    (6, 5000, 1024, 300, 17),
    (9, 4100, 2048, 1024, 1000),
    (33, 900, 128, 64, 64),
])
def test_edge_shapes(C, T, L, H, M, mode):
    x = np.random.default_rng(C * 1000 + L).standard_normal((C, T)).astype(np.float32)
    x += 0.5 * x[0:1]  # some coherence between channels
    _, out = gpu_analyze(x, L, H, M, contraction=mode)
    ref = oracle_for(x, L, H, M)
    assert out["G"].shape == ref["G"].shape and out["R"].shape == ref["R"].shape
    compare(out, ref, o.all_pairs(C), f"edge C={C} L={L}")


def test_strided_rows_and_scalings(mode):
    x = np.random.default_rng(5).standard_normal((6, 2000)).astype(np.float32)
    b = binding()
    for scaling in (b.SCALE_NONE, b.SCALE_DENSITY, b.SCALE_SPECTRUM):
        _, out = gpu_analyze(x, 256, 128, 64, scaling=scaling, fs=500e3, ld_pad=37, contraction=mode)
        ref = oracle_for(x, 256, 128, 64, scaling=scaling, fs=500e3)
        compare(out, ref, o.all_pairs(6), f"scaling {scaling}")


def test_degenerate_zero_channel(mode):
    """A dead channel: S_ii = 0 -> coherence and rho are 0 by definition (R16), nothing is NaN."""
    x = np.random.default_rng(6).standard_normal((4, 1500)).astype(np.float32)
    x[2] = 0.0
    _, out = gpu_analyze(x, 128, 64, 64, contraction=mode)
    ref = oracle_for(x, 128, 64, 64)
    compare(out, ref, o.all_pairs(4), "dead channel")
    dead = [p for p, (i, j) in enumerate(o.all_pairs(4)) if 2 in (i, j)]
    assert np.all(out["G"][dead] == 0) and np.all(out["R"][dead] == 0) and np.all(out["P"][dead] == 0)


@pytest.mark.parametrize("norm_mode", [0, 1, 2])
def test_int16_and_normalisation_modes(norm_mode, mode):
    rng = np.random.default_rng(8)
    o_true = rng.uniform(2000, 3000, size=6)
    sig = rng.standard_normal((6, 6000))
    sig[1] += 0.7 * sig[0]
    counts = np.rint(o_true[:, None] + 200 * sig).astype(np.int16)
    plan, out = gpu_analyze(counts, 512, 256, 256, norm_mode=norm_mode, n_first=5000, contraction=mode)
    offs = o.offsets(counts[:, :5000])
    if norm_mode:
        assert np.array_equal(plan.get_offsets(), offs)   # integer-exact sums
    ref = oracle_for(counts, 512, 256, 256, norm_mode=norm_mode, offs=offs)
    compare(out, ref, o.all_pairs(6), f"int16 norm {norm_mode}")
    # float32 input with offsets
    xf = counts.astype(np.float32)
    plan, out = gpu_analyze(xf, 512, 256, 256, norm_mode=norm_mode, n_first=5000, contraction=mode)
    ref = oracle_for(xf, 512, 256, 256, norm_mode=norm_mode, offs=o.offsets(xf[:, :5000]))
    compare(out, ref, o.all_pairs(6), f"f32 norm {norm_mode}")


def test_offsets_required():
    b = binding()
    plan = b.Plan(4, 1000, 128, 64, 64, norm_mode=b.NORM_RELATIVE)
    with pytest.raises(b.DeltaError) as e:
        plan.analyze_chunk(torch.zeros((4, 1000), device="cuda"))
    assert e.value.status == b.ERR_STATE
    with pytest.raises(b.DeltaError) as e:
        plan.analyze_chunk(torch.zeros((4, 1000), device="cuda")[:, :500])  # ld < T is caught first? T mismatch
    assert e.value.status in (b.ERR_STATE, b.ERR_INVALID_ARG)


def _sampled_pairs(C, n_ch, seed):
    rng = np.random.default_rng(seed)
    ch = np.sort(rng.choice(C, size=n_ch, replace=False))
    ch[0], ch[-1] = 0, C - 1   # include the corners of the pair triangle
    ch = np.unique(ch)
    loc = o.all_pairs(len(ch))
    glob = np.stack([ch[loc[:, 0]], ch[loc[:, 1]]], axis=1)
    return ch, loc, glob


TOLS = dict(P_rel=TOL_P_REL, P_abs=1e-5, G=TOL_G, A=TOL_A, R=TOL_R)


def _full_size_check(x, w_nfft, w_hop, w_max_lag, label, n_ch, seed):
    """Both contraction modes at full size, EVERY output element of every pair compared in float64.

    The oracle's direct DFT with its Python loop over pairs would take hours at these sizes, so all rows are checked
    with tests/fastcheck.py (float64, numpy rfft / irfft / matmul) -- after that checker has itself been compared with
    the oracle on a sample of channels of this very input (all pairs among them, first and last channel included)."""
    import fastcheck as fc
    b = binding()
    C = x.shape[0]
    ch, loc, glob = _sampled_pairs(C, n_ch, seed)
    ref = oracle_for(x[ch], w_nfft, w_hop, w_max_lag)
    fast = fc.analyze_sampled(x[ch], w_nfft, w_hop, w_max_lag)
    for k in ("G", "P", "R", "Sauto"):
        assert np.max(np.abs(fast[k] - ref[k])) <= 1e-9 * max(1.0, float(np.abs(ref[k]).max())), k
    assert np.max(np.abs(np.angle(np.exp(1j * (fast["A"] - ref["A"]))))) <= 1e-8
    outs = {}
    for name, mode in (("fp32", b.CONTRACT_FP32), ("tc", b.CONTRACT_TC)):
        _, out = gpu_analyze(x, w_nfft, w_hop, w_max_lag, contraction=mode)
        P = C * (C - 1) // 2
        assert out["G"].shape == (P, w_nfft // 2 + 1) and out["R"].shape == (P, 2 * w_max_lag + 1)
        for k in ("G", "A", "P", "R", "Sauto"):
            assert np.isfinite(out[k]).all(), (name, k)
        # the sampled pairs against the oracle itself
        idx = np.array([o.pair_index(int(i), int(j), C) for i, j in glob])
        sub = {k: out[k][idx] for k in ("G", "A", "P", "R")}
        sub["Sauto"] = out["Sauto"][ch]
        compare(sub, ref, loc, f"{label} sampled {name}")
        outs[name] = out
    st = fc.check_all_pairs(x, w_nfft, w_hop, w_max_lag, outs, TOLS, label)
    print(label, st)


@pytest.mark.parametrize("name,n_ch", [("long", 12), ("wide", 10)])
def test_full_size_configs_all_pairs(name, n_ch):
    """Configs 3 and 5 at BASELINE's full sizes (checked in full): all 18,336 / 73,536 rows of
    G, A, P, rho and the autospectra, both contraction modes."""
    w = es.WORKLOADS[name]
    _full_size_check(es.make(name), w.nfft, w.hop, w.max_lag, name, n_ch, 42)


def test_config4_streamed_shot():
    """Config 4: int16 counts, offsets from the first 5,000 samples of the shot, 250 chunks streamed
    from pinned host memory with the H2D copy of chunk n+1 overlapping the analysis of chunk n.
    Checked chunks: 0, 1, 124, 249 + 4 seeded random ones; also P9 (chunk independence): a chunk
    analysed alone gives bit-identical results to the same chunk inside the stream."""
    b = binding()
    w = es.WORKLOADS["streamed"]
    n_chunks = w.n_chunks
    counts, _ = es.streamed(n_chunks=n_chunks)
    h_x = torch.from_numpy(counts).pin_memory()
    plan = b.Plan(w.C, w.T, w.nfft, w.hop, w.max_lag, in_dtype=b.I16, norm_mode=b.NORM_RELATIVE)
    s = plan.sizes
    check = sorted({0, 1, 124, 249} | set(np.random.default_rng(4).choice(n_chunks, 4, replace=False).tolist()))
    slots = torch.empty(plan.slot_bytes(), dtype=torch.uint8, device="cuda")
    # keep every chunk's coherence on the device, the other quantities in a rotating set of 2
    G = torch.empty((n_chunks, s.P, s.F), dtype=torch.float32, device="cuda")
    A = torch.empty((n_chunks, s.P, s.F), dtype=torch.float32, device="cuda")
    P = torch.empty((n_chunks, s.P, s.F), dtype=torch.float32, device="cuda")
    R = torch.empty((n_chunks, s.P, s.n_lags), dtype=torch.float32, device="cuda")
    Sa = torch.empty((n_chunks, w.C, s.F), dtype=torch.float32, device="cuda")
    plan.analyze_shot_host(h_x, slots, dict(G=G, A=A, P=P, R=R, Sauto=Sa),
                           strides=(s.P * s.F, s.P * s.n_lags, w.C * s.F), set_offsets=True, n_first=w.n_first)
    torch.cuda.synchronize()
    offs = o.offsets(counts[0][:, :w.n_first])
    assert np.array_equal(plan.get_offsets(), offs)
    pairs = o.all_pairs(w.C)
    for n in check:
        ref = oracle_for(counts[n], w.nfft, w.hop, w.max_lag, norm_mode=o.NORM_RELATIVE, offs=offs)
        out = dict(G=G[n].cpu().numpy(), A=A[n].cpu().numpy(), P=P[n].cpu().numpy(), R=R[n].cpu().numpy(),
                   Sauto=Sa[n].cpu().numpy())
        st = compare(out, ref, pairs, f"streamed chunk {n}")
        print("chunk", n, st)
    # P9: chunk 124 alone
    alone = plan.analyze_chunk(dev(counts[124]))
    torch.cuda.synchronize()
    for k, t in (("G", G), ("A", A), ("P", P), ("R", R), ("Sauto", Sa)):
        assert torch.equal(alone[k], t[124]), k


@pytest.mark.parametrize("ring", [0, 2, 3])
def test_host_output_path_roundtrip(ring):
    """delta_analyze_shot_host with host outputs (the e2e path bench.py times): the device->host copies run on the
    library's second copy stream under the kernels of the next chunks.  ring = 0 with zero strides: one device output
    set, overwritten chunk after chunk (every overwrite must wait for the copy-back); ring = 2, 3: rotating sets."""
    b = binding()
    n = 7
    x = np.random.default_rng(3).standard_normal((n, 12, 1024)).astype(np.float32)
    plan = b.Plan(12, 1024, 128, 64, 64)
    s = plan.sizes
    h_x = torch.from_numpy(x).pin_memory()
    slots = torch.empty(plan.slot_bytes(), dtype=torch.uint8, device="cuda")
    sets = max(ring, 1)
    dev_out = dict(G=torch.empty((sets, s.P, s.F), device="cuda"), A=torch.empty((sets, s.P, s.F), device="cuda"),
                   P=torch.empty((sets, s.P, s.F), device="cuda"), R=torch.empty((sets, s.P, s.n_lags), device="cuda"),
                   Sauto=torch.empty((sets, 12, s.F), device="cuda"))
    strides = (s.P * s.F, s.P * s.n_lags, 12 * s.F) if ring else (0, 0, 0)
    host = dict(G=torch.empty((n, s.P, s.F)).pin_memory(), A=torch.empty((n, s.P, s.F)).pin_memory(),
                P=torch.empty((n, s.P, s.F)).pin_memory(), R=torch.empty((n, s.P, s.n_lags)).pin_memory(),
                Sauto=torch.empty((n, 12, s.F)).pin_memory())
    for rep in range(2):   # twice back to back: the second shot must wait for the first one's copies
        plan.analyze_shot_host(h_x, slots, dev_out, strides=strides, host_out=host, ring=ring)
    torch.cuda.synchronize()
    for k in range(n):
        ref = oracle_for(x[k], 128, 64, 64)
        compare({q: host[q][k].numpy() for q in host}, ref, o.all_pairs(12), f"host chunk {k}")


def test_chunks_in_flight_two_plans_two_streams():
    """bench.py keeps two independent chunks in flight (two plans = two workspaces, two streams).  Results must be
    bit-identical to the same chunks analysed one after the other on one stream (P9: chunks are independent)."""
    b = binding()
    w = es.WORKLOADS["single"]
    xs = [dev(es.turbulence(w.T, 700 + i)[:64]) for i in range(4)]
    serial_plan = b.Plan(64, w.T, w.nfft, w.hop, w.max_lag)
    serial = [{k: v.clone() for k, v in serial_plan.analyze_chunk(x).items()} for x in xs]
    torch.cuda.synchronize()
    plans = [b.Plan(64, w.T, w.nfft, w.hop, w.max_lag) for _ in range(2)]
    streams = [torch.cuda.Stream() for _ in range(2)]
    torch.cuda.synchronize()
    outs = []
    for rep in range(3):          # several rounds so that the kernels of the two streams really interleave
        outs = []
        for k, x in enumerate(xs):
            with torch.cuda.stream(streams[k % 2]):
                outs.append(plans[k % 2].analyze_chunk(x))
    torch.cuda.synchronize()
    for k in range(4):
        for name in ("G", "A", "P", "R", "Sauto"):
            assert torch.equal(outs[k][name], serial[k][name]), (k, name)


def test_programmatic_dependent_launch_does_not_change_results(monkeypatch):
    """The three kernels are chained by programmatic dependent launch; DELTA_NO_PDL=1 (read at plan creation)
    launches them with plain stream order.  Same bits either way, also back to back on one stream."""
    b = binding()
    w = es.WORKLOADS["single"]
    xs = [dev(es.turbulence(w.T, 800 + i)[:48]) for i in range(3)]
    pdl = b.Plan(48, w.T, w.nfft, w.hop, w.max_lag)
    monkeypatch.setenv("DELTA_NO_PDL", "1")
    plain = b.Plan(48, w.T, w.nfft, w.hop, w.max_lag)
    monkeypatch.delenv("DELTA_NO_PDL")
    a = [pdl.analyze_chunk(x) for x in xs]        # no sync in between: chunk n+1 is launched while n runs
    c = [plain.analyze_chunk(x) for x in xs]
    torch.cuda.synchronize()
    for k in range(3):
        for name in ("G", "A", "P", "R", "Sauto"):
            assert torch.equal(a[k][name], c[k][name]), (k, name)


@pytest.mark.parametrize("band", [(5e3, 9e3), (15e3, 60e3), (0.0, 250e3)])
def test_bandpass_preprocessing(band, mode):
    """f1: band-pass pre-processing as a mask on the transform's bins (R19), here the demo's
    5-9 kHz band of PAPER.md L231, a band around the 20 kHz mode, and the whole band (= no filter).  Outside the
    band every output is exactly 0; rho is normalised with the filtered autospectra."""
    w = es.WORKLOADS["single"]
    x = es.single()[:40]
    _, out = gpu_analyze(x, w.nfft, w.hop, w.max_lag, contraction=mode, band=band)
    ref = oracle_for(x, w.nfft, w.hop, w.max_lag, band=band)
    st = compare(out, ref, o.all_pairs(40), f"band {band}")
    print(band, st)
    mask = o.band_mask(w.nfft, 500e3, band[0], band[1])
    for k in ("G", "A", "P"):
        assert np.all(out[k][:, ~mask] == 0.0), k
    assert np.all(out["Sauto"][:, ~mask] == 0.0)
    if mask.all():   # the whole band must reproduce the unfiltered call (up to the source of R_cc[0]: Parseval)
        _, plain = gpu_analyze(x, w.nfft, w.hop, w.max_lag, contraction=mode)
        for k in ("G", "A", "P", "Sauto"):
            assert np.array_equal(out[k], plain[k]), k
        assert np.abs(out["R"] - plain["R"]).max() < 5e-6


@pytest.mark.parametrize("window,detrend,L,H", [(1, 0, 512, 256), (2, 1, 512, 256), (3, 1, 256, 64), (0, 1, 2048, 1024),
                                                (2, 0, 64, 32)])
def test_window_variants_and_detrend(window, detrend, L, H, mode):
    """f1: Hamming / rectangular / Blackman windows and the per-segment constant detrend, on
    a signal with large per-channel offsets (so that a missing detrend or a wrong window shows).  L = 2048 uses
    transforms wider than a warp (the detrend sum crosses warps), L = 64 the smallest."""
    rng = np.random.default_rng(77)
    C, T = 12, 9000
    # white noise mixed over neighbouring channels (flat spectrum: the float32 dynamic-range question of R13 is
    # config 2's business, not this test's) plus per-channel offsets
    g = rng.standard_normal((C + 1, T))
    x = (g[:C] + 0.7 * g[1:] + rng.uniform(-1, 1, size=(C, 1))).astype(np.float32)
    M = L // 2
    _, out = gpu_analyze(x, L, H, M, contraction=mode, window=window, detrend=detrend)
    ref = oracle_for(x, L, H, M, win=window, detrend=detrend)
    if window == 2 and detrend == 1:
        # rectangular window + detrend: the DC bin is exactly empty (pin P13), so G and A are 0/0 there and the
        # autospectrum is rounding residue on both sides; compare bins 1.. and bound the residue
        assert np.abs(out["Sauto"][:, 0]).max() <= 1e-9 * out["Sauto"].max()
        out = {k: (v if k == "R" else v[:, 1:]) for k, v in out.items()}
        ref = {k: (v if k == "R" else v[:, 1:]) for k, v in ref.items()}
    st = compare(out, ref, o.all_pairs(C), f"window {window} detrend {detrend} L {L}")
    print(window, detrend, L, st)


def test_accumulation_over_chunks(mode):
    """f2: the expectation of Eq. (1a) over the segments of several chunks: per-chunk spectra
    accumulated with delta_accumulate, then the staged coherence / phase / power / correlation calls on the sum,
    against the oracle's accumulated estimate."""
    b = binding()
    w = es.WORKLOADS["single"]
    C, n = 32, 5
    chunks = [es.turbulence(w.T, 900 + i)[:C] for i in range(n)]
    plan = b.Plan(C, w.T, w.nfft, w.hop, w.max_lag, contraction=mode)
    S_acc, Sa_acc = plan.empty_S(), torch.empty((C, plan.sizes.F), dtype=torch.float32, device="cuda")
    S_acc.fill_(float("nan"))          # w_acc = 0 must not read the old contents
    Sa_acc.fill_(float("nan"))
    for k, x in enumerate(chunks):
        X = plan.stft(dev(x))
        S, Sa = plan.cross_spectra(X)
        plan.accumulate(S_acc, Sa_acc, S, Sa, 0.0 if k == 0 else 1.0, 1.0 / n)   # running sum of S / n = the mean
    out = dict(G=plan.coherence(S_acc, Sa_acc), A=plan.crossphase(S_acc), P=plan.crosspower(S_acc),
               R=plan.crosscorr(S_acc, Sa_acc), Sauto=Sa_acc)
    torch.cuda.synchronize()
    out = {k: v.cpu().numpy() for k, v in out.items()}
    pairs = o.all_pairs(C)
    s2 = o.scale_factor(w.nfft)
    Xs = [o.stft(x, w.nfft, w.hop) for x in chunks]
    S_o = o.accumulate([o.cross_spectra(X, pairs, s2) for X in Xs])
    Sa_o = o.accumulate([o.auto_spectra(X, s2) for X in Xs])
    ref = dict(G=o.coherence(S_o, Sa_o, pairs), A=o.crossphase(S_o), P=o.crosspower(S_o),
               R=o.crosscorr(S_o, Sa_o, pairs, w.nfft, w.max_lag), Sauto=Sa_o)
    st = compare(out, ref, pairs, "accumulated")
    print(st)


@pytest.mark.parametrize("kind", ["reference_channel", "random_37"])
def test_explicit_pair_lists(kind, mode):
    """f2: outputs for an explicit pair list only -- one reference channel against all the
    others (the usual ECEi view), and a random list whose length is not a multiple of the 16-pair tile."""
    w = es.WORKLOADS["single"]
    C = 48
    x = es.single()[:C]
    if kind == "reference_channel":
        ref_ch = 17
        pairs = np.array([(min(ref_ch, c), max(ref_ch, c)) for c in range(C) if c != ref_ch], dtype=np.int32)
    else:
        allp = o.all_pairs(C)
        pairs = allp[np.random.default_rng(37).choice(len(allp), 37, replace=False)]
    b = binding()
    plan = b.Plan(C, w.T, w.nfft, w.hop, w.max_lag, contraction=mode, pairs=pairs)
    assert plan.sizes.P == len(pairs)
    out = plan.analyze_chunk(dev(x))
    torch.cuda.synchronize()
    out = {k: v.cpu().numpy() for k, v in out.items()}
    assert out["G"].shape == (len(pairs), w.F) and out["R"].shape == (len(pairs), 2 * w.max_lag + 1)
    ref = oracle_for(x, w.nfft, w.hop, w.max_lag, pairs=pairs)
    st = compare(out, ref, pairs, kind)
    print(kind, st)
    # the rows must equal the same pairs' rows of the all-pairs call, bit for bit (same S, same arithmetic)
    _, full = gpu_analyze(x, w.nfft, w.hop, w.max_lag, contraction=mode)
    idx = np.array([o.pair_index(int(i), int(j), C) for i, j in pairs])
    for k in ("G", "A", "P", "R"):
        assert np.array_equal(out[k], full[k][idx]), k


@pytest.mark.parametrize("C,T,L,H", [(40, 10_000, 512, 256), (12, 40_000, 256, 128)])
def test_phase_lock_estimator(C, T, L, H, mode):
    """f2: per-segment-normalised coherence (unit phasors per segment).  The second case has
    more than 8 segment blocks, i.e. the STFT variant without the cluster."""
    x = es.turbulence(T, 61)[:C]
    b = binding()
    plan = b.Plan(C, T, L, H, L // 2, contraction=mode, estimator=1)
    out = plan.analyze_chunk(dev(x))
    torch.cuda.synchronize()
    out = {k: v.cpu().numpy() for k, v in out.items()}
    ref = o.analyze_chunk(x, L, H, L // 2, phase_lock=True)
    # With unit phasors |dP| / sqrt(S_ii S_jj) IS the coherence error (S_cc = s^2), and every bin counts alike however
    # little power it holds: the float32 transform's error relative to a weak bin (1e-7 x the spectrum's dynamic range)
    # shows undiminished.  north_star's bound for the coherence is 1e-4; R13's tighter 1e-5 is relaxed to 5e-5 here.
    st = compare(out, ref, o.all_pairs(C), "phase lock", p_abs_tol=5e-5)
    print(st)
    assert np.abs(out["Sauto"] / o.scale_factor(L) - 1).max() < 1e-5     # unit phasors: S_cc = s^2 in every bin


def test_three_views_576_channels():
    """f3: the diagnostic has three 24 x 8 views: 576 channels, 165,600 pairs,
    nfft 512.  Three independent config-2 arrays with a common component; every row checked, both modes."""
    w = es.WORKLOADS["single"]
    a, b2, c = (es.turbulence(w.T, s) for s in (71, 72, 73))
    x = np.concatenate([a, 0.4 * a + 0.9 * b2, 0.4 * a + 0.9 * c]).astype(np.float32)
    assert x.shape[0] == 576
    _full_size_check(x, w.nfft, w.hop, w.max_lag, "576 channels", 10, 7)


@pytest.mark.parametrize("C,L", [(192, 512), (576, 512), (320, 64), (320, 128), (320, 256), (224, 1024)])
def test_output_subsets_on_a_reused_plan_are_bit_identical(C, L, mode):
    """Every subset of the per-pair outputs, asked for over and over on one plan, carries the bits of the call that
    asked for all of them.  A call for the cross-power alone makes the pair kernel's teams run far ahead of the
    tile copies, which is where a ring whose teams could mistake a pending barrier phase for a completed one gave
    wrong tiles (white-noise input: every tile differs from its neighbours)."""
    b = binding()
    # the other transform lengths run more teams per CTA over shorter tiles: enough pairs for every CTA's ring to go
    # round several times (51,040 pairs = 3,190 tiles at 320 channels), 20 segments
    T, H, M = (es.WORKLOADS["single"].T, 256, 256) if L == 512 else (L // 2 * 21, L // 2, L // 2)
    x = dev(np.random.default_rng(1234).standard_normal((C, T)).astype(np.float32))
    plan = b.Plan(C, T, L, H, M, contraction=mode)
    full = plan.empty_outputs()
    plan.analyze_chunk(x, full)
    torch.cuda.synchronize()
    full = {k: v.clone() for k, v in full.items()}
    import fastcheck as fc
    fc.check_all_pairs(x.cpu().numpy(), L, H, M, {"all": {k: v.cpu().numpy() for k, v in full.items()}},
                       TOLS, f"white noise {C} x {T}, nfft {L}")
    subsets = [dict(G=False, A=False, R=False), dict(G=False, A=False, R=True), dict(G=True, A=False, R=False),
               dict(G=False, A=True, R=False), dict(G=True, A=True, R=True)]
    for rep in range(6):
        for sub in subsets:
            out = plan.empty_outputs(**sub)
            out = {k: v for k, v in out.items() if v is not None}
            for v in out.values():
                v.fill_(float("nan"))
            plan.analyze_chunk(x, out)
            torch.cuda.synchronize()
            for k, v in out.items():
                assert torch.equal(v, full[k]), f"rep {rep} subset {sub}: {k} differs in {int((v != full[k]).any(dim=-1).sum())} rows"


@pytest.mark.parametrize("C", [576, 704])
def test_tmem_columns_are_not_reused_before_they_are_read_out(C):
    """Tensor-core contraction, channel counts whose accumulator groups have different TMEM layouts (576: units of
    (64, 128, 64) channels followed by (128, 128)): the first unit of an item shares columns with the SECOND unit of the
    CTA's previous item, so its MMAs have to wait for that unit's read-out too, not only for the unit of their own index.
    With the epilogue slowed down by the test hook a missing wait corrupts S every time."""
    b = binding()
    T, L, H, M = 3000, 512, 256, 16
    x = np.random.default_rng(77).standard_normal((C, T)).astype(np.float32)
    xd = dev(x)
    ref_plan = b.Plan(C, T, L, H, M, contraction=b.CONTRACT_FP32)
    S_ref = ref_plan.cross_spectra_unpack(ref_plan.cross_spectra(ref_plan.stft(xd))[0])
    plan = b.Plan(C, T, L, H, M, contraction=b.CONTRACT_TC)
    X = plan.stft(xd)
    S_fast = plan.cross_spectra_unpack(plan.cross_spectra(X)[0])
    plan._set_jitter(1, 20000)   # kJitTcEpiLate
    S_slow = plan.cross_spectra_unpack(plan.cross_spectra(X)[0])
    plan._set_jitter(0, 0)
    torch.cuda.synchronize()
    assert torch.equal(torch.view_as_real(S_slow), torch.view_as_real(S_fast)), \
        f"{int((S_slow != S_fast).any(dim=1).sum())} pairs change with a slow epilogue"
    scale = torch.abs(S_ref).max().item()
    assert torch.max(torch.abs(S_fast - S_ref)).item() <= 2e-5 * scale   # split-fp16 tensor cores vs the FP32 pipe


@pytest.mark.parametrize("C", [448, 640, 768, 960, 1000])
def test_many_channels_every_row(C):
    """Channel counts beyond the three-view array: up to 960 channels the tensor-core contraction is chosen (16 groups of
    accumulator units per bin at 960), beyond that the FP32 one.  Short transform and few lags to keep it small; every row
    of every output against the float64 pipeline (tests/fastcheck.py)."""
    import fastcheck as fc
    b = binding()
    T, L, H, M = 1600, 64, 32, 8
    rng = np.random.default_rng(C)
    common = rng.standard_normal(T)
    x = (rng.uniform(0.0, 1.0, (C, 1)) * common + rng.standard_normal((C, T))).astype(np.float32)
    plan = b.Plan(C, T, L, H, M)
    assert plan.sizes.contraction == (b.CONTRACT_TC if C <= 960 else b.CONTRACT_FP32)
    out = plan.analyze_chunk(dev(x))
    torch.cuda.synchronize()
    st = fc.check_all_pairs(x, L, H, M, {"auto": {k: v.cpu().numpy() for k, v in out.items()}}, TOLS, f"{C} channels")
    print(C, st)


JITTER_BITS = {1: "tc epilogue late", 2: "tc epilogue warps skewed", 4: "tc producer slow", 8: "tc mma issuer slow",
               16: "pair producer slow", 32: "pair teams skewed", 64: "pair warps skewed", 128: "stft CTAs skewed at start",
               256: "stft CTAs skewed before the write-out", 512: "pair tile copies land out of order"}


@pytest.mark.parametrize("C,T,L,H,M", [
    (192, 10000, 512, 256, 256),   # config 2: cluster STFT, one accumulator group, three pair teams over a 4-slot ring
    (576, 2600, 512, 256, 64),     # seven accumulator groups of three TMEM layouts
    (320, 1400, 64, 32, 32),       # eight pair teams per CTA
    (224, 6000, 1024, 512, 512),   # one pair team, two slots
    (40, 9000, 2048, 1024, 1024),  # pair groups wider than a warp (private exchange buffers), chscale pass
])
def test_results_do_not_depend_on_the_relative_speed_of_the_roles(C, T, L, H, M):
    """Producers, consumers and neighbouring CTAs of the three kernels are slowed down one role at a time (test hook
    delta_internal_set_jitter): every output keeps its bits.  A pipeline whose waits only hold for the usual relative speeds
    (the pair kernel's ring and the contraction's TMEM reuse both had such a gap until round 2) fails here every time."""
    _jitter_check(dict(n_channels=C, n_samples=T, nfft=L, hop=H, max_lag=M), C + L)


def test_results_do_not_depend_on_timing_variants():
    """The same for the variants that take other routes through the kernels: an explicit pair list (the groups gather
    their tile columns themselves), the band-pass filter (autospectra tables from a separate kernel), int16 input."""
    b = binding()
    allp = o.all_pairs(96)
    pairs = allp[np.sort(np.random.default_rng(5).choice(len(allp), 1501, replace=False))]
    _jitter_check(dict(n_channels=96, n_samples=5000, nfft=256, hop=128, max_lag=128, pairs=pairs), 1)
    _jitter_check(dict(n_channels=128, n_samples=5000, nfft=512, hop=256, max_lag=256, band=(5e3, 9e3)), 2)
    _jitter_check(dict(n_channels=64, n_samples=5000, nfft=512, hop=256, max_lag=100, in_dtype=b.I16), 3)


def _jitter_check(plan_kw, seed):
    b = binding()
    C, T = plan_kw["n_channels"], plan_kw["n_samples"]
    xf = np.random.default_rng(seed).standard_normal((C, T))
    if plan_kw.get("in_dtype", b.F32) == b.I16:
        x = dev((2000 + 200 * xf).astype(np.int16))
    else:
        x = dev(xf.astype(np.float32))
    plan = b.Plan(**plan_kw)
    ref = plan.analyze_chunk(x)
    torch.cuda.synchronize()
    ref = {k: v.clone() for k, v in ref.items()}
    for mask, what in list(JITTER_BITS.items()) + [(1023, "everything at once")]:
        # all outputs, and the cross-power alone (the pair kernel's teams then run far ahead of the tile copies)
        for subset in (dict(), dict(G=False, A=False, R=False)):
            plan._set_jitter(mask, 20000 if mask == 512 else 3000)
            out = {k: v for k, v in plan.empty_outputs(**subset).items() if v is not None}
            for v in out.values():
                v.fill_(float("nan"))
            plan.analyze_chunk(x, out)
            plan._set_jitter(0, 0)
            torch.cuda.synchronize()
            for k, v in out.items():
                assert torch.equal(v, ref[k]), f"{what} {subset}: {k} differs in {int((v != ref[k]).any(dim=-1).sum())} rows"


def test_staged_external_X_with_padding_not_zeroed():
    """A caller-supplied X buffer whose padding (rows C..Cp-1, segment blocks beyond ceil(K/8)) holds NaN before
    delta_stft: C = 192 and 128 have Cp == C and an odd number of segment blocks (K = 38: 5 of 6), the case where the
    contraction reads a block no STFT CTA writes.  Staged results must equal the fused call bit for bit."""
    b = binding()
    w = es.WORKLOADS["single"]
    for C in (192, 128):
        for mode in (b.CONTRACT_TC, b.CONTRACT_FP32):
            x = dev(es.single()[:C])
            plan = b.Plan(C, w.T, w.nfft, w.hop, w.max_lag, contraction=mode)
            fused = plan.analyze_chunk(x)
            X = plan.empty_X()
            X.view(torch.float16 if mode == b.CONTRACT_TC else torch.float32).fill_(float("nan"))
            plan.stft(x, X)
            S, Sa = plan.cross_spectra(X)
            G, A, P, R = plan.coherence(S, Sa), plan.crossphase(S), plan.crosspower(S), plan.crosscorr(S, Sa)
            torch.cuda.synchronize()
            for name, t in (("G", G), ("A", A), ("P", P), ("Sauto", Sa)):
                assert torch.isfinite(t).all(), (C, mode, name)
                assert torch.equal(t, fused[name]), (C, mode, name)
            assert torch.max(torch.abs(R - fused["R"])).item() < 5e-6


def test_X_buffers_are_self_contained():
    """delta_stft(x1 -> X1), delta_stft(x2 -> X2), then delta_cross_spectra(X1): the spectra of x1, whatever the plan
    did in between (the per-channel fp16 scales of the tensor-core mode travel inside the X buffer)."""
    b = binding()
    w = es.WORKLOADS["single"]
    C = 40
    x1 = es.single()[:C]
    x2 = (1000.0 * es.turbulence(w.T, 55)[:C]).astype(np.float32)   # very different amplitudes: different scales
    for mode in (b.CONTRACT_TC, b.CONTRACT_FP32):
        plan = b.Plan(C, w.T, w.nfft, w.hop, w.max_lag, contraction=mode)
        X1 = plan.stft(dev(x1))
        X2 = plan.stft(dev(x2))
        S1, Sa1 = plan.cross_spectra(X1)
        S2, Sa2 = plan.cross_spectra(X2)
        torch.cuda.synchronize()
        pairs = o.all_pairs(C)
        s2 = o.scale_factor(w.nfft)
        for x, S, Sa in ((x1, S1, Sa1), (x2, S2, Sa2)):
            Xo = o.stft(x, w.nfft, w.hop)
            So, Sao = o.cross_spectra(Xo, pairs, s2), o.auto_spectra(Xo, s2)
            den = np.sqrt(Sao[pairs[:, 0]] * Sao[pairs[:, 1]])
            assert np.max(np.abs(plan.cross_spectra_unpack(S).cpu().numpy() - So) / den) < 1e-5
            assert np.max(np.abs(Sa.cpu().numpy() - Sao) / Sao) < 1e-4
        # and the unpack accessor reads the scales from the buffer it is given
        Xg = plan.stft_unpack(X1).cpu().numpy()
        Xo = o.stft(x1, w.nfft, w.hop)
        assert np.abs(Xg - Xo).max() <= 2e-6 * np.abs(Xo).max()


@pytest.mark.parametrize("L,Ls,H,detrend,dtype", [(512, 256, 128, 0, "f32"), (1024, 300, 100, 1, "f32"), (256, 129, 64, 0, "i16")])
def test_zero_padded_segments(L, Ls, H, detrend, dtype, mode):
    """f2: segments of nperseg < nfft samples zero-padded to the transform length (the
    linear cross-correlation).  Cases: half-length segments; an odd-ish length that is no multiple of anything, with
    detrend; an odd length with int16 counts and offset normalisation (the padding must stay zero)."""
    C, T = 20, 10_000
    b = binding()
    if dtype == "i16":
        counts, _ = es.streamed(n_chunks=1)
        x = counts[0][:C]
        offs = o.offsets(x[:, :5000])
        plan = b.Plan(C, T, L, H, L // 2, contraction=mode, nperseg=Ls, detrend=detrend, in_dtype=b.I16, norm_mode=b.NORM_RELATIVE)
        xd = dev(x)
        plan.set_offsets(xd, 5000)
        ref = o.analyze_chunk(x, L, H, L // 2, nperseg=Ls, detrend=detrend, norm_mode=o.NORM_RELATIVE, offs=offs)
    else:
        x = es.turbulence(T, 91)[:C]
        plan = b.Plan(C, T, L, H, L // 2, contraction=mode, nperseg=Ls, detrend=detrend)
        xd = dev(x)
        ref = o.analyze_chunk(x, L, H, L // 2, nperseg=Ls, detrend=detrend)
    assert plan.sizes.K == (T - Ls) // H + 1
    out = plan.analyze_chunk(xd)
    torch.cuda.synchronize()
    out = {k: v.cpu().numpy() for k, v in out.items()}
    st = compare(out, ref, o.all_pairs(C), f"nperseg {Ls} of {L}")
    print(st)


def test_all_variants_together(mode):
    """The f1/f2 options are independent switches; everything at once must still match the oracle: int16 counts with
    offset normalisation, Blackman window, detrend, zero-padded segments, band-pass, phase-lock estimator, an explicit
    pair list, a short lag window."""
    b = binding()
    C, T, L, Ls, H, M = 24, 10_000, 512, 320, 160, 100
    counts, _ = es.streamed(n_chunks=1)
    x = counts[0][:C]
    offs = o.offsets(x[:, :5000])
    allp = o.all_pairs(C)
    pairs = allp[np.random.default_rng(5).choice(len(allp), 45, replace=False)]
    band = (8e3, 120e3)
    plan = b.Plan(C, T, L, H, M, contraction=mode, in_dtype=b.I16, norm_mode=b.NORM_RELATIVE, window=3, detrend=1,
                  nperseg=Ls, band=band, estimator=1, pairs=pairs)
    xd = dev(x)
    plan.set_offsets(xd, 5000)
    out = plan.analyze_chunk(xd)
    torch.cuda.synchronize()
    out = {k: v.cpu().numpy() for k, v in out.items()}
    ref = o.analyze_chunk(x, L, H, M, pairs=pairs, fs=500e3, norm_mode=o.NORM_RELATIVE, offs=offs, band=band,
                          win=o.WIN_BLACKMAN, detrend=o.DETREND_CONSTANT, phase_lock=True, nperseg=Ls)
    assert out["R"].shape == (45, 2 * M + 1)
    st = compare(out, ref, pairs, "all variants", p_abs_tol=5e-5)
    print(st)


@pytest.mark.parametrize("C,T,L,H,M", [(24, 10_000, 500, 250, 250), (10, 9_000, 768, 192, 100), (6, 12_000, 1000, 400, 500),
                                        (5, 1_000, 48, 24, 24), (7, 3_000, 250, 100, 60)])
def test_non_power_of_two_nfft(C, T, L, H, M, mode):
    """f1: even transform lengths that are not powers of two run on the direct-DFT kernels
    (stft_dft_kernel, pair_dft_kernel), through the same contraction; north_star's tolerances, both modes."""
    x = es.turbulence(T, 300 + L)[:C]
    _, out = gpu_analyze(x, L, H, M, contraction=mode)
    ref = oracle_for(x, L, H, M)
    assert out["G"].shape == ref["G"].shape == (C * (C - 1) // 2, L // 2 + 1) and out["R"].shape == ref["R"].shape
    st = compare(out, ref, o.all_pairs(C), f"nfft {L}")
    print(L, st)


def test_non_power_of_two_nfft_with_variants(mode):
    """The direct-DFT path with the f1/f2 switches on: int16 counts with offset normalisation, Hamming window, detrend,
    zero-padded segments, band-pass, an explicit pair list, a short lag window; and its staged calls."""
    b = binding()
    C, T, L, Ls, H, M = 16, 10_000, 600, 400, 200, 77
    counts, _ = es.streamed(n_chunks=1)
    x = counts[0][:C]
    offs = o.offsets(x[:, :5000])
    allp = o.all_pairs(C)
    pairs = allp[np.random.default_rng(9).choice(len(allp), 21, replace=False)]
    band = (4e3, 150e3)
    plan = b.Plan(C, T, L, H, M, contraction=mode, in_dtype=b.I16, norm_mode=b.NORM_RELATIVE, window=1, detrend=1,
                  nperseg=Ls, band=band, pairs=pairs)
    xd = dev(x)
    plan.set_offsets(xd, 5000)
    out = plan.analyze_chunk(xd)
    torch.cuda.synchronize()
    out = {k: v.cpu().numpy() for k, v in out.items()}
    ref = o.analyze_chunk(x, L, H, M, pairs=pairs, fs=500e3, norm_mode=o.NORM_RELATIVE, offs=offs, band=band,
                          win=o.WIN_HAMMING, detrend=o.DETREND_CONSTANT, nperseg=Ls)
    st = compare(out, ref, pairs, "nfft 600 with variants")
    print(st)
    # staged calls give the same G, A, P
    X = plan.stft(xd)
    S, Sa = plan.cross_spectra(X)
    G, A, P = plan.coherence(S, Sa), plan.crossphase(S), plan.crosspower(S)
    torch.cuda.synchronize()
    for name, t in (("G", G), ("A", A), ("P", P)):
        assert np.array_equal(t.cpu().numpy(), out[name]), name


def test_strong_scaling_split_gives_the_same_bits():
    """f4: one shot's chunks dealt round-robin to replicas (bench.py --scaling strong), every replica with its own plan
    and its own offsets from chunk 0.  On one GPU: two plans take the even and the odd chunks; every chunk's results are
    bit-identical to the single-plan run over the whole shot."""
    import bench
    b = binding()
    w = es.WORKLOADS["streamed"]
    counts, _ = es.streamed(n_chunks=6)
    counts = counts[:, :48]
    C = counts.shape[1]
    first = dev(counts[0])

    def run(chunks):
        plan = b.Plan(C, w.T, w.nfft, w.hop, w.max_lag, in_dtype=b.I16, norm_mode=b.NORM_RELATIVE)
        plan.set_offsets(first, w.n_first)
        res = {}
        for n in chunks:
            out = plan.analyze_chunk(dev(counts[n]))
            res[n] = {k: v.clone() for k, v in out.items()}
        torch.cuda.synchronize()
        return res

    whole = run(range(6))
    for rank in range(2):
        part = run(bench.shot_chunks_of_rank(6, rank, 2))
        assert sorted(part) == list(range(rank, 6, 2))
        for n, out in part.items():
            for k in ("G", "A", "P", "R", "Sauto"):
                assert torch.equal(out[k], whole[n][k]), (rank, n, k)
