"""CPU-side checks of the C-ABI boundary (include/delta.h): the library loads, exports every
declared symbol, validates arguments with the documented status codes, and reports the sizes
SURVEY.md section 8 tabulates.  No compute call is made (there is no GPU here)."""
import ctypes as C
import os
import re

import pytest

from paper_2108_08896_b200 import binding as b

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "delta.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(delta_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    syms = declared_symbols()
    assert len(syms) >= 19
    assert set(syms) == set(b.EXPORTS)
    for s in syms:
        assert getattr(b.LIB, s) is not None
    for name in ("delta_stft", "delta_cross_spectra", "delta_coherence", "delta_crossphase", "delta_crosspower",
                 "delta_crosscorr"):   # the six calls BASELINE.json's north_star names
        assert name in syms
    assert b.LIB.delta_version() == 201
    assert os.path.dirname(b.LIB_PATH).endswith("paper_2108_08896_b200")  # in-tree, not site-packages


def mk(**kw):
    base = dict(n_channels=192, n_samples=10_000, nfft=512, hop=256, window=0, scaling=0, fs=500e3, in_dtype=0,
                norm_mode=0, max_lag=256, n_pairs=0, h_pairs=None, contraction=0)
    base.update(kw)
    return b.DeltaConfig(**base)


def create(cfg):
    h = C.c_void_p()
    rc = b.LIB.delta_plan_create(C.byref(cfg), C.byref(h))
    if rc == 0:
        b.LIB.delta_plan_destroy(h)
    else:
        assert not h.value
    return rc


@pytest.mark.parametrize("kw,status", [
    (dict(), b.OK),
    (dict(nfft=501, hop=250, max_lag=250), b.ERR_UNSUPPORTED),   # odd transform length
    (dict(nfft=8, hop=4, max_lag=4), b.ERR_UNSUPPORTED),
    (dict(nfft=8192, hop=4096, n_samples=100_000), b.ERR_UNSUPPORTED),
    (dict(n_samples=300), b.ERR_UNSUPPORTED),     # T < L
    (dict(max_lag=257), b.ERR_UNSUPPORTED),       # M > L/2
    (dict(hop=513), b.ERR_UNSUPPORTED),
    (dict(hop=0), b.ERR_INVALID_ARG),
    (dict(n_channels=0), b.ERR_INVALID_ARG),
    (dict(n_channels=5000), b.ERR_UNSUPPORTED),
    (dict(window=9), b.ERR_INVALID_ARG),
    (dict(scaling=9), b.ERR_INVALID_ARG),
    (dict(scaling=2, fs=0.0), b.ERR_INVALID_ARG),
    (dict(in_dtype=7), b.ERR_INVALID_ARG),
    (dict(norm_mode=-1), b.ERR_INVALID_ARG),
    (dict(max_lag=-1), b.ERR_INVALID_ARG),
    (dict(contraction=5), b.ERR_INVALID_ARG),
    (dict(n_pairs=3), b.ERR_INVALID_ARG),         # list announced but NULL
])
def test_plan_create_validation(kw, status):
    assert create(mk(**kw)) == status


def test_null_arguments():
    assert b.LIB.delta_plan_create(None, None) == b.ERR_INVALID_ARG
    h = C.c_void_p()
    assert b.LIB.delta_plan_create(None, C.byref(h)) == b.ERR_INVALID_ARG
    assert b.LIB.delta_plan_destroy(None) == b.ERR_INVALID_ARG
    assert b.LIB.delta_plan_sizes(None, None) == b.ERR_INVALID_ARG


def test_explicit_pair_list_through_the_raw_struct():
    arr = (C.c_int32 * 4)(0, 1, 0, 2)
    assert create(mk(n_pairs=2, h_pairs=C.cast(arr, C.POINTER(C.c_int32)))) == b.OK
    assert create(mk(n_pairs=2, h_pairs=None)) == b.ERR_INVALID_ARG


@pytest.mark.parametrize("name,K,F,P,nl", [("tiny", 15, 129, 28, 257), ("single", 38, 257, 18336, 513),
                                           ("long", 194, 513, 18336, 1025), ("wide", 94, 1025, 73536, 2049)])
def test_sizes_match_survey_table(name, K, F, P, nl):
    import ecei_synth as es
    w = es.WORKLOADS[name]
    p = b.Plan(w.C, w.T, w.nfft, w.hop, w.max_lag, allocate=False)
    s = p.sizes
    assert (s.K, s.F, s.P, s.n_lags) == (K, F, P, nl) == (w.K, w.F, w.P, 2 * w.max_lag + 1)
    B = s.s_block_pairs
    assert B in (4, 8, 16)
    assert s.s_bytes == -(-P // B) * s.F * B * 8
    assert s.workspace_bytes >= s.x_bytes + s.s_bytes


def test_compute_calls_refuse_without_workspace():
    p = b.Plan(8, 2048, 256, 128, allocate=False)
    assert b.LIB.delta_stft(p._h, 16, 2048, 16, None) == b.ERR_NO_WORKSPACE
    assert b.LIB.delta_analyze_chunk(p._h, 16, 2048, None, None, None, None, None, None) == b.ERR_NO_WORKSPACE
    assert b.LIB.delta_plan_set_workspace(p._h, None, 0, None) == b.ERR_INVALID_ARG
    assert b.LIB.delta_plan_set_workspace(p._h, 8, 1 << 30, None) == b.ERR_ALIGNMENT
    assert b.LIB.delta_plan_set_workspace(p._h, 256, 16, None) == b.ERR_NO_WORKSPACE
    assert b.LIB.delta_strerror(b.ERR_UNSUPPORTED).decode().startswith("unsupported")


def test_plan_needs_a_gpu_for_allocation():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        b.Plan(8, 2048, 256, 128)


def test_bandpass_config_validation():
    """include/delta.h: both band edges 0 = off; otherwise fs > 0 and 0 <= lo <= hi."""
    assert b.Plan(8, 2048, 256, 128, allocate=False, band=(5e3, 9e3)).sizes.F == 129
    assert b.Plan(8, 2048, 256, 128, allocate=False, band=None).sizes.F == 129
    for bad in [(9e3, 5e3), (-1.0, 5e3)]:
        with pytest.raises(b.DeltaError) as e:
            b.Plan(8, 2048, 256, 128, allocate=False, band=bad)
        assert e.value.status == b.ERR_INVALID_ARG
    with pytest.raises(b.DeltaError) as e:
        b.Plan(8, 2048, 256, 128, allocate=False, band=(5e3, 9e3), fs=0.0)
    assert e.value.status == b.ERR_INVALID_ARG
    assert b.LIB.delta_version() >= 101


def test_window_and_detrend_validation():
    for w in (0, 1, 2, 3):
        assert b.Plan(8, 2048, 256, 128, allocate=False, window=w, detrend=1).sizes.K == 15
    for kw in (dict(window=4), dict(window=-1), dict(detrend=2), dict(detrend=-1)):
        with pytest.raises(b.DeltaError) as e:
            b.Plan(8, 2048, 256, 128, allocate=False, **kw)
        assert e.value.status == b.ERR_INVALID_ARG


def test_explicit_pair_list_validation():
    """f2: explicit pair lists (e.g. one reference channel against all others); entries must satisfy 0 <= i < j < C."""
    p = b.Plan(8, 2048, 256, 128, allocate=False, pairs=[(0, 3), (2, 7), (0, 1)])
    assert p.sizes.P == 3
    for bad in ([(3, 3)], [(4, 2)], [(0, 8)], [(-1, 2)]):
        with pytest.raises(b.DeltaError) as e:
            b.Plan(8, 2048, 256, 128, allocate=False, pairs=bad)
        assert e.value.status == b.ERR_INVALID_ARG


def test_nperseg_validation():
    assert b.Plan(8, 2048, 256, 64, allocate=False, nperseg=128).sizes.K == (2048 - 128) // 64 + 1
    assert b.Plan(8, 2048, 256, 128, allocate=False, nperseg=0).sizes.K == 15
    for kw, st in ((dict(nperseg=300), b.ERR_INVALID_ARG), (dict(nperseg=-1), b.ERR_INVALID_ARG),
                   (dict(nperseg=100, hop=128), b.ERR_UNSUPPORTED)):
        args = dict(hop=128)
        args.update(kw)
        with pytest.raises(b.DeltaError) as e:
            b.Plan(8, 2048, 256, allocate=False, **args)
        assert e.value.status == st


def test_header_is_plain_c_and_links(tmp_path):
    """The boundary is a C ABI: include/delta.h must compile as C99 (no C++ or CUDA types in the signatures) and a
    plain C program must link against the shared library and create / destroy a plan without a GPU."""
    import shutil
    import subprocess
    gcc = shutil.which("gcc")
    if gcc is None:
        pytest.skip("no gcc")
    src = tmp_path / "use_delta.c"
    src.write_text('''
#include <stdio.h>
#include <string.h>
#include "delta.h"
int main(void) {
  delta_config c;
  memset(&c, 0, sizeof c);
  c.n_channels = 192; c.n_samples = 10000; c.nfft = 512; c.hop = 256; c.max_lag = 256; c.fs = 500e3f;
  delta_plan *p = NULL;
  delta_sizes s;
  if (delta_plan_create(&c, &p) != DELTA_OK || delta_plan_sizes(p, &s) != DELTA_OK) return 1;
  printf("%d %d %lld %d\\n", s.n_segments, s.n_bins, (long long)s.n_pairs, delta_version());
  c.nfft = 501;
  delta_plan *q = NULL;
  if (delta_plan_create(&c, &q) != DELTA_ERR_UNSUPPORTED || q != NULL) return 2;
  return delta_plan_destroy(p) == DELTA_OK ? 0 : 3;
}
''')
    exe = tmp_path / "use_delta"
    libdir = os.path.dirname(b.LIB_PATH)
    subprocess.run([gcc, "-std=c99", "-Wall", "-Wextra", "-pedantic", "-Werror", "-I", os.path.join(ROOT, "include"),
                    str(src), "-o", str(exe), "-L", libdir, "-ldelta_b200", f"-Wl,-rpath,{libdir}"], check=True)
    out = subprocess.run([str(exe)], capture_output=True, text=True)
    assert out.returncode == 0, out
    assert out.stdout.split()[:3] == ["38", "257", "18336"]


def test_non_power_of_two_nfft_is_accepted():
    """Even transform lengths that are not powers of two take the direct-DFT kernels (f1): the plan is created and
    reports K, F as the definitions give them."""
    p = b.Plan(192, 10_000, 500, 250, 250, allocate=False)
    assert p.sizes.K == (10_000 - 500) // 250 + 1 and p.sizes.F == 251 and p.sizes.n_lags == 501
