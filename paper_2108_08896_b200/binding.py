"""Thin ctypes binding over libdelta_b200.so (include/delta.h): argument marshalling only.

PyTorch is used for device memory and streams; every step of the path runs in the library's CUDA
kernels.  There is no CPU fallback: if the library cannot be loaded, importing this module raises.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import torch

from . import build as _build

# ---- enums (include/delta.h) --------------------------------------------------------------
OK = 0
ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_ALIGNMENT, ERR_NO_WORKSPACE, ERR_CUDA, ERR_STATE, ERR_NO_MEMORY = -1, -2, -3, -4, -5, -6, -7
ERR_TOO_LARGE = -8
STATIC_SCRATCH_BYTES = 8 << 20   # DELTA_STATIC_SCRATCH_BYTES
WIN_HANN_PERIODIC = 0
SCALE_WINPOW, SCALE_NONE, SCALE_DENSITY, SCALE_SPECTRUM = 0, 1, 2, 3
F32, I16 = 0, 1
NORM_NONE, NORM_SUBTRACT, NORM_RELATIVE = 0, 1, 2
CONTRACT_AUTO, CONTRACT_FP32, CONTRACT_TC = 0, 1, 2


class DeltaConfig(C.Structure):
    _fields_ = [("n_channels", C.c_int32), ("n_samples", C.c_int32), ("nfft", C.c_int32), ("hop", C.c_int32),
                ("window", C.c_int32), ("scaling", C.c_int32), ("fs", C.c_float), ("in_dtype", C.c_int32),
                ("norm_mode", C.c_int32), ("max_lag", C.c_int32), ("n_pairs", C.c_int32),
                ("h_pairs", C.POINTER(C.c_int32)), ("contraction", C.c_int32),
                ("bp_lo_hz", C.c_float), ("bp_hi_hz", C.c_float), ("detrend", C.c_int32), ("estimator", C.c_int32), ("nperseg", C.c_int32)]


class DeltaSizes(C.Structure):
    _fields_ = [("n_segments", C.c_int32), ("n_bins", C.c_int32), ("n_lags", C.c_int32), ("contraction", C.c_int32),
                ("n_pairs", C.c_int64), ("workspace_bytes", C.c_int64), ("x_bytes", C.c_int64),
                ("s_bytes", C.c_int64), ("s_block_pairs", C.c_int64)]


EXPORTS = ["delta_plan_create", "delta_plan_destroy", "delta_plan_sizes", "delta_plan_set_workspace",
           "delta_set_offsets", "delta_get_offsets", "delta_stft", "delta_stft_unpack", "delta_cross_spectra",
           "delta_cross_spectra_unpack",
           "delta_coherence", "delta_coherence_static", "delta_crossphase", "delta_crosspower", "delta_crosscorr", "delta_accumulate", "delta_analyze_chunk",
           "delta_analyze_shot_host", "delta_plan_set_stage_events", "delta_last_launch_count", "delta_strerror", "delta_last_cuda_error",
           "delta_version"]


def _load() -> C.CDLL:
    path = _build.LIB
    if not os.path.exists(path) or _build.is_stale():
        path = _build.build()
    lib = C.CDLL(path)
    vp, i64, i32 = C.c_void_p, C.c_int64, C.c_int32
    lib.delta_plan_create.argtypes = [C.POINTER(DeltaConfig), C.POINTER(vp)]
    lib.delta_plan_destroy.argtypes = [vp]
    lib.delta_plan_sizes.argtypes = [vp, C.POINTER(DeltaSizes)]
    lib.delta_plan_set_workspace.argtypes = [vp, vp, C.c_size_t, vp]
    lib.delta_set_offsets.argtypes = [vp, vp, i64, i32, vp]
    lib.delta_get_offsets.argtypes = [vp, vp, vp]
    lib.delta_stft.argtypes = [vp, vp, i64, vp, vp]
    lib.delta_stft_unpack.argtypes = [vp, vp, vp, vp]
    lib.delta_cross_spectra.argtypes = [vp, vp, vp, vp, vp]
    lib.delta_cross_spectra_unpack.argtypes = [vp, vp, vp, vp]
    lib.delta_internal_set_trace.argtypes = [vp, vp]   # development hook, not part of the C ABI
    lib.delta_internal_set_jitter.argtypes = [vp, i32, i32]   # test hook, not part of the C ABI
    lib.delta_internal_probe_fabric.argtypes = [vp, C.c_size_t, vp, C.c_size_t, vp]   # measurement aid (csrc/probe.cu)
    lib.delta_coherence.argtypes = [vp, vp, vp, vp, vp]
    lib.delta_coherence_static.argtypes = [vp, vp, vp, vp, vp]
    lib.delta_crossphase.argtypes = [vp, vp, vp, vp]
    lib.delta_crosspower.argtypes = [vp, vp, vp, vp]
    lib.delta_crosscorr.argtypes = [vp, vp, vp, vp, vp]
    lib.delta_accumulate.argtypes = [vp, vp, vp, vp, vp, C.c_float, C.c_float, vp]
    lib.delta_analyze_chunk.argtypes = [vp, vp, i64, vp, vp, vp, vp, vp, vp]
    lib.delta_analyze_shot_host.argtypes = [vp, vp, i32, vp, i32, i32, vp, vp, vp, vp, vp, i64, i64, i64, i32,
                                            vp, vp, vp, vp, vp, vp]
    lib.delta_last_launch_count.argtypes = [vp]
    lib.delta_plan_set_stage_events.argtypes = [vp, C.POINTER(vp)]
    lib.delta_strerror.argtypes = [C.c_int]
    lib.delta_strerror.restype = C.c_char_p
    lib.delta_last_cuda_error.argtypes = []
    lib.delta_version.argtypes = []
    return lib


LIB = _load()
LIB_PATH = _build.LIB


class DeltaError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = LIB.delta_strerror(status).decode()
        if status == ERR_CUDA:
            msg += f" [cudaError {LIB.delta_last_cuda_error()}]"
        super().__init__(f"{where}: {msg} ({status})")


def _check(status: int, where: str) -> None:
    if status != OK:
        raise DeltaError(status, where)


def _ptr(t) -> int | None:
    return None if t is None else t.data_ptr()


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


@dataclass
class Sizes:
    K: int
    F: int
    n_lags: int
    contraction: int
    P: int
    workspace_bytes: int
    x_bytes: int
    s_bytes: int
    s_block_pairs: int


class Plan:
    """delta_plan + its workspace.  Method names follow the C entry points."""

    def __init__(self, n_channels, n_samples, nfft, hop, max_lag=None, in_dtype=F32, norm_mode=NORM_NONE,
                 scaling=SCALE_WINPOW, fs=500e3, contraction=CONTRACT_AUTO, window=WIN_HANN_PERIODIC,
                 device=None, allocate=True, band=None, detrend=0, pairs=None, estimator=0, nperseg=0):
        """band = (lo_hz, hi_hz): optional band-pass pre-processing (include/delta.h), None = off."""
        lo_hz, hi_hz = (0.0, 0.0) if band is None else band
        n_list, p_list = 0, None
        if pairs is not None:   # explicit pair list [n][2], i < j (copied by delta_plan_create)
            import numpy as np
            self._pairs = np.ascontiguousarray(np.asarray(pairs, dtype=np.int32).reshape(-1, 2))
            n_list, p_list = self._pairs.shape[0], self._pairs.ctypes.data_as(C.POINTER(C.c_int32))
        self.cfg = DeltaConfig(n_channels, n_samples, nfft, hop, window, scaling, fs, in_dtype, norm_mode,
                               nfft // 2 if max_lag is None else max_lag, n_list, p_list, contraction, lo_hz, hi_hz, detrend, estimator, nperseg)
        self._h = C.c_void_p()
        _check(LIB.delta_plan_create(C.byref(self.cfg), C.byref(self._h)), "delta_plan_create")
        sz = DeltaSizes()
        _check(LIB.delta_plan_sizes(self._h, C.byref(sz)), "delta_plan_sizes")
        self.sizes = Sizes(sz.n_segments, sz.n_bins, sz.n_lags, sz.contraction, sz.n_pairs, sz.workspace_bytes,
                           sz.x_bytes, sz.s_bytes, sz.s_block_pairs)
        self.C, self.T = n_channels, n_samples
        self.workspace = None
        if allocate:
            if not torch.cuda.is_available():
                raise RuntimeError("libdelta_b200 needs a CUDA device (there is no CPU fallback)")
            self.device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
            self.workspace = torch.empty(self.sizes.workspace_bytes, dtype=torch.uint8, device=self.device)
            _check(LIB.delta_plan_set_workspace(self._h, self.workspace.data_ptr(), self.workspace.numel(), _stream()),
                   "delta_plan_set_workspace")

    def __del__(self):
        h = getattr(self, "_h", None)
        if h and LIB is not None:
            LIB.delta_plan_destroy(h)
            self._h = None

    # -- allocation helpers (device memory comes from torch) -----------------------------------
    def empty_X(self):
        return torch.empty(self.sizes.x_bytes, dtype=torch.uint8, device=self.device)

    def empty_S(self):
        return torch.empty(self.sizes.s_bytes // 4, dtype=torch.float32, device=self.device)

    def empty_outputs(self, G=True, A=True, P=True, R=True, Sauto=True):
        s = self.sizes
        mk = lambda shape: torch.empty(shape, dtype=torch.float32, device=self.device)
        return dict(G=mk((s.P, s.F)) if G else None, A=mk((s.P, s.F)) if A else None,
                    P=mk((s.P, s.F)) if P else None, R=mk((s.P, s.n_lags)) if R else None,
                    Sauto=mk((self.C, s.F)) if Sauto else None)

    # -- C entry points ------------------------------------------------------------------------
    def set_offsets(self, x, n_first):
        _check(LIB.delta_set_offsets(self._h, x.data_ptr(), x.stride(0), n_first, _stream()), "delta_set_offsets")

    def get_offsets(self):
        import numpy as np
        out = np.empty(self.C, dtype=np.float64)
        _check(LIB.delta_get_offsets(self._h, out.ctypes.data, _stream()), "delta_get_offsets")
        return out

    def stft(self, x, X=None):
        X = self.empty_X() if X is None else X
        _check(LIB.delta_stft(self._h, x.data_ptr(), x.stride(0), X.data_ptr(), _stream()), "delta_stft")
        return X

    def stft_unpack(self, X):
        out = torch.empty((self.C, self.sizes.K, self.sizes.F, 2), dtype=torch.float32, device=self.device)
        _check(LIB.delta_stft_unpack(self._h, X.data_ptr(), out.data_ptr(), _stream()), "delta_stft_unpack")
        return torch.view_as_complex(out)

    def cross_spectra(self, X, S=None, Sauto=None):
        S = self.empty_S() if S is None else S
        Sauto = torch.empty((self.C, self.sizes.F), dtype=torch.float32, device=self.device) if Sauto is None else Sauto
        _check(LIB.delta_cross_spectra(self._h, X.data_ptr(), S.data_ptr(), Sauto.data_ptr(), _stream()),
               "delta_cross_spectra")
        return S, Sauto

    def cross_spectra_unpack(self, S):
        out = torch.empty((self.sizes.P, self.sizes.F, 2), dtype=torch.float32, device=self.device)
        _check(LIB.delta_cross_spectra_unpack(self._h, S.data_ptr(), out.data_ptr(), _stream()),
               "delta_cross_spectra_unpack")
        return torch.view_as_complex(out)

    def _set_trace(self, buf):
        _check(LIB.delta_internal_set_trace(self._h, None if buf is None else buf.data_ptr()), "delta_internal_set_trace")

    def _set_jitter(self, mask, ns):
        """Test hook (kJit* bits in csrc/delta_internal.h): the kernels' roles sleep at the named places."""
        _check(LIB.delta_internal_set_jitter(self._h, mask, ns), "delta_internal_set_jitter")

    def coherence(self, S, Sauto, G=None):
        G = torch.empty((self.sizes.P, self.sizes.F), dtype=torch.float32, device=self.device) if G is None else G
        _check(LIB.delta_coherence(self._h, S.data_ptr(), Sauto.data_ptr(), G.data_ptr(), _stream()), "delta_coherence")
        return G

    def coherence_static(self, S, Sauto, G=None):
        """delta_coherence with its scratch in the library's static device array: nothing is allocated by the call (pass
        G to keep torch from allocating the output)."""
        G = torch.empty((self.sizes.P, self.sizes.F), dtype=torch.float32, device=self.device) if G is None else G
        _check(LIB.delta_coherence_static(self._h, S.data_ptr(), Sauto.data_ptr(), G.data_ptr(), _stream()),
               "delta_coherence_static")
        return G

    def crossphase(self, S, A=None):
        A = torch.empty((self.sizes.P, self.sizes.F), dtype=torch.float32, device=self.device) if A is None else A
        _check(LIB.delta_crossphase(self._h, S.data_ptr(), A.data_ptr(), _stream()), "delta_crossphase")
        return A

    def crosspower(self, S, P=None):
        P = torch.empty((self.sizes.P, self.sizes.F), dtype=torch.float32, device=self.device) if P is None else P
        _check(LIB.delta_crosspower(self._h, S.data_ptr(), P.data_ptr(), _stream()), "delta_crosspower")
        return P

    def crosscorr(self, S, Sauto, R=None):
        R = torch.empty((self.sizes.P, self.sizes.n_lags), dtype=torch.float32, device=self.device) if R is None else R
        _check(LIB.delta_crosscorr(self._h, S.data_ptr(), Sauto.data_ptr(), R.data_ptr(), _stream()), "delta_crosscorr")
        return R

    def accumulate(self, S_acc, Sauto_acc, S, Sauto, w_acc, w_new):
        _check(LIB.delta_accumulate(self._h, _ptr(S_acc), _ptr(Sauto_acc), _ptr(S), _ptr(Sauto), w_acc, w_new, _stream()),
               "delta_accumulate")

    def analyze_chunk(self, x, out=None, stream=None):
        """stream: a torch.cuda.Stream (default: torch's current stream)."""
        out = self.empty_outputs() if out is None else out
        _check(LIB.delta_analyze_chunk(self._h, x.data_ptr(), x.stride(0), _ptr(out.get("G")), _ptr(out.get("A")),
                                       _ptr(out.get("P")), _ptr(out.get("R")), _ptr(out.get("Sauto")),
                                       _stream() if stream is None else stream.cuda_stream),
               "delta_analyze_chunk")
        return out

    def analyze_shot_host(self, h_x, slots, dev_out, strides=(0, 0, 0), host_out=None, set_offsets=False, n_first=0, ring=0):
        """h_x: pinned host tensor [n_chunks][C][T]; slots: device uint8 buffer (2 input slots);
        dev_out: dict of device tensors (chunk n in set n mod ring, or n if ring == 0, at set*stride elements);
        host_out: dict of pinned host tensors [n_chunks][...] or None."""
        host_out = host_out or {}
        _check(LIB.delta_analyze_shot_host(
            self._h, h_x.data_ptr(), h_x.shape[0], slots.data_ptr(), int(set_offsets), n_first,
            _ptr(dev_out.get("G")), _ptr(dev_out.get("A")), _ptr(dev_out.get("P")), _ptr(dev_out.get("R")),
            _ptr(dev_out.get("Sauto")), strides[0], strides[1], strides[2], ring,
            _ptr(host_out.get("G")), _ptr(host_out.get("A")), _ptr(host_out.get("P")), _ptr(host_out.get("R")),
            _ptr(host_out.get("Sauto")), _stream()), "delta_analyze_shot_host")

    def set_stage_events(self, events):
        """events: 4 torch.cuda.Event(enable_timing=True) that have been recorded once (so that their
        CUDA handles exist), or None to switch the hook off."""
        if events is None:
            _check(LIB.delta_plan_set_stage_events(self._h, None), "delta_plan_set_stage_events")
            return
        arr = (C.c_void_p * 4)(*[e.cuda_event for e in events])
        _check(LIB.delta_plan_set_stage_events(self._h, arr), "delta_plan_set_stage_events")

    def slot_bytes(self):
        esz = 2 if self.cfg.in_dtype == I16 else 4
        return 2 * ((self.C * self.T * esz + 255) // 256 * 256)

    @property
    def last_launch_count(self):
        return LIB.delta_last_launch_count(self._h)


def _probe_fabric(src, read_bytes, dst, write_bytes):
    """One launch of the SM <-> L2 probe (csrc/probe.cu; not part of the C ABI): bulk-copies `read_bytes` of `src` into
    shared memory and writes `write_bytes` of `dst`, one persistent CTA per SM."""
    _check(LIB.delta_internal_probe_fabric(None if src is None else src.data_ptr(), read_bytes,
                                           None if dst is None else dst.data_ptr(), write_bytes, _stream()),
           "delta_internal_probe_fabric")
