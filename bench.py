#!/usr/bin/env python
"""bench.py -- throughput of the all-channel-pairs spectral path (delta_analyze_chunk) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload single|long|streamed|wide|views3] [--scaling weak|strong]

One "step" = one pass of the whole hot path (STFT -> cross-spectra -> coherence, cross-phase,
cross-power, cross-correlation for all pairs) over one synthetic ECEi-shaped chunk.  The default
workload is BASELINE.json configs[1] (192 channels x 10,000 float32 samples, nfft 512, 50 %
overlap, 18,336 pairs).  Prints ONE JSON line (rank 0).  See DESIGN.md section 8 for what each
number means.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import ecei_synth as es  # noqa: E402

METRIC = "channel_pair_spectra_per_s"
UNIT = "pair-spectra/s"
N_IN = 4            # rotating input chunks
L2_BYTES = 126e6    # outputs rotate over enough buffer sets to exceed this
REPEATS = 5         # the K-step timed region is repeated and the median reported (steps stays K)

# the three-view workload: not a BASELINE config, so it lives here
VIEWS3 = es.Workload("views3", 576, 10_000, 512, 256, 256, "f32")


def workload(name):
    return VIEWS3 if name == "views3" else es.WORKLOADS[name]


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            d = json.load(fh)
        return dict(hbm_gbs=float(d["hbm_gbs"]), bf16_tflops=float(d.get("bf16_tflops", 1590.0)),
                    bf16_tflops_sustained=float(d.get("bf16_tflops_sustained", 1400.0)),
                    sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler:
    """Polls NVML for SM clock and throttle reasons while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.002):
        self.index, self.period = index, period_s
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _poll(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                 "hw_power_brake_slowdown": 0x80, "sw_power_cap": 0x4, "sync_boost": 0x10}
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def start(self):
        if self.nv is not None:
            self._thread = threading.Thread(target=self._poll, daemon=True)
            self._thread.start()

    def stop(self):
        self._stop.set()
        if self._thread is not None:
            self._thread.join()
        if not self.samples and self.nv is not None:   # region shorter than one period: one sample now
            try:
                self.samples.append(float(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
            except Exception:
                pass
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def max_over_ranks(value: float, world: int, device: str = "cuda") -> float:
    """Timing rule: the step time of a multi-rank run is the MAX over ranks."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def rank_chunk_seeds(rank: int, n: int = N_IN):
    """Weak scaling: every rank analyses its own chunks (disjoint seeds), no data-path collective."""
    return [2 + 100 * i + 1000 * rank for i in range(n)]


def shot_chunks_of_rank(n_chunks: int, rank: int, world: int):
    """Strong scaling of one shot (chunks are independent): chunk n goes to rank n mod world."""
    return list(range(rank, n_chunks, world))


def aggregate_value(pairs_per_step: int, steps: int, world: int, ms_max: float) -> float:
    """Whole-job throughput: units processed by all ranks / max-over-ranks time."""
    return world * pairs_per_step * steps / (ms_max * 1e-3)


def physical_gpu_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


def alg_bytes(w):
    """Algorithmic bytes per chunk: read the chunk once, write every requested
    output once.  X, S and tables are implementation intermediates and are not counted."""
    inp = w.C * w.T * (2 if w.dtype == "i16" else 4)
    gap = 3 * w.P * w.F * 4
    rho = w.P * (2 * w.max_lag + 1) * 4
    auto = w.C * w.F * 4
    return dict(input=inp, gap=gap, rho=rho, auto=auto, total=inp + gap + rho + auto)


def host_chunks(w, rank, n):
    """n float32 (or, for the streamed shot, int16) chunks [C][T] of the workload, seeded per rank."""
    if w.name == "views3":
        out = []
        for s in rank_chunk_seeds(rank, n):
            a, b2, c = (es.turbulence(w.T, s + k) for k in (0, 7, 13))
            out.append(np.concatenate([a, 0.4 * a + 0.9 * b2, 0.4 * a + 0.9 * c]).astype(np.float32))
        return out
    if w.name == "wide":
        return [es.wide(s, s + 50) for s in rank_chunk_seeds(rank, n)]
    return [es.turbulence(w.T, s) for s in rank_chunk_seeds(rank, n)]


def oracle_chunk(x, w):
    from oracle import delta_oracle as o
    return o.analyze_chunk(x, w.nfft, w.hop, w.max_lag)


def blas_threads():
    try:
        import threadpoolctl
        return max([p.get("num_threads", 1) for p in threadpoolctl.threadpool_info()] or [1])
    except Exception:
        return os.cpu_count() or 1


def cpu_baseline(w, budget_s=10.0):
    """Two CPU figures on this box's host cores, on a bounded sample of the workload (same generator, float32 input):
    the oracle as it stands (float64, direct DFT) and -- labelled as such -- the same float64 pipeline with numpy's FFT
    (BASELINE.md section 3).  Channel subsets keep each at ~10 s; the unit is still pair-spectra/s."""
    from oracle import fft_baseline as fb
    x_full = host_chunks(w, 0, 1)[0] if w.dtype == "f32" else es.turbulence(w.T, 9000)
    # cost grows with the pairs: time a few channels first, then as many as the budget allows; if a whole chunk takes less
    # than the budget, whole chunks are repeated until ~budget seconds of CPU work have been timed
    def timed(fn, x):
        t0 = time.perf_counter()
        fn(x)
        return time.perf_counter() - t0

    def sample(fn, n0):
        t_small = timed(fn, x_full[:n0])
        n = int(max(n0, min(w.C, n0 * np.sqrt(budget_s / max(t_small, 1e-3)))))
        reps, t = 0, 0.0
        while True:
            t += timed(fn, x_full[:n])
            reps += 1
            if t >= budget_s or n < w.C or reps >= 64:
                break
        return n, reps, t

    n_or, r_or, t_or = sample(lambda x: oracle_chunk(x, w), min(16, w.C))
    P_or = r_or * (n_or * (n_or - 1) // 2)
    n_fb, r_fb, t_fb = sample(lambda x: fb.analyze_chunk(x, w.nfft, w.hop, w.max_lag), min(48, w.C))
    P_fb = r_fb * (n_fb * (n_fb - 1) // 2)
    cores = blas_threads()
    return {"value": P_or / t_or, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{r_or} x the first {n_or} channels ({n_or * (n_or - 1) // 2} pairs) of one '{w.name}' chunk ({w.T} samples, "
                      f"nfft {w.nfft}), all four quantities, float64 direct-DFT numpy oracle, {t_or:.1f} s", "seconds": t_or,
            "library_fft": {"value": P_fb / t_fb, "unit": UNIT, "cores": cores, "kind": "CPU, library FFT",
                            "sample": f"{r_fb} x the first {n_fb} channels ({n_fb * (n_fb - 1) // 2} pairs) of the same chunk, float64 numpy "
                                      f"rfft / matmul / ifft (oracle/fft_baseline.py, pinned to the oracle), {t_fb:.1f} s",
                            "seconds": t_fb}}


# --------------------------------------------------------------------------------------------
def run_reference(args):
    """--impl reference: for this tier the reference arm is the oracle, timed on host cores."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = workload(args.workload)
    x_full = host_chunks(w, 0, 1)[0]
    # bounded sample per step so that (W + K) steps end within a few minutes
    n0 = min(32, w.C)
    t0 = time.perf_counter()
    oracle_chunk(x_full[:n0], w)
    t32 = time.perf_counter() - t0
    budget = 150.0
    steps_total = args.steps + args.warmup
    n_ch = int(max(8, min(w.C, n0 * np.sqrt(budget / steps_total / max(t32, 1e-3)))))
    x = x_full[:n_ch]
    P = n_ch * (n_ch - 1) // 2
    for _ in range(args.warmup):
        oracle_chunk(x, w)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_chunk(x, w)
    dt = time.perf_counter() - t0
    val = P * args.steps / dt
    sample = (f"each step = the first {n_ch} channels ({P} pairs) of one '{w.name}' chunk "
              f"({w.T} samples, nfft {w.nfft}), all four quantities")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "channels": w.C, "samples": w.T, "nfft": w.nfft, "hop": w.hop,
                       "segments": w.K, "pairs": w.P, "max_lag": w.max_lag, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": blas_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libdelta_b200 has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    from paper_2108_08896_b200 import binding as b

    w = workload(args.workload)
    streamed = w.name == "streamed"
    strong = args.scaling == "strong"
    if strong and not streamed:
        raise SystemExit("--scaling strong splits the chunks of one shot over the ranks: use --workload streamed")
    peaks = load_peaks()
    contraction = {"auto": b.CONTRACT_AUTO, "fp32": b.CONTRACT_FP32, "tc": b.CONTRACT_TC}[args.contraction]
    plan_kw = dict(contraction=contraction)
    if streamed:
        plan_kw.update(in_dtype=b.I16, norm_mode=b.NORM_RELATIVE)
    # chunks are independent, so `inflight` of them are kept in flight: one plan (= one workspace)
    # and one CUDA stream each; a plan is never used from two streams at once (include/delta.h)
    plans = [b.Plan(w.C, w.T, w.nfft, w.hop, w.max_lag, **plan_kw) for _ in range(max(1, args.inflight))]
    streams = [torch.cuda.Stream() for _ in plans]
    plan = plans[0]
    s = plan.sizes
    ab = alg_bytes(w)
    K, W = args.steps, args.warmup

    # ---- inputs resident in HBM before the timed region ------------------------------------------
    if streamed:
        # one shot: 250 int16 chunks; weak scaling: every rank its own shot; strong: rank r takes chunks r, r + world, ...
        counts, _ = es.streamed(seed=4 + (0 if strong else 1000 * rank), n_chunks=w.n_chunks)
        mine = shot_chunks_of_rank(w.n_chunks, rank, world) if strong else list(range(w.n_chunks))
        shot_dev = torch.from_numpy(counts).cuda()
        xs = [shot_dev[n] for n in mine]
        first = shot_dev[0]                                      # the offsets come from the first chunk of the shot (R1);
        for p_ in plans:                                         # every rank recomputes them from chunk 0, no broadcast
            p_.set_offsets(first, w.n_first)
        xs_host = None
    else:
        xs_host = host_chunks(w, rank, N_IN)
        xs = [torch.from_numpy(x).cuda() for x in xs_host]
    out_bytes = ab["gap"] + ab["rho"] + ab["auto"]
    n_out = max(2 * len(plans), int(np.ceil(4.5 * L2_BYTES / out_bytes)))
    n_out = (n_out + len(plans) - 1) // len(plans) * len(plans)
    outs = [plan.empty_outputs() for _ in range(n_out)]
    n_in = len(xs)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    per_stream = n_out // len(plans)

    def out_set(k):
        # every stream rotates over its own output sets (no two streams ever write the same buffers)
        i = k % len(plans)
        return i * per_stream + (k // len(plans)) % per_stream

    def steps(n, first_k=0):
        # step k runs on stream k % inflight; a buffer set is reused only after n_out further steps
        for k in range(first_k, first_k + n):
            i = k % len(plans)
            plans[i].analyze_chunk(xs[k % n_in], outs[out_set(k)], stream=streams[i])

    main = torch.cuda.current_stream()

    def timed(n):
        # CUDA events on the launching stream; the side streams fork from e0 and join before e1
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(main)
        for st in streams:
            st.wait_event(e0)
        steps(n)
        for st in streams:
            main.wait_stream(st)
        e1.record(main)
        return e0, e1

    steps(max(W, 3))
    torch.cuda.synchronize()
    launches_per_step = plan.last_launch_count

    # ---- timed region: exactly K steps, repeated; the median of the repeats is reported --------
    sampler = ClockSampler(physical_gpu_index(local_rank))
    barrier()
    sampler.start()
    reps, t_cpu = [], []
    for _ in range(REPEATS):
        barrier()
        t0 = time.perf_counter()
        e0, e1 = timed(K)
        t_cpu.append(time.perf_counter() - t0)   # host time to enqueue the K steps (must stay below the device time)
        barrier()
        reps.append(max_over_ranks(e0.elapsed_time(e1), world))
    clocks = sampler.stop()
    ms = float(np.median(reps))

    # the same K steps on ONE stream (no chunk overlap), for reference
    serial = []
    for _ in range(3):
        barrier()
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record()
        for k in range(K):
            plan.analyze_chunk(xs[k % n_in], outs[k % n_out])
        g1.record()
        barrier()
        serial.append(max_over_ranks(g0.elapsed_time(g1), world))
    ms_serial = float(np.median(serial))

    # ---- per-stage durations (same steps again, events recorded between the kernels) -------------
    Ks = min(K, 400)
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(Ks)]
    for row in evs:
        for e in row:
            e.record()
    torch.cuda.synchronize()
    for k in range(Ks):
        plan.set_stage_events(evs[k])
        plan.analyze_chunk(xs[k % n_in], outs[k % n_out])
    plan.set_stage_events(None)
    torch.cuda.synchronize()
    stage_ms = np.array([[row[i].elapsed_time(row[i + 1]) for i in range(3)] for row in evs])
    stage_mean = np.median(stage_ms, axis=0)
    tc = s.contraction == b.CONTRACT_TC
    flops_contract = 8.0 * (w.P + w.C) * w.F * w.K   # useful FP32-equivalent flops of Eq. (1a), Hermitian half
    alu_peak_tf = 148 * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
    stages = [
        {"kernel": "stft_kernel" + ("+chscale_kernel" if tc and s.K > 64 else ""), "ms": float(stage_mean[0]), "bound": "hbm",
         "alg_bytes": ab["input"], "achieved": ab["input"] / (stage_mean[0] * 1e-3) / 1e9, "unit": "GB/s"},
        {"kernel": "contract_tc_kernel" if tc else "contract_fp32_kernel", "ms": float(stage_mean[1]),
         "bound": "tensor" if tc else "alu", "alg_flops": flops_contract,
         "achieved": flops_contract / (stage_mean[1] * 1e-3) / 1e12, "unit": "TFLOP/s"},
        {"kernel": "pair_kernel", "ms": float(stage_mean[2]), "bound": "hbm",
         "alg_bytes": ab["gap"] + ab["rho"], "achieved": (ab["gap"] + ab["rho"]) / (stage_mean[2] * 1e-3) / 1e9,
         "unit": "GB/s"},
    ]
    dom = int(np.argmax(stage_mean))
    d = stages[dom]
    if d["bound"] == "hbm":
        peak, peak_src = peaks["hbm_gbs"], f"MEASURED_PEAKS.json hbm_gbs ({peaks['source']})"
    elif d["bound"] == "alu":
        peak, peak_src = alu_peak_tf, "148 SMs x 128 FP32 lanes x 2 flop x sm_max_mhz (DESIGN.md section 7)"
    else:
        peak, peak_src = peaks["bf16_tflops"], f"MEASURED_PEAKS.json bf16_tflops burst ({peaks['source']}); fp16 kind::f16"
    # DRAM traffic of the dominant kernel per launch: from the committed ncu capture of this workload (dram bytes summed over
    # consecutive steps with --cache-control none, profiles/r02_traffic.json.txt); null if there is none for it
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "r02_traffic.json.txt")
    if os.path.exists(tpath):
        try:
            traffic = json.load(open(tpath)).get(w.name, {}).get(d["kernel"].split("+")[0])
        except Exception:
            traffic = None
    # SM <-> L2 crossbar bytes of the dominant kernel per launch (ncu, profiles/r02_xbar.json.txt) held against the rates
    # `bench.py --probe-fabric` measured (profiles/r02_probe_fabric.json.txt): reads and writes add up on that path, so
    # bound_us = write / write rate + read / read rate.  Committed captures, not live values; null without them.
    xbar = None
    try:
        xb = json.load(open(os.path.join(ROOT, "profiles", "r02_xbar.json.txt"))).get(w.name, {}).get(d["kernel"].split("+")[0])
        pr = {c["case"].split(" ")[0]: c["gbs"] for c in json.load(open(os.path.join(ROOT, "profiles", "r02_probe_fabric.json.txt")))["cases"][:2]}
        if xb:
            bound_us = xb["write_bytes"] / pr["write"] / 1e3 + xb["read_bytes"] / pr["read"] / 1e3
            xbar = {"read_bytes": xb["read_bytes"], "write_bytes": xb["write_bytes"], "probe_read_gbs": pr["read"],
                    "probe_write_gbs": pr["write"], "bound_us": bound_us, "frac": bound_us / (d["ms"] * 1e3)}
    except Exception:
        xbar = None
    roofline = {"kernel": d["kernel"], "bound": d["bound"], "achieved": d["achieved"], "peak": peak, "unit": d["unit"],
                "frac": d["achieved"] / peak, "traffic": traffic, "peak_source": peak_src,
                "kernel_ms": d["ms"], "kernel_share_of_step": float(stage_mean[dom] / stage_mean.sum()), "xbar": xbar,
                "stages": stages,
                "pipeline": {"alg_bytes_per_step": ab["total"], "achieved": ab["total"] / (ms / K * 1e-3) / 1e9,
                             "unit": "GB/s", "frac_of_measured_hbm": ab["total"] / (ms / K * 1e-3) / 1e9 / peaks["hbm_gbs"],
                             "frac_of_8TBs": ab["total"] / (ms / K * 1e-3) / 1e9 / 8000.0}}

    # ---- end to end through the C ABI with HOST buffers (H2D + D2H inside the timed region) ------
    if streamed:
        # the whole shot (this rank's chunks) from pinned host memory through delta_analyze_shot_host: H2D of chunk n+1 on
        # the side stream under the kernels of chunk n; outputs stay on the device, the
        # autospectra of every chunk are read back (the per-step result)
        sel = counts[mine]
        h_x = torch.from_numpy(np.ascontiguousarray(sel)).pin_memory()
        n_e2e = h_x.shape[0]
        host_out = dict(Sauto=torch.empty((n_e2e, w.C, s.F)).pin_memory())
        d2h = ab["auto"]
        call = ("delta_analyze_shot_host: the shot's int16 chunks from pinned host memory, H2D on the side stream, G/A/P/rho "
                "left on the device (rotating sets), autospectra of every chunk copied back")
    else:
        n_e2e = max(1, min(K, 12 if out_bytes < 200e6 else 3))
        h_x = torch.from_numpy(np.stack([xs_host[i % N_IN] for i in range(n_e2e)])).pin_memory()
        host_out = dict(G=torch.empty((n_e2e, s.P, s.F)).pin_memory(), A=torch.empty((n_e2e, s.P, s.F)).pin_memory(),
                        P=torch.empty((n_e2e, s.P, s.F)).pin_memory(), R=torch.empty((n_e2e, s.P, s.n_lags)).pin_memory(),
                        Sauto=torch.empty((n_e2e, w.C, s.F)).pin_memory())
        d2h = out_bytes
        call = "delta_analyze_shot_host: pinned host chunks in, all five outputs copied back to pinned host memory"
    slots = torch.empty(plan.slot_bytes(), dtype=torch.uint8, device="cuda")
    dev_out = dict(G=torch.empty((2, s.P, s.F), device="cuda"), A=torch.empty((2, s.P, s.F), device="cuda"),
                   P=torch.empty((2, s.P, s.F), device="cuda"), R=torch.empty((2, s.P, s.n_lags), device="cuda"),
                   Sauto=torch.empty((2, w.C, s.F), device="cuda"))

    def e2e_once():
        # two device output sets: the copy-back of chunk n runs on the library's copy stream under the kernels of chunk n + 1
        plan.analyze_shot_host(h_x, slots, dev_out, strides=(s.P * s.F, s.P * s.n_lags, w.C * s.F), host_out=host_out,
                               set_offsets=streamed, n_first=w.n_first, ring=2)

    e2e_once()
    barrier()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record()
    e2e_once()
    f1.record()
    barrier()
    e2e_ms = max_over_ranks(f0.elapsed_time(f1), world)
    e2e = {"value": aggregate_value(w.P, n_e2e, world, e2e_ms), "unit": UNIT, "h2d_bytes_per_step": ab["input"],
           "d2h_bytes_per_step": d2h, "steps": n_e2e, "ms_per_step": e2e_ms / n_e2e, "call": call}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(w)

    if rank == 0:
        value = aggregate_value(w.P, K, world, ms)
        scaling = "strong" if strong else "weak"
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": ms / K, "higher_is_better": True, "scaling": scaling, "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "config": {"workload": w.name, "channels": w.C, "samples": w.T, "nfft": w.nfft, "hop": w.hop,
                           "segments": w.K, "pairs": w.P, "max_lag": w.max_lag, "input": w.dtype, "outputs": "G,A,P,rho,autospectra",
                           "contraction": "tcgen05 split-fp16" if tc else "fp32 fma",
                           "l2_policy": f"inputs rotate over {n_in} chunks, outputs over {n_out} buffer sets "
                                        f"({n_out * out_bytes / 1e6:.0f} MB > 126 MB L2)",
                           "chunks_in_flight": len(plans), "timed_region_repeats": REPEATS,
                           "parallelism": (f"one shot's chunks dealt round-robin to {world} replicas, no collective" if strong
                                           else f"chunk-parallel replicas x{world}, no collective")},
                "ms_per_step_repeats": [r / K for r in reps],
                "ms_per_step_one_stream": ms_serial / K, "host_enqueue_ms_per_step": 1e3 * float(np.median(t_cpu)) / K,
                "samples_per_s": world * w.C * w.T * K / (ms * 1e-3),
                "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_step * K, "roofline": roofline,
                "cpu_baseline": cpu}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def probe_fabric():
    """What the path between the SMs and L2 sustains (paper_2108_08896_b200/csrc/probe.cu): the rate the crossbar bytes
    of the kernels (ncu: l1tex__m_xbar2l1tex_read_bytes + l1tex__m_l1tex2xbar_write_bytes) are held against in
    DESIGN.md section 7.  Sizes are those of config 2: S (37.9 MB, L2 resident) read, the outputs (94.2 MB, rotating over
    six buffers so that they drain to HBM) written.  Prints one JSON line."""
    import torch
    from paper_2108_08896_b200 import binding as b
    dev = torch.device("cuda", 0)
    rbytes, wbytes = 37978112 // 32768 * 32768, 94173696 // 16 * 16
    src = torch.ones(rbytes, dtype=torch.uint8, device=dev)
    dsts = [torch.empty(wbytes, dtype=torch.uint8, device=dev) for _ in range(6)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    out = {"probe": "sm_l2_fabric", "unit": "GB/s", "launch": "one CTA per SM, 800 threads", "cases": []}
    for name, rb, wb in (("read (bulk copy to shared memory)", rbytes, 0), ("write (16-byte streaming stores)", 0, wbytes),
                         ("read + write", rbytes, wbytes)):
        for r in range(12):
            b._probe_fabric(src, rb, dsts[r % 6], wb)
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()   # 60 launches back to back: a 5 us kernel is not to be timed at the host's launch rate
        with torch.cuda.graph(graph):
            for r in range(60):
                b._probe_fabric(src, rb, dsts[r % 6], wb)
        graph.replay()
        torch.cuda.synchronize()
        times = []
        for rep in range(5):
            e0.record()
            graph.replay()
            e1.record()
            torch.cuda.synchronize()
            times.append(e0.elapsed_time(e1) / 60)
        ms = sorted(times)[2]
        out["cases"].append({"case": name, "read_bytes": rb, "write_bytes": wb, "us_per_launch": round(ms * 1e3, 2),
                             "gbs": round((rb + wb) / ms / 1e6, 1)})
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="single", choices=["single", "long", "streamed", "wide", "views3"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--contraction", default="auto", choices=["auto", "fp32", "tc"])
    ap.add_argument("--inflight", type=int, default=None,
                    help="independent chunks kept in flight (plans x streams); default 2, 1 for `wide`, whose kernels are long "
                         "enough to fill the GPU on their own (two in flight measured 919 vs 871 us per chunk)")
    ap.add_argument("--probe-fabric", action="store_true", help="measure the SM <-> L2 rates instead of the workload")
    args = ap.parse_args()
    if args.inflight is None:
        args.inflight = 1 if args.workload == "wide" else 2
    if args.probe_fabric:
        probe_fabric()
        return
    if args.impl == "reference":
        args.steps = 20 if args.steps is None else args.steps   # defaults sized per arm
        args.warmup = 3 if args.warmup is None else args.warmup
        run_reference(args)
    else:
        big = args.workload in ("long", "wide", "views3")
        args.steps = (100 if big else 1000) if args.steps is None else args.steps
        args.warmup = (10 if big else 100) if args.warmup is None else args.warmup
        run_ours(args)


if __name__ == "__main__":
    main()
