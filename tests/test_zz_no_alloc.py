"""delta_coherence_static (include/delta.h): the coherence stage with its scratch in the library's static device array,
for callers that cannot allocate.  Checked against the existing path (delta_coherence, scratch in the plan's workspace) within
the coherence tolerance of the parity tests, on calls in a row that share the array.

Collected last on purpose (the suite runs with pytest -x); it passes alone in a fresh process and after the others.
"""
import numpy as np
import pytest
import torch

TOL_G = 1e-4   # north_star's bound for the coherence, as in tests/test_parity_gpu.py


def binding():
    from paper_2108_08896_b200 import binding as b
    return b


def spectra(b, C, T, L, H, M, seed):
    """A plan and the S, Sauto of one seeded chunk: a common component + white noise, so coherences spread over (0, 1)."""
    rng = np.random.default_rng(seed)
    common = rng.standard_normal(T)
    x = (rng.uniform(0.1, 1.5, (C, 1)) * common + rng.standard_normal((C, T))).astype(np.float32)
    plan = b.Plan(C, T, L, H, M)
    X = plan.stft(torch.from_numpy(x).cuda())
    S, Sa = plan.cross_spectra(X)
    torch.cuda.synchronize()
    return plan, S, Sa


def check(plan, S, Sa, label):
    ref = plan.coherence(S, Sa)
    G = torch.full_like(ref, float("nan"))
    plan.coherence_static(S, Sa, G)
    torch.cuda.synchronize()
    assert torch.isfinite(G).all(), label
    err = torch.max(torch.abs(G - ref)).item()
    assert err <= TOL_G, f"{label}: |G_static - G| = {err:.3g}"
    assert 0.05 < ref.mean().item() < 0.95 and ref.max().item() <= 1.0 + TOL_G   # a non-trivial case
    return err


@pytest.mark.gpu
def test_static_scratch_matches_the_workspace_path_on_calls_in_a_row():
    b = binding()
    # three plans of different shapes share the array: a larger one first, so that the smaller ones find its leftovers
    cases = [(96, 6000, 512, 256, 256, 11), (40, 3000, 256, 128, 128, 12), (24, 9000, 2048, 1024, 1024, 13)]
    made = [spectra(b, *c) for c in cases]
    for rep in range(2):
        for (plan, S, Sa), c in zip(made, cases):
            check(plan, S, Sa, f"rep {rep} {c[:3]}")
    # two calls in a row on one plan with different inputs
    plan, S, Sa = made[0]
    plan2, S2, Sa2 = spectra(b, *cases[0][:5], seed=99)
    check(plan, S, Sa, "first input")
    check(plan, S2, Sa2, "second input, same plan")


@pytest.mark.gpu
def test_static_call_allocates_no_device_memory():
    b = binding()
    plan, S, Sa = spectra(b, 64, 4000, 512, 256, 256, 5)
    G = torch.empty((plan.sizes.P, plan.sizes.F), dtype=torch.float32, device="cuda")
    plan.coherence_static(S, Sa, G)   # first use: module loading, symbol address
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        plan.coherence_static(S, Sa, G)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0


def test_plans_beyond_the_static_scratch_are_refused():
    """Host logic only (the size check comes before anything touches the device): runs without a GPU too."""
    b = binding()
    C, L = 576, 4096   # 4 C ceil4(F) floats = 18.9 MB > DELTA_STATIC_SCRATCH_BYTES
    assert 4 * C * ((L // 2 + 1 + 3) // 4 * 4) * 4 > b.STATIC_SCRATCH_BYTES
    plan = b.Plan(C, L, L, L, 0, allocate=False)
    fake = 4096   # never dereferenced: the call is refused first
    status = b.LIB.delta_coherence_static(plan._h, fake, fake, fake, None)
    assert status == b.ERR_TOO_LARGE
    assert b"DELTA_STATIC_SCRATCH_BYTES" in b.LIB.delta_strerror(status)
    # a plan that fits is not refused for its size (without a workspace it stops at the next check)
    small = b.Plan(192, 10000, 512, 256, 256, allocate=False)
    assert b.LIB.delta_coherence_static(small._h, fake, fake, fake, None) == b.ERR_NO_WORKSPACE
    assert b.LIB.delta_coherence_static(small._h, None, fake, fake, None) == b.ERR_INVALID_ARG
