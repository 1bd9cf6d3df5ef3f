"""tc_direct_static — the direct sum for callers that cannot allocate device memory — against tc_direct.  `-m gpu`.

Who needs it: a library loaded into an application whose own pool has taken the whole GPU and only lends out fixed
buffers; a latency-critical step that must not touch the driver's allocator (cudaMalloc takes a global lock, cudaFree
synchronises the device); a process whose 180 GB are already full.  tc_direct serves everyone else: it creates a
context and cudaMallocs the packed source array.  tc_direct_static keeps that array in a 4 MiB block compiled into the
library (one per GPU, shared by all callers, limit TC_DIRECT_STATIC_MAX_N = 262 144 particles) and allocates nothing.

What is checked: two calls in a row (the second with FEWER particles, so the block still holds the first call's
sources beyond the new n — they must not leak into the result) equal the existing path's results within the tolerance
of tests/test_gpu_direct.py (same kernels: the only difference is the order of fp64 atomics); the device's free memory
is the same before and after a repeated call; sizes beyond the limit and host pointers are refused with a clear message.

This file is named to be collected LAST: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It passes alone in a fresh process (it then performs the per-device set-up itself) and after the others."""
import numpy as np
import pytest

from paper_1005_5384_b200 import binding as B
from paper_1005_5384_b200 import build as tc_build
from paper_1005_5384_b200 import inputs

pytestmark = pytest.mark.gpu
ACC_TOL, POT_TOL = 2e-6, 1e-6          # the bars of tests/test_gpu_direct.py


@pytest.fixture(scope="module", autouse=True)
def _built():
    tc_build.build()


def _existing_path(pos, mass, eps, targets):
    with B.TreeCode() as tc:
        tc.set_particles(pos, mass)
        return tc.direct(eps, targets)


def _rel(a, b):
    return np.linalg.norm(a - b, axis=-1) / np.linalg.norm(b, axis=-1)


def test_static_direct_equals_existing_path_on_two_calls_in_a_row():
    import torch
    eps = 0.01
    pos_a, mass_a = inputs.plummer(5000 + 13, 31)                 # several source tiles and a ragged tail
    pos_b, mass_b = inputs.plummer(3000 - 7, 32)                  # second call: fewer particles, other positions
    mass_b = (mass_b * np.random.default_rng(5).uniform(0.5, 2.0, len(mass_b))).astype(np.float32)
    tg_b = inputs.sample_targets(len(mass_b), 700 + 3, seed=9)
    d = lambda x: torch.from_numpy(np.ascontiguousarray(x)).cuda()
    # every device buffer exists before the calls: the entry point is given memory, it never obtains any
    dpa, dma, dpb, dmb, dtb = d(pos_a), d(mass_a), d(pos_b), d(mass_b), d(tg_b)
    acc_a = torch.full((len(mass_a), 3), float("nan"), dtype=torch.float64, device="cuda")
    pot_a = torch.full((len(mass_a),), float("nan"), dtype=torch.float64, device="cuda")
    acc_b = torch.full((len(tg_b), 3), float("nan"), dtype=torch.float64, device="cuda")
    pot_b = torch.full((len(tg_b),), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()

    # call 1: all particles, legacy default stream (also the per-device set-up when this file runs alone)
    B.tc_direct_static(dpa, dma, eps, None, acc_a, pot_a, 0)
    # call 2, right behind it on the same stream: targets, fewer sources than the block still holds from call 1
    B.tc_direct_static(dpb, dmb, eps, dtb, acc_b, pot_b, 0)
    torch.cuda.synchronize()

    ra, rpa = _existing_path(pos_a, mass_a, eps, None)
    rb, rpb = _existing_path(pos_b, mass_b, eps, tg_b)
    for got, gpot, ref, rpot, what in ((acc_a, pot_a, ra, rpa, "call 1"), (acc_b, pot_b, rb, rpb, "call 2")):
        got, gpot = got.cpu().numpy(), gpot.cpu().numpy()
        ea, ep = _rel(got, ref).max(), (np.abs(gpot - rpot) / np.abs(rpot)).max()
        print(f"tc_direct_static {what}: max rel diff to tc_direct acc {ea:.2e}, pot {ep:.2e}")
        assert np.isfinite(got).all() and np.isfinite(gpot).all(), what
        assert ea <= ACC_TOL and ep <= POT_TOL, what

    # the same call again on a stream of the caller: identical results, and the GPU's free memory does not move
    s = torch.cuda.Stream()
    acc_c, pot_c = torch.empty_like(acc_b), torch.empty_like(pot_b)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    with torch.cuda.stream(s):
        B.tc_direct_static(dpb, dmb, eps, dtb, acc_c, pot_c, s.cuda_stream)
    s.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    assert free1 == free0, f"device memory changed across the call: {free0} -> {free1}"
    assert _rel(acc_c.cpu().numpy(), rb).max() <= ACC_TOL
    assert (np.abs(pot_c.cpu().numpy() - rpb) / np.abs(rpb)).max() <= POT_TOL

    # pot = NULL is allowed
    acc_d = torch.empty_like(acc_b)
    B.tc_direct_static(dpb, dmb, eps, dtb, acc_d, None, 0)
    torch.cuda.synchronize()
    assert _rel(acc_d.cpu().numpy(), rb).max() <= ACC_TOL


def test_static_direct_refuses_what_it_cannot_hold():
    import torch
    lim = B.TC_DIRECT_STATIC_MAX_N
    pos = torch.zeros((lim + 1, 3), dtype=torch.float32, device="cuda")
    mass = torch.ones(lim + 1, dtype=torch.float32, device="cuda")
    acc = torch.zeros((4, 3), dtype=torch.float64, device="cuda")
    tg = torch.arange(4, dtype=torch.int64, device="cuda")
    with pytest.raises(B.TcError) as e:                            # one particle too many
        B.tc_direct_static(pos, mass, 0.01, tg, acc)
    assert e.value.code == B.TC_EINVAL and str(lim) in str(e.value) and "TC_DIRECT_STATIC_MAX_N" in str(e.value)
    B.tc_direct_static(pos[:lim], mass[:lim], 0.01, tg, acc)       # exactly the limit is fine
    torch.cuda.synchronize()
    assert torch.isfinite(acc).all()
    with pytest.raises(B.TcError) as e:                            # host memory: there is nowhere to stage it
        B.tc_direct_static(np.zeros((8, 3), np.float32), np.ones(8, np.float32), 0.01, None, np.zeros((8, 3)))
    assert e.value.code == B.TC_EINVAL and "DEVICE" in str(e.value)
    with pytest.raises(B.TcError) as e:
        B.tc_direct_static(pos[:8], mass[:8], -1.0, None, torch.zeros((8, 3), dtype=torch.float64, device="cuda"))
    assert e.value.code == B.TC_EINVAL
