"""Several contexts at once — `-m gpu`.

`include/tc.h` promises "no global state; multiple contexts allowed" (`tc_create`).
Two things can break that promise without any single-context test noticing: state shared between
contexts (a static scratch buffer of the host builder, the device-side group counter, the spill
buffer) and work of one context overtaking work of another on a different stream.  Here two contexts
with DIFFERENT particle sets are driven (a) interleaved call by call on two CUDA streams with
device buffers and no synchronisation in between, and (b) from two host threads at the same time
(ctypes releases the GIL, so the two `tc_build`s and the two kernels really overlap).  Every result is
compared with the oracle (counts exactly, accelerations within the bar of `test_gpu_parity.py`) and
with the same context run alone.
"""
import threading

import numpy as np
import pytest

from oracle import Oracle
from paper_1005_5384_b200 import binding as B
from paper_1005_5384_b200 import build as tc_build
from paper_1005_5384_b200 import inputs

pytestmark = pytest.mark.gpu

ACC_Q999, ACC_MAX, POT_MAX = 1e-4, 1e-3, 1e-4


@pytest.fixture(scope="module", autouse=True)
def _built():
    tc_build.build()


# two workloads that differ in everything a shared buffer would mix up: size, tree depth, options
CASES = [
    dict(make=lambda: inputs.plummer(30011, 41), n_leaf=16, n_group=96, theta=0.5, eps=0.01, opts={}),
    dict(make=lambda: inputs.uniform_cube(17003, 42), n_leaf=8, n_group=32, theta=0.75, eps=0.02, opts={"device_build": 1}),
]


def oracle_ref(case, pos, mass):
    o = Oracle(pos, mass, case["n_leaf"], case["n_group"])
    return o.forces(case["theta"], case["eps"], shadow32=True)


def check(acc, pot, n_pc, n_pp, ref):
    assert np.array_equal(n_pc, ref["n_pc"]) and np.array_equal(n_pp, ref["n_pp"])
    rel = np.linalg.norm(acc.astype(np.float64) - ref["acc"], axis=1) / np.linalg.norm(ref["acc"], axis=1)
    assert np.isfinite(rel).all()
    assert np.quantile(rel, 0.999) <= ACC_Q999 and rel.max() <= ACC_MAX
    assert (np.abs(pot - ref["pot"]) / np.abs(ref["pot"])).max() <= POT_MAX


def solo(case, pos, mass):
    with B.TreeCode(n_group=case["n_group"]) as tc:
        for k, v in case["opts"].items():
            tc.set_option(k, v)
        tc.set_particles(pos, mass)
        tc.build(case["n_leaf"])
        acc, pot = tc.forces(case["theta"], case["eps"])
        n_pc, n_pp = tc.counts()
    return acc, pot, n_pc, n_pp


def test_two_contexts_interleaved_on_two_streams():
    import torch
    data = [c["make"]() for c in CASES]
    refs = [oracle_ref(c, *d) for c, d in zip(CASES, data)]
    alone = [solo(c, *d) for c, d in zip(CASES, data)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    tcs = [B.TreeCode(n_group=c["n_group"]) for c in CASES]
    try:
        bufs = []
        for tc, c, (pos, mass), st in zip(tcs, CASES, data, streams):
            for k, v in c["opts"].items():
                tc.set_option(k, v)
            tc.set_stream(st.cuda_stream)
            n = len(mass)
            with torch.cuda.stream(st):
                bufs.append(dict(pos=torch.from_numpy(pos).cuda(), mass=torch.from_numpy(mass).cuda(),
                                 acc=torch.full((n, 3), float("nan"), dtype=torch.float32, device="cuda"),
                                 pot=torch.full((n,), float("nan"), dtype=torch.float32, device="cuda")))
            st.synchronize()
        # call by call, alternating between the contexts; nothing waits for the other stream
        for rep in range(3):
            for tc, b in zip(tcs, bufs):
                tc.set_particles(b["pos"], b["mass"])
            for tc, c in zip(tcs, CASES):
                tc.build(c["n_leaf"])
            for tc, c, b in zip(tcs, CASES, bufs):
                B.tc_forces(tc.ctx, c["theta"], c["eps"], b["acc"], b["pot"])
        for tc in tcs:
            tc.sync()
        for tc, b, ref, al in zip(tcs, bufs, refs, alone):
            acc, pot = b["acc"].cpu().numpy(), b["pot"].cpu().numpy()
            n_pc, n_pp = tc.counts()
            check(acc, pot, n_pc, n_pp, ref)
            # a group is evaluated by one warp in a fixed order: the same context alone gives the same bits
            assert np.array_equal(acc, al[0]) and np.array_equal(pot, al[1])
            assert np.array_equal(n_pc, al[2]) and np.array_equal(n_pp, al[3])
    finally:
        for tc in tcs:
            tc.close()


def test_two_contexts_driven_from_two_host_threads():
    data = [c["make"]() for c in CASES]
    refs = [oracle_ref(c, *d) for c, d in zip(CASES, data)]
    alone = [solo(c, *d) for c, d in zip(CASES, data)]
    out, errors = [None, None], []
    start = threading.Barrier(2)

    def worker(i):
        try:
            c, (pos, mass) = CASES[i], data[i]
            with B.TreeCode(n_group=c["n_group"]) as tc:
                for k, v in c["opts"].items():
                    tc.set_option(k, v)
                start.wait()
                for rep in range(5):               # host buffers: set + build + forces, synchronous per call
                    tc.set_particles(pos, mass)
                    tc.build(c["n_leaf"])
                    acc, pot = tc.forces(c["theta"], c["eps"])
                    n_pc, n_pp = tc.counts()
                    if rep and not (np.array_equal(acc, out[i][0]) and np.array_equal(n_pc, out[i][2])):
                        raise AssertionError(f"context {i}: repetition {rep} differs from repetition 0")
                    out[i] = (acc, pot, n_pc, n_pp)
        except BaseException as e:                 # surfaced in the main thread below
            errors.append((i, e))
            start.abort()

    threads = [threading.Thread(target=worker, args=(i,)) for i in range(2)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=300)
    assert not any(t.is_alive() for t in threads), "a worker thread hangs"
    assert not errors, errors
    for o, ref, al in zip(out, refs, alone):
        check(*o, ref)
        assert np.array_equal(o[0], al[0]) and np.array_equal(o[1], al[1])
        assert np.array_equal(o[2], al[2]) and np.array_equal(o[3], al[3])
