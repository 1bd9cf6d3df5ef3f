"""The paper-literal two-pass pipeline (option "two_pass") — `-m gpu`.

count kernel -> scan -> write kernel (lists in global memory) -> body-node kernel -> body-leaf kernel must
give the same lists as the fused kernel: identical counts, forces equal up to summation order, and the
usual parity with the oracle."""
import numpy as np
import pytest

from oracle import Oracle
from paper_1005_5384_b200 import binding as B
from paper_1005_5384_b200 import build as tc_build
from paper_1005_5384_b200 import inputs
from test_gpu_parity import check, rel_err

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    tc_build.build()


def _run(pos, mass, theta, eps, n_leaf, n_group, two_pass, opts=None):
    with B.TreeCode(n_group=n_group) as tc:
        tc.set_option("two_pass", two_pass)
        for k, v in (opts or {}).items():
            tc.set_option(k, v)
        tc.set_particles(pos, mass)
        tc.build(n_leaf)
        acc, pot = tc.forces(theta, eps)
        n_pc, n_pp = tc.counts()
        return acc, pot, n_pc, n_pp, tc.stats()


@pytest.mark.parametrize("name,n_leaf,n_group,eps", [("plummer_1k", 16, 64, None), ("plummer_64k", 16, 96, None),
                                                       ("cube_64k", 8, 32, None), ("plummer_64k", 4, 256, 0.0)])
def test_two_pass_equals_fused_and_oracle(name, n_leaf, n_group, eps):
    pos, mass, theta, eps0, _ = inputs.make(name)
    eps = eps0 if eps is None else eps
    f = _run(pos, mass, theta, eps, n_leaf, n_group, 0)
    t = _run(pos, mass, theta, eps, n_leaf, n_group, 1)
    assert np.array_equal(f[2], t[2]) and np.array_equal(f[3], t[3])
    for k in ("n_pc_total", "n_pp_total"):
        assert f[4][k] == t[4][k], k
    assert rel_err(t[0].astype(np.float64), f[0].astype(np.float64)).max() <= 5e-5
    assert t[4]["list_bytes"] > 0 and t[4]["t_node_ms"] > 0 and f[4]["list_bytes"] == 0
    o = Oracle(pos, mass, n_leaf, n_group)
    ref = o.forces(theta, eps, shadow32=True, stats=True)
    check(t[0], t[1], t[2], t[3], ref)
    # opening tests EXECUTED: the count pass walks every group once; the fused kernel walks a group once per
    # 128 of its particles (include/tc.h, tc_stats.n_tests_total), i.e. once for every N_group <= 128
    m = o.cells()["count"][o.groups()]
    assert t[4]["n_tests_total"] == int(ref["tests"].sum())
    assert f[4]["n_tests_total"] == int((ref["tests"] * ((m + 127) // 128)).sum())


def test_two_pass_degenerate_and_spill():
    # root is a leaf; coincident particles (level-21 leaf > 64 bodies); spilling walk stack
    pos = np.array([[0, 0, 0], [3, 4, 0]], np.float32); mass = np.array([2.0, 5.0], np.float32)
    t = _run(pos, mass, 0.5, 0.1, 16, 64, 1)
    f = _run(pos, mass, 0.5, 0.1, 16, 64, 0)
    assert np.allclose(t[0], f[0], rtol=1e-6) and np.allclose(t[1], f[1], rtol=1e-6) and (t[3] == 1).all()
    pos, mass = inputs.plummer(2048, 11)
    pos[:200] = pos[0]
    t = _run(pos, mass, 0.5, 0.01, 16, 64, 1)
    check(t[0], t[1], t[2], t[3], Oracle(pos, mass, 16, 64).forces(0.5, 0.01, shadow32=True))
    pos, mass = inputs.plummer(32768, 14)
    t = _run(pos, mass, 0.2, 0.01, 2, 16, 1, {"stack_smem": 64})
    f = _run(pos, mass, 0.2, 0.01, 2, 16, 0)
    assert t[4]["n_spills"] > 0
    assert np.array_equal(f[2], t[2]) and np.array_equal(f[3], t[3])
    assert rel_err(t[0].astype(np.float64), f[0].astype(np.float64)).max() <= 5e-5


def test_two_pass_timing_breakdown_1m():
    """The paper's per-kernel metrics at config 3, beside the fused kernel."""
    pos, mass, theta, eps, n_leaf = inputs.make("plummer_1m")
    n = len(mass)
    with B.TreeCode() as tc:
        tc.set_particles(pos, mass)
        tc.build(n_leaf)
        acc_f, pot_f = tc.forces(theta, eps)
        tc.forces(theta, eps)
        sf = tc.stats()
        cf = tc.counts()
        tc.set_option("two_pass", 1)
        acc_t, pot_t = tc.forces(theta, eps)
        tc.forces(theta, eps)
        st = tc.stats()
        ct = tc.counts()
    assert np.array_equal(cf[0], ct[0]) and np.array_equal(cf[1], ct[1])
    assert rel_err(acc_t.astype(np.float64), acc_f.astype(np.float64)).max() <= 5e-5
    tests, npc, npp = st["n_tests_total"], st["n_pc_total"], st["n_pp_total"]
    print(f"fused: {sf['t_gpu_ms']:.3f} ms | two-pass total {st['t_gpu_ms']:.3f} ms = count+scan {st['t_walk_count_ms']:.3f} "
          f"+ write {st['t_walk_write_ms']:.3f} + node {st['t_node_ms']:.3f} + leaf {st['t_leaf_ms']:.3f}; "
          f"lists {st['list_bytes'] / 1e6:.0f} MB")
    print(f"paper metrics: walk-count {64 * tests / st['t_walk_count_ms'] / 1e6:.0f} GB/s, walk-write "
          f"{64 * tests / st['t_walk_write_ms'] / 1e6:.0f} GB/s, node kernel {70 * npc / st['t_node_ms'] / 1e9:.1f} TFLOP/s "
          f"(paper's 70 flops), leaf kernel {38 * npp / st['t_leaf_ms'] / 1e9:.1f} TFLOP/s (paper's 38 flops)")
    assert st["t_gpu_ms"] > sf["t_gpu_ms"]          # fusing wins: no list traffic, one walk instead of two
