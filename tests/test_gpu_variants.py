"""Variant readings on the GPU (options "open_rule", "quadrupole"; R21, R22) against the oracle
run with the same variant — `-m gpu`.  Same bars as the default path: counts exact against the fp32
shadow, accelerations 1e-4 (99.9 %) / 1e-3 (max), potentials 1e-4."""
import numpy as np
import pytest

from oracle import Oracle, direct
from paper_1005_5384_b200 import binding as B
from paper_1005_5384_b200 import build as tc_build
from paper_1005_5384_b200 import inputs
from test_gpu_parity import check, rel_err

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    tc_build.build()


def _run(pos, mass, theta, eps, n_leaf, n_group, open_rule, quadrupole, two_pass=0, group_box=0, device_build=0):
    with B.TreeCode(n_group=n_group) as tc:
        tc.set_option("group_box", group_box)
        tc.set_option("device_build", device_build)
        tc.set_option("open_rule", open_rule)
        tc.set_option("quadrupole", quadrupole)
        tc.set_option("two_pass", two_pass)
        tc.set_particles(pos, mass)
        tc.build(n_leaf)
        acc, pot = tc.forces(theta, eps)
        n_pc, n_pp = tc.counts()
        return acc, pot, n_pc, n_pp, tc.stats()


@pytest.mark.parametrize("open_rule,quadrupole", [(1, 1), (0, 0), (1, 0)])
@pytest.mark.parametrize("name,n_leaf,n_group", [("plummer_1k", 16, 64), ("plummer_64k", 16, 96), ("cube_64k", 8, 32)])
def test_variants_match_the_oracle_variant(open_rule, quadrupole, name, n_leaf, n_group):
    pos, mass, theta, eps, _ = inputs.make(name)
    acc, pot, n_pc, n_pp, st = _run(pos, mass, theta, eps, n_leaf, n_group, open_rule, quadrupole)
    o = Oracle(pos, mass, n_leaf, n_group, open_rule=open_rule, quadrupole=bool(quadrupole))
    ref = o.forces(theta, eps, shadow32=True, stats=True)
    check(acc, pot, n_pc, n_pp, ref)
    assert st["n_tests_total"] == int(ref["tests"].sum())


@pytest.mark.parametrize("open_rule,device_build,two_pass", [(0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1)])
@pytest.mark.parametrize("name,n_leaf,n_group", [("plummer_1k", 16, 64), ("plummer_64k", 16, 96), ("cube_64k", 4, 32)])
def test_group_box_matches_the_oracle_variant(open_rule, device_build, two_pass, name, n_leaf, n_group):
    """R23 (option "group_box"): the group enters the opening test as its tight box — host and device builds,
    with the COM rule, in the two-pass pipeline; counts exact against the oracle's fp32 shadow of R23."""
    pos, mass, theta, eps, _ = inputs.make(name)
    acc, pot, n_pc, n_pp, st = _run(pos, mass, theta, eps, n_leaf, n_group, open_rule, 1, two_pass=two_pass,
                                    group_box=1, device_build=device_build)
    o = Oracle(pos, mass, n_leaf, n_group, open_rule=open_rule, group_box=True)
    ref = o.forces(theta, eps, shadow32=True, stats=True)
    check(acc, pot, n_pc, n_pp, ref)
    assert st["n_tests_total"] == int(ref["tests"].sum())
    base = Oracle(pos, mass, n_leaf, n_group, open_rule=open_rule).forces(theta, eps, shadow32=True)
    assert ref["interactions"] < base["interactions"]


def test_group_box_device_build_boxes_identical():
    pos, mass, *_ = inputs.make("plummer_64k")
    out = []
    for dev in (0, 1):
        with B.TreeCode(n_group=96) as tc:
            tc.set_option("device_build", dev)
            tc.set_particles(pos, mass)
            tc.build(16)
            out.append(B.tc_get_group_boxes(tc.ctx))
    assert np.array_equal(out[0], out[1])


def test_variants_in_the_two_pass_pipeline_and_eps0():
    pos, mass, theta, _, n_leaf = inputs.make("plummer_64k")
    for eps in (0.01, 0.0):
        a, p, c, d, _ = _run(pos, mass, theta, eps, n_leaf, 64, 1, 0, two_pass=1)
        check(a, p, c, d, Oracle(pos, mass, n_leaf, 64, open_rule=1, quadrupole=False).forces(theta, eps, shadow32=True))


def test_com_rule_trades_accuracy_for_interactions_1m():
    """about 45 % fewer interactions and about twice the error at equal theta (config 3)."""
    pos, mass, theta, eps, n_leaf = inputs.make("plummer_1m")
    tg = inputs.sample_targets(len(mass), 2048, seed=4)
    with B.TreeCode() as tc:
        tc.set_particles(pos, mass)
        dacc, _ = tc.direct(eps, tg)
        tc.build(n_leaf)
        out = {}
        for rule in (0, 1):
            tc.set_option("open_rule", rule)
            acc, _ = tc.forces(theta, eps)
            tc.forces(theta, eps)
            s = tc.stats()
            out[rule] = (s["t_gpu_ms"], s["n_pc_total"] + s["n_pp_total"], np.median(rel_err(acc[tg].astype(np.float64), dacc)))
    print("open_rule 0: %.3f ms, %.3e interactions, median error %.2e | open_rule 1: %.3f ms, %.3e interactions, median error %.2e"
          % (out[0] + out[1]))
    assert out[1][1] < 0.75 * out[0][1] and out[1][0] < out[0][0]
    assert out[0][2] < out[1][2] < 6 * out[0][2]


def test_group_box_1m_sampled_groups():
    """R23 at config 3 (full size, the launch configuration of bench.py): counts exact and forces within the bars on
    sampled groups; fewer interactions than the cube rule."""
    pos, mass, theta, eps, n_leaf = inputs.make("plummer_1m")
    with B.TreeCode() as tc:                                   # default N_group
        tc.set_particles(pos, mass)
        tc.build(n_leaf)
        n_group = tc.stats()["n_group"]
        tc.forces(theta, eps)
        base = tc.stats()
        tc.set_option("group_box", 1)
        acc, pot = tc.forces(theta, eps)
        tc.forces(theta, eps)
        n_pc, n_pp = tc.counts()
        st = tc.stats()
    o = Oracle(pos, mass, n_leaf, n_group, group_box=True)
    gsel = np.sort(np.random.default_rng(23).choice(o.n_groups, 192, replace=False)).astype(np.int64)
    ref = o.forces(theta, eps, shadow32=True, groups=gsel)
    check(acc, pot, n_pc, n_pp, ref, ref["n_pc"] >= 0)
    tot, tot0 = st["n_pc_total"] + st["n_pp_total"], base["n_pc_total"] + base["n_pp_total"]
    print("group_box at config 3: %.3f ms, %.4e interactions (cube rule: %.3f ms, %.4e)" % (st["t_gpu_ms"], tot, base["t_gpu_ms"], tot0))
    assert tot < tot0 and st["n_tests_total"] < base["n_tests_total"]
