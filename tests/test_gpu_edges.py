"""Edge and degenerate cases of the CUDA path against the oracle — `-m gpu`.

Empty / tiny inputs, a root that is a leaf, coincident particles (level-21
leaves larger than N_leaf, R7), eps = 0 and eps whose square is subnormal, theta
extremes, N_group > 128 (a group is walked once per 128 of its particles),
N_group = 1, the global-memory spill path of the walk stack, unequal masses,
call-order errors.
"""
import numpy as np
import pytest

from oracle import Oracle, direct
from paper_1005_5384_b200 import binding as B
from paper_1005_5384_b200 import build as tc_build
from paper_1005_5384_b200 import inputs
from test_gpu_parity import check, gpu_forces, rel_err

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    tc_build.build()


def test_single_particle():
    pos = np.array([[0.25, -1.0, 3.0]], np.float32)
    mass = np.array([2.0], np.float32)
    acc, pot, n_pc, n_pp, st = gpu_forces(pos, mass, 0.5, 0.01, 16, 64)
    assert (acc == 0).all() and n_pc[0] == 0 and n_pp[0] == 0
    assert abs(pot[0]) <= 1e-6 * 2.0 / 0.01          # the self term -m/eps is added and removed in fp32
    assert st["n_cells"] == 1 and st["n_groups"] == 1


@pytest.mark.parametrize("eps", [0.0, 0.1])
def test_two_particles_closed_form(eps):
    """N = 2: a = m d / (d^2 + eps^2)^(3/2) (root is a leaf, never tested)."""
    pos = np.array([[0, 0, 0], [3, 4, 0]], np.float32)
    mass = np.array([2.0, 5.0], np.float32)
    acc, pot, _, n_pp, _ = gpu_forces(pos, mass, 0.5, eps, 16, 64)
    s3 = (25.0 + eps * eps) ** 1.5
    assert np.allclose(acc[0], 5.0 * np.array([3, 4, 0]) / s3, rtol=2e-6)
    assert np.allclose(acc[1], -2.0 * np.array([3, 4, 0]) / s3, rtol=2e-6)
    assert np.allclose(pot, [-5.0 / np.sqrt(25 + eps * eps), -2.0 / np.sqrt(25 + eps * eps)], rtol=1e-5)
    assert (n_pp == 1).all()


@pytest.mark.parametrize("eps", [0.0, 0.01])
def test_coincident_particles_level21_leaf(eps):
    """200 particles at one point + a Plummer cloud: the point is a level-21 leaf with count > N_leaf
    and > 64 (R7); with eps = 0 coincident pairs contribute nothing (O6)."""
    pos, mass = inputs.plummer(2048, 11)
    pos[:200] = pos[0]
    acc, pot, n_pc, n_pp, st = gpu_forces(pos, mass, 0.5, eps, 16, 64)
    o = Oracle(pos, mass, 16, 64)
    assert st["depth"] == 21 == o.depth
    ref = o.forces(0.5, eps, shadow32=True)
    check(acc, pot, n_pc, n_pp, ref)


@pytest.mark.parametrize("n_leaf,n_group", [(1, 1), (4, 256), (16, 1000), (64, 64), (2048, 2048)])
def test_leaf_and_group_sizes(n_leaf, n_group):
    pos, mass = inputs.plummer(3000, 12)
    acc, pot, n_pc, n_pp, st = gpu_forces(pos, mass, 0.6, 0.02, n_leaf, n_group)
    o = Oracle(pos, mass, n_leaf, n_group)
    assert st["n_groups"] == o.n_groups
    check(acc, pot, n_pc, n_pp, o.forces(0.6, 0.02, shadow32=True))


@pytest.mark.parametrize("theta", [0.0, 0.05, 2.0, 1e3])
def test_theta_extremes(theta):
    pos, mass = inputs.uniform_cube(4096, 13)
    acc, pot, n_pc, n_pp, _ = gpu_forces(pos, mass, theta, 0.01, 8, 32)
    ref = Oracle(pos, mass, 8, 32).forces(theta, 0.01, shadow32=True)
    assert np.array_equal(n_pc, ref["n_pc"]) and np.array_equal(n_pp, ref["n_pp"])
    if theta <= 2.0:       # beyond that the method itself is meaningless; counts still agree
        check(acc, pot, n_pc, n_pp, ref)


@pytest.mark.parametrize("cfg", [0, 1, 2])
def test_spill_path_matches_and_is_exercised(cfg):
    """stack_smem = 64 forces the walk stack through its global-memory spill: same result — in the automatic choice and in
    each build of the fused kernel forced (kernel_config 1 = sparse, 2 = dense: both compile the spill path)."""
    pos, mass = inputs.plummer(32768, 14)
    a0, p0, c0, d0, s0 = gpu_forces(pos, mass, 0.2, 0.01, 2, 16, opts={"kernel_config": cfg})
    a1, p1, c1, d1, s1 = gpu_forces(pos, mass, 0.2, 0.01, 2, 16, opts={"stack_smem": 64, "kernel_config": cfg})
    assert s1["n_spills"] > 1000 and s0["n_spills"] <= 16      # (theta = 0.2, N_leaf = 2: a handful of spills even with 256 entries)
    assert np.array_equal(c0, c1) and np.array_equal(d0, d1)
    assert s0["n_tests_total"] == s1["n_tests_total"]
    # traversal order changes => summation order changes; both are within fp32 rounding of each other
    assert rel_err(a1.astype(np.float64), a0.astype(np.float64)).max() <= 2e-5
    gsel = np.arange(0, 2000, 50, dtype=np.int64)
    ref = Oracle(pos, mass, 2, 16).forces(0.2, 0.01, shadow32=True, groups=gsel)
    check(a1, p1, c1, d1, ref, ref["n_pc"] >= 0)


def test_unequal_masses_and_massless():
    rng = np.random.default_rng(15)
    pos, _ = inputs.plummer(5000, 15)
    mass = rng.uniform(0.0, 2.0, 5000).astype(np.float32)
    mass[::7] = 0.0
    acc, pot, n_pc, n_pp, _ = gpu_forces(pos, mass, 0.5, 0.01, 16, 64)
    check(acc, pot, n_pc, n_pp, Oracle(pos, mass, 16, 64).forces(0.5, 0.01, shadow32=True))


def test_eps0_against_direct():
    pos, mass = inputs.plummer(2000, 16)
    acc, pot, _, _, _ = gpu_forces(pos, mass, 0.0, 0.0, 16, 64)
    dacc, dpot = direct(pos, mass, 0.0)
    assert rel_err(acc.astype(np.float64), dacc).max() <= 2e-5
    assert (np.abs(pot - dpot) / np.abs(dpot)).max() <= 1e-5


def test_repeat_calls_and_rebuild_are_deterministic_in_counts():
    pos, mass = inputs.plummer(20000, 17)
    with B.TreeCode(n_group=64) as tc:
        tc.set_particles(pos, mass)
        tc.build(16)
        a0, p0 = tc.forces(0.5, 0.01)
        c0 = tc.counts()
        a1, p1 = tc.forces(0.5, 0.01)
        c1 = tc.counts()
        assert np.array_equal(c0[0], c1[0]) and np.array_equal(c0[1], c1[1])
        assert rel_err(a1.astype(np.float64), a0.astype(np.float64)).max() <= 2e-5
        # new particles invalidate the tree
        tc.set_particles(pos[:100], mass[:100])
        with pytest.raises(B.TcError) as e:
            tc.forces(0.5, 0.01)
        assert e.value.code == B.TC_ESTATE
        tc.build(16)
        a2, _ = tc.forces(0.5, 0.01)
        assert a2.shape == (100, 3) and np.isfinite(a2).all()


def test_argument_errors_on_device_context():
    pos, mass = inputs.plummer(64, 18)
    with B.TreeCode() as tc:
        with pytest.raises(B.TcError) as e:
            tc.build(16)
        assert e.value.code == B.TC_ESTATE
        tc.set_particles(pos, mass)
        tc.build(16)
        acc = np.zeros((64, 3), np.float32)
        for theta, eps in [(-1.0, 0.01), (0.5, -0.01), (float("nan"), 0.01), (0.5, float("inf"))]:
            with pytest.raises(B.TcError) as e:
                B.tc_forces(tc.ctx, theta, eps, acc, None)
            assert e.value.code == B.TC_EINVAL
        B.tc_forces(tc.ctx, 0.5, 0.01, acc, None)       # pot = NULL is allowed
        assert np.isfinite(acc).all() and np.abs(acc).max() > 0


def test_tiny_eps_is_eps_zero_and_huge_theta_is_refused():
    """eps in (4e-23, 1.1e-19) has a non-zero SUBNORMAL square that rsqrt.approx.ftz flushes to 0 (inf for
    the self pair and coincident pairs, then NaN), and below ~1e-13 m / eps^3 of those pairs overflows (inf * 0);
    theta > 1.8e19 squares to inf (0 * inf = NaN in the test of a group's own ancestors).  The library takes
    eps < 1e-10 as 0 and refuses such a theta."""
    pos, mass = inputs.plummer(2048, 21)
    pos[:40] = pos[0]                                            # coincident particles too
    o = Oracle(pos, mass, 16, 64)
    ref0 = o.forces(0.5, 0.0, shadow32=True)
    for eps in (9e-11, 2e-19, 1e-20, 3e-22, 1e-30):
        acc, pot, n_pc, n_pp, _ = gpu_forces(pos, mass, 0.5, eps, 16, 64)
        assert np.isfinite(acc).all() and np.isfinite(pot).all()
        check(acc, pot, n_pc, n_pp, ref0)
        dacc, dpot = gpu_direct(pos, mass, eps)
        assert np.isfinite(dacc).all() and np.isfinite(dpot).all()
    # the smallest eps that runs the eps > 0 kernel stays finite (the potential then carries the documented 6e-8 m/eps)
    acc, pot, n_pc, n_pp, _ = gpu_forces(pos, mass, 0.5, 1e-10, 16, 64)
    assert np.isfinite(acc).all() and np.isfinite(pot).all()
    assert rel_err(acc.astype(np.float64), ref0["acc"]).max() < 1e-3
    with B.TreeCode(n_group=64) as tc:
        tc.set_particles(pos, mass)
        tc.build(16)
        for theta in (1e20, 2e18, float("inf")):
            with pytest.raises(B.TcError) as e:
                tc.forces(theta, 0.01)
            assert e.value.code == B.TC_EINVAL
        # a theta that large but legal opens nothing beyond what touches the group: finite, counts as the oracle's
        acc, pot = tc.forces(1e18, 0.01)
        n_pc, n_pp = tc.counts()
    check(acc, pot, n_pc, n_pp, o.forces(1e18, 0.01, shadow32=True))


def gpu_direct(pos, mass, eps):
    with B.TreeCode() as tc:
        tc.set_particles(pos, mass)
        return tc.direct(eps, targets=np.arange(0, len(mass), 7, dtype=np.int64))


def test_binding_checks_dtype_and_shape_before_the_c_call():
    """a float64 array would be reinterpreted byte by byte by the C library."""
    pos, mass, theta, eps, n_leaf = inputs.make("plummer_1k")
    with B.TreeCode() as tc:
        with pytest.raises(TypeError):
            tc.set_particles(pos.astype(np.float64), mass)
        with pytest.raises(TypeError):
            tc.set_particles(pos, mass.astype(np.float64))
        with pytest.raises(TypeError):
            tc.set_particles(np.ascontiguousarray(pos.T), mass)
        with pytest.raises(TypeError):
            tc.set_particles(pos, mass[:-1])
        tc.set_particles(pos, mass)
        tc.build(n_leaf)
        with pytest.raises(TypeError):
            B.tc_forces(tc.ctx, theta, eps, np.empty((len(mass), 3), np.float64))
        with pytest.raises(TypeError):
            B.tc_forces(tc.ctx, theta, eps, np.empty((len(mass), 3), np.float32), np.empty(len(mass) + 1, np.float32))
        with pytest.raises(TypeError):
            B.tc_direct(tc.ctx, eps, None, np.empty((len(mass), 3), np.float32))


@pytest.mark.parametrize("cfg", [1, 2])
def test_both_launch_configurations_match_the_oracle(cfg):
    """The fused kernel exists in two builds (sparse / dense, option kernel_config): each is forced
    here on small AND large groups, coincident particles (a level-21 leaf above the pass size), eps = 0, a variant
    reading, the stack-spill-sized walk and a sharded evaluation — same lists, same tolerances."""
    import torch
    pos, mass = inputs.plummer(12000, 41)
    pos[:150] = pos[0]
    for n_leaf, n_group, theta, eps, extra in [(16, 128, 0.5, 0.01, {}), (4, 8, 0.4, 0.0, {}), (16, 96, 0.6, 0.01, {"open_rule": 1, "group_box": 1}),
                                               (8, 256, 0.3, 0.01, {"quadrupole": 0})]:
        opts = dict(extra, kernel_config=cfg)
        acc, pot, n_pc, n_pp, st = gpu_forces(pos, mass, theta, eps, n_leaf, n_group, opts=opts)
        o = Oracle(pos, mass, n_leaf, n_group, open_rule=extra.get("open_rule", 0), quadrupole=bool(extra.get("quadrupole", 1)),
                   group_box=bool(extra.get("group_box", 0)))
        check(acc, pot, n_pc, n_pp, o.forces(theta, eps, shadow32=True))
    # the two builds agree with each other to summation-order rounding, and a sharded evaluation in a forced build
    # is bit for bit the unsharded one of the same build
    n = len(mass)
    with B.TreeCode(n_group=128) as tc:
        tc.set_option("kernel_config", cfg)
        tc.set_particles(pos, mass)
        tc.build(16)
        a0, p0 = tc.forces(0.5, 0.01)
        tc.set_option("shard_count", 3)
        ns = tc.shard_size()
        g = torch.zeros((3, ns, 4), dtype=torch.float32, device="cuda")
        for r in range(3):
            tc.set_option("shard_rank", r)
            tc.forces_shard(0.5, 0.01, g[r])
        acc = torch.empty((n, 3), dtype=torch.float32, device="cuda"); pot = torch.empty(n, dtype=torch.float32, device="cuda")
        tc.shard_scatter(g, None, acc, pot)
        tc.sync()
        assert np.array_equal(acc.cpu().numpy(), a0) and np.array_equal(pot.cpu().numpy(), p0)
        tc.set_option("shard_count", 1); tc.set_option("shard_rank", 0)
        tc.set_option("kernel_config", 3 - cfg)
        a1, _ = tc.forces(0.5, 0.01)
        assert rel_err(a1.astype(np.float64), a0.astype(np.float64)).max() <= 5e-5
        with pytest.raises(B.TcError):
            tc.set_option("kernel_config", 3)


@pytest.mark.parametrize("two_pass", [0, 1])
def test_self_pair_is_excluded_not_cancelled_at_large_m_over_eps(two_pass):
    """O6 sums over j != i.  With m / eps = 1e4 and |phi| ~ 1, a self term -m/eps that is added to the fp32 potential sum and
    taken out again leaves ~6e-8 * 1e4 = 6e-4 of relative error (the library did that until round 3: this test failed);
    excluded by index, the potential is accurate to fp32 rounding.  Tree path (fused and two-pass) and tc_direct."""
    pos = np.array([[0.0, 0.0, 0.0], [1.0, 0.25, 0.0], [-0.5, 0.75, 0.5], [0.25, -1.0, 0.75], [0.5, 0.5, -1.25]], np.float32)
    mass = np.array([1.0, 0.5, 2.0, 1.5, 0.75], np.float32)
    eps = 1e-4
    for n_leaf, n_group in ((1, 1), (2, 8), (16, 128)):
        acc, pot, n_pc, n_pp, _ = gpu_forces(pos, mass, 0.5, eps, n_leaf, n_group, opts={"two_pass": two_pass})
        ref = Oracle(pos, mass, n_leaf, n_group).forces(0.5, eps, shadow32=True)
        assert np.array_equal(n_pc, ref["n_pc"]) and np.array_equal(n_pp, ref["n_pp"])
        assert (np.abs(pot - ref["pot"]) / np.abs(ref["pot"])).max() <= 2e-6
        assert rel_err(acc.astype(np.float64), ref["acc"]).max() <= 1e-5
    if not two_pass:
        with B.TreeCode() as tc:
            tc.set_particles(pos, mass)
            dacc, dpot = tc.direct(eps)
            tg = np.array([3, 0, 3], np.int64)             # targets out of order, one twice
            tacc, tpot = tc.direct(eps, tg)
        racc, rpot = direct(pos, mass, eps)
        assert (np.abs(dpot - rpot) / np.abs(rpot)).max() <= 1e-6 and rel_err(dacc, racc).max() <= 2e-6
        assert np.array_equal(tpot, dpot[tg]) and np.array_equal(tacc, dacc[tg])
