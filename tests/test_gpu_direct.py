"""tc_direct (GPU direct summation) against the oracle's fp64 direct sum — `-m gpu`.

Tolerance: relative error <= 2e-6 on accelerations and <= 1e-6 on potentials (fp32 interactions with a
Newton-refined rsqrt, fp64 accumulation: per-term error ~1e-7, no growth with N)."""
import numpy as np
import pytest

from oracle import direct
from paper_1005_5384_b200 import binding as B
from paper_1005_5384_b200 import build as tc_build
from paper_1005_5384_b200 import inputs
from test_gpu_parity import rel_err

pytestmark = pytest.mark.gpu
ACC_TOL, POT_TOL = 2e-6, 1e-6


@pytest.fixture(scope="module", autouse=True)
def _built():
    tc_build.build()


def _check(acc, pot, racc, rpot):
    assert rel_err(acc, racc).max() <= ACC_TOL
    assert (np.abs(pot - rpot) / np.abs(rpot)).max() <= POT_TOL


@pytest.mark.parametrize("eps", [0.01, 0.0])
def test_direct_all_particles_config1(eps):
    pos, mass, *_ = inputs.make("plummer_1k")
    with B.TreeCode() as tc:
        tc.set_particles(pos, mass)
        acc, pot = tc.direct(eps)                 # no tree needed
    _check(acc, pot, *direct(pos, mass, eps))


def test_direct_sampled_targets_64k_and_ragged_sizes():
    pos, mass, *_ = inputs.make("plummer_64k")
    pos, mass = pos[:65536 - 37], mass[:65536 - 37]          # ragged source tail
    tg = inputs.sample_targets(len(mass), 1000 + 3, seed=7)  # ragged target tile
    with B.TreeCode() as tc:
        tc.set_particles(pos, mass)
        acc, pot = tc.direct(0.01, tg)
        _check(acc, pot, *direct(pos, mass, 0.01, targets=tg))
        # one target, and the same target twice
        one = np.array([5, 5], np.int64)
        a1, p1 = tc.direct(0.01, one)
        r = direct(pos, mass, 0.01, targets=one)
        _check(a1, p1, *r)
        assert np.array_equal(a1[0], a1[1])


def test_direct_coincident_and_unequal_masses():
    rng = np.random.default_rng(21)
    pos, _ = inputs.plummer(3000, 21)
    pos[10:20] = pos[10]
    mass = rng.uniform(0.0, 2.0, 3000).astype(np.float32)
    with B.TreeCode() as tc:
        tc.set_particles(pos, mass)
        for eps in (0.0, 0.05):
            acc, pot = tc.direct(eps)
            racc, rpot = direct(pos, mass, eps)
            # coincident partners at eps = 0 make |a| of those particles small sums of large terms: absolute check
            assert np.abs(acc - racc).max() <= ACC_TOL * np.linalg.norm(racc, axis=1).max()
            assert (np.abs(pot - rpot) / np.abs(rpot)).max() <= POT_TOL


def test_direct_device_pointers_and_errors():
    import torch
    pos, mass, *_ = inputs.make("plummer_1k")
    with B.TreeCode() as tc:
        with pytest.raises(B.TcError) as e:
            tc.direct(0.01)
        assert e.value.code == B.TC_ESTATE
        tc.set_particles(pos, mass)
        tc.use_torch_stream()
        d_acc = torch.empty((1024, 3), dtype=torch.float64, device="cuda")
        d_pot = torch.empty(1024, dtype=torch.float64, device="cuda")
        B.tc_direct(tc.ctx, 0.01, None, d_acc, d_pot)
        tc.sync()
        _check(d_acc.cpu().numpy(), d_pot.cpu().numpy(), *direct(pos, mass, 0.01))
        with pytest.raises(B.TcError) as e:
            tc.direct(0.01, np.array([0, 1024], np.int64))
        assert e.value.code == B.TC_EINVAL
        with pytest.raises(B.TcError) as e:
            tc.direct(-1.0)
        assert e.value.code == B.TC_EINVAL


def test_tree_error_against_gpu_direct_matches_oracle_direct_1m():
    """Config-4 style use: the tree's error measured against tc_direct equals the one measured against the
    oracle's direct sum (4096 targets, N = 2^20) — and times the direct kernel."""
    pos, mass, theta, eps, n_leaf = inputs.make("plummer_1m")
    tg = inputs.sample_targets(len(mass), 4096, seed=4)
    with B.TreeCode() as tc:
        tc.set_particles(pos, mass)
        gacc, gpot = tc.direct(eps, tg)
        t_direct = tc.stats()["t_gpu_ms"]
        tc.build(n_leaf)
        acc, _ = tc.forces(theta, eps)
    racc, rpot = direct(pos, mass, eps, targets=tg)
    _check(gacc, gpot, racc, rpot)
    e_g, e_o = rel_err(acc[tg].astype(np.float64), gacc), rel_err(acc[tg].astype(np.float64), racc)
    assert abs(np.median(e_g) / np.median(e_o) - 1) < 0.01
    print(f"tc_direct: 4096 x 2^20 interactions in {t_direct:.3f} ms = {4096 * (1 << 20) / (t_direct * 1e-3) / 1e9:.0f} G interactions/s; "
          f"tree median error vs GPU direct {np.median(e_g):.3e}, vs oracle direct {np.median(e_o):.3e}")
