"""Pins of the oracle's kick-drift-kick leapfrog (oracle.leapfrog_kdk; BASELINE.json config 5) — `-m "not gpu"`.

The integrator is pinned with force laws written out HERE in plain numpy (not the oracle's), so that a wrong
factor (dt instead of dt/2, a drift before the kick, a stale acceleration) fails one of:
  * two-body circular orbit: closed-form radius / period, error falling as dt^2 (second order);
  * exact time reversibility of KDK (forward K steps, flip the velocities, K steps: back at the start);
  * momentum conservation with pairwise antisymmetric forces; energy error bounded and ~dt^2;
  * with the tree force on a Plummer sphere: energy conserved at the level of the tree error.
"""
import numpy as np

import oracle
from paper_1005_5384_b200 import inputs


def _direct64(mass, eps):
    m = np.asarray(mass, np.float64)

    def f(x):
        d = x[None, :, :] - x[:, None, :]                # d[i, j] = x_j - x_i
        s2 = (d * d).sum(-1) + eps * eps
        np.fill_diagonal(s2, np.inf)
        ri = 1.0 / np.sqrt(s2)
        acc = (m[None, :, None] * d * (ri ** 3)[:, :, None]).sum(1)
        pot = -(m[None, :] * ri).sum(1)
        return acc, pot
    return f


def _two_body():
    # equal masses 1/2 a distance 1 apart on a circle of radius 1/2: a = m/d^2 = 1/2 = v^2/r  ->  v = 1/2, period 2 pi
    pos = np.array([[-0.5, 0, 0], [0.5, 0, 0]], np.float64)
    vel = np.array([[0, -0.5, 0], [0, 0.5, 0]], np.float64)
    return pos, vel, np.array([0.5, 0.5])


def test_two_body_circular_orbit_second_order():
    pos, vel, m = _two_body()
    f = _direct64(m, 0.0)
    errs = []
    for steps in (200, 400, 800):
        x, v, a, p = oracle.leapfrog_kdk(pos, vel, 2 * np.pi / steps, steps, f)
        r = np.linalg.norm(x, axis=1)
        assert np.abs(r - 0.5).max() < 1e-3                       # stays on the circle
        errs.append(np.abs(x - pos).max())                         # one period later: back at the start
        assert np.allclose(p, -0.5, atol=1e-3)                     # phi_i = -m_j / d
    assert errs[0] < 2e-3
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.5 < errs[1] / errs[2] < 4.5   # second order in dt


def test_quarter_period_closed_form():
    pos, vel, m = _two_body()
    x, v, *_ = oracle.leapfrog_kdk(pos, vel, (np.pi / 2) / 1000, 1000, _direct64(m, 0.0))
    assert np.allclose(x, [[0, -0.5, 0], [0, 0.5, 0]], atol=2e-6)  # counter-clockwise quarter turn
    assert np.allclose(v, [[0.5, 0, 0], [-0.5, 0, 0]], atol=2e-6)


def test_time_reversible_and_momentum():
    rng = np.random.default_rng(7)
    pos, vel, m = rng.normal(size=(12, 3)), 0.3 * rng.normal(size=(12, 3)), rng.uniform(0.5, 1.5, 12) / 12
    f = _direct64(m, 0.05)
    x1, v1, a1, _ = oracle.leapfrog_kdk(pos, vel, 0.01, 50, f)
    assert np.abs(x1 - pos).max() > 1e-2
    x2, v2, *_ = oracle.leapfrog_kdk(x1, -v1, 0.01, 50, f)
    assert np.abs(x2 - pos).max() < 1e-12 and np.abs(v2 + vel).max() < 1e-12
    p0, p1 = (m[:, None] * vel).sum(0), (m[:, None] * v1).sum(0)
    assert np.abs(p1 - p0).max() < 1e-15
    # acc0: handing in the accelerations of the start gives the same trajectory
    a0, _ = f(pos)
    x3, v3, *_ = oracle.leapfrog_kdk(pos, vel, 0.01, 50, f, acc0=a0)
    assert np.array_equal(x3, x1) and np.array_equal(v3, v1)


def test_energy_error_is_second_order():
    rng = np.random.default_rng(8)
    pos, vel, m = rng.normal(size=(10, 3)), 0.2 * rng.normal(size=(10, 3)), np.full(10, 0.1)
    f = _direct64(m, 0.1)

    def energy(x, v):
        return 0.5 * (m * (v * v).sum(1)).sum() + 0.5 * (m * f(x)[1]).sum()
    e0 = energy(pos, vel)
    de = []
    for steps in (40, 80, 160):
        x, v, *_ = oracle.leapfrog_kdk(pos, vel, 1.0 / steps, steps, f)
        de.append(abs(energy(x, v) - e0))
    assert de[0] < 1e-3 * abs(e0)
    assert 3.0 < de[0] / de[1] < 5.0 and 3.0 < de[1] / de[2] < 5.0


def test_tree_force_leapfrog_conserves_energy_on_a_plummer_sphere():
    n = 512
    pos, mass = inputs.plummer(n, 21)
    vel = inputs.plummer_velocities64(pos.astype(np.float64), 22, 1.0, 1.0)
    f = oracle.tree_force(mass, 0.4, 0.05, n_leaf=8, n_group=16)
    a0, p0 = f(pos.astype(np.float64))
    m = mass.astype(np.float64)
    e0 = 0.5 * (m * (vel * vel).sum(1)).sum() + 0.5 * (m * p0).sum()
    x, v, a, p = oracle.leapfrog_kdk(pos, vel, 1.0 / 128, 10, f)
    e1 = 0.5 * (m * (v * v).sum(1)).sum() + 0.5 * (m * p).sum()
    assert abs((e1 - e0) / e0) < 2e-4
    # against the exact force law on the same start: the trajectories agree at the tree-error level
    xd, vd, *_ = oracle.leapfrog_kdk(pos, vel, 1.0 / 128, 10, _direct64(m, 0.05))
    assert np.abs(x - xd).max() < 1e-5 and np.abs(v - vd).max() < 2e-4
