"""Pins for the oracle's evaluation (O6) and its direct-summation reference.

Cited passages: body-node / body-leaf interaction Lists 3-4 PAPER.md:105-135; quadrupole moments
PAPER.md:49 (formula only cited -> textbook, R10); error metric PAPER.md:149; error ~ theta^4 PAPER.md:151.
"""
import numpy as np
import pytest

import oracle
from paper_1005_5384_b200 import inputs
from conftest import read_golden


# ---------------------------------------------------------------- direct summation
def test_direct_two_body_closed_form():
    """a = m d / (d^2 + eps^2)^(3/2) toward the other body; phi = -m/(d^2+eps^2)^(1/2)."""
    pos = np.array([[0, 0, 0], [3, 4, 0]], np.float32)       # d = 5
    m = np.array([2.0, 0.5], np.float32)
    eps = 0.5
    a, p = oracle.direct(pos, m, eps)
    s3 = (25 + 0.25) ** 1.5
    assert np.allclose(a[0], 0.5 * np.array([3, 4, 0]) / s3, rtol=1e-14)
    assert np.allclose(a[1], -2.0 * np.array([3, 4, 0]) / s3, rtol=1e-14)
    assert np.allclose(p, [-0.5 / 25.25 ** 0.5, -2.0 / 25.25 ** 0.5], rtol=1e-14)


def test_direct_equilateral_triangle():
    """Three equal masses on an equilateral triangle of side L: |a| = sqrt(3) m / L^2 toward the centre."""
    L, mm = 2.0, 1.0
    pos = np.array([[0, 0, 0], [L, 0, 0], [L / 2, L * np.sqrt(3) / 2, 0]], np.float64)
    a, p = oracle.direct(pos.astype(np.float32), np.full(3, mm, np.float32), 0.0)
    cen = pos.mean(0)
    for i in range(3):
        u = (cen - pos[i]) / np.linalg.norm(cen - pos[i])
        assert np.allclose(a[i], np.sqrt(3) * mm / L ** 2 * u, atol=1e-6)
        assert abs(p[i] + 2 * mm / L) < 1e-6


def test_direct_momentum_and_targets():
    pos, m = inputs.plummer(700, 5)
    a, p = oracle.direct(pos, m, 0.01)
    ma = m[:, None].astype(np.float64) * a
    assert np.linalg.norm(ma.sum(0)) < 1e-13 * np.linalg.norm(ma, axis=1).sum()
    t = np.array([3, 77, 650], np.int64)
    at, pt = oracle.direct(pos, m, 0.01, targets=t)
    assert np.array_equal(at, a[t]) and np.array_equal(pt, p[t])
    # potential energy symmetric: sum_i m_i phi_i = 2 W, W from pairs
    x = pos.astype(np.float64)
    d = np.sqrt(((x[:, None] - x[None]) ** 2).sum(-1) + 1e-4)
    m64 = m.astype(np.float64)
    W = -(np.triu(np.outer(m64, m64) / d, 1)).sum()
    assert abs((m64 * p).sum() - 2 * W) < 1e-12 * abs(W)


def test_direct_coincident_eps0():
    pos = np.array([[1, 1, 1], [1, 1, 1], [2, 1, 1]], np.float32)
    a, p = oracle.direct(pos, np.ones(3, np.float32), 0.0)
    assert np.isfinite(a).all() and np.allclose(a[0], [1, 0, 0]) and np.allclose(p[0], -1)


# ---------------------------------------------------------------- particle-cell closed form
def _two_mass_setup(field):
    G = read_golden("quadrupole_two_mass.txt")
    s, mm = G["s"], G["m"]
    pos = np.array([[-s, 0, 0], [s, 0, 0], field], np.float32)
    m = np.array([mm, mm, 1e-3], np.float32)
    O = oracle.Oracle(pos, m, 2)
    # the two masses share one leaf A, the field point sits alone in leaf B (checked, not assumed)
    c = O.cells()
    assert O.n_cells == 3
    A = int(np.nonzero(c["count"] == 2)[0][0])
    gB = [k for k, gc in enumerate(O.groups()) if c["count"][gc] == 1][0]
    cl, ll, *_ = O.walk(gB, 0.5)
    assert cl.tolist() == [A] and ll.size == 1
    return G, O


def test_quadrupole_on_axis_golden():
    G, O = _two_mass_setup([8, 0, 0])
    r = O.forces(0.5, 0.0)
    assert r["n_pc"][2] == 1 and r["n_pp"][2] == 0
    assert abs(r["acc"][2, 0] - G["onaxis_ax"]) < 1e-15 and abs(r["acc"][2, 1]) < 1e-18 and abs(r["acc"][2, 2]) < 1e-18
    assert abs(r["pot"][2] - G["onaxis_phi"]) < 1e-15
    # the residual against the exact two-body force is O((s/r)^4) relative (next even multipole)
    rel = abs(r["acc"][2, 0] - G["onaxis_ax_exact"]) / abs(G["onaxis_ax_exact"])
    assert 1e-8 < rel < 10 * (G["s"] / 8.0) ** 4
    assert abs(r["pot"][2] - G["onaxis_phi_exact"]) / 0.25 < 3 * (G["s"] / 8.0) ** 4


def test_quadrupole_off_axis_golden():
    """Exercises the Q r term and the off-diagonal geometry (field point (6, 8, 0))."""
    G, O = _two_mass_setup([6, 8, 0])
    r = O.forces(0.5, 0.0)
    assert abs(r["acc"][2, 0] - G["offaxis_ax"]) < 1e-14
    assert abs(r["acc"][2, 1] - G["offaxis_ay"]) < 1e-14
    assert abs(r["acc"][2, 2]) < 1e-18
    assert abs(r["pot"][2] - G["offaxis_phi"]) < 1e-14
    # and against the exact pair force: error O((s/r)^4)
    ex, _ = oracle.direct(O.pos, np.array([1, 1, 0], np.float32), 0.0, targets=np.array([2]))
    assert np.linalg.norm(r["acc"][2] - ex[0]) / np.linalg.norm(ex[0]) < 10 * (G["s"] / 10.0) ** 4


def test_quadrupole_residual_scales_as_fourth_power():
    """Halving s/R must cut the relative residual ~16x (monopole-only would give 4x, a wrong
    quadrupole coefficient would not converge at that order at all)."""
    res = []
    for R in (4.0, 8.0, 16.0):
        pos = np.array([[-0.125, 0.0625, 0], [0.125, -0.0625, 0], [R * 0.6, R * 0.8, 0]], np.float32)
        m = np.array([1, 1, 1e-3], np.float32)
        O = oracle.Oracle(pos, m, 2)
        assert O.n_cells == 3
        r = O.forces(1.0, 0.0)
        assert r["n_pc"][2] == 1
        ex, exp_ = oracle.direct(pos, np.array([1, 1, 0], np.float32), 0.0, targets=np.array([2]))
        res.append(np.linalg.norm(r["acc"][2] - ex[0]) / np.linalg.norm(ex[0]))
    assert 12 < res[0] / res[1] < 20 and 12 < res[1] / res[2] < 20


def test_softened_particle_cell_reduces_to_softened_monopole_for_point_cell():
    """R11: a single-particle cell (Q = 0) seen as a cell gives exactly -m r/(r^2+eps^2)^(3/2)."""
    pos = np.array([[0, 0, 0], [3, 4, 12]], np.float32)      # r = 13
    m = np.array([2.0, 1.0], np.float32)
    O = oracle.Oracle(pos, m, 1)
    eps = 0.75
    r = O.forces(0.5, eps)
    assert r["n_pc"].tolist() == [1, 1] and r["n_pp"].tolist() == [0, 0]
    a, p = oracle.direct(pos, m, eps)
    assert np.allclose(r["acc"], a, rtol=1e-14, atol=0) and np.allclose(r["pot"], p, rtol=1e-14)
    s2 = 169 + eps * eps
    assert np.allclose(r["acc"][1], -2.0 * np.array([3, 4, 12]) / s2 ** 1.5, rtol=1e-14)


# ---------------------------------------------------------------- softened quadrupole (R11)
def _two_mass_field(field, theta=2.0):
    """Two masses in one leaf A (the cell), the field point alone in leaf B; B's walk lists A un-opened."""
    G = read_golden("quadrupole_two_mass_softened.txt")
    d, mm = G["d"], G["m"]
    pos = np.array([[-d, 0, 0], [d, 0, 0], field], np.float32)
    m = np.array([mm, mm, 1e-3], np.float32)
    O = oracle.Oracle(pos, m, 2)
    c = O.cells()
    assert O.n_cells == 3
    A = int(np.nonzero(c["count"] == 2)[0][0])
    gB = [k for k, gc in enumerate(O.groups()) if c["count"][gc] == 1][0]
    cl, ll, *_ = O.walk(gB, theta)
    assert cl.tolist() == [A] and ll.size == 1
    return G, O


def test_softened_quadrupole_on_axis_golden():
    """R11 pin with Q != 0 and eps ~ |r|: sigma^2 = r^2 + eps^2 in the s^-5 AND s^-7 terms.  With r in place of sigma in
    either term the on-axis a_x would be -3.62 or -6.27 instead of -4.292608 (golden header)."""
    G, O = _two_mass_field([0.5, 0, 0])
    r = O.forces(2.0, G["A_eps"])
    assert r["n_pc"][2] == 1 and r["n_pp"][2] == 0
    assert abs(r["acc"][2, 0] - G["A_ax"]) < 1e-14 and abs(r["acc"][2, 1]) < 1e-18 and abs(r["acc"][2, 2]) < 1e-18
    assert abs(r["pot"][2] - G["A_phi"]) < 1e-14
    r = O.forces(2.0, G["C_eps"])
    assert abs(r["acc"][2, 0] - G["C_ax"]) < 1e-12 and abs(r["pot"][2] - G["C_phi"]) < 1e-12


def test_softened_quadrupole_off_axis_golden():
    """Off axis: exercises Q r with two components and the mixed geometry at eps > 0."""
    G, O = _two_mass_field([0.5, 0.25, 0])
    r = O.forces(2.0, G["B_eps"])
    assert r["n_pc"][2] == 1 and r["n_pp"][2] == 0
    assert abs(r["acc"][2, 0] - G["B_ax"]) < 1e-14 and abs(r["acc"][2, 1] - G["B_ay"]) < 1e-14
    assert abs(r["acc"][2, 2]) < 1e-18 and abs(r["pot"][2] - G["B_phi"]) < 1e-14


@pytest.mark.parametrize("eps", [0.0, 0.1, 0.5])
def test_particle_cell_acceleration_is_minus_gradient_of_its_potential(eps):
    """O6 is self-consistent at any softening: a = -grad(phi) of the SAME cell term (central differences of the oracle's
    potential over displaced field points).  A power of sigma wrong in a or in phi alone, or a wrong sign or
    coefficient on Q r or (r^T Q r) r, breaks this by far more than the 1e-6 of the difference quotient."""
    base = np.array([0.5, 0.25, 0.125])
    hstep = 2.0 ** -10                                   # fp32-exact displacements
    def phi_at(x):
        pos = np.array([[-0.125, 0.03125, 0], [0.125, -0.03125, 0.03125], x], np.float32)
        assert np.array_equal(pos[2].astype(np.float64), x)
        O = oracle.Oracle(pos, np.array([1.0, 0.5, 1e-3], np.float32), 2)
        r = O.forces(2.0, eps)
        assert r["n_pc"][2] == 1 and r["n_pp"][2] == 0
        return r["pot"][2], r["acc"][2]
    _, a0 = phi_at(base)
    grad = np.zeros(3)
    for k in range(3):
        e = np.zeros(3); e[k] = hstep
        grad[k] = (phi_at(base + e)[0] - phi_at(base - e)[0]) / (2 * hstep)
    assert np.linalg.norm(a0 + grad) / np.linalg.norm(a0) < 2e-5


# ---------------------------------------------------------------- whole evaluation
@pytest.mark.parametrize("n,n_leaf,n_group", [(1024, 16, 16), (4096, 16, 64), (777, 3, 3)])
def test_theta_zero_equals_direct_sum(n, n_leaf, n_group):
    pos, m = inputs.plummer(n, 1)
    O = oracle.Oracle(pos, m, n_leaf, n_group)
    r = O.forces(0.0, 0.01)
    a, p = oracle.direct(pos, m, 0.01)
    assert (r["n_pc"] == 0).all() and (r["n_pp"] == n - 1).all()
    assert np.abs(r["acc"] - a).max() <= 1e-12 * np.abs(a).max()
    assert np.abs(r["pot"] - p).max() <= 1e-12 * np.abs(p).max()


def test_convergence_with_theta_and_fourth_power_slope():
    """Error vs direct sum falls monotonically as theta -> 0, roughly as theta^4."""
    pos, m = inputs.plummer(8192, 3)
    O = oracle.Oracle(pos, m, 16)
    a, _ = oracle.direct(pos, m, 0.01)
    an = np.linalg.norm(a, axis=1)
    med, mx = [], []
    thetas = [1.0, 0.75, 0.5, 0.3, 0.1]
    for th in thetas:
        r = O.forces(th, 0.01)
        e = np.linalg.norm(r["acc"] - a, axis=1) / an
        med.append(np.median(e))
        mx.append(e.max())
    assert all(med[i] > med[i + 1] for i in range(4)) and all(mx[i] > mx[i + 1] for i in range(4))
    slope = np.log(med[1] / med[3]) / np.log(0.75 / 0.3)
    assert 2.5 < slope < 5.0
    assert med[2] < 5e-4 and mx[4] < 1e-4


def test_counts_definition():
    pos, m = inputs.plummer(2048, 6)
    O = oracle.Oracle(pos, m, 16, 32)
    c = O.cells()
    perm = O.perm()
    r = O.forces(0.5, 0.01)
    tot = 0
    for g in range(O.n_groups):
        cl, ll, *_ = O.walk(g, 0.5)
        gc = O.groups()[g]
        mem = perm[c["begin"][gc]: c["begin"][gc] + c["count"][gc]]
        assert (r["n_pc"][mem] == cl.size).all()
        assert (r["n_pp"][mem] == c["count"][ll].sum() - 1).all()
        tot += len(mem) * (cl.size + c["count"][ll].sum() - 1)
    assert tot == r["interactions"] == int((r["n_pc"] + r["n_pp"]).sum())


def test_momentum_residual_small():
    """Tree forces are not exactly antisymmetric; the residual sits well below the median error."""
    pos, m = inputs.plummer(4096, 7)
    O = oracle.Oracle(pos, m, 16)
    r = O.forces(0.5, 0.01)
    a, _ = oracle.direct(pos, m, 0.01)
    med = np.median(np.linalg.norm(r["acc"] - a, axis=1) / np.linalg.norm(a, axis=1))
    ma = m[:, None] * r["acc"]
    assert np.linalg.norm(ma.sum(0)) / np.linalg.norm(ma, axis=1).sum() < med


def test_plummer_analytic_field():
    """Radially binned mean radial acceleration and potential follow the Plummer model
    a_r = -M(<r)/r^2 with M(<r) = r^3/(1+r^2)^(3/2) (truncation only removes mass outside r = 10,
    which by Newton's shell theorem does not change a_r inside)."""
    n = 16384
    pos, m = inputs.plummer(n, 12)
    O = oracle.Oracle(pos, m, 16)
    r = O.forces(0.5, 0.01)
    x = pos.astype(np.float64)
    rad = np.linalg.norm(x, axis=1)
    ar = (r["acc"] * x).sum(1) / rad
    # total mass is 1 (all n particles inside r = 10), so the model's enclosed fraction is scaled by 1/X_max
    want = -(rad / (1 + rad ** 2) ** 1.5) / inputs.PLUMMER_X_MAX
    for lo, hi in [(0.3, 0.5), (0.5, 0.8), (0.8, 1.2), (1.2, 2.0), (2.0, 4.0)]:
        s = (rad >= lo) & (rad < hi)
        assert s.sum() > 500
        assert abs(ar[s].mean() / want[s].mean() - 1) < 0.05
    # potential at the centre-most particles.  Full model of mass M = 1/X_max: phi(0) = -M; the shells
    # removed outside R = 10 contributed -int_R^inf dM/r = phi_full(R) + M(<R)/R = -M/sqrt(101) + 1/10,
    # so the truncated model has phi(0) = -M (1 - 1/sqrt(101)) - 1/10.
    s = rad < 0.1
    phi0 = -(1 - 1 / np.sqrt(101.0)) / inputs.PLUMMER_X_MAX - 0.1
    assert abs(r["pot"][s].mean() / phi0 - 1) < 0.03


def test_subset_of_groups_and_order_independence():
    pos, m = inputs.plummer(3000, 2)
    O = oracle.Oracle(pos, m, 16, 64)
    full = O.forces(0.5, 0.01)
    sel = np.array([0, 5, O.n_groups - 1], np.int64)
    part = O.forces(0.5, 0.01, groups=sel)
    done = ~np.isnan(part["pot"])
    c = O.cells()
    assert done.sum() == c["count"][O.groups()[sel]].sum()
    assert np.array_equal(part["acc"][done], full["acc"][done])
    # a permutation of the input particles gives the same forces (tree is a function of positions)
    p = np.random.default_rng(0).permutation(3000)
    O2 = oracle.Oracle(pos[p], m[p], 16, 64)
    r2 = O2.forces(0.5, 0.01)
    assert np.allclose(r2["acc"], full["acc"][p], rtol=1e-11, atol=1e-13)
    assert np.array_equal(r2["n_pc"], full["n_pc"][p]) and np.array_equal(r2["n_pp"], full["n_pp"][p])
