"""Pins of the oracle's VARIANT readings (R21: opening test against the cell's centre of mass;
R22: monopole-only cells) — `-m "not gpu"`.  The default readings are pinned in test_oracle_{tree,walk,eval}.py.

R21  brute force: the lists re-derived here from the recursive definition with plain numpy on the cell
     table; coverage invariant; theta = 0 is the direct sum; every cell inside a group still opens in the
     fp32 shadow (R14 under R20); fewer interactions and a larger, still converging, error than R1.
R22  closed form: two equal masses seen as ONE cell give exactly the point-mass field -2m/R^2 (the
     quadrupole of tests/golden/quadrupole_two_mass.txt switched off); error larger than with quadrupoles
     and ~theta^3 instead of ~theta^4.
"""
import numpy as np
import pytest

import oracle
from paper_1005_5384_b200 import inputs
from conftest import read_golden


def _lists_from_definition(c, gcell, theta, rule):
    """Recursive definition of the walk on the cell table `c` (fp64), independent of the oracle's loop."""
    cell_list, leaf_list = [], []
    gb, gh = c["b"][gcell], c["h"][gcell]

    def opened(ch):
        if rule == 0:
            d = np.maximum(0.0, np.abs(c["b"][ch] - gb) - c["h"][ch] - gh)
        else:
            d = np.maximum(0.0, np.abs(c["X"][ch] - gb) - gh)
        return (d * d).sum() * theta * theta <= (2.0 * c["h"][ch]) ** 2

    def visit(node):
        for ch in c["child"][node]:
            if ch < 0:
                continue
            if opened(ch):
                if c["n_child"][ch]:
                    visit(ch)
                else:
                    leaf_list.append(ch)
            else:
                cell_list.append(ch)

    if c["n_child"][0] == 0:
        return [], [0]
    visit(0)
    return cell_list, leaf_list


@pytest.mark.parametrize("rule", [0, 1])
@pytest.mark.parametrize("theta", [0.3, 0.7])
def test_walk_lists_against_recursive_definition(rule, theta):
    pos, mass = inputs.plummer(700, 41)
    o = oracle.Oracle(pos, mass, 4, 16, open_rule=rule)
    c = o.cells()
    groups = o.groups()
    for g in range(0, o.n_groups, 5):
        cl, ll, *_ = o.walk(g, theta)
        wc, wl = _lists_from_definition(c, groups[g], theta, rule)
        assert sorted(cl.tolist()) == sorted(wc) and sorted(ll.tolist()) == sorted(wl)
        assert c["count"][cl].sum() + c["count"][ll].sum() == o.n      # coverage: every particle exactly once


def test_com_rule_theta0_is_direct_sum_and_converges():
    pos, mass = inputs.plummer(1500, 42)
    dacc, dpot = oracle.direct(pos, mass, 0.01)
    o1 = oracle.Oracle(pos, mass, 8, 32, open_rule=1)
    r = o1.forces(0.0, 0.01)
    assert (r["n_pc"] == 0).all() and (r["n_pp"] == 1499).all()
    assert np.abs(r["acc"] - dacc).max() <= 1e-12 * np.abs(dacc).max()
    o0 = oracle.Oracle(pos, mass, 8, 32)
    err = lambda a: np.median(np.linalg.norm(a - dacc, axis=1) / np.linalg.norm(dacc, axis=1))
    prev = None
    for theta in (1.0, 0.7, 0.5, 0.3):
        r1, r0 = o1.forces(theta, 0.01), o0.forces(theta, 0.01)
        assert r1["interactions"] < r0["interactions"]                 # the COM rule opens fewer cells ...
        assert err(r1["acc"]) > err(r0["acc"])                         # ... and pays with a larger error
        if prev is not None:
            assert err(r1["acc"]) < prev                               # which still falls with theta
        prev = err(r1["acc"])


@pytest.mark.parametrize("n_leaf,n_group", [(4, 64), (1, 8)])
def test_com_rule_own_cells_open_in_fp32(n_leaf, n_group):
    """R14 under the COM rule: the centre of mass of a cell inside the group lies in the group's tight box,
    hence (R20) in its fp32 cube: d = 0 in the fp32 shadow too."""
    pos, mass = inputs.plummer(3000, 12)
    o = oracle.Oracle(pos, mass, n_leaf, n_group, open_rule=1)
    c = o.cells()
    groups = o.groups()
    for g in range(0, o.n_groups, 3):
        gb, ge = c["begin"][groups[g]], c["begin"][groups[g]] + c["count"][groups[g]]
        cl, ll, *_ = o.walk(g, 0.6, shadow32=True)
        assert not ((c["begin"][cl] < ge) & (c["begin"][cl] + c["count"][cl] > gb)).any()
        assert c["count"][cl].sum() + c["count"][ll].sum() == o.n


def test_monopole_only_closed_form_and_error_order():
    G = read_golden("quadrupole_two_mass.txt")
    s, mm = G["s"], G["m"]
    pos = np.array([[-s, 0, 0], [s, 0, 0], [8, 0, 0]], np.float32)
    m = np.array([mm, mm, 1e-3], np.float32)
    o = oracle.Oracle(pos, m, 2, quadrupole=False)
    r = o.forces(0.5, 0.0)
    assert r["n_pc"][2] == 1 and r["n_pp"][2] == 0
    assert abs(r["acc"][2, 0] - (-2.0 * mm / 64.0)) < 1e-16 and abs(r["pot"][2] - (-2.0 * mm / 8.0)) < 1e-16
    # the quadrupole term of the golden file is exactly what is missing
    assert abs((G["onaxis_ax"] - r["acc"][2, 0]) - (-6.0 * mm * s * s / 8.0 ** 4)) < 1e-15
    # on a real distribution: larger error than with quadrupoles, and a lower order in theta
    pos, mass = inputs.plummer(4000, 43)
    dacc, _ = oracle.direct(pos, mass, 0.01)
    om, oq = oracle.Oracle(pos, mass, 8, 32, quadrupole=False), oracle.Oracle(pos, mass, 8, 32)
    err = lambda a: np.median(np.linalg.norm(a - dacc, axis=1) / np.linalg.norm(dacc, axis=1))
    e_m = [err(om.forces(t, 0.01)["acc"]) for t in (0.8, 0.4)]
    e_q = [err(oq.forces(t, 0.01)["acc"]) for t in (0.8, 0.4)]
    assert e_m[0] > e_q[0] and e_m[1] > e_q[1]
    assert np.log2(e_m[0] / e_m[1]) < np.log2(e_q[0] / e_q[1])         # monopole: lower order in theta
    assert 1.5 < np.log2(e_m[0] / e_m[1]) and np.log2(e_q[0] / e_q[1]) < 5.0
