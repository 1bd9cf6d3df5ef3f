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


# ---- R23: the group enters the opening test as its tight box (per-axis half extents) ---------------------

def _lists_group_box(c, gcell, theta, rule):
    """Recursive definition under R23, with the distance written as the gap between INTERVALS
    ([bmin, bmax] of the group against the cell's cube, or against the cell's COM) — not the oracle's
    |db| - h - e form."""
    cell_list, leaf_list = [], []
    glo, ghi = c["bmin"][gcell], c["bmax"][gcell]

    def opened(ch):
        if rule == 0:
            clo, chi = c["b"][ch] - c["h"][ch], c["b"][ch] + c["h"][ch]
        else:
            clo = chi = c["X"][ch]
        gap = np.maximum(0.0, np.maximum(clo - ghi, glo - chi))
        return (gap * gap).sum() * theta * theta <= (2.0 * c["h"][ch]) ** 2

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


def test_group_box_threshold_golden():
    G = read_golden("group_box_threshold.txt")
    pos = np.array([[G["f"]] * 3, [G["gx0"], G["gy"], G["z"]], [G["gx1"], G["gy"], G["z"]],
                    [G["cx0"], G["cy"], G["z"]], [G["cx1"], G["cy"], G["z"]]], np.float32)
    m = np.full(5, 0.2, np.float32)
    assert abs(G["theta_star_cube"] - 0.5 / G["d_cube"]) < 1e-12 and abs(G["theta_star_box"] - 0.5 / G["d_box"]) < 1e-12
    for gbox, tstar in ((False, G["theta_star_cube"]), (True, G["theta_star_box"])):
        O = oracle.Oracle(pos, m, 2, group_box=gbox)
        c = O.cells()
        grp = O.groups().tolist()
        # the tree holds the two pairs as leaves with the boxes the golden file states
        gi = [g for g in grp if c["count"][g] == 2 and np.allclose(c["b"][g], [2.5, 1, 1])]
        ci = [g for g in grp if c["count"][g] == 2 and np.allclose(c["b"][g], [2.5, 6, 1])]
        assert len(gi) == 1 and len(ci) == 1
        g_cell, c_cell = gi[0], ci[0]
        assert c["h"][g_cell] == 1.0 and c["h"][c_cell] == 0.25
        assert np.allclose(c["bmax"][g_cell] - c["bmin"][g_cell], [2, 0, 0])
        gidx = grp.index(g_cell)
        for shadow in (False, True):
            cl, ll, *_ = O.walk(gidx, tstar * 0.999, shadow)
            assert c_cell in ll.tolist() and c_cell not in cl.tolist()         # opened: particle-particle
            cl, ll, *_ = O.walk(gidx, tstar * 1.001, shadow)
            assert c_cell in cl.tolist() and c_cell not in ll.tolist()         # not opened: multipole
    # between the two thresholds the two readings disagree
    th = 0.12
    Oc, Ob = oracle.Oracle(pos, m, 2), oracle.Oracle(pos, m, 2, group_box=True)
    gidx = Oc.groups().tolist().index(g_cell)
    assert c_cell in Oc.walk(gidx, th)[1].tolist() and c_cell in Ob.walk(gidx, th)[0].tolist()


@pytest.mark.parametrize("rule", [0, 1])
@pytest.mark.parametrize("theta", [0.3, 0.7])
def test_group_box_lists_against_recursive_definition(rule, theta):
    pos, mass = inputs.plummer(700, 43)
    o = oracle.Oracle(pos, mass, 4, 16, open_rule=rule, group_box=True)
    c = o.cells()
    groups = o.groups()
    for g in range(0, o.n_groups, 5):
        cl, ll, *_ = o.walk(g, theta)
        wc, wl = _lists_group_box(c, groups[g], theta, rule)
        assert sorted(cl.tolist()) == sorted(wc) and sorted(ll.tolist()) == sorted(wl)
        assert c["count"][cl].sum() + c["count"][ll].sum() == o.n      # coverage: every particle exactly once


def test_group_box_theta0_fewer_interactions_same_error_order():
    pos, mass = inputs.plummer(1500, 44)
    dacc, dpot = oracle.direct(pos, mass, 0.01)
    ob = oracle.Oracle(pos, mass, 8, 32, group_box=True)
    r = ob.forces(0.0, 0.01)
    assert (r["n_pc"] == 0).all() and (r["n_pp"] == 1499).all()
    assert np.abs(r["acc"] - dacc).max() <= 1e-12 * np.abs(dacc).max()
    oc = oracle.Oracle(pos, mass, 8, 32)
    err = lambda a: np.median(np.linalg.norm(a - dacc, axis=1) / np.linalg.norm(dacc, axis=1))
    prev = None
    for theta in (1.0, 0.7, 0.5, 0.3):
        rb, rc = ob.forces(theta, 0.01, stats=True), oc.forces(theta, 0.01, stats=True)
        # the tight box lies inside the cube: distances can only grow, so no test that fails to open under
        # the cube rule opens under R23: fewer opening tests, fewer particle-particle terms, fewer interactions
        assert (rb["tests"] <= rc["tests"]).all() and rb["n_pp"].sum() <= rc["n_pp"].sum()
        assert rb["interactions"] < rc["interactions"]
        # every particle of the group is still at least d away from the cell: same error order
        assert err(rb["acc"]) < 1.5 * err(rc["acc"])
        if prev is not None:
            assert err(rb["acc"]) < prev
        prev = err(rb["acc"])


@pytest.mark.parametrize("n_leaf,n_group,rule", [(4, 64, 0), (1, 8, 0), (1, 8, 1)])
def test_group_box_own_cells_open_in_fp32(n_leaf, n_group, rule):
    """R14 under R23: a cell inside the group has its fp32 centre (and its COM) inside the group's tight
    box, whose fp32 half extents are rounded up from the rounded centre: d = 0 in the fp32 shadow too."""
    pos, mass = inputs.plummer(3000, 13)
    o = oracle.Oracle(pos, mass, n_leaf, n_group, open_rule=rule, group_box=True)
    c = o.cells()
    e32, (b32, h32) = o.ext32(), o.bnd32()
    # containment of the tight box in the fp32 box, and of the fp32 box in the fp32 cube
    assert (b32.astype(np.float64) + e32 >= c["bmax"]).all() and (b32.astype(np.float64) - e32 <= c["bmin"]).all()
    assert (e32.max(axis=1) == h32).all()
    groups = o.groups()
    for g in range(0, o.n_groups, 3):
        gb, ge = c["begin"][groups[g]], c["begin"][groups[g]] + c["count"][groups[g]]
        cl, ll, *_ = o.walk(g, 0.6, shadow32=True)
        assert not ((c["begin"][cl] < ge) & (c["begin"][cl] + c["count"][cl] > gb)).any()
        assert c["count"][cl].sum() + c["count"][ll].sum() == o.n
