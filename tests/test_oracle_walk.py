"""Pins for the oracle's walk (O5): List 2 PAPER.md:73-91, prose PAPER.md:93, boundary cube Fig. 1 PAPER.md:39.

* a hand-computed opening threshold (tests/golden/opening_threshold.txt): direction of the
  inequality, that l is the CELL's side, that both half sides enter d;
* the coverage invariant: every particle is seen exactly once by every group;
* theta = 0 opens everything; huge theta opens only touching cells;
* brute force: lists derived from the recursive definition over all (group, cell) pairs
  with the box distance computed min-over-corner-pairs style (interval gap), not the
  oracle's |db| - h - h form;
* the fp32 shadow (R16) only flips tests whose fp64 margin is at rounding level.
"""
import numpy as np
import pytest

import oracle
from paper_1005_5384_b200 import inputs
from conftest import read_golden


def test_opening_threshold_golden():
    G = read_golden("opening_threshold.txt")
    pos = np.array([[G["xa0"], 0, 0], [G["xa1"], 0, 0], [G["xb0"], 0, 0], [G["xb1"], 0, 0]], np.float32)
    m = np.full(4, 0.25, np.float32)
    O = oracle.Oracle(pos, m, 2)
    c = O.cells()
    assert O.n_cells == 3 and O.n_groups == 2
    grp = O.groups()
    A, B = grp[0], grp[1]
    assert np.allclose(c["b"][A], [0, 0, 0]) and c["h"][A] == 0.25
    assert np.allclose(c["b"][B], [8, 0, 0]) and c["h"][B] == 0.5
    tA, tB = G["theta_star_A"], G["theta_star_B"]
    assert abs(tA - 0.5 / G["d"]) < 1e-12 and abs(tB - 1.0 / G["d"]) < 1e-12
    for shadow in (False, True):
        # group B (index 1) testing cell A: opened (-> leaf list, A is a leaf) iff theta <= tA
        cl, ll, *_ = O.walk(1, tA * 0.999, shadow)
        assert sorted(ll.tolist()) == [A, B] and cl.size == 0
        cl, ll, *_ = O.walk(1, tA * 1.001, shadow)
        assert cl.tolist() == [A] and ll.tolist() == [B]
        # group A testing cell B: threshold is tB (the CELL's side is what counts)
        cl, ll, *_ = O.walk(0, tB * 0.999, shadow)
        assert sorted(ll.tolist()) == [A, B] and cl.size == 0
        cl, ll, *_ = O.walk(0, tB * 1.001, shadow)
        assert cl.tolist() == [B] and ll.tolist() == [A]
        # between the thresholds the two groups disagree
        th = 0.1
        assert O.walk(1, th, shadow)[0].tolist() == [A] and O.walk(0, th, shadow)[0].size == 0


def test_root_leaf_case():
    """O5: if the root is a leaf the leaf list is {root}."""
    pos, m = inputs.plummer(10, 3)
    O = oracle.Oracle(pos, m, 16)
    cl, ll, *_ = O.walk(0, 0.5)
    assert cl.size == 0 and ll.tolist() == [0]
    r = O.forces(0.5, 0.01)
    assert (r["n_pc"] == 0).all() and (r["n_pp"] == 9).all()


@pytest.mark.parametrize("n_leaf,n_group", [(16, 16), (16, 64), (4, 32)])
@pytest.mark.parametrize("theta", [0.0, 0.3, 0.5, 1.0, 1e6])
def test_coverage_invariant(n_leaf, n_group, theta):
    pos, _ = inputs.plummer(2048, 21)
    m = (np.random.default_rng(1).random(2048) + 0.5).astype(np.float32)
    O = oracle.Oracle(pos, m, n_leaf, n_group)
    c = O.cells()
    leaves = set(np.nonzero(c["n_child"] == 0)[0].tolist())
    for g in range(0, O.n_groups, 5):
        cl, ll, *_ = O.walk(g, theta)
        assert len(set(cl.tolist())) == cl.size and len(set(ll.tolist())) == ll.size
        assert set(ll.tolist()) <= leaves
        assert c["count"][cl].sum() + c["count"][ll].sum() == 2048
        assert abs(c["M"][cl].sum() + c["M"][ll].sum() - c["M"][0]) < 1e-12 * c["M"][0]
        if theta == 0.0:
            assert cl.size == 0 and set(ll.tolist()) == leaves
        # the group's own particles are always reached particle-particle
        gcell = O.groups()[g]
        own = [l for l in ll if c["begin"][gcell] <= c["begin"][l] < c["begin"][gcell] + c["count"][gcell]]
        assert c["count"][own].sum() == c["count"][gcell]


def _gap(lo1, hi1, lo2, hi2):
    """Distance between two axis-aligned boxes, per-axis interval gap (textbook AABB distance)."""
    g = np.maximum(0.0, np.maximum(lo1 - hi2, lo2 - hi1))
    return np.sqrt((g * g).sum(-1))


@pytest.mark.parametrize("theta", [0.35, 0.5, 0.8])
def test_walk_brute_force_all_pairs(theta):
    """cell c is in cell-list(g) iff every proper ancestor of c below the root... is opened and c is not;
    c is in leaf-list(g) iff c and all its ancestors are opened and c is a leaf (recursive definition)."""
    pos, m = inputs.uniform_cube(600, 8)
    O = oracle.Oracle(pos, m, 4, 16)
    c = O.cells()
    nc = O.n_cells
    lo = c["b"] - c["h"][:, None]
    hi = c["b"] + c["h"][:, None]
    for g in range(O.n_groups):
        gc = O.groups()[g]
        d = _gap(lo, hi, lo[gc], hi[gc])
        opened = d * theta <= 2 * c["h"]
        opened[0] = True                                  # the root is always expanded
        anc_open = np.ones(nc, bool)                      # all proper ancestors opened
        for i in range(1, nc):                            # parents precede children (pre-order ids)
            p = c["parent"][i]
            anc_open[i] = anc_open[p] and opened[p]
        want_cell = sorted(np.nonzero(anc_open & ~opened)[0].tolist())
        want_leaf = sorted(np.nonzero(anc_open & opened & (c["n_child"] == 0))[0].tolist())
        cl, ll, *_ = O.walk(g, theta)
        assert sorted(cl.tolist()) == want_cell
        assert sorted(ll.tolist()) == want_leaf


def test_huge_theta_opens_only_touching_cells():
    pos, m = inputs.plummer(1024, 1)
    O = oracle.Oracle(pos, m, 16)
    c = O.cells()
    lo = c["b"] - c["h"][:, None]
    hi = c["b"] + c["h"][:, None]
    for g in range(0, O.n_groups, 9):
        gc = O.groups()[g]
        cl, ll, *_ = O.walk(g, 1e9)
        assert (_gap(lo[ll], hi[ll], lo[gc], hi[gc]) == 0).all()
        assert (_gap(lo[cl], hi[cl], lo[gc], hi[gc]) > 0).all()


def test_fp32_shadow_flips_are_borderline():
    """R16: the fp32 decision differs from the fp64 one only where the fp64 margin is at fp32 rounding level."""
    pos, m = inputs.plummer(65536, 2)
    O = oracle.Oracle(pos, m, 16)
    sel = np.arange(0, O.n_groups, 3)
    r64 = O.forces(0.5, 0.01, shadow32=False, groups=sel, stats=True)
    r32 = O.forces(0.5, 0.01, shadow32=True, groups=sel, stats=True)
    assert (r64["tests"] > 0).all()
    flipped = r64["flips"] > 0
    assert flipped.sum() <= 1e-3 * sel.size + 5         # "a handful per 1e5 groups"
    # a flip needs a margin of a few fp32 ulps relative to the coordinates (|b| <~ 10, l >~ 1e-3)
    assert (r64["min_margin"][flipped] < 1e-4).all()
    # groups without a flip have identical counts
    grp = O.groups()[sel]
    c = O.cells()
    perm = O.perm()
    for k in np.nonzero(~flipped)[0][::50]:
        i = perm[c["begin"][grp[k]]]
        assert r64["n_pc"][i] == r32["n_pc"][i] and r64["n_pp"][i] == r32["n_pp"][i]
    # total flips counted the same way in both modes
    assert np.array_equal(r64["flips"], r32["flips"])


# ---- R20: the fp32 form of the boundary contains the tight box, so R14 survives in FP32 ----
@pytest.mark.parametrize("n_leaf,n_group", [(4, 64), (1, 8), (16, 64)])
def test_fp32_boundary_contains_box_and_own_cells_always_open(n_leaf, n_group):
    """Regression pin (found on the GPU): with b32 = fp32(b), h32 = fp32(h) a particle on a face of
    its group's tight box can fall outside the fp32 cube; alone in a leaf (h = 0) it is then NOT
    opened and meets its own monopole.  Under R20 every cell inside a group opens in fp32 too."""
    pos, mass = inputs.plummer(3000, 12)
    o = oracle.Oracle(pos, mass, n_leaf, n_group)
    c = o.cells()
    b32, h32 = o.bnd32()
    perm = o.perm()
    x = pos.astype(np.float32)
    # containment as the FP32 test evaluates it: fl32(|x - b32|) <= h32 for every member of every cell
    for i in range(o.n_cells):
        mem = perm[c["begin"][i]:c["begin"][i] + c["count"][i]]
        reach = np.abs(x[mem] - b32[i]).astype(np.float32).max()
        assert reach <= h32[i]
    assert (h32 >= c["h"]).all()
    ulp = 1.2e-7 * (np.abs(c["b"]).max(1) + c["h"])
    assert (h32 - c["h"] <= 2 * ulp).all()          # ... and by no more than rounding
    # consequence: in the fp32 shadow no cell overlapping a group's own particles is left unopened,
    # and the shadow lists still cover every particle exactly once
    groups = o.groups()
    for g in range(0, o.n_groups, 3):
        gb, ge = c["begin"][groups[g]], c["begin"][groups[g]] + c["count"][groups[g]]
        cl, ll, _, _, _ = o.walk(g, 0.6, shadow32=True)
        assert not ((c["begin"][cl] < ge) & (c["begin"][cl] + c["count"][cl] > gb)).any()
        assert c["count"][cl].sum() + c["count"][ll].sum() == o.n


def test_flip_audit_finds_exactly_the_flipped_tests_within_survey_bound():
    """R16 in SURVEY 8(c)'s absolute form (oracle.flip_audit): for every group whose fp32-shadow walk differs from the fp64
    one, the cells decided differently are as many as the walk counted flips, and each has a slack |d theta - 2h| within
    8 * 2^-23 * (max_k(|b_c,k| + |b_g,k|) + h_c + h_g) * max(theta, 1).  Groups without a flip are not listed."""
    pos, m = inputs.plummer(65536, 2)
    O = oracle.Oracle(pos, m, 16)
    r = O.forces(0.3, 0.01, shadow32=True, stats=True)
    rows = oracle.flip_audit(O, 0.3, r["flips"])
    assert int(r["flips"].sum()) >= 3                    # the case has flips to audit (5 with this seed)
    assert sorted(g for g, _, _ in rows) == sorted(np.nonzero(r["flips"] > 0)[0].tolist())
    for g, f, cells in rows:
        assert len(cells) == f == int(r["flips"][g])
        for x, slack, bound in cells:
            assert 0.0 <= slack <= bound < 1e-4
    # with a subset of groups the indices are mapped back to group numbers
    sel = np.array(sorted(g for g, _, _ in rows)[:2] + [7], dtype=np.int64)
    rs = O.forces(0.3, 0.01, shadow32=True, groups=sel, stats=True)
    assert [g for g, _, _ in oracle.flip_audit(O, 0.3, rs["flips"], sel)] == sel[:2].tolist()
