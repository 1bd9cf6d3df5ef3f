"""Pins for the oracle's tree (O1-O4) and cell properties (O3).

Cited passages: octree definition PAPER.md:45-47 (§2.1); tight bounding box and
boundary cube Fig. 1; cell properties; groups
PAPER.md:49,65.  Readings R4-R8 of DESIGN.md.

The oracle builds its tree by top-down recursion (partition by bit).  These
tests re-derive the cell set from the *definition* in a different way (group
particles by key prefix level by level, in numpy), and check moments against
the parallel-axis merge of the children — neither is how the oracle computes.
"""
import numpy as np
import pytest

import oracle
from paper_1005_5384_b200 import inputs


def brute_cells(pos, n_leaf):
    """Set of (level, ix, iy, iz, count, is_leaf) from the definition (O1, O2)."""
    x = pos.astype(np.float64)
    lo, hi = x.min(0), x.max(0)
    side = (hi - lo).max() * (1.0 + 2.0 ** -20)
    if side == 0.0:
        side = 1.0
    org = (lo + hi) / 2.0 - side / 2.0
    g = np.clip(np.floor((x - org) * (2.0 ** 21 / side)), 0, 2 ** 21 - 1).astype(np.int64)
    out = set()
    alive = {(0, 0, 0): np.arange(len(x))}  # cells of the current level that exist
    for level in range(0, 22):
        nxt = {}
        for key, members in alive.items():
            leaf = (len(members) <= n_leaf) or (level == 21)
            out.add((level,) + key + (len(members), leaf))
            if leaf:
                continue
            sub = g[members] >> (21 - (level + 1))
            for k in {tuple(r) for r in sub}:
                nxt[k] = members[(sub == np.array(k)).all(1)]
        alive = nxt
        if not alive:
            break
    return out, g


def oracle_cells(O, g):
    c = O.cells()
    perm = O.perm()
    out = set()
    for i in range(O.n_cells):
        lev = int(c["level"][i])
        first = perm[c["begin"][i]]
        key = tuple(int(v) for v in (g[first] >> (21 - lev))) if lev > 0 else (0, 0, 0)
        out.add((lev,) + key + (int(c["count"][i]), bool(c["n_child"][i] == 0)))
    return out


@pytest.mark.parametrize("n,seed,n_leaf", [(1, 0, 4), (7, 1, 2), (64, 2, 1), (300, 3, 4), (1024, 1, 16)])
def test_tree_matches_definition(n, seed, n_leaf):
    pos, m = inputs.plummer(n, seed)
    O = oracle.Oracle(pos, m, n_leaf)
    want, g = brute_cells(pos, n_leaf)
    assert np.array_equal(O.grid().astype(np.int64), g)
    assert oracle_cells(O, g) == want
    assert O.n_leaves == sum(1 for t in want if t[-1])


def test_tree_invariants_and_order():
    pos, m = inputs.plummer(4096, 11)
    n_leaf = 16
    O = oracle.Oracle(pos, m, n_leaf, n_group=64)
    c = O.cells()
    perm = O.perm()
    assert sorted(perm.tolist()) == list(range(4096))  # a permutation
    leaf = c["n_child"] == 0
    assert c["count"][leaf].sum() == 4096
    assert (c["count"][leaf & (c["level"] < 21)] <= n_leaf).all()   # R4
    assert (c["count"][~leaf] > n_leaf).all()
    # children partition the parent into contiguous ranges, in octant order (R6)
    for i in np.nonzero(~leaf)[0]:
        ch = c["child"][i][c["child"][i] >= 0]
        assert len(ch) == c["n_child"][i] >= 1
        assert c["begin"][ch[0]] == c["begin"][i]
        assert (c["begin"][ch[1:]] == c["begin"][ch[:-1]] + c["count"][ch[:-1]]).all()
        assert c["count"][ch].sum() == c["count"][i]
        assert (c["parent"][ch] == i).all() and (c["level"][ch] == c["level"][i] + 1).all()
    # Morton order of the particle permutation
    g = O.grid().astype(np.uint64)[perm]
    key = np.zeros(4096, dtype=np.uint64)
    for b in range(21):
        for k, sh in ((0, 2), (1, 1), (2, 0)):
            key |= ((g[:, k] >> np.uint64(b)) & np.uint64(1)) << np.uint64(3 * b + sh)
    key = key.astype(np.int64)
    # the recursion orders particles down to leaf resolution: leaves, taken by `begin`,
    # occupy disjoint increasing key ranges (order inside a leaf is unspecified)
    lv = np.nonzero(leaf)[0]
    lv = lv[np.argsort(c["begin"][lv])]
    kmin = np.array([key[c["begin"][i]: c["begin"][i] + c["count"][i]].min() for i in lv])
    kmax = np.array([key[c["begin"][i]: c["begin"][i] + c["count"][i]].max() for i in lv])
    assert (kmin[1:] > kmax[:-1]).all()
    # mean leaf occupancy is a factor 3-4 below N_leaf
    occ = c["count"][leaf].mean()
    assert n_leaf / 4.5 < occ < n_leaf / 2.5
    # groups (O4, R5): a partition of the particles; maximal cells with count <= N_group
    grp = O.groups()
    assert c["count"][grp].sum() == 4096
    assert (np.diff(c["begin"][grp]) > 0).all()                     # Morton order
    for gcell in grp:
        assert c["count"][gcell] <= 64 or c["n_child"][gcell] == 0
        p = c["parent"][gcell]
        if p >= 0:
            assert c["count"][p] > 64


def test_groups_equal_leaves_when_ngroup_equals_nleaf():
    pos, m = inputs.uniform_cube(2000, 5)
    O = oracle.Oracle(pos, m, 8)            # n_group defaults to n_leaf
    c = O.cells()
    assert sorted(O.groups().tolist()) == sorted(np.nonzero(c["n_child"] == 0)[0].tolist())


def test_depth_cap_coincident_particles():
    """R7: coincident particles cannot be split; the level-21 cell is a leaf whatever its count."""
    pos = np.zeros((40, 3), np.float32)
    pos[:20] = [0.25, 0.5, 0.75]
    pos[20:] = [-1.0, -1.0, -1.0]
    m = np.full(40, 1 / 40, np.float32)
    O = oracle.Oracle(pos, m, 4)
    c = O.cells()
    leaf = c["n_child"] == 0
    assert O.depth == 21 and c["count"][leaf].sum() == 40
    assert sorted(c["count"][leaf].tolist()) == [20, 20]
    assert (c["level"][leaf] == 21).all()
    assert (c["h"][leaf] == 0).all()


def test_single_point_root_side():
    """O1: side == 0 -> side = 1."""
    O = oracle.Oracle(np.array([[3.0, -2.0, 1.0]], np.float32), np.array([2.0], np.float32), 4)
    org, side = O.root()
    assert side == 1.0 and np.allclose(org, [2.5, -2.5, 0.5])
    assert O.n_cells == 1 and O.n_groups == 1


def test_bbox_and_boundary_cube():
    """Fig. 1: tight bbox of the members; cube with the same centre, side = largest bbox side."""
    pos, m = inputs.plummer(2000, 4)
    O = oracle.Oracle(pos, m, 8)
    c = O.cells()
    perm = O.perm()
    x = pos.astype(np.float64)
    org, side = O.root()
    for i in range(0, O.n_cells, 7):
        mem = perm[c["begin"][i]: c["begin"][i] + c["count"][i]]
        assert np.array_equal(c["bmin"][i], x[mem].min(0)) and np.array_equal(c["bmax"][i], x[mem].max(0))
        assert np.array_equal(c["b"][i], (x[mem].min(0) + x[mem].max(0)) / 2)
        assert c["h"][i] == (x[mem].max(0) - x[mem].min(0)).max() / 2
        # bbox inside the geometric cell of that level
        w = side / 2 ** c["level"][i]
        cell_lo = org + np.floor((x[mem[0]] - org) / w) * w
        assert (c["bmin"][i] >= cell_lo - 1e-9).all() and (c["bmax"][i] <= cell_lo + w + 1e-9).all()


def test_moments_parallel_axis_and_invariants():
    """PAPER.md:49 (mass, centre of mass, quadrupole; R10).  Children merge by the parallel-axis
    theorem: Q_parent = sum_c [Q_c + M_c (3 d d^T - |d|^2 I)], d = X_c - X_parent."""
    rng = np.random.default_rng(0)
    pos, _ = inputs.plummer(3000, 9)
    m = (rng.random(3000) + 0.1).astype(np.float32)       # unequal masses
    O = oracle.Oracle(pos, m, 8)
    c = O.cells()
    assert abs(c["M"][0] - m.astype(np.float64).sum()) < 1e-12 * c["M"][0]
    assert np.allclose(c["X"][0], (m[:, None].astype(np.float64) * pos).sum(0) / m.astype(np.float64).sum(), rtol=0, atol=1e-12)
    tr = c["Q"][:, 0] + c["Q"][:, 1] + c["Q"][:, 2]
    scale = np.abs(c["Q"]).max(1) + 1e-300
    assert (np.abs(tr) <= 1e-12 * scale + 1e-18).all()                  # traceless
    assert ((c["X"] >= c["bmin"] - 1e-12) & (c["X"] <= c["bmax"] + 1e-12)).all()   # COM in bbox
    assert (c["Q"][c["count"] == 1] == 0).all()                         # a point has no quadrupole

    def full(q):
        return np.array([[q[0], q[3], q[4]], [q[3], q[1], q[5]], [q[4], q[5], q[2]]])

    for i in np.nonzero(c["n_child"] > 0)[0]:
        ch = c["child"][i][c["child"][i] >= 0]
        M = c["M"][ch].sum()
        X = (c["M"][ch, None] * c["X"][ch]).sum(0) / M
        Q = np.zeros((3, 3))
        for k in ch:
            d = c["X"][k] - X
            Q += full(c["Q"][k]) + c["M"][k] * (3 * np.outer(d, d) - d.dot(d) * np.eye(3))
        assert abs(M - c["M"][i]) <= 1e-12 * M
        assert np.allclose(X, c["X"][i], rtol=0, atol=1e-12)
        assert np.allclose(Q, full(c["Q"][i]), rtol=0, atol=1e-12 * max(1.0, np.abs(Q).max()))


def test_quadrupole_of_known_configuration():
    """Two masses m at (+-s,0,0): Q = diag(4 m s^2, -2 m s^2, -2 m s^2) (textbook; golden file header)."""
    s, mm = 0.125, 1.0
    pos = np.array([[-s, 0, 0], [s, 0, 0]], np.float32)
    O = oracle.Oracle(pos, np.array([mm, mm], np.float32), 2)
    c = O.cells()
    assert O.n_cells == 1
    assert np.allclose(c["Q"][0], [4 * mm * s * s, -2 * mm * s * s, -2 * mm * s * s, 0, 0, 0], atol=1e-15)
    assert c["M"][0] == 2.0 and np.allclose(c["X"][0], 0)
    # an off-diagonal case: masses at +-(s, s, 0)/sqrt(2)-free version: (+-s, +-s, 0) -> Qxy = 3*2*m*s*s
    pos = np.array([[-s, -s, 0], [s, s, 0]], np.float32)
    c = oracle.Oracle(pos, np.array([mm, mm], np.float32), 2).cells()
    # y = (s,s,0): 3 y y^T - |y|^2 I = [[s2, 3 s2, 0], [3 s2, s2, 0], [0, 0, -2 s2]], times 2 m
    s2 = s * s
    assert np.allclose(c["Q"][0], [2 * s2, 2 * s2, -4 * s2, 6 * s2, 0, 0], atol=1e-15)
