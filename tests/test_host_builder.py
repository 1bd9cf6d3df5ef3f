"""Host logic of the library (step A0: tc_build) against the oracle's own tree.

The two builders share no code: the oracle partitions recursively top-down and
sums moments directly over members (oracle/treecode_oracle.cpp), the library
sorts Morton keys, splits breadth-first and shifts children's moments
(csrc/tc_build.cpp).  Same readings O1-O4 => identical cell sets, bit-identical
fp32 boundaries, moments equal to fp32 rounding.  Runs without a GPU
(TC_FLAG_HOST_ONLY)."""
import numpy as np
import pytest

from oracle import Oracle
from paper_1005_5384_b200 import binding as B
from paper_1005_5384_b200 import build as tc_build
from paper_1005_5384_b200 import inputs


@pytest.fixture(scope="module", autouse=True)
def _built():
    tc_build.build()


def _compare(pos, mass, n_leaf, n_group):
    with B.TreeCode(host_only=True, n_group=n_group) as tc:
        tc.set_particles(pos, mass)
        tc.build(n_leaf)
        s, tr = tc.stats(), tc.tree()
        gbox = B.tc_get_group_boxes(tc.ctx)
    o = Oracle(pos, mass, n_leaf, n_group)
    assert (s["n_cells"], s["n_leaves"], s["n_groups"], s["depth"]) == (o.n_cells, o.n_leaves, o.n_groups, o.depth)
    n = len(mass)
    assert np.array_equal(np.sort(tr["perm"]), np.arange(n))
    oc = o.cells()
    # match cells by (level, first member, count): a single-child chain shares (begin, count)
    lvl = np.zeros(s["n_cells"], np.int64)
    for c in range(s["n_cells"]):                        # breadth-first: parents come first
        f, k = tr["link"][c, 0], tr["link"][c, 1]
        if k:
            lvl[f:f + k] = lvl[c] + 1
    key_o = {(int(l), int(b), int(c)): i for i, (l, b, c) in enumerate(zip(oc["level"], oc["begin"], oc["count"]))}
    idx = np.array([key_o[(int(l), int(b), int(c))] for l, (b, c) in zip(lvl, tr["link"][:, 2:4])])
    assert len(set(idx.tolist())) == o.n_cells
    # members of every cell are the same SET (order inside a leaf may differ)
    operm = o.perm()
    for c in np.random.default_rng(0).choice(o.n_cells, size=min(64, o.n_cells), replace=False):
        b, k = tr["link"][c, 2], tr["link"][c, 3]
        assert set(tr["perm"][b:b + k].tolist()) == set(operm[b:b + k].tolist())
    # leaf / node flags and child structure
    assert np.array_equal(tr["link"][:, 1], oc["n_child"][idx])
    for c in range(min(o.n_cells, 2000)):
        f, k = tr["link"][c, 0], tr["link"][c, 1]
        if k:
            want = [x for x in oc["child"][idx[c]] if x >= 0]
            assert idx[f:f + k].tolist() == want     # octant order 4bx+2by+bz
    # boundary cubes: bit-identical fp32 (Fig. 1; fp32 form = reading R20)
    b32, h32 = o.bnd32()
    assert np.array_equal(tr["bnd"][:, :3], b32[idx])
    assert np.array_equal(tr["bnd"][:, 3], h32[idx])
    assert np.array_equal(b32, oc["b"].astype(np.float32))
    assert (h32 >= oc["h"]).all() and (h32 <= oc["h"] * (1 + 3e-7) + 1.2e-7 * np.abs(oc["b"]).max(1)).all()
    # moments: fp64 parallel-axis vs fp64 direct sums, compared after fp32 rounding
    assert np.allclose(tr["xm"][:, 3], oc["M"][idx], rtol=2e-7, atol=0)
    ext = np.abs(pos).max()
    assert np.abs(tr["xm"][:, :3] - oc["X"][idx]).max() <= 1.2e-7 * ext
    qs = np.abs(oc["Q"][idx]).max(axis=1, keepdims=True) + 1e-300
    assert (np.abs(tr["q"] - oc["Q"][idx]) / qs).max() <= 2e-7
    # groups in the same (Morton) order
    assert np.array_equal(idx[tr["groups"]], o.groups())
    # tight boxes of the groups (variant R23): bit-identical fp32 half extents, their maximum is the cube's half side
    assert np.array_equal(gbox, o.ext32()[o.groups()])
    assert np.array_equal(gbox.max(axis=1), tr["bnd"][tr["groups"], 3])


@pytest.mark.parametrize("name,n_group", [("plummer_1k", 16), ("plummer_1k", 64), ("plummer_64k", 64), ("cube_64k", 16)])
def test_tree_matches_oracle(name, n_group):
    pos, mass, _, _, n_leaf = inputs.make(name)
    _compare(pos, mass, n_leaf, n_group)


@pytest.mark.parametrize("n_leaf", [1, 8, 32])
def test_tree_matches_oracle_n_leaf(n_leaf):
    pos, mass = inputs.plummer(4096, 11)
    _compare(pos, mass, n_leaf, max(n_leaf, 24))


def test_degenerate_inputs():
    rng = np.random.default_rng(5)
    one = np.array([[0.25, -1.0, 3.0]], np.float32)
    _compare(one, np.ones(1, np.float32), 16, 16)                       # single particle: root is a leaf
    same = np.repeat(one, 100, axis=0)
    _compare(same, np.full(100, 0.01, np.float32), 16, 64)              # all coincident: side = 1, level-21 leaf
    pos = rng.random((300, 3)).astype(np.float32)
    pos[:150] = pos[0]                                                  # a coincident clump inside a cloud
    _compare(pos, rng.random(300).astype(np.float32), 8, 32)
    mass = rng.random(500).astype(np.float32)
    mass[::3] = 0.0                                                     # massless particles
    _compare(rng.standard_normal((500, 3)).astype(np.float32), mass, 4, 16)
    line = np.zeros((64, 3), np.float32)
    line[:, 0] = np.linspace(-1, 1, 64)                                 # collinear: two axes have zero extent
    _compare(line, np.ones(64, np.float32), 4, 8)


def test_deep_clusters_through_the_radix_sort_fixup():
    """n large enough for the parallel radix sort (3 passes of 11 bits = 11 levels): a tight cluster and a
    coincident clump make cells far below level 11, i.e. long runs of equal prefixes that the fix-up must order."""
    rng = np.random.default_rng(9)
    n = 70000
    pos = rng.uniform(-1, 1, (n, 3)).astype(np.float32)
    pos[:9000] = (np.array([0.3, -0.2, 0.1]) + 1e-5 * rng.standard_normal((9000, 3))).astype(np.float32)   # levels 15-18
    pos[9000:9300] = pos[9000]                                                                            # level-21 leaf
    mass = np.full(n, 1.0 / n, np.float32)
    _compare(pos, mass, 8, 32)


def test_far_outlier_takes_the_lopsided_sort_path():
    """One escaper stretches the root cube: every other particle shares the top digits of its key, so the bucketed
    sort would run on one thread and the builder falls back to three global passes — same tree either way."""
    rng = np.random.default_rng(10)
    n = 70000
    pos = (1e-3 * rng.standard_normal((n, 3))).astype(np.float32)
    pos[123] = (100.0, 100.0, 100.0)
    _compare(pos, np.full(n, 1.0 / n, np.float32), 16, 64)


def test_sort_with_the_13_level_prefix_above_4m_particles():
    """N just above 2^22 takes the sort plan of the large runs (13-level prefix, 25 index bits, 3 passes;
    csrc/tc_build.cpp::sort_plan).  Checked against the oracle's tree without the per-cell Python loops of
    `_compare`: same cell / leaf / group counts and depth, and the same leaves — (first, count) of every leaf
    in Morton order and, leaf by leaf, the same member set."""
    n = (1 << 22) + 1237
    pos, mass = inputs.plummer(n, 77)
    with B.TreeCode(host_only=True, n_group=64) as tc:
        tc.set_particles(pos, mass)
        tc.build(16)
        s, tr = tc.stats(), tc.tree()
    o = Oracle(pos, mass, 16, 64)
    assert (s["n_cells"], s["n_leaves"], s["n_groups"], s["depth"]) == (o.n_cells, o.n_leaves, o.n_groups, o.depth)
    oc = o.cells()

    def leaves(begin, count, perm):
        order = np.argsort(begin, kind="stable")
        b, c = begin[order].astype(np.int64), count[order].astype(np.int64)
        assert np.array_equal(np.concatenate([[0], np.cumsum(c)[:-1]]), b) and c.sum() == n   # a partition of [0, n)
        leaf_id = np.repeat(np.arange(len(b)), c)
        return b, c, perm[np.lexsort((perm, leaf_id))]          # members sorted inside every leaf

    link = tr["link"]
    is_leaf = link[:, 1] == 0
    lb, lc, lp = leaves(link[is_leaf, 2], link[is_leaf, 3], np.asarray(tr["perm"]).astype(np.int64))
    m = oc["n_child"] == 0
    ob, on, op = leaves(oc["begin"][m], oc["count"][m], np.asarray(o.perm()).astype(np.int64))
    assert np.array_equal(lb, ob) and np.array_equal(lc, on)
    assert np.array_equal(lp, op)


def test_rebuilds_in_one_context_equal_fresh_contexts():
    """The builder's per-cell arrays and sort buffers live in the context between builds and are not cleared
    (csrc/tc_build.cpp): a big problem, then smaller and differently shaped ones in the SAME context must give,
    array for array, the tree a fresh context builds."""
    cases = [(inputs.plummer(40000, 51), 16, 64), (inputs.uniform_cube(3000, 52), 4, 16), (inputs.plummer(700, 53), 1, 1),
             (inputs.plummer(25000, 54), 8, 96), (inputs.uniform_cube(9000, 55), 16, 64)]
    with B.TreeCode(host_only=True) as reused:
        for (pos, mass), n_leaf, n_group in cases:
            reused.set_option("n_group", n_group)
            reused.set_particles(pos, mass)
            reused.build(n_leaf)
            s1, t1, g1 = reused.stats(), reused.tree(), B.tc_get_group_boxes(reused.ctx)
            with B.TreeCode(host_only=True, n_group=n_group) as fresh:
                fresh.set_particles(pos, mass)
                fresh.build(n_leaf)
                s2, t2, g2 = fresh.stats(), fresh.tree(), B.tc_get_group_boxes(fresh.ctx)
            for k in ("n_cells", "n_leaves", "n_groups", "depth"):
                assert s1[k] == s2[k]
            assert t1.keys() == t2.keys()
            for k in t1:
                assert np.array_equal(np.asarray(t1[k]), np.asarray(t2[k])), k
            assert np.array_equal(g1, g2)
