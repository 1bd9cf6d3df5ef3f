"""ORACLE — test infrastructure only (see oracle/treecode_oracle.cpp header).

Only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports the CUDA
binding and shares no code with ``paper_1005_5384_b200/csrc``.

``build()`` compiles the plain C++ oracle with g++ (``-ffp-contract=off``) into
``oracle/liboracle_tc.so``; ``Oracle`` is a thin ctypes wrapper.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "treecode_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle_tc.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle if the .so is missing or older than its source."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-fopenmp",
           "-ffp-contract=off", "-fno-fast-math", "-o", _LIB, _SRC]
    subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    L = C.CDLL(_LIB)
    vp, i64, i32, f64 = C.c_void_p, C.c_int64, C.c_int, C.c_double
    L.orc_create.restype = vp
    L.orc_create.argtypes = [i64, vp, vp, i32, i32]
    L.orc_destroy.argtypes = [vp]
    L.orc_set_variant.argtypes = [vp, i32, i32]
    L.orc_set_group_box.argtypes = [vp, i32]
    L.orc_get_ext32.argtypes = [vp, vp]
    for f in ("orc_n_cells", "orc_n_leaves", "orc_n_groups"):
        getattr(L, f).restype = i64
        getattr(L, f).argtypes = [vp]
    L.orc_depth.restype = i32
    L.orc_depth.argtypes = [vp]
    L.orc_get_root.argtypes = [vp, vp, vp]
    L.orc_get_grid.argtypes = [vp, vp]
    L.orc_get_perm.argtypes = [vp, vp]
    L.orc_get_groups.argtypes = [vp, vp]
    L.orc_get_cells.argtypes = [vp] + [vp] * 13
    L.orc_get_bnd32.argtypes = [vp, vp, vp]
    L.orc_walk.restype = i32
    L.orc_walk.argtypes = [vp, i64, f64, i32, vp, i64, vp, i64, vp, vp, vp, vp, vp]
    L.orc_forces.restype = i64
    L.orc_forces.argtypes = [vp, f64, f64, i32, i64, vp, vp, vp, vp, vp, vp, vp, vp]
    L.orc_direct.argtypes = [i64, vp, vp, f64, i64, vp, vp, vp]
    L.orc_num_threads.restype = i32
    _lib = L
    return L


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def num_threads() -> int:
    return int(_load().orc_num_threads())


class Oracle:
    """fp64 CPU tree-code: own tree (O1-O4), own walk (O5), own evaluation (O6)."""

    def __init__(self, pos, mass, n_leaf: int = 16, n_group: int | None = None, open_rule: int = 0,
                 quadrupole: bool = True, group_box: bool = False):
        L = _load()
        self.pos = np.ascontiguousarray(pos, dtype=np.float32)
        self.mass = np.ascontiguousarray(mass, dtype=np.float32)
        assert self.pos.ndim == 2 and self.pos.shape[1] == 3 and self.mass.shape == (self.pos.shape[0],)
        self.n = self.pos.shape[0]
        self.n_leaf = int(n_leaf)
        self.n_group = int(n_group if n_group is not None else n_leaf)
        self._h = L.orc_create(self.n, _p(self.pos), _p(self.mass), self.n_leaf, self.n_group)
        if not self._h:
            raise ValueError("orc_create failed (n, n_leaf, n_group must be >= 1)")
        # variants: open_rule 1 = group cube to cell COM (R21); quadrupole False = monopole only (R22)
        L.orc_set_variant(self._h, int(open_rule), int(bool(quadrupole)))
        self.open_rule, self.quadrupole = int(open_rule), bool(quadrupole)
        # variant R23: the group enters the opening test as its tight box (per-axis half extents)
        L.orc_set_group_box(self._h, int(bool(group_box)))
        self.group_box = bool(group_box)
        self.n_cells = int(L.orc_n_cells(self._h))
        self.n_leaves = int(L.orc_n_leaves(self._h))
        self.n_groups = int(L.orc_n_groups(self._h))
        self.depth = int(L.orc_depth(self._h))

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.orc_destroy(self._h)
            self._h = None

    # ---- tree inspection -------------------------------------------------
    def root(self):
        org = np.zeros(3)
        side = np.zeros(1)
        _lib.orc_get_root(self._h, _p(org), _p(side))
        return org, float(side[0])

    def grid(self):
        g = np.zeros((self.n, 3), dtype=np.int32)
        _lib.orc_get_grid(self._h, _p(g))
        return g

    def perm(self):
        p = np.zeros(self.n, dtype=np.int64)
        _lib.orc_get_perm(self._h, _p(p))
        return p

    def groups(self):
        g = np.zeros(self.n_groups, dtype=np.int32)
        _lib.orc_get_groups(self._h, _p(g))
        return g

    def cells(self) -> dict:
        nc = self.n_cells
        d = dict(level=np.zeros(nc, np.int32), parent=np.zeros(nc, np.int32),
                 child=np.zeros((nc, 8), np.int32), n_child=np.zeros(nc, np.int32),
                 begin=np.zeros(nc, np.int64), count=np.zeros(nc, np.int64),
                 bmin=np.zeros((nc, 3)), bmax=np.zeros((nc, 3)), b=np.zeros((nc, 3)), h=np.zeros(nc),
                 M=np.zeros(nc), X=np.zeros((nc, 3)), Q=np.zeros((nc, 6)))
        _lib.orc_get_cells(self._h, *[_p(d[k]) for k in
                                      ("level", "parent", "child", "n_child", "begin", "count",
                                       "bmin", "bmax", "b", "h", "M", "X", "Q")])
        return d

    def bnd32(self):
        """fp32 boundary cubes of the shadow test (R20): (b32 [n_cells,3], h32 [n_cells])."""
        b = np.zeros((self.n_cells, 3), np.float32)
        h = np.zeros(self.n_cells, np.float32)
        _lib.orc_get_bnd32(self._h, _p(b), _p(h))
        return b, h

    # ---- walk / forces ---------------------------------------------------
    def ext32(self):
        """fp32 half extents of every cell's tight box about its fp32 centre (R23): [n_cells,3]."""
        e = np.zeros((self.n_cells, 3), np.float32)
        _lib.orc_get_ext32(self._h, _p(e))
        return e

    def walk(self, group: int, theta: float, shadow32: bool = False):
        """(cell_list, leaf_list, min_margin, n_flips, n_tests) of one group (O5)."""
        cap = self.n_cells
        cl = np.zeros(cap, np.int32)
        ll = np.zeros(cap, np.int32)
        nc = np.zeros(1, np.int64)
        nl = np.zeros(1, np.int64)
        mm = np.zeros(1)
        nf = np.zeros(1, np.int64)
        nt = np.zeros(1, np.int64)
        rc = _lib.orc_walk(self._h, int(group), float(theta), int(shadow32), _p(cl), cap, _p(ll), cap,
                           _p(nc), _p(nl), _p(mm), _p(nf), _p(nt))
        assert rc == 0
        return cl[: nc[0]].copy(), ll[: nl[0]].copy(), float(mm[0]), int(nf[0]), int(nt[0])

    def forces(self, theta: float, eps: float, shadow32: bool = False, groups=None, stats: bool = False):
        """acc fp64 [n,3], pot fp64 [n], n_pc int64 [n], n_pp int64 [n] (+ per-group stats).

        ``groups``: optional int64 array of group indices; particles of other
        groups keep NaN (acc, pot) / -1 (counts).
        """
        acc = np.full((self.n, 3), np.nan)
        pot = np.full(self.n, np.nan)
        npc = np.full(self.n, -1, np.int64)
        npp = np.full(self.n, -1, np.int64)
        sel = None
        ng = self.n_groups
        if groups is not None:
            sel = np.ascontiguousarray(groups, dtype=np.int64)
            ng = sel.size
        gm = np.zeros(ng)
        gf = np.zeros(ng, np.int64)
        gt = np.zeros(ng, np.int64)
        total = _lib.orc_forces(self._h, float(theta), float(eps), int(shadow32), ng, _p(sel),
                                _p(acc), _p(pot), _p(npc), _p(npp), _p(gm), _p(gf), _p(gt))
        out = dict(acc=acc, pot=pot, n_pc=npc, n_pp=npp, interactions=int(total))
        if stats:
            out.update(min_margin=gm, flips=gf, tests=gt)
        return out


def flip_audit(o: "Oracle", theta: float, flips, groups=None, cells=None):
    """R16 audit in SURVEY.md 8(c)'s own form: a group whose fp32-shadow walk differs from the fp64 walk is accepted only
    if every test that was decided differently has an ABSOLUTE slack |d theta - 2 h_c| (fp64, O5) within a few fp32 ulps
    of the coordinates that enter it:  slack <= 8 * 2^-23 * (max_k(|b_c,k| + |b_g,k|) + h_c + h_g) * max(theta, 1).

    ``flips`` is the per-group flip count of ``forces(..., stats=True)`` (aligned with ``groups``, or with all groups).
    For every group with a flip both walks are repeated; the cells that sit on a list of one walk but not of the other,
    and whose parent does not, are exactly the tests decided differently (a parent of such a cell was opened by both
    walks; cells below it differ only as a consequence).  Default opening rule only (R1 / R9).
    Returns ``[(group, n_flips, [(cell, slack, bound), ...]), ...]``; the caller asserts slack <= bound and
    len(list) == n_flips.  Bookkeeping on the oracle's own tree data; no part of the force arithmetic."""
    assert o.open_rule == 0 and not o.group_box, "flip_audit: written for the default opening test (R1 / R9)"
    flips = np.asarray(flips)
    idx = np.nonzero(flips > 0)[0]
    if idx.size == 0:
        return []
    c = cells if cells is not None else o.cells()
    gcell = o.groups()
    out = []
    for k in idx:
        g = int(k if groups is None else np.asarray(groups)[k])
        c64, l64 = o.walk(g, theta, False)[:2]
        c32, l32 = o.walk(g, theta, True)[:2]
        cand = (set(c64.tolist()) ^ set(c32.tolist())) | (set(l64.tolist()) ^ set(l32.tolist()))
        top = sorted(x for x in cand if int(c["parent"][x]) not in cand)
        gc = int(gcell[g])
        bg, hg = c["b"][gc], float(c["h"][gc])
        rows = []
        for x in top:
            bc, hc = c["b"][x], float(c["h"][x])
            d = np.maximum(0.0, np.abs(bc - bg) - hc - hg)
            slack = abs(float(np.sqrt((d * d).sum())) * theta - 2.0 * hc)
            bound = 8.0 * 2.0 ** -23 * (float(np.max(np.abs(bc) + np.abs(bg))) + hc + hg) * max(theta, 1.0)
            rows.append((int(x), slack, bound))
        out.append((g, int(flips[k]), rows))
    return out


def direct(pos, mass, eps: float, targets=None):
    """fp64 direct summation: (acc [n_t,3], pot [n_t])."""
    L = _load()
    pos = np.ascontiguousarray(pos, dtype=np.float32)
    mass = np.ascontiguousarray(mass, dtype=np.float32)
    n = pos.shape[0]
    t = None if targets is None else np.ascontiguousarray(targets, dtype=np.int64)
    nt = n if t is None else t.size
    acc = np.zeros((nt, 3))
    pot = np.zeros(nt)
    L.orc_direct(n, _p(pos), _p(mass), float(eps), nt, _p(t), _p(acc), _p(pot))
    return acc, pot


# ---- time integration (BASELINE.json config 5; the paper leaves it on the host) -------------
def leapfrog_kdk(pos, vel, dt: float, steps: int, force, acc0=None):
    """Kick-drift-kick leapfrog in fp64, step by step as BASELINE.json config 5 writes it:

        v += a dt/2 ;  x += v dt ;  a = force(x) ;  v += a dt/2

    ``force(x64) -> (acc64, pot64)`` is any force law (``tree_force`` below, or an exact one in the pins).
    Returns (pos, vel, acc, pot) after ``steps`` steps; the inputs are not modified.
    Pins (tests/test_oracle_leapfrog.py): two-body circular orbit closed form, second-order convergence,
    exact time reversibility, momentum conservation.
    """
    x = np.array(pos, dtype=np.float64, copy=True)
    v = np.array(vel, dtype=np.float64, copy=True)
    a, p = force(x) if acc0 is None else (np.array(acc0, dtype=np.float64, copy=True), None)
    for _ in range(int(steps)):
        v += a * (0.5 * dt)
        x += v * dt
        a, p = force(x)
        v += a * (0.5 * dt)
    return x, v, a, p


def tree_force(mass, theta: float, eps: float, n_leaf: int = 16, n_group=None, shadow32: bool = True, **variants):
    """Force law for ``leapfrog_kdk``: a new Oracle tree on the positions ROUNDED TO fp32 (what the library is
    handed each step), opening decisions in the fp32 shadow by default (R16)."""
    def f(x64):
        o = Oracle(x64.astype(np.float32), mass, n_leaf, n_group, **variants)
        r = o.forces(theta, eps, shadow32=shadow32)
        return r["acc"], r["pot"]
    return f
