"""The C-ABI library builds, loads and exports every symbol include/*.h declares.
No compute call needs a GPU here; the host-only context covers call-order errors."""
import os
import re

import numpy as np
import pytest

from paper_1005_5384_b200 import binding as B
from paper_1005_5384_b200 import build as tc_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    tc_build.build()


def test_header_symbols_are_exported():
    hdr = "".join(open(os.path.join(ROOT, "include", h)).read() for h in sorted(os.listdir(os.path.join(ROOT, "include"))))
    declared = set(re.findall(r"\b(tc_[a-z0-9_]+)\s*\(", hdr)) - {"tc_ctx"}
    assert declared == set(B.SYMBOLS), declared ^ set(B.SYMBOLS)
    L = B.lib()
    for s in declared:
        assert getattr(L, s) is not None


def test_stats_struct_size_matches_header():
    # 4 int64 + 4 int32 + 4 int64 + 3 double + 1 int64 + 4 double + 2 int64
    import ctypes
    assert ctypes.sizeof(B.tc_stats) == 4 * 8 + 4 * 4 + 4 * 8 + 3 * 8 + 8 + 4 * 8 + 2 * 8


def test_no_cpu_fallback_host_only_refuses_forces():
    with B.TreeCode(host_only=True) as tc:
        pos = np.random.default_rng(0).random((100, 3)).astype(np.float32)
        mass = np.full(100, 0.01, np.float32)
        tc.set_particles(pos, mass)
        tc.build(8)
        with pytest.raises(B.TcError) as e:
            tc.forces(0.5, 0.01)
        assert e.value.code == B.TC_ESTATE
        with pytest.raises(B.TcError) as e:                       # no CPU leapfrog either
            B.tc_leapfrog(tc.ctx, pos, pos.copy(), mass, 0.01, 1, 8, 0.5, 0.01, np.zeros_like(pos))
        assert e.value.code == B.TC_ESTATE


def test_error_codes():
    with B.TreeCode(host_only=True) as tc:
        with pytest.raises(B.TcError) as e:
            tc.build(16)
        assert e.value.code == B.TC_ESTATE
        pos = np.zeros((4, 3), np.float32)
        mass = np.ones(4, np.float32)
        bad = pos.copy(); bad[2, 1] = np.nan
        with pytest.raises(B.TcError) as e:
            tc.set_particles(bad, mass)
        assert e.value.code == B.TC_EINVAL
        with pytest.raises(B.TcError) as e:
            tc.set_particles(pos, -mass)
        assert e.value.code == B.TC_EINVAL
        with pytest.raises(B.TcError) as e:
            B.tc_set_particles(tc.ctx, pos, mass, 0)
        assert e.value.code == B.TC_EINVAL
        tc.set_particles(pos, mass)
        with pytest.raises(B.TcError) as e:
            tc.build(0)
        assert e.value.code == B.TC_EINVAL
        with pytest.raises(B.TcError) as e:
            tc.set_option("no_such_key", 1)
        assert e.value.code == B.TC_EINVAL
        with pytest.raises(B.TcError) as e:
            tc.set_option("n_group", 0)
        assert e.value.code == B.TC_EINVAL
        with pytest.raises(B.TcError) as e:
            tc.tree()
        assert e.value.code == B.TC_ESTATE
    B.tc_destroy(None)  # NULL is a no-op


def test_product_path_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1005_5384_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cpp", ".cu", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "treecode_oracle" not in src and "liboracle" not in src, f
