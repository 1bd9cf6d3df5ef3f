"""Device-side tree build (option "device_build") — `-m gpu`.

The GPU builder must produce the SAME tree as the host builder and as the oracle: identical cells, links,
groups (Morton order), bit-identical fp32 boundary cubes, moments equal up to the last fp32 bit (the
particle order inside a leaf — hence the fp64 summation order — may differ), and therefore exactly the same
interaction counts and forces within the usual tolerances."""
import numpy as np
import pytest

from oracle import Oracle
from paper_1005_5384_b200 import binding as B
from paper_1005_5384_b200 import build as tc_build
from paper_1005_5384_b200 import inputs
from test_gpu_parity import check

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    tc_build.build()


def _trees(pos, mass, n_leaf, n_group):
    out = []
    for dev in (0, 1):
        with B.TreeCode(n_group=n_group) as tc:
            tc.set_option("device_build", dev)
            tc.set_particles(pos, mass)
            tc.build(n_leaf)
            out.append((tc.stats(), tc.tree()))
    return out


def _same_tree(h, d, pos):
    (sh, th), (sd, td) = h, d
    for k in ("n", "n_cells", "n_leaves", "n_groups", "depth", "tree_bytes"):
        assert sh[k] == sd[k], k
    assert np.array_equal(th["link"], td["link"])
    assert np.array_equal(th["groups"], td["groups"])
    assert np.array_equal(th["bnd"], td["bnd"])                      # boundary cubes: bit-identical
    n = sh["n"]
    assert np.array_equal(np.sort(td["perm"]), np.arange(n))
    # same members per leaf (order inside a leaf may differ)
    leaves = np.where(th["link"][:, 1] == 0)[0]
    for c in leaves[:: max(1, len(leaves) // 500)]:
        b, k = th["link"][c, 2], th["link"][c, 3]
        assert set(th["perm"][b:b + k].tolist()) == set(td["perm"][b:b + k].tolist())
    # moments: equal up to fp32 rounding of slightly different fp64 sums
    ext = max(1.0, float(np.abs(pos).max()))
    assert np.allclose(th["xm"][:, 3], td["xm"][:, 3], rtol=2e-7, atol=0)
    assert np.abs(th["xm"][:, :3] - td["xm"][:, :3]).max() <= 2.4e-7 * ext
    qs = np.abs(th["q"]).max(1) + 1e-30
    assert (np.abs(th["q"] - td["q"]).max(1) <= 1e-5 * qs + 1e-12 * th["xm"][:, 3] * ext * ext).all()


@pytest.mark.parametrize("name,n_leaf,n_group", [("plummer_1k", 16, 64), ("plummer_64k", 16, 96), ("cube_64k", 8, 32),
                                                   ("plummer_64k", 1, 1), ("plummer_1m", 16, 96)])
def test_device_tree_equals_host_tree(name, n_leaf, n_group):
    pos, mass, *_ = inputs.make(name)
    h, d = _trees(pos, mass, n_leaf, n_group)
    _same_tree(h, d, pos)


def test_device_tree_degenerate_inputs():
    # one particle; two particles; coincident particles (level-21 leaf); all particles in one leaf
    for pos, mass, n_leaf in [
        (np.array([[0.5, 0.25, -1.0]], np.float32), np.array([1.0], np.float32), 16),
        (np.array([[0, 0, 0], [1, 2, 3]], np.float32), np.array([1.0, 2.0], np.float32), 1),
        (None, None, 16),
        (inputs.plummer(12, 3)[0], inputs.plummer(12, 3)[1], 16),
    ]:
        if pos is None:
            pos, mass = inputs.plummer(2048, 11)
            pos[:200] = pos[0]
        h, d = _trees(pos, mass, n_leaf, 64)
        _same_tree(h, d, pos)


@pytest.mark.parametrize("name", ["plummer_1k", "plummer_64k"])
def test_forces_on_device_built_tree_match_oracle(name):
    pos, mass, theta, eps, n_leaf = inputs.make(name)
    with B.TreeCode(n_group=64) as tc:
        tc.set_option("device_build", 1)
        tc.set_particles(pos, mass)
        tc.build(n_leaf)
        acc, pot = tc.forces(theta, eps)
        n_pc, n_pp = tc.counts()
    check(acc, pot, n_pc, n_pp, Oracle(pos, mass, n_leaf, 64).forces(theta, eps, shadow32=True))


def test_device_and_host_build_times_1m():
    """Prints both build times.  The host side of the box varies from run to run, so the guard is loose: the device
    build (measured 1.1-1.3 ms) must not take more than twice the host build + copy (6-8 ms) at N = 2^20."""
    pos, mass, theta, eps, n_leaf = inputs.make("plummer_1m")
    t = {}
    for dev in (0, 1):
        with B.TreeCode() as tc:
            tc.set_option("device_build", dev)
            tc.set_particles(pos, mass)
            ts = []
            for _ in range(4):
                tc.build(n_leaf)
                ts.append(tc.stats()["t_host_ms"] + tc.stats()["t_copy_ms"])
            t[dev] = min(ts[1:])
    print(f"tc_build N=2^20: host {t[0]:.2f} ms (build + copy), device {t[1]:.2f} ms")
    assert t[0] > 0 and 0 < t[1] <= 2.0 * t[0]


def test_device_inputs_device_build_leapfrog_matches_host_build():
    """Device pointers + device build: nothing crosses PCIe per step; the trajectory equals the host-build one."""
    import torch
    from paper_1005_5384_b200 import integrate
    pos, mass, vel = inputs.two_plummer(1 << 18, with_velocities=True)
    logs = []
    for dev in (0, 1):
        st = torch.cuda.Stream()
        with torch.cuda.stream(st), B.TreeCode() as tc:
            tc.set_option("device_build", dev)
            tc.set_stream(st.cuda_stream)
            d_pos, d_vel, d_mass = torch.from_numpy(pos).cuda(), torch.from_numpy(vel).cuda(), torch.from_numpy(mass).cuda()
            logs.append(integrate.leapfrog_kdk(tc, d_pos, d_vel, d_mass, 1.0 / 128, 3, 0.5, 0.005, 16))
            x_end = d_pos.cpu().numpy()
        logs[-1].append(x_end)
    (h, d) = logs
    assert np.abs(h[-1] - d[-1]).max() <= 1e-6                     # same positions after 3 steps
    for a, b in zip(h[:-1], d[:-1]):
        assert a["interactions"] == b["interactions"]              # identical trees -> identical lists
        assert abs(a["E"] - b["E"]) <= 1e-7 * abs(a["E"])
    print(f"leapfrog N=2^18: per-step build host {np.mean([r['t_host_ms'] + r['t_copy_ms'] for r in h[1:-1]]):.2f} ms, "
          f"device {np.mean([r['t_host_ms'] for r in d[1:-1]]):.2f} ms")


def test_device_build_rejects_bad_particles_and_switches_back_to_host():
    import torch
    pos, mass, *_ = inputs.make("plummer_1k")
    with B.TreeCode(n_group=96) as tc:
        tc.set_option("device_build", 1)
        bad = torch.from_numpy(pos).cuda().clone()
        bad[5, 1] = float("nan")
        with pytest.raises(B.TcError) as e:
            tc.set_particles(bad, torch.from_numpy(mass).cuda())
        assert e.value.code == B.TC_EINVAL
        badm = mass.copy(); badm[7] = -1.0
        with pytest.raises(B.TcError) as e:
            tc.set_particles(pos, badm)
        assert e.value.code == B.TC_EINVAL
        # device-only particles, then a HOST build: the host copy is fetched from the device
        tc.set_particles(torch.from_numpy(pos).cuda(), torch.from_numpy(mass).cuda())
        tc.set_option("device_build", 0)
        tc.build(16)
        acc, pot = tc.forces(0.5, 0.01)
        n_pc, n_pp = tc.counts()
    check(acc, pot, n_pc, n_pp, Oracle(pos, mass, 16, 96).forces(0.5, 0.01, shadow32=True))


def test_pinned_host_inputs_take_the_direct_dma_path_and_bad_values_are_still_refused():
    """Device build with PAGE-LOCKED host inputs: DMA + pack kernel, no host pass — same tree, same forces as with
    pageable inputs; validation now happens in the pack kernel."""
    import torch
    pos, mass, theta, eps, n_leaf = inputs.make("plummer_64k")
    p_pin, m_pin = torch.from_numpy(pos).pin_memory().numpy(), torch.from_numpy(mass).pin_memory().numpy()
    out = []
    for p, m in ((pos, mass), (p_pin, m_pin), (p_pin, mass)):       # pageable, pinned, mixed
        with B.TreeCode() as tc:
            tc.set_option("device_build", 1)
            tc.set_particles(p, m)
            tc.build(n_leaf)
            acc, pot = tc.forces(theta, eps)
            out.append((acc, pot, tc.counts(), tc.stats()["n_cells"]))
    for o in out[1:]:
        assert np.array_equal(o[0], out[0][0]) and np.array_equal(o[1], out[0][1]) and o[3] == out[0][3]
        assert np.array_equal(o[2][0], out[0][2][0]) and np.array_equal(o[2][1], out[0][2][1])
    bad = torch.from_numpy(pos.copy()).pin_memory().numpy()
    bad[7, 1] = np.inf
    with B.TreeCode() as tc:
        tc.set_option("device_build", 1)
        with pytest.raises(B.TcError) as e:
            tc.set_particles(bad, m_pin)
        assert e.value.code == B.TC_EINVAL
        tc.set_particles(p_pin, m_pin)                                # the context is still usable
        tc.build(n_leaf)
        tc.set_option("device_build", 0)                              # host build needs the host copy: fetched lazily
        tc.build(n_leaf)
        acc, _ = tc.forces(theta, eps)
        assert np.abs(acc - out[0][0]).max() <= 2e-6 * np.abs(out[0][0]).max()


def test_pure_morton_schedule_with_very_many_groups():
    """>= 400 000 groups: both builders schedule in pure Morton order (tc_lanes.h, schedule_class_shift); the schedule
    changes only WHEN a group runs, so counts are identical and forces agree to summation-order rounding."""
    pos, mass = inputs.uniform_cube(1 << 19, 33)
    res = {}
    for dev in (0, 1):
        with B.TreeCode(n_group=1) as tc:
            tc.set_option("device_build", dev)
            tc.set_particles(pos, mass)
            tc.build(1)
            assert tc.stats()["n_groups"] >= 400000
            acc, pot = tc.forces(0.7, 0.01)
            res[dev] = (acc, pot) + tc.counts()
    assert np.array_equal(res[0][2], res[1][2]) and np.array_equal(res[0][3], res[1][3])
    assert np.allclose(res[0][0], res[1][0], rtol=2e-5, atol=1e-7) and np.allclose(res[0][1], res[1][1], rtol=2e-5)
    o = Oracle(pos, mass, 1, 1)
    gsel = np.arange(0, o.n_groups, o.n_groups // 500, dtype=np.int64)
    ref = o.forces(0.7, 0.01, shadow32=True, groups=gsel)
    check(res[1][0], res[1][1], res[1][2], res[1][3], ref, ref["n_pc"] >= 0)
