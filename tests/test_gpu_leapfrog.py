"""tc_leapfrog (device-side kick-drift-kick steps, SURVEY.md 8(f)-4 / BASELINE.json config 5) against the
oracle's fp64 leapfrog with the oracle's tree force — `-m gpu`.

The library keeps x and v in fp32 and fuses a dt/2 and v dt with one rounding each; the oracle integrates in
fp64 and hands its tree the positions rounded to fp32.  After a few steps the two states differ by a few fp32
ulps of the coordinates (bar: 1e-5 of max(1, |x|)); the accelerations of the last step are then checked with
the usual bars against the oracle evaluated on the LIBRARY's own final positions."""
import numpy as np
import pytest

import oracle
from oracle import Oracle
from paper_1005_5384_b200 import binding as B
from paper_1005_5384_b200 import build as tc_build
from paper_1005_5384_b200 import inputs
from test_gpu_parity import check

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", autouse=True)
def _built():
    tc_build.build()


def _start(n, seed):
    pos, mass = inputs.plummer(n, seed)
    vel = inputs.plummer_velocities64(pos.astype(np.float64), seed + 100, 1.0, 1.0).astype(np.float32)
    return pos, vel, mass


def _native(pos, vel, mass, dt, chunks, n_leaf, n_group, theta, eps, device_build, **opts):
    import torch
    with B.TreeCode(n_group=n_group) as tc:
        tc.set_option("device_build", device_build)
        for k, v in opts.items():
            tc.set_option(k, v)
        d = [torch.from_numpy(a.copy()).cuda() for a in (pos, vel, mass)]
        acc = torch.empty((len(mass), 3), dtype=torch.float32, device="cuda")
        pot = torch.empty(len(mass), dtype=torch.float32, device="cuda")
        for i, steps in enumerate(chunks):
            B.tc_leapfrog(tc.ctx, d[0], d[1], d[2], dt, steps, n_leaf, theta, eps, acc, pot, have_acc=i > 0)
        tc.sync()
        n_pc, n_pp = tc.counts()
        return d[0].cpu().numpy(), d[1].cpu().numpy(), acc.cpu().numpy(), pot.cpu().numpy(), n_pc, n_pp


@pytest.mark.parametrize("device_build", [0, 1])
@pytest.mark.parametrize("n,n_leaf,n_group,steps", [(2048, 8, 32, 4), (3001, 16, 96, 3)])
def test_leapfrog_matches_the_oracle_leapfrog(device_build, n, n_leaf, n_group, steps):
    theta, eps, dt = 0.5, 0.02, 1.0 / 128
    pos, vel, mass = _start(n, 31)
    x, v, a, p, n_pc, n_pp = _native(pos, vel, mass, dt, [steps], n_leaf, n_group, theta, eps, device_build)
    ox, ov, oa, op = oracle.leapfrog_kdk(pos, vel, dt, steps, oracle.tree_force(mass, theta, eps, n_leaf, n_group))
    assert np.abs(ox - pos).max() > 10 * dt * dt                                  # they did move
    assert (np.abs(x - ox) <= 1e-5 * np.maximum(1.0, np.abs(ox))).all()
    assert (np.abs(v - ov) <= 1e-5 * np.maximum(1.0, np.abs(ov))).all()
    # the last force evaluation, on the library's own final positions
    ref = Oracle(x, mass, n_leaf, n_group).forces(theta, eps, shadow32=True)
    check(a, p, n_pc, n_pp, ref)


def test_leapfrog_have_acc_continues_bit_for_bit_and_zero_steps_is_a_force_call():
    theta, eps, dt = 0.6, 0.02, 1.0 / 64
    pos, vel, mass = _start(1500, 33)
    one = _native(pos, vel, mass, dt, [4], 8, 32, theta, eps, 1)
    two = _native(pos, vel, mass, dt, [1, 2, 1], 8, 32, theta, eps, 1)
    for a, b in zip(one, two):
        assert np.array_equal(a, b)
    x, v, a, p, n_pc, n_pp = _native(pos, vel, mass, dt, [0], 8, 32, theta, eps, 0)
    assert np.array_equal(x, pos) and np.array_equal(v, vel)
    check(a, p, n_pc, n_pp, Oracle(pos, mass, 8, 32).forces(theta, eps, shadow32=True))


def test_leapfrog_with_variants_and_ragged_sizes():
    """n not a multiple of 4 (scalar tail of the kick/drift kernels), group_box + COM rule."""
    theta, eps, dt = 0.5, 0.02, 1.0 / 128
    for n in (1, 2, 1023):
        pos, vel, mass = _start(n, 35)
        x, v, a, p, n_pc, n_pp = _native(pos, vel, mass, dt, [2], 4, 16, theta, eps, 1, group_box=1, open_rule=1)
        f = oracle.tree_force(mass, theta, eps, 4, 16, open_rule=1, group_box=True)
        ox, ov, oa, op = oracle.leapfrog_kdk(pos, vel, dt, 2, f)
        assert (np.abs(x - ox) <= 1e-5 * np.maximum(1.0, np.abs(ox))).all()
        assert (np.abs(v - ov) <= 1e-5 * np.maximum(1.0, np.abs(ov))).all()


def test_leapfrog_argument_errors():
    import torch
    pos, vel, mass = _start(64, 37)
    with B.TreeCode() as tc:
        d_pos, d_vel, d_mass = (torch.from_numpy(a).cuda() for a in (pos, vel, mass))
        acc = torch.empty((64, 3), dtype=torch.float32, device="cuda")
        with pytest.raises(B.TcError) as e:                       # host pointer
            B.tc_leapfrog(tc.ctx, pos, d_vel, d_mass, 0.01, 1, 16, 0.5, 0.01, acc)
        assert e.value.code == B.TC_EINVAL
        big = torch.empty(64 * 3 + 1, dtype=torch.float32, device="cuda")
        with pytest.raises(B.TcError) as e:                       # misaligned view
            B.tc_leapfrog(tc.ctx, d_pos, big[1:].view(64, 3), d_mass, 0.01, 1, 16, 0.5, 0.01, acc)
        assert e.value.code == B.TC_EINVAL
        with pytest.raises(B.TcError) as e:
            B.tc_leapfrog(tc.ctx, d_pos, d_vel, d_mass, 0.01, -1, 16, 0.5, 0.01, acc)
        assert e.value.code == B.TC_EINVAL
        with pytest.raises(B.TcError) as e:                       # theta < 0 is refused by the tc_forces inside
            B.tc_leapfrog(tc.ctx, d_pos, d_vel, d_mass, 0.01, 1, 16, -0.5, 0.01, acc)
        assert e.value.code == B.TC_EINVAL


def test_native_leapfrog_equals_the_torch_harness():
    """integrate.leapfrog_kdk(native=True) (tc_leapfrog) and the torch elementwise harness on the same start."""
    import torch
    from paper_1005_5384_b200 import integrate
    pos, vel, mass = _start(4096, 39)
    out = []
    for native in (False, True):
        with B.TreeCode(n_group=64) as tc:
            tc.set_option("device_build", 1)
            d_pos, d_vel, d_mass = (torch.from_numpy(a.copy()).cuda() for a in (pos, vel, mass))
            log = integrate.leapfrog_kdk(tc, d_pos, d_vel, d_mass, 1.0 / 128, 5, 0.5, 0.02, 16, native=native)
            out.append((d_pos.cpu().numpy(), d_vel.cpu().numpy(), log[-1]["dE_rel"]))
    assert np.allclose(out[0][0], out[1][0], rtol=0, atol=2e-6) and np.allclose(out[0][1], out[1][1], rtol=0, atol=2e-6)
    assert out[1][2] < 2e-4
