"""Stream ordering between torch and the library on torch's DEFAULT stream — `-m gpu`.

The raw handle of the legacy default stream is 0, and tc_set_stream(NULL) means "the context's own stream", which is
non-blocking: work queued there is not ordered with the default stream at all.  `TreeCode.use_torch_stream` passes the
default stream as cudaStreamLegacy instead (include/tc.h, tc_set_stream).  Each test below queues a long spin kernel on
the default stream in front of the write the library depends on (or behind the library's kernel, in front of the read):
without the ordering the library would see the buffer as it was BEFORE the write."""
import numpy as np
import pytest

from paper_1005_5384_b200 import binding as B
from paper_1005_5384_b200 import build as tc_build
from paper_1005_5384_b200 import inputs, integrate, parallel

pytestmark = pytest.mark.gpu
SPIN = 300_000_000          # cycles of torch.cuda._sleep: ~0.15 s at 1.9 GHz


@pytest.fixture(scope="module", autouse=True)
def _built():
    tc_build.build()


def test_default_stream_handle_is_passed_as_legacy():
    import torch
    assert torch.cuda.current_stream().cuda_stream == 0
    assert B.torch_stream_handle() == B.CUDA_STREAM_LEGACY
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        assert B.torch_stream_handle() == s.cuda_stream != 0


def test_forces_on_default_stream_wait_for_a_late_write_of_the_positions():
    import torch
    pos, mass, theta, eps, n_leaf = inputs.make("plummer_64k")
    n = len(mass)
    with B.TreeCode() as tc:                                         # synchronised reference, host buffers
        tc.set_particles(pos, mass)
        tc.build(n_leaf)
        a0, p0 = tc.forces(theta, eps)
    d_src, d_mass = torch.from_numpy(pos).cuda(), torch.from_numpy(mass).cuda()
    d_pos = d_src * 2.0                                              # what a too-early read would see: another (valid) system
    acc = torch.empty((n, 3), dtype=torch.float32, device="cuda")
    pot = torch.empty(n, dtype=torch.float32, device="cuda")
    torch.cuda.synchronize()
    with B.TreeCode() as tc:
        tc.use_torch_stream()
        tc.set_option("device_build", 1)                             # everything stays stream-ordered on the device
        # one pass up front: every buffer of the context exists afterwards, so that nothing in the pass under test
        # synchronises the device by accident (a first-use cudaMalloc) and hides a missing stream order
        tc.set_particles(d_pos, d_mass)
        tc.build(n_leaf)
        B.tc_forces(tc.ctx, theta, eps, acc, pot)
        tc.sync()
        torch.cuda._sleep(SPIN)
        d_pos.copy_(d_src)                                           # lands ~0.15 s from now
        tc.set_particles(d_pos, d_mass)
        tc.build(n_leaf)
        B.tc_forces(tc.ctx, theta, eps, acc, pot)
        torch.cuda._sleep(SPIN // 10)
        ha, hp = acc.cpu().numpy(), pot.cpu().numpy()                # torch's read, ordered behind the library's kernel
    from test_gpu_parity import rel_err
    assert rel_err(ha, a0).max() < 1e-4 and np.abs(hp - p0).max() < 1e-4 * np.abs(p0).max()


def test_leapfrog_on_default_stream_equals_side_stream():
    import torch
    pos, mass, vel = inputs.two_plummer(4096, with_velocities=True)
    res = []
    for side in (True, False):
        d_pos, d_vel, d_mass = (torch.from_numpy(np.ascontiguousarray(x)).cuda() for x in (pos, vel, mass))
        st = torch.cuda.Stream() if side else torch.cuda.current_stream()
        with torch.cuda.stream(st), B.TreeCode() as tc:
            integrate.leapfrog_kdk(tc, d_pos, d_vel, d_mass, 1.0 / 64, 3, 0.5, 0.01, n_leaf=16)
            torch.cuda.synchronize()
        res.append((d_pos.cpu().numpy(), d_vel.cpu().numpy()))
    assert np.array_equal(res[0][0], res[1][0]) and np.array_equal(res[0][1], res[1][1])


def test_forces_sharded_on_default_stream_without_set_stream():
    """The all-gather (here: a torch copy) reads the shard's rows on torch's stream: forces_sharded must have put the
    shard kernel on that stream itself — the caller never called set_stream."""
    import torch
    pos, mass, theta, eps, n_leaf = inputs.make("plummer_64k")
    n = len(mass)
    with B.TreeCode() as tc:
        tc.set_particles(pos, mass)
        tc.build(n_leaf)
        a0, p0 = tc.forces(theta, eps)
        n_slots = tc.shard_size()
        sc = {"rows": torch.full((n_slots, 4), float("nan"), dtype=torch.float32, device="cuda")}
        acc = torch.empty((n, 3), dtype=torch.float32, device="cuda")
        pot = torch.empty(n, dtype=torch.float32, device="cuda")
        torch.cuda.synchronize()
        parallel.forces_sharded(tc, theta, eps, acc, pot, scratch=sc)
        ha, hp = acc.cpu().numpy(), pot.cpu().numpy()
        assert np.array_equal(ha, a0) and np.array_equal(hp, p0)
