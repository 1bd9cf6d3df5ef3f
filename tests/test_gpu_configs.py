"""BASELINE.json configs 4 and 5 at FULL size on the GPU — `-m gpu`.

Config 4: Plummer N = 2^20, theta in {0.3, 0.5, 0.75, 1.0} x N_leaf in {8, 16, 32}: rms relative force
error against fp64 direct summation on 4096 sampled particles versus time.
Config 5: two offset Plummer spheres, N = 2^24, eps = 0.005: oracle parity over EVERY particle at step 0 (all
443 844 groups; the maximum error is a statement about the whole system) and on sampled groups at
step 10, 10 leapfrog KDK steps with a host tree rebuild each step (energy and momentum conservation).
Every comparison carries the R16 flip audit (test_gpu_parity.flip_audit).
The tables are printed (run with -s) and written to gpurun_out/ when that directory exists.
"""
import json
import os

import numpy as np
import pytest

from oracle import Oracle, direct
from paper_1005_5384_b200 import binding as B
from paper_1005_5384_b200 import build as tc_build
from paper_1005_5384_b200 import inputs
from test_gpu_parity import check, flip_audit, rel_err

pytestmark = pytest.mark.gpu
N_GROUP = 128          # the library's default and bench.py's setting
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    tc_build.build()


def _dump(name, obj):
    d = os.path.join(ROOT, "gpurun_out")
    if os.path.isdir(d):
        with open(os.path.join(d, name), "w") as f:
            json.dump(obj, f, indent=1)


def test_config4_accuracy_versus_time_1m():
    import torch
    import bench
    peak = bench.fp32_peak_tflops(1965.0)                 # nominal FP32 peak at the B200's maximum SM clock (bench.py)
    pos, mass, _, eps, _ = inputs.make("plummer_1m")
    n = len(mass)
    tg = inputs.sample_targets(n, 4096, seed=4)
    dacc, _ = direct(pos, mass, eps, targets=tg)          # fp64 direct sum over all N
    rows = []
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        d_acc = torch.empty((n, 3), dtype=torch.float32, device="cuda")
        d_pot = torch.empty(n, dtype=torch.float32, device="cuda")
        for n_leaf in (8, 16, 32):
            with B.TreeCode(n_group=N_GROUP) as tc:
                tc.set_stream(st.cuda_stream)
                tc.set_particles(pos, mass)
                tc.build(n_leaf)
                for theta in (0.3, 0.5, 0.75, 1.0):
                    ts = []
                    for _ in range(4):
                        B.tc_forces(tc.ctx, theta, eps, d_acc, d_pot)
                        tc.sync()
                        ts.append(tc.stats()["t_gpu_ms"])
                    s = tc.stats()
                    e = rel_err(d_acc[torch.from_numpy(tg).cuda()].cpu().numpy().astype(np.float64), dacc)
                    # the paper's device-utilisation picture versus theta (Fig. 8's axes): flop rate of
                    # the evaluation and data rate of the walk alone (option walk_only: one more launch per point)
                    tc.set_option("walk_only", 1)
                    tw = []
                    for _ in range(3):
                        B.tc_forces(tc.ctx, theta, eps, d_acc, d_pot)
                        tc.sync()
                        tw.append(tc.stats()["t_gpu_ms"])
                    sw = tc.stats()
                    tc.set_option("walk_only", 0)
                    ms, wms = float(np.median(ts[1:])), float(np.median(tw[1:]))
                    rows.append(dict(n_leaf=n_leaf, theta=theta, ms=ms,
                                     rms=float(np.sqrt((e ** 2).mean())), median=float(np.median(e)),
                                     p99=float(np.quantile(e, 0.99)), n_pc=s["n_pc_total"] / n, n_pp=s["n_pp_total"] / n,
                                     tflops=(bench.FLOPS_PC * s["n_pc_total"] + bench.FLOPS_PP * s["n_pp_total"]) / (ms * 1e-3) / 1e12,
                                     gflops_paper=(bench.PAPER_FLOPS_PC * s["n_pc_total"] + bench.PAPER_FLOPS_PP * s["n_pp_total"]) / (ms * 1e-3) / 1e9,
                                     walk_ms=wms, tests=sw["n_tests_total"], opened=sw["n_opened_total"],
                                     walk_gbs=16.0 * (sw["n_tests_total"] + sw["n_opened_total"]) / (wms * 1e-3) / 1e9))
                    rows[-1]["frac"] = rows[-1]["tflops"] / peak
    for r in rows:
        print("config4 N_leaf={n_leaf:2d} theta={theta:4.2f}: {ms:7.3f} ms  rms={rms:.3e} median={median:.3e} "
              "p99={p99:.3e}  p-c/particle={n_pc:7.0f} p-p/particle={n_pp:6.0f}  {tflops:5.1f} TFLOP/s = {frac:.3f} of FP32 peak "
              "({gflops_paper:7.0f} GFLOP/s in the paper's 70/38 convention)  walk {walk_ms:6.3f} ms = {walk_gbs:6.1f} GB/s".format(**r))
    _dump("config4_sweep.json", rows)
    for n_leaf in (8, 16, 32):
        rr = [r for r in rows if r["n_leaf"] == n_leaf]
        # error rises steeply with theta (~theta^4), time falls
        assert all(a["rms"] < b["rms"] for a, b in zip(rr, rr[1:]))
        assert all(a["ms"] > b["ms"] for a, b in zip(rr, rr[1:]))
        assert rr[0]["median"] * 4 < rr[1]["median"]                 # 0.3 -> 0.5: at least (5/3)^3
    r05 = [r for r in rows if r["n_leaf"] == 16 and r["theta"] == 0.5][0]
    assert 2e-5 < r05["median"] < 4e-4                               # SURVEY 8(c) sanity band around 8.7e-5


def test_config4_oracle_parity_at_every_sweep_point_1m():
    """Oracle parity at ALL twelve (theta, N_leaf) points of config 4, full size: EVERY particle at N_leaf = 16 (the
    four theta of the headline leaf size), 2048 evenly spaced groups at N_leaf = 8 / 32, plus the paper's own setting
    N_leaf = N_group = 64 at theta = 0.5 on 2048 groups.  Flip audit (R16) at every point."""
    pos, mass, _, eps, _ = inputs.make("plummer_1m")
    rows = []
    for n_leaf, n_group, thetas in ((8, N_GROUP, (0.3, 0.5, 0.75, 1.0)), (16, N_GROUP, (0.3, 0.5, 0.75, 1.0)),
                                    (32, N_GROUP, (0.3, 0.5, 0.75, 1.0)), (64, 64, (0.5,))):
        o = Oracle(pos, mass, n_leaf, n_group)
        gsel = None if n_leaf == 16 else np.unique(np.linspace(0, o.n_groups - 1, 2048).astype(np.int64))
        with B.TreeCode(n_group=n_group) as tc:
            tc.set_particles(pos, mass)
            tc.build(n_leaf)
            for theta in thetas:
                ref = o.forces(theta, eps, shadow32=True, groups=gsel, stats=True)
                acc, pot = tc.forces(theta, eps)
                n_pc, n_pp = tc.counts()
                sel = ref["n_pc"] >= 0
                assert gsel is not None or sel.all()
                rel, prel = check(acc, pot, n_pc, n_pp, ref, sel)
                fl = flip_audit(o, ref, theta, gsel, tag=f"config4 N_leaf={n_leaf} theta={theta}")
                rows.append(dict(n_leaf=n_leaf, n_group=n_group, theta=theta, particles=int(sel.sum()),
                                 groups=int(o.n_groups if gsel is None else len(gsel)), n_groups=int(o.n_groups),
                                 acc_q50=float(np.median(rel)), acc_q999=float(np.quantile(rel, 0.999)), acc_max=float(rel.max()),
                                 pot_max=float(prel.max()), flips=fl))
                print(f"config4 parity N_leaf={n_leaf:2d} N_group={n_group:3d} theta={theta:4.2f}: {int(sel.sum())} particles of "
                      f"{rows[-1]['groups']} / {o.n_groups} groups, acc q99.9={np.quantile(rel, 0.999):.2e} max={rel.max():.2e} "
                      f"pot max={prel.max():.2e} flips={sum(f for _, f, _ in fl)}")
    _dump("config4_parity.json", rows)


def _sampled_parity(tag, pos_host, mass, d_acc, d_pot, n_pc, n_pp, theta, eps, n_leaf, n_group, n_sample, seed):
    """Oracle (own tree on these positions) on n_sample random groups (None: ALL groups, every particle) against the
    library's result; R16 flip audit on the groups walked."""
    o = Oracle(pos_host, mass, n_leaf, n_group)
    gsel = None if n_sample is None else np.sort(np.random.default_rng(seed).choice(o.n_groups, n_sample, replace=False)).astype(np.int64)
    ref = o.forces(theta, eps, shadow32=True, groups=gsel, stats=True)
    shape = (o.n_cells, o.n_leaves, o.n_groups, o.depth)
    sel = ref["n_pc"] >= 0
    assert n_sample is not None or sel.all()            # whole population: the oracle evaluated every particle
    rel, prel = check(d_acc.cpu().numpy(), d_pot.cpu().numpy(), n_pc, n_pp, ref, sel)
    fl = flip_audit(o, ref, theta, gsel, tag=f"config5 {tag}")
    del o
    print(f"config5 {tag}: {int(sel.sum())} particles of {shape[2] if n_sample is None else n_sample} groups, flips={int(ref['flips'].sum())}, "
          f"acc q50={np.median(rel):.2e} q99.9={np.quantile(rel, 0.999):.2e} max={rel.max():.2e} pot max={prel.max():.2e}")
    _dump(f"config5_parity_{tag.replace(' ', '_').replace('(', '').replace(')', '')}.json",
          dict(particles=int(sel.sum()), groups=int(shape[2] if n_sample is None else n_sample), n_groups=int(shape[2]),
               interactions=int(ref["interactions"]), acc_q50=float(np.median(rel)), acc_q999=float(np.quantile(rel, 0.999)),
               acc_max=float(rel.max()), pot_max=float(prel.max()), flips=fl))
    return shape


def test_config5_two_plummer_16m_parity_and_leapfrog():
    """Config 5 at full size: oracle parity at step 0 over EVERY particle (all groups) and on the step-10 positions
     on 4096 sampled groups,
    10 KDK steps with a host tree rebuild each step (the torch harness), then the same 10 steps with the library's own
    device-side leapfrog (`tc_leapfrog`, device tree build) ending in the same state."""
    import torch
    from paper_1005_5384_b200 import integrate
    n, theta, eps, n_leaf, dt, steps, n_group = 1 << 24, 0.5, 0.005, 16, 1.0 / 128, 10, N_GROUP
    pos, mass, vel = inputs.two_plummer(n, with_velocities=True)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st), B.TreeCode(n_group=n_group) as tc:
        tc.set_stream(st.cuda_stream)
        d_pos, d_vel, d_mass = torch.from_numpy(pos).cuda(), torch.from_numpy(vel).cuda(), torch.from_numpy(mass).cuda()
        # ---- parity at step 0 over the whole population (full size, the configuration the loop runs)
        d_acc = torch.empty((n, 3), dtype=torch.float32, device="cuda")
        d_pot = torch.empty(n, dtype=torch.float32, device="cuda")
        tc.set_particles(d_pos, d_mass)
        tc.build(n_leaf)
        B.tc_forces(tc.ctx, theta, eps, d_acc, d_pot)
        tc.sync()
        s0 = tc.stats()
        n_pc, n_pp = tc.counts()
        shape = _sampled_parity("step 0", pos, mass, d_acc, d_pot, n_pc, n_pp, theta, eps, n_leaf, n_group, None, 5)
        assert (s0["n_cells"], s0["n_leaves"], s0["n_groups"], s0["depth"]) == shape
        print(f"config5 step 0: cells={s0['n_cells']} groups={s0['n_groups']} T_host={s0['t_host_ms']:.0f} ms "
              f"T_copy={s0['t_copy_ms']:.1f} ms T_gpu={s0['t_gpu_ms']:.1f} ms interactions={s0['n_pc_total'] + s0['n_pp_total']:.3e}")
        # ---- 10 KDK steps, host tree rebuild each step
        state = {}
        log = integrate.leapfrog_kdk(tc, d_pos, d_vel, d_mass, dt, steps, theta, eps, n_leaf, state=state,
                                     log=lambda r: print("config5 step {step:2d}: T_host={t_host_ms:6.0f} ms T_copy={t_copy_ms:5.1f} ms "
                                                         "T_gpu={t_gpu_ms:6.1f} ms wall={wall_ms:6.0f} ms dE/E={dE_rel:.2e} |dP|={dP:.2e}".format(**r)))
        _dump("config5_leapfrog.json", log)
        assert len(log) == steps + 1
        assert max(r["dE_rel"] for r in log) < 2e-4          # tree-force + leapfrog energy error over 10 steps
        assert max(r["dP"] for r in log) < 1e-4              # total momentum (tree forces are not exactly symmetric)
        # the spheres approach: separation of the two centres of mass shrinks by ~ 0.5 * 10/128
        n1 = (3 * n) // 4
        x1 = float(d_pos[:n1, 0].double().mean()); x2 = float(d_pos[n1:, 0].double().mean())
        assert 6.0 - 0.06 < (x2 - x1) < 6.0 - 0.02
        # ---- parity on the step-10 positions: the loop's last force evaluation against an oracle tree built on them
        pos10 = d_pos.cpu().numpy()
        n_pc, n_pp = tc.counts()
        shape10 = _sampled_parity("step 10", pos10, mass, state["acc"], state["pot"], n_pc, n_pp, theta, eps, n_leaf, n_group, 4096, 6)
        s10 = tc.stats()
        assert (s10["n_cells"], s10["n_leaves"], s10["n_groups"], s10["depth"]) == shape10
        # ---- the same 10 steps with the library's device-side leapfrog (native=True, device tree build)
        d_pos2, d_vel2 = torch.from_numpy(pos).cuda(), torch.from_numpy(vel).cuda()
        tc.set_option("device_build", 1)
        state2 = {}
        log2 = integrate.leapfrog_kdk(tc, d_pos2, d_vel2, d_mass, dt, steps, theta, eps, n_leaf, native=True, state=state2)
        _dump("config5_leapfrog_native.json", log2)
        print("config5 native (tc_leapfrog, device build): " + ", ".join(f"{r['wall_ms']:.0f}" for r in log2[1:]) + " ms per step; "
              f"dE/E max={max(r['dE_rel'] for r in log2):.2e}")
        assert max(r["dE_rel"] for r in log2) < 2e-4 and max(r["dP"] for r in log2) < 1e-4
        # same algorithm, same fp32 arithmetic per step (fma kicks vs torch's mul-add differ by an ulp per step)
        dx = (d_pos2 - d_pos).abs().max().item(); dv = (d_vel2 - d_vel).abs().max().item()
        print(f"config5 native vs torch harness after {steps} steps: max |dx|={dx:.2e} max |dv|={dv:.2e}")
        assert dx < 1e-4 and dv < 1e-4
        n_pc2, n_pp2 = tc.counts()
        _sampled_parity("step 10 (native)", d_pos2.cpu().numpy(), mass, state2["acc"], state2["pot"], n_pc2, n_pp2, theta, eps,
                        n_leaf, n_group, 1024, 7)
