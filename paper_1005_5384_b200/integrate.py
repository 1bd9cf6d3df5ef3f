"""Config-5 harness: leapfrog KDK time integration around the force library.

The paper keeps time integration on the host and only mentions it; BASELINE.json
config 5 prescribes 10 kick-drift-kick steps with a host tree rebuild each step.  This module is
harness code, not part of the hot path: positions / velocities live in torch device tensors and every
force evaluation is one ``tc_set_particles`` + ``tc_build`` + ``tc_forces`` through the C ABI (device
pointers).  The kicks and the drift are either plain elementwise torch ops (default) or, with
``native=True``, the library's own ``tc_leapfrog`` (device-side KDK), called one step at a
time so that the energy can be logged between steps.
"""
from __future__ import annotations

import time

import torch

from . import binding as B


def energy(mass, vel, pot):
    """(kinetic, potential, total) in fp64; potential energy = 1/2 sum m_i phi_i (G = 1)."""
    m = mass.double()
    ke = 0.5 * (m * (vel.double() ** 2).sum(1)).sum()
    pe = 0.5 * (m * pot.double()).sum()
    return float(ke), float(pe), float(ke + pe)


def leapfrog_kdk(tc: "B.TreeCode", pos, vel, mass, dt: float, steps: int, theta: float, eps: float,
                 n_leaf: int = 16, log=None, native: bool = False, state: dict | None = None):
    """Advance (pos, vel) in place by `steps` KDK steps; returns a list of per-step dicts.

    v += a dt/2 ; x += v dt ; rebuild tree ; a = forces(x) ; v += a dt/2     (BASELINE.json config 5)
    Each entry: step, t_host_ms, t_copy_ms, t_gpu_ms (PAPER.md:155,165 split), wall_ms, E, dE_rel, |sum m v|.
    `state`, if given, receives the accelerations and potentials of the last force evaluation (`acc`, `pot`).
    The library works on its own stream: it is pointed at torch's current stream here, so that the torch
    kicks / drift and the library's reads of `pos` are ordered (tc.h: device pointers are stream-ordered).
    Torch's default stream has the raw handle 0, which tc_set_stream takes as "the context's own stream":
    `use_torch_stream` passes it as cudaStreamLegacy instead.
    """
    tc.use_torch_stream(pos.device)
    n = pos.shape[0]
    dev = pos.device
    acc = torch.empty((n, 3), dtype=torch.float32, device=dev)
    pot = torch.empty(n, dtype=torch.float32, device=dev)
    if state is not None:
        state["acc"], state["pot"] = acc, pot

    def force():
        tc.set_particles(pos, mass)
        tc.build(n_leaf)
        B.tc_forces(tc.ctx, theta, eps, acc, pot)
        tc.sync()
        return tc.stats()

    st = force()
    e0 = energy(mass, vel, pot)[2]
    p0 = (mass.double()[:, None] * vel.double()).sum(0)
    out = [dict(step=0, t_host_ms=st["t_host_ms"], t_copy_ms=st["t_copy_ms"], t_gpu_ms=st["t_gpu_ms"], wall_ms=0.0,
                E=e0, dE_rel=0.0, dP=0.0, interactions=st["n_pc_total"] + st["n_pp_total"])]
    for k in range(1, steps + 1):
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        if native:
            B.tc_leapfrog(tc.ctx, pos, vel, mass, dt, 1, n_leaf, theta, eps, acc, pot, have_acc=True)
            tc.sync()
            st = tc.stats()
        else:
            vel.add_(acc, alpha=0.5 * dt)
            pos.add_(vel, alpha=dt)
            st = force()
            vel.add_(acc, alpha=0.5 * dt)
        torch.cuda.synchronize(dev)
        wall = (time.perf_counter() - t0) * 1e3
        e = energy(mass, vel, pot)[2]
        dp = float(((mass.double()[:, None] * vel.double()).sum(0) - p0).norm())
        rec = dict(step=k, t_host_ms=st["t_host_ms"], t_copy_ms=st["t_copy_ms"], t_gpu_ms=st["t_gpu_ms"], wall_ms=wall,
                   E=e, dE_rel=abs((e - e0) / e0), dP=dp, interactions=st["n_pc_total"] + st["n_pp_total"])
        out.append(rec)
        if log:
            log(rec)
    return out
