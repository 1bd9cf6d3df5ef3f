"""Thin Python binding of the C ABI in include/tc.h — argument marshalling only.

Same names as the C functions (``tc_create`` ... ``tc_destroy``) plus a small
``TreeCode`` convenience class.  Every step of the hot path runs inside
``libtc_b200.so`` (hand-written CUDA for sm_100a); there is no Python or CPU
fallback: if the library is missing or no CUDA device exists, calls raise.

Arrays may be numpy arrays (host pointers) or torch CUDA tensors (device
pointers, passed as ``data_ptr()``); PyTorch is used for device memory and
streams only.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
#: the in-tree library; TC_B200_LIB points at another build of the same sources (tuning variants)
LIB_PATH = os.environ.get("TC_B200_LIB") or os.path.join(_HERE, "libtc_b200.so")

TC_OK, TC_EINVAL, TC_ESTATE, TC_ECUDA, TC_ENOMEM, TC_EOVERFLOW = 0, -1, -2, -3, -4, -5
TC_FLAG_HOST_ONLY = 1

#: every symbol include/tc.h and include/tc_bench.h declare (checked by tests/test_abi.py)
SYMBOLS = ["tc_create", "tc_create_ex", "tc_destroy", "tc_set_particles", "tc_build", "tc_forces",
           "tc_set_option", "tc_get_counts", "tc_get_stats", "tc_set_stream", "tc_sync",
           "tc_last_error", "tc_get_tree", "tc_get_group_boxes", "tc_leapfrog", "tc_fp32_peak", "tc_direct",
           "tc_shard_size", "tc_forces_shard", "tc_shard_scatter", "tc_direct_static"]

#: most sources / targets tc_direct_static accepts (TC_DIRECT_STATIC_MAX_N of include/tc.h: its 4 MiB static block)
TC_DIRECT_STATIC_MAX_N = 262144


class tc_stats(C.Structure):
    _fields_ = [("n", C.c_int64), ("n_cells", C.c_int64), ("n_leaves", C.c_int64), ("n_groups", C.c_int64),
                ("depth", C.c_int32), ("n_leaf", C.c_int32), ("n_group", C.c_int32), ("reserved", C.c_int32),
                ("n_pc_total", C.c_int64), ("n_pp_total", C.c_int64), ("n_tests_total", C.c_int64),
                ("n_spills", C.c_int64), ("t_host_ms", C.c_double), ("t_copy_ms", C.c_double),
                ("t_gpu_ms", C.c_double), ("tree_bytes", C.c_int64),
                ("t_walk_count_ms", C.c_double), ("t_walk_write_ms", C.c_double), ("t_node_ms", C.c_double),
                ("t_leaf_ms", C.c_double), ("list_bytes", C.c_int64), ("n_opened_total", C.c_int64)]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "reserved"}


class TcError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"tc error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load libtc_b200.so (built by ``paper_1005_5384_b200.build``); fail loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1005_5384_b200.build` "
                          "(there is no Python/CPU fallback for the CUDA path)")
    L = C.CDLL(LIB_PATH)
    vp, i64, i32, f32, f64 = C.c_void_p, C.c_int64, C.c_int, C.c_float, C.c_double
    L.tc_create.restype = vp
    L.tc_create.argtypes = []
    L.tc_create_ex.restype = vp
    L.tc_create_ex.argtypes = [C.c_uint32]
    L.tc_destroy.restype = None
    L.tc_destroy.argtypes = [vp]
    L.tc_set_particles.argtypes = [vp, vp, vp, i64]
    L.tc_build.argtypes = [vp, i32]
    L.tc_forces.argtypes = [vp, f32, f32, vp, vp]
    L.tc_set_option.argtypes = [vp, C.c_char_p, f64]
    L.tc_get_counts.argtypes = [vp, vp, vp]
    L.tc_get_stats.argtypes = [vp, C.POINTER(tc_stats)]
    L.tc_set_stream.argtypes = [vp, vp]
    L.tc_sync.argtypes = [vp]
    L.tc_last_error.restype = C.c_char_p
    L.tc_last_error.argtypes = [vp]
    L.tc_get_tree.argtypes = [vp] + [vp] * 6
    L.tc_get_group_boxes.argtypes = [vp, vp]
    L.tc_leapfrog.argtypes = [vp, vp, vp, vp, i64, f32, i32, i32, f32, f32, vp, vp, i32]
    L.tc_fp32_peak.argtypes = [vp, C.POINTER(C.c_double)]
    L.tc_direct.argtypes = [vp, f32, vp, i64, vp, vp]
    L.tc_shard_size.argtypes = [vp, C.POINTER(C.c_int64)]
    L.tc_forces_shard.argtypes = [vp, f32, f32, vp, vp]
    L.tc_shard_scatter.argtypes = [vp, vp, vp, vp, vp, vp, vp]
    L.tc_direct_static.argtypes = [vp, vp, i64, f32, vp, i64, vp, vp, vp]
    _lib = L
    return L


def _ptr(a, dtype=None, shape=None, name="buffer"):
    """Raw pointer of a numpy array (host) or a torch tensor (host or device); None -> NULL.

    `dtype` (numpy dtype) and `shape` (tuple, None = any extent) are CHECKED before the C call: the library sees
    plain pointers and would reinterpret a float64 array, or a [3,n] one, byte by byte."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        if not a.flags["C_CONTIGUOUS"]:
            raise TypeError(f"{name}: array must be C-contiguous")
        got, p = a.dtype, C.c_void_p(a.ctypes.data)
    elif hasattr(a, "data_ptr"):
        if not a.is_contiguous():
            raise TypeError(f"{name}: tensor must be contiguous")
        got, p = np.dtype(str(a.dtype).replace("torch.", "")), C.c_void_p(a.data_ptr())
    else:
        raise TypeError(f"{name}: unsupported buffer type {type(a)}")
    if dtype is not None and got != np.dtype(dtype):
        raise TypeError(f"{name}: dtype must be {np.dtype(dtype)}, got {got}")
    if shape is not None:
        sh = tuple(a.shape)
        if len(sh) != len(shape) or any(w is not None and int(w) != int(g) for w, g in zip(shape, sh)):
            raise TypeError(f"{name}: shape must be {tuple('n' if w is None else w for w in shape)}, got {sh}")
    return p


def _check(ctx, rc):
    if rc != TC_OK:
        raise TcError(rc, lib().tc_last_error(ctx).decode())


# ---- the C functions, one to one ------------------------------------------------
def tc_create(flags: int = 0):
    ctx = lib().tc_create_ex(flags)
    if not ctx:
        raise TcError(TC_ECUDA, lib().tc_last_error(None).decode())
    return ctx


def tc_destroy(ctx):
    lib().tc_destroy(ctx)


def tc_set_particles(ctx, pos, mass, n=None):
    n = int(pos.shape[0]) if n is None else int(n)
    _check(ctx, lib().tc_set_particles(ctx, _ptr(pos, np.float32, (None, 3), "pos"), _ptr(mass, np.float32, (pos.shape[0],), "mass"), n))


def tc_build(ctx, n_leaf: int):
    _check(ctx, lib().tc_build(ctx, int(n_leaf)))


def tc_forces(ctx, theta: float, eps: float, acc, pot=None):
    _check(ctx, lib().tc_forces(ctx, float(theta), float(eps), _ptr(acc, np.float32, (None, 3), "acc"),
                                _ptr(pot, np.float32, (acc.shape[0],), "pot")))


def tc_set_option(ctx, key: str, value: float):
    _check(ctx, lib().tc_set_option(ctx, key.encode(), float(value)))


def tc_get_counts(ctx, n: int | None = None):
    n = tc_get_stats(ctx)["n"]          # the library writes one entry per particle of the built tree
    n_pc = np.zeros(n, np.int32)
    n_pp = np.zeros(n, np.int32)
    _check(ctx, lib().tc_get_counts(ctx, _ptr(n_pc), _ptr(n_pp)))
    return n_pc, n_pp


def tc_get_stats(ctx) -> dict:
    s = tc_stats()
    _check(ctx, lib().tc_get_stats(ctx, C.byref(s)))
    return s.asdict()


def tc_set_stream(ctx, cuda_stream: int):
    _check(ctx, lib().tc_set_stream(ctx, C.c_void_p(cuda_stream)))


#: cudaStreamLegacy of cuda_runtime_api.h: the handle that NAMES the legacy default stream.  The raw handle of that
#: stream is 0, which tc_set_stream reads as "the context's own (non-blocking) stream" — not ordered with it at all.
CUDA_STREAM_LEGACY = 0x1


def torch_stream_handle(device=None) -> int:
    """Handle of torch's CURRENT stream on `device` in the form tc_set_stream needs: torch's default stream is the
    legacy default stream (handle 0) and is passed as cudaStreamLegacy, any other stream as itself."""
    import torch
    h = int(torch.cuda.current_stream(device).cuda_stream)
    return h if h != 0 else CUDA_STREAM_LEGACY


def tc_sync(ctx):
    _check(ctx, lib().tc_sync(ctx))


def tc_get_tree(ctx) -> dict:
    s = tc_get_stats(ctx)
    n, nc, ng = s["n"], s["n_cells"], s["n_groups"]
    out = dict(perm=np.zeros(n, np.int32), bnd=np.zeros((nc, 4), np.float32), xm=np.zeros((nc, 4), np.float32),
               q=np.zeros((nc, 6), np.float32), link=np.zeros((nc, 4), np.int32), groups=np.zeros(ng, np.int32))
    _check(ctx, lib().tc_get_tree(ctx, *[_ptr(out[k]) for k in ("perm", "bnd", "xm", "q", "link", "groups")]))
    return out


def tc_get_group_boxes(ctx) -> np.ndarray:
    """fp32 half extents [n_groups,3] of every group's tight box (variant R23), groups in Morton order."""
    out = np.zeros((tc_get_stats(ctx)["n_groups"], 3), np.float32)
    _check(ctx, lib().tc_get_group_boxes(ctx, _ptr(out)))
    return out


def tc_leapfrog(ctx, pos, vel, mass, dt: float, steps: int, n_leaf: int, theta: float, eps: float, acc, pot=None,
                have_acc: bool = False):
    """`steps` KDK steps on the device; pos, vel, mass, acc, pot are torch CUDA tensors updated in place."""
    n = int(mass.shape[0])
    _check(ctx, lib().tc_leapfrog(ctx, _ptr(pos, np.float32, (n, 3), "pos"), _ptr(vel, np.float32, (n, 3), "vel"),
                                  _ptr(mass, np.float32, (n,), "mass"), n, float(dt), int(steps), int(n_leaf), float(theta),
                                  float(eps), _ptr(acc, np.float32, (n, 3), "acc"), _ptr(pot, np.float32, (n,), "pot"),
                                  int(bool(have_acc))))


def tc_direct(ctx, eps: float, targets, acc, pot=None):
    """Direct summation for `targets` (host int64 array or None = all particles) into fp64 acc / pot."""
    nt = 0 if targets is None else int(len(targets))
    if targets is not None:
        assert isinstance(targets, np.ndarray) and targets.dtype == np.int64, "targets must be a host int64 array"
    _check(ctx, lib().tc_direct(ctx, float(eps), _ptr(targets, np.int64, (nt,), "targets"), nt, _ptr(acc, np.float64, (None, 3), "acc"),
                                _ptr(pot, np.float64, (acc.shape[0],), "pot")))


def tc_direct_static(pos, mass, eps: float, targets, acc, pot=None, cuda_stream: int = 0):
    """Direct summation for callers that may not allocate device memory (a plugin inside an application whose pool
    owns the GPU, a latency-critical step that must stay clear of the allocator's lock, a full device): no context,
    no cudaMalloc — the packed sources live in a 4 MiB block inside the library, one per GPU, shared by all callers.

    Every array is a torch CUDA tensor of the caller: pos [n,3] / mass [n] float32, targets int64 [n_t] or None (all),
    acc [n_t,3] / pot [n_t] float64 outputs.  Work is queued on `cuda_stream` (0 = legacy default stream), nothing is
    synchronised.  n, n_t <= TC_DIRECT_STATIC_MAX_N or TcError(TC_EINVAL).  Calls that overlap on the GPU race on
    the shared block; make the first call per device outside stream capture (include/tc.h has the full contract)."""
    n = int(mass.shape[0])
    nt = 0 if targets is None else int(targets.shape[0])
    rc = lib().tc_direct_static(_ptr(pos, np.float32, (n, 3), "pos"), _ptr(mass, np.float32, (n,), "mass"), n, float(eps),
                                _ptr(targets, np.int64, (nt,), "targets"), nt, _ptr(acc, np.float64, (None, 3), "acc"),
                                _ptr(pot, np.float64, (acc.shape[0],), "pot"), C.c_void_p(cuda_stream))
    _check(None, rc)


def tc_shard_size(ctx) -> int:
    """Rows every rank contributes to the all-gather of a sharded evaluation (options shard_count / shard_rank)."""
    v = C.c_int64(0)
    _check(ctx, lib().tc_shard_size(ctx, C.byref(v)))
    return int(v.value)


def tc_forces_shard(ctx, theta: float, eps: float, out4, cnt2=None):
    """This rank's shard into compact DEVICE rows out4 [n_slots,4] (+ cnt2 [n_slots,2] int32)."""
    _check(ctx, lib().tc_forces_shard(ctx, float(theta), float(eps), _ptr(out4, np.float32, (None, 4), "out4"),
                                      _ptr(cnt2, np.int32, (out4.shape[0], 2), "cnt2")))


def tc_shard_scatter(ctx, gathered4, gathered_cnt2, acc, pot=None, n_pc=None, n_pp=None):
    """All-gathered rows [k,n_slots,4] (+ counts) -> acc / pot / counts in the caller's order (DEVICE tensors)."""
    n = int(acc.shape[0])
    _check(ctx, lib().tc_shard_scatter(ctx, _ptr(gathered4, np.float32, (None, None, 4), "gathered4"),
                                       _ptr(gathered_cnt2, np.int32, tuple(gathered4.shape[:2]) + (2,), "gathered_cnt2"),
                                       _ptr(acc, np.float32, (n, 3), "acc"), _ptr(pot, np.float32, (n,), "pot"),
                                       _ptr(n_pc, np.int32, (n,), "n_pc"), _ptr(n_pp, np.int32, (n,), "n_pp")))


def tc_fp32_peak(ctx) -> float:
    """Measured FFMA-only FP32 throughput of the current device in TFLOP/s."""
    v = C.c_double(0.0)
    _check(ctx, lib().tc_fp32_peak(ctx, C.byref(v)))
    return float(v.value)


class TreeCode:
    """Context manager around one tc_ctx (marshalling only)."""

    def __init__(self, host_only: bool = False, n_group: int | None = None):
        self.ctx = tc_create(TC_FLAG_HOST_ONLY if host_only else 0)
        self.n = 0
        if n_group is not None:
            self.set_option("n_group", n_group)

    def close(self):
        if self.ctx:
            tc_destroy(self.ctx)
            self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, key, value):
        tc_set_option(self.ctx, key, value)

    def set_particles(self, pos, mass):
        self.n = int(pos.shape[0])
        tc_set_particles(self.ctx, pos, mass, self.n)

    def build(self, n_leaf: int = 16):
        tc_build(self.ctx, n_leaf)

    def forces(self, theta, eps, acc=None, pot=None):
        """Host path: allocates numpy outputs if none are given and returns (acc, pot)."""
        if acc is None:
            acc = np.empty((self.n, 3), np.float32)
            pot = np.empty(self.n, np.float32)
        tc_forces(self.ctx, theta, eps, acc, pot)
        return acc, pot

    def direct(self, eps, targets=None):
        """Host path of tc_direct: returns (acc fp64 [n_t,3], pot fp64 [n_t])."""
        nt = self.n if targets is None else len(targets)
        acc = np.empty((nt, 3), np.float64)
        pot = np.empty(nt, np.float64)
        t = None if targets is None else np.ascontiguousarray(targets, dtype=np.int64)
        tc_direct(self.ctx, eps, t, acc, pot)
        return acc, pot

    def counts(self):
        return tc_get_counts(self.ctx)

    # one evaluation over k GPUs (include/tc.h, "ONE force evaluation over k GPUs"): this context is one rank
    def shard_size(self) -> int:
        return tc_shard_size(self.ctx)

    def forces_shard(self, theta, eps, out4, cnt2=None):
        tc_forces_shard(self.ctx, theta, eps, out4, cnt2)

    def shard_scatter(self, gathered4, gathered_cnt2, acc, pot=None, n_pc=None, n_pp=None):
        tc_shard_scatter(self.ctx, gathered4, gathered_cnt2, acc, pot, n_pc, n_pp)

    def stats(self):
        return tc_get_stats(self.ctx)

    def tree(self):
        return tc_get_tree(self.ctx)

    def sync(self):
        tc_sync(self.ctx)

    def set_stream(self, s):
        tc_set_stream(self.ctx, s)

    def use_torch_stream(self, device=None):
        """Queue the context's work on torch's current stream (default stream included): torch ops before and after a
        call with device pointers are then ordered with it."""
        tc_set_stream(self.ctx, torch_stream_handle(device))
