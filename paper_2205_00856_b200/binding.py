"""Thin ctypes binding of include/cn_nshape.h -- argument marshalling only.

Every step of the path runs in the CUDA kernels of libcn_nshape.so.  There is no CPU fallback and this
module never imports `oracle/`: if the shared library is missing or no CUDA device is present the calls
fail loudly.  PyTorch is used by callers only to hold device memory and streams; this module accepts
torch tensors (their data_ptr), numpy arrays (host pointers) or raw integer addresses.
"""
from __future__ import annotations

import ctypes
import os

PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(PKG, "libcn_nshape.so")

CN_OK, CN_EINVAL, CN_ENOMEM, CN_ECUDA, CN_ENOTFACTORIZED, CN_EBREAKDOWN, CN_ETOOLARGE = range(7)
CN_STATIC_NMAX = 4096
CN_OPT_PATH, CN_OPT_TILE_THREADS, CN_OPT_RS_TOPMAX, CN_OPT_RS_LEVELS, CN_OPT_PROFILE, CN_OPT_PDL, CN_OPT_ONCHIP = 1, 2, 3, 5, 6, 7, 8
CN_OPT_RS_GROUP, CN_OPT_RS_SERIAL_TOP, CN_OPT_RS_TOP_IN_SUBST, CN_OPT_KEEP_P, CN_OPT_BY_COLS = 10, 11, 12, 13, 14
PATH_AUTO, PATH_GENERIC, PATH_TILED, PATH_ONCHIP = 0, 1, 2, 3

EXPORTS = ["cn_plan_create", "cn_plan_set_device_budget", "cn_plan_set_option", "cn_factorize", "cn_step",
           "cn_batched_sweep", "cn_destroy", "cn_plan_get_info", "cn_plan_get_profile", "cn_status_string",
           "cn_last_cuda_error", "cn_version", "cn_plan_set_td_shape", "cn_step_td",
           "cn_tridiag_create", "cn_tridiag_solve", "cn_tridiag_destroy",
           "cn_tridiag_create_blocks", "cn_plan_set_systems", "cn_batched_sweep_v",
           "cn_shard_plan_create", "cn_shard_counts", "cn_shard_factorize_local", "cn_shard_factorize_finish",
           "cn_shard_edge", "cn_shard_prologue", "cn_shard_advance", "cn_shard_epilogue",
           "cn_shard_factorize", "cn_shard_run", "cn_step_static"]

# cn_exchange_fn: cn_status (*)(void *ctx, const void *send, void *recv, int64_t count, void *stream)
EXCHANGE_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64,
                               ctypes.c_void_p)


class CnError(RuntimeError):
    def __init__(self, status: int, where: str, cuda_err: int = 0):
        self.status = status
        self.cuda_err = cuda_err
        msg = lib().cn_status_string(status).decode()
        super().__init__("%s failed: %s%s" % (where, msg, (" [cudaError %d]" % cuda_err) if cuda_err else ""))


class cn_plan_info(ctypes.Structure):
    _fields_ = [("N", ctypes.c_int64), ("P", ctypes.c_int64), ("path", ctypes.c_int32),
                ("tile_threads", ctypes.c_int32), ("tile_points", ctypes.c_int64), ("rs_levels", ctypes.c_int32),
                ("out_of_core", ctypes.c_int32), ("device_bytes", ctypes.c_size_t), ("launches", ctypes.c_int64),
                ("bytes_per_point_step", ctypes.c_double), ("P_effective", ctypes.c_int64)]


_lib = None


def lib():
    """Load libcn_nshape.so (built in-tree by build.py / __graft_entry__.build()).  No fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libcn_nshape.so is missing: run `python -m paper_2205_00856_b200.build` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, i64, dbl, sz, i32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_double, ctypes.c_size_t, ctypes.c_int
        L.cn_plan_create.restype = i32
        L.cn_plan_create.argtypes = [ctypes.POINTER(vp), i64, i64, dbl, dbl, vp]
        L.cn_plan_set_device_budget.restype = i32
        L.cn_plan_set_device_budget.argtypes = [vp, sz]
        L.cn_plan_set_option.restype = i32
        L.cn_plan_set_option.argtypes = [vp, i32, i64]
        L.cn_factorize.restype = i32
        L.cn_factorize.argtypes = [vp, vp]
        L.cn_step.restype = i32
        L.cn_step.argtypes = [vp, vp, i64, vp]
        L.cn_plan_set_td_shape.restype = i32
        L.cn_plan_set_td_shape.argtypes = [vp, vp]
        L.cn_step_td.restype = i32
        L.cn_step_td.argtypes = [vp, vp, i64, vp, vp]
        L.cn_tridiag_create.restype = i32
        L.cn_tridiag_create.argtypes = [ctypes.POINTER(vp), i64, vp, vp, vp, vp]
        L.cn_tridiag_create_blocks.restype = i32
        L.cn_tridiag_create_blocks.argtypes = [ctypes.POINTER(vp), i64, vp, vp, vp, i64, vp, vp]
        L.cn_plan_set_systems.restype = i32
        L.cn_plan_set_systems.argtypes = [vp, i64, i64, i64]
        L.cn_batched_sweep_v.restype = i32
        L.cn_batched_sweep_v.argtypes = [vp, vp, i64, vp]
        L.cn_tridiag_solve.restype = i32
        L.cn_tridiag_solve.argtypes = [vp, vp, vp, vp]
        L.cn_tridiag_destroy.restype = i32
        L.cn_tridiag_destroy.argtypes = [vp]
        L.cn_batched_sweep.restype = i32
        L.cn_batched_sweep.argtypes = [vp, vp, i64, i64, i64, i64, vp]
        L.cn_shard_plan_create.restype = i32
        L.cn_shard_plan_create.argtypes = [ctypes.POINTER(vp), i64, i64, dbl, dbl, vp, ctypes.c_int32, ctypes.c_int32]
        L.cn_shard_counts.restype = i32
        L.cn_shard_counts.argtypes = [vp, ctypes.POINTER(i64), ctypes.POINTER(i64)]
        for name, n in (("cn_shard_factorize_local", 3), ("cn_shard_factorize_finish", 3), ("cn_shard_edge", 4),
                        ("cn_shard_prologue", 5), ("cn_shard_advance", 5), ("cn_shard_epilogue", 4)):
            getattr(L, name).restype = i32
            getattr(L, name).argtypes = [vp] * n
        L.cn_shard_factorize.restype = i32
        L.cn_shard_factorize.argtypes = [vp, EXCHANGE_FN, vp, vp]
        L.cn_shard_run.restype = i32
        L.cn_shard_run.argtypes = [vp, vp, i64, EXCHANGE_FN, vp, vp]
        L.cn_step_static.restype = i32
        L.cn_step_static.argtypes = [i64, dbl, dbl, vp, vp, i64, vp]
        L.cn_destroy.restype = i32
        L.cn_destroy.argtypes = [vp]
        L.cn_plan_get_info.restype = i32
        L.cn_plan_get_info.argtypes = [vp, ctypes.POINTER(cn_plan_info)]
        L.cn_plan_get_profile.restype = i32
        L.cn_plan_get_profile.argtypes = [vp, ctypes.POINTER(dbl)]
        L.cn_status_string.restype = ctypes.c_char_p
        L.cn_status_string.argtypes = [i32]
        L.cn_last_cuda_error.restype = i32
        L.cn_last_cuda_error.argtypes = [vp, ctypes.POINTER(i32)]
        L.cn_version.restype = ctypes.c_char_p
        L.cn_version.argtypes = []
        _lib = L
    return _lib


def _ptr(x) -> int:
    """Address of a torch tensor / numpy array / int."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return int(x.data_ptr())
    if hasattr(x, "ctypes"):
        return int(x.ctypes.data)
    raise TypeError("expected a torch tensor, a numpy array or an integer address, got %r" % type(x))


def _stream(stream) -> int:
    if stream is None:
        import torch
        return int(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return stream
    return int(stream.cuda_stream)


def _check(plan, st: int, where: str):
    if st != CN_OK:
        err = ctypes.c_int(0)
        if plan:
            lib().cn_last_cuda_error(plan, ctypes.byref(err))
        raise CnError(st, where, err.value)


# ---- the C-ABI, same names ------------------------------------------------------------------------------
def cn_plan_create(N: int, P: int, dx: float, dt: float, V):
    """V: N float64 values, numpy (host) or torch CUDA tensor (device); copied by the library."""
    if hasattr(V, "dtype"):
        assert str(V.dtype).endswith("float64"), "V must be float64"
    h = ctypes.c_void_p()
    st = lib().cn_plan_create(ctypes.byref(h), N, P, dx, dt, _ptr(V))
    _check(None, st, "cn_plan_create")
    return h


def cn_plan_set_device_budget(plan, nbytes: int):
    _check(plan, lib().cn_plan_set_device_budget(plan, nbytes), "cn_plan_set_device_budget")


def cn_plan_set_option(plan, key: int, value: int):
    _check(plan, lib().cn_plan_set_option(plan, key, value), "cn_plan_set_option")


def cn_factorize(plan, stream=None):
    _check(plan, lib().cn_factorize(plan, _stream(stream)), "cn_factorize")


def cn_step(plan, psi, nsteps: int = 1, stream=None):
    """psi: N complex128, torch CUDA tensor (or pinned host tensor in out-of-core mode); updated in place."""
    _check(plan, lib().cn_step(plan, _ptr(psi), nsteps, _stream(stream)), "cn_step")


def cn_step_static(N: int, dx: float, dt: float, V, psi, nsteps: int = 1, stream=None):
    """The stepper that allocates nothing (N <= CN_STATIC_NMAX).  V: N float64, psi: N complex128, both torch CUDA
    tensors on the current device; psi updated in place.  Calls that overlap on the GPU race on the library's scratch."""
    assert getattr(V, "is_cuda", False) and getattr(psi, "is_cuda", False), "cn_step_static takes DEVICE pointers"
    _check(None, lib().cn_step_static(N, dx, dt, _ptr(V), _ptr(psi), nsteps, _stream(stream)), "cn_step_static")


def cn_plan_set_td_shape(plan, g):
    _check(plan, lib().cn_plan_set_td_shape(plan, _ptr(g)), "cn_plan_set_td_shape")


def cn_step_td(plan, psi, field, stream=None):
    # field: host float64 array, one value f(t_k + dt/2) per step
    import numpy as np
    f = np.ascontiguousarray(field, dtype=np.float64)
    _check(plan, lib().cn_step_td(plan, _ptr(psi), f.size, f.ctypes.data, _stream(stream)), "cn_step_td")


def cn_batched_sweep(plan, psi, nsys: int, elem_stride: int, sys_stride: int, nsteps: int = 1, stream=None):
    _check(plan, lib().cn_batched_sweep(plan, _ptr(psi), nsys, elem_stride, sys_stride, nsteps, _stream(stream)),
           "cn_batched_sweep")


def cn_plan_set_systems(plan, nsys: int, elem_stride: int, sys_stride: int):
    _check(plan, lib().cn_plan_set_systems(plan, nsys, elem_stride, sys_stride), "cn_plan_set_systems")


def cn_batched_sweep_v(plan, psi, nsteps: int = 1, stream=None):
    _check(plan, lib().cn_batched_sweep_v(plan, _ptr(psi), nsteps, _stream(stream)), "cn_batched_sweep_v")


def cn_destroy(plan):
    _check(None, lib().cn_destroy(plan), "cn_destroy")


def cn_plan_get_info(plan) -> dict:
    info = cn_plan_info()
    _check(plan, lib().cn_plan_get_info(plan, ctypes.byref(info)), "cn_plan_get_info")
    return {k: getattr(info, k) for k, _ in cn_plan_info._fields_}


def cn_plan_get_profile(plan) -> dict:
    out = (ctypes.c_double * 4)()
    _check(plan, lib().cn_plan_get_profile(plan, out), "cn_plan_get_profile")
    return {"pass_ms": out[0], "pass_count": int(out[1]), "rs_ms": out[2], "rs_count": int(out[3])}


def cn_version() -> str:
    return lib().cn_version().decode()


class Tridiag:
    """General complex tridiagonal system (cn_tridiag_*): marshalling only."""

    def __init__(self, b, a, c, stream=None, joints=None):
        """joints: optional caller-placed joint lines (increasing 0-based row indices, the last one N - 1)."""
        n = int(a.shape[0])
        h = ctypes.c_void_p()
        if joints is None:
            st = lib().cn_tridiag_create(ctypes.byref(h), n, _ptr(b), _ptr(a), _ptr(c), _stream(stream))
        else:
            J = (ctypes.c_int64 * len(joints))(*[int(j) for j in joints])
            st = lib().cn_tridiag_create_blocks(ctypes.byref(h), n, _ptr(b), _ptr(a), _ptr(c), len(joints),
                                                ctypes.cast(J, ctypes.c_void_p), _stream(stream))
        if st != CN_OK:
            raise CnError(st, "cn_tridiag_create")
        self.h, self.N = h, n

    def solve(self, d, x=None, stream=None):
        x = d if x is None else x
        st = lib().cn_tridiag_solve(self.h, _ptr(d), _ptr(x), _stream(stream))
        if st != CN_OK:
            raise CnError(st, "cn_tridiag_solve")
        return x

    def close(self):
        if self.h:
            lib().cn_tridiag_destroy(self.h)
            self.h = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class ShardPlan:
    """One shard of a system spread over several processes (cn_shard_*): marshalling only.  The records are device
    tensors owned by the caller; `paper_2205_00856_b200.sharded` holds the protocol that moves them."""

    def __init__(self, N_local, P_local, dx, dt, V_local, shard, nshards, **opts):
        h = ctypes.c_void_p()
        st = lib().cn_shard_plan_create(ctypes.byref(h), N_local, P_local, dx, dt, _ptr(V_local), shard, nshards)
        _check(None, st, "cn_shard_plan_create")
        self.h, self.N, self.shard, self.nshards = h, N_local, shard, nshards
        for k, v in opts.items():
            cn_plan_set_option(self.h, {"rs_topmax": CN_OPT_RS_TOPMAX, "pdl": CN_OPT_PDL, "keep_p": CN_OPT_KEEP_P,
                                        "tile_threads": CN_OPT_TILE_THREADS,
                                        "rs_top_in_subst": CN_OPT_RS_TOP_IN_SUBST}[k], v)

    def counts(self):
        m, s = ctypes.c_int64(0), ctypes.c_int64(0)
        _check(self.h, lib().cn_shard_counts(self.h, ctypes.byref(m), ctypes.byref(s)), "cn_shard_counts")
        return int(m.value), int(s.value)

    def factorize_local(self, matrix_send, stream=None):
        _check(self.h, lib().cn_shard_factorize_local(self.h, _ptr(matrix_send), _stream(stream)), "cn_shard_factorize_local")

    def factorize_finish(self, matrix_all, stream=None):
        _check(self.h, lib().cn_shard_factorize_finish(self.h, _ptr(matrix_all), _stream(stream)), "cn_shard_factorize_finish")

    def edge(self, psi, edge_send, stream=None):
        _check(self.h, lib().cn_shard_edge(self.h, _ptr(psi), _ptr(edge_send), _stream(stream)), "cn_shard_edge")

    def prologue(self, psi, edges_all, step_send, stream=None):
        _check(self.h, lib().cn_shard_prologue(self.h, _ptr(psi), _ptr(edges_all), _ptr(step_send), _stream(stream)),
               "cn_shard_prologue")

    def advance(self, psi, step_all, step_send, stream=None):
        _check(self.h, lib().cn_shard_advance(self.h, _ptr(psi), _ptr(step_all), _ptr(step_send), _stream(stream)),
               "cn_shard_advance")

    def epilogue(self, psi, step_all, stream=None):
        _check(self.h, lib().cn_shard_epilogue(self.h, _ptr(psi), _ptr(step_all), _stream(stream)), "cn_shard_epilogue")

    # the same protocol driven by the library: `exchange` is a Python callable (send_ptr, recv_ptr, count, stream_ptr)
    # that enqueues the all-gather of `count` complex128 values per shard and returns CN_OK
    def _wrap(self, exchange):
        def cb(ctx, send, recv, count, stream):
            try:
                return int(exchange(send, recv, count, stream) or CN_OK)
            except Exception:  # an exception must not unwind through the C frames
                import traceback
                traceback.print_exc()
                return CN_ECUDA
        return EXCHANGE_FN(cb)

    def factorize(self, exchange, stream=None):
        fn = self._wrap(exchange)
        _check(self.h, lib().cn_shard_factorize(self.h, fn, None, _stream(stream)), "cn_shard_factorize")

    def run(self, psi, nsteps, exchange, stream=None):
        fn = self._wrap(exchange)
        _check(self.h, lib().cn_shard_run(self.h, _ptr(psi), nsteps, fn, None, _stream(stream)), "cn_shard_run")

    def info(self):
        return cn_plan_get_info(self.h)

    def close(self):
        if self.h:
            cn_destroy(self.h)
            self.h = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Plan:
    """RAII convenience around the handle; still marshalling only."""

    def __init__(self, N, P, dx, dt, V, path=PATH_AUTO, tile_threads=0, device_budget=0, **opts):
        self.h = cn_plan_create(N, P, dx, dt, V)
        self.N, self.P = N, P
        if path:
            cn_plan_set_option(self.h, CN_OPT_PATH, path)
        if tile_threads:
            cn_plan_set_option(self.h, CN_OPT_TILE_THREADS, tile_threads)
        if device_budget:
            cn_plan_set_device_budget(self.h, device_budget)
        for k, v in opts.items():
            cn_plan_set_option(self.h, {"rs_topmax": CN_OPT_RS_TOPMAX,
                                        "rs_levels": CN_OPT_RS_LEVELS, "profile": CN_OPT_PROFILE,
                                        "pdl": CN_OPT_PDL, "onchip": CN_OPT_ONCHIP, "rs_group": CN_OPT_RS_GROUP,
                                        "rs_serial_top": CN_OPT_RS_SERIAL_TOP, "rs_top_in_subst": CN_OPT_RS_TOP_IN_SUBST, "keep_p": CN_OPT_KEEP_P,
                                        "by_cols": CN_OPT_BY_COLS}[k], v)

    def factorize(self, stream=None):
        cn_factorize(self.h, stream)
        return self

    def step(self, psi, nsteps=1, stream=None):
        cn_step(self.h, psi, nsteps, stream)

    def set_td_shape(self, g):
        cn_plan_set_td_shape(self.h, g)

    def step_td(self, psi, field, stream=None):
        cn_step_td(self.h, psi, field, stream)

    def batched_sweep(self, psi, nsys, elem_stride, sys_stride, nsteps=1, stream=None):
        cn_batched_sweep(self.h, psi, nsys, elem_stride, sys_stride, nsteps, stream)

    def set_systems(self, nsys, elem_stride, sys_stride):
        cn_plan_set_systems(self.h, nsys, elem_stride, sys_stride)
        return self

    def batched_sweep_v(self, psi, nsteps=1, stream=None):
        cn_batched_sweep_v(self.h, psi, nsteps, stream)

    def info(self):
        return cn_plan_get_info(self.h)

    def set_option(self, key, value):
        cn_plan_set_option(self.h, key, value)

    def profile(self):
        return cn_plan_get_profile(self.h)

    def close(self):
        if self.h:
            cn_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()
