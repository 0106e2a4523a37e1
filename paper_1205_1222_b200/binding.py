"""Thin ctypes binding of include/nbreg.h: argument marshalling only.

Same names as the C ABI (nb_create, nb_set_j, nb_predict_j, nb_regular_force, ...) wrapped in a small
class.  PyTorch supplies device memory and the CUDA stream; every step of the path runs in the CUDA
kernels of libnbreg.so.  There is no CPU fallback: a missing library or device raises.
"""
from __future__ import annotations

import ctypes
import os

import torch

from . import build as _build

NB_OK = 0
_lib = None


class NbregError(RuntimeError):
    pass


def lib_path() -> str:
    return _build.LIB


def load(build_if_missing: bool = True):
    """Load libnbreg.so (building it in-tree with nvcc if it is missing or stale)."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if build_if_missing and _build.stale():
        _build.build()
    if not os.path.exists(path):
        raise NbregError(f"{path} is missing: build it with `python -m paper_1205_1222_b200.build` (no CPU fallback)")
    lib = ctypes.CDLL(path)
    vp, i64, i32, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_double
    lib.nb_version.restype = ctypes.c_int
    lib.nb_strerror.restype = ctypes.c_char_p
    lib.nb_strerror.argtypes = [ctypes.c_int]
    lib.nb_workspace_bytes.restype = ctypes.c_size_t
    lib.nb_workspace_bytes.argtypes = [i64, i64, i32]
    lib.nb_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int, i64, i64, i32, vp, ctypes.c_size_t]
    lib.nb_destroy.argtypes = [vp]
    lib.nb_set_j.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp]
    lib.nb_predict_j.argtypes = [vp, dbl, vp]
    lib.nb_get_predicted.argtypes = [vp, vp, vp, vp]
    lib.nb_regular_force.argtypes = [vp, i32, vp, vp, dbl, vp, vp, vp, vp, vp, vp]
    lib.nb_regular_force_ex.argtypes = [vp, i32, vp, vp, vp, dbl, vp, vp, vp, vp, vp, vp, vp]
    lib.nb_irregular_force.argtypes = [vp, i32, vp, vp, vp, i32, dbl, vp, vp, vp]
    lib.nb_irregular_force_act.argtypes = [vp, i32, vp, vp, vp, i32, dbl, vp, vp, vp]
    lib.nb_regular_correct.argtypes = [vp, i32, ctypes.POINTER(CorrectorIO), dbl, vp]
    lib.nb_regular_force_host.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, i32, vp, vp, dbl, vp, vp, vp, vp, vp]
    lib.nb_regular_force_host_csr.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, i32, vp, vp, dbl, vp, vp, vp, vp, vp, i64, vp]
    lib.nb_set_option.argtypes = [vp, ctypes.c_char_p, i64]
    lib.nb_regular_force_static.argtypes = [ctypes.c_int, i64, vp, vp, vp, vp, vp, vp, i32, vp, vp, dbl, i32, vp, vp, vp, vp,
                                            vp, vp]
    lib.nb_static_limits.argtypes = [ctypes.POINTER(i64)]
    lib.nb_get_error_scale.argtypes = [vp, i32, vp, vp]
    lib.nb_fixup_stats.argtypes = [vp, ctypes.POINTER(i64), vp]
    lib.nb_last_launch_info.argtypes = [vp, ctypes.POINTER(i64)]
    lib.nb_plan.argtypes = [i64, i32, i32, ctypes.POINTER(i32), i64, i64, ctypes.POINTER(i64)]
    _lib = lib
    return lib


class CorrectorIO(ctypes.Structure):
    """nb_corrector_io of include/nbreg.h, field for field."""
    _fields_ = [(k, ctypes.c_void_p) for k in (
        "i_idx", "dt_r", "fr0", "frd0", "acc", "jerk", "nbr_count", "nbr_list", "old_count", "old_list", "r_s", "n_p",
        "f1", "fd1", "d2", "d3", "dx", "dv", "r_s_new")] + [("list_stride", ctypes.c_int32),
                                                             ("old_stride", ctypes.c_int32)]


def _check(rc: int):
    if rc != NB_OK:
        raise NbregError(f"nbreg error {rc}: {load().nb_strerror(rc).decode()}")


def _dev(t: torch.Tensor, dtype, what: str):
    if not t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise NbregError(f"{what}: expected a contiguous CUDA tensor of {dtype}")
    return ctypes.c_void_p(t.data_ptr())


def _host(t: torch.Tensor, dtype, what: str):
    if t.is_cuda or t.dtype != dtype or not t.is_contiguous():
        raise NbregError(f"{what}: expected a contiguous CPU tensor of {dtype}")
    return ctypes.c_void_p(t.data_ptr())


def _stream_ptr(stream):
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


_INFO_KEYS = ("rows_per_cta", "i_per_thread", "j_chunks", "ctas", "split_row_blocks", "launches", "j_tile",
              "ctas_per_sm")


def nb_plan(n: int, n_i: int, num_sms: int = 148, ctas_per_sm=(3, 6, 12, 24, 1), i_block: int = 0,
            j_split: int = 0) -> dict:
    """The launch planner alone (host only).  Same keys as nb_last_launch_info, with chunk_j (particles per j-chunk)
    in place of launches."""
    arr = (ctypes.c_int64 * 8)()
    occ = (ctypes.c_int32 * 5)(*[int(v) for v in ctas_per_sm])
    _check(load().nb_plan(int(n), int(n_i), int(num_sms), occ, int(i_block), int(j_split), arr))
    keys = tuple("chunk_j" if k == "launches" else k for k in _INFO_KEYS)
    return dict(zip(keys, [int(v) for v in arr]))


def nb_static_limits() -> dict:
    """Limits of nb_regular_force_static: n, n_i, nbr_cap, and the bytes of its file-scope device scratch array."""
    arr = (ctypes.c_int64 * 4)()
    _check(load().nb_static_limits(arr))
    return dict(n=int(arr[0]), n_i=int(arr[1]), nbr_cap=int(arr[2]), scratch_bytes=int(arr[3]))


def nb_regular_force_static(x0, v0, a0, j0, m, t0, i_idx, r_s, t: float, out: dict, device: int = 0, stream=None):
    """nb_regular_force_static: the allocation-free call (no context, no workspace; scratch in a fixed device array of the
    library).  All tensors on cuda:`device`; `out` holds acc, jerk, nbr_count, nbr_list [n_i][nbr_cap], n_overflow."""
    f64 = torch.float64
    n, n_i = int(x0.shape[0]), int(i_idx.shape[0])
    cap = int(out["nbr_list"].shape[1]) if out["nbr_list"].dim() == 2 else 1
    _check(load().nb_regular_force_static(
        int(device), n, _dev(x0, f64, "x0"), _dev(v0, f64, "v0"), _dev(a0, f64, "a0"), _dev(j0, f64, "j0"),
        _dev(m, f64, "m"), _dev(t0, f64, "t0"), n_i, _dev(i_idx, torch.int32, "i_idx"), _dev(r_s, f64, "r_s"), float(t),
        cap, _dev(out["acc"], f64, "acc"), _dev(out["jerk"], f64, "jerk"),
        _dev(out["nbr_count"], torch.int32, "nbr_count"), _dev(out["nbr_list"], torch.int32, "nbr_list"),
        _dev(out["n_overflow"], torch.int32, "n_overflow"), _stream_ptr(stream)))
    return out


class Context:
    """nb_ctx with a torch-allocated workspace."""

    def __init__(self, n_max: int, n_i_max: int, nbr_cap: int, device: int = 0):
        if not torch.cuda.is_available():
            raise NbregError("no CUDA device: the regular-force path has no CPU fallback")
        self.lib = load()
        self.n_max, self.n_i_max, self.cap, self.device = int(n_max), int(n_i_max), int(nbr_cap), int(device)
        nbytes = self.lib.nb_workspace_bytes(self.n_max, self.n_i_max, self.cap)
        if nbytes == 0:
            raise NbregError("nb_workspace_bytes: invalid sizes")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=f"cuda:{device}")
        self._h = ctypes.c_void_p()
        _check(self.lib.nb_create(ctypes.byref(self._h), device, self.n_max, self.n_i_max, self.cap,
                                  ctypes.c_void_p(self.workspace.data_ptr()), nbytes))
        self._keep = None
        self.n = 0

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self.lib.nb_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- nb_set_j
    def nb_set_j(self, x0, v0, a0, j0, m, t0):
        f64 = torch.float64
        n = x0.shape[0]
        ptrs = [_dev(t, f64, nm) for t, nm in ((x0, "x0"), (v0, "v0"), (a0, "a0"), (j0, "j0"), (m, "m"), (t0, "t0"))]
        _check(self.lib.nb_set_j(self._h, n, *ptrs))
        self._keep = (x0, v0, a0, j0, m, t0)  # the library keeps the pointers, keep the tensors alive
        self.n = n

    # -- nb_predict_j
    def nb_predict_j(self, t: float, stream=None):
        _check(self.lib.nb_predict_j(self._h, float(t), _stream_ptr(stream)))

    # -- nb_get_predicted
    def nb_get_predicted(self, stream=None):
        xp = torch.empty((self.n, 3), dtype=torch.float64, device=self.workspace.device)
        vp = torch.empty_like(xp)
        _check(self.lib.nb_get_predicted(self._h, ctypes.c_void_p(xp.data_ptr()), ctypes.c_void_p(vp.data_ptr()),
                                         _stream_ptr(stream)))
        return xp, vp

    # -- nb_regular_force
    def alloc_outputs(self, n_i: int):
        dev = self.workspace.device
        return dict(acc=torch.empty((n_i, 3), dtype=torch.float64, device=dev),
                    jerk=torch.empty((n_i, 3), dtype=torch.float64, device=dev),
                    nbr_count=torch.empty(n_i, dtype=torch.int32, device=dev),
                    nbr_list=torch.empty((n_i, self.cap), dtype=torch.int32, device=dev),
                    n_overflow=torch.zeros(1, dtype=torch.int32, device=dev))

    def nb_regular_force(self, i_idx, r_s, t: float, out=None, stream=None):
        n_i = int(i_idx.shape[0])
        if out is None:
            out = self.alloc_outputs(n_i)
        _check(self.lib.nb_regular_force(
            self._h, n_i, _dev(i_idx, torch.int32, "i_idx"), _dev(r_s, torch.float64, "r_s"), float(t),
            _dev(out["acc"], torch.float64, "acc"), _dev(out["jerk"], torch.float64, "jerk"),
            _dev(out["nbr_count"], torch.int32, "nbr_count"), _dev(out["nbr_list"], torch.int32, "nbr_list"),
            _dev(out["n_overflow"], torch.int32, "n_overflow"), _stream_ptr(stream)))
        return out

    # -- nb_regular_force_ex: velocity criterion (dtr) and / or potential output (out["pot"])
    def nb_regular_force_ex(self, i_idx, r_s, t: float, dtr=None, want_pot: bool = False, out=None, stream=None):
        n_i = int(i_idx.shape[0])
        if out is None:
            out = self.alloc_outputs(n_i)
        if want_pot and "pot" not in out:
            out["pot"] = torch.empty(n_i, dtype=torch.float64, device=self.workspace.device)
        null = ctypes.c_void_p()
        _check(self.lib.nb_regular_force_ex(
            self._h, n_i, _dev(i_idx, torch.int32, "i_idx"), _dev(r_s, torch.float64, "r_s"),
            null if dtr is None else _dev(dtr, torch.float64, "dtr"), float(t),
            _dev(out["acc"], torch.float64, "acc"), _dev(out["jerk"], torch.float64, "jerk"),
            _dev(out["pot"], torch.float64, "pot") if want_pot else null,
            _dev(out["nbr_count"], torch.int32, "nbr_count"), _dev(out["nbr_list"], torch.int32, "nbr_list"),
            _dev(out["n_overflow"], torch.int32, "n_overflow"), _stream_ptr(stream)))
        return out

    # -- nb_irregular_force: eq. (7), (8) over given neighbour lists
    def nb_irregular_force(self, i_idx, nbr_count, nbr_list, t: float, out=None, stream=None, act: bool = False):
        n_i = int(i_idx.shape[0])
        dev = self.workspace.device
        if out is None:
            out = dict(acc=torch.empty((n_i, 3), dtype=torch.float64, device=dev),
                       jerk=torch.empty((n_i, 3), dtype=torch.float64, device=dev))
        stride = int(nbr_list.shape[1]) if nbr_list.dim() == 2 else 1
        fn = self.lib.nb_irregular_force_act if act else self.lib.nb_irregular_force
        _check(fn(
            self._h, n_i, _dev(i_idx, torch.int32, "i_idx"), _dev(nbr_count, torch.int32, "nbr_count"),
            _dev(nbr_list, torch.int32, "nbr_list"), stride, float(t),
            _dev(out["acc"], torch.float64, "acc"), _dev(out["jerk"], torch.float64, "jerk"), _stream_ptr(stream)))
        return out

    def nb_irregular_force_act(self, i_idx, nbr_count, nbr_list, t: float, out=None, stream=None):
        """Prediction fused into the gather (PRED_ACT)."""
        return self.nb_irregular_force(i_idx, nbr_count, nbr_list, t, out=out, stream=stream, act=True)

    # -- nb_regular_correct: step (vii) and eq. (1)
    def nb_regular_correct(self, i_idx, dt_r, fr0, frd0, acc, jerk, nbr_count, nbr_list, old_count, old_list, t: float,
                           r_s=None, n_p=None, out=None, stream=None):
        n_i = int(i_idx.shape[0])
        dev = self.workspace.device
        f64 = torch.float64
        if out is None:
            out = {k: torch.empty((n_i, 3), dtype=f64, device=dev) for k in ("f1", "fd1", "d2", "d3", "dx", "dv")}
            if r_s is not None:
                out["r_s_new"] = torch.empty(n_i, dtype=f64, device=dev)
        io = CorrectorIO()
        for key, ten, dt in (("i_idx", i_idx, torch.int32), ("dt_r", dt_r, f64), ("fr0", fr0, f64),
                             ("frd0", frd0, f64), ("acc", acc, f64), ("jerk", jerk, f64),
                             ("nbr_count", nbr_count, torch.int32), ("nbr_list", nbr_list, torch.int32),
                             ("old_count", old_count, torch.int32), ("old_list", old_list, torch.int32),
                             ("r_s", r_s, f64), ("n_p", n_p, f64)) + tuple(
                                 (k, out.get(k), f64) for k in ("f1", "fd1", "d2", "d3", "dx", "dv", "r_s_new")):
            setattr(io, key, None if ten is None else _dev(ten, dt, key))
        io.list_stride = int(nbr_list.shape[1]) if nbr_list.dim() == 2 else 1
        io.old_stride = int(old_list.shape[1]) if old_list.dim() == 2 else 1
        _check(self.lib.nb_regular_correct(self._h, n_i, ctypes.byref(io), float(t), _stream_ptr(stream)))
        return out

    # -- nb_regular_force_host (all tensors on the CPU; pinned memory recommended)
    def nb_regular_force_host(self, x0, v0, a0, j0, m, t0, i_idx, r_s, t: float, out):
        f64 = torch.float64
        n, n_i = int(x0.shape[0]), int(i_idx.shape[0])
        _check(self.lib.nb_regular_force_host(
            self._h, n, _host(x0, f64, "x0"), _host(v0, f64, "v0"), _host(a0, f64, "a0"), _host(j0, f64, "j0"),
            _host(m, f64, "m"), _host(t0, f64, "t0"), n_i, _host(i_idx, torch.int32, "i_idx"),
            _host(r_s, f64, "r_s"), float(t), _host(out["acc"], f64, "acc"), _host(out["jerk"], f64, "jerk"),
            _host(out["nbr_count"], torch.int32, "nbr_count"), _host(out["nbr_list"], torch.int32, "nbr_list"),
            _host(out["n_overflow"], torch.int32, "n_overflow")))
        self.n = n
        return out

    def nb_regular_force_host_csr(self, x0, v0, a0, j0, m, t0, i_idx, r_s, t: float, out):
        """Lists in CSR form: out["nbr_offset"] int64 [n_i + 1], out["nbr_packed"] int32 [capacity] (CPU tensors)."""
        f64 = torch.float64
        n, n_i = int(x0.shape[0]), int(i_idx.shape[0])
        _check(self.lib.nb_regular_force_host_csr(
            self._h, n, _host(x0, f64, "x0"), _host(v0, f64, "v0"), _host(a0, f64, "a0"), _host(j0, f64, "j0"),
            _host(m, f64, "m"), _host(t0, f64, "t0"), n_i, _host(i_idx, torch.int32, "i_idx"),
            _host(r_s, f64, "r_s"), float(t), _host(out["acc"], f64, "acc"), _host(out["jerk"], f64, "jerk"),
            _host(out["nbr_count"], torch.int32, "nbr_count"), _host(out["nbr_offset"], torch.int64, "nbr_offset"),
            _host(out["nbr_packed"], torch.int32, "nbr_packed"), int(out["nbr_packed"].numel()),
            _host(out["n_overflow"], torch.int32, "n_overflow")))
        self.n = n
        return out

    def nb_set_option(self, key: str, value: int):
        _check(self.lib.nb_set_option(self._h, key.encode(), int(value)))

    def nb_get_error_scale(self, n_i: int, stream=None):
        """Test hook: (q_a, q_j) per row of the last force call, float32 [n_i][2]."""
        out = torch.empty((int(n_i), 2), dtype=torch.float32, device=self.workspace.device)
        _check(self.lib.nb_get_error_scale(self._h, int(n_i), ctypes.c_void_p(out.data_ptr()), _stream_ptr(stream)))
        return out

    def nb_fixup_stats(self, stream=None) -> dict:
        """Rows the last force call recomputed in fp64, and since nb_create (synchronises the stream)."""
        arr = (ctypes.c_int64 * 2)()
        _check(self.lib.nb_fixup_stats(self._h, arr, _stream_ptr(stream)))
        return dict(last=int(arr[0]), total=int(arr[1]))

    def nb_last_launch_info(self) -> dict:
        arr = (ctypes.c_int64 * 8)()
        _check(self.lib.nb_last_launch_info(self._h, arr))
        keys = _INFO_KEYS
        return dict(zip(keys, [int(v) for v in arr]))

    # -- convenience: upload a numpy State (inputs.State) and register it
    def set_state(self, state):
        dev = self.workspace.device
        ts = [torch.from_numpy(a).to(dev) for a in (state.x0, state.v0, state.a0, state.j0, state.m, state.t0)]
        self.nb_set_j(*ts)
        return ts
