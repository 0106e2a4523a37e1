"""ctypes loader for oracle.c -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It never imports the CUDA package and shares no code with it.  See oracle.c for the paper citations.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

_f64p = ctypes.POINTER(ctypes.c_double)
_i32p = ctypes.POINTER(ctypes.c_int32)


def build(force: bool = False) -> str:
    """Compile oracle.c with gcc (fp64, OpenMP, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True, capture_output=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_set_num_threads.argtypes = [ctypes.c_int]
        lib.oracle_predict.argtypes = [ctypes.c_int64, _f64p, _f64p, _f64p, _f64p, _f64p, ctypes.c_double, _f64p, _f64p]
        lib.oracle_regular_force.argtypes = [ctypes.c_int64, _f64p, _f64p, _f64p, ctypes.c_int64, _i32p, _f64p,
                                             _f64p, _f64p, _i32p, _i32p, ctypes.c_int64]
        lib.oracle_force_given_lists.argtypes = [ctypes.c_int64, _f64p, _f64p, _f64p, ctypes.c_int64, _i32p, _i32p,
                                                 _i32p, ctypes.c_int64, _f64p, _f64p]
        lib.oracle_regular_force_ex.argtypes = [ctypes.c_int64, _f64p, _f64p, _f64p, ctypes.c_int64, _i32p, _f64p,
                                                _f64p, _f64p, _f64p, _f64p, _i32p, _i32p, ctypes.c_int64]
        lib.oracle_irregular_force.argtypes = [ctypes.c_int64, _f64p, _f64p, _f64p, ctypes.c_int64, _i32p, _i32p, _i32p,
                                               ctypes.c_int64, _f64p, _f64p, _f64p, _f64p]
        _lib = lib
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(_f64p)


def _pi(a):
    return a.ctypes.data_as(_i32p)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(int(n))


def predict(x0, v0, a0, j0, t0, t):
    """Hermite predictor (PAPER.md:93 step iii; formula from north_star).  Returns xp, vp [n][3]."""
    x0, v0, a0, j0, t0 = map(_d, (x0, v0, a0, j0, t0))
    n = x0.shape[0]
    xp = np.empty((n, 3))
    vp = np.empty((n, 3))
    _load().oracle_predict(n, _p(x0), _p(v0), _p(a0), _p(j0), _p(t0), float(t), _p(xp), _p(vp))
    return xp, vp


def predict_state(state):
    """Convenience for inputs.State -> (xp, vp)."""
    return predict(state.x0, state.v0, state.a0, state.j0, state.t0, state.t)


def regular_force(xp, vp, m, i_idx, r_s, list_stride: int = 256, want_lists: bool = True):
    """eq. (9), (10), (11).  Returns acc[n_i][3], jerk[n_i][3], count[n_i] (true count)
    and lists: a python list of sorted int32 arrays (complete sets: re-runs with a larger stride if needed)."""
    xp, vp, m, r_s = map(_d, (xp, vp, m, r_s))
    i_idx = np.ascontiguousarray(i_idx, dtype=np.int32)
    n, n_i = xp.shape[0], i_idx.shape[0]
    acc = np.empty((n_i, 3))
    jerk = np.empty((n_i, 3))
    count = np.empty(n_i, dtype=np.int32)
    lib = _load()
    if not want_lists:
        lib.oracle_regular_force(n, _p(xp), _p(vp), _p(m), n_i, _pi(i_idx), _p(r_s), _p(acc), _p(jerk), _pi(count),
                                 None, 0)
        return acc, jerk, count, None
    stride = max(1, int(list_stride))
    while True:
        lists = np.empty((n_i, stride), dtype=np.int32)
        lib.oracle_regular_force(n, _p(xp), _p(vp), _p(m), n_i, _pi(i_idx), _p(r_s), _p(acc), _p(jerk), _pi(count),
                                 _pi(lists), stride)
        mx = int(count.max()) if n_i else 0
        if mx <= stride:
            break
        stride = mx
    return acc, jerk, count, [lists[q, : count[q]].copy() for q in range(n_i)]


def regular_force_ex(xp, vp, m, i_idx, r_s, dtr=None, list_stride: int = 256):
    """Variants of Listing B2: velocity criterion eq. (3) with per-row regular step dtr
    (None = plain criterion) and the potential sum.  Returns acc, jerk, pot, count, lists."""
    xp, vp, m, r_s = map(_d, (xp, vp, m, r_s))
    i_idx = np.ascontiguousarray(i_idx, dtype=np.int32)
    n, n_i = xp.shape[0], i_idx.shape[0]
    dtr_p = None
    if dtr is not None:
        dtr = _d(dtr)
        dtr_p = _p(dtr)
    acc = np.empty((n_i, 3))
    jerk = np.empty((n_i, 3))
    pot = np.empty(n_i)
    count = np.empty(n_i, dtype=np.int32)
    stride = max(1, int(list_stride))
    while True:
        lists = np.empty((n_i, stride), dtype=np.int32)
        _load().oracle_regular_force_ex(n, _p(xp), _p(vp), _p(m), n_i, _pi(i_idx), _p(r_s), dtr_p, _p(acc), _p(jerk),
                                        _p(pot), _pi(count), _pi(lists), stride)
        mx = int(count.max()) if n_i else 0
        if mx <= stride:
            break
        stride = mx
    return acc, jerk, pot, count, [lists[q, : count[q]].copy() for q in range(n_i)]


def force_given_lists(xp, vp, m, i_idx, lists, counts=None):
    """Same sums with the neighbour sets given (python list of index arrays, or a padded 2-D array + counts)."""
    xp, vp, m = map(_d, (xp, vp, m))
    i_idx = np.ascontiguousarray(i_idx, dtype=np.int32)
    n, n_i = xp.shape[0], i_idx.shape[0]
    if counts is None:
        counts = np.array([len(l) for l in lists], dtype=np.int32)
        stride = max(1, int(counts.max()) if n_i else 1)
        padded = np.zeros((n_i, stride), dtype=np.int32)
        for q, l in enumerate(lists):
            padded[q, : len(l)] = l
    else:
        padded = np.ascontiguousarray(lists, dtype=np.int32)
        counts = np.ascontiguousarray(counts, dtype=np.int32)
        stride = padded.shape[1]
    acc = np.empty((n_i, 3))
    jerk = np.empty((n_i, 3))
    _load().oracle_force_given_lists(n, _p(xp), _p(vp), _p(m), n_i, _pi(i_idx), _pi(padded), _pi(counts), stride,
                                     _p(acc), _p(jerk))
    return acc, jerk


def irregular_force(xp, vp, m, i_idx, lists, counts=None):
    """eq. (7), (8): force and jerk from the members of the given lists (python list of index
    arrays, or a padded 2-D int32 array + counts).  Returns acc, jerk, acc_scale, jerk_scale (sums of term norms)."""
    xp, vp, m = map(_d, (xp, vp, m))
    i_idx = np.ascontiguousarray(i_idx, dtype=np.int32)
    n, n_i = xp.shape[0], i_idx.shape[0]
    if counts is None:
        counts = np.array([len(l) for l in lists], dtype=np.int32)
        stride = max(1, int(counts.max()) if n_i else 1)
        padded = np.zeros((n_i, stride), dtype=np.int32)
        for q, l in enumerate(lists):
            padded[q, : len(l)] = l
    else:
        padded = np.ascontiguousarray(lists, dtype=np.int32)
        counts = np.ascontiguousarray(counts, dtype=np.int32)
        stride = padded.shape[1]
    acc = np.empty((n_i, 3))
    jerk = np.empty((n_i, 3))
    sa = np.empty(n_i)
    sj = np.empty(n_i)
    _load().oracle_irregular_force(n, _p(xp), _p(vp), _p(m), n_i, _pi(i_idx), _pi(padded), _pi(counts), stride,
                                   _p(acc), _p(jerk), _p(sa), _p(sj))
    return acc, jerk, sa, sj


def total_force(x, v, m):
    """All particles active, r_s = 0: total force and jerk (used as a0, jerk0 "from a first oracle pass",
    BASELINE.json config 1)."""
    n = np.asarray(x).shape[0]
    acc, jerk, _, _ = regular_force(x, v, m, np.arange(n, dtype=np.int32), np.zeros(n), want_lists=False)
    return acc, jerk
