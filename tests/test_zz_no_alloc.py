"""nb_regular_force_static: the entry point that allocates nothing (scratch in a file-scope device array of the library)
-- needs a B200 (-m gpu).  Collected last on purpose (the suite runs with pytest -x).

Checked against the existing path (nb_create + nb_regular_force through binding.Context) on the same seeded inputs, on
two calls in a row that share the scratch array: neighbour counts and lists identical, acc and jerk within the tolerances
every parity test uses (tests/parity.py: 1e-6 / 1e-5; the two paths may split the j-range differently, so the fp64 sums of
the same fp32 terms can differ in their last bits), and against the fp64 oracle as usual.  Sizes beyond the array's fixed
limits are rejected with NB_E_LIMIT before anything is enqueued."""
import ctypes

import numpy as np
import pytest
import torch

from paper_1205_1222_b200 import binding, inputs
import parity
from gpu_util import run_gpu

pytestmark = pytest.mark.gpu


def _static_call(wl, dev):
    s = wl.state
    ts = [torch.from_numpy(a).to(dev) for a in (s.x0, s.v0, s.a0, s.j0, s.m, s.t0)]
    i_idx = torch.from_numpy(np.ascontiguousarray(wl.i_idx, dtype=np.int32)).to(dev)
    r_s = torch.from_numpy(np.ascontiguousarray(wl.r_s, dtype=np.float64)).to(dev)
    out = dict(acc=torch.empty((wl.n_i, 3), dtype=torch.float64, device=dev),
               jerk=torch.empty((wl.n_i, 3), dtype=torch.float64, device=dev),
               nbr_count=torch.empty(wl.n_i, dtype=torch.int32, device=dev),
               nbr_list=torch.full((wl.n_i, wl.cap), -7, dtype=torch.int32, device=dev),
               n_overflow=torch.full((1,), -1, dtype=torch.int32, device=dev))
    binding.nb_regular_force_static(*ts, i_idx, r_s, s.t, out)
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in out.items()}


def _same_as_existing_path(oracle, wl, got):
    ref, _ = run_gpu(wl)  # nb_create + nb_set_j + nb_regular_force
    assert np.array_equal(got["nbr_count"], ref["nbr_count"])
    assert int(got["n_overflow"][0]) == int(ref["n_overflow"][0])
    for q in range(wl.n_i):
        c = min(int(ref["nbr_count"][q]), wl.cap)
        if ref["nbr_count"][q] <= wl.cap:  # (an overflowed j-split row may keep other cap entries, reading R7)
            assert np.array_equal(got["nbr_list"][q, :c], ref["nbr_list"][q, :c]), q
        assert np.all(got["nbr_list"][q, c:] == -7)  # nothing written past the stored entries
    assert parity.relerr(got["acc"], ref["acc"]).max() <= parity.TOL_ACC
    assert parity.relerr(got["jerk"], ref["jerk"]).max() <= parity.TOL_JERK
    xp, vp = oracle.predict_state(wl.state)
    rep = parity.compare(oracle, xp, vp, wl.state.m, wl.i_idx, wl.r_s, wl.cap, got)
    parity.check_overflow_flag(got, wl.cap)
    return rep


def test_static_scratch_entry_point_matches_the_existing_path_twice_in_a_row(oracle):
    dev = torch.device("cuda:0")
    pred = lambda s: oracle.predict_state(s)[0]
    # two different calls back to back on the shared array: a j-split mid-size block with one overflowing row, then a
    # small block of another system (different n, n_i and cap: nothing of the first call may leak into the second)
    wl1 = inputs.make_custom(6001, 700, 20, 64, seed_sub=21, predict=pred)
    wl1.r_s[3] *= 3.0
    wl2 = inputs.make_custom(2500, 45, 12, 32, seed_sub=22, masses="salpeter", predict=pred)
    got1 = _static_call(wl1, dev)
    got2 = _static_call(wl2, dev)
    rep1 = _same_as_existing_path(oracle, wl1, got1)
    rep2 = _same_as_existing_path(oracle, wl2, got2)
    assert int(got1["n_overflow"][0]) >= 1
    # ... and the first workload again, after the second: same bits as its first run (same plan, fixed summation order)
    again = _static_call(wl1, dev)
    for k in ("acc", "jerk", "nbr_count", "n_overflow"):
        assert np.array_equal(again[k], got1[k]), k
    print(rep1, rep2)


def test_static_scratch_entry_point_rejects_sizes_beyond_its_array():
    lib = binding.load()
    lim = binding.nb_static_limits()
    assert lim == dict(n=65536, n_i=4096, nbr_cap=512, scratch_bytes=8 << 20)
    dummy = torch.zeros(64, dtype=torch.float64, device="cuda:0")
    p = ctypes.c_void_p(dummy.data_ptr())
    args = lambda n, n_i, cap: (0, n, p, p, p, p, p, p, n_i, p, p, 1.0, cap, p, p, p, p, p, None)
    for n, n_i, cap in ((lim["n"] + 1, 1, 8), (100, lim["n_i"] + 1, 8), (100, 1, lim["nbr_cap"] + 1)):
        rc = lib.nb_regular_force_static(*args(n, n_i, cap))
        assert rc == -5 and b"nb_regular_force_static" in lib.nb_strerror(rc)
    assert lib.nb_regular_force_static(*args(0, 1, 8)) == -1
    with pytest.raises(binding.NbregError, match="static-scratch"):
        binding._check(lib.nb_regular_force_static(*args(lim["n"] + 1, 1, 8)))
