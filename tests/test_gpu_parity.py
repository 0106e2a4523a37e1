"""Parity of the CUDA path with the fp64 oracle on BASELINE.json's five configs -- needs a B200 (-m gpu).

All calls go through the C ABI (include/nbreg.h) via the thin binding.  Tolerances are north_star's:
|acc| 1e-6, |jerk| 1e-5 relative per row, lists bit-exact as sets outside the 1e-6 boundary band
(tests/parity.py).  Inputs are seeded (paper_1205_1222_b200/inputs.py); nothing is read from /root/reference.
"""
import numpy as np
import pytest

from paper_1205_1222_b200 import inputs
import parity
from gpu_util import run_gpu

pytestmark = pytest.mark.gpu


def _pred_pos(oracle):
    return lambda s: oracle.predict_state(s)[0]


def _check_pred(oracle, s, xp_g, vp_g):
    """Predicted state vs oracle: <= 1e-15 relative to the largest Taylor term (Horner/FMA ordering only)."""
    xp_o, vp_o = oracle.predict_state(s)
    dt = (s.t - s.t0)[:, None]
    sx = np.maximum.reduce([np.abs(s.x0), np.abs(s.v0 * dt), np.abs(s.a0 * dt ** 2 / 2), np.abs(s.j0 * dt ** 3 / 6)])
    sv = np.maximum.reduce([np.abs(s.v0), np.abs(s.a0 * dt), np.abs(s.j0 * dt ** 2 / 2)])
    assert np.max(np.abs(xp_g - xp_o) / sx) <= 4e-16
    assert np.max(np.abs(vp_g - vp_o) / sv) <= 4e-16
    return xp_o, vp_o


@pytest.mark.parametrize("config", [1, 2])
def test_configs_1_2_all_rows(oracle, config):
    wl = inputs.make_workload(config, forces=oracle.total_force, predict=_pred_pos(oracle))
    gpu, info, xp_g, vp_g = run_gpu(wl, want_pred=True)
    xp, vp = _check_pred(oracle, wl.state, xp_g, vp_g)
    rep = parity.compare(oracle, xp, vp, wl.state.m, wl.i_idx, wl.r_s, wl.cap, gpu)
    assert parity.check_overflow_flag(gpu, wl.cap) == 0
    assert abs(rep["mean_count"] - wl.k) < 1.0  # r_s calibrated on the predicted positions: k neighbours
    assert np.all(gpu["nbr_list"][np.arange(wl.cap)[None, :] >= gpu["nbr_count"][:, None]] == -7)
    print(config, info, rep)


def test_config3_block_sweep(oracle):
    """N = 65536 Salpeter masses; active-block sizes 32 ... 65536 exercise the j-split path and the gather."""
    st = inputs.make_state(3)
    xp, vp = oracle.predict_state(st)
    full = inputs.make_workload(3, predict=lambda s: xp, state=st)
    saw_split = False
    for n_i in inputs.CONFIG3_BLOCKS:
        wl = inputs.Workload(st, full.i_idx[:n_i].copy(), full.r_s[:n_i].copy(), full.k, full.cap)
        gpu, info = run_gpu(wl)
        rows = None if n_i <= 8192 else np.random.default_rng(n_i).choice(n_i, 8192, replace=False)
        rep = parity.compare(oracle, xp, vp, st.m, wl.i_idx, wl.r_s, wl.cap, gpu, rows=rows)
        parity.check_overflow_flag(gpu, wl.cap)
        saw_split |= info["j_chunks"] > 1
        print(n_i, info, rep)
    assert saw_split  # the direct (one chunk per row) path is config 5's


def test_config4_binaries_and_overflow(oracle):
    """N = 200000 with 10 % hard binaries; 1 % of the rows have r_s doubled so their list overflows cap = 512."""
    wl = inputs.make_workload(4, predict=_pred_pos(oracle))
    gpu, info, xp_g, vp_g = run_gpu(wl, want_pred=True)
    xp, vp = _check_pred(oracle, wl.state, xp_g, vp_g)
    rep = parity.compare(oracle, xp, vp, wl.state.m, wl.i_idx, wl.r_s, wl.cap, gpu, list_stride=2048)
    n_over = parity.check_overflow_flag(gpu, wl.cap)
    assert n_over >= 40 and rep["overflow_rows"] >= n_over
    # a binary member always lists its companion
    nb2 = wl.state.n_binary_members
    for q in np.nonzero(wl.i_idx < nb2)[0][:200]:
        if gpu["nbr_count"][q] <= wl.cap:
            assert (wl.i_idx[q] ^ 1) in gpu["nbr_list"][q, : gpu["nbr_count"][q]]
    print(info, rep)


def test_config5_full_block_sampled(oracle):
    """N = N_i = 1048576 in the launch configuration bench.py times; oracle on a seeded 8192-row subset plus
    whole-block invariants."""
    wl = inputs.make_workload(5, predict=_pred_pos(oracle))
    gpu, info = run_gpu(wl)
    xp, vp = oracle.predict_state(wl.state)
    rows = np.random.default_rng(5).choice(wl.n_i, 8192, replace=False)
    rep = parity.compare(oracle, xp, vp, wl.state.m, wl.i_idx, wl.r_s, wl.cap, gpu, rows=rows)
    parity.check_overflow_flag(gpu, wl.cap)
    cnt = gpu["nbr_count"]
    assert cnt.min() >= wl.k - 1 and cnt.max() <= wl.k + 8  # exactly-k calibration holds over the whole block
    assert np.all(np.isfinite(gpu["acc"])) and np.all(np.isfinite(gpu["jerk"]))
    # whole waves of CTAs run the full j-range unsplit; only the last partial wave of row blocks is j-split
    assert info["split_row_blocks"] * info["rows_per_cta"] < 0.15 * wl.n_i
    print(info, rep)
