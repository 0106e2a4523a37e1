"""Parity of the CUDA path with the fp64 oracle on BASELINE.json's five configs -- needs a B200 (-m gpu).

All calls go through the C ABI (include/nbreg.h) via the thin binding.  Tolerances are north_star's:
|acc| 1e-6, |jerk| 1e-5 relative per row, lists bit-exact as sets outside the 1e-6 boundary band
(tests/parity.py).  Inputs are seeded (paper_1205_1222_b200/inputs.py); nothing is read from /root/reference.
"""
import os

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
    assert rep["overflow_bestfit"] == 0
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
        rep = parity.compare(oracle, xp, vp, st.m, wl.i_idx, wl.r_s, wl.cap, gpu)  # EVERY row of every block size
        parity.check_overflow_flag(gpu, wl.cap)
        assert rep["overflow_bestfit"] == 0
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
    assert rep["overflow_bestfit"] == 0
    # a binary member always lists its companion
    nb2 = wl.state.n_binary_members
    for q in np.nonzero(wl.i_idx < nb2)[0][:200]:
        if gpu["nbr_count"][q] <= wl.cap:
            assert (wl.i_idx[q] ^ 1) in gpu["nbr_list"][q, : gpu["nbr_count"][q]]
    print(info, rep)


def _p5_on_gpu_output(oracle, wl, xp, vp, gpu, rows):
    """P5 on the GPU's own output (eq. (7) + (9) = total force, eq. (8) + (10) = total jerk): the
    GPU's regular sums plus the oracle's irregular sums over the GPU's LIST must give the total force of those rows --
    list and force of a row are consistent with each other whatever side of r_s a boundary pair fell on."""
    m = wl.state.m
    idx = np.ascontiguousarray(wl.i_idx[rows], dtype=np.int32)
    a_tot, j_tot, _, _ = oracle.regular_force(xp, vp, m, idx, np.zeros(len(rows)), want_lists=False)
    cnt = np.minimum(gpu["nbr_count"][rows], wl.cap)
    a_irr, j_irr, _, _ = oracle.irregular_force(xp, vp, m, idx, gpu["nbr_list"][rows], cnt)
    full = gpu["nbr_count"][rows] <= wl.cap  # an overflowed row has lost list members
    a_reg, j_reg = a_tot - a_irr, j_tot - j_irr  # what the regular sums must be, given the GPU's list
    ea = parity.relerr(gpu["acc"][rows], a_reg)[full]
    ej = parity.relerr(gpu["jerk"][rows], j_reg)[full]
    assert ea.max() <= parity.TOL_ACC and ej.max() <= parity.TOL_JERK, (ea.max(), ej.max())
    return dict(rows=int(full.sum()), max_acc=float(ea.max()), max_jerk=float(ej.max()))


def test_config5_full_block_sampled(oracle):
    """N = N_i = 1048576 in the launch configuration bench.py times.  SURVEY 8(c): the oracle on a seeded 8192-row subset
    plus every row the GPU flagged as overflowed, P5 on the GPU output for a further 1024 random rows, and whole-block
    invariants.  (Every one of the 1048576 rows: test_config5_every_row below, run on demand.)"""
    wl = inputs.make_workload(5, predict=_pred_pos(oracle))
    gpu, info = run_gpu(wl)
    xp, vp = oracle.predict_state(wl.state)
    rng = np.random.default_rng(5)
    rows = rng.choice(wl.n_i, 8192, replace=False)
    over = np.nonzero(gpu["nbr_count"] > wl.cap)[0]
    rows = np.union1d(rows, over)
    rep = parity.compare(oracle, xp, vp, wl.state.m, wl.i_idx, wl.r_s, wl.cap, gpu, rows=rows, list_stride=2048)
    parity.check_overflow_flag(gpu, wl.cap)
    assert rep["overflow_bestfit"] == 0
    p5 = _p5_on_gpu_output(oracle, wl, xp, vp, gpu, np.setdiff1d(rng.choice(wl.n_i, 1100, replace=False), rows)[:1024])
    cnt = gpu["nbr_count"]
    assert cnt.min() >= wl.k - 1 and cnt.max() <= wl.k + 8  # exactly-k calibration holds over the whole block
    assert np.all(np.isfinite(gpu["acc"])) and np.all(np.isfinite(gpu["jerk"]))
    # whole waves of CTAs run the full j-range unsplit; only the last partial wave of row blocks is j-split
    assert info["split_row_blocks"] * info["rows_per_cta"] < 0.15 * wl.n_i
    # the fp64 fix-up pass took the rows whose sums cancel: a few per 10^4
    assert 0 < info["fixup_rows"] < 0.01 * wl.n_i
    print(info, rep, p5)


@pytest.mark.skipif(os.environ.get("NBREG_FULL_PARITY") != "1",
                    reason="1.1e12 fp64 oracle pairs (~8 min on 16 cores): set NBREG_FULL_PARITY=1; the kept run is "
                           "profiles/r2_full_parity.md")
def test_config5_every_row(oracle):
    """north_star: |acc| <= 1e-6 and |jerk| <= 1e-5 PER PARTICLE.  The oracle on all 1048576 rows of config 5, in chunks;
    lists compared as sets on every row.  Writes gpurun_out/full_parity_c5.json."""
    import json
    import time
    wl = inputs.make_workload(5, predict=_pred_pos(oracle))
    xp, vp = oracle.predict_state(wl.state)
    summary = {}
    for label, opts in (("fixup_on", {}), ("fixup_off", {"fixup": 0})):
        gpu, info = run_gpu(wl, options=opts)
        worst_a = worst_j = 0.0
        band = over_half = n_rows = over_a = over_j = 0
        t0 = time.time()
        for r0 in range(0, wl.n_i, 65536):
            rows = np.arange(r0, min(r0 + 65536, wl.n_i))
            # with the fix-up off a few rows per million are expected to miss the bound: counted, not raised
            rep = parity.compare(oracle, xp, vp, wl.state.m, wl.i_idx, wl.r_s, wl.cap, gpu, rows=rows,
                                 strict=(label == "fixup_on"))
            worst_a, worst_j = max(worst_a, rep["max_acc_err"]), max(worst_j, rep["max_jerk_err"])
            band += rep["band_pairs"]
            over_half += rep["rows_over_half_tol"]
            over_a += rep["rows_over_acc"]
            over_j += rep["rows_over_jerk"]
            n_rows += rep["rows"]
        summary[label] = dict(rows_checked=n_rows, max_acc_err=worst_a, max_jerk_err=worst_j, band_pairs=band,
                              rows_over_acc_tolerance=over_a, rows_over_jerk_tolerance=over_j,
                              rows_over_half_tolerance=over_half, fixup_rows=info["fixup_rows"],
                              oracle_and_compare_seconds=time.time() - t0)
        print(label, summary[label], flush=True)
    os.makedirs("gpurun_out", exist_ok=True)
    json.dump(summary, open("gpurun_out/full_parity_c5.json", "w"), indent=1)
    assert summary["fixup_on"]["rows_checked"] == wl.n_i
    assert summary["fixup_on"]["rows_over_acc_tolerance"] == 0 and summary["fixup_on"]["rows_over_jerk_tolerance"] == 0
