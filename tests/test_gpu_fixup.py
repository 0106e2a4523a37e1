"""The fp64 fix-up pass (csrc/fixflag.cuh, csrc/fixup.cuh) -- needs a B200 (-m gpu).

north_star's bound is per particle; the fp32 pair arithmetic misses it on rows whose sums cancel (DESIGN.md section 5.8,
profiles/r2_full_parity.md).  Tested here: (1) the pass itself, forced onto EVERY row, reproduces the fp64 oracle to
rounding on every launch shape and for every queue length (1, 2, 3-4, >= 5 rows take different work mappings); (2) it
never changes a list, a count or the overflow flag; (3) the failure mode it is for -- rows near the cluster centre, where
the regular force cancels -- passes with it and is measurably worse without it; (4) the error-scale estimate the
decision rests on bounds the real error."""
import numpy as np
import pytest
import torch

from paper_1205_1222_b200 import binding, inputs
import parity
from gpu_util import run_gpu

pytestmark = pytest.mark.gpu
ALL_ROWS = {"fixup_ca_milli": 10 ** 12, "fixup_cj_milli": 10 ** 12}  # C so large that every row is queued


def _wl(oracle, n, n_i, k, cap, **kw):
    return inputs.make_custom(n, n_i, k, cap, predict=lambda s: oracle.predict_state(s)[0], **kw)


@pytest.mark.parametrize("n_i", [1, 2, 3, 4, 5, 9, 300])
@pytest.mark.parametrize("opts", [{}, {"i_block": 256, "j_split": 1}, {"i_block": 32, "j_split": 7}])
def test_forced_on_every_row_it_is_the_fp64_sum(oracle, n_i, opts):
    wl = _wl(oracle, 2777, n_i, 16, 48, masses="salpeter")
    wl.r_s[0] *= 3.0  # one overflowing row: its sums must still exclude every neighbour
    xp, vp = oracle.predict_state(wl.state)
    plain, _ = run_gpu(wl, options=dict(opts, fixup=0, ovf_first_in_j=1))
    fixed, info = run_gpu(wl, options=dict(opts, ovf_first_in_j=1, **ALL_ROWS))
    assert info["fixup_rows"] == n_i
    # lists, counts, overflow: untouched
    # (which cap entries an overflowed j-split row keeps may differ between two runs, reading R7: compared with the
    # option that makes them reproducible)
    assert np.array_equal(fixed["nbr_count"], plain["nbr_count"]) and np.array_equal(fixed["nbr_list"], plain["nbr_list"])
    assert np.array_equal(fixed["n_overflow"], plain["n_overflow"])
    # forces: the oracle re-summed with the GPU's own neighbour decisions (counts are the true counts; row 0 overflowed,
    # so take the oracle's full list for it after checking that the counts agree)
    acc_o, jerk_o, cnt_o, lists_o = oracle.regular_force(xp, vp, wl.state.m, wl.i_idx, wl.r_s, list_stride=4096)
    assert np.array_equal(cnt_o, fixed["nbr_count"])  # no band pair in this workload
    ea, ej = parity.relerr(fixed["acc"], acc_o), parity.relerr(fixed["jerk"], jerk_o)
    assert ea.max() < 1e-12 and ej.max() < 1e-11, (ea.max(), ej.max())
    # ... and the fp32 results it replaced were within the fp32 bounds of the same numbers
    assert parity.relerr(plain["acc"], acc_o).max() < 1e-5


def test_forced_with_velocity_criterion_potential_and_fused_prediction(oracle):
    wl = _wl(oracle, 5003, 100, 20, 64)
    xp, vp = oracle.predict_state(wl.state)
    dtr = (wl.state.t - wl.state.t0[wl.i_idx]) * 4.0
    g, info = run_gpu(wl, options=ALL_ROWS, dtr=dtr, want_pot=True)
    assert info["fixup_rows"] == wl.n_i
    a, j, pot, cnt, _ = oracle.regular_force_ex(xp, vp, wl.state.m, wl.i_idx, wl.r_s, dtr)
    assert np.array_equal(cnt, g["nbr_count"])
    assert parity.relerr(g["acc"], a).max() < 1e-12 and parity.relerr(g["jerk"], j).max() < 1e-11
    assert np.max(np.abs(g["pot"] - pot) / pot) < parity.TOL_POT  # the potential stays the fp32 sum
    # the call predicts inside the force kernel: the pass predicts from the registered state as well
    g2, info2 = run_gpu(wl, options=dict(ALL_ROWS, fuse_pred=2))
    a2, j2, cnt2, _ = oracle.regular_force(xp, vp, wl.state.m, wl.i_idx, wl.r_s)
    assert info2["fixup_rows"] == wl.n_i and info2["launches"] == 3  # force, gather, fix-up: no predictor pass
    assert np.array_equal(cnt2, g2["nbr_count"])
    assert parity.relerr(g2["acc"], a2).max() < 1e-12 and parity.relerr(g2["jerk"], j2).max() < 1e-11


@pytest.mark.parametrize("seed", [1, 2, 3, 4])
def test_rows_near_the_cluster_centre(oracle, seed):
    """The failure mode of fp32 pair arithmetic: a particle near the centre of the cluster, where the regular force
    cancels (sum of |terms| 20-200 times |acc|).  Active block = the 512 particles nearest to the centre of mass."""
    full = _wl(oracle, 6000 + 700 * seed, 6000 + 700 * seed, 14, 64, seed_sub=50 + seed, masses="salpeter", active="all")
    xp, vp = oracle.predict_state(full.state)
    centre = (full.state.m[:, None] * xp).sum(axis=0) / full.state.m.sum()
    rows = np.argsort(np.linalg.norm(xp - centre, axis=1))[:512]
    wl = inputs.Workload(full.state, full.i_idx[rows].copy(), full.r_s[rows].copy(), full.k, full.cap)
    acc_o, jerk_o, cnt_o, _ = oracle.regular_force(xp, vp, wl.state.m, wl.i_idx, wl.r_s)
    res = {}
    for label, opts in (("on", {}), ("off", {"fixup": 0})):
        g, info = run_gpu(wl, options=opts)
        ok = g["nbr_count"] == cnt_o  # rows with a band pair are left to tests/parity.py
        res[label] = (parity.relerr(g["acc"], acc_o)[ok], parity.relerr(g["jerk"], jerk_o)[ok], info["fixup_rows"], g)
    ea, ej, n_fix, g = res["on"]
    assert ea.max() <= parity.TOL_ACC and ej.max() <= parity.TOL_JERK, (ea.max(), ej.max())
    parity.compare(oracle, xp, vp, wl.state.m, wl.i_idx, wl.r_s, wl.cap, g)
    assert 0 < n_fix < wl.n_i  # some of these rows need the pass, not all
    # the pass only ever replaces a row by the fp64 sum: nowhere worse than the fp32 path, and its worst row is better
    ea0, ej0, _, _ = res["off"]
    assert ej.max() <= ej0.max() and ea.max() <= ea0.max()
    print(seed, dict(fixup_rows=n_fix, on=(float(ea.max()), float(ej.max())), off=(float(ea0.max()), float(ej0.max()))))


def test_error_scale_bounds_the_error(oracle):
    """nb_get_error_scale: sqrt(q - |s|^2 / T) is the yardstick of a row's fp32 error.  With the pass off, every row's
    error stays below 4e-6 of it (the per-term rounding error is a few 1e-7: a scale 10 x too small would show)."""
    wl = _wl(oracle, 9000, 2000, 24, 96, masses="salpeter")
    xp, vp = oracle.predict_state(wl.state)
    s = wl.state
    ctx = binding.Context(s.n, wl.n_i, wl.cap)
    ctx.nb_set_option("fixup", 0)
    ctx.set_state(s)
    dev = ctx.workspace.device
    out = ctx.nb_regular_force(torch.from_numpy(wl.i_idx.astype(np.int32)).to(dev), torch.from_numpy(wl.r_s).to(dev), s.t)
    torch.cuda.synchronize()
    info = ctx.nb_last_launch_info()
    q = ctx.nb_get_error_scale(wl.n_i).cpu().numpy().astype(np.float64)
    acc_o, jerk_o, cnt_o, _ = oracle.regular_force(xp, vp, s.m, wl.i_idx, wl.r_s)
    ok = out["nbr_count"].cpu().numpy() == cnt_o
    n_pad = (s.n + 255) // 256 * 256
    if info["j_chunks"] > 1:  # equal chunks, a multiple of 4 particles, at least 64 (the planner's rule)
        chunk_j = max(64, -(-(-(-n_pad // info["j_chunks"])) // 4) * 4)
        tiles = info["j_chunks"] * -(-chunk_j // info["j_tile"])
    else:
        tiles = -(-n_pad // info["j_tile"])
    for k, (g, o) in enumerate(((out["acc"], acc_o), (out["jerk"], jerk_o))):
        err = np.linalg.norm(g.cpu().numpy() - o, axis=1)[ok]
        scale = np.sqrt(np.maximum(q[ok, k] - np.sum(o[ok] ** 2, axis=1) / tiles, 0.0))
        big = scale > 0.05 * np.linalg.norm(o[ok], axis=1)  # rows where the spread of the terms matters at all
        assert big.sum() > 50
        ratio = err[big] / scale[big]
        assert ratio.max() < 4e-6 and np.median(ratio) > 2e-8, (ratio.max(), np.median(ratio))
    ctx.close()
