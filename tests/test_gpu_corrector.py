"""Regular corrector of step (vii) and eq. (1) through nb_regular_correct against
oracle/corrector.py (-m gpu).

Acceptance:
 * f1, fd1 (regular force with respect to the OLD list).  The oracle sums eq. (9), (10) over every j outside the old
   list (the plain definition); the GPU adds the list difference to the new-list force.  Its error is that of the
   new-list force (north_star: 1e-6 |acc|, 1e-5 |jerk|) plus that of the fp32 pair terms that do NOT cancel, the
   members of L_new xor L_old, measured against their summed norms as for the irregular force (1e-6).  The common
   members are never evaluated.
 * d2, d3, dx, dv are linear in (f1, fd1): with e_f = |f1_gpu - f1_or|, e_d = |fd1_gpu - fd1_or| of the row,
   |e d2| <= 6 e_f/h^2 + 4 e_d/h, |e d3| <= 12 e_f/h^3 + 6 e_d/h^2, |e dx| <= 0.15 h^2 e_f + h^3 e_d/30,
   |e dv| <= 0.5 h e_f + h^2 e_d/12 (coefficients of f1, fd1 in the formulas of reading R17), plus fp64 rounding.
   With exact inputs and L_old = L_new the whole output is fp64 arithmetic: <= 1e-12 of the term magnitudes.
 * r_s_new: fp64 cbrt, <= 1e-14 relative.
"""
import numpy as np
import pytest
import torch

from oracle import corrector
from paper_1205_1222_b200 import binding, inputs

pytestmark = pytest.mark.gpu


def _t(a, dev, dtype=None):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).to(dev)


def _norm(a):
    return np.linalg.norm(a, axis=1)


def _step_inputs(n_i, k, a_scale, seed):
    """Seeded stand-ins for what the host integrator keeps per particle (no arithmetic of the method)."""
    rng = np.random.default_rng(seed)
    dt = 2.0 ** -rng.integers(3, 9, size=n_i).astype(np.float64)
    fr0 = rng.normal(size=(n_i, 3)) * a_scale
    frd0 = rng.normal(size=(n_i, 3)) * a_scale
    n_p = k * rng.uniform(0.5, 2.0, size=n_i)
    return dt, fr0, frd0, n_p


def _propagated(h, e_f, e_d):
    return dict(d2=6 * e_f / h ** 2 + 4 * e_d / h, d3=12 * e_f / h ** 3 + 6 * e_d / h ** 2,
                dx=0.15 * h ** 2 * e_f + h ** 3 * e_d / 30, dv=0.5 * h * e_f + h ** 2 * e_d / 12)


@pytest.mark.parametrize("config", [1, 2, 4])
def test_full_regular_step_chain(oracle, config):
    """Old list and new list both from nb_regular_force (two radii), then nb_regular_correct, all on the device."""
    wl = inputs.make_workload(config, predict=lambda s: oracle.predict_state(s)[0])
    s = wl.state
    rs_old = wl.r_s * np.random.default_rng(100 + config).uniform(0.8, 1.2, size=wl.n_i)
    ctx = binding.Context(s.n, wl.n_i, wl.cap)
    ctx.set_state(s)
    dev = ctx.workspace.device
    i_idx = _t(wl.i_idx, dev, np.int32)
    old = ctx.nb_regular_force(i_idx, _t(rs_old, dev), s.t)
    new = ctx.nb_regular_force(i_idx, _t(wl.r_s, dev), s.t)
    a_scale = float(np.median(_norm(new["acc"].cpu().numpy())))
    dt, fr0, frd0, n_p = _step_inputs(wl.n_i, wl.k, a_scale, 7 + config)
    out = ctx.nb_regular_correct(i_idx, _t(dt, dev), _t(fr0, dev), _t(frd0, dev), new["acc"], new["jerk"],
                                 new["nbr_count"], new["nbr_list"], old["nbr_count"], old["nbr_list"], s.t,
                                 r_s=_t(wl.r_s, dev), n_p=_t(n_p, dev))
    torch.cuda.synchronize()
    g = {k: v.cpu().numpy() for k, v in out.items()}
    c_old, l_old = old["nbr_count"].cpu().numpy(), old["nbr_list"].cpu().numpy()
    c_new, l_new = new["nbr_count"].cpu().numpy(), new["nbr_list"].cpu().numpy()
    ctx.close()

    # the oracle: plain definition, every j outside the (stored) old list is summed
    xp, vp = oracle.predict_state(s)
    full = (c_old <= wl.cap) & (c_new <= wl.cap)          # rows with a dropped member are outside the contract
    assert full.mean() > 0.9
    rows = np.flatnonzero(full)
    ii = wl.i_idx[rows]
    ref = corrector.regular_corrector(xp, vp, s.m, ii, l_old[rows], c_new[rows], dt[rows], fr0[rows], frd0[rows],
                                      wl.r_s[rows], n_p[rows], old_counts=c_old[rows])
    a_new, j_new = oracle.force_given_lists(xp, vp, s.m, ii, l_new[rows], c_new[rows])
    diff = [np.setxor1d(l_old[q, :c_old[q]], l_new[q, :c_new[q]]).astype(np.int32) for q in rows]
    assert sum(len(d) for d in diff) > len(rows)          # the lists really changed
    _, _, sa, sj = oracle.irregular_force(xp, vp, s.m, ii, diff)
    e_f, e_d = _norm(g["f1"][rows] - ref["f1"]), _norm(g["fd1"][rows] - ref["fd1"])
    assert np.all(e_f <= 1e-6 * _norm(a_new) + 1e-6 * sa), (e_f / (_norm(a_new) + sa)).max()
    assert np.all(e_d <= 1e-5 * _norm(j_new) + 1e-6 * sj), (e_d / (_norm(j_new) + sj)).max()
    # the correction is not a no-op
    assert np.median(_norm(g["f1"][rows] - new["acc"].cpu().numpy()[rows]) / _norm(a_new)) > 1e-5
    h = dt[rows]
    tol = _propagated(h, e_f, e_d)
    for key in ("d2", "d3", "dx", "dv"):
        err = _norm(g[key][rows] - ref[key])
        mag = _propagated(h, _norm(ref["f1"]) + _norm(fr0[rows]), _norm(ref["fd1"]) + _norm(frd0[rows]))[key]
        assert np.all(err <= np.sqrt(3) * tol[key] * (1 + 1e-9) + 1e-13 * mag), key
    # eq. (1), on the rows whose true count the oracle confirms
    _, _, c_or, _ = oracle.regular_force(xp, vp, s.m, ii, wl.r_s[rows], list_stride=wl.cap, want_lists=False)
    same = c_or == c_new[rows]
    assert same.mean() > 0.999
    r_ref = corrector.neighbour_radius_update(wl.r_s[rows], n_p[rows], c_or)
    assert np.abs(g["r_s_new"][rows][same] / r_ref[same] - 1).max() < 1e-14
    print(config, dict(rows=len(rows), f1_err=float((e_f / _norm(ref["f1"])).max()),
                       fd1_err=float((e_d / _norm(ref["fd1"])).max())))


def test_exact_inputs_same_list_is_fp64_arithmetic(oracle):
    """acc, jerk and both lists from the ORACLE, L_old = L_new: every output is then fp64 arithmetic on the GPU."""
    wl = inputs.make_custom(3000, 700, 24, 64, predict=lambda s: oracle.predict_state(s)[0])
    s = wl.state
    xp, vp = oracle.predict_state(s)
    a, j, cnt, lists = oracle.regular_force(xp, vp, s.m, wl.i_idx, wl.r_s, list_stride=64)
    stride = max(1, int(cnt.max()))
    padded = np.full((wl.n_i, stride), -1, dtype=np.int32)
    for q, l in enumerate(lists):
        padded[q, :len(l)] = l
    dt, fr0, frd0, n_p = _step_inputs(wl.n_i, 24, float(np.median(_norm(a))), 3)
    cnt[:3] = 0                                           # rows with an empty list: n_i = 0 in eq. (1) (R18)
    ref = corrector.regular_corrector(xp, vp, s.m, wl.i_idx, padded, cnt, dt, fr0, frd0, wl.r_s, n_p, old_counts=cnt)
    a_in, j_in = oracle.force_given_lists(xp, vp, s.m, wl.i_idx, padded, cnt)
    _, _, sa, sj = oracle.irregular_force(xp, vp, s.m, wl.i_idx, padded, cnt)
    ctx = binding.Context(s.n, wl.n_i, 64)
    ctx.set_state(s)
    dev = ctx.workspace.device
    lst, c = _t(padded, dev), _t(cnt, dev, np.int32)
    out = ctx.nb_regular_correct(_t(wl.i_idx, dev, np.int32), _t(dt, dev), _t(fr0, dev), _t(frd0, dev), _t(a_in, dev),
                                 _t(j_in, dev), c, lst, c, lst, s.t, r_s=_t(wl.r_s, dev), n_p=_t(n_p, dev))
    torch.cuda.synchronize()
    g = {k: v.cpu().numpy() for k, v in out.items()}
    assert np.all(_norm(g["f1"] - ref["f1"]) <= 1e-14 * (sa + _norm(a_in)))
    assert np.all(_norm(g["fd1"] - ref["fd1"]) <= 1e-14 * (sj + _norm(j_in)))
    mags = _propagated(dt, _norm(ref["f1"]) + _norm(fr0) + sa, _norm(ref["fd1"]) + _norm(frd0) + sj)
    for key in ("d2", "d3", "dx", "dv"):
        assert np.all(_norm(g[key] - ref[key]) <= 1e-12 * mags[key]), key
    assert np.abs(g["r_s_new"] / ref["r_s_new"] - 1).max() < 1e-14
    assert np.allclose(g["r_s_new"][:3], wl.r_s[:3] * np.cbrt(n_p[:3]), rtol=1e-14)

    # without r_s / n_p step 3 is skipped; n_i = 0 enqueues nothing; bad arguments are rejected
    out2 = ctx.nb_regular_correct(_t(wl.i_idx, dev, np.int32), _t(dt, dev), _t(fr0, dev), _t(frd0, dev), _t(a_in, dev),
                                  _t(j_in, dev), c, lst, c, lst, s.t)
    torch.cuda.synchronize()
    assert "r_s_new" not in out2 and torch.equal(out2["dx"], out["dx"])
    empty = torch.empty((0, 3), dtype=torch.float64, device=dev)
    e1 = torch.empty(0, dtype=torch.float64, device=dev)
    ei = torch.empty(0, dtype=torch.int32, device=dev)
    ctx.nb_regular_correct(ei, e1, empty, empty, empty, empty, ei, lst[:0], ei, lst[:0], s.t)
    io = binding.CorrectorIO()
    assert ctx.lib.nb_regular_correct(ctx._h, 5, io, float(s.t), None) == -1   # null pointers
    ctx.close()


def test_hermite_on_the_device_reproduces_a_quintic(oracle):
    """Force cubic in time fed through acc/jerk with empty lists: predictor + dx, dv land on the numpy-integrated
    trajectory (the pin of the oracle, applied to the GPU path directly)."""
    from numpy.polynomial import polynomial as P
    rng = np.random.default_rng(4)
    n = 257
    coef = rng.normal(size=(n, 3, 4))
    dt = 2.0 ** -rng.integers(1, 7, size=n).astype(np.float64)
    f1 = np.empty((n, 3)); fd1 = np.empty((n, 3)); x_beyond = np.empty((n, 3)); v_beyond = np.empty((n, 3))
    for q in range(n):
        for c in range(3):
            pf = coef[q, c]
            f1[q, c], fd1[q, c] = P.polyval(dt[q], pf), P.polyval(dt[q], P.polyder(pf))
            hi = np.array([0, 0, pf[2], pf[3]])           # the part of F beyond the predictor's f0 + fd0 tau
            pv = P.polyint(hi)
            v_beyond[q, c], x_beyond[q, c] = P.polyval(dt[q], pv), P.polyval(dt[q], P.polyint(pv))
    wl = inputs.make_custom(512, n, 8, 16, predict=lambda s: oracle.predict_state(s)[0])
    ctx = binding.Context(wl.state.n, n, 16)
    ctx.set_state(wl.state)
    dev = ctx.workspace.device
    zc = torch.zeros(n, dtype=torch.int32, device=dev)
    zl = torch.zeros((n, 16), dtype=torch.int32, device=dev)
    out = ctx.nb_regular_correct(_t(wl.i_idx, dev, np.int32), _t(dt, dev), _t(coef[..., 0], dev), _t(coef[..., 1], dev),
                                 _t(f1, dev), _t(fd1, dev), zc, zl, zc, zl, wl.state.t)
    torch.cuda.synchronize()
    assert np.abs(out["dx"].cpu().numpy() - x_beyond).max() < 1e-13
    assert np.abs(out["dv"].cpu().numpy() - v_beyond).max() < 1e-13
    assert torch.equal(out["f1"].cpu(), torch.from_numpy(f1))
    ctx.close()


def test_unsorted_lists_take_the_general_path(oracle):
    """nb_regular_force writes ascending lists (binary-search membership); any order must give the same result
    (shuffle-scan membership): same fp32 terms, fp64 sums in another order."""
    wl = inputs.make_custom(6000, 900, 40, 128, predict=lambda s: oracle.predict_state(s)[0])
    s = wl.state
    rs_old = wl.r_s * np.random.default_rng(9).uniform(0.8, 1.2, size=wl.n_i)
    ctx = binding.Context(s.n, wl.n_i, 128)
    ctx.set_state(s)
    dev = ctx.workspace.device
    i_idx = _t(wl.i_idx, dev, np.int32)
    old = ctx.nb_regular_force(i_idx, _t(rs_old, dev), s.t)
    new = ctx.nb_regular_force(i_idx, _t(wl.r_s, dev), s.t)
    dt, fr0, frd0, n_p = _step_inputs(wl.n_i, 40, 1.0, 5)
    common = (i_idx, _t(dt, dev), _t(fr0, dev), _t(frd0, dev), new["acc"], new["jerk"])
    ref = ctx.nb_regular_correct(*common, new["nbr_count"], new["nbr_list"], old["nbr_count"], old["nbr_list"], s.t)
    rng = np.random.default_rng(10)
    shuffled = {}
    for name, d in (("old", old), ("new", new)):
        lst, cnt = d["nbr_list"].cpu().numpy().copy(), d["nbr_count"].cpu().numpy()
        assert all(np.all(np.diff(lst[q, :cnt[q]]) > 0) for q in range(wl.n_i))     # ascending as written
        for q in range(wl.n_i):
            lst[q, :cnt[q]] = rng.permutation(lst[q, :cnt[q]])
        shuffled[name] = _t(lst, dev)
    for new_l, old_l in ((shuffled["new"], shuffled["old"]), (new["nbr_list"], shuffled["old"]),
                         (shuffled["new"], old["nbr_list"])):
        got = ctx.nb_regular_correct(*common, new["nbr_count"], new_l, old["nbr_count"], old_l, s.t)
        torch.cuda.synchronize()
        for key in ("f1", "fd1"):
            d = (got[key] - ref[key]).abs().max().item()
            assert d <= 1e-13 * ref[key].abs().max().item(), (key, d)
    assert (ref["f1"] - new["acc"]).abs().max().item() > 1e-6     # lists differ, the correction is not zero
    ctx.close()


def test_small_block_regular_step_runs_without_a_prediction_pass(oracle):
    """N >= 262144, small block: the force call predicts inside force_kernel, the corrector predicts what it gathers
    (corrector_kernel<true>): force + gather + fix-up + corrector = 4 launches per regular step, results identical bit for bit
    to the chain with the predictor pass."""
    wl = inputs.make_custom(300001, 96, 30, 128, seed_sub=4, predict=lambda s: oracle.predict_state(s)[0])
    s = wl.state
    rs_old = wl.r_s * np.random.default_rng(8).uniform(0.8, 1.2, size=wl.n_i)
    ctx = binding.Context(s.n, wl.n_i, wl.cap)
    state_dev = ctx.set_state(s)
    dev = ctx.workspace.device
    i_idx = _t(wl.i_idx, dev, np.int32)
    dt, fr0, frd0, n_p = _step_inputs(wl.n_i, 30, 1.0, 6)
    res = {}
    # both chains on the same launch plan (the fused-prediction kernels hold fewer warps per SM, so the planner may split
    # the j-range differently; the order in which the chunks' fp64 sums are added decides the last bits)
    ctx.nb_set_option("fuse_pred", 0)
    ctx.nb_regular_force(i_idx, _t(wl.r_s, dev), s.t)
    plan = ctx.nb_last_launch_info()
    ctx.nb_set_option("i_block", plan["rows_per_cta"])
    ctx.nb_set_option("j_split", plan["j_chunks"])
    for mode in ("fused", "pass"):
        ctx.nb_set_option("fuse_pred", 1 if mode == "fused" else 0)
        ctx.nb_set_option("irr_pred", 0 if mode == "fused" else 1)
        ctx.nb_set_j(*state_dev)
        old = ctx.nb_regular_force(i_idx, _t(rs_old, dev), s.t)
        ctx.nb_set_j(*state_dev)                      # a new step: no prediction in the context
        new = ctx.nb_regular_force(i_idx, _t(wl.r_s, dev), s.t)
        launches = ctx.nb_last_launch_info()["launches"]
        out = ctx.nb_regular_correct(i_idx, _t(dt, dev), _t(fr0, dev), _t(frd0, dev), new["acc"], new["jerk"],
                                     new["nbr_count"], new["nbr_list"], old["nbr_count"], old["nbr_list"], s.t)
        torch.cuda.synchronize()
        res[mode] = (launches, {k: v.clone() for k, v in out.items()}, new["acc"].clone())
    assert res["fused"][0] == 3 and res["pass"][0] == 4   # force, gather, fp64 fix-up (, predictor pass)
    assert torch.equal(res["fused"][2], res["pass"][2])
    for k in ("f1", "fd1", "d2", "d3", "dx", "dv"):
        assert torch.equal(res["fused"][1][k], res["pass"][1][k]), k
    assert (res["fused"][1]["f1"] - res["fused"][2]).abs().max().item() > 0   # the lists differ
    ctx.close()
