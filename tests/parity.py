"""GPU-vs-oracle acceptance of BASELINE.json north_star, shared by the -m gpu tests and smoke().

Per active row: |acc_gpu - acc_or| / |acc_or| <= 1e-6, |jerk_gpu - jerk_or| / |jerk_or| <= 1e-5 (Euclidean
norms).  Neighbour lists equal as SETS, except pairs with |r_ij - r_s| / r_s < 1e-6 (fp64 r), which may fall
on either side and are reported; rows holding such a pair are force-checked against the oracle re-summed
with the GPU's list.  Overflowed rows (count > cap): counts equal, stored entries are a
subset of the true set of size cap (reading R7).
"""
from __future__ import annotations

import itertools

import numpy as np

TOL_ACC = 1e-6
TOL_JERK = 1e-5
TOL_POT = 1e-6  # the potential is a sum of positive terms like acc's dominant part: same bound
BAND = 1e-6


def relerr(a, b):
    den = np.linalg.norm(b, axis=-1)
    den = np.where(den == 0.0, 1.0, den)
    return np.linalg.norm(a - b, axis=-1) / den


def _rmin(xp, vp, i, j, dt):
    """r_min of eq. (3) for the pairs (i, j): min(|R|, |R + dt V|); dt = 0 gives |R|."""
    R = xp[j] - xp[i]
    d = np.linalg.norm(R, axis=-1)
    if dt != 0.0:
        d = np.minimum(d, np.linalg.norm(R + dt * (vp[j] - vp[i]), axis=-1))
    return d


def _pair_terms(xp, vp, m, i, js):
    """Sum over js of the eq. (9), (10) pair terms and of m / r for particle i (fp64, plain numpy)."""
    R = xp[js] - xp[i]
    V = vp[js] - vp[i]
    r = np.linalg.norm(R, axis=1)
    rv = np.einsum("jc,jc->j", R, V)
    da = (m[js, None] * R / r[:, None] ** 3).sum(axis=0)
    dj = (m[js, None] * (V / r[:, None] ** 3 - 3.0 * rv[:, None] * R / r[:, None] ** 5)).sum(axis=0)
    return da, dj, float((m[js] / r).sum())


def compare(oracle, xp, vp, m, i_idx, r_s, cap, gpu, rows=None, list_stride=None, dtr=None, check_pot=False,
            precomputed=None, strict=True):
    """gpu: dict of numpy arrays acc, jerk, nbr_count, nbr_list, n_overflow (full block).
    rows: optional subset of row numbers to check (oracle runs only on those).
    dtr: per-row regular steps -> velocity criterion eq. (3) (band measured on r_min); check_pot: compare gpu["pot"].
    precomputed: (acc, jerk, count, lists) of oracle.regular_force on exactly these rows (bench.py times that call as
    its cpu_baseline and hands the results in, so the oracle runs once).
    strict=False: rows over the acc / jerk tolerance are counted (rows_over_acc, rows_over_jerk) instead of raising
    (list violations still raise): for measuring how many rows the fp32 path alone would miss.
    Returns a report dict; raises AssertionError on a violation."""
    i_idx = np.asarray(i_idx)
    if rows is None:
        rows = np.arange(i_idx.shape[0])
    rows = np.asarray(rows)
    sub_idx = np.ascontiguousarray(i_idx[rows], dtype=np.int32)
    sub_rs = np.ascontiguousarray(r_s[rows])
    stride = list_stride or max(2 * cap, 64)
    ex = dtr is not None or check_pot
    sub_dt = np.zeros(rows.shape[0]) if dtr is None else np.ascontiguousarray(np.asarray(dtr)[rows], dtype=np.float64)
    if precomputed is not None:
        assert not ex
        acc_o, jerk_o, cnt_o, lists_o = (np.array(precomputed[0]), np.array(precomputed[1]), precomputed[2],
                                         precomputed[3])
    elif ex:
        acc_o, jerk_o, pot_o, cnt_o, lists_o = oracle.regular_force_ex(xp, vp, m, sub_idx, sub_rs,
                                                                       None if dtr is None else sub_dt, list_stride=stride)
    else:
        acc_o, jerk_o, cnt_o, lists_o = oracle.regular_force(xp, vp, m, sub_idx, sub_rs, list_stride=stride)
    acc_g, jerk_g = gpu["acc"][rows].copy(), gpu["jerk"][rows].copy()
    cnt_g = gpu["nbr_count"][rows]
    list_g = gpu["nbr_list"][rows]
    n_band_pairs, worst_band, n_over, n_bestfit = 0, 0.0, 0, 0
    recheck = []  # rows whose list differs only inside the band
    for q in range(rows.shape[0]):
        so = lists_o[q]
        stored = min(int(cnt_g[q]), cap)
        sg = list_g[q, :stored]
        assert np.all(np.diff(sg) > 0), f"row {rows[q]}: GPU list not strictly ascending"
        if cnt_g[q] > cap or cnt_o[q] > cap:
            n_over += 1
        if cnt_g[q] == cnt_o[q] and stored == cnt_o[q] and np.array_equal(sg, so):
            continue
        set_o, set_g = set(so.tolist()), set(sg.tolist())
        if cnt_g[q] > cap:  # overflowed row: only `cap` entries are stored
            diff = set_g - set_o
            extra_needed = int(cnt_g[q]) != int(cnt_o[q])
        else:
            diff = set_g ^ set_o
            extra_needed = True
        if not diff and not extra_needed:
            continue
        # every disagreeing j must sit inside the boundary band
        i = sub_idx[q]
        if cnt_g[q] > cap:
            # Overflowed row: the stored list is cut at cap.  Entries the GPU lists and the oracle sums are named
            # (diff) and must be band pairs; what the count difference leaves unexplained are band pairs that did not
            # make it into the stored list: the best-fitting ones are moved across.  The oracle's sums are adjusted
            # accordingly (H4: a row with a band pair is force-checked with the GPU's own classification).
            d = _rmin(xp, vp, i, np.arange(xp.shape[0]), sub_dt[q])
            in_band = np.abs(d - sub_rs[q]) < BAND * sub_rs[q]
            for j in diff:
                assert in_band[j], f"row {rows[q]} (i={i}): list differs at j={j} outside the band"
            if diff:
                da, dj, dp = _pair_terms(xp, vp, m, i, np.array(sorted(diff)))
                acc_o[q] -= da
                jerk_o[q] -= dj
                if ex:
                    pot_o[q] -= dp
            delta = int(cnt_o[q]) + len(diff) - int(cnt_g[q])  # > 0: the GPU summed `delta` pairs the oracle listed
            n_band_pairs += len(diff) + abs(delta)
            cand = [int(j) for j in np.nonzero(in_band)[0]
                    if j != i and j not in diff and j not in set_g and ((d[j] < sub_rs[q]) == (delta > 0))]
            assert abs(delta) <= len(cand), f"row {rows[q]}: overflow count mismatch"
            best = None
            if delta != 0:
                # The only place where the harness fits something to the output under test: WHICH band pairs of an
                # overflowed row were left out of the stored list cannot be read off the list.  Counted and reported
                # (overflow_bestfit); 0 on configs 1-5.
                n_bestfit += 1
                for combo in itertools.islice(itertools.combinations(cand, abs(delta)), 256):
                    da, dj, dp = _pair_terms(xp, vp, m, i, np.array(combo))
                    sign = 1.0 if delta > 0 else -1.0
                    trial = acc_o[q] + sign * da
                    err = np.linalg.norm(acc_g[q] - trial)
                    if best is None or err < best[0]:
                        best = (err, trial, jerk_o[q] + sign * dj, sign * dp)
            if best is not None:
                acc_o[q], jerk_o[q] = best[1], best[2]
                if ex:
                    pot_o[q] += best[3]
            continue
        for j in diff:
            d = float(_rmin(xp, vp, i, j, sub_dt[q]))
            off = abs(d - sub_rs[q]) / sub_rs[q]
            assert off < BAND, f"row {rows[q]} (i={i}): list differs at j={j}, |r-r_s|/r_s={off:.3e} outside band"
            worst_band = max(worst_band, off)
            n_band_pairs += 1
        if cnt_g[q] <= cap:
            assert int(cnt_g[q]) == len(set_g)
            recheck.append(q)
    if recheck:  # H4: force parity against the oracle re-summed with the GPU's own list
        rq = np.array(recheck)
        a2, j2 = oracle.force_given_lists(xp, vp, m, sub_idx[rq], [list_g[q, : cnt_g[q]] for q in rq])
        acc_o[rq], jerk_o[rq] = a2, j2
        if check_pot:  # the same re-summation for the potential: move the band pairs' m / r across
            for q in recheck:
                i = sub_idx[q]
                so, sg = set(lists_o[q].tolist()), set(list_g[q, : cnt_g[q]].tolist())
                for j in so - sg:  # oracle excluded it, the GPU summed it
                    pot_o[q] += m[j] / np.linalg.norm(xp[j] - xp[i])
                for j in sg - so:
                    pot_o[q] -= m[j] / np.linalg.norm(xp[j] - xp[i])
    ea, ej = relerr(acc_g, acc_o), relerr(jerk_g, jerk_o)
    # rows where everything is a neighbour have acc = jerk = 0 exactly on both sides
    zero = (np.linalg.norm(acc_o, axis=1) == 0)
    if zero.any():
        assert np.all(acc_g[zero] == 0) and np.all(jerk_g[zero] == 0)
    worst_a = int(np.argmax(ea))
    if strict:
        assert ea.max() <= TOL_ACC, f"acc rel err {ea.max():.3e} at row {rows[worst_a]} > {TOL_ACC}"
        assert ej.max() <= TOL_JERK, f"jerk rel err {ej.max():.3e} at row {rows[int(np.argmax(ej))]} > {TOL_JERK}"
    max_pot = 0.0
    if check_pot:
        pot_g = gpu["pot"][rows]
        den = np.where(pot_o == 0.0, 1.0, np.abs(pot_o))
        ep = np.abs(pot_g - pot_o) / den
        if zero.any():
            assert np.all(pot_g[zero] == 0)
        assert ep.max() <= TOL_POT, f"pot rel err {ep.max():.3e} at row {rows[int(np.argmax(ep))]} > {TOL_POT}"
        max_pot = float(ep.max())
    return dict(max_pot_err=max_pot, rows=int(rows.shape[0]), max_acc_err=float(ea.max()), max_jerk_err=float(ej.max()),
                median_acc_err=float(np.median(ea)), band_pairs=int(n_band_pairs), worst_band=float(worst_band),
                overflow_rows=int(n_over), overflow_bestfit=int(n_bestfit), mean_count=float(cnt_o.mean()),
                p999_jerk_err=float(np.quantile(ej, 0.999)) if len(ej) else 0.0,
                rows_over_half_tol=int(((ea > 0.5 * TOL_ACC) | (ej > 0.5 * TOL_JERK)).sum()),
                rows_over_acc=int((ea > TOL_ACC).sum()), rows_over_jerk=int((ej > TOL_JERK).sum()))


def check_overflow_flag(gpu, cap):
    n_over = int((gpu["nbr_count"] > cap).sum())
    assert int(gpu["n_overflow"][0]) == n_over, (int(gpu["n_overflow"][0]), n_over)
    return n_over
