"""Second, independent statement of the oracle in numpy -- TEST INFRASTRUCTURE, tiny N only.

Guards oracle.c (pin P10): vectorised over j, python loop over rows.  Written from the equations, not
from oracle.c: eq. (9)-(11) at PAPER.md:102-108, criterion eq. (2) at PAPER.md:65-67, predictor per
north_star (PAPER.md:93 names the step).  Shares no code with the CUDA path.
"""
from __future__ import annotations

import numpy as np


def predict(x0, v0, a0, j0, t0, t):
    dt = (t - np.asarray(t0, dtype=np.float64))[:, None]
    xp = x0 + v0 * dt + a0 * dt ** 2 / 2.0 + j0 * dt ** 3 / 6.0
    vp = v0 + a0 * dt + j0 * dt ** 2 / 2.0
    return xp, vp


def regular_force(xp, vp, m, i_idx, r_s):
    xp = np.asarray(xp, dtype=np.float64)
    vp = np.asarray(vp, dtype=np.float64)
    m = np.asarray(m, dtype=np.float64)
    n_i = len(i_idx)
    acc = np.zeros((n_i, 3))
    jerk = np.zeros((n_i, 3))
    lists = []
    for q, (i, h) in enumerate(zip(i_idx, r_s)):
        R = xp - xp[i]
        V = vp - vp[i]
        r2 = np.einsum("jc,jc->j", R, R)
        other = np.arange(xp.shape[0]) != i
        nb = other & (r2 < h * h)
        summed = other & ~nb & (r2 > 0.0)
        Rs, Vs, r2s, ms = R[summed], V[summed], r2[summed], m[summed]
        r = np.sqrt(r2s)
        rv = np.einsum("jc,jc->j", Rs, Vs)
        acc[q] = (ms[:, None] * Rs / r[:, None] ** 3).sum(axis=0)
        jerk[q] = (ms[:, None] * (Vs / r[:, None] ** 3 - 3.0 * rv[:, None] * Rs / r[:, None] ** 5)).sum(axis=0)
        lists.append(np.nonzero(nb)[0].astype(np.int32))
    count = np.array([len(l) for l in lists], dtype=np.int32)
    return acc, jerk, count, lists


def regular_force_ex(xp, vp, m, i_idx, r_s, dtr=None):
    """Velocity criterion eq. (3) and the potential of Listing B2, written
    from the equations: neighbour iff min(|R|, |R + dtr V|) < r_s; pot = sum m / r over the summed pairs."""
    xp = np.asarray(xp, dtype=np.float64)
    vp = np.asarray(vp, dtype=np.float64)
    m = np.asarray(m, dtype=np.float64)
    n_i = len(i_idx)
    dtr = np.zeros(n_i) if dtr is None else np.asarray(dtr, dtype=np.float64)
    acc = np.zeros((n_i, 3))
    jerk = np.zeros((n_i, 3))
    pot = np.zeros(n_i)
    lists = []
    for q, (i, h) in enumerate(zip(i_idx, r_s)):
        R = xp - xp[i]
        V = vp - vp[i]
        r = np.linalg.norm(R, axis=1)
        rp = np.linalg.norm(R + dtr[q] * V, axis=1)
        other = np.arange(xp.shape[0]) != i
        nb = other & (np.minimum(r * r, rp * rp) < h * h)
        summed = other & ~nb & (r > 0.0)
        Rs, Vs, rs_, ms = R[summed], V[summed], r[summed], m[summed]
        rv = np.einsum("jc,jc->j", Rs, Vs)
        acc[q] = (ms[:, None] * Rs / rs_[:, None] ** 3).sum(axis=0)
        jerk[q] = (ms[:, None] * (Vs / rs_[:, None] ** 3 - 3.0 * rv[:, None] * Rs / rs_[:, None] ** 5)).sum(axis=0)
        pot[q] = (ms / rs_).sum()
        lists.append(np.nonzero(nb)[0].astype(np.int32))
    count = np.array([len(l) for l in lists], dtype=np.int32)
    return acc, jerk, pot, count, lists


def irregular_force(xp, vp, m, i_idx, lists):
    """eq. (7), (8), from the equations: sums over the given neighbour lists."""
    xp = np.asarray(xp, dtype=np.float64)
    vp = np.asarray(vp, dtype=np.float64)
    m = np.asarray(m, dtype=np.float64)
    acc = np.zeros((len(i_idx), 3))
    jerk = np.zeros((len(i_idx), 3))
    for q, i in enumerate(i_idx):
        js = np.asarray([j for j in lists[q] if j != i], dtype=np.int64)
        if js.size == 0:
            continue
        R = xp[js] - xp[i]
        V = vp[js] - vp[i]
        r = np.linalg.norm(R, axis=1)
        ok = r > 0
        R, V, r, mj = R[ok], V[ok], r[ok], m[js][ok]
        rv = np.einsum("jc,jc->j", R, V)
        acc[q] = (mj[:, None] * R / r[:, None] ** 3).sum(axis=0)
        jerk[q] = (mj[:, None] * (V / r[:, None] ** 3 - 3.0 * rv[:, None] * R / r[:, None] ** 5)).sum(axis=0)
    return acc, jerk
