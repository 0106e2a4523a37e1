"""Pins for oracle/corrector.py (step (vii); eq. (1)) -- CPU only.

The paper prints no corrector formula (readings R16-R18), so the pins are what the
mathematics fixes: exactness on polynomial force (integrated by numpy's polynomial routines, not by the oracle's
formula), the convergence order on a Kepler circle, the list-difference identity that follows from eq. (7) + (9),
and eq. (1) against hand-derived values and the n ~ r^3 count of a uniform medium.
"""
import json
import os

import numpy as np
from numpy.polynomial import polynomial as P

from oracle import corrector, oracle
from paper_1205_1222_b200 import inputs

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "corrector_closed_forms.json")))


def test_hermite_golden_cubic():
    g = GOLD["hermite_cubic"]
    col = lambda v: np.array([[v, 0.0, -v]])
    d2, d3, dx, dv = corrector.hermite_corrector(col(g["f0"]), col(g["fd0"]), col(g["f1"]), col(g["fd1"]),
                                                 np.array([g["dt"]]))
    for got, key in ((d2, "d2_end"), (d3, "d3"), (dx, "dx"), (dv, "dv")):
        assert np.allclose(got[0], [g[key], 0.0, -g[key]], rtol=1e-13, atol=1e-15), key


def test_hermite_reproduces_quintic_trajectory():
    """Force cubic in time => trajectory quintic.  numpy integrates the polynomial; predictor + corrector must land
    on it to rounding, and recover the derivatives at the END of the step."""
    rng = np.random.default_rng(11)
    n = 50
    coef = rng.normal(size=(n, 3, 4))               # F(tau) = c0 + c1 tau + c2 tau^2 + c3 tau^3, per row/component
    x0, v0 = rng.normal(size=(n, 3)), rng.normal(size=(n, 3))
    dt = 2.0 ** -rng.integers(1, 8, size=n)
    f0, fd0 = coef[..., 0], coef[..., 1]
    f1, fd1, x_true, v_true, d2_true = (np.empty((n, 3)) for _ in range(5))
    for q in range(n):
        for c in range(3):
            pf = coef[q, c]
            pv = P.polyint(pf, k=[v0[q, c]])        # v(tau)
            px = P.polyint(pv, k=[x0[q, c]])        # x(tau)
            f1[q, c], fd1[q, c] = P.polyval(dt[q], pf), P.polyval(dt[q], P.polyder(pf))
            d2_true[q, c] = P.polyval(dt[q], P.polyder(pf, 2))
            x_true[q, c], v_true[q, c] = P.polyval(dt[q], px), P.polyval(dt[q], pv)
    h = dt[:, None]
    xp = x0 + v0 * h + f0 * h ** 2 / 2 + fd0 * h ** 3 / 6      # the predictor of north_star
    vp = v0 + f0 * h + fd0 * h ** 2 / 2
    d2, d3, dx, dv = corrector.hermite_corrector(f0, fd0, f1, fd1, dt)
    assert np.abs(xp + dx - x_true).max() < 1e-13 and np.abs(vp + dv - v_true).max() < 1e-13
    assert np.abs(dx).max() > 1e-4                  # the increments are not negligible in this test
    scale = np.abs(coef).max() / dt.min() ** 2      # d2, d3 divide rounding errors of f by dt^2, dt^3
    assert np.abs(d2 - d2_true).max() < 1e-13 * scale
    assert np.abs(d3 - 6 * coef[..., 3]).max() < 1e-13 * scale / dt.min()


def test_hermite_order_on_kepler_circle():
    """Test particle on the unit circle around a unit point mass: F = -(cos t, sin t, 0).  The corrected position
    converges as dt^6 and the velocity as dt^5 (cubic Hermite: F'' to O(dt^2), F''' to O(dt)); a wrong
    coefficient anywhere lowers the order."""
    errs = []
    for h in (0.2, 0.1, 0.05):
        x0, v0 = np.array([[1.0, 0, 0]]), np.array([[0, 1.0, 0]])
        f = lambda t: np.array([[-np.cos(t), -np.sin(t), 0]])
        fd = lambda t: np.array([[np.sin(t), -np.cos(t), 0]])
        xp = x0 + v0 * h + f(0) * h ** 2 / 2 + fd(0) * h ** 3 / 6
        vp = v0 + f(0) * h + fd(0) * h ** 2 / 2
        _, _, dx, dv = corrector.hermite_corrector(f(0), fd(0), f(h), fd(h), np.array([h]))
        ex = np.linalg.norm(xp + dx - [[np.cos(h), np.sin(h), 0]])
        ev = np.linalg.norm(vp + dv - [[-np.sin(h), np.cos(h), 0]])
        e_pred = np.linalg.norm(xp - [[np.cos(h), np.sin(h), 0]])
        assert ex < e_pred * h                       # the corrector gains more than one order
        errs.append((ex, ev))
    for k in (0, 1):
        rx, rv = errs[k][0] / errs[k + 1][0], errs[k][1] / errs[k + 1][1]
        assert 50 < rx < 80 and 25 < rv < 40, (rx, rv)


def test_old_list_force_is_new_force_plus_list_difference():
    """F_R(L_old) = F_R(L_new) + F_I(L_new) - F_I(L_old), same for the derivative (eq. (7) + (9) = total for ANY list,
    PAPER.md:94-104): the route the GPU takes, checked between three different loops of the oracle."""
    rngs = inputs.streams(6, 21)
    x, v = inputs.plummer_points(rngs, 700)
    m = inputs.salpeter_masses(rngs["mass"], 700)
    ii = np.arange(0, 700, 3, dtype=np.int32)
    rs_old = inputs.kth_neighbour_distance(x, ii, 24, brute=True) * 1.0001
    rs_new = rs_old * np.random.default_rng(5).uniform(0.7, 1.4, size=len(ii))
    _, _, _, l_old = oracle.regular_force(x, v, m, ii, rs_old)
    a_new, j_new, c_new, l_new = oracle.regular_force(x, v, m, ii, rs_new)
    assert any(set(a) != set(b) for a, b in zip(l_old, l_new))
    ai_new, ji_new, sa, sj = oracle.irregular_force(x, v, m, ii, l_new)
    ai_old, ji_old, sa2, sj2 = oracle.irregular_force(x, v, m, ii, l_old)
    a_ref, j_ref = corrector.regular_force_old_list(x, v, m, ii, l_old)
    assert (np.linalg.norm(a_new + ai_new - ai_old - a_ref, axis=1) / (sa + sa2 + 1)).max() < 1e-13
    assert (np.linalg.norm(j_new + ji_new - ji_old - j_ref, axis=1) / (sj + sj2 + 1)).max() < 1e-13
    # and it is NOT the new-list force: the correction matters
    assert np.linalg.norm(a_new - a_ref, axis=1).max() > 1e-3


def test_radius_update_golden_and_uniform_medium():
    for c in GOLD["radius_update"]["cases"]:
        got = corrector.neighbour_radius_update([c["r_s"]], [c["n_p"]], [c["n_i"]])[0]
        assert abs(got - c["r_s_new"]) < 1e-15, c
    # uniform medium: the count inside r grows as r^3, so the new radius holds about n_p particles
    rng = np.random.default_rng(3)
    pts = rng.uniform(-1, 1, size=(400000, 3))
    r = np.linalg.norm(pts, axis=1)
    r_old, n_p = 0.3, 12000.0
    n_i = int((r < r_old).sum())
    r_new = corrector.neighbour_radius_update([r_old], [n_p], [n_i])[0]
    n_new = int((r < r_new).sum())
    assert abs(n_new - n_p) < 6 * np.sqrt(n_p) and r_new < 1.0


def test_regular_corrector_chain():
    """The block function is the three steps in order."""
    rngs = inputs.streams(6, 22)
    x, v = inputs.plummer_points(rngs, 300)
    m = np.full(300, 1 / 300)
    ii = np.array([5, 17, 100], dtype=np.int32)
    rs = inputs.kth_neighbour_distance(x, ii, 10, brute=True) * 1.0001
    _, _, cnt, lists = oracle.regular_force(x, v, m, ii, rs)
    rng = np.random.default_rng(1)
    f0, fd0 = rng.normal(size=(3, 3)), rng.normal(size=(3, 3))
    dt = np.array([0.125, 0.25, 0.0625])
    out = corrector.regular_corrector(x, v, m, ii, lists, cnt, dt, f0, fd0, rs, np.array([20.0, 5.0, 10.0]))
    a, j = oracle.force_given_lists(x, v, m, ii, lists)
    assert np.array_equal(out["f1"], a) and np.array_equal(out["fd1"], j)
    d2, d3, dx, dv = corrector.hermite_corrector(f0, fd0, a, j, dt)
    assert np.array_equal(out["dx"], dx) and np.array_equal(out["d3"], d3)
    assert np.allclose(out["r_s_new"], rs * np.cbrt(np.array([20.0, 5.0, 10.0]) / np.maximum(cnt, 1)))
