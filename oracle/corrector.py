"""Oracle for the regular corrector of step (vii) and the neighbour-radius update eq. (1) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this.  It never imports the CUDA
package and shares no code with it.  fp64 numpy, one plain statement per step, in the order of the text.

What the paper fixes (step (vii)): "Execute the regular corrector.  Since the neighbour list L_i has
been updated, the force polynomials should be corrected to reflect the difference between the old and new list."
It prints no corrector formula; it names the scheme: "fourth-order ... Hermite formulation (Makino 1991) for the
case of two force polynomials (Makino & Aarseth 1992)", i.e. the cubic force polynomial through
(F, dF/dt) at both ends of the step.  Readings R16-R19 of DESIGN.md section 2 state what is taken here:

  1. regular_force_old_list: the regular force at the END of the step with respect to the OLD list, by the plain
     definition eq. (9), (10) with "neighbour" := member of L_old (oracle.force_given_lists): the polynomial of
     the step that just ended was built on L_old, so its end point must exclude the same particles (R16).
  2. hermite_corrector: the unique cubic F(tau) with F(0) = F0, F'(0) = Fd0, F(dt) = F1, F'(dt) = Fd1; its second
     and third derivatives; and the terms of the Taylor series of x and v the predictor (x0 + v0 dt + F0 dt^2/2 +
     Fd0 dt^3/6, north_star) left out: dx = F2 dt^4/24 + F3 dt^5/120, dv = F2 dt^3/6 + F3 dt^4/24 (R17).
  3. neighbour_radius_update: eq. (1), R_s_new = R_s_old (n_p / n_i)^(1/3); n_i = 0 is "catered for"
      without saying how: n_i := 1 (R18).

Pins (tests/test_oracle_corrector.py): a quintic trajectory integrated by numpy's polynomial routines is
reproduced exactly; on a Kepler circle the corrected position converges as dt^6 and the velocity as dt^5; the
old-list force equals new-list force + F_I(L_new) - F_I(L_old) (eq. (7) + (9), three different oracle loops);
eq. (1) against the uniform-density count n ~ r^3 and printed closed-form values.
"""
from __future__ import annotations

import numpy as np

from . import oracle


def regular_force_old_list(xp, vp, m, i_idx, old_lists, old_counts=None):
    """F_R, dF_R/dt at the predicted state, excluding the members of the OLD lists (eq. (9), (10), PAPER.md:102-106,
    with the condition replaced by list membership; R16)."""
    return oracle.force_given_lists(xp, vp, m, i_idx, old_lists, old_counts)


def hermite_corrector(f0, fd0, f1, fd1, dt):
    """Cubic Hermite interpolation of the regular force over one regular step and the corrector increments (R17).

    f0, fd0: [n_i, 3] regular force and derivative at the start of the step; f1, fd1: at the end, SAME list.
    dt: [n_i] length of the step (> 0).  Returns d2 (second derivative at the END of the step), d3 (third
    derivative, constant), dx, dv (to be added to the predicted position and velocity).
    Derivation: F(tau) = f0 + fd0 tau + A tau^2/2 + B tau^3/6 with F(dt) = f1, F'(dt) = fd1 gives
      A = [-6 (f0 - f1) - dt (4 fd0 + 2 fd1)] / dt^2,   B = [12 (f0 - f1) + 6 dt (fd0 + fd1)] / dt^3."""
    f0, fd0, f1, fd1 = (np.asarray(a, dtype=np.float64) for a in (f0, fd0, f1, fd1))
    h = np.asarray(dt, dtype=np.float64)[:, None]
    a = (-6.0 * (f0 - f1) - h * (4.0 * fd0 + 2.0 * fd1)) / h ** 2
    b = (12.0 * (f0 - f1) + 6.0 * h * (fd0 + fd1)) / h ** 3
    dx = a * h ** 4 / 24.0 + b * h ** 5 / 120.0
    dv = a * h ** 3 / 6.0 + b * h ** 4 / 24.0
    d2 = a + h * b
    d3 = b
    return d2, d3, dx, dv


def neighbour_radius_update(r_s, n_p, n_i):
    """eq. (1): R_s_new = R_s_old (n_p / n_i)^(1/3); n_i = 0 counts as 1 (R18)."""
    r_s = np.asarray(r_s, dtype=np.float64)
    n_p = np.asarray(n_p, dtype=np.float64)
    n_i = np.maximum(np.asarray(n_i, dtype=np.float64), 1.0)
    return r_s * np.cbrt(n_p / n_i)


def regular_corrector(xp, vp, m, i_idx, old_lists, new_counts, dt_r, fr0, frd0, r_s, n_p, old_counts=None):
    """Step (vii) for a block of rows: 1., 2., 3. above in that order.
    Returns dict(f1, fd1, d2, d3, dx, dv, r_s_new)."""
    f1, fd1 = regular_force_old_list(xp, vp, m, i_idx, old_lists, old_counts)
    d2, d3, dx, dv = hermite_corrector(fr0, frd0, f1, fd1, dt_r)
    r_new = neighbour_radius_update(r_s, n_p, new_counts)
    return dict(f1=f1, fd1=fd1, d2=d2, d3=d3, dx=dx, dv=dv, r_s_new=r_new)
