"""Seeded synthetic inputs for the regular-force path (serves the CUDA path, the oracle and the tests).

This module holds only the INPUT RECIPE of DESIGN.md section "Inputs": Plummer spheres in N-body units
(section 4: "isolated Plummer models in virial equilibrium ... standard N-body units with
total energy E=-0.25 and total mass 1"), the Salpeter masses and primordial binaries BASELINE.json's
configs add, block time-steps, active sets and neighbour radii.  It holds none of the
method's arithmetic: no predictor, no pair force, no neighbour test.  Where a config needs the
predicted positions or a first force pass, the caller passes them in (`predict=`, `forces=`).

All draws come from numpy Generator(PCG64) streams spawned from SeedSequence(12051222): one child per
config, one grandchild per named stream, so that changing one recipe never shifts another.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Callable, Optional

import numpy as np

SEED = 12051222
STREAMS = ("radius", "dir_x", "speed", "dir_v", "mass", "binary", "active", "dt", "overflow")
N_CONFIGS = 5

# Plummer scale length in N-body units (G = M = 1, E = -1/4): b = 3*pi/16.
B_PLUMMER = 3.0 * np.pi / 16.0
R_TRUNC = 20.0  # truncation radius in Plummer-scale units (the paper is silent; our choice)

# (N, N_i, k target neighbours, nbr cap) per BASELINE.json config; N_i None = swept (config 3).
CONFIG_TABLE = {
    1: dict(n=1024, n_i=1024, k=32, cap=128),
    2: dict(n=16384, n_i=2048, k=50, cap=256),
    3: dict(n=65536, n_i=65536, k=80, cap=256),
    4: dict(n=200000, n_i=8192, k=100, cap=512),
    5: dict(n=1048576, n_i=1048576, k=100, cap=512),
}
CONFIG3_BLOCKS = tuple(2 ** e for e in range(5, 17))  # 32 ... 65536
N_BINARIES_4 = 10000  # config 4: 10 % of 200000 particles sit in binaries


def streams(config: int, sub: int = 0) -> dict:
    """Named generators for one config.  `sub` > 0 gives independent streams for custom workloads."""
    root = np.random.SeedSequence(SEED)
    child = root.spawn(N_CONFIGS + 1)[config - 1 if 1 <= config <= N_CONFIGS else N_CONFIGS]
    if sub:
        child = child.spawn(sub + 1)[sub]
    grand = child.spawn(len(STREAMS))
    return {name: np.random.Generator(np.random.PCG64(s)) for name, s in zip(STREAMS, grand)}


# ----------------------------------------------------------------------------- Plummer sampling
def _unit_vectors(rng, n):
    z = rng.uniform(-1.0, 1.0, n)
    phi = rng.uniform(0.0, 2.0 * np.pi, n)
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)


def _plummer_radii(rng, n):
    r = np.empty(n)
    todo = np.arange(n)
    while todo.size:
        u = rng.uniform(0.0, 1.0, todo.size)
        u = np.where(u <= 0.0, 0.5, u)
        rr = 1.0 / np.sqrt(u ** (-2.0 / 3.0) - 1.0 + 1e-300)
        ok = rr <= R_TRUNC
        r[todo[ok]] = rr[ok]
        todo = todo[~ok]
    return r


def _plummer_speed_fraction(rng, n):
    """q = v / v_esc by von Neumann rejection on g(q) = q^2 (1 - q^2)^(7/2) <= 0.1."""
    q = np.empty(n)
    todo = np.arange(n)
    while todo.size:
        qq = rng.uniform(0.0, 1.0, todo.size)
        yy = rng.uniform(0.0, 0.1, todo.size)
        ok = yy < qq * qq * (1.0 - qq * qq) ** 3.5
        q[todo[ok]] = qq[ok]
        todo = todo[~ok]
    return q


def plummer_points(rngs: dict, n: int):
    """n phase-space points of a Plummer model in N-body units (not yet centred)."""
    r = _plummer_radii(rngs["radius"], n)
    x = r[:, None] * _unit_vectors(rngs["dir_x"], n)
    q = _plummer_speed_fraction(rngs["speed"], n)
    speed = q * np.sqrt(2.0) * (1.0 + r * r) ** (-0.25)
    v = speed[:, None] * _unit_vectors(rngs["dir_v"], n)
    x *= B_PLUMMER
    v *= np.sqrt(1.0 / B_PLUMMER)
    return x, v


def _centre(x, v, m):
    mt = m.sum()
    x -= (m[:, None] * x).sum(axis=0) / mt
    v -= (m[:, None] * v).sum(axis=0) / mt


def salpeter_masses(rng, n, m_lo=0.1, m_hi=10.0, alpha=2.35):
    p = 1.0 - alpha  # -1.35
    u = rng.uniform(0.0, 1.0, n)
    m = (m_lo ** p + u * (m_hi ** p - m_lo ** p)) ** (1.0 / p)
    return m / m.sum()


# ----------------------------------------------------------------------------- smooth field for a0, jerk0
def plummer_field(x, v):
    """Acceleration and its time derivative of the smooth Plummer potential (M = 1, b = 3 pi / 16)
    seen by a particle at x moving with v.  Input recipe for a0, jerk0 where no force pass is given."""
    d2 = (x * x).sum(axis=1) + B_PLUMMER ** 2
    d3 = d2 * np.sqrt(d2)
    xv = (x * v).sum(axis=1)
    a = -x / d3[:, None]
    j = -v / d3[:, None] + 3.0 * (xv / (d3 * d2))[:, None] * x
    return a, j


# ----------------------------------------------------------------------------- binaries (config 4)
def _kepler_relative_orbit(rng, nb, mu):
    """Relative position and velocity of nb bound two-body orbits with total mass mu (G = 1):
    semi-major axis log-uniform in [1e-5, 1e-3], thermal eccentricity e = sqrt(u), uniform mean anomaly,
    uniformly random orientation."""
    a = 10.0 ** rng.uniform(-5.0, -3.0, nb)
    e = np.sqrt(rng.uniform(0.0, 1.0, nb))
    e = np.minimum(e, 0.99)  # keep pericentre resolved; the thermal tail above 0.99 is 2 % of draws
    M = rng.uniform(0.0, 2.0 * np.pi, nb)
    E = M + e * np.sin(M)
    for _ in range(60):  # Newton on Kepler's equation E - e sin E = M
        E -= (E - e * np.sin(E) - M) / (1.0 - e * np.cos(E))
    cosE, sinE = np.cos(E), np.sin(E)
    r = a * (1.0 - e * cosE)
    px = a * (cosE - e)
    py = a * np.sqrt(1.0 - e * e) * sinE
    fac = np.sqrt(mu * a) / r
    vx = -fac * sinE
    vy = fac * np.sqrt(1.0 - e * e) * cosE
    # uniform random rotation from a normalised Gaussian quaternion
    qn = rng.normal(size=(nb, 4))
    qn /= np.linalg.norm(qn, axis=1)[:, None]
    w, qx, qy, qz = qn.T
    R = np.empty((nb, 3, 3))
    R[:, 0, 0] = 1 - 2 * (qy * qy + qz * qz)
    R[:, 0, 1] = 2 * (qx * qy - qz * w)
    R[:, 0, 2] = 2 * (qx * qz + qy * w)
    R[:, 1, 0] = 2 * (qx * qy + qz * w)
    R[:, 1, 1] = 1 - 2 * (qx * qx + qz * qz)
    R[:, 1, 2] = 2 * (qy * qz - qx * w)
    R[:, 2, 0] = 2 * (qx * qz - qy * w)
    R[:, 2, 1] = 2 * (qy * qz + qx * w)
    R[:, 2, 2] = 1 - 2 * (qx * qx + qy * qy)
    rel = R[:, :, 0] * px[:, None] + R[:, :, 1] * py[:, None]
    vrel = R[:, :, 0] * vx[:, None] + R[:, :, 1] * vy[:, None]
    return rel, vrel, a


# ----------------------------------------------------------------------------- state
@dataclass
class State:
    """fp64 j-particle state at each particle's own last time t0 (what nb_set_j registers)."""
    config: int
    n: int
    x0: np.ndarray
    v0: np.ndarray
    a0: np.ndarray
    j0: np.ndarray
    m: np.ndarray
    t0: np.ndarray
    t: float
    n_binary_members: int = 0  # particles [0, n_binary_members) are binary components (2b, 2b+1)
    a0_source: str = "plummer_field"


@dataclass
class Workload:
    state: State
    i_idx: np.ndarray  # int32[n_i], 0-based
    r_s: np.ndarray  # float64[n_i]
    k: int
    cap: int
    name: str = ""
    rs_positions: str = "x0"
    extra: dict = field(default_factory=dict)

    @property
    def n_i(self):
        return int(self.i_idx.shape[0])

    @property
    def pairs(self):
        return self.n_i * self.state.n


def _block_dt(rng, n, k_lo, k_hi):
    k = rng.integers(k_lo, k_hi + 1, n)
    return 2.0 ** (-k.astype(np.float64))


def _finish_state(config, x, v, m, rngs, dt_rule, forces, n_binary_members=0, companion=None):
    n = x.shape[0]
    src = "plummer_field"
    if forces is not None:
        a0, j0 = forces(x, v, m)
        a0 = np.ascontiguousarray(a0, dtype=np.float64)
        j0 = np.ascontiguousarray(j0, dtype=np.float64)
        src = "force_pass"
    else:
        a0, j0 = plummer_field(x, v)
        if companion is not None:
            # binary members also feel their companion: textbook two-body term, part of the recipe for
            # realistic a0/jerk0 (|a| ~ 5e4, |jerk| ~ 5e9 at a = 1e-5), see DESIGN.md "Inputs".
            nb2 = n_binary_members
            R = x[companion] - x[:nb2]
            V = v[companion] - v[:nb2]
            r2 = (R * R).sum(axis=1)
            r3 = r2 * np.sqrt(r2)
            rv = (R * V).sum(axis=1)
            mc = m[companion]
            a0[:nb2] += (mc / r3)[:, None] * R
            j0[:nb2] += (mc / r3)[:, None] * (V - (3.0 * rv / r2)[:, None] * R)
    t = 1.0
    if dt_rule[0] == "const":
        dt = np.full(n, dt_rule[1])
    else:
        dt = _block_dt(rngs["dt"], n, dt_rule[1], dt_rule[2])
    if n_binary_members:
        an = np.linalg.norm(a0[:n_binary_members], axis=1)
        jn = np.linalg.norm(j0[:n_binary_members], axis=1)
        kb = np.ceil(-np.log2(an / (32.0 * jn)))
        kb = np.clip(kb, 3, 40)
        dt[:n_binary_members] = 2.0 ** (-kb)
    t0 = t - dt
    return State(config, n, np.ascontiguousarray(x), np.ascontiguousarray(v), a0, j0,
                 np.ascontiguousarray(m), t0, t, n_binary_members, src)


def make_state(config: int, forces: Optional[Callable] = None) -> State:
    """State of BASELINE.json config 1..5.  `forces(x, v, m) -> (a, jerk)` supplies a0, jerk0 from a
    first force pass (configs 1-2 in the tests); without it the smooth Plummer field is used."""
    spec = CONFIG_TABLE[config]
    n = spec["n"]
    rngs = streams(config)
    if config == 4:
        nb = N_BINARIES_4
        npts = n - nb  # 190000 Plummer points: nb centres of mass, then the singles
        xc, vc = plummer_points(rngs, npts)
        m1 = 1.0 / n
        mp = np.full(npts, m1)
        mp[:nb] = 2.0 * m1
        _centre(xc, vc, mp)
        rel, vrel, _a = _kepler_relative_orbit(rngs["binary"], nb, 2.0 * m1)
        x = np.empty((n, 3))
        v = np.empty((n, 3))
        x[0:2 * nb:2] = xc[:nb] - 0.5 * rel
        x[1:2 * nb:2] = xc[:nb] + 0.5 * rel
        v[0:2 * nb:2] = vc[:nb] - 0.5 * vrel
        v[1:2 * nb:2] = vc[:nb] + 0.5 * vrel
        x[2 * nb:] = xc[nb:]
        v[2 * nb:] = vc[nb:]
        m = np.full(n, m1)
        companion = np.arange(2 * nb) ^ 1
        return _finish_state(config, x, v, m, rngs, ("block", 3, 10), forces, 2 * nb, companion)
    x, v = plummer_points(rngs, n)
    if config == 3:
        m = salpeter_masses(rngs["mass"], n)
    else:
        m = np.full(n, 1.0 / n)
    _centre(x, v, m)
    dt_rule = {1: ("const", 1.0 / 64.0), 2: ("block", 3, 10), 3: ("block", 3, 10), 5: ("block", 3, 12)}[config]
    return _finish_state(config, x, v, m, rngs, dt_rule, forces)


def make_active(config: int, state: State, n_i: Optional[int] = None) -> np.ndarray:
    """Active block (0-based int32 indices into the j arrays)."""
    spec = CONFIG_TABLE[config]
    rng = streams(config)["active"]
    n = state.n
    if config in (1, 5):
        idx = np.arange(n)
        if n_i is not None:
            idx = idx[:n_i]
    elif config == 2:
        idx = rng.choice(n, size=spec["n_i"], replace=False)
    elif config == 3:
        perm = rng.permutation(n)
        idx = perm[: (n_i if n_i is not None else n)]
    else:  # config 4: exactly 10 % of the block are binary members
        nbm = state.n_binary_members
        n_b = (spec["n_i"] * 10) // 100
        ib = rng.choice(nbm, size=n_b, replace=False)
        isg = nbm + rng.choice(n - nbm, size=spec["n_i"] - n_b, replace=False)
        idx = np.concatenate([ib, isg])
        rng.shuffle(idx)
    return np.ascontiguousarray(idx, dtype=np.int32)


def kth_neighbour_distance(pos: np.ndarray, idx: np.ndarray, k: int, brute: bool = False) -> np.ndarray:
    """Distance from pos[idx[q]] to its k-th nearest OTHER particle."""
    idx = np.asarray(idx, dtype=np.int64)
    n = pos.shape[0]
    k = min(k, n - 1)
    if k <= 0:
        return np.zeros(idx.shape[0])
    if brute:
        out = np.empty(idx.shape[0])
        for lo in range(0, idx.shape[0], 256):
            sel = idx[lo:lo + 256]
            d2 = ((pos[sel, None, :] - pos[None, :, :]) ** 2).sum(axis=2)
            d2[np.arange(sel.shape[0]), sel] = np.inf
            out[lo:lo + 256] = np.sqrt(np.partition(d2, k - 1, axis=1)[:, k - 1])
        return out
    from scipy.spatial import cKDTree

    tree = cKDTree(pos)
    d, j = tree.query(pos[idx], k=k + 1, workers=-1)
    # column 0 is the particle itself unless another particle coincides with it; take the k-th other.
    self_first = j[:, 0] == idx
    out = d[:, k].copy()
    if not self_first.all():
        for q in np.nonzero(~self_first)[0]:
            others = d[q][j[q] != idx[q]]
            out[q] = others[k - 1] if others.shape[0] >= k else d[q, k]
    return out


def calibrate_rs(config: int, pos_t: np.ndarray, i_idx: np.ndarray, k: Optional[int] = None,
                 factor: float = 1.0001, brute: bool = False) -> np.ndarray:
    """r_s,i = distance to the k-th nearest other particle (in the given positions) x 1.0001.
    Config 4 additionally doubles a seeded 1 % of the rows so that the list overflows (cap 512)."""
    if k is None:
        k = CONFIG_TABLE[config]["k"]
    rs = kth_neighbour_distance(pos_t, i_idx, k, brute=brute) * factor
    if config == 4:
        rng = streams(4)["overflow"]
        n_over = max(1, i_idx.shape[0] // 100)
        rows = rng.choice(i_idx.shape[0], size=n_over, replace=False)
        rs[rows] *= 2.0
    return rs


def make_workload(config: int, forces: Optional[Callable] = None, predict: Optional[Callable] = None,
                  n_i: Optional[int] = None, state: Optional[State] = None) -> Workload:
    """One BASELINE.json config.  `predict(state) -> x_p` gives the predicted positions at t on which
    r_s is calibrated (the tests pass the oracle's predictor); without it r_s is calibrated on x0."""
    spec = CONFIG_TABLE[config]
    if state is None:
        state = make_state(config, forces)
    i_idx = make_active(config, state, n_i)
    pos = state.x0 if predict is None else np.ascontiguousarray(predict(state))
    r_s = calibrate_rs(config, pos, i_idx)
    return Workload(state, i_idx, r_s, spec["k"], spec["cap"], name=f"config{config}",
                    rs_positions="x0" if predict is None else "predicted")


def make_custom(n: int, n_i: int, k: int, cap: int, seed_sub: int = 1, dt_k=(3, 10), masses: str = "equal",
                forces: Optional[Callable] = None, predict: Optional[Callable] = None,
                active: str = "random", brute_rs: bool = False) -> Workload:
    """A Plummer workload of arbitrary size (ragged-tail and edge-case tests, quick benches).
    Uses its own streams (config slot 6, sub-stream seed_sub) so it never perturbs configs 1-5."""
    rngs = streams(N_CONFIGS + 1, seed_sub)
    x, v = plummer_points(rngs, n)
    m = salpeter_masses(rngs["mass"], n) if masses == "salpeter" else np.full(n, 1.0 / n)
    _centre(x, v, m)
    state = _finish_state(0, x, v, m, rngs, ("block", dt_k[0], dt_k[1]), forces)
    if active == "all":
        idx = np.arange(min(n_i, n))
    else:
        idx = rngs["active"].choice(n, size=n_i, replace=n_i > n)
    idx = np.ascontiguousarray(idx, dtype=np.int32)
    pos = state.x0 if predict is None else np.ascontiguousarray(predict(state))
    r_s = kth_neighbour_distance(pos, idx, k, brute=brute_rs) * 1.0001 if k > 0 else np.zeros(idx.shape[0])
    return Workload(state, idx, r_s, k, cap, name=f"custom_n{n}_ni{n_i}_k{k}",
                    rs_positions="x0" if predict is None else "predicted")
