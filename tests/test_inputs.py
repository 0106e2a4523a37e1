"""The seeded input recipe (BASELINE.json configs) -- CPU only."""
import numpy as np

from paper_1205_1222_b200 import inputs


def test_streams_are_reproducible_and_independent():
    a = inputs.streams(2)["radius"].uniform(size=4)
    b = inputs.streams(2)["radius"].uniform(size=4)
    c = inputs.streams(3)["radius"].uniform(size=4)
    assert np.array_equal(a, b) and not np.array_equal(a, c)


def test_config1_state_properties():
    s = inputs.make_state(1)
    assert s.n == 1024 and s.x0.shape == (1024, 3) and s.x0.dtype == np.float64
    assert abs(s.m.sum() - 1.0) < 1e-12
    np.testing.assert_allclose((s.m[:, None] * s.x0).sum(axis=0), 0, atol=1e-14)
    np.testing.assert_allclose((s.m[:, None] * s.v0).sum(axis=0), 0, atol=1e-14)
    assert np.all(s.t - s.t0 == 1.0 / 64.0)
    # N-body units: virial ratio about 1 and E about -1/4 (statistical at N = 1024)
    ke = 0.5 * (s.m * (s.v0 ** 2).sum(axis=1)).sum()
    d = np.sqrt(((s.x0[:, None] - s.x0[None]) ** 2).sum(axis=2))
    np.fill_diagonal(d, np.inf)
    pe = -0.5 * (s.m[:, None] * s.m[None] / d).sum()
    assert -0.32 < ke + pe < -0.19 and 0.8 < -2 * ke / pe < 1.2


def test_config2_block_steps_and_active_set():
    s = inputs.make_state(2)
    dt = s.t - s.t0
    k = -np.log2(dt)
    assert np.all(k == np.round(k)) and k.min() == 3 and k.max() == 10
    idx = inputs.make_active(2, s)
    assert idx.dtype == np.int32 and idx.shape == (2048,) and np.unique(idx).shape == (2048,)
    assert not np.array_equal(idx, np.sort(idx))


def test_config3_masses_and_nested_blocks():
    s = inputs.make_state(3)
    assert abs(s.m.sum() - 1.0) < 1e-12 and 50 < s.m.max() / s.m.min() <= 100.0001
    full = inputs.make_active(3, s)
    for n_i in (32, 1024):
        assert np.array_equal(inputs.make_active(3, s, n_i), full[:n_i])
    assert np.array_equal(np.sort(full), np.arange(65536))


def test_config4_binaries():
    s = inputs.make_state(4)
    nb2 = s.n_binary_members
    assert s.n == 200000 and nb2 == 20000
    sep = np.linalg.norm(s.x0[0:nb2:2] - s.x0[1:nb2:2], axis=1)
    assert 1e-7 < sep.min() and sep.max() < 2.1e-3  # a in [1e-5, 1e-3], e <= 0.99
    # bound pairs: relative energy negative
    vrel = np.linalg.norm(s.v0[0:nb2:2] - s.v0[1:nb2:2], axis=1)
    mu = s.m[0] + s.m[1]
    assert np.all(0.5 * vrel ** 2 - mu / sep < 0)
    # predictor step stays inside the orbit: dt * |jerk| / |a| <= 1/32 (block-step rule of the recipe)
    an = np.linalg.norm(s.a0[:nb2], axis=1)
    jn = np.linalg.norm(s.j0[:nb2], axis=1)
    dt = (s.t - s.t0)[:nb2]
    assert np.all(dt * jn / an <= 1.0 / 32.0 * 1.0000001) or np.all(dt >= 2.0 ** -40)
    idx = inputs.make_active(4, s)
    assert idx.shape == (8192,) and (idx < nb2).sum() == 819 and np.unique(idx).shape == (8192,)


def test_rs_calibration_kdtree_matches_bruteforce():
    s = inputs.make_state(2)
    idx = inputs.make_active(2, s)[:200]
    a = inputs.kth_neighbour_distance(s.x0, idx, 50)
    b = inputs.kth_neighbour_distance(s.x0, idx, 50, brute=True)
    np.testing.assert_allclose(a, b, rtol=1e-14)
    # by construction exactly k others are strictly inside r_s = d_k * 1.0001 unless the (k+1)-th is within 1e-4
    rs = a * 1.0001
    d = np.linalg.norm(s.x0[idx][:, None, :] - s.x0[None, :, :], axis=2)
    cnt = (d < rs[:, None]).sum(axis=1) - 1
    assert cnt.min() == 50 and cnt.max() <= 52
