"""Edge cases of the CUDA path against the oracle (-m gpu): ragged sizes, every CTA shape and j-split,
degenerate radii, overflow, duplicates, translation, coincident particles, host-buffer entry point."""
import ctypes

import numpy as np
import pytest
import torch

from paper_1205_1222_b200 import binding, inputs
import parity
from gpu_util import run_gpu

pytestmark = pytest.mark.gpu


def _wl(oracle, n, n_i, k, cap, **kw):
    return inputs.make_custom(n, n_i, k, cap, predict=lambda s: oracle.predict_state(s)[0], **kw)


def _full_check(oracle, wl, gpu, cap=None):
    xp, vp = oracle.predict_state(wl.state)
    rep = parity.compare(oracle, xp, vp, wl.state.m, wl.i_idx, wl.r_s, cap or wl.cap, gpu)
    parity.check_overflow_flag(gpu, cap or wl.cap)
    return rep


@pytest.mark.parametrize("i_block", [32, 64, 128, 256, 512])
@pytest.mark.parametrize("j_split", [1, 3, 0])
def test_every_cta_shape_and_split_ragged(oracle, i_block, j_split):
    # n odd and not a multiple of any tile; n_i not a multiple of any CTA width; several tiles per chunk
    wl = _wl(oracle, 2999, 777, 24, 64, masses="salpeter")
    gpu, info = run_gpu(wl, options={"i_block": i_block, "j_split": j_split})
    assert info["rows_per_cta"] == i_block and (j_split == 0 or info["j_chunks"] == j_split)
    _full_check(oracle, wl, gpu)


def test_shapes_and_splits_agree_bitwise_on_lists_and_closely_on_sums(oracle):
    wl = _wl(oracle, 4096, 512, 30, 64)
    ref, _ = run_gpu(wl, options={"i_block": 256, "j_split": 1})
    for ib, sp in ((32, 7), (128, 2), (512, 1)):
        g, _ = run_gpu(wl, options={"i_block": ib, "j_split": sp})
        assert np.array_equal(g["nbr_count"], ref["nbr_count"])
        for q in range(wl.n_i):
            c = ref["nbr_count"][q]
            assert np.array_equal(g["nbr_list"][q, :c], ref["nbr_list"][q, :c])
        assert parity.relerr(g["acc"], ref["acc"]).max() < 1e-6  # two fp32 evaluations, each within ~3e-7 of fp64


@pytest.mark.parametrize("i_block", [32, 256])
def test_main_blocks_plus_split_tail(oracle, i_block):
    """More row blocks than CTA slots: whole waves run unsplit, the remaining blocks are j-split (atomic list
    slots + ordering in the gather kernel).  Rows are drawn with replacement so that N stays small."""
    probe = _wl(oracle, 3001, 64, 24, 64)
    _, info0 = run_gpu(probe, options={"i_block": i_block})
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    slots = sms * info0["ctas_per_sm"]
    n_i = (slots + slots // 16) * i_block + 1  # one full wave of row blocks plus a 1/16 wave that must be split
    wl = _wl(oracle, 3001, n_i, 24, 64)
    gpu, info = run_gpu(wl, options={"i_block": i_block})
    n_blocks = -(-wl.n_i // info["rows_per_cta"])
    assert 0 < info["split_row_blocks"] < n_blocks and info["j_chunks"] > 1
    assert info["ctas"] == n_blocks - info["split_row_blocks"] + info["split_row_blocks"] * info["j_chunks"]
    _full_check(oracle, wl, gpu)


def test_deterministic_repeat(oracle):
    wl = _wl(oracle, 5000, 300, 20, 64)
    a, _ = run_gpu(wl)
    b, _ = run_gpu(wl)
    for k in ("acc", "jerk", "nbr_count", "n_overflow"):
        assert np.array_equal(a[k], b[k])


def test_degenerate_radii_and_tiny_blocks(oracle):
    wl = _wl(oracle, 1500, 64, 16, 32)
    # r_s = 0: empty list, total force; r_s huge: everything a neighbour, zero force, overflow
    wl.r_s[:8] = 0.0
    wl.r_s[8:12] = 1e3
    gpu, _ = run_gpu(wl)
    rep = _full_check(oracle, wl, gpu)
    assert np.all(gpu["nbr_count"][:8] == 0)
    assert np.all(gpu["nbr_count"][8:12] == wl.state.n - 1)
    assert np.all(gpu["acc"][8:12] == 0) and np.all(gpu["jerk"][8:12] == 0)
    assert int(gpu["n_overflow"][0]) >= 4 and rep["overflow_rows"] >= 4
    # n_i = 1 and n_i = 0
    one = inputs.Workload(wl.state, wl.i_idx[20:21].copy(), wl.r_s[20:21].copy(), wl.k, wl.cap)
    g1, _ = run_gpu(one)
    assert np.array_equal(g1["acc"][0], gpu["acc"][20]) or parity.relerr(g1["acc"], gpu["acc"][20:21]).max() < 1e-6
    _full_check(oracle, one, g1)
    zero = inputs.Workload(wl.state, wl.i_idx[:0].copy(), wl.r_s[:0].copy(), wl.k, wl.cap)
    g0, _ = run_gpu(zero)
    assert int(g0["n_overflow"][0]) == 0


def test_duplicate_indices_and_self_exclusion(oracle):
    wl = _wl(oracle, 1200, 96, 12, 32)
    wl.i_idx[1] = wl.i_idx[0]
    wl.r_s[1] = wl.r_s[0]
    gpu, _ = run_gpu(wl)
    _full_check(oracle, wl, gpu)
    assert np.array_equal(gpu["acc"][0], gpu["acc"][1]) and gpu["nbr_count"][0] == gpu["nbr_count"][1]
    for q in range(wl.n_i):
        assert wl.i_idx[q] not in gpu["nbr_list"][q, : min(gpu["nbr_count"][q], wl.cap)]


def test_translation_by_100_needs_double_single(oracle):
    """with plain fp32 positions this fails by orders of magnitude."""
    wl = _wl(oracle, 4000, 500, 40, 128)
    g0, _ = run_gpu(wl)
    wl.state.x0 = wl.state.x0 + np.array([100.0, -100.0, 50.0])
    g1, _ = run_gpu(wl)
    _full_check(oracle, wl, g1)
    assert parity.relerr(g1["acc"], g0["acc"]).max() < 1e-6
    same = sum(np.array_equal(g0["nbr_list"][q, :g0["nbr_count"][q]], g1["nbr_list"][q, :g1["nbr_count"][q]])
               for q in range(wl.n_i))
    assert same >= wl.n_i - 2


def test_coincident_particles(oracle):
    wl = _wl(oracle, 800, 800, 10, 32, active="all")
    s = wl.state
    s.x0[5] = s.x0[9]
    s.v0[5], s.a0[5], s.j0[5], s.t0[5] = s.v0[9], s.a0[9], s.j0[9], s.t0[9]  # stay coincident after prediction
    wl.r_s[5] = 0.0      # R4: singular term skipped, not listed
    wl.r_s[9] = 1e-3     # neighbour (0 < r_s^2)
    gpu, _ = run_gpu(wl)
    assert gpu["nbr_count"][5] == 0 and np.all(np.isfinite(gpu["acc"][5]))
    assert 5 in gpu["nbr_list"][9, : gpu["nbr_count"][9]]
    _full_check(oracle, wl, gpu)


@pytest.mark.parametrize("n,n_i", [(3001, 257), (270001, 48)])
def test_host_entry_point_matches_device_entry_point(oracle, n, n_i):
    """(270001, 48): small block of a large system, the prediction runs inside the force kernel on the context's own
    device mirrors of the host arrays."""
    wl = _wl(oracle, n, n_i, 20, 64)
    dev_out, _ = run_gpu(wl)
    s = wl.state
    ctx = binding.Context(s.n, wl.n_i, wl.cap)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    out = dict(acc=torch.empty((wl.n_i, 3), dtype=torch.float64).pin_memory(),
               jerk=torch.empty((wl.n_i, 3), dtype=torch.float64).pin_memory(),
               nbr_count=torch.empty(wl.n_i, dtype=torch.int32).pin_memory(),
               nbr_list=torch.empty((wl.n_i, wl.cap), dtype=torch.int32).pin_memory(),
               n_overflow=torch.zeros(1, dtype=torch.int32).pin_memory())
    ctx.nb_regular_force_host(pin(s.x0), pin(s.v0), pin(s.a0), pin(s.j0), pin(s.m), pin(s.t0),
                              pin(wl.i_idx.astype(np.int32)), pin(wl.r_s), s.t, out)
    for k in ("acc", "jerk", "nbr_count"):
        assert np.array_equal(out[k].numpy(), dev_out[k]), k
    for q in range(wl.n_i):
        c = dev_out["nbr_count"][q]
        assert np.array_equal(out["nbr_list"].numpy()[q, :c], dev_out["nbr_list"][q, :c])
    ctx.close()


def test_error_codes_on_device():
    lib = binding.load()
    ctx = binding.Context(1000, 100, 16)
    dummy = torch.zeros(8, dtype=torch.int32, device="cuda")
    p = ctypes.c_void_p(dummy.data_ptr())
    # force before set_j -> NB_E_STATE; n_i > n_i_max -> NB_E_INVAL; null n_overflow -> NB_E_INVAL
    assert lib.nb_regular_force(ctx._h, 4, p, p, 1.0, p, p, p, p, p, None) == -2
    assert lib.nb_regular_force(ctx._h, 101, p, p, 1.0, p, p, p, p, p, None) == -1
    assert lib.nb_regular_force(ctx._h, 4, p, p, 1.0, p, p, p, p, None, None) == -1
    assert lib.nb_predict_j(ctx._h, 1.0, None) == -2
    with pytest.raises(binding.NbregError):
        ctx.nb_set_option("no_such_option", 1)
    ctx.close()


def test_large_cap_and_overflow_on_every_path(oracle):
    """cap = 2048 with lists of ~1000 entries (sort of long j-split rows), and overflow on rows that one CTA owns
    (j_split = 1) as well as on j-split rows."""
    wl = _wl(oracle, 1800, 96, 16, 2048)
    wl.r_s[:6] = 1e3            # everything a neighbour: 1799 entries, fits cap 2048
    wl.r_s[6:12] *= 4.0         # ~1000 neighbours
    for opts in ({"j_split": 1}, {"i_block": 32, "j_split": 7}, {}):
        gpu, _ = run_gpu(wl, options=opts)
        _full_check(oracle, wl, gpu)
        assert np.all(gpu["nbr_count"][:6] == wl.state.n - 1) and int(gpu["n_overflow"][0]) == 0
    small = inputs.Workload(wl.state, wl.i_idx, wl.r_s, wl.k, 64)
    for opts in ({"j_split": 1}, {"i_block": 64, "j_split": 5}):
        gpu, _ = run_gpu(small, options=opts)
        _full_check(oracle, small, gpu, cap=64)
        assert int(gpu["n_overflow"][0]) >= 12


def _check_random_case(oracle, wl, gpu, cap, dtr, use_pot):
    """Rows with r_s > 0 under north_star's bounds; rows with r_s = 0 sum EVERY pair, the closest ones included,
    which is outside the method's regime ("all close interactions are skipped"): their error is
    measured against the summed term magnitudes instead (as for the irregular force)."""
    xp, vp = oracle.predict_state(wl.state)
    pos = np.nonzero(wl.r_s > 0)[0]
    if pos.size:
        parity.compare(oracle, xp, vp, wl.state.m, wl.i_idx, wl.r_s, cap, gpu, rows=pos, dtr=dtr, check_pot=use_pot,
                       list_stride=max(2 * cap, 512))
    zero = np.nonzero(wl.r_s == 0)[0]
    if zero.size:
        assert np.all(gpu["nbr_count"][zero] == 0)
        everyone = [np.delete(np.arange(wl.state.n, dtype=np.int32), i) for i in wl.i_idx[zero]]
        a_o, j_o, sa, sj = oracle.irregular_force(xp, vp, wl.state.m, wl.i_idx[zero], everyone)
        assert np.all(np.linalg.norm(gpu["acc"][zero] - a_o, axis=1) <= 1e-6 * sa)
        assert np.all(np.linalg.norm(gpu["jerk"][zero] - j_o, axis=1) <= 1e-6 * sj)
    parity.check_overflow_flag(gpu, cap)
    live = np.arange(cap)[None, :] < np.minimum(gpu["nbr_count"], cap)[:, None]
    assert np.all(gpu["nbr_list"][~live] == -7)  # nothing written past the count


@pytest.mark.parametrize("seed", range(12))
def test_seeded_random_shapes(oracle, seed):
    """Seeded random sizes, caps, radii scales, CTA shapes, splits, row orders and variants against the oracle."""
    rng = np.random.default_rng(1000 + seed)
    n = int(rng.integers(20, 6000))
    n_i = int(rng.integers(1, 1500))
    k = int(min(rng.integers(12, 60), n - 1))
    cap = int(rng.choice([8, 32, 64, 200]))
    wl = _wl(oracle, n, n_i, k, cap, masses=str(rng.choice(["equal", "salpeter"])), seed_sub=2 + seed)
    wl.r_s *= rng.choice([1.0, 1.0, 1.7], size=wl.n_i)            # some lists overflow small caps
    wl.r_s[rng.random(wl.n_i) < 0.03] = 0.0
    opts = {"i_block": int(rng.choice([0, 0, 32, 64, 128, 256, 512])), "j_split": int(rng.choice([0, 0, 1, 2, 9])),
            "order_rows": int(rng.choice([0, 1, 2]))}
    use_vel, use_pot = bool(rng.integers(0, 2)), bool(rng.integers(0, 2))
    dtr = (wl.state.t - wl.state.t0[wl.i_idx]) * float(rng.choice([1.0, 8.0])) if use_vel else None
    gpu, info = run_gpu(wl, options=opts, dtr=dtr, want_pot=use_pot)
    _check_random_case(oracle, wl, gpu, cap, dtr, use_pot)


def test_two_contexts_with_different_caps(oracle):
    """Kernel function attributes are per process: creating a second context with a small cap must not shrink what
    the first one may launch (its gather kernel stages cap entries per row in shared memory)."""
    big = _wl(oracle, 1500, 200, 16, 4096)
    big.r_s[:4] = 1e3
    ctx_big = binding.Context(big.state.n, big.n_i, big.cap)
    ctx_small = binding.Context(64, 8, 4)  # created later, smaller in every way
    gpu, _ = run_gpu(big, ctx=ctx_big, options={"i_block": 32, "j_split": 3})
    _full_check(oracle, big, gpu)
    assert np.all(gpu["nbr_count"][:4] == big.state.n - 1)
    ctx_small.close()
    ctx_big.close()


def test_calls_are_cuda_graph_capturable(oracle):
    """Device-pointer calls only enqueue kernels on the caller's stream (no allocation, no synchronisation), so a
    whole step -- predictor, force, gather -- can be captured once and replayed (small active blocks are bound by
    enqueue latency otherwise)."""
    wl = _wl(oracle, 5000, 96, 20, 64)
    s = wl.state
    ctx = binding.Context(s.n, wl.n_i, wl.cap)
    ctx.set_state(s)
    dev = ctx.workspace.device
    i_idx = torch.from_numpy(np.ascontiguousarray(wl.i_idx, dtype=np.int32)).to(dev)
    r_s = torch.from_numpy(np.ascontiguousarray(wl.r_s)).to(dev)
    out = ctx.alloc_outputs(wl.n_i)
    ctx.nb_predict_j(s.t)
    ctx.nb_regular_force(i_idx, r_s, s.t, out=out)  # warm-up outside the capture
    torch.cuda.synchronize()
    ref = {k: v.clone() for k, v in out.items()}
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        ctx.nb_predict_j(s.t)
        ctx.nb_regular_force(i_idx, r_s, s.t, out=out)
    for k in ("acc", "jerk", "nbr_count", "nbr_list"):
        out[k].zero_()
    graph.replay()
    graph.replay()
    torch.cuda.synchronize()
    for k in ("acc", "jerk", "nbr_count", "n_overflow"):
        assert torch.equal(out[k], ref[k]), k
    gpu = {k: v.cpu().numpy() for k, v in out.items()}
    _full_check(oracle, wl, gpu)
    ctx.close()


def test_host_entry_point_in_row_chunks(oracle):
    """nb_regular_force_host splits blocks of more than 16384 rows into row chunks (copy-back overlapped with the
    next chunk): same lists and counts as the device entry point, sums equal to rounding, overflow count summed."""
    wl = _wl(oracle, 2500, 40001, 20, 32)
    wl.r_s[::1000] *= 3.0  # a few overflowing rows in every chunk
    dev_out, _ = run_gpu(wl)
    s = wl.state
    ctx = binding.Context(s.n, wl.n_i, wl.cap)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    out = dict(acc=torch.empty((wl.n_i, 3), dtype=torch.float64).pin_memory(),
               jerk=torch.empty((wl.n_i, 3), dtype=torch.float64).pin_memory(),
               nbr_count=torch.empty(wl.n_i, dtype=torch.int32).pin_memory(),
               nbr_list=torch.full((wl.n_i, wl.cap), -7, dtype=torch.int32).pin_memory(),
               n_overflow=torch.zeros(1, dtype=torch.int32).pin_memory())
    ctx.nb_regular_force_host(pin(s.x0), pin(s.v0), pin(s.a0), pin(s.j0), pin(s.m), pin(s.t0),
                              pin(wl.i_idx.astype(np.int32)), pin(wl.r_s), s.t, out)
    host = {k: v.numpy() for k, v in out.items()}
    assert np.array_equal(host["nbr_count"], dev_out["nbr_count"])
    assert int(host["n_overflow"][0]) == int(dev_out["n_overflow"][0]) >= 40
    ok = dev_out["nbr_count"] <= wl.cap
    for q in np.nonzero(ok)[0][::7]:
        c = dev_out["nbr_count"][q]
        assert np.array_equal(host["nbr_list"][q, :c], dev_out["nbr_list"][q, :c])
    assert parity.relerr(host["acc"], dev_out["acc"]).max() < 1e-6  # two fp32 evaluations, each within ~3e-7 of fp64
    assert parity.relerr(host["jerk"], dev_out["jerk"]).max() < 1e-5
    _full_check(oracle, wl, host)
    ctx.close()


@pytest.mark.parametrize("fuse", [0, 2])
def test_overflowed_split_rows_keep_the_first_cap_in_j_on_request(oracle, fuse):
    """Option "ovf_first_in_j": the list of an overflowed j-split row is rewritten as the first nbr_cap neighbours in
    ascending j (what a row run by one CTA keeps anyway): equal to the head of the oracle's list, and identical in two
    runs.  fuse = 2: the call predicts inside the force kernel, the rewrite predicts what it tests."""
    wl = _wl(oracle, 6000, 200, 20, 32)
    wl.r_s[::7] *= 2.5  # ~300 neighbours > cap 32 on every 7th row
    xp, vp = oracle.predict_state(wl.state)
    _, _, cnt_o, lists_o = oracle.regular_force(xp, vp, wl.state.m, wl.i_idx, wl.r_s, list_stride=1024)
    opts = {"ovf_first_in_j": 1, "i_block": 64, "j_split": 9, "fuse_pred": fuse}
    g1, info = run_gpu(wl, options=opts)
    g2, _ = run_gpu(wl, options=opts)
    assert info["j_chunks"] == 9 and int(g1["n_overflow"][0]) >= 25
    over = np.nonzero(g1["nbr_count"] > wl.cap)[0]
    assert len(over) == int(g1["n_overflow"][0])
    for q in over:
        assert np.array_equal(g1["nbr_list"][q], lists_o[q][: wl.cap]), q      # the first cap in ascending j
        assert np.array_equal(g1["nbr_list"][q], g2["nbr_list"][q])
    assert np.array_equal(g1["nbr_count"], cnt_o)
    _full_check(oracle, wl, g1)
    # ... and with the velocity criterion
    dtr = np.full(wl.n_i, 1.0 / 64)
    g3, _ = run_gpu(wl, options={"ovf_first_in_j": 1, "i_block": 64, "j_split": 9}, dtr=dtr)
    _, _, _, cnt_v, lists_v = oracle.regular_force_ex(xp, vp, wl.state.m, wl.i_idx, wl.r_s, dtr, list_stride=1024)
    for q in np.nonzero(g3["nbr_count"] > wl.cap)[0]:
        assert np.array_equal(g3["nbr_list"][q], lists_v[q][: wl.cap]), q


@pytest.mark.parametrize("n,n_i", [(3001, 257), (2500, 40001), (900, 0)])
def test_host_entry_point_csr_lists(oracle, n, n_i):
    """nb_regular_force_host_csr: the same outputs with the lists packed back to back (CSR), in one chunk and in several
    row chunks (40001 rows: three), overflowing rows cut at cap; too small a buffer is reported with the size needed."""
    wl = _wl(oracle, n, max(n_i, 1), 20, 32)
    if n_i == 0:
        wl = inputs.Workload(wl.state, wl.i_idx[:0].copy(), wl.r_s[:0].copy(), wl.k, wl.cap)
    wl.r_s[::1000] *= 3.0
    s = wl.state
    ctx = binding.Context(s.n, max(wl.n_i, 1), wl.cap)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_in = [pin(a) for a in (s.x0, s.v0, s.a0, s.j0, s.m, s.t0)] + [pin(wl.i_idx.astype(np.int32)), pin(wl.r_s)]
    dense = dict(acc=torch.empty((wl.n_i, 3), dtype=torch.float64), jerk=torch.empty((wl.n_i, 3), dtype=torch.float64),
                 nbr_count=torch.empty(wl.n_i, dtype=torch.int32),
                 nbr_list=torch.full((wl.n_i, wl.cap), -7, dtype=torch.int32), n_overflow=torch.zeros(1, dtype=torch.int32))
    ctx.nb_regular_force_host(*h_in, s.t, dense)
    stored = np.minimum(dense["nbr_count"].numpy(), wl.cap).astype(np.int64)
    total = int(stored.sum())
    csr = dict(acc=torch.empty((wl.n_i, 3), dtype=torch.float64), jerk=torch.empty((wl.n_i, 3), dtype=torch.float64),
               nbr_count=torch.empty(wl.n_i, dtype=torch.int32), nbr_offset=torch.full((wl.n_i + 1,), -1, dtype=torch.int64),
               nbr_packed=torch.full((total + 5,), -7, dtype=torch.int32), n_overflow=torch.zeros(1, dtype=torch.int32))
    ctx.nb_regular_force_host_csr(*h_in, s.t, csr)
    for k in ("acc", "jerk", "nbr_count", "n_overflow"):
        assert torch.equal(csr[k], dense[k]), k
    off = csr["nbr_offset"].numpy()
    assert np.array_equal(off, np.concatenate([[0], np.cumsum(stored)]))
    packed = csr["nbr_packed"].numpy()
    assert np.all(packed[total:] == -7)  # nothing written past the entries
    ref = dense["nbr_list"].numpy()
    cnt = dense["nbr_count"].numpy()
    for q in range(0, wl.n_i, max(1, wl.n_i // 3000)):
        if cnt[q] <= wl.cap:
            assert np.array_equal(packed[off[q]:off[q + 1]], ref[q, : stored[q]])
        else:  # an overflowed j-split row keeps cap of its neighbours, not necessarily the same ones in two runs (R7)
            assert off[q + 1] - off[q] == wl.cap and np.all(np.diff(packed[off[q]:off[q + 1]]) > 0)
    if wl.n_i > 0:  # a buffer that is too small: NB_E_NOMEM, and the offsets say what is needed
        csr["nbr_packed"] = torch.empty(max(total // 2, 1), dtype=torch.int32)
        csr["nbr_offset"].fill_(-1)
        with pytest.raises(binding.NbregError):
            ctx.nb_regular_force_host_csr(*h_in, s.t, csr)
        assert int(csr["nbr_offset"][-1]) == total and torch.equal(csr["nbr_count"], dense["nbr_count"])
    ctx.close()


@pytest.mark.parametrize("n_i", [300, 4096, 4097, 8192, 9001])
def test_row_ordering_paths(oracle, n_i):
    """Rows processed in Morton order of the predicted positions (one-CTA sorts of 512 x 8 and 1024 x 8 rows, device-wide
    sort above 8192): outputs land in the caller's rows; lists and counts identical to the unordered run, sums to rounding."""
    wl = _wl(oracle, 3001, n_i, 24, 64, masses="salpeter")
    wl.i_idx[5] = wl.i_idx[4]  # duplicates keep their own rows
    wl.r_s[5] = wl.r_s[4]
    dtr = (wl.state.t - wl.state.t0[wl.i_idx]) * 4.0
    plain, _ = run_gpu(wl, options={"order_rows": 0}, dtr=dtr, want_pot=True)
    for opts in ({"order_rows": 2}, {"order_rows": 2, "i_block": 32, "j_split": 5}, {"order_rows": 2, "j_split": 1}):
        g, info = run_gpu(wl, options=opts, dtr=dtr, want_pot=True)
        assert np.array_equal(g["nbr_count"], plain["nbr_count"]) and int(g["n_overflow"][0]) == int(plain["n_overflow"][0])
        ok = plain["nbr_count"] <= wl.cap
        for q in np.nonzero(ok)[0][:: max(1, n_i // 500)]:
            c = plain["nbr_count"][q]
            assert np.array_equal(g["nbr_list"][q, :c], plain["nbr_list"][q, :c])
        assert parity.relerr(g["acc"], plain["acc"]).max() < 1e-6
    xp, vp = oracle.predict_state(wl.state)
    parity.compare(oracle, xp, vp, wl.state.m, wl.i_idx, wl.r_s, wl.cap, g, dtr=dtr, check_pot=True)
    parity.check_overflow_flag(g, wl.cap)


@pytest.mark.parametrize("n,n_i", [(5001, 1), (5001, 32), (70001, 64), (70001, 100), (30000, 128), (30000, 129), (30000, 256),
                                  (300001, 100), (900001, 128)])
def test_prediction_fused_into_the_force_kernel_gives_the_same_bits(oracle, n, n_i):
    """A small block (<= 128 rows) predicts inside force_kernel (PRED variant) instead of running the predictor
    first: same records, same pair arithmetic, same row order, identical outputs; checked against the path with the
    predictor pass (option fuse_pred = 0) bit for bit, and against the oracle as usual.  129 and 256 rows keep the pass.
    (900001, 128) runs with the row ordering forced, which then predicts its rows' positions itself."""
    wl = inputs.make_custom(n, n_i, 20, 64, seed_sub=7, predict=lambda s: oracle.predict_state(s)[0])
    s = wl.state
    ctx = binding.Context(s.n, max(n_i, 1), wl.cap)
    ctx.nb_set_option("order_rows", 2 if n == 900001 else 1)
    res = {}
    big = n >= 262144                             # there the default setting (1) fuses by itself
    # Both paths on the SAME launch plan: the fused-prediction kernels hold 24 warps per SM against 28, so the planner
    # may split the j-range differently, and the order in which the chunks' fp64 sums are added decides the last bits.
    ctx.nb_set_option("fuse_pred", 0)
    _, plan = run_gpu(wl, ctx=ctx)
    fixed = {"i_block": plan["rows_per_cta"], "j_split": plan["j_chunks"]}
    for fuse in (2, 0):
        ctx.nb_set_option("fuse_pred", 1 if (fuse and big) else fuse)   # 2: fuse a small block whatever n
        gpu, info = run_gpu(wl, ctx=ctx, options=fixed)  # set_state invalidates the prediction: the call is the fused one
        res[fuse] = (gpu, info)
    ctx.nb_set_option("i_block", 0)
    ctx.nb_set_option("j_split", 0)
    (g1, i1), (g0, i0) = res[2], res[0]
    assert i1["j_chunks"] == i0["j_chunks"] and i1["rows_per_cta"] == i0["rows_per_cta"]
    # predictor, [row ordering: one kernel up to 8192 rows, when the call is long enough], force, gather
    assert i0["launches"] - i1["launches"] == (1 if n_i <= 128 else 0)
    for k in ("acc", "jerk", "nbr_count", "n_overflow"):
        assert np.array_equal(g1[k], g0[k]), k
    for q in range(n_i):
        c = min(g1["nbr_count"][q], wl.cap)
        assert np.array_equal(g1["nbr_list"][q, :c], g0["nbr_list"][q, :c])
    xp, vp = oracle.predict_state(s)
    parity.compare(oracle, xp, vp, s.m, wl.i_idx, wl.r_s, wl.cap, g1)
    # the context holds no prediction after the fused call: a second call at the same time fuses again, and a
    # call that needs the predicted records (velocity criterion) predicts first
    ctx.nb_set_option("fuse_pred", 1)
    g3, i3 = run_gpu(wl, ctx=ctx)
    assert i3["launches"] == (i1["launches"] if big else i0["launches"])   # n < 262144: the predictor pass stays
    ctx.nb_set_option("fuse_pred", 2)
    g2, i2 = run_gpu(wl, ctx=ctx, dtr=np.zeros(n_i))
    assert i2["launches"] == i0["launches"] and np.allclose(g2["acc"], g1["acc"], rtol=1e-5, atol=0)
    ctx.close()


def test_launch_and_copy_options_do_not_change_the_bits(oracle):
    """Options that only change HOW the kernels are launched or what else the predictor writes: "pdl" (programmatic
    dependent launch along the kernel chain) and "gather_copy" (the particle-major copy of the records, written for the
    gathering kernels): identical outputs bit for bit, on a j-split block with the fix-up pass at work."""
    wl = _wl(oracle, 7001, 900, 20, 64, masses="salpeter")
    ref, info = run_gpu(wl)
    assert info["j_chunks"] > 1
    try:
        for opts in ({"pdl": 0}, {"pdl": 1, "gather_copy": 1}, {"pdl": 0, "gather_copy": 1}):
            g, _ = run_gpu(wl, options=opts)
            for k in ("acc", "jerk", "nbr_count", "nbr_list", "n_overflow"):
                assert np.array_equal(g[k], ref[k]), (opts, k)
    finally:  # "pdl" is process-wide: leave it on for the tests that follow
        ctx = binding.Context(16, 16, 8)
        ctx.nb_set_option("pdl", 1)
        ctx.close()
    _full_check(oracle, wl, ref)
