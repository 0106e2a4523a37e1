"""Host-side launch planner of the C ABI (nb_plan): CPU only.

The planner decides the CTA shape, which row blocks run the whole j-range in one CTA and how the remaining
("tail") row blocks are split along j so that the CTA count fills whole waves of the SMs.
These tests check its invariants, not a particular tuning.
"""
import itertools

import pytest

from paper_1205_1222_b200 import binding

OCC = (3, 6, 12, 24, 1)  # CTAs per SM of the shapes 256, 128, 64, 32, 512 rows (what a B200 reports)
SHAPE = {256: 0, 128: 1, 64: 2, 32: 3, 512: 4}


def _check_plan(p, n, n_i):
    rows = p["rows_per_cta"]
    n_pad = (n + 255) // 256 * 256
    n_blocks = -(-n_i // rows)
    tail, S = p["split_row_blocks"], p["j_chunks"]
    assert 0 <= tail <= n_blocks and S >= 1
    assert (S == 1) == (tail == 0)
    assert p["ctas"] == (n_blocks - tail) + tail * S
    assert tail * rows * S <= min(max(256 * n_i, 131072), 2097152)  # (row, chunk) slots of the j-split workspace
    if S > 1:  # equal chunks (a multiple of 4 particles, not of the tile) cover the j-range exactly, none is empty
        cj = p["chunk_j"]
        assert cj % 4 == 0 and cj >= 64 and (S - 1) * cj < n_pad <= S * cj
    return n_blocks


@pytest.mark.parametrize("n,n_i", [(1024, 1024), (16384, 2048), (200000, 8192), (1048576, 1048576), (2999, 777),
                                   (65536, 1), (300, 300), (1 << 20, 3)] + [(65536, 2 ** e) for e in range(5, 17)])
def test_plan_invariants(n, n_i):
    p = binding.nb_plan(n, n_i, 148, OCC)
    _check_plan(p, n, n_i)
    assert p["ctas_per_sm"] == OCC[SHAPE[p["rows_per_cta"]]]


def test_full_waves_run_unsplit_and_the_tail_fills_the_last_wave():
    # config 5: 4096 blocks of 256 rows on 444 slots = 9 full waves + 100 blocks; those are j-split
    p = binding.nb_plan(1 << 20, 1 << 20, 148, OCC)
    slots = 148 * p["ctas_per_sm"]
    n_blocks = _check_plan(p, 1 << 20, 1 << 20)
    assert p["split_row_blocks"] == n_blocks % slots
    # modelled time (in j per CTA slot) within 4 % of a perfectly balanced machine
    n_pad = 1 << 20
    waves_tail = -(-p["split_row_blocks"] * p["j_chunks"] // slots)
    modelled = (n_blocks // slots) * n_pad + waves_tail * p["chunk_j"]
    assert modelled <= 1.04 * n_blocks * n_pad / slots
    # an exact multiple of the slots needs no split at all
    q = binding.nb_plan(1 << 20, 444 * 256, 148, OCC, i_block=256)
    assert q["j_chunks"] == 1 and q["split_row_blocks"] == 0 and q["ctas"] == 444


def test_small_blocks_are_split_to_fill_the_machine():
    for n_i in (32, 64, 128, 256, 512):
        p = binding.nb_plan(65536, n_i, 148, OCC)
        _check_plan(p, 65536, n_i)
        assert p["j_chunks"] > 1
        assert p["ctas"] >= 148  # at least one CTA per SM
    # ... but no chunk shorter than 64 particles
    p = binding.nb_plan(300, 32, 148, OCC)
    assert p["j_chunks"] <= 512 // 64


def test_forced_options_are_honoured():
    for ib, sp in itertools.product((32, 64, 128, 256, 512), (1, 3, 7)):
        p = binding.nb_plan(2999, 777, 148, OCC, i_block=ib, j_split=sp)
        assert p["rows_per_cta"] == ib
        cj = max(64, -(-(-(-3072 // sp)) // 4) * 4)   # equal chunks, a multiple of 4 particles, at least 64
        want = -(-3072 // cj)                          # ... none empty
        assert p["j_chunks"] == want and (want == 1 or p["split_row_blocks"] == -(-777 // ib))
        _check_plan(p, 2999, 777)
    lib = binding.load()
    import ctypes
    info = (ctypes.c_int64 * 8)()
    occ = (ctypes.c_int32 * 5)(*OCC)
    assert lib.nb_plan(0, 1, 148, occ, 0, 0, info) == -1
    assert lib.nb_plan(10, 1, 148, occ, 48, 0, info) == -1
    assert lib.nb_plan(10, 1, 148, None, 0, 0, info) == -1


def test_plan_depends_on_machine_size():
    a = binding.nb_plan(65536, 4096, 148, OCC)
    b = binding.nb_plan(65536, 4096, 16, OCC)
    assert a["ctas"] > b["ctas"] or a["j_chunks"] >= b["j_chunks"]


@pytest.mark.parametrize("n", [65536, 1 << 20])
def test_shapes_much_taller_than_the_block_are_left_out(n):
    """A CTA shape at least twice as tall as the whole active block would compute rows that do not exist."""
    for n_i in (1, 7, 32):
        assert binding.nb_plan(n, n_i, 148, OCC)["rows_per_cta"] == 32
    for n_i in (33, 64):
        assert binding.nb_plan(n, n_i, 148, OCC)["rows_per_cta"] <= 64
    for n_i in (65, 128):
        assert binding.nb_plan(n, n_i, 148, OCC)["rows_per_cta"] <= 128
    assert binding.nb_plan(n, 64, 148, OCC, i_block=256)["rows_per_cta"] == 256   # a forced shape is obeyed
