"""The C-ABI library loads on a CPU-only box and exports every symbol include/nbreg.h declares."""
import ctypes
import os
import re

from paper_1205_1222_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "nbreg.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(nb_[a-z_]+)\s*\(", src)))


def test_header_symbols_are_exported():
    lib = binding.load()
    names = _declared()
    assert {"nb_predict_j", "nb_regular_force", "nb_create", "nb_destroy", "nb_set_j"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in nbreg.h but not exported by libnbreg.so"


def test_host_side_logic_without_gpu():
    lib = binding.load()
    assert lib.nb_version() >= 100
    assert lib.nb_workspace_bytes(0, 1, 1) == 0 and lib.nb_workspace_bytes(10, 1, 0) == 0
    small, big = lib.nb_workspace_bytes(1024, 1024, 128), lib.nb_workspace_bytes(1 << 20, 1 << 20, 512)
    assert 1024 * 40 <= small < big
    assert big >= (1 << 20) * 40
    assert lib.nb_strerror(0) == b"ok" and b"invalid" in lib.nb_strerror(-1)
    # null / bad arguments are rejected before any CUDA call
    assert lib.nb_create(None, 0, 10, 10, 8, None, 0) == -1
    h = ctypes.c_void_p()
    assert lib.nb_create(ctypes.byref(h), 0, 0, 10, 8, None, 0) == -1
    assert lib.nb_destroy(None) == 0
    assert lib.nb_set_option(None, b"j_split", 1) == -1


def test_static_entry_point_limits_are_checked_before_any_cuda_call():
    """nb_regular_force_static (scratch in a fixed 8 MiB device array of the library) rejects sizes beyond its limits with
    NB_E_LIMIT and a text that names the entry point -- on a box without a GPU too."""
    lib = binding.load()
    assert binding.nb_static_limits() == dict(n=65536, n_i=4096, nbr_cap=512, scratch_bytes=8 << 20)
    one = ctypes.c_int32(0)
    p = ctypes.cast(ctypes.pointer(one), ctypes.c_void_p)
    call = lambda n, n_i, cap: lib.nb_regular_force_static(0, n, p, p, p, p, p, p, n_i, p, p, 1.0, cap, p, p, p, p, p, None)
    for args in ((65537, 1, 8), (100, 4097, 8), (100, 1, 513)):
        rc = call(*args)
        assert rc == -5 and b"nb_regular_force_static" in lib.nb_strerror(rc)
    assert call(0, 1, 8) == -1 and call(100, -1, 8) == -1 and call(100, 1, 0) == -1


def test_binding_fails_loudly_without_cuda():
    import pytest
    import torch

    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(binding.NbregError):
        binding.Context(16, 16, 8)
