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


def test_binding_fails_loudly_without_cuda():
    import pytest
    import torch

    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(binding.NbregError):
        binding.Context(16, 16, 8)
