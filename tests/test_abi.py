"""CPU-side checks of the boundary (-m "not gpu"): the shared library loads without a GPU and exports
every function include/cfd.h declares; argument validation that needs no device; independence of the
oracle and the CUDA path (no shared code, neither imports the other)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "cfd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cfd_[a-z0-9_]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_2006_07964_b200 import build

    build.build()
    from paper_2006_07964_b200 import binding

    return binding


def test_header_functions_all_exported(lib):
    names = _declared_functions()
    assert {"cfd_create_blocks", "cfd_compute_metrics", "cfd_rhs", "cfd_rk_stage", "cfd_apply_bc",
            "cfd_exchange_interfaces"} <= set(names)  # the six calls BASELINE.json north_star names
    raw = C.CDLL(lib.LIB_PATH)
    for n in names:
        assert hasattr(raw, n), f"{n} declared in include/cfd.h but not exported"
    assert set(lib.ABI_SYMBOLS) == set(names)


def test_workspace_bytes_is_pure_host_arithmetic(lib):
    d = (lib._Dims * 2)(lib._Dims(32, 32, 32), lib._Dims(10, 20, 30))
    p = lib._Params()
    got = lib.lib.cfd_workspace_bytes(2, d, C.byref(p))
    M = 44 ** 3 + 22 * 32 * 42  # every block has its own 12 M doubles of scratch (blocks run concurrently)
    assert got >= 12 * M * 8
    assert got < 12 * M * 8 + 2 * 16384 * 5 * 8 + (1 << 12)  # + residual partials (16384 CTAs x 5 per block)


def test_no_cuda_device_fails_loudly(lib):
    import torch

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2006_07964_b200 import workloads as W

    case = W.c1_vortex(8)
    with pytest.raises(lib.CfdError):
        lib.Context(case.dims, case.faces, case.params)


def test_oracle_and_cuda_path_share_nothing():
    """Neither side includes / imports the other; no file appears in both trees."""
    csrc = os.path.join(ROOT, "paper_2006_07964_b200")
    orc = os.path.join(ROOT, "oracle")
    for dirpath, _, files in os.walk(csrc):
        for f in files:
            if f.endswith((".cu", ".cuh", ".h", ".py")):
                s = open(os.path.join(dirpath, f)).read()
                assert "oracle_core" not in s and "pyoracle" not in s and "liboracle" not in s, f
                assert not re.search(r"^\s*(from|import)\s+oracle", s, flags=re.M), f
    for f in os.listdir(orc):
        if f.endswith((".cpp", ".hpp", ".py")):
            s = open(os.path.join(orc, f)).read()
            assert "cfd.h" not in s and "cfd_internal" not in s and "libcfd_b200" not in s, f
            assert "paper_2006_07964_b200" not in s.replace("paper_2006_07964_b200/csrc", "").replace(
                "paper_2006_07964_b200/binding.py", ""), f
