"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol include/semb200.h declares, its
host-only entry point (semb_gll) agrees with the oracle, and compute entry points fail loudly without a CUDA
device (there is no CPU fallback).  No compute call is made."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def semb():
    from paper_2501_13240_b200 import build, semb as S
    build.build()
    S.lib()
    return S


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "semb200.h")).read()
    return sorted(set(re.findall(r"SEMB_API\s+[\w\s\*]+?\b(semb_\w+)\s*\(", text)))


def test_header_symbols_are_all_exported(semb):
    names = declared_symbols()
    assert len(names) >= 20, names
    L = semb.lib()
    for nme in names:
        assert hasattr(L, nme), f"{nme} is declared in include/semb200.h but not exported by libsemb200.so"
    # the binding's own list is the header's list
    assert sorted(semb.SYMBOLS) == names


def test_no_torch_types_in_the_abi():
    text = open(os.path.join(ROOT, "include", "semb200.h")).read()
    code = re.sub(r"/\*.*?\*/", "", text, flags=re.S)          # comments may mention torch's allocator
    assert "torch" not in code.lower() and "at::" not in code and "#include <cuda" not in code
    assert 'extern "C"' in text


def test_version_names_the_target(semb):
    assert "sm_100a" in semb.version() and "fp64" in semb.version()


@pytest.mark.parametrize("N", [1, 2, 3, 5, 7, 9, 10])
def test_gll_host_entry_point_against_oracle(semb, orc, N):
    """semb_gll (long-double Newton on P_{N+1} - P_{N-1}, barycentric D) vs the oracle (fp64 Newton on P'_N,
    closed-form D): two independent constructions of the same basis."""
    xi, rho, D = semb.gll(N)
    oxi, orho = orc.gll(N)
    oD = orc.dhat(N)
    assert np.abs(xi - oxi).max() <= 4e-16
    assert np.abs(rho - orho).max() <= 1e-15
    assert np.abs(D - oD).max() <= 2e-13 * np.abs(oD).max()
    assert np.all(D.sum(axis=1) == 0.0) or np.abs(D.sum(axis=1)).max() <= 1e-14   # reading R2
    # centro-antisymmetry, which the even-odd contractions of the axhelm kernel rely on
    assert np.abs(D + D[::-1, ::-1]).max() <= 1e-14 * np.abs(D).max()


def test_gll_rejects_bad_order(semb):
    L = semb.lib()
    buf = np.zeros(200)
    p = buf.ctypes.data_as(C.c_void_p)
    assert L.semb_gll(C.c_int(0), p, p, p) == -1
    assert L.semb_gll(C.c_int(11), p, p, p) == -1


def test_setup_fails_loudly_without_a_device(semb):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    L = semb.lib()
    h = C.c_void_p()
    x = np.zeros(8); ft = np.zeros(6, dtype=np.int32); per = np.zeros(3)
    p = x.ctypes.data_as(C.c_void_p)
    rc = L.semb_setup(C.c_int64(1), C.c_int(1), p, p, p, ft.ctypes.data_as(C.c_void_p), per.ctypes.data_as(C.c_void_p),
                      None, None, None, C.byref(h))
    assert rc == -3 and not h.value                      # SEMB_ECUDA, no handle
    assert b"no CUDA device" in L.semb_last_error(None)
    # bad arguments are rejected before anything else
    assert L.semb_setup(C.c_int64(0), C.c_int(1), p, p, p, None, None, None, None, None, C.byref(h)) == -1
    assert L.semb_export_field(None, b"temperature", None) < 0


def test_bench_byte_model_matches_the_survey():
    """bench.py's per-iteration byte model: 171.6 B/node at N = 7, 169.8 at N = 9."""
    import importlib.util
    import os
    spec = importlib.util.spec_from_file_location("bench", os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "bench.py"))
    bench = importlib.util.module_from_spec(spec); spec.loader.exec_module(bench)
    assert abs(bench.model_bytes_per_iteration(7) - 171.6) < 0.05 and abs(bench.model_bytes_per_iteration(9) - 169.8) < 0.05
    assert bench.B_ITER == 171.6 and bench.B_AXHELM == 64.0 and bench.B_AXHELM_HELM == 72.0 and bench.B_AXHELM_PCG == 104.0
