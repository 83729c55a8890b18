"""The C ABI without a GPU: liblcs_b200.so builds (nvcc cross-compiles sm_100a), loads, exports every entry point that
include/lcs.h declares, and its host-side argument checks answer as the header says.  No compute call is made."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_in_header():
    text = open(os.path.join(ROOT, "include", "lcs.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)           # comments mention function names too
    return sorted(set(re.findall(r"\b(lcs_[a-z0-9_]+)\s*\(", text)))


@pytest.fixture(scope="module")
def lib():
    import paper_2604_11008_b200 as pkg
    return pkg.load_library(build_if_missing=True)


def test_every_declared_entry_point_is_exported(lib):
    import paper_2604_11008_b200 as pkg
    names = declared_in_header()
    assert len(names) >= 18
    for n in names:
        assert getattr(lib, n) is not None, n
    assert sorted(pkg.EXPORTED_SYMBOLS) == names                 # the binding and the header list the same calls


def test_version_and_workspace_size_checks(lib):
    from paper_2604_11008_b200.binding import LcsParams
    assert b"sm_100a" in lib.lcs_version()
    prm = LcsParams(1.5e-5, 1000.0, (C.c_double * 3)(0, 0, 0), 0, 0, 0)
    ok = lib.lcs_workspace_bytes(32, 2, 2, 2, 4096, C.byref(prm))
    assert ok > 8 * 8 * 4096 * 8                                 # at least the eight slabs
    prm_rk2 = LcsParams(1.5e-5, 1000.0, (C.c_double * 3)(0, 0, 0), 0, 0, 1)
    assert lib.lcs_workspace_bytes(32, 2, 2, 2, 4096, C.byref(prm_rk2)) >= ok + 8 * 8 * 4096 * 8   # + the RK2 group
    assert lib.lcs_workspace_bytes(1623, 1, 1, 1, 4096, C.byref(prm)) > 1625 ** 3 * 32          # 1625^3 records < 2^32
    bad = [
        (33, 2, 2, 2, 4096, prm),                                # N not divisible by Px
        (1, 1, 1, 1, 4096, prm),                                 # N < 2
        (32, 2, 2, 2, 4095, prm),                                # odd capacity
        (32, 2, 2, 2, 0, prm),                                   # no capacity
        (2048, 2, 2, 2, 4096, prm),                              # N > 1625 (32-bit record indices)
        (1624, 1, 1, 1, 4096, prm),                              # one brick of 1626^3 records >= 2^32 (1623 is the limit)
        (1616, 8, 8, 8, 4096, prm),                              # 512 bricks of 204^3 records >= 2^32
        (32, 2, 2, 2, 1 << 31, prm),                             # capacity beyond 2^31 - 1
        (32, 2, 2, 2, 1 << 28, prm),                             # P * capacity = 2^31: slot indices and copy coordinates
        (32, 2, 2, 2, 4096, LcsParams(0.0, 1000.0, (C.c_double * 3)(0, 0, 0), 0, 0, 0)),        # nu <= 0
        (32, 2, 2, 2, 4096, LcsParams(1.5e-5, 1000.0, (C.c_double * 3)(0, 0, 0), 0, 2, 0)),     # unknown drag model
        (32, 2, 2, 2, 4096, LcsParams(1.5e-5, 1000.0, (C.c_double * 3)(0, 0, 0), 4098, 0, 0)),  # send region > capacity
    ]
    for N, px, py, pz, cap, p in bad:
        assert lib.lcs_workspace_bytes(N, px, py, pz, cap, C.byref(p)) == 0, (N, px, py, pz, cap)
    assert lib.lcs_workspace_bytes(32, 2, 2, 2, 4096, None) == 0


def test_staging_size_formula(lib):
    """lcs_staging_bytes is what lcs_step_fused_host checks against: eight arrays of n words, each rounded up to 256
    bytes, plus the P counts rounded up to 256 bytes (include/lcs.h)."""
    up = lambda v: (v + 255) // 256 * 256
    lib.lcs_staging_bytes.restype = C.c_size_t
    lib.lcs_staging_bytes.argtypes = [C.c_int64, C.c_int]
    for n, P in ((0, 1), (1, 8), (30011, 8), (1 << 26, 512)):
        assert lib.lcs_staging_bytes(n, P) == 8 * up(8 * n) + up(8 * P)
    assert lib.lcs_staging_bytes(-1, 8) == 0 and lib.lcs_staging_bytes(10, 0) == 0


def test_null_handles_are_rejected(lib):
    from paper_2604_11008_b200 import LCS_ERR_INVALID_ARG
    for name in ("lcs_destroy", "lcs_migrate", "lcs_migrate_sweeps"):
        assert getattr(lib, name)(None) == LCS_ERR_INVALID_ARG, name
    assert lib.lcs_step_fused(None, 0.1) == LCS_ERR_INVALID_ARG
    assert lib.lcs_step_rk2(None, 0.1) == LCS_ERR_INVALID_ARG
    assert lib.lcs_particle_step(None, 0.1) == LCS_ERR_INVALID_ARG


def test_the_binding_has_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2604_11008_b200 import LCS
    with pytest.raises(Exception):
        LCS(32, 2, 2, 2, 4096)
