"""-m "not gpu": the C-ABI library loads and exports every symbol include/emugemm.h declares; host-only
helpers agree with the oracle; compute calls fail loudly (never fall back) without a GPU."""
import ctypes

import pytest

import paper_2606_25453_b200 as E
from oracle import oracle as O


def test_library_exports_every_declared_symbol():
    lib = E.load_library()
    syms = E.exported_symbols()
    assert len(syms) >= 20
    for s in syms:
        assert hasattr(lib, s), s
    for must in ("emugemm_dgemm_oz1", "emugemm_sgemm_oz1", "emugemm_dgemm_oz2", "emugemm_zgemm_oz2_3m"):
        assert must in syms


def test_probes_build_exports_the_probe_calls_and_the_product_does_not():
    """The experiment switches ("results become WRONG") and probe kernels live only in libemugemm_probes.so."""
    prod, probes = E.load_library(), E.load_library(probes=True)
    extra = sorted(set(E.exported_symbols(probes=True)) - set(E.exported_symbols()))
    assert extra == ["emugemm_dbg_i8_probe", "emugemm_dbg_oz1_issue_probe", "emugemm_dbg_set_flags"]
    for s in E.exported_symbols(probes=True):
        assert hasattr(probes, s), s
    for s in extra:
        assert not hasattr(prod, s), s


def test_host_helpers_match_oracle():
    for N in (2, 12, 14, 16, 18, 20):
        for k in (1, 4096, 8192, 65536):
            assert E.oz2_budget(N, k) == O.oz2_budget(N, k)
            assert E.oz2_budget(N, k, True) == O.oz2_budget(N, k, True)
    # overflow-safe chunk (R7), a multiple of 128.  Sign-magnitude digits (R1): p k_c 127^2 <= 2^31 - 1.  Default two's-complement
    # digits (R24): the leading digit reaches -128, the fullest accumulator sums 2 pairs <= 128 * 127 and p - 2 pairs <= 127^2.
    for p in range(1, 9):
        ck = E.oz1_chunk_k(p, E.DIGITS_SIGN_MAGNITUDE)
        assert ck % 128 == 0 and p * ck * 127 * 127 <= 2 ** 31 - 1 < p * (ck + 128) * 127 * 127
        per_k = 128 * 128 if p == 1 else 2 * 128 * 127 + (p - 2) * 127 * 127
        ck = E.oz1_chunk_k(p)
        assert ck % 128 == 0 and ck * per_k <= 2 ** 31 - 1 < (ck + 128) * per_k
        ck8 = E.oz1_chunk_k(p, 8)
        assert ck8 % 128 == 0 and p * ck8 * 128 * 128 <= 2 ** 31 - 1 < p * (ck8 + 128) * 128 * 128


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    lib = E.load_library()
    h = ctypes.c_void_p()
    st = lib.emugemm_create(ctypes.byref(h))
    assert st == -5  # EMUGEMM_ERR_DEVICE: no silent fallback
    assert lib.emugemm_status_string(st) == b"no sm_100 CUDA device"


def test_workspace_bytes_monotone():
    lib = E.load_library()
    a = lib.emugemm_workspace_bytes(1, 8, 1024, 1024, 1024, 4)
    b = lib.emugemm_workspace_bytes(1, 8, 1024, 1024, 1024, 8)
    c = lib.emugemm_workspace_bytes(2, 8, 1024, 1024, 1024, 16)
    d = lib.emugemm_workspace_bytes(3, 16, 1024, 1024, 1024, 16)
    assert 0 < a < b and c > 0 and d > c
    assert lib.emugemm_workspace_bytes(1, 8, 1024, 1024, 1024, 9) == 0


def test_static_limit_and_chunked_workspace_sizes():
    """Host-only sizing rules: the static-array limit of emugemm_dgemm_oz1_static, the room for balanced Scheme I
    k-chunks (few tiles, long k) and the second output-residue buffer of a k-chunked Scheme II call."""
    lib = E.load_library()
    lib.emugemm_static_workspace_limit.restype = ctypes.c_size_t
    assert lib.emugemm_static_workspace_limit() == 32 << 20
    assert lib.emugemm_workspace_bytes(1, 8, 1024, 1024, 1024, 8) <= 32 << 20 < lib.emugemm_workspace_bytes(1, 8, 1024, 1024, 2176, 8)
    planes = 2 * 7 * 1024 * 65536
    # 1024 x 1024 x 65536, p = 7: both digit modes need 4 overflow-safe chunks (18,944 / 18,688 columns), balanced up to 8
    # partial buffers of 16 MB
    ws = lib.emugemm_workspace_bytes(1, 8, 1024, 1024, 65536, 7)
    assert planes + 8 * 1024 * 1024 * 16 <= ws <= planes + 8 * 1024 * 1024 * 16 + (1 << 20)
    # many tiles: no balancing, the partials stay at the minimum count (p = 8, 8-bit mode: ceil(65536 / 16256) = 5)
    ws_big = lib.emugemm_workspace_bytes(1, 8, 8192, 8192, 65536, 8)
    assert ws_big <= 2 * 8 * 8192 * 65536 + 5 * 8192 * 8192 * 16 + (1 << 20)
    # Scheme II: one set of output residue planes up to k = 130,944, two beyond
    one = lib.emugemm_workspace_bytes(2, 8, 256, 256, 130944, 16) - 2 * 16 * 256 * 130944
    two = lib.emugemm_workspace_bytes(2, 8, 256, 256, 131072, 16) - 2 * 16 * 256 * 131072
    assert 16 * 256 * 256 <= one < 16 * 256 * 256 + (1 << 16)
    assert 2 * 16 * 256 * 256 <= two < 2 * 16 * 256 * 256 + (1 << 16)
