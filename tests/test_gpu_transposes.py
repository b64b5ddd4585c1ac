"""-m gpu: transposed operands (emugemm_*_t): op(A) op(B) for all four flag combinations equals the oracle run
on explicitly transposed copies (numpy transposition: independent of the CUDA path).  Integer stages are shared
with the untransposed path, so the check is on the final values (2 ulp) plus bit-identity between the four
storage variants of the same mathematical operands."""
import numpy as np
import pytest

import emugemm_inputs as G
from gpu_util import assert_within_ulps

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import oracle as O
    import paper_2606_25453_b200 as E
    h = E.EmuGemm()
    yield torch, O, h
    h.close()


def dev(torch, x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("scheme,pn", [("oz1", 5), ("oz1", 3), ("oz2", 14)])
def test_real_all_flag_combinations(env, scheme, pn):
    torch, O, h = env
    m, n, k = 200, 136, 333
    A, B = G.real_pair(m, n, k, 1.0, 12)
    want = O.dgemm_oz1(A, B, pn) if scheme == "oz1" else O.dgemm_oz2(A, B, pn)
    _, absAB = O.bf128_dgemm(A, B)
    call = h.dgemm_oz1 if scheme == "oz1" else h.dgemm_oz2
    outs = []
    for ta in (False, True):
        for tb in (False, True):
            Ad = dev(torch, A.T if ta else A)
            Bd = dev(torch, B.T if tb else B)
            C = torch.full((m, n), float("nan"), dtype=torch.float64, device="cuda")
            call(Ad, Bd, C, pn, transa=ta, transb=tb)
            got = C.cpu().numpy()
            assert_within_ulps(got, want, absAB, 2, what=f"{scheme} ta={ta} tb={tb}")
            outs.append(got)
    for o in outs[1:]:
        assert np.array_equal(o, outs[0])  # same digits / residues whatever the storage order


def test_sgemm_and_complex_transposed(env):
    torch, O, h = env
    m, n, k = 130, 70, 260
    A, B = G.real_pair(m, n, k, 1.0, 4, dtype=np.float32)
    C = torch.zeros((m, n), dtype=torch.float32, device="cuda")
    h.sgemm_oz1(dev(torch, A.T), dev(torch, B.T), C, 4, transa=True, transb=True)
    _, ab = O.bf128_dgemm(A.astype(np.float64), B.astype(np.float64))
    assert_within_ulps(C.cpu().numpy(), O.sgemm_oz1(A, B, 4), ab, 2, bits=23, what="sgemm TT")
    Az, Bz = G.complex_pair(100, 64, 128, 1.0, 8)
    Cz = torch.zeros((100, 64), dtype=torch.complex128, device="cuda")
    h.zgemm_oz2_3m(dev(torch, Az.T), dev(torch, Bz), Cz, 14, transa=True)
    wantz = O.zgemm_oz2_3m(Az, Bz, 14)
    _, absZ = O.bf128_zgemm(Az, Bz)
    got = Cz.cpu().numpy()
    assert_within_ulps(got.real, wantz.real, absZ, 2, what="3M T re")
    assert_within_ulps(got.imag, wantz.imag, absZ, 2, what="3M T im")


def test_column_major_call_is_swapped_row_major_call(env):
    """Column-major C = A B (BLAS convention) == row-major C^T = B^T A^T on the same buffers."""
    torch, O, h = env
    m, n, k, p = 96, 150, 200, 6
    A, B = G.real_pair(m, n, k, 1.0, 3)
    A_cm, B_cm = dev(torch, A.T), dev(torch, B.T)          # column-major storage of A (m x k) and B (k x n)
    C_cm = torch.zeros((n, m), dtype=torch.float64, device="cuda")  # column-major m x n == row-major n x m
    # row-major view: C^T (n x m) = B^T (n x k, stored as is) * A^T (k x m, stored as is)
    h.dgemm_oz1(B_cm, A_cm, C_cm, p)
    want = O.dgemm_oz1(np.ascontiguousarray(B.T), np.ascontiguousarray(A.T), p)
    _, absAB = O.bf128_dgemm(np.ascontiguousarray(B.T), np.ascontiguousarray(A.T))
    assert_within_ulps(C_cm.cpu().numpy(), want, absAB, 2, what="column-major")


def test_bad_flags(env):
    import ctypes as C
    torch, O, h = env
    A = torch.zeros((16, 16), dtype=torch.float64, device="cuda")
    i64, dbl, vp = C.c_int64, C.c_double, C.c_void_p
    st = h._lib.emugemm_dgemm_oz1_t(h._h, C.c_int(2), C.c_int(0), i64(16), i64(16), i64(16), dbl(1.0), vp(A.data_ptr()), i64(16),
                                    vp(A.data_ptr()), i64(16), dbl(0.0), vp(A.data_ptr()), i64(16), C.c_int(4))
    assert st == -1
