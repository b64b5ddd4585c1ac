"""-m gpu: pre-decomposed operands (emugemm_decompose + emugemm_gemm_pre):
bit-identical to the one-shot calls, an operand decomposed once is reused against several partners, and the results
match the ORACLE on the same inputs (2 ulp of (|A||B|)_ij), including transposed-storage operands."""
import numpy as np
import pytest

import emugemm_inputs as G
from gpu_util import assert_within_ulps

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    import paper_2606_25453_b200 as E
    h = E.EmuGemm()
    yield torch, E, h
    h.close()


def dev(torch, x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("p,bits", [(6, 7), (3, 7), (7, 8)])
def test_oz1_reuse_bit_identical(env, p, bits):
    torch, E, h = env
    h.set_slice_bits(bits)
    try:
        m, n, k = 200, 136, 333
        A, B1 = G.real_pair(m, n, k, 1.0, 12)
        _, B2 = G.real_pair(m, n, k, 1.0, 13)
        Ad = dev(torch, A)
        opA = h.decompose(E.OZ1, 0, Ad, p)
        for B in (B1, B2):
            Bd = dev(torch, B)
            opB = h.decompose(E.OZ1, 1, Bd, p)
            C1 = torch.zeros((m, n), dtype=torch.float64, device="cuda")
            C2 = torch.zeros((m, n), dtype=torch.float64, device="cuda")
            h.gemm_pre(opA, opB, C1, alpha=1.25)
            h.dgemm_oz1(Ad, Bd, C2, p, alpha=1.25)
            assert torch.equal(C1, C2)
        # transposed storage of the right operand decomposes to the same planes
        opBt = h.decompose(E.OZ1, 1, dev(torch, B2.T), p, trans=True)
        C3 = torch.zeros((m, n), dtype=torch.float64, device="cuda")
        h.gemm_pre(opA, opBt, C3, alpha=1.25)
        assert torch.equal(C3, C2)
    finally:
        h.set_slice_bits(7)


def test_oz2_and_3m_bit_identical(env):
    torch, E, h = env
    m, n, k, N = 130, 260, 300, 14
    A, B = G.real_pair(m, n, k, 1.0, 2)
    Ad, Bd = dev(torch, A), dev(torch, B)
    opA, opB = h.decompose(E.OZ2, 0, Ad, N), h.decompose(E.OZ2, 1, Bd, N)
    C1 = torch.zeros((m, n), dtype=torch.float64, device="cuda")
    C2 = torch.zeros((m, n), dtype=torch.float64, device="cuda")
    h.gemm_pre(opA, opB, C1)
    h.dgemm_oz2(Ad, Bd, C2, N)
    assert torch.equal(C1, C2)
    Az, Bz = G.complex_pair(100, 64, 128, 1.0, 8)
    Azd, Bzd = dev(torch, Az), dev(torch, Bz)
    oa, ob = h.decompose(E.OZ2_3M, 0, Azd, N), h.decompose(E.OZ2_3M, 1, Bzd, N)
    Z1 = torch.zeros((100, 64), dtype=torch.complex128, device="cuda")
    Z2 = torch.zeros((100, 64), dtype=torch.complex128, device="cuda")
    h.gemm_pre(oa, ob, Z1, alpha=0.5 - 2j)
    h.zgemm_oz2_3m(Azd, Bzd, Z2, N, alpha=0.5 - 2j)
    assert torch.equal(Z1, Z2)


def test_mismatched_operands_rejected(env):
    torch, E, h = env
    A, B = G.real_pair(64, 64, 128, 1.0, 1)
    opA = h.decompose(E.OZ1, 0, dev(torch, A), 4)
    opB5 = h.decompose(E.OZ1, 1, dev(torch, B), 5)
    Cc = torch.zeros((64, 64), dtype=torch.float64, device="cuda")
    with pytest.raises(E.EmuGemmError) as ei:
        h.gemm_pre(opA, opB5, Cc)
    assert ei.value.status == -1
    with pytest.raises(E.EmuGemmError):
        h.gemm_pre(opA, opA, Cc)  # two left operands


@pytest.mark.parametrize("transa,transb", [(False, False), (True, False), (False, True), (True, True)])
def test_oz1_operands_against_oracle(env, transa, transb):
    """emugemm_decompose with either storage of either operand, then emugemm_gemm_pre, against oracle_dgemm_oz1."""
    torch, E, h = env
    from oracle import oracle as O
    m, n, k, p = 150, 200, 260, 6
    A, B, Cin = G.real_pair(m, n, k, 1.0, 31, with_c=True)
    opA = h.decompose(E.OZ1, 0, dev(torch, A.T if transa else A), p, trans=transa)
    opB = h.decompose(E.OZ1, 1, dev(torch, B.T if transb else B), p, trans=transb)
    C = dev(torch, Cin)
    h.gemm_pre(opA, opB, C, alpha=-0.75, beta=1.5)
    want = O.dgemm_oz1(A, B, p, alpha=-0.75, beta=1.5, Cin=Cin)
    _, absAB = O.bf128_dgemm(A, B)
    assert_within_ulps(C.cpu().numpy(), want, 0.75 * absAB + 1.5 * np.abs(Cin), 2, what=f"operands oz1 {transa} {transb}")


@pytest.mark.parametrize("transa,transb", [(False, False), (True, True)])
def test_oz2_operands_against_oracle(env, transa, transb):
    torch, E, h = env
    from oracle import oracle as O
    m, n, k, N = 130, 140, 300, 15
    A, B = G.real_pair(m, n, k, 1.0, 32)
    opA = h.decompose(E.OZ2, 0, dev(torch, A.T if transa else A), N, trans=transa)
    opB = h.decompose(E.OZ2, 1, dev(torch, B.T if transb else B), N, trans=transb)
    C = torch.full((m, n), float("nan"), dtype=torch.float64, device="cuda")
    h.gemm_pre(opA, opB, C)
    _, absAB = O.bf128_dgemm(A, B)
    assert_within_ulps(C.cpu().numpy(), O.dgemm_oz2(A, B, N), absAB, 2, what=f"operands oz2 {transa} {transb}")


def test_3m_operands_against_oracle(env):
    torch, E, h = env
    from oracle import oracle as O
    m, n, k, N = 90, 70, 200, 14
    A, B = G.complex_pair(m, n, k, 1.0, 33)
    oa = h.decompose(E.OZ2_3M, 0, dev(torch, A), N)
    ob = h.decompose(E.OZ2_3M, 1, dev(torch, B.T), N, trans=True)
    Z = torch.zeros((m, n), dtype=torch.complex128, device="cuda")
    h.gemm_pre(oa, ob, Z, alpha=0.5 - 2j)
    want = O.zgemm_oz2_3m(A, B, N, alpha=0.5 - 2j)
    _, absZ = O.bf128_zgemm(A, B)
    got = Z.cpu().numpy()
    scale = abs(0.5 - 2j) * 2 * absZ
    assert_within_ulps(got.real, want.real, scale, 2, what="operands 3M re")
    assert_within_ulps(got.imag, want.imag, scale, 2, what="operands 3M im")
