"""-m gpu parity tests, Scheme II and 3M: residues and per-modulus output residues bit-exact, final
FP64 within 2 ulp of (|A||B|)_ij against the oracle."""
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
    yield torch, O, h, E
    h.close()


def dev(torch, x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def test_budget_matches_oracle(env):
    torch, O, h, E = env
    for N in (2, 8, 12, 14, 16, 18, 20):
        for k in (1, 100, 4096, 8192, 100000):
            for is3m in (False, True):
                assert E.oz2_budget(N, k, is3m) == O.oz2_budget(N, k, is3m)


@pytest.mark.parametrize("N", [2, 12, 20])
def test_residues_bit_exact(env, N):
    torch, O, h, E = env
    m, n, k = 130, 70, 333
    A, B = G.real_pair(m, n, k, 1.0, 2)
    A[0, 0] = 0.0
    _, tA, tB = O.oz2_budget(N, k)
    RA, eA = h.dbg_oz2_residues(dev(torch, A), False, N, tA)
    RB, eB = h.dbg_oz2_residues(dev(torch, B), True, N, tB)
    oA, oB = O.row_exponents(A), O.col_exponents(B)
    assert np.array_equal(eA.cpu().numpy(), oA) and np.array_equal(eB.cpu().numpy(), oB)
    assert np.array_equal(RA.cpu().numpy(), O.oz2_residues_rows(A, oA, tA, N))
    assert np.array_equal(RB.cpu().numpy(), O.oz2_residues_cols(B, oB, tB, N))


def test_residues_complex_bit_exact(env):
    torch, O, h, E = env
    N, m, n, k = 18, 70, 90, 200
    A, B = G.complex_pair(m, n, k, 1.0, 3)
    _, tA, tB = O.oz2_budget(N, k, True)
    RA, eA = h.dbg_oz2_residues(dev(torch, A), False, N, tA)
    RB, eB = h.dbg_oz2_residues(dev(torch, B), True, N, tB)
    oA, oB = O.row_exponents_z(A), O.col_exponents_z(B)
    assert np.array_equal(RA.cpu().numpy(), O.oz2_residues_z(A, oA, tA, N, False))
    assert np.array_equal(RB.cpu().numpy(), O.oz2_residues_z(B, oB, tB, N, True))


@pytest.mark.parametrize("shape", [(256, 512, 256), (200, 300, 333)])
def test_modgemm_bit_exact(env, shape):
    """fused mod-reduction epilogue: extreme residues (+-127/-128) so the INT32 range is exercised."""
    torch, O, h, E = env
    m, n, k = shape
    N = 6
    rng = np.random.default_rng(0)
    RA = rng.integers(-128, 128, size=(N, m, k)).astype(np.int8)
    RB = rng.integers(-128, 128, size=(N, n, k)).astype(np.int8)
    RA[1, :8, :] = 127; RB[1, :8, :] = 127; RA[0, 8:16, :] = -128; RB[0, :8, :] = -128
    got = h.dbg_oz2_modgemm(dev(torch, RA), dev(torch, RB)).cpu().numpy()
    want, _, _ = O.oz2_modprod(RA, RB)
    assert np.array_equal(got, want)


def test_modgemm_3m_bit_exact(env):
    torch, O, h, E = env
    N, m, n, k = 4, 200, 300, 256
    A, B = G.complex_pair(m, n, k, 1.0, 3)
    _, tA, tB = O.oz2_budget(N, k, True)
    RA3 = O.oz2_residues_z(A, O.row_exponents_z(A), tA, N, False)
    RB3 = O.oz2_residues_z(B, O.col_exponents_z(B), tB, N, True)
    got = h.dbg_oz2_modgemm(dev(torch, RA3), dev(torch, RB3), is3m=True).cpu().numpy()
    assert np.array_equal(got, O.oz2_modprod_3m(RA3, RB3))


@pytest.mark.parametrize("N", [8, 12, 16, 20])
def test_crt_alone(env, N):
    torch, O, h, E = env
    m, n, k = 96, 100, 128
    A, B = G.real_pair(m, n, k, 1.0, N)
    _, tA, tB = O.oz2_budget(N, k)
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    CR, _, _ = O.oz2_modprod(O.oz2_residues_rows(A, eA, tA, N), O.oz2_residues_cols(B, eB, tB, N))
    C = torch.zeros((m, n), dtype=torch.float64, device="cuda")
    h.dbg_oz2_crt(dev(torch, CR), dev(torch, eA), dev(torch, eB), tA, tB, C)
    _, absAB = O.bf128_dgemm(A, B)
    assert_within_ulps(C.cpu().numpy(), O.oz2_crt(CR, eA, eB, tA, tB), absAB, 2, what=f"crt N={N}")


@pytest.mark.parametrize("N,shape", [(12, (256, 256, 256)), (14, (200, 300, 333)), (16, (129, 513, 140)), (18, (384, 256, 512)),
                                     (20, (130, 70, 1000))])
def test_dgemm_oz2(env, N, shape):
    torch, O, h, E = env
    m, n, k = shape
    A, B = G.real_pair(m, n, k, 1.0, 2)
    C = torch.full((m, n), float("nan"), dtype=torch.float64, device="cuda")
    h.dgemm_oz2(dev(torch, A), dev(torch, B), C, N)
    _, absAB = O.bf128_dgemm(A, B)
    assert_within_ulps(C.cpu().numpy(), O.dgemm_oz2(A, B, N), absAB, 2, what=f"oz2 N={N}")


def test_dgemm_oz2_alpha_beta(env):
    torch, O, h, E = env
    m, n, k, N = 140, 90, 260, 14
    A, B, Cin = G.real_pair(m, n, k, 1.0, 6, with_c=True)
    C = dev(torch, Cin)
    h.dgemm_oz2(dev(torch, A), dev(torch, B), C, N, alpha=2.5, beta=-0.5)
    _, absAB = O.bf128_dgemm(A, B)
    assert_within_ulps(C.cpu().numpy(), O.dgemm_oz2(A, B, N, alpha=2.5, beta=-0.5, Cin=Cin), 2.5 * absAB + 0.5 * np.abs(Cin), 2)


@pytest.mark.parametrize("N,shape", [(14, (256, 256, 256)), (18, (150, 270, 333))])
def test_zgemm_oz2_3m(env, N, shape):
    torch, O, h, E = env
    m, n, k = shape
    A, B = G.complex_pair(m, n, k, 1.0, 3)
    C = torch.zeros((m, n), dtype=torch.complex128, device="cuda")
    h.zgemm_oz2_3m(dev(torch, A), dev(torch, B), C, N)
    want = O.zgemm_oz2_3m(A, B, N)
    _, absZ = O.bf128_zgemm(A, B)
    got = C.cpu().numpy()
    assert_within_ulps(got.real, want.real, absZ, 2, what="3M re")
    assert_within_ulps(got.imag, want.imag, absZ, 2, what="3M im")


def test_zgemm_alpha_beta(env):
    torch, O, h, E = env
    m, n, k, N = 100, 64, 128, 14
    A, B, Cin = G.complex_pair(m, n, k, 1.0, 8, with_c=True)
    C = dev(torch, Cin)
    al, be = 0.5 - 2j, 1.5 + 0.25j
    h.zgemm_oz2_3m(dev(torch, A), dev(torch, B), C, N, alpha=al, beta=be)
    want = O.zgemm_oz2_3m(A, B, N, alpha=al, beta=be, Cin=Cin)
    _, absZ = O.bf128_zgemm(A, B)
    scale = abs(al) * 2 * absZ + abs(be) * 2 * np.abs(Cin)
    got = C.cpu().numpy()
    assert_within_ulps(got.real, want.real, scale, 2)
    assert_within_ulps(got.imag, want.imag, scale, 2)


# ---- Scheme II on FP32 inputs (emugemm_sgemm_oz2) ----
@pytest.mark.parametrize("N,shape", [(8, (256, 256, 256)), (11, (200, 300, 333)), (9, (129, 513, 140))])
def test_sgemm_oz2(env, N, shape):
    torch, O, h, E = env
    m, n, k = shape
    A, B = G.real_pair(m, n, k, 1.0, 4, dtype=np.float32)
    C = torch.full((m, n), float("nan"), dtype=torch.float32, device="cuda")
    h.sgemm_oz2(dev(torch, A), dev(torch, B), C, N)
    _, absAB = O.bf128_dgemm(A.astype(np.float64), B.astype(np.float64))
    assert_within_ulps(C.cpu().numpy(), O.sgemm_oz2(A, B, N), absAB, 2, bits=23, what=f"sgemm_oz2 N={N}")


def test_sgemm_oz2_residues_alpha_beta_transposed(env):
    torch, O, h, E = env
    m, n, k, N = 140, 90, 260, 10
    A, B, Cin = G.real_pair(m, n, k, 1.0, 6, dtype=np.float32, with_c=True)
    _, tA, tB = O.oz2_budget(N, k)
    RA, _ = h.dbg_oz2_residues(dev(torch, A), False, N, tA)
    A64 = A.astype(np.float64)
    assert np.array_equal(RA.cpu().numpy(), O.oz2_residues_rows(A64, O.row_exponents(A64), tA, N))
    C = dev(torch, Cin)
    h.sgemm_oz2(dev(torch, A.T), dev(torch, B), C, N, alpha=2.5, beta=-0.5, transa=True)
    _, absAB = O.bf128_dgemm(A64, B.astype(np.float64))
    assert_within_ulps(C.cpu().numpy(), O.sgemm_oz2(A, B, N, alpha=2.5, beta=-0.5, Cin=Cin), 2.5 * absAB + 0.5 * np.abs(Cin), 2,
                       bits=23, what="sgemm_oz2 alpha/beta")
