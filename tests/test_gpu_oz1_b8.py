"""-m gpu parity tests, Scheme I with 8-bit balanced digits (emugemm_set_slice_bits(h, 8); R23):
digits and INT32 accumulators bit-exact against the oracle's 8-bit mode, final FP64 / FP32 within 2 ulp of
(|A||B|)_ij, k-chunking with the shorter overflow-safe chunk (p k_c 128^2 <= 2^31 - 1)."""
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
    h.set_slice_bits(8)
    O.set_slice_bits(8)
    yield torch, O, h
    O.set_slice_bits(7)
    h.close()


def dev(torch, x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("p", [1, 3, 4, 7, 8])
@pytest.mark.parametrize("shape", [(256, 256, 256), (130, 70, 333)])
def test_digits_bit_exact(env, p, shape):
    torch, O, h = env
    m, n, k = shape
    A, B = G.real_pair(m, n, k, 2.0, 5)
    A[0, 0] = 0.0
    A[1, 1] = -np.abs(A[1]).max() * 3
    A[2, 2] = np.abs(A[2]).max() * 1.999
    SA, eA = h.dbg_oz1_slices(dev(torch, A), False, p)
    SB, eB = h.dbg_oz1_slices(dev(torch, B), True, p)
    oA, oB = O.row_exponents(A), O.col_exponents(B)
    assert np.array_equal(eA.cpu().numpy(), oA) and np.array_equal(eB.cpu().numpy(), oB)
    assert np.array_equal(SA.cpu().numpy(), O.oz1_slices_rows(A, oA, p))
    assert np.array_equal(SB.cpu().numpy(), O.oz1_slices_cols(B, oB, p))


def test_digits_f32_bit_exact(env):
    torch, O, h = env
    A, B = G.real_pair(100, 60, 200, 1.0, 4, dtype=np.float32)
    SA, _ = h.dbg_oz1_slices(dev(torch, A), False, 3)
    SB, _ = h.dbg_oz1_slices(dev(torch, B), True, 3)
    A64, B64 = A.astype(np.float64), B.astype(np.float64)
    assert np.array_equal(SA.cpu().numpy(), O.oz1_slices_rows(A64, O.row_exponents(A64), 3))
    assert np.array_equal(SB.cpu().numpy(), O.oz1_slices_cols(B64, O.col_exponents(B64), 3))


@pytest.mark.parametrize("p", [2, 4, 5, 7, 8])
def test_int32_accumulators_bit_exact(env, p):
    torch, O, h = env
    m, n, k = (256, 320, 384) if p % 2 else (200, 150, 300)
    A, B = G.real_pair(m, n, k, 0.5, 100 + p)
    acc = h.dbg_oz1_accumulators(dev(torch, A), dev(torch, B), p).cpu().numpy()
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    CS = O.oz1_accumulators(O.oz1_slices_rows(A, eA, p), O.oz1_slices_cols(B, eB, p))
    assert acc.shape == (1, p, m, n)
    assert np.array_equal(acc[0].astype(np.int64), CS)


@pytest.mark.parametrize("p,shape,phi", [(3, (384, 320, 512), 0.5), (4, (129, 257, 130), 2.0), (6, (300, 200, 333), 2.0),
                                         (7, (256, 256, 256), 0.5), (7, (515, 130, 700), 2.0), (8, (128, 64, 128), 1.0)])
def test_dgemm_full_matrix(env, p, shape, phi):
    torch, O, h = env
    m, n, k = shape
    A, B = G.real_pair(m, n, k, phi, 1)
    C = torch.full((m, n), float("nan"), dtype=torch.float64, device="cuda")
    h.dgemm_oz1(dev(torch, A), dev(torch, B), C, p)
    _, absAB = O.bf128_dgemm(A, B)
    assert_within_ulps(C.cpu().numpy(), O.dgemm_oz1(A, B, p), absAB, 2, what=f"b8 p={p} {shape}")


def test_alpha_beta_and_sgemm(env):
    torch, O, h = env
    m, n, k, p = 200, 136, 260, 7
    A, B, Cin = G.real_pair(m, n, k, 1.0, 9, with_c=True)
    Cd = dev(torch, Cin)
    h.dgemm_oz1(dev(torch, A), dev(torch, B), Cd, p, alpha=-1.5, beta=0.75)
    _, absAB = O.bf128_dgemm(A, B)
    assert_within_ulps(Cd.cpu().numpy(), O.dgemm_oz1(A, B, p, alpha=-1.5, beta=0.75, Cin=Cin), 1.5 * absAB + 0.75 * np.abs(Cin), 2)
    A32, B32 = G.real_pair(260, 200, 300, 1.0, 4, dtype=np.float32)
    C32 = torch.zeros((260, 200), dtype=torch.float32, device="cuda")
    h.sgemm_oz1(dev(torch, A32), dev(torch, B32), C32, 3)
    _, ab32 = O.bf128_dgemm(A32.astype(np.float64), B32.astype(np.float64))
    assert_within_ulps(C32.cpu().numpy(), O.sgemm_oz1(A32, B32, 3), ab32, 2, bits=23, what="sgemm b8 p=3")


def test_k_chunked(env):
    """p = 8: the 8-bit chunk bound is 16,256 columns, so k = 17,000 takes 2 chunks + the exact reduction."""
    torch, O, h = env
    import paper_2606_25453_b200 as E
    assert E.oz1_chunk_k(8, 8) == 16256 and 8 * 16256 * 128 * 128 <= 2 ** 31 - 1 < 8 * (16256 + 128) * 128 * 128
    m, n, k, p = 64, 48, 17000, 8
    A, B = G.real_pair(m, n, k, 1.0, 4)
    C = torch.zeros((m, n), dtype=torch.float64, device="cuda")
    h.dgemm_oz1(dev(torch, A), dev(torch, B), C, p)
    _, absAB = O.bf128_dgemm(A, B)
    assert_within_ulps(C.cpu().numpy(), O.dgemm_oz1(A, B, p), absAB, 2, what="chunked b8")
    acc = h.dbg_oz1_accumulators(dev(torch, A[:, :1000]), dev(torch, B[:1000]), 4, chunk_k=384).cpu().numpy()
    eA, eB = O.row_exponents(A[:, :1000]), O.col_exponents(B[:1000])
    CS = O.oz1_accumulators(O.oz1_slices_rows(A[:, :1000], eA, 4), O.oz1_slices_cols(B[:1000], eB, 4))
    assert np.array_equal(acc.astype(np.int64).sum(0), CS)


def test_full_size_sampled_p7(env):
    """The f1 operating point: 8192^3, 7 balanced slices (28 products) at FP64-level accuracy."""
    torch, O, h = env
    size, p = 8192, 7
    A, B = G.real_pair(size, size, size, 0.5, 1)
    C = torch.full((size, size), float("nan"), dtype=torch.float64, device="cuda")
    h.dgemm_oz1(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), C, p)
    rows, cols = G.sample_indices(size, 36, 7)[:48], G.sample_indices(size, 36, 8)[:48]
    got = C[torch.from_numpy(rows).cuda()][:, torch.from_numpy(cols).cuda()].cpu().numpy()
    absab = np.abs(A[rows, :]) @ np.abs(B[:, cols])
    assert_within_ulps(got, O.oz1_sampled(A, B, p, rows, cols), absab, 2, what="b8 8192 p=7")
    assert torch.isfinite(C).all()
