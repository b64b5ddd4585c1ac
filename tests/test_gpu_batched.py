"""-m gpu parity tests, strided batched Scheme I: every entry of a batched call
against the oracle run on that entry (2 ulp of (|A||B|)_ij) and bit-identical to the single call on it."""
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
    assert torch.cuda.is_available()
    h = E.EmuGemm()
    yield torch, O, h
    h.close()


def entries(batch, m, n, k, phi, seed, dtype=np.float64):
    AB = [G.real_pair(m, n, k, phi, seed + 17 * b, dtype=dtype) for b in range(batch)]
    return np.stack([a for a, _ in AB]), np.stack([b for _, b in AB])


@pytest.mark.parametrize("p,batch,shape", [(6, 5, (100, 70, 300)), (8, 3, (129, 66, 130)), (3, 4, (260, 330, 256)),
                                           (4, 7, (64, 64, 64)), (5, 2, (300, 200, 333)), (2, 3, (257, 514, 128))])
def test_dgemm_batched_vs_oracle_and_single(env, p, batch, shape):
    """Ragged m, n (tiles of one entry spill into the next entry's plane rows) for every kernel family:
    p <= 3 CTA pairs, p >= 4 multicast clusters."""
    torch, O, h = env
    m, n, k = shape
    A, B = entries(batch, m, n, k, 1.0, 40 + p)
    Ad, Bd = torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()
    C = torch.full((batch, m, n), float("nan"), dtype=torch.float64, device="cuda")  # beta = 0: C not read
    h.dgemm_oz1_strided_batched(Ad, Bd, C, p)
    got = C.cpu().numpy()
    for b in range(batch):
        _, absAB = O.bf128_dgemm(A[b], B[b])
        assert_within_ulps(got[b], O.dgemm_oz1(A[b], B[b], p), absAB, 2, what=f"entry {b} p={p} {shape}")
        single = torch.zeros((m, n), dtype=torch.float64, device="cuda")
        h.dgemm_oz1(Ad[b], Bd[b], single, p)
        assert np.array_equal(got[b], single.cpu().numpy()), f"entry {b} differs from the single call"


def test_batched_alpha_beta_strides_shared_b(env):
    """alpha / beta, padded leading dimensions, a batch stride larger than the matrix, and ONE B shared by all
    entries (strideB = 0)."""
    torch, O, h = env
    batch, m, n, k, p = 4, 90, 72, 200, 6
    A, _ = entries(batch, m, n, k, 2.0, 3)
    _, B = G.real_pair(m, n, k, 2.0, 99)
    rng = np.random.default_rng(5)
    Cin = rng.standard_normal((batch, m, n))
    Abuf = torch.zeros((batch, m + 2, k + 6), dtype=torch.float64, device="cuda")
    Abuf[:, :m, :k] = torch.from_numpy(A).cuda()
    Bbuf = torch.zeros((k, n + 10), dtype=torch.float64, device="cuda")
    Bbuf[:, :n] = torch.from_numpy(B).cuda()
    Cbuf = torch.full((batch, m + 1, n + 4), 7.0, dtype=torch.float64, device="cuda")
    Cbuf[:, :m, :n] = torch.from_numpy(Cin).cuda()
    h.dgemm_oz1_strided_batched(Abuf[:, :m, :k], Bbuf[:, :n], Cbuf[:, :m, :n], p, alpha=-1.5, beta=0.75)
    got = Cbuf.cpu().numpy()
    assert (got[:, m:, :] == 7.0).all() and (got[:, :, n:] == 7.0).all(), "wrote outside C"
    for b in range(batch):
        _, absAB = O.bf128_dgemm(A[b], B)
        want = O.dgemm_oz1(A[b], B, p, alpha=-1.5, beta=0.75, Cin=Cin[b])
        scale = 1.5 * absAB + 0.75 * np.abs(Cin[b])
        assert_within_ulps(got[b, :m, :n], want, scale, 2, what=f"entry {b}")


def test_sgemm_batched(env):
    torch, O, h = env
    batch, m, n, k, p = 3, 130, 96, 260, 4
    A, B = entries(batch, m, n, k, 1.0, 8, dtype=np.float32)
    C = torch.zeros((batch, m, n), dtype=torch.float32, device="cuda")
    h.sgemm_oz1_strided_batched(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), C, p)
    got = C.cpu().numpy()
    for b in range(batch):
        _, absAB = O.bf128_dgemm(A[b].astype(np.float64), B[b].astype(np.float64))
        assert_within_ulps(got[b], O.sgemm_oz1(A[b], B[b], p), absAB, 2, bits=23, what=f"entry {b}")


def test_batched_8bit_slices(env):
    """R23 digits through the batched path."""
    torch, O, h = env
    batch, m, n, k, p = 3, 140, 100, 384, 7
    A, B = entries(batch, m, n, k, 1.0, 21)
    C = torch.zeros((batch, m, n), dtype=torch.float64, device="cuda")
    h.set_slice_bits(8)
    O.set_slice_bits(8)
    try:
        h.dgemm_oz1_strided_batched(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), C, p)
        got = C.cpu().numpy()
        for b in range(batch):
            _, absAB = O.bf128_dgemm(A[b], B[b])
            assert_within_ulps(got[b], O.dgemm_oz1(A[b], B[b], p), absAB, 2, what=f"entry {b}")
    finally:
        h.set_slice_bits(7)
        O.set_slice_bits(7)


def test_batched_long_k_runs_entry_by_entry(env):
    """k above the overflow-safe chunk length: the batched call falls back to one (chunked) call per entry."""
    torch, O, h = env
    import paper_2606_25453_b200 as E
    p = 8
    k = int(E.oz1_chunk_k(p)) + 256
    batch, m, n = 2, 40, 24
    A, B = entries(batch, m, n, k, 0.5, 2)
    C = torch.zeros((batch, m, n), dtype=torch.float64, device="cuda")
    h.dgemm_oz1_strided_batched(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), C, p)
    got = C.cpu().numpy()
    for b in range(batch):
        _, absAB = O.bf128_dgemm(A[b], B[b])
        assert_within_ulps(got[b], O.dgemm_oz1(A[b], B[b], p), absAB, 2, what=f"entry {b}")


def test_batched_degenerate_and_errors(env):
    torch, O, h = env
    import paper_2606_25453_b200 as E
    A = torch.zeros((2, 8, 16), dtype=torch.float64, device="cuda")
    B = torch.zeros((2, 16, 8), dtype=torch.float64, device="cuda")
    C = torch.full((2, 8, 8), 3.0, dtype=torch.float64, device="cuda")
    # k = 0: C scaled by beta, entry by entry
    h.dgemm_oz1_strided_batched(A[:, :, :0], B[:, :0, :], C, 4, beta=0.5)
    assert (C.cpu().numpy() == 1.5).all()
    # overlapping outputs are refused
    lib, hh = h._lib, h._h
    import ctypes as ct
    st = lib.emugemm_dgemm_oz1_strided_batched(hh, ct.c_int64(2), ct.c_int64(8), ct.c_int64(8), ct.c_int64(16),
                                               ct.c_double(1.0), ct.c_void_p(A.data_ptr()), ct.c_int64(16), ct.c_int64(128),
                                               ct.c_void_p(B.data_ptr()), ct.c_int64(8), ct.c_int64(128), ct.c_double(0.0),
                                               ct.c_void_p(C.data_ptr()), ct.c_int64(8), ct.c_int64(8), ct.c_int(4))
    assert st == -1  # EMUGEMM_ERR_ARG
    # misaligned batch stride
    st = lib.emugemm_dgemm_oz1_strided_batched(hh, ct.c_int64(2), ct.c_int64(8), ct.c_int64(8), ct.c_int64(16),
                                               ct.c_double(1.0), ct.c_void_p(A.data_ptr()), ct.c_int64(16), ct.c_int64(129),
                                               ct.c_void_p(B.data_ptr()), ct.c_int64(8), ct.c_int64(128), ct.c_double(0.0),
                                               ct.c_void_p(C.data_ptr()), ct.c_int64(8), ct.c_int64(64), ct.c_int(4))
    assert st == -2  # EMUGEMM_ERR_ALIGNMENT


# ---- Scheme II ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,batch,shape", [(16, 4, (100, 80, 300)), (12, 3, (257, 272, 130)), (20, 2, (300, 200, 333)),
                                           (14, 5, (64, 64, 128))])
def test_dgemm_oz2_batched_vs_oracle_and_single(env, N, batch, shape):
    torch, O, h = env
    m, n, k = shape
    A, B = entries(batch, m, n, k, 1.0, 300 + N)
    Ad, Bd = torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()
    C = torch.full((batch, m, n), float("nan"), dtype=torch.float64, device="cuda")  # beta = 0: C not read
    h.dgemm_oz2_strided_batched(Ad, Bd, C, N)
    got = C.cpu().numpy()
    for b in range(batch):
        _, absAB = O.bf128_dgemm(A[b], B[b])
        assert_within_ulps(got[b], O.dgemm_oz2(A[b], B[b], N), absAB, 2, what=f"entry {b} N={N} {shape}")
        single = torch.zeros((m, n), dtype=torch.float64, device="cuda")
        h.dgemm_oz2(Ad[b], Bd[b], single, N)
        assert np.array_equal(got[b], single.cpu().numpy()), f"entry {b} differs from the single call"


def test_oz2_batched_alpha_beta_strides_shared_a(env):
    """alpha / beta, padded leading dimensions and batch strides, ONE A shared by all entries (strideA = 0)."""
    torch, O, h = env
    batch, m, n, k, N = 3, 90, 72, 200, 15
    A, _ = G.real_pair(m, n, k, 2.0, 77)
    _, B = entries(batch, m, n, k, 2.0, 5)
    Cin = np.random.default_rng(6).standard_normal((batch, m, n))
    Abuf = torch.zeros((m, k + 6), dtype=torch.float64, device="cuda")
    Abuf[:, :k] = torch.from_numpy(A).cuda()
    Bbuf = torch.zeros((batch, k + 2, n + 10), dtype=torch.float64, device="cuda")
    Bbuf[:, :k, :n] = torch.from_numpy(B).cuda()
    Cbuf = torch.full((batch, m + 1, n + 4), 7.0, dtype=torch.float64, device="cuda")
    Cbuf[:, :m, :n] = torch.from_numpy(Cin).cuda()
    h.dgemm_oz2_strided_batched(Abuf[:, :k], Bbuf[:, :k, :n], Cbuf[:, :m, :n], N, alpha=-1.5, beta=0.75)
    got = Cbuf.cpu().numpy()
    assert (got[:, m:, :] == 7.0).all() and (got[:, :, n:] == 7.0).all(), "wrote outside C"
    for b in range(batch):
        _, absAB = O.bf128_dgemm(A, B[b])
        want = O.dgemm_oz2(A, B[b], N, alpha=-1.5, beta=0.75, Cin=Cin[b])
        assert_within_ulps(got[b, :m, :n], want, 1.5 * absAB + 0.75 * np.abs(Cin[b]), 2, what=f"entry {b}")


def test_sgemm_oz2_batched(env):
    torch, O, h = env
    batch, m, n, k, N = 3, 130, 96, 260, 9
    A, B = entries(batch, m, n, k, 1.0, 18, dtype=np.float32)
    C = torch.zeros((batch, m, n), dtype=torch.float32, device="cuda")
    h.sgemm_oz2_strided_batched(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), C, N)
    got = C.cpu().numpy()
    for b in range(batch):
        _, absAB = O.bf128_dgemm(A[b].astype(np.float64), B[b].astype(np.float64))
        assert_within_ulps(got[b], O.sgemm_oz2(A[b], B[b], N), absAB, 2, bits=23, what=f"entry {b}")


@pytest.mark.parametrize("N,batch,shape", [(14, 3, (100, 80, 200)), (18, 2, (257, 272, 130))])
def test_zgemm_3m_batched(env, N, batch, shape):
    """complex128 by 3M: every entry against the oracle, bit-identical to the single call; alpha / beta complex."""
    torch, O, h = env
    m, n, k = shape
    trip = [G.complex_pair(m, n, k, 1.0, 60 + 7 * b, with_c=True) for b in range(batch)]
    A, B, Cin = (np.stack([t[i] for t in trip]) for i in range(3))
    al, be = 0.5 - 2j, 1.5 + 0.25j
    Ad, Bd = torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()
    C = torch.from_numpy(Cin).cuda()
    h.zgemm_oz2_3m_strided_batched(Ad, Bd, C, N, alpha=al, beta=be)
    got = C.cpu().numpy()
    for b in range(batch):
        want = O.zgemm_oz2_3m(A[b], B[b], N, alpha=al, beta=be, Cin=Cin[b])
        _, absZ = O.bf128_zgemm(A[b], B[b])
        scale = abs(al) * 2 * absZ + abs(be) * 2 * np.abs(Cin[b])
        assert_within_ulps(got[b].real, want.real, scale, 2, what=f"entry {b} re")
        assert_within_ulps(got[b].imag, want.imag, scale, 2, what=f"entry {b} im")
        single = torch.from_numpy(Cin[b]).cuda()
        h.zgemm_oz2_3m(Ad[b], Bd[b], single, N, alpha=al, beta=be)
        assert np.array_equal(got[b], single.cpu().numpy()), f"entry {b} differs from the single call"
