"""-m gpu parity tests, Scheme I: the CUDA path (through the C ABI) against the oracle on the same
seeded inputs.  Integer intermediates (exponents, slices, INT32 accumulators) bit-exact; final FP64
within 2 ulp of (|A||B|)_ij (north_star), FP32 path 2 ulp in FP32."""
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


def dev(torch, x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_exponents(env, dtype):
    torch, O, h = env
    A, B = G.real_pair(300, 200, 333, 2.0, 11, dtype=dtype)
    A[3, :] = 0
    B[:, 5] = 0
    if dtype == np.float64:
        A[4, 7] = 5e-324
    eA = h.dbg_exponents(dev(torch, A), False).cpu().numpy()
    eB = h.dbg_exponents(dev(torch, B), True).cpu().numpy()
    assert np.array_equal(eA, O.row_exponents(A.astype(np.float64)))
    assert np.array_equal(eB, O.col_exponents(B.astype(np.float64)))


def test_exponents_complex(env):
    torch, O, h = env
    A, B = G.complex_pair(70, 90, 130, 1.0, 3)
    assert np.array_equal(h.dbg_exponents(dev(torch, A), False).cpu().numpy(), O.row_exponents_z(A))
    assert np.array_equal(h.dbg_exponents(dev(torch, B), True).cpu().numpy(), O.col_exponents_z(B))


@pytest.mark.parametrize("p", [1, 3, 6, 8])
@pytest.mark.parametrize("shape", [(256, 256, 256), (130, 70, 333)])
def test_slices_bit_exact(env, p, shape):
    torch, O, h = env
    m, n, k = shape
    A, B = G.real_pair(m, n, k, 2.0, 5)
    A[0, 0] = 0.0
    SA, eA = h.dbg_oz1_slices(dev(torch, A), False, p)
    SB, eB = h.dbg_oz1_slices(dev(torch, B), True, p)
    oA, oB = O.row_exponents(A), O.col_exponents(B)
    assert np.array_equal(eA.cpu().numpy(), oA) and np.array_equal(eB.cpu().numpy(), oB)
    assert np.array_equal(SA.cpu().numpy(), O.oz1_slices_rows(A, oA, p))
    assert np.array_equal(SB.cpu().numpy(), O.oz1_slices_cols(B, oB, p))


def test_slices_f32_bit_exact(env):
    torch, O, h = env
    A, B = G.real_pair(100, 60, 200, 1.0, 4, dtype=np.float32)
    SA, eA = h.dbg_oz1_slices(dev(torch, A), False, 4)
    SB, eB = h.dbg_oz1_slices(dev(torch, B), True, 4)
    A64, B64 = A.astype(np.float64), B.astype(np.float64)
    assert np.array_equal(SA.cpu().numpy(), O.oz1_slices_rows(A64, O.row_exponents(A64), 4))
    assert np.array_equal(SB.cpu().numpy(), O.oz1_slices_cols(B64, O.col_exponents(B64), 4))


@pytest.mark.parametrize("p", [1, 2, 3, 4, 5, 6, 7, 8])
def test_int32_accumulators_bit_exact(env, p):
    """tcgen05 path: the p INT32 accumulators of the fused kernel == the oracle's int64 C_s."""
    torch, O, h = env
    m, n, k = (256, 320, 384) if p % 2 else (200, 150, 300)
    A, B = G.real_pair(m, n, k, 0.5, 100 + p)
    acc = h.dbg_oz1_accumulators(dev(torch, A), dev(torch, B), p).cpu().numpy()
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    CS = O.oz1_accumulators(O.oz1_slices_rows(A, eA, p), O.oz1_slices_cols(B, eB, p))
    assert acc.shape == (1, p, m, n)
    assert np.array_equal(acc[0].astype(np.int64), CS)


def test_int32_accumulators_chunked(env):
    """k-chunking (R7, R8): per-chunk INT32 dumps summed in int64 equal the chunk-free oracle."""
    torch, O, h = env
    p, m, n, k = 4, 140, 100, 1000
    A, B = G.real_pair(m, n, k, 1.0, 77)
    acc = h.dbg_oz1_accumulators(dev(torch, A), dev(torch, B), p, chunk_k=384).cpu().numpy()
    assert acc.shape[0] == 3
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    CS = O.oz1_accumulators(O.oz1_slices_rows(A, eA, p), O.oz1_slices_cols(B, eB, p))
    assert np.array_equal(acc.astype(np.int64).sum(0), CS)


def test_config0_dgemm_oz1(env):
    """BASELINE config 1 (index 0): 256^3, phi 0.5, seed 0, p 6: full oracle + __float128 brute force."""
    torch, O, h = env
    A, B = G.real_pair(256, 256, 256, 0.5, 0)
    C = torch.full((256, 256), float("nan"), dtype=torch.float64, device="cuda")  # beta = 0: C not read
    h.dgemm_oz1(dev(torch, A), dev(torch, B), C, 6)
    want = O.dgemm_oz1(A, B, 6)
    exact, absAB = O.bf128_dgemm(A, B)
    worst = assert_within_ulps(C.cpu().numpy(), want, absAB, 2, what="config0 vs oracle")
    assert worst <= 2
    # and the GPU result obeys the same closed-form truncation bound as the oracle
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    x = np.abs(A) * np.exp2(-eA.astype(float))[:, None]
    y = np.abs(B) * np.exp2(-eB.astype(float))[None, :]
    bound = np.exp2(eA[:, None].astype(float) + eB[None, :] - 42) * (x.sum(1)[:, None] + y.sum(0)[None, :] + 256 * 5 / (1 - 2.0 ** -7))
    assert (np.abs(C.cpu().numpy() - exact) < bound + 3 * np.spacing(np.abs(absAB))).all()


@pytest.mark.parametrize("p,shape,phi", [(3, (384, 320, 512), 0.5), (4, (129, 257, 130), 2.0), (5, (300, 200, 333), 2.0),
                                         (7, (128, 64, 128), 1.0), (8, (515, 130, 700), 2.0), (2, (260, 520, 256), 0.5)])
def test_dgemm_oz1_full_matrix(env, p, shape, phi):
    torch, O, h = env
    m, n, k = shape
    A, B = G.real_pair(m, n, k, phi, 1)
    C = torch.zeros((m, n), dtype=torch.float64, device="cuda")
    h.dgemm_oz1(dev(torch, A), dev(torch, B), C, p)
    _, absAB = O.bf128_dgemm(A, B)
    assert_within_ulps(C.cpu().numpy(), O.dgemm_oz1(A, B, p), absAB, 2, what=f"p={p} {shape}")


def test_dgemm_oz1_alpha_beta_strides(env):
    torch, O, h = env
    m, n, k, p = 200, 136, 260, 6
    A, B, Cin = G.real_pair(m, n, k, 1.0, 9, with_c=True)
    # non-trivial leading dimensions
    Ad = torch.zeros((m, k + 6), dtype=torch.float64, device="cuda"); Ad[:, :k] = dev(torch, A)
    Bd = torch.zeros((k, n + 10), dtype=torch.float64, device="cuda"); Bd[:, :n] = dev(torch, B)
    Cd = torch.zeros((m, n + 3), dtype=torch.float64, device="cuda"); Cd[:, :n] = dev(torch, Cin)
    Cd[:, n:] = 7.0
    h.dgemm_oz1(Ad[:, :k], Bd[:, :n], Cd[:, :n], p, alpha=-1.5, beta=0.75)
    want = O.dgemm_oz1(A, B, p, alpha=-1.5, beta=0.75, Cin=Cin)
    _, absAB = O.bf128_dgemm(A, B)
    assert_within_ulps(Cd[:, :n].cpu().numpy(), want, 1.5 * absAB + 0.75 * np.abs(Cin), 2, what="alpha/beta")
    assert (Cd[:, n:] == 7.0).all()  # padding columns untouched


def test_dgemm_oz1_k_chunked_final(env):
    """k > overflow-safe chunk: p = 8 bound is 16640, so k = 17000 takes 2 chunks + double-double reduce."""
    torch, O, h = env
    m, n, k, p = 64, 48, 17000, 8
    A, B = G.real_pair(m, n, k, 1.0, 4)
    C = torch.zeros((m, n), dtype=torch.float64, device="cuda")
    h.dgemm_oz1(dev(torch, A), dev(torch, B), C, p)
    _, absAB = O.bf128_dgemm(A, B)
    assert_within_ulps(C.cpu().numpy(), O.dgemm_oz1(A, B, p), absAB, 2, what="chunked")


@pytest.mark.parametrize("p", [3, 4])
def test_sgemm_oz1(env, p):
    torch, O, h = env
    m, n, k = 260, 200, 300
    A, B = G.real_pair(m, n, k, 1.0, 4, dtype=np.float32)
    C = torch.zeros((m, n), dtype=torch.float32, device="cuda")
    h.sgemm_oz1(dev(torch, A), dev(torch, B), C, p)
    _, absAB = O.bf128_dgemm(A.astype(np.float64), B.astype(np.float64))
    assert_within_ulps(C.cpu().numpy(), O.sgemm_oz1(A, B, p), absAB, 2, bits=23, what=f"sgemm p={p}")


def test_degenerate_sizes(env):
    torch, O, h = env
    A = torch.zeros((5, 0), dtype=torch.float64, device="cuda")
    B = torch.zeros((0, 4), dtype=torch.float64, device="cuda")
    C = torch.ones((5, 4), dtype=torch.float64, device="cuda")
    h.dgemm_oz1(A, B, C, 4, beta=2.0)  # k = 0: C <- beta C
    assert (C == 2.0).all()
    A1, B1 = G.real_pair(1, 1, 1, 0.5, 3)
    C1 = torch.zeros((1, 1), dtype=torch.float64, device="cuda")
    h.dgemm_oz1(dev(torch, A1), dev(torch, B1), C1, 8)
    assert C1.cpu().numpy()[0, 0] == O.dgemm_oz1(A1, B1, 8)[0, 0]
    Z = torch.zeros((130, 130), dtype=torch.float64, device="cuda")
    Cz = torch.ones((130, 130), dtype=torch.float64, device="cuda")
    h.dgemm_oz1(Z, Z, Cz, 5)  # all-zero operands
    assert (Cz == 0).all()


def test_dgemm_oz1_extreme_exponents(env):
    """operands near DBL_MIN / DBL_MAX: 2^(eA_i + eB_j - 7(p+1)) must flush to zero / subnormals / infinity
    correctly instead of wrapping the exponent field."""
    torch, O, h = env
    m, n, k, p = 70, 66, 130, 6
    A, B = G.real_pair(m, n, k, 1.0, 21)
    for sa, sb in ((2.0 ** -1000, 2.0 ** -1000), (2.0 ** -1020, 2.0 ** -40), (2.0 ** 500, 2.0 ** 500), (2.0 ** -600, 2.0 ** -440),
                   (2.0 ** -1021, 2.0 ** 0)):
        As, Bs = A * sa, B * sb
        C = torch.full((m, n), float("nan"), dtype=torch.float64, device="cuda")
        h.dgemm_oz1(dev(torch, As), dev(torch, Bs), C, p)
        want = O.dgemm_oz1(As, Bs, p)
        got = C.cpu().numpy()
        with np.errstate(over="ignore", under="ignore"):
            scale = np.abs(As) @ np.abs(Bs)
        tiny = scale < 2.0 ** -1021
        if (~tiny).any():
            assert_within_ulps(got[~tiny], want[~tiny], scale[~tiny], 2, what=f"scales {sa} {sb}")
        assert (np.abs(got[tiny] - want[tiny]) <= 2 * 2.0 ** -1074).all()   # subnormal range: two subnormal spacings


@pytest.mark.parametrize("bits", [7, 8])
@pytest.mark.parametrize("p,shape", [(8, (40, 24, 34000)), (7, (130, 70, 39000)), (3, (64, 48, 90000)), (8, (256, 200, 17000))])
def test_dgemm_oz1_balanced_chunks_fit_the_declared_workspace(env, bits, p, shape):
    """Long k on few tiles: the chunk count is balanced against the worker count (api.cu oz1_chunks_balanced, up to twice
    the overflow-safe minimum).  A FRESH handle reserves exactly emugemm_workspace_bytes(), so the call fails with
    EMUGEMM_ERR_WORKSPACE if the declared size does not cover the chunk count the call picks in either digit mode; the
    result must not depend on the split (exact double-double partials)."""
    torch, O, _ = env
    import paper_2606_25453_b200 as E
    m, n, k = shape
    A, B = G.real_pair(m, n, k, 1.0, 21)
    h = E.EmuGemm()
    try:
        h.set_slice_bits(bits)
        O.set_slice_bits(bits)
        C = torch.zeros((m, n), dtype=torch.float64, device="cuda")
        h.dgemm_oz1(dev(torch, A), dev(torch, B), C, p)
        want = O.dgemm_oz1(A, B, p)
    finally:
        O.set_slice_bits(7)
        h.close()
    assert_within_ulps(C.cpu().numpy(), want, np.abs(A) @ np.abs(B), 2, what=f"balanced chunks p={p} bits={bits}")
