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


# ---- the CRT is exact for EVERY residue vector (R17, round 2) ----
@pytest.mark.parametrize("N", [2, 3, 8, 11, 12, 14, 15, 16, 18, 20])
def test_crt_correctly_rounded_for_any_magnitude(env, N):
    """X of every magnitude from 0 to P/4 (the budget's range, R12), both signs: the kernel must return the
    correctly rounded double of the big integer.  The expected value is Python's int -> float conversion (correctly
    rounded, independent of oracle and kernel); the oracle is held to 1 ulp of it (its __float128 step may round twice)."""
    torch, O, h, E = env
    mods = [int(x) for x in O.oz2_moduli(N)]
    P = O.oz2_P(N)
    rng = np.random.default_rng(1000 + N)
    m, n = 37, 52   # ragged: scalar tail path of the kernel
    Xs = []
    top = (P // 4).bit_length() - 1
    for idx in range(m * n):
        bits = idx % (top + 1)
        x = int(rng.integers(0, 2**62)) * int(rng.integers(0, 2**62)) * int(rng.integers(0, 2**62))
        x = (x % (1 << bits)) | (1 << bits) if bits > 0 else idx % 3
        x = min(x, P // 4 - 1)
        Xs.append(-x if (idx // (top + 1)) % 2 else x)
    Xs[0], Xs[1], Xs[2], Xs[3] = 0, 1, -1, P // 4 - 1
    CR = np.empty((N, m, n), np.int8)
    for l, mod in enumerate(mods):
        r = np.array([x % mod for x in Xs], np.int64)
        r = np.where(r >= (mod + 1) // 2, r - mod, r)
        CR[l] = r.reshape(m, n)
    eA = np.zeros(m, np.int32); eB = np.zeros(n, np.int32)
    want = np.array([float(x) for x in Xs]).reshape(m, n)
    for (mm, nn) in ((m, n), (m, 48)):   # ragged and vector path
        C = torch.full((mm, nn), float("nan"), dtype=torch.float64, device="cuda")
        h.dbg_oz2_crt(dev(torch, CR[:, :mm, :nn]), dev(torch, eA[:mm]), dev(torch, eB[:nn]), 0, 0, C)
        assert np.array_equal(C.cpu().numpy(), want[:mm, :nn]), f"N={N}: CRT is not the correctly rounded integer"
    orc = O.oz2_crt(CR, eA, eB, 0, 0)
    assert (np.abs(orc - want) <= np.spacing(np.abs(want))).all()


def _adversarial_pairs(m, n, k):
    """(|A||B|)_ij << k 2^(eA_i + eB_j): each row / column maximum meets a tiny or zero partner."""
    rng = np.random.default_rng(42)
    out = {}
    # one 1.0 per row of A at h = i mod k over 2^-40 noise; column j of B is 1.0 at h = (j + 1) mod k, tiny elsewhere
    A = rng.uniform(-1, 1, (m, k)) * 2.0 ** -40
    B = rng.uniform(-1, 1, (k, n)) * 2.0 ** -40
    A[np.arange(m), np.arange(m) % k] = 1.0
    B[(np.arange(n) + 1) % k, np.arange(n)] = 1.0
    out["unit_over_noise"] = (A, B)
    # B = I (k = n): C = A truncated to tA bits; each column of B has one nonzero
    A2 = rng.uniform(-1, 1, (m, n)) * np.exp(2.0 * rng.standard_normal((m, n)))
    out["identity"] = (A2, np.eye(n))
    # the row maximum of A meets an exact zero of B, the rest of the row is 2^-30 smaller
    A3 = rng.uniform(-1, 1, (m, k)) * 2.0 ** -30
    A3[:, 0] = rng.uniform(0.5, 1.0, m)
    B3 = rng.uniform(-1, 1, (k, n))
    B3[0, :] = 0.0
    out["max_meets_zero"] = (A3, B3)
    # integers: exact products with heavy cancellation (result 0 or tiny against k 2^(eA+eB))
    A4 = rng.integers(-3, 4, (m, k)).astype(np.float64)
    A4[:, 1] = 2.0 ** 20
    B4 = rng.integers(-3, 4, (k, n)).astype(np.float64)
    B4[1, :] = 0.0
    B4[2, ::2] = 2.0 ** 20
    out["integers"] = (A4, B4)
    return out


@pytest.mark.parametrize("N", [12, 16, 20])
@pytest.mark.parametrize("case", ["unit_over_noise", "identity", "max_meets_zero", "integers"])
def test_dgemm_oz2_adversarial(env, N, case):
    torch, O, h, E = env
    m, n, k = 150, 136, 136 if case == "identity" else 200
    A, B = _adversarial_pairs(m, n, k)[case]
    C = torch.full((m, n), float("nan"), dtype=torch.float64, device="cuda")
    h.dgemm_oz2(dev(torch, A), dev(torch, B), C, N)
    _, absAB = O.bf128_dgemm(A, B)
    got, want = C.cpu().numpy(), O.dgemm_oz2(A, B, N)
    assert_within_ulps(got, want, absAB, 2, what=f"adversarial {case} N={N}")
    zero = absAB == 0
    assert (got[zero] == 0).all()   # ulp_of(0) = 0: an exact zero must come out as zero


def test_zgemm_oz2_3m_adversarial(env):
    torch, O, h, E = env
    m, n, k, N = 100, 96, 128, 18
    Ar, Br = _adversarial_pairs(m, n, k)["unit_over_noise"]
    Ai, Bi = _adversarial_pairs(m, n, k)["max_meets_zero"]
    A, B = Ar + 1j * Ai * 2.0 ** -20, Br + 1j * Bi * 2.0 ** -35
    C = torch.zeros((m, n), dtype=torch.complex128, device="cuda")
    h.zgemm_oz2_3m(dev(torch, A), dev(torch, B), C, N)
    want = O.zgemm_oz2_3m(A, B, N)
    _, absZ = O.bf128_zgemm(A, B)
    got = C.cpu().numpy()
    assert_within_ulps(got.real, want.real, absZ, 2, what="3M adversarial re")
    assert_within_ulps(got.imag, want.imag, absZ, 2, what="3M adversarial im")


def test_dgemm_oz2_extreme_exponents(env):
    """operands near DBL_MIN / DBL_MAX: the power-of-two scaling must flush to zero / subnormals / infinity
    correctly instead of building a garbage exponent field."""
    torch, O, h, E = env
    m, n, k, N = 64, 64, 128, 14
    A, B = G.real_pair(m, n, k, 1.0, 21)
    for sa, sb in ((2.0 ** -1000, 2.0 ** -1000), (2.0 ** -1020, 2.0 ** -40), (2.0 ** 500, 2.0 ** 500), (2.0 ** -600, 2.0 ** -440)):
        As, Bs = A * sa, B * sb
        C = torch.full((m, n), float("nan"), dtype=torch.float64, device="cuda")
        h.dgemm_oz2(dev(torch, As), dev(torch, Bs), C, N)
        want = O.dgemm_oz2(As, Bs, N)
        got = C.cpu().numpy()
        with np.errstate(over="ignore", under="ignore"):
            scale = np.abs(As) @ np.abs(Bs)
        tiny = scale < 2.0 ** -1021
        if (~tiny).any():
            assert_within_ulps(got[~tiny], want[~tiny], scale[~tiny], 2, what=f"scales {sa} {sb}")
        # results in the subnormal range: absolute error of two subnormal spacings
        assert (np.abs(got[tiny] - want[tiny]) <= 2 * 2.0 ** -1074).all()


# ---- fused reconstruction: the CRT runs inside the per-modulus GEMM kernel ----
@pytest.mark.parametrize("N,shape", [(12, (256, 256, 256)), (14, (520, 300, 333)), (16, (512, 1024, 384)), (18, (600, 530, 260)),
                                     (20, (300, 770, 200)), (8, (512, 512, 256)), (15, (770, 512, 140))])
def test_dgemm_oz2_fused_matches_oracle_and_unfused(env, N, shape):
    torch, O, h, E = env
    m, n, k = shape
    A, B, Cin = G.real_pair(m, n, k, 1.0, 40 + N, with_c=True)
    Ad, Bd = dev(torch, A), dev(torch, B)
    out = {}
    for fused in (True, False):
        h.set_oz2_fusion(fused)
        C = torch.full((m, n), float("nan"), dtype=torch.float64, device="cuda")
        h.enable_stage_timing(True)
        h.dgemm_oz2(Ad, Bd, C, N)
        _, launches = h.stage_ms()
        h.enable_stage_timing(False)
        assert launches == (4 if fused else 5), "the fused path must not launch a separate CRT kernel"
        C2 = dev(torch, Cin)
        h.dgemm_oz2(Ad, Bd, C2, N, alpha=-1.5, beta=0.25)
        out[fused] = (C, C2)
    h.set_oz2_fusion(False)
    assert torch.equal(out[True][0], out[False][0]) and torch.equal(out[True][1], out[False][1])  # same arithmetic, same bits
    _, absAB = O.bf128_dgemm(A, B)
    assert_within_ulps(out[True][0].cpu().numpy(), O.dgemm_oz2(A, B, N), absAB, 2, what=f"fused oz2 N={N}")
    assert_within_ulps(out[True][1].cpu().numpy(), O.dgemm_oz2(A, B, N, alpha=-1.5, beta=0.25, Cin=Cin), 1.5 * absAB + 0.25 * np.abs(Cin), 2,
                       what=f"fused oz2 alpha/beta N={N}")


def test_dgemm_oz2_fused_adversarial_and_strided(env):
    """the fused path on the inputs that broke the round-1 CRT, with a C that has a leading-dimension slack"""
    torch, O, h, E = env
    m, n, k, N = 512, 512, 300, 16
    A, B = _adversarial_pairs(m, n, k)["unit_over_noise"]
    Cd = torch.full((m, n + 5), 7.0, dtype=torch.float64, device="cuda")
    h.set_oz2_fusion(True)
    try:
        h.dgemm_oz2(dev(torch, A), dev(torch, B), Cd[:, :n], N)
    finally:
        h.set_oz2_fusion(False)
    _, absAB = O.bf128_dgemm(A, B)
    assert_within_ulps(Cd[:, :n].cpu().numpy(), O.dgemm_oz2(A, B, N), absAB, 2, what="fused adversarial")
    assert (Cd[:, n:] == 7.0).all()


# ---- k beyond one INT32-safe range (k 128^2 < 2^31): one GEMM launch per k-chunk, output residues added modulo m_l ----------
@pytest.mark.parametrize("N,shape", [(12, (48, 40, 133000)), (16, (130, 70, 131072)), (20, (33, 17, 270001))])
def test_dgemm_oz2_k_chunked(env, N, shape):
    """k > 130,944: 2 chunks (133,000; 131,072 = one k-block over the limit) and 3 chunks (270,001, ragged), against the
    oracle, whose per-modulus products accumulate in int64 over the whole k."""
    torch, O, h, E = env
    m, n, k = shape
    A, B = G.real_pair(m, n, k, 1.0, 12)
    C = torch.full((m, n), float("nan"), dtype=torch.float64, device="cuda")
    h.dgemm_oz2(dev(torch, A), dev(torch, B), C, N, alpha=1.5)
    absAB = np.abs(A) @ np.abs(B)
    assert_within_ulps(C.cpu().numpy(), O.dgemm_oz2(A, B, N, alpha=1.5), 1.5 * absAB, 2, what=f"oz2 k={k} N={N}")


def test_zgemm_oz2_3m_k_chunked_and_operand_handles(env):
    torch, O, h, E = env
    m, n, k, N = 40, 24, 131500, 14
    A, B = G.complex_pair(m, n, k, 1.0, 13)
    C = torch.zeros((m, n), dtype=torch.complex128, device="cuda")
    h.zgemm_oz2_3m(dev(torch, A), dev(torch, B), C, N)
    want = O.zgemm_oz2_3m(A, B, N)
    absZ = (np.abs(A.real) + np.abs(A.imag)) @ (np.abs(B.real) + np.abs(B.imag))
    got = C.cpu().numpy()
    assert_within_ulps(got.real, want.real, absZ, 2, what="3M chunked re")
    assert_within_ulps(got.imag, want.imag, absZ, 2, what="3M chunked im")
    # pre-decomposed operands take the same chunked path and give the same bits
    Ar, Br = G.real_pair(m, n, k, 1.0, 14)
    C1 = torch.empty((m, n), dtype=torch.float64, device="cuda")
    C2 = torch.empty_like(C1)
    h.dgemm_oz2(dev(torch, Ar), dev(torch, Br), C1, 15)
    opA = h.decompose(E.OZ2, 0, dev(torch, Ar), 15)
    opB = h.decompose(E.OZ2, 1, dev(torch, Br), 15)
    h.gemm_pre(opA, opB, C2)
    assert torch.equal(C1, C2)
