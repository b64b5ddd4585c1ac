"""-m gpu: parity at BASELINE.json's full sizes, in the launch configuration bench.py times (same C-ABI
calls, same workspace path), on SAMPLED outputs the oracle computes one by one (SURVEY 8(c) "Parity at large
sizes"): ~40 x 40 sampled elements incl. first/last rows/columns and both sides of tile boundaries.
Tolerance: 2 ulp of (|A||B|)_ij at the sampled elements (FP32 path: 2 ulp in FP32)."""
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


def _abs_ab(A, B, rows, cols):
    return np.abs(A[rows, :]).astype(np.float64) @ np.abs(B[:, cols]).astype(np.float64)


def _samples(m, n, seed, count=36):
    return G.sample_indices(m, count, seed)[:48], G.sample_indices(n, count, seed + 1)[:48]


@pytest.mark.parametrize("size,p,phi", [(8192, 8, 2.0), (8192, 3, 0.5), (4096, 5, 2.0), (2048, 6, 0.5), (8192, 4, 0.5), (8192, 6, 2.0),
                                        (4096, 7, 0.5), (2048, 3, 2.0), (16384, 8, 0.5), (16384, 3, 2.0)])
def test_config1_oz1_sweep_points(env, size, p, phi):
    """BASELINE configs[1]: Scheme I DGEMM square sweep, seed 1."""
    torch, O, h = env
    A, B = G.real_pair(size, size, size, phi, 1)
    C = torch.full((size, size), float("nan"), dtype=torch.float64, device="cuda")
    h.dgemm_oz1(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), C, p)
    rows, cols = _samples(size, size, 7)
    got = C[torch.from_numpy(rows).cuda()][:, torch.from_numpy(cols).cuda()].cpu().numpy()
    want = O.oz1_sampled(A, B, p, rows, cols)
    assert_within_ulps(got, want, _abs_ab(A, B, rows, cols), 2, what=f"oz1 {size} p={p}")
    assert torch.isfinite(C).all()


@pytest.mark.parametrize("N", [12, 14, 16, 18, 20])
def test_config2_oz2_8192(env, N):
    """BASELINE configs[2]: Scheme II DGEMM 8192^3, phi 1, seed 2."""
    torch, O, h = env
    size = 8192
    A, B = G.real_pair(size, size, size, 1.0, 2)
    C = torch.full((size, size), float("nan"), dtype=torch.float64, device="cuda")
    h.dgemm_oz2(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), C, N)
    rows, cols = _samples(size, size, 9)
    got = C[torch.from_numpy(rows).cuda()][:, torch.from_numpy(cols).cuda()].cpu().numpy()
    want = O.oz2_sampled(A, B, N, rows, cols)
    assert_within_ulps(got, want, _abs_ab(A, B, rows, cols), 2, what=f"oz2 N={N}")
    assert torch.isfinite(C).all()


@pytest.mark.parametrize("size,N", [(4096, 14), (4096, 18), (8192, 14), (8192, 18)])
def test_config3_zgemm_3m(env, size, N):
    """BASELINE configs[3]: ZGEMM via 3M, phi 1 on re and im, seed 3."""
    torch, O, h = env
    A, B = G.complex_pair(size, size, size, 1.0, 3)
    C = torch.zeros((size, size), dtype=torch.complex128, device="cuda")
    h.zgemm_oz2_3m(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), C, N)
    rows, cols = _samples(size, size, 11, count=24)
    got = C[torch.from_numpy(rows).cuda()][:, torch.from_numpy(cols).cuda()].cpu().numpy()
    want = O.oz2_sampled(A, B, N, rows, cols, is3m=True)
    scale = (np.abs(A.real[rows]) + np.abs(A.imag[rows])) @ (np.abs(B.real[:, cols]) + np.abs(B.imag[:, cols]))
    assert_within_ulps(got.real, want.real, scale, 2, what="3M re")
    assert_within_ulps(got.imag, want.imag, scale, 2, what="3M im")


def test_config4_tall_skinny_k_chunked(env):
    """BASELINE configs[4]: p = 7, m = n = 1024, k = 65536 -> 4 overflow-safe k-chunks + exact reduction."""
    torch, O, h = env
    m, n, k, p = 1024, 1024, 65536, 7
    A, B = G.real_pair(m, n, k, 1.0, 4)
    C = torch.zeros((m, n), dtype=torch.float64, device="cuda")
    h.dgemm_oz1(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), C, p)
    rows, cols = _samples(m, n, 13)
    got = C[torch.from_numpy(rows).cuda()][:, torch.from_numpy(cols).cuda()].cpu().numpy()
    assert_within_ulps(got, O.oz1_sampled(A, B, p, rows, cols), _abs_ab(A, B, rows, cols), 2, what="k=65536")


def test_config4_wide_m_narrow_n(env):
    """BASELINE configs[4]: p = 7, m = 16384, n = 256, k = 4096."""
    torch, O, h = env
    m, n, k, p = 16384, 256, 4096, 7
    A, B = G.real_pair(m, n, k, 1.0, 4)
    C = torch.zeros((m, n), dtype=torch.float64, device="cuda")
    h.dgemm_oz1(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), C, p)
    rows, cols = _samples(m, n, 15)
    got = C[torch.from_numpy(rows).cuda()][:, torch.from_numpy(cols).cuda()].cpu().numpy()
    assert_within_ulps(got, O.oz1_sampled(A, B, p, rows, cols), _abs_ab(A, B, rows, cols), 2, what="16384x256")


@pytest.mark.parametrize("p", [3, 4])
def test_config4_sgemm_16384(env, p):
    """BASELINE configs[4]: FP32-input emulation at m = n = k = 16384."""
    torch, O, h = env
    size = 16384
    A, B = G.real_pair(size, size, size, 1.0, 4, dtype=np.float32)
    C = torch.zeros((size, size), dtype=torch.float32, device="cuda")
    h.sgemm_oz1(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), C, p)
    rows, cols = _samples(size, size, 17, count=24)
    got = C[torch.from_numpy(rows).cuda()][:, torch.from_numpy(cols).cuda()].cpu().numpy()
    want = O.oz1_sampled(A, B, p, rows, cols, is_f32=True)
    assert_within_ulps(got, want, _abs_ab(A, B, rows, cols), 2, bits=23, what=f"sgemm 16384 p={p}")


# ---- SURVEY 8(d) "Checks" column at full size: integer intermediates ----
def test_full_size_slices_bit_exact(env):
    """configs[1]: ALL slices of the 8192 x 8192 operands (p = 8, phi = 2), rows of A and columns of B, bit for bit."""
    torch, O, h = env
    size, p = 8192, 8
    A, B = G.real_pair(size, size, size, 2.0, 1)
    for X, by_cols in ((A, False), (B, True)):
        S, e = h.dbg_oz1_slices(torch.from_numpy(X).cuda(), by_cols, p)
        oe = O.col_exponents(X) if by_cols else O.row_exponents(X)
        assert np.array_equal(e.cpu().numpy(), oe)
        want = O.oz1_slices_cols(X, oe, p) if by_cols else O.oz1_slices_rows(X, oe, p)
        got = S.cpu().numpy()
        del S
        assert np.array_equal(got, want), f"slices differ (by_cols={by_cols})"


def test_full_size_residues_bit_exact(env):
    """configs[2]: ALL residues of the 8192 x 8192 operands (N = 16, phi = 1, seed 2), bit for bit."""
    torch, O, h = env
    size, N = 8192, 16
    A, B = G.real_pair(size, size, size, 1.0, 2)
    _, tA, tB = O.oz2_budget(N, size)
    for X, by_cols, t in ((A, False, tA), (B, True, tB)):
        R, e = h.dbg_oz2_residues(torch.from_numpy(X).cuda(), by_cols, N, t)
        oe = O.col_exponents(X) if by_cols else O.row_exponents(X)
        assert np.array_equal(e.cpu().numpy(), oe)
        want = O.oz2_residues_cols(X, oe, t, N) if by_cols else O.oz2_residues_rows(X, oe, t, N)
        got = R.cpu().numpy()
        del R
        assert np.array_equal(got, want), f"residues differ (by_cols={by_cols})"


@pytest.mark.parametrize("p", [8, 3])
def test_int32_dump_4096(env, p):
    """INT32 accumulators of the fused kernel at 4096^3 (p = 8: N-concatenated one-CTA kernel; p = 3: the cta_group::2
    pair kernel): 96 sampled rows x 160 sampled columns of all p accumulators, bit for bit against the oracle's int64
    slice products (the full dump is 4096^2 p values; the oracle's plain loops finish the sample in seconds)."""
    torch, O, h = env
    size = 4096
    A, B = G.real_pair(size, size, size, 0.5, 1)
    acc = h.dbg_oz1_accumulators(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), p)
    assert acc.shape == (1, p, size, size)
    rows = G.sample_indices(size, 88, 21)[:96]
    cols = G.sample_indices(size, 152, 22)[:160]
    got = acc[0][:, torch.from_numpy(rows).cuda()][:, :, torch.from_numpy(cols).cuda()].cpu().numpy().astype(np.int64)
    del acc
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    SA = O.oz1_slices_rows(A[rows], eA[rows], p)
    SB = O.oz1_slices_cols(np.ascontiguousarray(B[:, cols]), eB[cols], p)
    assert np.array_equal(got, O.oz1_accumulators(SA, SB))


def test_output_residues_8192(env):
    """configs[2]: per-modulus output residues of the fused mod-GEMM at 8192^3, N = 16, sampled 64 x 64 per modulus."""
    torch, O, h = env
    size, N = 8192, 16
    A, B = G.real_pair(size, size, size, 1.0, 2)
    _, tA, tB = O.oz2_budget(N, size)
    eA, eB = O.row_exponents(A), O.col_exponents(B)
    RA, RB = O.oz2_residues_rows(A, eA, tA, N), O.oz2_residues_cols(B, eB, tB, N)
    out = h.dbg_oz2_modgemm(torch.from_numpy(RA).cuda(), torch.from_numpy(RB).cuda())
    rows = G.sample_indices(size, 56, 23)[:64]
    cols = G.sample_indices(size, 56, 24)[:64]
    got = out[:, torch.from_numpy(rows).cuda()][:, :, torch.from_numpy(cols).cuda()].cpu().numpy()
    del out
    want, _, _ = O.oz2_modprod(np.ascontiguousarray(RA[:, rows]), np.ascontiguousarray(RB[:, cols]))
    assert np.array_equal(got, want)


def test_output_residues_3m_4096(env):
    """configs[3]: 3M output residues (re, im) at 4096^3, N = 14, sampled."""
    torch, O, h = env
    size, N = 4096, 14
    A, B = G.complex_pair(size, size, size, 1.0, 3)
    _, tA, tB = O.oz2_budget(N, size, True)
    RA3 = O.oz2_residues_z(A, O.row_exponents_z(A), tA, N, False)
    RB3 = O.oz2_residues_z(B, O.col_exponents_z(B), tB, N, True)
    out = h.dbg_oz2_modgemm(torch.from_numpy(RA3).cuda(), torch.from_numpy(RB3).cuda(), is3m=True)
    rows = G.sample_indices(size, 40, 25)[:48]
    cols = G.sample_indices(size, 40, 26)[:48]
    got = out[:, :, torch.from_numpy(rows).cuda()][:, :, :, torch.from_numpy(cols).cuda()].cpu().numpy()
    del out
    want = O.oz2_modprod_3m(np.ascontiguousarray(RA3[:, :, rows]), np.ascontiguousarray(RB3[:, :, cols]))
    assert np.array_equal(got, want)


# ---- SURVEY 8(f) features at the sizes bench.py's `detail` legs run them ----------------------------------------
def test_8bit_digits_p7_8192(env):
    """R23: balanced base-256 digits, p = 7 at 8192^3 (bench detail f1), sampled against the oracle's 8-bit mode."""
    torch, O, _ = env
    import paper_2606_25453_b200 as E
    size, p = 8192, 7
    A, B = G.real_pair(size, size, size, 0.5, 1)
    h = E.EmuGemm()
    try:
        h.set_slice_bits(8)
        O.set_slice_bits(8)
        C = torch.full((size, size), float("nan"), dtype=torch.float64, device="cuda")
        h.dgemm_oz1(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), C, p)
        rows, cols = _samples(size, size, 23)
        got = C[torch.from_numpy(rows).cuda()][:, torch.from_numpy(cols).cuda()].cpu().numpy()
        want = O.oz1_sampled(A, B, p, rows, cols)
    finally:
        O.set_slice_bits(7)
        h.close()
    assert_within_ulps(got, want, _abs_ab(A, B, rows, cols), 2, what="8-bit digits p=7 8192")
    assert torch.isfinite(C).all()


def test_strided_batched_64x512_p8(env):
    """64 products of 512^3 through ONE fused launch (bench detail f2); every entry sampled."""
    torch, O, h = env
    batch, s, p = 64, 512, 8
    rng = np.random.default_rng(31)
    A = (rng.random((batch, s, s)) - 0.5) * np.exp(0.5 * rng.standard_normal((batch, s, s)))
    B = (rng.random((batch, s, s)) - 0.5) * np.exp(0.5 * rng.standard_normal((batch, s, s)))
    C = torch.full((batch, s, s), float("nan"), dtype=torch.float64, device="cuda")
    h.dgemm_oz1_strided_batched(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), C, p)
    rows, cols = _samples(s, s, 29, count=8)
    Cs = C[:, torch.from_numpy(rows).cuda()][:, :, torch.from_numpy(cols).cuda()].cpu().numpy()
    for b in range(batch):
        want = O.oz1_sampled(A[b], B[b], p, rows, cols)
        assert_within_ulps(Cs[b], want, _abs_ab(A[b], B[b], rows, cols), 2, what=f"batched entry {b}")
    assert torch.isfinite(C).all()


def test_zgemm_4m_2048_p8(env):
    """Scheme I complex by 4M at 2048^3, p = 8: sampled against the oracle's real products of the embedding
    (re = Re A Re B - Im A Im B as ONE sliced product of [Re A, -Im A] [Re B; Im B], likewise im: oracle_zgemm_oz1_4m's definition)."""
    torch, O, h = env
    size, p = 2048, 8
    A, B = G.complex_pair(size, size, size, 1.0, 3)
    C = torch.zeros((size, size), dtype=torch.complex128, device="cuda")
    h.zgemm_oz1_4m(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), C, p)
    rows, cols = _samples(size, size, 37, count=12)
    got = C[torch.from_numpy(rows).cuda()][:, torch.from_numpy(cols).cuda()].cpu().numpy()
    # the real embedding: A' = [[Re A, -Im A], [Im A, Re A]] (2m x 2k), B' = [[Re B], [Im B]] (2k x n)
    Ae = np.block([[A.real, -A.imag], [A.imag, A.real]])
    Be = np.vstack([B.real, B.imag])
    want_re = O.oz1_sampled(Ae, Be, p, rows, cols)
    want_im = O.oz1_sampled(Ae, Be, p, rows + size, cols)
    scale = (np.abs(A.real[rows]) + np.abs(A.imag[rows])) @ (np.abs(B.real[:, cols]) + np.abs(B.imag[:, cols]))
    assert_within_ulps(got.real, want_re, scale, 2, what="4M re")
    assert_within_ulps(got.imag, want_im, scale, 2, what="4M im")


# ---- SURVEY 8(c) reading R1 (sign-magnitude digits, emugemm_set_slice_form(h, 1)) at full size ----------------------
# The default digit form is R24; R1, the reading SURVEY 8(c) lists, stays a complete mode: the same checks as above
# on BASELINE configs[1] points, against the oracle's R1 mode.
def test_sign_magnitude_form_full_size(env):
    torch, O, _ = env
    import paper_2606_25453_b200 as E
    size = 8192
    A, B = G.real_pair(size, size, size, 2.0, 1)
    dA, dB = torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()
    h = E.EmuGemm()
    try:
        h.set_slice_form(1)
        O.set_slice_bits(O.DIGITS_SIGNMAG)
        # all slices of the 8192 x 8192 operands, bit for bit
        for X, dX, by_cols in ((A, dA, False), (B, dB, True)):
            S, e = h.dbg_oz1_slices(dX, by_cols, 8)
            oe = O.col_exponents(X) if by_cols else O.row_exponents(X)
            want = O.oz1_slices_cols(X, oe, 8) if by_cols else O.oz1_slices_rows(X, oe, 8)
            got = S.cpu().numpy()
            del S
            assert np.array_equal(e.cpu().numpy(), oe) and np.array_equal(got, want), f"R1 slices differ (by_cols={by_cols})"
            assert got.min() >= -127 and got[1:].min() < 0          # sign-magnitude: lower slices carry signs
        rows, cols = _samples(size, size, 7)
        for p in (8, 3):
            C = torch.full((size, size), float("nan"), dtype=torch.float64, device="cuda")
            h.dgemm_oz1(dA, dB, C, p)
            got = C[torch.from_numpy(rows).cuda()][:, torch.from_numpy(cols).cuda()].cpu().numpy()
            assert_within_ulps(got, O.oz1_sampled(A, B, p, rows, cols), _abs_ab(A, B, rows, cols), 2, what=f"R1 8192 p={p}")
            assert torch.isfinite(C).all()
    finally:
        O.set_slice_bits(7)
        h.close()
