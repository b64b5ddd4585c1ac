"""-m gpu: seeded random sweep over shapes (ragged, tiny, tile-boundary), slice / moduli counts, digit formats,
transposition flags, leading dimensions and alpha / beta for every entry point, each case against the oracle
(2 ulp of |alpha| (|A||B|)_ij + |beta| |C_in|_ij; FP32 entry points in FP32 ulps)."""
import numpy as np
import pytest

import emugemm_inputs as G
from gpu_util import assert_within_ulps

pytestmark = pytest.mark.gpu

SIZES = [1, 2, 7, 31, 63, 64, 65, 127, 128, 129, 160, 255, 256, 257, 300]


@pytest.fixture(scope="module")
def env():
    import torch
    from oracle import oracle as O
    import paper_2606_25453_b200 as E
    h = E.EmuGemm()
    yield torch, O, h
    O.set_slice_bits(7)
    h.close()


def _padded(torch, X, pad):
    """device copy of X inside a wider allocation (ld = cols + pad), returned as the strided view"""
    r, c = X.shape
    buf = torch.zeros((r, c + pad), dtype=torch.from_numpy(X[:0]).dtype, device="cuda")
    buf[:, :c] = torch.from_numpy(np.ascontiguousarray(X)).cuda()
    return buf[:, :c]


def _pick(rng, cplx, f32):
    m, n, k = (int(rng.choice(SIZES)) for _ in range(3))
    phi = float(rng.choice([0.5, 1.0, 2.0]))
    seed = int(rng.integers(0, 10 ** 6))
    if cplx:
        A, B, Cin = G.complex_pair(m, n, k, phi, seed, with_c=True)
    else:
        A, B, Cin = G.real_pair(m, n, k, phi, seed, dtype=np.float32 if f32 else np.float64, with_c=True)
    return m, n, k, A, B, Cin


@pytest.mark.parametrize("case", range(40))
def test_random_real(env, case):
    torch, O, h = env
    rng = np.random.default_rng(1000 + case)
    scheme = ["oz1d", "oz1s", "oz2d", "oz2s"][case % 4]
    f32 = scheme.endswith("s")
    m, n, k, A, B, Cin = _pick(rng, False, f32)
    ta, tb = bool(rng.integers(0, 2)), bool(rng.integers(0, 2))
    use_beta = bool(rng.integers(0, 2))
    alpha = float(rng.choice([1.0, -1.5, 0.25]))
    beta = float(rng.choice([0.75, -2.0])) if use_beta else 0.0
    bits = 8 if (scheme.startswith("oz1") and rng.integers(0, 2)) else 7
    if scheme.startswith("oz1"):
        pn = int(rng.integers(1, 5 if f32 else 9))
    else:
        pn = int(rng.integers(8, 12)) if f32 else int(rng.integers(10, 21))
    Ad = _padded(torch, A.T if ta else A, int(rng.choice([0, 2, 6])) * (2 if not f32 else 4))
    Bd = _padded(torch, B.T if tb else B, int(rng.choice([0, 2, 6])) * (2 if not f32 else 4))
    Cd = _padded(torch, Cin, int(rng.choice([0, 4])) * (1 if not f32 else 1))
    h.set_slice_bits(bits)
    O.set_slice_bits(bits)
    try:
        call = {"oz1d": h.dgemm_oz1, "oz1s": h.sgemm_oz1, "oz2d": h.dgemm_oz2, "oz2s": h.sgemm_oz2}[scheme]
        ora = {"oz1d": O.dgemm_oz1, "oz1s": O.sgemm_oz1, "oz2d": O.dgemm_oz2, "oz2s": O.sgemm_oz2}[scheme]
        call(Ad, Bd, Cd, pn, alpha=alpha, beta=beta, transa=ta, transb=tb)
        want = ora(A, B, pn, alpha=alpha, beta=beta, Cin=Cin if use_beta else None)
    finally:
        h.set_slice_bits(7)
        O.set_slice_bits(7)
    _, absAB = O.bf128_dgemm(A.astype(np.float64), B.astype(np.float64))
    scale = abs(alpha) * absAB + abs(beta) * np.abs(Cin).astype(np.float64)
    assert_within_ulps(Cd.cpu().numpy(), want, scale, 2, bits=23 if f32 else 52,
                       what=f"{scheme} m={m} n={n} k={k} pn={pn} bits={bits} ta={ta} tb={tb} a={alpha} b={beta}")


@pytest.mark.parametrize("case", range(16))
def test_random_complex(env, case):
    torch, O, h = env
    rng = np.random.default_rng(5000 + case)
    m, n, k, A, B, Cin = _pick(rng, True, False)
    use_beta = bool(rng.integers(0, 2))
    alpha = complex(rng.choice([1.0, 0.5 - 2j, -1j]))
    beta = complex(rng.choice([1.5 + 0.25j, -1.0])) if use_beta else 0j
    Ad, Bd, Cd = _padded(torch, A, int(rng.choice([0, 3]))), _padded(torch, B, int(rng.choice([0, 5]))), _padded(torch, Cin, 0)
    if case % 2 == 0:
        N = int(rng.integers(12, 21))
        h.zgemm_oz2_3m(Ad, Bd, Cd, N, alpha=alpha, beta=beta)
        want = O.zgemm_oz2_3m(A, B, N, alpha=alpha, beta=beta, Cin=Cin if use_beta else None)
        what = f"3M m={m} n={n} k={k} N={N}"
    else:
        p = int(rng.integers(2, 9))
        h.zgemm_oz1_4m(Ad, Bd, Cd, p, alpha=alpha, beta=beta)
        want = O.zgemm_oz1_4m(A, B, p, alpha=alpha, beta=beta, Cin=Cin if use_beta else None)
        what = f"4M m={m} n={n} k={k} p={p}"
    _, absZ = O.bf128_zgemm(A, B)
    scale = abs(alpha) * 2 * absZ + abs(beta) * 2 * np.abs(Cin)
    got = Cd.cpu().numpy()
    assert_within_ulps(got.real, want.real, scale, 2, what=what + " re")
    assert_within_ulps(got.imag, want.imag, scale, 2, what=what + " im")


@pytest.mark.parametrize("case", range(12))
def test_random_batched(env, case):
    """strided batched Scheme I: random shapes (sizes that keep every entry 16-byte aligned), counts, digit formats,
    batch strides with slack, optionally one shared operand."""
    torch, O, h = env
    rng = np.random.default_rng(7000 + case)
    f32 = bool(case % 3 == 2)
    q = 4 if f32 else 2                                   # elements per 16 bytes
    m, n, k = (int(rng.choice([2, 8, 30, 64, 66, 128, 130, 160, 258])) for _ in range(3))
    batch = int(rng.integers(2, 7))
    p = int(rng.integers(1, 5 if f32 else 9))
    bits = 8 if rng.integers(0, 2) else 7
    share_b = bool(rng.integers(0, 2))
    use_beta = bool(rng.integers(0, 2))
    alpha = float(rng.choice([1.0, -1.5, 0.25]))
    beta = float(rng.choice([0.75, -2.0])) if use_beta else 0.0
    dt = np.float32 if f32 else np.float64
    tdt = torch.float32 if f32 else torch.float64
    A = np.stack([G.real_pair(m, n, k, 1.0, 10 * case + b, dtype=dt)[0] for b in range(batch)])
    Bs = [G.real_pair(m, n, k, 1.0, 500 + 10 * case + b, dtype=dt)[1] for b in range(1 if share_b else batch)]
    Cin = np.random.default_rng(case).standard_normal((batch, m, n)).astype(dt)
    rows_pad, pad = int(rng.integers(0, 3)), q * int(rng.integers(0, 3))   # slack rows between entries, ld slack
    Ab = torch.zeros((batch, m + rows_pad, k + pad), dtype=tdt, device="cuda")
    Ab[:, :m, :k] = torch.from_numpy(A).cuda()
    if share_b:
        Bb = torch.zeros((k, n + pad), dtype=tdt, device="cuda")
        Bb[:, :n] = torch.from_numpy(Bs[0]).cuda()
        Bv = Bb[:, :n]
    else:
        Bb = torch.zeros((batch, k + rows_pad, n + pad), dtype=tdt, device="cuda")
        Bb[:, :k, :n] = torch.from_numpy(np.stack(Bs)).cuda()
        Bv = Bb[:, :k, :n]
    Cb = torch.zeros((batch, m + rows_pad, n + pad), dtype=tdt, device="cuda")
    Cb[:, :m, :n] = torch.from_numpy(Cin).cuda()
    for t in (Ab, Bb, Cb):   # entries must stay 16-byte aligned: skip draws whose batch stride is not
        if t.dim() == 3 and (t.stride(0) * t.element_size()) % 16:
            pytest.skip("batch stride not 16-byte aligned for this draw")
    h.set_slice_bits(bits)
    O.set_slice_bits(bits)
    try:
        call = h.sgemm_oz1_strided_batched if f32 else h.dgemm_oz1_strided_batched
        call(Ab[:, :m, :k], Bv, Cb[:, :m, :n], p, alpha=alpha, beta=beta)
        got = Cb.cpu().numpy()
        for b in range(batch):
            Bm = Bs[0] if share_b else Bs[b]
            _, absAB = O.bf128_dgemm(A[b].astype(np.float64), Bm.astype(np.float64))
            ref = (O.sgemm_oz1 if f32 else O.dgemm_oz1)(A[b], Bm, p, alpha=alpha, beta=beta, Cin=Cin[b] if use_beta else None)
            scale = abs(alpha) * absAB + abs(beta) * np.abs(Cin[b].astype(np.float64))
            assert_within_ulps(got[b, :m, :n], ref, scale, 2, bits=23 if f32 else 52,
                               what=f"case {case} entry {b} {m}x{n}x{k} p={p} bits={bits} f32={f32}")
    finally:
        h.set_slice_bits(7)
        O.set_slice_bits(7)
