"""-m gpu: Scheme I complex GEMM by 4M (emugemm_zgemm_oz1_4m) against the oracle's 4M on the real
embedding: final values within 2 ulp of (|A||B|)_ij per component, both digit formats, alpha / beta, ragged sizes."""
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
    O.set_slice_bits(7)
    h.close()


def dev(torch, x):
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("bits,p,shape", [(7, 6, (256, 256, 256)), (7, 3, (150, 270, 333)), (7, 8, (130, 70, 200)),
                                          (8, 7, (200, 136, 260)), (8, 4, (129, 257, 130))])
def test_zgemm_oz1_4m(env, bits, p, shape):
    torch, O, h = env
    m, n, k = shape
    h.set_slice_bits(bits)
    O.set_slice_bits(bits)
    try:
        A, B = G.complex_pair(m, n, k, 1.0, 3)
        C = torch.full((m, n), float("nan"), dtype=torch.complex128, device="cuda")
        h.zgemm_oz1_4m(dev(torch, A), dev(torch, B), C, p)
        want = O.zgemm_oz1_4m(A, B, p)
        _, absZ = O.bf128_zgemm(A, B)
        got = C.cpu().numpy()
        assert_within_ulps(got.real, want.real, absZ, 2, what=f"4M re bits={bits} p={p}")
        assert_within_ulps(got.imag, want.imag, absZ, 2, what=f"4M im bits={bits} p={p}")
    finally:
        h.set_slice_bits(7)
        O.set_slice_bits(7)


def test_alpha_beta_and_k_zero(env):
    torch, O, h = env
    m, n, k, p = 100, 64, 128, 6
    A, B, Cin = G.complex_pair(m, n, k, 1.0, 8, with_c=True)
    C = dev(torch, Cin)
    al, be = 0.5 - 2j, 1.5 + 0.25j
    h.zgemm_oz1_4m(dev(torch, A), dev(torch, B), C, p, alpha=al, beta=be)
    want = O.zgemm_oz1_4m(A, B, p, alpha=al, beta=be, Cin=Cin)
    _, absZ = O.bf128_zgemm(A, B)
    scale = abs(al) * 2 * absZ + abs(be) * 2 * np.abs(Cin)
    got = C.cpu().numpy()
    assert_within_ulps(got.real, want.real, scale, 2)
    assert_within_ulps(got.imag, want.imag, scale, 2)
    Az = torch.zeros((3, 0), dtype=torch.complex128, device="cuda")
    Bz = torch.zeros((0, 2), dtype=torch.complex128, device="cuda")
    Cz = torch.full((3, 2), 1 + 2j, dtype=torch.complex128, device="cuda")
    h.zgemm_oz1_4m(Az, Bz, Cz, 4, beta=1j)
    assert torch.allclose(Cz, torch.full((3, 2), -2 + 1j, dtype=torch.complex128, device="cuda"))


def test_gaussian_integers_exact(env):
    torch, O, h = env
    rng = np.random.default_rng(3)
    A = (rng.integers(-31, 32, size=(140, 200)) + 1j * rng.integers(-31, 32, size=(140, 200))).astype(np.complex128)
    B = (rng.integers(-31, 32, size=(200, 90)) + 1j * rng.integers(-31, 32, size=(200, 90))).astype(np.complex128)
    C = torch.zeros((140, 90), dtype=torch.complex128, device="cuda")
    h.zgemm_oz1_4m(dev(torch, A), dev(torch, B), C, 4)
    assert np.array_equal(C.cpu().numpy(), A @ B)
