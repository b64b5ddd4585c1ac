"""-m gpu: complex64 GEMM (emugemm_cgemm_oz1_4m, emugemm_cgemm_oz2_3m) against the oracle: 2 FP32 ulp of
(|A||B|)_ij per component."""
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


@pytest.mark.parametrize("kind,pn,shape", [("4m", 3, (256, 256, 256)), ("4m", 4, (150, 270, 333)), ("3m", 9, (200, 136, 260)),
                                           ("3m", 11, (129, 257, 130))])
def test_cgemm(env, kind, pn, shape):
    torch, O, h = env
    m, n, k = shape
    Az, Bz, Cz = G.complex_pair(m, n, k, 1.0, 3, with_c=True)
    A, B, Cin = Az.astype(np.complex64), Bz.astype(np.complex64), Cz.astype(np.complex64)
    al, be = 0.5 - 2j, 1.5 + 0.25j
    C = dev(torch, Cin)
    if kind == "4m":
        h.cgemm_oz1_4m(dev(torch, A), dev(torch, B), C, pn, alpha=al, beta=be)
        want = O.cgemm_oz1_4m(A, B, pn, alpha=al, beta=be, Cin=Cin)
    else:
        h.cgemm_oz2_3m(dev(torch, A), dev(torch, B), C, pn, alpha=al, beta=be)
        want = O.cgemm_oz2_3m(A, B, pn, alpha=al, beta=be, Cin=Cin)
    _, absZ = O.bf128_zgemm(A.astype(np.complex128), B.astype(np.complex128))
    scale = abs(al) * 2 * absZ + abs(be) * 2 * np.abs(Cin).astype(np.float64)
    got = C.cpu().numpy()
    assert_within_ulps(got.real, want.real, scale, 2, bits=23, what=f"cgemm {kind} re")
    assert_within_ulps(got.imag, want.imag, scale, 2, bits=23, what=f"cgemm {kind} im")


def test_cgemm_gaussian_integers_exact_and_k_zero(env):
    torch, O, h = env
    rng = np.random.default_rng(3)
    A = (rng.integers(-31, 32, size=(140, 200)) + 1j * rng.integers(-31, 32, size=(140, 200))).astype(np.complex64)
    B = (rng.integers(-31, 32, size=(200, 90)) + 1j * rng.integers(-31, 32, size=(200, 90))).astype(np.complex64)
    want = (A.astype(np.complex128) @ B.astype(np.complex128)).astype(np.complex64)
    C = torch.zeros((140, 90), dtype=torch.complex64, device="cuda")
    h.cgemm_oz1_4m(dev(torch, A), dev(torch, B), C, 3)
    assert np.array_equal(C.cpu().numpy(), want)
    h.cgemm_oz2_3m(dev(torch, A), dev(torch, B), C, 8)
    assert np.array_equal(C.cpu().numpy(), want)
    Az = torch.zeros((3, 0), dtype=torch.complex64, device="cuda")
    Bz = torch.zeros((0, 2), dtype=torch.complex64, device="cuda")
    Cz = torch.full((3, 2), 1 + 2j, dtype=torch.complex64, device="cuda")
    h.cgemm_oz2_3m(Az, Bz, Cz, 8, beta=1j)
    assert torch.allclose(Cz, torch.full((3, 2), -2 + 1j, dtype=torch.complex64, device="cuda"))
