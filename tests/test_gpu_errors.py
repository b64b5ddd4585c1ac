"""-m gpu: error behaviour of the C ABI (include/emugemm.h "Return value"): invalid arguments, alignment,
workspace and precision errors are reported as negative status codes -- no exception from the library, no
silent fallback -- and degenerate sizes are no-ops."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    import paper_2606_25453_b200 as E
    h = E.EmuGemm()
    yield torch, E, h
    h.close()


def _call_d(E, h, fn, m, n, k, A, lda, B, ldb, Cc, ldc, pn):
    i64, dbl, vp = C.c_int64, C.c_double, C.c_void_p
    return getattr(h._lib, fn)(h._h, i64(m), i64(n), i64(k), dbl(1.0), vp(A), i64(lda), vp(B), i64(ldb), dbl(0.0), vp(Cc), i64(ldc),
                               C.c_int(pn))


def test_status_codes(env):
    torch, E, h = env
    m = n = k = 256
    A = torch.zeros((m, k), dtype=torch.float64, device="cuda")
    B = torch.zeros((k, n), dtype=torch.float64, device="cuda")
    Cm = torch.zeros((m, n), dtype=torch.float64, device="cuda")
    h.reserve(h.workspace_bytes(E.binding.OZ2, 8, m, n, k, 20))
    a, b, c = A.data_ptr(), B.data_ptr(), Cm.data_ptr()
    assert _call_d(E, h, "emugemm_dgemm_oz1", m, n, k, a, k, b, n, c, n, 4) == 0
    assert _call_d(E, h, "emugemm_dgemm_oz1", m, n, k, a, k, b, n, c, n, 0) == -1       # p out of range
    assert _call_d(E, h, "emugemm_dgemm_oz1", m, n, k, a, k, b, n, c, n, 9) == -1
    assert _call_d(E, h, "emugemm_dgemm_oz1", m, n, k, a, k - 1, b, n, c, n, 4) == -1   # lda < k
    assert _call_d(E, h, "emugemm_dgemm_oz1", -1, n, k, a, k, b, n, c, n, 4) == -1      # negative size
    assert _call_d(E, h, "emugemm_dgemm_oz1", m, n, k, a + 8, k, b, n, c, n, 4) == -2   # A not 16-byte aligned
    assert _call_d(E, h, "emugemm_dgemm_oz2", m, n, k, a, k, b, n, c, n, 1) == -1       # n_moduli out of range
    assert _call_d(E, h, "emugemm_dgemm_oz2", m, n, k, a, k, b, n, c, n, 21) == -1
    assert _call_d(E, h, "emugemm_dgemm_oz1", 0, n, k, a, k, b, n, c, n, 4) == 0        # m = 0: no-op
    assert h._lib.emugemm_set_slice_bits(h._h, C.c_int(9)) == -1
    assert h._lib.emugemm_status_string(C.c_int(-3)) == b"workspace missing or too small"


def test_workspace_too_small(env):
    torch, E, h = env
    m = n = k = 512
    A = torch.zeros((m, k), dtype=torch.float64, device="cuda")
    B = torch.zeros((k, n), dtype=torch.float64, device="cuda")
    Cm = torch.zeros((m, n), dtype=torch.float64, device="cuda")
    small = torch.empty(4096 + 1024, dtype=torch.uint8, device="cuda")
    off = (-small.data_ptr()) % 1024
    assert h._lib.emugemm_set_workspace(h._h, C.c_void_p(small.data_ptr() + off), C.c_size_t(4096)) == 0
    assert _call_d(E, h, "emugemm_dgemm_oz1", m, n, k, A.data_ptr(), k, B.data_ptr(), n, Cm.data_ptr(), n, 8) == -3
    assert h._lib.emugemm_set_workspace(h._h, C.c_void_p(small.data_ptr() + off + 8), C.c_size_t(2048)) == -2
    h._ws = None  # let the binding re-reserve for the next test
    h.dgemm_oz1(A, B, Cm, 8)
    assert (Cm == 0).all()


def test_precision_error_and_tiny_budget(env):
    torch, E, h = env
    # 2 moduli: P = 65280; k = 16320 leaves T = 0 < 2 bits -> EMUGEMM_ERR_PRECISION
    T, _, _ = E.oz2_budget(2, 16320)
    assert T < 2
    m, n, k = 8, 8, 16320
    A = torch.ones((m, k), dtype=torch.float64, device="cuda")
    B = torch.ones((k, n), dtype=torch.float64, device="cuda")
    Cm = torch.zeros((m, n), dtype=torch.float64, device="cuda")
    h.reserve(h.workspace_bytes(E.binding.OZ2, 8, m, n, k, 2))
    assert _call_d(E, h, "emugemm_dgemm_oz2", m, n, k, A.data_ptr(), k, B.data_ptr(), n, Cm.data_ptr(), n, 2) == -4


def test_degenerate_oz2_and_3m(env):
    torch, E, h = env
    A = torch.zeros((5, 0), dtype=torch.float64, device="cuda")
    B = torch.zeros((0, 4), dtype=torch.float64, device="cuda")
    Cm = torch.ones((5, 4), dtype=torch.float64, device="cuda")
    h.dgemm_oz2(A, B, Cm, 12, beta=3.0)  # k = 0: C <- beta C
    assert (Cm == 3.0).all()
    Az = torch.zeros((3, 0), dtype=torch.complex128, device="cuda")
    Bz = torch.zeros((0, 2), dtype=torch.complex128, device="cuda")
    Cz = torch.full((3, 2), 1 + 2j, dtype=torch.complex128, device="cuda")
    h.zgemm_oz2_3m(Az, Bz, Cz, 14, beta=1j)
    assert torch.allclose(Cz, torch.full((3, 2), -2 + 1j, dtype=torch.complex128, device="cuda"))
    Z = torch.zeros((130, 130), dtype=torch.float64, device="cuda")
    Cc = torch.ones((130, 130), dtype=torch.float64, device="cuda")
    h.dgemm_oz2(Z, Z, Cc, 16)  # all-zero operands
    assert (Cc == 0).all()


def test_nonfinite_flag(env):
    """non-finite inputs give an unspecified result and no fault; the pre-pass raises a flag."""
    import numpy as np
    torch, E, h = env[0], env[1], env[2]
    A = torch.rand((70, 130), dtype=torch.float64, device="cuda") - 0.5
    B = torch.rand((130, 50), dtype=torch.float64, device="cuda") - 0.5
    C = torch.zeros((70, 50), dtype=torch.float64, device="cuda")
    h.dgemm_oz1(A, B, C, 4)
    assert h.nonfinite_seen() is False
    for bad, where in ((float("inf"), "A"), (float("nan"), "B"), (-float("inf"), "B")):
        A2, B2 = A.clone(), B.clone()
        (A2 if where == "A" else B2)[3, 7] = bad
        h.dgemm_oz1(A2, B2, C, 4)
        assert h.nonfinite_seen() is True
        h.dgemm_oz2(A2, B2, C, 12)
        assert h.nonfinite_seen() is True
    h.dgemm_oz2(A, B, C, 12)
    assert h.nonfinite_seen() is False   # the flag describes the last call only
    Z = (torch.rand((40, 64), dtype=torch.float64, device="cuda") - 0.5).to(torch.complex128)
    Z[1, 2] = complex(0.0, float("nan"))
    W = (torch.rand((64, 30), dtype=torch.float64, device="cuda") - 0.5).to(torch.complex128)
    Cz = torch.zeros((40, 30), dtype=torch.complex128, device="cuda")
    h.zgemm_oz2_3m(Z, W, Cz, 14)
    assert h.nonfinite_seen() is True
    torch.cuda.synchronize()  # no fault: the device is still usable
    h.dgemm_oz1(A, B, C, 4)
    assert torch.isfinite(C).all()


def test_two_handles_on_two_streams_with_wave_barrier(env):
    """The grid-wide wave barrier of the fused kernels is an optimisation with a bounded wait that gives up
    (csrc/ptx.cuh): two handles issuing such kernels on two streams at once -- their CTAs are then NOT all co-resident --
    must complete and give the results of the serial calls."""
    torch, E, h = env
    m, n, k, p = 4096, 4096, 8192, 8   # 64 KB of slices per operand row: the barrier is on
    A = torch.rand((m, k), dtype=torch.float64, device="cuda") - 0.5
    B = torch.rand((k, n), dtype=torch.float64, device="cuda") - 0.5
    ref = torch.empty((m, n), dtype=torch.float64, device="cuda")
    h.dgemm_oz1(A, B, ref, p)
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    h1, h2 = E.EmuGemm(), E.EmuGemm()
    h1.set_stream(s1); h2.set_stream(s2)
    C1 = torch.empty_like(ref); C2 = torch.empty_like(ref)
    try:
        for _ in range(3):
            with torch.cuda.stream(s1):
                h1.dgemm_oz1(A, B, C1, p)
            with torch.cuda.stream(s2):
                h2.dgemm_oz1(A, B, C2, p)
        torch.cuda.synchronize()
        assert torch.equal(C1, ref) and torch.equal(C2, ref)
    finally:
        h1.close(); h2.close()
