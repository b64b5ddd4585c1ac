"""gpu: emugemm_dgemm_oz1_static -- the Scheme I DGEMM whose scratch lives in the library's static device array
(include/emugemm.h; csrc/static_ws.cu), for callers that cannot call cudaMalloc.

Collected LAST on purpose (the file name sorts after every other test file): the suite runs with `pytest -x`, and a
failure here must not hide the parity tests.  The tests pass alone in a fresh process and after the rest of the suite.

The existing path (emugemm_dgemm_oz1 with a caller workspace) is the reference: both run the same kernels over the same
workspace layout on integer accumulators, so the results must agree BIT FOR BIT (tighter than the 2-ulp parity bar)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2606_25453_b200 as E
    h = E.EmuGemm()
    yield torch, E, h
    h.close()


def _operands(torch, m, n, k, seed):
    import emugemm_inputs as I
    A, B = I.real_pair(m, n, k, 1.0, seed)
    return torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()


def test_static_entry_matches_workspace_path_two_calls_in_a_row(env):
    torch, E, h = env
    # call 1: several tiles, ragged m / n, k not a multiple of the 128-column k-block; call 2: another shape and p, so
    # that what call 1 left in the shared array (planes of another geometry, barrier counter) must not matter
    cases = [(300, 260, 1000, 8, 1.0, 0.0), (515, 129, 2300, 5, -0.75, 0.5), (300, 260, 1000, 8, 1.0, 0.0)]
    ref_h = E.EmuGemm()      # its own handle and workspace: the static call must not depend on either
    try:
        outs = []
        for i, (m, n, k, p, alpha, beta) in enumerate(cases):
            A, B = _operands(torch, m, n, k, seed=100 + i)
            C0 = torch.from_numpy(np.random.default_rng(i).standard_normal((m, n))).cuda()
            want = C0.clone()
            ref_h.dgemm_oz1(A, B, want, p, alpha=alpha, beta=beta)
            got = C0.clone()
            h.dgemm_oz1_static(A, B, got, p, alpha=alpha, beta=beta)     # back to back on one stream, no sync between
            outs.append((got, want))
        torch.cuda.synchronize()
        for got, want in outs:
            assert torch.isfinite(want).all()
            assert torch.equal(got, want)
    finally:
        ref_h.close()


def test_static_entry_needs_no_workspace_and_allocates_nothing(env):
    torch, E, _ = env
    h = E.EmuGemm()          # fresh handle: no workspace was ever registered
    try:
        m = n = k = 1024     # the documented maximum at p = 8
        p = 8
        assert h.workspace_bytes(E.OZ1, 8, m, n, k, p) <= h.static_workspace_limit() == 32 << 20
        A, B = _operands(torch, m, n, k, seed=7)
        C1 = torch.empty((m, n), dtype=torch.float64, device="cuda")
        C2 = torch.empty_like(C1)
        want = torch.empty_like(C1)
        h.dgemm_oz1_static(A, B, C1, p)          # first call: module load, per-device set-up of the symbol address
        torch.cuda.synchronize()
        free0, _ = torch.cuda.mem_get_info()
        h.dgemm_oz1_static(A, B, C2, p)
        torch.cuda.synchronize()
        free1, _ = torch.cuda.mem_get_info()
        assert free1 == free0                    # device memory in use did not change: nothing was allocated
        assert h._ws is None                     # the binding reserved no torch workspace either
        E.EmuGemm().dgemm_oz1(A, B, want, p)
        torch.cuda.synchronize()
        assert torch.equal(C1, want) and torch.equal(C2, want)
        assert h.nonfinite_seen() is False       # the diagnostics words of the static call are readable
    finally:
        h.close()


def test_static_entry_rejects_sizes_beyond_the_array(env):
    torch, E, h = env
    m = n = 1024
    k = 2176                 # 2 * 8 * 1024 * 2176 bytes of planes = 34 MiB > 32 MiB
    assert h.workspace_bytes(E.OZ1, 8, m, n, k, 8) > h.static_workspace_limit()
    A = torch.zeros((m, k), dtype=torch.float64, device="cuda")
    B = torch.zeros((k, n), dtype=torch.float64, device="cuda")
    C = torch.full((m, n), 3.0, dtype=torch.float64, device="cuda")
    with pytest.raises(E.EmuGemmError) as ei:
        h.dgemm_oz1_static(A, B, C, 8)
    assert ei.value.status == -7 and "static scratch" in str(ei.value)
    torch.cuda.synchronize()
    assert (C == 3.0).all()  # nothing was enqueued
    h.dgemm_oz1_static(A, B, C, 3)   # the same shape fits with fewer slices
    torch.cuda.synchronize()
    assert (C == 0.0).all()
    with pytest.raises(E.EmuGemmError) as ei:
        h.dgemm_oz1_static(A, B, C, 9)
    assert ei.value.status == -1


def test_static_entry_under_cuda_graph_capture(env):
    """The use case the entry point exists for: the call is captured into a CUDA graph in GLOBAL capture-error mode (a
    cudaMalloc / cudaFree or any other capture-unsafe call during the capture would fail it) and replayed twice."""
    torch, E, _ = env
    h = E.EmuGemm()
    try:
        m, n, k, p = 512, 384, 1000, 8
        A, B = _operands(torch, m, n, k, seed=5)
        want = torch.empty((m, n), dtype=torch.float64, device="cuda")
        E.EmuGemm().dgemm_oz1(A, B, want, p)
        C = torch.empty_like(want)
        h.dgemm_oz1_static(A, B, C, p)     # outside the capture: module load and the per-device symbol-address set-up
        torch.cuda.synchronize()
        s = torch.cuda.Stream()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.stream(s):
            h.set_stream(s)
            with torch.cuda.graph(g, stream=s, capture_error_mode="global"):
                h.dgemm_oz1_static(A, B, C, p)
        for _ in range(2):
            C.zero_()
            torch.cuda.synchronize()
            g.replay()
            torch.cuda.synchronize()
            assert torch.equal(C, want)
    finally:
        h.close()
