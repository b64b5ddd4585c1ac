"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side tests / bench.

Holds NONE of the method's arithmetic: only the paper's input distribution
(Eq. 19: a_ij = (rand - 0.5) * exp(phi * randn)) and the config
table of BASELINE.json.  Recipe: rng = numpy.random.default_rng(seed);
for each matrix in the order A, B (then C if beta != 0): U = rng.random(shape),
Z = rng.standard_normal(shape), M = (U - 0.5) * exp(phi * Z) in FP64.  Complex: the
real part is drawn first, then the imaginary part, same recipe.  FP32 configs cast
the FP64 draw to float32.  The identical bytes go to the oracle and to the GPU.
"""
import numpy as np


def _draw(rng, shape, phi):
    u = rng.random(shape)
    z = rng.standard_normal(shape)
    return (u - 0.5) * np.exp(phi * z)


def real_pair(m, n, k, phi, seed, dtype=np.float64, with_c=False):
    """(A m x k, B k x n[, C m x n]) in the paper's distribution."""
    rng = np.random.default_rng(seed)
    A = _draw(rng, (m, k), phi)
    B = _draw(rng, (k, n), phi)
    out = [A.astype(dtype), B.astype(dtype)]
    if with_c:
        out.append(_draw(rng, (m, n), phi).astype(dtype))
    return tuple(out)


def complex_pair(m, n, k, phi, seed, with_c=False):
    rng = np.random.default_rng(seed)

    def z(shape):
        re = _draw(rng, shape, phi)
        im = _draw(rng, shape, phi)
        return re + 1j * im

    out = [z((m, k)), z((k, n))]
    if with_c:
        out.append(z((m, n)))
    return tuple(out)


def sample_indices(size, count, seed, tile=128):
    """Sorted unique indices: `count` random ones plus the first/last index and both
    sides of every `tile` boundary near the ends (SURVEY 8(c) 'Parity at large sizes')."""
    rng = np.random.default_rng(seed)
    idx = set(int(x) for x in rng.integers(0, size, size=min(count, size)))
    for x in (0, 1, size - 1, size - 2, tile - 1, tile, size - tile - 1, size - tile):
        if 0 <= x < size:
            idx.add(int(x))
    return np.array(sorted(idx), dtype=np.int64)


# BASELINE.json configs (index -> description), used by tests and bench.py.
CONFIGS = {
    0: dict(kind="oz1_d", shapes=[(256, 256, 256)], phi=[0.5], seed=0, p=[6]),
    1: dict(kind="oz1_d", shapes=[(s, s, s) for s in (2048, 4096, 8192, 16384)], phi=[0.5, 2.0], seed=1,
            p=[3, 4, 5, 6, 7, 8]),
    2: dict(kind="oz2_d", shapes=[(8192, 8192, 8192)], phi=[1.0], seed=2, N=[12, 14, 16, 18, 20]),
    3: dict(kind="oz2_z3m", shapes=[(4096, 4096, 4096), (8192, 8192, 8192)], phi=[1.0], seed=3, N=[14, 18]),
    4: dict(kind="oz1_mixed", seed=4, phi=[1.0],
            cases=[dict(prec="s", shape=(16384, 16384, 16384), p=3), dict(prec="s", shape=(16384, 16384, 16384), p=4),
                   dict(prec="d", shape=(1024, 1024, 65536), p=7), dict(prec="d", shape=(16384, 256, 4096), p=7)]),
}
