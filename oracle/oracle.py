"""ctypes view of oracle/liboracle.so (TEST INFRASTRUCTURE; see emugemm_oracle.c).

Argument marshalling only: numpy arrays in, numpy arrays out (dtype widening of float32 / complex64 inputs to the
C routines' double interface and the matching narrowing of their results included).  Every function cites the C
routine it calls; the arithmetic and its paper citations live there.
"""
import ctypes as C
import numpy as np

from . import build as _build

_lib = C.CDLL(_build.build())

_i64, _i32, _dbl, _flt = C.c_int64, C.c_int32, C.c_double, C.c_float
_p = C.c_void_p
BETA = 7


def _ptr(a):
    return a.ctypes.data_as(_p)


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def threads():
    _lib.oracle_threads.restype = C.c_int
    return int(_lib.oracle_threads())


def set_threads(t):
    _lib.oracle_set_threads(C.c_int(int(t)))


# ---------------------------------------------------------------- exponents
DIGITS_SIGNMAG = 0x207


def set_slice_bits(code):
    """Scheme I digit mode: 7 (default, R24) = 7-bit two's-complement digits, signed leading slice and non-negative
    remaining slices (PAPER.md:345 at beta = 7); DIGITS_SIGNMAG (0x207, R1) = 7-bit sign-magnitude digits; 8 (R23) =
    balanced signed base-256 digits."""
    _lib.oracle_set_slice_bits(C.c_int(code))


def get_slice_bits():
    return int(_lib.oracle_get_slice_bits())


def row_exponents(A):
    A = _f64(A)
    m, k = A.shape
    e = np.empty(m, np.int32)
    _lib.oracle_row_exponents(_i64(m), _i64(k), _ptr(A), _i64(k), _ptr(e))
    return e


def col_exponents(B):
    B = _f64(B)
    k, n = B.shape
    e = np.empty(n, np.int32)
    _lib.oracle_col_exponents(_i64(k), _i64(n), _ptr(B), _i64(n), _ptr(e))
    return e


def _zview(Z):
    Z = np.ascontiguousarray(Z, dtype=np.complex128)
    return Z, Z.view(np.float64)


def row_exponents_z(Z):
    Z, Zf = _zview(Z)
    m, k = Z.shape
    e = np.empty(m, np.int32)
    _lib.oracle_row_exponents_z(_i64(m), _i64(k), _ptr(Zf), _i64(k), _ptr(e))
    return e


def col_exponents_z(Z):
    Z, Zf = _zview(Z)
    k, n = Z.shape
    e = np.empty(n, np.int32)
    _lib.oracle_col_exponents_z(_i64(k), _i64(n), _ptr(Zf), _i64(n), _ptr(e))
    return e


# ---------------------------------------------------------------- Scheme I
def oz1_slices_rows(A, eA, p):
    """int8 [p][m][k] (oracle_oz1_slices_rows)."""
    A = _f64(A)
    m, k = A.shape
    eA = np.ascontiguousarray(eA, np.int32)
    S = np.empty((p, m, k), np.int8)
    _lib.oracle_oz1_slices_rows(_i64(m), _i64(k), _ptr(A), _i64(k), _ptr(eA), C.c_int(p), _ptr(S))
    return S


def oz1_slices_cols(B, eB, p):
    """int8 [p][n][k]: slices of the COLUMNS of B (oracle_oz1_slices_cols)."""
    B = _f64(B)
    k, n = B.shape
    eB = np.ascontiguousarray(eB, np.int32)
    S = np.empty((p, n, k), np.int8)
    _lib.oracle_oz1_slices_cols(_i64(k), _i64(n), _ptr(B), _i64(n), _ptr(eB), C.c_int(p), _ptr(S))
    return S


def oz1_accumulators(SA, SB):
    """int64 [p][m][n], C_s = sum_{t<=s} A'_t B'_{s-t} (oracle_oz1_accumulators)."""
    SA = np.ascontiguousarray(SA, np.int8)
    SB = np.ascontiguousarray(SB, np.int8)
    p, m, k = SA.shape
    _, n, _ = SB.shape
    CS = np.empty((p, m, n), np.int64)
    _lib.oracle_oz1_accumulators(_i64(m), _i64(n), _i64(k), C.c_int(p), _ptr(SA), _ptr(SB), _ptr(CS))
    return CS


def oz1_reduce(CS, eA, eB, alpha=1.0, beta=0.0, Cin=None):
    CS = np.ascontiguousarray(CS, np.int64)
    p, m, n = CS.shape
    out = np.zeros((m, n), np.float64) if Cin is None else _f64(Cin).copy()
    eA = np.ascontiguousarray(eA, np.int32)
    eB = np.ascontiguousarray(eB, np.int32)
    _lib.oracle_oz1_reduce(_i64(m), _i64(n), C.c_int(p), _ptr(CS), _ptr(eA), _ptr(eB),
                           _dbl(alpha), _dbl(beta), _ptr(out), _i64(n))
    return out


def dgemm_oz1(A, B, p, alpha=1.0, beta=0.0, Cin=None):
    A, B = _f64(A), _f64(B)
    m, k = A.shape
    _, n = B.shape
    out = np.zeros((m, n), np.float64) if Cin is None else _f64(Cin).copy()
    _lib.oracle_dgemm_oz1.restype = C.c_int
    rc = _lib.oracle_dgemm_oz1(_i64(m), _i64(n), _i64(k), _dbl(alpha), _ptr(A), _i64(k), _ptr(B),
                               _i64(n), _dbl(beta), _ptr(out), _i64(n), C.c_int(p))
    if rc:
        raise ValueError(f"oracle_dgemm_oz1 rc={rc}")
    return out


def sgemm_oz1(A, B, p, alpha=1.0, beta=0.0, Cin=None):
    A = np.ascontiguousarray(A, np.float32)
    B = np.ascontiguousarray(B, np.float32)
    m, k = A.shape
    _, n = B.shape
    out = np.zeros((m, n), np.float32) if Cin is None else np.ascontiguousarray(Cin, np.float32).copy()
    _lib.oracle_sgemm_oz1.restype = C.c_int
    rc = _lib.oracle_sgemm_oz1(_i64(m), _i64(n), _i64(k), _flt(alpha), _ptr(A), _i64(k), _ptr(B),
                               _i64(n), _flt(beta), _ptr(out), _i64(n), C.c_int(p))
    if rc:
        raise ValueError(f"oracle_sgemm_oz1 rc={rc}")
    return out


def oz1_sampled(A, B, p, rows, cols, alpha=1.0, is_f32=False):
    """out[r][c] = element (rows[r], cols[c]) of the Scheme I result (oracle_oz1_sampled)."""
    A, B = _f64(A), _f64(B)
    m, k = A.shape
    _, n = B.shape
    rows = np.ascontiguousarray(rows, np.int64)
    cols = np.ascontiguousarray(cols, np.int64)
    out = np.empty((len(rows), len(cols)), np.float64)
    _lib.oracle_oz1_sampled(_i64(m), _i64(n), _i64(k), _dbl(alpha), _ptr(A), _i64(k), _ptr(B), _i64(n),
                            C.c_int(p), _i64(len(rows)), _ptr(rows), _i64(len(cols)), _ptr(cols),
                            C.c_int(1 if is_f32 else 0), _ptr(out))
    return out


def zgemm_oz1_4m(A, B, p, alpha=1.0 + 0j, beta=0j, Cin=None, _f32=False):
    """Scheme I complex GEMM by 4M as four separate real slice products (oracle_zgemm_oz1_4m)."""
    A, Af = _zview(A)
    B, Bf = _zview(B)
    m, k = A.shape
    _, n = B.shape
    out = np.zeros((m, n), np.complex128) if Cin is None else np.ascontiguousarray(Cin, np.complex128).copy()
    al = np.array([complex(alpha).real, complex(alpha).imag], np.float64)
    be = np.array([complex(beta).real, complex(beta).imag], np.float64)
    _lib.oracle_zgemm_oz1_4m.restype = C.c_int
    rc = _lib.oracle_zgemm_oz1_4m(_i64(m), _i64(n), _i64(k), _ptr(al), _ptr(Af), _i64(k), _ptr(Bf), _i64(n), _ptr(be),
                                  _ptr(out.view(np.float64)), _i64(n), C.c_int(p), C.c_int(1 if _f32 else 0))
    if rc:
        raise ValueError(f"oracle_zgemm_oz1_4m rc={rc}")
    return out


def cgemm_oz1_4m(A, B, p, alpha=1.0 + 0j, beta=0j, Cin=None):
    """CGEMM by Scheme I / 4M (oracle_zgemm_oz1_4m with is_f32): complex64 inputs widened exactly (marshalling), each
    component rounded once to float inside the C routine."""
    A = np.ascontiguousarray(A, np.complex64).astype(np.complex128)
    B = np.ascontiguousarray(B, np.complex64).astype(np.complex128)
    C0 = None if Cin is None else np.ascontiguousarray(Cin, np.complex64).astype(np.complex128)
    return zgemm_oz1_4m(A, B, p, alpha=alpha, beta=beta, Cin=C0, _f32=True).astype(np.complex64)


def cgemm_oz2_3m(A, B, N, alpha=1.0 + 0j, beta=0j, Cin=None):
    """CGEMM by Scheme II / 3M on complex64 inputs (oracle_zgemm_oz2_3m on the exactly widened inputs; the last step,
    one more rounding of each component to float, is a dtype conversion of the routine's double result: at most 2^-29
    relative beyond 1/2 ulp of float, far inside the 2-ulp FP32 tolerance)."""
    A = np.ascontiguousarray(A, np.complex64).astype(np.complex128)
    B = np.ascontiguousarray(B, np.complex64).astype(np.complex128)
    C0 = None if Cin is None else np.ascontiguousarray(Cin, np.complex64).astype(np.complex128)
    return zgemm_oz2_3m(A, B, N, alpha=alpha, beta=beta, Cin=C0).astype(np.complex64)


# ---------------------------------------------------------------- brute force
def bf128_dgemm(A, B):
    """(C, absAB): __float128 product of the original operands and (|A||B|)_ij."""
    A, B = _f64(A), _f64(B)
    m, k = A.shape
    _, n = B.shape
    out = np.empty((m, n), np.float64)
    ab = np.empty((m, n), np.float64)
    _lib.oracle_bf128_dgemm(_i64(m), _i64(n), _i64(k), _ptr(A), _i64(k), _ptr(B), _i64(n), _ptr(out),
                            _i64(n), _ptr(ab))
    return out, ab


def bf128_zgemm(X, Y):
    X, Xf = _zview(X)
    Y, Yf = _zview(Y)
    m, k = X.shape
    _, n = Y.shape
    out = np.empty((m, n), np.complex128)
    ab = np.empty((m, n), np.float64)
    _lib.oracle_bf128_zgemm(_i64(m), _i64(n), _i64(k), _ptr(Xf), _i64(k), _ptr(Yf), _i64(n),
                            _ptr(out.view(np.float64)), _i64(n), _ptr(ab))
    return out, ab


# ---------------------------------------------------------------- Scheme II
def oz2_moduli(N):
    mod = np.empty(N, np.int32)
    _lib.oracle_oz2_moduli.restype = C.c_int
    if _lib.oracle_oz2_moduli(C.c_int(N), _ptr(mod)):
        raise ValueError("bad N")
    return mod


def _limbs_to_int(l):
    return sum(int(l[i]) << (64 * i) for i in range(4))


def oz2_P(N):
    l = np.empty(4, np.uint64)
    _lib.oracle_oz2_P_limbs(C.c_int(N), _ptr(l))
    return _limbs_to_int(l)


def oz2_weights(N):
    l = np.empty((N, 4), np.uint64)
    _lib.oracle_oz2_weights_limbs(C.c_int(N), _ptr(l))
    return [_limbs_to_int(l[i]) for i in range(N)]


def oz2_budget(N, k, is3m=False):
    """(T, tA, tB) (oracle_oz2_budget)."""
    tA, tB = _i32(0), _i32(0)
    _lib.oracle_oz2_budget.restype = C.c_int
    T = _lib.oracle_oz2_budget(C.c_int(N), _i64(k), C.c_int(1 if is3m else 0), C.byref(tA), C.byref(tB))
    return int(T), int(tA.value), int(tB.value)


def oz2_residues_rows(A, eA, tA, N):
    A = _f64(A)
    m, k = A.shape
    eA = np.ascontiguousarray(eA, np.int32)
    R = np.empty((N, m, k), np.int8)
    _lib.oracle_oz2_residues_rows(_i64(m), _i64(k), _ptr(A), _i64(k), _ptr(eA), C.c_int(tA), C.c_int(N), _ptr(R))
    return R


def oz2_residues_cols(B, eB, tB, N):
    B = _f64(B)
    k, n = B.shape
    eB = np.ascontiguousarray(eB, np.int32)
    R = np.empty((N, n, k), np.int8)
    _lib.oracle_oz2_residues_cols(_i64(k), _i64(n), _ptr(B), _i64(n), _ptr(eB), C.c_int(tB), C.c_int(N), _ptr(R))
    return R


def oz2_residues_z(Z, e, t, N, by_cols):
    """int8 [3][N][rows][k]: re, im, Sigma planes (oracle_oz2_residues_z)."""
    Z, Zf = _zview(Z)
    if by_cols:
        k, rows = Z.shape
        ld = rows
    else:
        rows, k = Z.shape
        ld = k
    e = np.ascontiguousarray(e, np.int32)
    R = np.empty((3, N, rows, k), np.int8)
    _lib.oracle_oz2_residues_z(_i64(rows), _i64(k), _ptr(Zf), _i64(ld), C.c_int(1 if by_cols else 0),
                               _ptr(e), C.c_int(t), C.c_int(N), _ptr(R))
    return R


def oz2_modprod(RA, RB, want_acc=False):
    """(CR int8 [N][m][n], max|acc|, ACC int64 or None) (oracle_oz2_modprod)."""
    RA = np.ascontiguousarray(RA, np.int8)
    RB = np.ascontiguousarray(RB, np.int8)
    N, m, k = RA.shape
    _, n, _ = RB.shape
    CR = np.empty((N, m, n), np.int8)
    ACC = np.empty((N, m, n), np.int64) if want_acc else None
    _lib.oracle_oz2_modprod.restype = C.c_int64
    mx = _lib.oracle_oz2_modprod(_i64(m), _i64(n), _i64(k), C.c_int(N), _ptr(RA), _ptr(RB), _ptr(CR),
                                 _ptr(ACC) if want_acc else None)
    return CR, int(mx), ACC


def oz2_modprod_3m(RA3, RB3):
    """int8 [2][N][m][n] (re, im) (oracle_oz2_modprod_3m)."""
    RA3 = np.ascontiguousarray(RA3, np.int8)
    RB3 = np.ascontiguousarray(RB3, np.int8)
    _, N, m, k = RA3.shape
    _, _, n, _ = RB3.shape
    CZ = np.empty((2, N, m, n), np.int8)
    _lib.oracle_oz2_modprod_3m(_i64(m), _i64(n), _i64(k), C.c_int(N), _ptr(RA3), _ptr(RB3), _ptr(CZ))
    return CZ


def oz2_crt_int(c):
    """Exact CRT of one residue vector -> Python int in (-P/2, P/2] (oracle_oz2_crt_limbs)."""
    c = np.ascontiguousarray(c, np.int32)
    l = np.empty(4, np.uint64)
    _lib.oracle_oz2_crt_limbs.restype = C.c_int
    s = _lib.oracle_oz2_crt_limbs(C.c_int(len(c)), _ptr(c), _ptr(l))
    return s * _limbs_to_int(l)


def oz2_crt(CR, eA, eB, tA, tB, alpha=1.0, beta=0.0, Cin=None, want_X=False):
    CR = np.ascontiguousarray(CR, np.int8)
    N, m, n = CR.shape
    out = np.zeros((m, n), np.float64) if Cin is None else _f64(Cin).copy()
    eA = np.ascontiguousarray(eA, np.int32)
    eB = np.ascontiguousarray(eB, np.int32)
    X = np.empty((m, n, 5), np.int64) if want_X else None
    _lib.oracle_oz2_crt(_i64(m), _i64(n), C.c_int(N), _ptr(CR), _ptr(eA), _ptr(eB), C.c_int(tA), C.c_int(tB),
                        _dbl(alpha), _dbl(beta), _ptr(out), _i64(n), _i64(1), _ptr(X) if want_X else None)
    if want_X:
        Xu = X.view(np.uint64)
        Xi = [[int(X[i, j, 0]) * _limbs_to_int(Xu[i, j, 1:5]) for j in range(n)] for i in range(m)]
        return out, Xi
    return out


def dgemm_oz2(A, B, N, alpha=1.0, beta=0.0, Cin=None):
    A, B = _f64(A), _f64(B)
    m, k = A.shape
    _, n = B.shape
    out = np.zeros((m, n), np.float64) if Cin is None else _f64(Cin).copy()
    _lib.oracle_dgemm_oz2.restype = C.c_int
    rc = _lib.oracle_dgemm_oz2(_i64(m), _i64(n), _i64(k), _dbl(alpha), _ptr(A), _i64(k), _ptr(B), _i64(n),
                               _dbl(beta), _ptr(out), _i64(n), C.c_int(N))
    if rc:
        raise ValueError(f"oracle_dgemm_oz2 rc={rc}")
    return out


def sgemm_oz2(A, B, N, alpha=1.0, beta=0.0, Cin=None):
    """Scheme II on float32 inputs, float32 output (oracle_sgemm_oz2)."""
    A = np.ascontiguousarray(A, np.float32)
    B = np.ascontiguousarray(B, np.float32)
    m, k = A.shape
    _, n = B.shape
    out = np.zeros((m, n), np.float32) if Cin is None else np.ascontiguousarray(Cin, np.float32).copy()
    _lib.oracle_sgemm_oz2.restype = C.c_int
    rc = _lib.oracle_sgemm_oz2(_i64(m), _i64(n), _i64(k), C.c_float(alpha), _ptr(A), _i64(k), _ptr(B), _i64(n),
                               C.c_float(beta), _ptr(out), _i64(n), C.c_int(N))
    if rc:
        raise ValueError(f"oracle_sgemm_oz2 rc={rc}")
    return out


def zgemm_oz2_3m(A, B, N, alpha=1.0 + 0j, beta=0j, Cin=None):
    A, Af = _zview(A)
    B, Bf = _zview(B)
    m, k = A.shape
    _, n = B.shape
    out = np.zeros((m, n), np.complex128) if Cin is None else np.ascontiguousarray(Cin, np.complex128).copy()
    al = np.array([complex(alpha).real, complex(alpha).imag], np.float64)
    be = np.array([complex(beta).real, complex(beta).imag], np.float64)
    _lib.oracle_zgemm_oz2_3m.restype = C.c_int
    rc = _lib.oracle_zgemm_oz2_3m(_i64(m), _i64(n), _i64(k), _ptr(al), _ptr(Af), _i64(k), _ptr(Bf), _i64(n),
                                  _ptr(be), _ptr(out.view(np.float64)), _i64(n), C.c_int(N))
    if rc:
        raise ValueError(f"oracle_zgemm_oz2_3m rc={rc}")
    return out


def oz2_sampled(A, B, N, rows, cols, alpha=1.0, is3m=False):
    rows = np.ascontiguousarray(rows, np.int64)
    cols = np.ascontiguousarray(cols, np.int64)
    if is3m:
        A, Af = _zview(A)
        B, Bf = _zview(B)
        out = np.empty((len(rows), len(cols)), np.complex128)
        of = out.view(np.float64)
    else:
        A, B = _f64(A), _f64(B)
        Af, Bf = A, B
        out = np.empty((len(rows), len(cols)), np.float64)
        of = out
    k = A.shape[1]
    n = B.shape[1]
    al = np.array([complex(alpha).real, complex(alpha).imag], np.float64)
    _lib.oracle_oz2_sampled.restype = C.c_int
    rc = _lib.oracle_oz2_sampled(_i64(k), _ptr(al), _ptr(Af), _i64(k), _ptr(Bf), _i64(n), C.c_int(N),
                                 C.c_int(1 if is3m else 0), _i64(len(rows)), _ptr(rows), _i64(len(cols)),
                                 _ptr(cols), _ptr(of))
    if rc:
        raise ValueError(f"oracle_oz2_sampled rc={rc}")
    return out
