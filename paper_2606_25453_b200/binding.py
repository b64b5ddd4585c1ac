"""ctypes binding for libemugemm.so: same names as include/emugemm.h, argument marshalling only.

PyTorch is used for device memory and streams (tensor.data_ptr(), torch.cuda.current_stream());
every step of the hot path runs in the library's CUDA kernels.  There is no CPU fallback.
"""
import ctypes as C
import os
import re

LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libemugemm.so")
PROBES_LIB_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "libemugemm_probes.so")
_HEADER = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "emugemm.h")

OZ1, OZ2, OZ2_3M, OZ1_4M = 1, 2, 3, 4
DIGITS_SIGN_MAGNITUDE = 0x207   # EMUGEMM_DIGITS_SIGN_MAGNITUDE: code of the sign-magnitude digit form for oz1_chunk_k
_i64, _int, _dbl, _flt, _vp, _sz = C.c_int64, C.c_int, C.c_double, C.c_float, C.c_void_p, C.c_size_t


class Operand(C.Structure):
    """emugemm_operand_t (include/emugemm.h): a pre-decomposed operand; `tensor` keeps the device buffer alive."""
    _fields_ = [("scheme", C.c_int), ("role", C.c_int), ("elem", C.c_int), ("pn", C.c_int), ("slice_bits", C.c_int),
                ("t_bits", C.c_int), ("rows", C.c_int64), ("k", C.c_int64), ("kpad", C.c_int64), ("buf", C.c_void_p),
                ("bytes", C.c_size_t)]


class EmuGemmError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"emugemm status {status}: {msg}")
        self.status = status


_libs = {}


def load_library(probes=False):
    """dlopen the in-tree library; raises (never falls back) if it has not been built.  probes=True: the PROBES build
    (same sources + -DEMUGEMM_PROBES: emugemm_dbg_set_flags and the tensor-pipe probes), used only by bench.py's probe leg."""
    if probes not in _libs:
        path = PROBES_LIB_PATH if probes else LIB_PATH
        if not os.path.exists(path):
            raise FileNotFoundError(f"{path} not built: run `python -m paper_2606_25453_b200.build` "
                                    "(the product path has no CPU fallback)")
        lib = C.CDLL(path)
        lib.emugemm_status_string.restype = C.c_char_p
        lib.emugemm_workspace_bytes.restype = _sz
        lib.emugemm_workspace_bytes.argtypes = [_int, _int, _i64, _i64, _i64, _int]
        lib.emugemm_operand_bytes.restype = _sz
        lib.emugemm_operand_bytes.argtypes = [_int, _i64, _i64, _int]
        lib.emugemm_static_workspace_limit.restype = _sz
        lib.emugemm_oz1_chunk_k.restype = _i64
        lib.emugemm_oz1_chunk_k_bits.restype = _i64
        _libs[probes] = lib
    return _libs[probes]


def exported_symbols(probes=False):
    """Names declared in include/emugemm.h (used by the not-gpu load test); the `#ifdef EMUGEMM_PROBES` block only for
    the PROBES build."""
    text = open(_HEADER).read()
    if not probes:
        text = re.sub(r"#ifdef EMUGEMM_PROBES.*?#endif /\* EMUGEMM_PROBES \*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(emugemm_[a-z0-9_]+)\s*\(", text)))


def oz2_budget(n_moduli, k, is3m=False):
    a, b = _int(0), _int(0)
    T = load_library().emugemm_oz2_budget(_int(n_moduli), _i64(k), _int(1 if is3m else 0), C.byref(a), C.byref(b))
    return int(T), a.value, b.value


def crt_constants(n_moduli):
    """emugemm_dbg_crt_constants (host only) -> dict(n_pairs, n_digits, digit_bits, W=[digit lists], P=[digits], pair=[(M, K1, K2, C0, magic)])."""
    npairs, nd, g = _int(0), _int(0), _int(0)
    digits = (C.c_longlong * 55)()
    pair = (C.c_uint * 50)()
    st = load_library().emugemm_dbg_crt_constants(_int(n_moduli), C.byref(npairs), C.byref(nd), C.byref(g), digits, pair)
    if st != 0:
        raise EmuGemmError(st, "emugemm_dbg_crt_constants")
    NP, J = npairs.value, nd.value
    rows = [[int(digits[q * J + j]) for j in range(J)] for q in range(NP + 1)]
    return dict(n_pairs=NP, n_digits=J, digit_bits=g.value, W=rows[:NP], P=rows[NP],
                pair=[tuple(int(pair[5 * q + i]) for i in range(5)) for q in range(NP)])


def oz1_chunk_k(p, slice_bits=7):
    return int(load_library().emugemm_oz1_chunk_k_bits(_int(p), _int(slice_bits)))


def _ptr(t):
    return _vp(t.data_ptr()) if t is not None else _vp(None)


class EmuGemm:
    """One handle (= one host thread, one stream).  Tensors are row-major CUDA tensors; strides are taken
    from the tensors (last dim contiguous).  Workspace is a torch uint8 tensor owned by this object and
    grown on demand OUTSIDE the timed hot path via reserve()."""

    def __init__(self, probes=False):
        import torch
        self._torch = torch
        self._lib = load_library(probes)
        self._h = _vp(None)
        self._check(self._lib.emugemm_create(C.byref(self._h)))
        self._ws = None
        self.slice_bits = 7
        self._device = torch.cuda.current_device()
        self._stream = None
        self.set_stream(torch.cuda.current_stream())

    def close(self):
        if self._h:
            self._lib.emugemm_destroy(self._h)
            self._h = _vp(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st):
        if st != 0:
            raise EmuGemmError(st, self._lib.emugemm_status_string(_int(st)).decode())

    # ---- handle ------------------------------------------------------------
    def set_stream(self, stream):
        self._check(self._lib.emugemm_set_stream(self._h, _vp(stream.cuda_stream)))
        self._stream = stream

    def set_slice_bits(self, bits):
        """Scheme I digits: 7 (default, form per set_slice_form) or 8 = balanced base 256 (see include/emugemm.h)."""
        self._check(self._lib.emugemm_set_slice_bits(self._h, _int(bits)))
        self.slice_bits = bits

    def set_slice_form(self, form):
        """7-bit Scheme I digits: 0 = two's-complement fields (default, R24), 1 = sign-magnitude (R1; include/emugemm.h)."""
        self._check(self._lib.emugemm_set_slice_form(self._h, _int(form)))
        if self.slice_bits != 8:
            self.slice_bits = DIGITS_SIGN_MAGNITUDE if form else 7

    def set_oz2_fusion(self, on):
        """Scheme II real DGEMM: fused reconstruction inside the GEMM kernel, or (default) the separate CRT kernel."""
        self._check(self._lib.emugemm_set_oz2_fusion(self._h, _int(1 if on else 0)))
        self._fusion = bool(on)

    def workspace_bytes(self, scheme, elem, m, n, k, pn):
        return int(self._lib.emugemm_workspace_bytes(scheme, elem, m, n, k, pn))

    def reserve(self, nbytes):
        torch = self._torch
        if self._ws is None or self._ws.numel() < nbytes + 1024:
            if self._ws is not None and self._stream is not None:
                # kernels of earlier calls may still use the old workspace on the handle's stream, which need not be
                # torch's current stream: the caching allocator must not hand the block out before they are done
                self._ws.record_stream(self._stream)
            self._ws = None
            raw = torch.empty(int(nbytes) + 2048, dtype=torch.uint8, device="cuda")
            if self._stream is not None:
                raw.record_stream(self._stream)
            self._ws = raw
        off = (-self._ws.data_ptr()) % 1024
        self._check(self._lib.emugemm_set_workspace(self._h, _vp(self._ws.data_ptr() + off), _sz(self._ws.numel() - off)))

    def _reserve_for(self, scheme, elem, m, n, k, pn):
        need = self.workspace_bytes(scheme, elem, m, n, k, pn)
        if scheme == OZ2 and getattr(self, "_fusion", False):
            need += 160 * 2 * pn * 32768  # room for the per-CTA scratch of the fused reconstruction (include/emugemm.h)
        if self._ws is None or self._ws.numel() - 1024 < need:
            self.reserve(need)

    def enable_stage_timing(self, on=True):
        self._check(self._lib.emugemm_enable_stage_timing(self._h, _int(1 if on else 0)))

    def stage_ms(self):
        ms = (_flt * 3)()
        n = _int(0)
        self._check(self._lib.emugemm_stage_ms(self._h, ms, C.byref(n)))
        return [float(x) for x in ms], n.value

    def nonfinite_seen(self):
        """True if the last compute call's pre-pass met an Inf or a NaN in A or B (synchronises the stream)."""
        v = _int(0)
        self._check(self._lib.emugemm_nonfinite_seen(self._h, C.byref(v)))
        return bool(v.value)

    def last_gemm_cycles(self):
        c = C.c_ulonglong(0)
        self._check(self._lib.emugemm_last_gemm_cycles(self._h, C.byref(c)))
        return int(c.value)

    # ---- compute (names follow include/emugemm.h) --------------------------
    @staticmethod
    def _ld(t):
        assert t.stride(-1) == 1, "row-major tensors with a contiguous last dimension are required"
        return t.stride(0)

    # transa / transb: the tensor holds the TRANSPOSE of the operand (A: k x m, B: n x k), row-major
    def _dims(self, A, B, transa=False, transb=False, C_=None, dtype=None):
        """(m, n, k) after checking what the C ABI cannot see from raw pointers: every matrix is a 2-D CUDA tensor of
        the entry point's dtype on the handle's device, the inner dimensions agree and C is m x n (ValueError before
        the library is entered: a wrong dtype or shape would make the kernels read or write out of bounds)."""
        torch = self._torch
        for name, X in (("A", A), ("B", B), ("C", C_)):
            if X is None:
                continue
            if not isinstance(X, torch.Tensor) or X.dim() != 2:
                raise ValueError(f"{name}: a 2-D torch tensor is required")
            if not X.is_cuda or X.device.index != self._device:
                raise ValueError(f"{name}: must live on cuda:{self._device}, the device of this handle (got {X.device})")
            if dtype is not None and X.dtype != dtype:
                raise ValueError(f"{name}: dtype {X.dtype} given, this entry point takes {dtype}")
            if X.stride(-1) != 1 and X.shape[-1] > 1:
                raise ValueError(f"{name}: the last dimension must be contiguous")
        m, k = (A.shape[1], A.shape[0]) if transa else A.shape
        kb, n = (B.shape[1], B.shape[0]) if transb else B.shape
        if k != kb:
            raise ValueError(f"inner dimensions differ: op(A) is {m} x {k}, op(B) is {kb} x {n}")
        if C_ is not None and tuple(C_.shape) != (m, n):
            raise ValueError(f"C is {tuple(C_.shape)}, expected ({m}, {n})")
        return m, n, k

    def dgemm_oz1(self, A, B, C_, p, alpha=1.0, beta=0.0, transa=False, transb=False):
        m, n, k = self._dims(A, B, transa, transb, C_, self._torch.float64)
        self._reserve_for(OZ1, 8, m, n, k, p)
        self._check(self._lib.emugemm_dgemm_oz1_t(self._h, _int(transa), _int(transb), _i64(m), _i64(n), _i64(k), _dbl(alpha),
                                                   _ptr(A), _i64(self._ld(A)), _ptr(B), _i64(self._ld(B)), _dbl(beta), _ptr(C_),
                                                   _i64(self._ld(C_)), _int(p)))
        return C_

    def static_workspace_limit(self):
        return int(self._lib.emugemm_static_workspace_limit())

    def dgemm_oz1_static(self, A, B, C_, p, alpha=1.0, beta=0.0):
        """emugemm_dgemm_oz1_static: scratch in the library's static device array -- nothing is allocated or reserved
        here (no torch workspace either); EmuGemmError with status -7 beyond static_workspace_limit()."""
        m, n, k = self._dims(A, B, False, False, C_, self._torch.float64)
        self._check(self._lib.emugemm_dgemm_oz1_static(self._h, _i64(m), _i64(n), _i64(k), _dbl(alpha), _ptr(A), _i64(self._ld(A)),
                                                        _ptr(B), _i64(self._ld(B)), _dbl(beta), _ptr(C_), _i64(self._ld(C_)),
                                                        _int(p)))
        return C_

    def sgemm_oz1(self, A, B, C_, p, alpha=1.0, beta=0.0, transa=False, transb=False):
        m, n, k = self._dims(A, B, transa, transb, C_, self._torch.float32)
        self._reserve_for(OZ1, 4, m, n, k, p)
        self._check(self._lib.emugemm_sgemm_oz1_t(self._h, _int(transa), _int(transb), _i64(m), _i64(n), _i64(k), _flt(alpha),
                                                   _ptr(A), _i64(self._ld(A)), _ptr(B), _i64(self._ld(B)), _flt(beta), _ptr(C_),
                                                   _i64(self._ld(C_)), _int(p)))
        return C_

    def _batched(self, fn, cvt, elem, A, B, C_, p, alpha, beta, scheme=OZ1):
        # A: (batch, m, k) or (m, k) shared by all entries; B: (batch, k, n) or (k, n); C_: (batch, m, n).
        # The last dimension is contiguous, dimension -2 carries the leading dimension, dimension 0 the batch stride.
        torch = self._torch
        want = {4: torch.float32, 8: torch.float64, 16: torch.complex128}[elem]
        for name, X in (("A", A), ("B", B), ("C", C_)):
            if not isinstance(X, torch.Tensor) or not X.is_cuda or X.device.index != self._device or X.dtype != want:
                raise ValueError(f"{name}: a {want} tensor on cuda:{self._device} is required")
        if C_.dim() != 3 or A.dim() not in (2, 3) or B.dim() not in (2, 3):
            raise ValueError("batched operands: A (batch, m, k) or (m, k), B (batch, k, n) or (k, n), C (batch, m, n)")
        batch, m, n = C_.shape
        k = A.shape[-1]
        for X, shp in ((A, (m, k)), (B, (k, n))):
            if tuple(X.shape[-2:]) != shp or X.stride(-1) != 1 or (X.dim() == 3 and X.shape[0] != batch):
                raise ValueError("batched operands: A (batch, m, k), B (batch, k, n), C (batch, m, n), last dimension contiguous")
        if C_.stride(-1) != 1:
            raise ValueError("C must be contiguous in its last dimension")
        sa = A.stride(0) if A.dim() == 3 else 0
        sb = B.stride(0) if B.dim() == 3 else 0
        self._reserve_for(scheme, elem, batch * m, batch * n, k, p)
        self._check(fn(self._h, _i64(batch), _i64(m), _i64(n), _i64(k), cvt(alpha), _ptr(A), _i64(A.stride(-2)), _i64(sa),
                       _ptr(B), _i64(B.stride(-2)), _i64(sb), cvt(beta), _ptr(C_), _i64(C_.stride(-2)), _i64(C_.stride(0)),
                       _int(p)))
        return C_

    def dgemm_oz1_strided_batched(self, A, B, C_, p, alpha=1.0, beta=0.0):
        """C_[b] = alpha A[b] B[b] + beta C_[b] (float64 CUDA tensors; a 2-D A or B is shared by all entries)."""
        return self._batched(self._lib.emugemm_dgemm_oz1_strided_batched, _dbl, 8, A, B, C_, p, alpha, beta)

    def sgemm_oz1_strided_batched(self, A, B, C_, p, alpha=1.0, beta=0.0):
        return self._batched(self._lib.emugemm_sgemm_oz1_strided_batched, _flt, 4, A, B, C_, p, alpha, beta)

    def dgemm_oz2_strided_batched(self, A, B, C_, n_moduli, alpha=1.0, beta=0.0):
        return self._batched(self._lib.emugemm_dgemm_oz2_strided_batched, _dbl, 8, A, B, C_, n_moduli, alpha, beta, OZ2)

    def sgemm_oz2_strided_batched(self, A, B, C_, n_moduli, alpha=1.0, beta=0.0):
        return self._batched(self._lib.emugemm_sgemm_oz2_strided_batched, _flt, 4, A, B, C_, n_moduli, alpha, beta, OZ2)

    def dgemm_oz2(self, A, B, C_, n_moduli, alpha=1.0, beta=0.0, transa=False, transb=False):
        m, n, k = self._dims(A, B, transa, transb, C_, self._torch.float64)
        self._reserve_for(OZ2, 8, m, n, k, n_moduli)
        self._check(self._lib.emugemm_dgemm_oz2_t(self._h, _int(transa), _int(transb), _i64(m), _i64(n), _i64(k), _dbl(alpha),
                                                   _ptr(A), _i64(self._ld(A)), _ptr(B), _i64(self._ld(B)), _dbl(beta), _ptr(C_),
                                                   _i64(self._ld(C_)), _int(n_moduli)))
        return C_

    def zgemm_oz1_4m(self, A, B, C_, p, alpha=1.0 + 0j, beta=0j):
        """A, B, C_: complex128 CUDA tensors (Scheme I, 4M)."""
        m, n, k = self._dims(A, B, False, False, C_, self._torch.complex128)
        self._reserve_for(OZ1_4M, 16, m, n, k, p)
        al = (_dbl * 2)(complex(alpha).real, complex(alpha).imag)
        be = (_dbl * 2)(complex(beta).real, complex(beta).imag)
        self._check(self._lib.emugemm_zgemm_oz1_4m(self._h, _i64(m), _i64(n), _i64(k), al, _ptr(A), _i64(self._ld(A)), _ptr(B),
                                                    _i64(self._ld(B)), be, _ptr(C_), _i64(self._ld(C_)), _int(p)))
        return C_

    def cgemm_oz1_4m(self, A, B, C_, p, alpha=1.0 + 0j, beta=0j):
        """A, B, C_: complex64 CUDA tensors (Scheme I, 4M)."""
        m, n, k = self._dims(A, B, False, False, C_, self._torch.complex64)
        self._reserve_for(OZ1_4M, 16, m, n, k, p)
        al = (_dbl * 2)(complex(alpha).real, complex(alpha).imag)
        be = (_dbl * 2)(complex(beta).real, complex(beta).imag)
        self._check(self._lib.emugemm_cgemm_oz1_4m(self._h, _i64(m), _i64(n), _i64(k), al, _ptr(A), _i64(self._ld(A)), _ptr(B),
                                                    _i64(self._ld(B)), be, _ptr(C_), _i64(self._ld(C_)), _int(p)))
        return C_

    def cgemm_oz2_3m(self, A, B, C_, n_moduli, alpha=1.0 + 0j, beta=0j):
        """A, B, C_: complex64 CUDA tensors (Scheme II, 3M)."""
        m, n, k = self._dims(A, B, False, False, C_, self._torch.complex64)
        self._reserve_for(OZ2_3M, 16, m, n, k, n_moduli)
        al = (_dbl * 2)(complex(alpha).real, complex(alpha).imag)
        be = (_dbl * 2)(complex(beta).real, complex(beta).imag)
        self._check(self._lib.emugemm_cgemm_oz2_3m(self._h, _i64(m), _i64(n), _i64(k), al, _ptr(A), _i64(self._ld(A)), _ptr(B),
                                                    _i64(self._ld(B)), be, _ptr(C_), _i64(self._ld(C_)), _int(n_moduli)))
        return C_

    def sgemm_oz2(self, A, B, C_, n_moduli, alpha=1.0, beta=0.0, transa=False, transb=False):
        m, n, k = self._dims(A, B, transa, transb, C_, self._torch.float32)
        self._reserve_for(OZ2, 8, m, n, k, n_moduli)
        self._check(self._lib.emugemm_sgemm_oz2_t(self._h, _int(transa), _int(transb), _i64(m), _i64(n), _i64(k), _flt(alpha),
                                                   _ptr(A), _i64(self._ld(A)), _ptr(B), _i64(self._ld(B)), _flt(beta), _ptr(C_),
                                                   _i64(self._ld(C_)), _int(n_moduli)))
        return C_

    def zgemm_oz2_3m(self, A, B, C_, n_moduli, alpha=1.0 + 0j, beta=0j, transa=False, transb=False):
        """A, B, C_: complex128 CUDA tensors."""
        m, n, k = self._dims(A, B, transa, transb, C_, self._torch.complex128)
        self._reserve_for(OZ2_3M, 16, m, n, k, n_moduli)
        al = (_dbl * 2)(complex(alpha).real, complex(alpha).imag)
        be = (_dbl * 2)(complex(beta).real, complex(beta).imag)
        self._check(self._lib.emugemm_zgemm_oz2_3m_t(self._h, _int(transa), _int(transb), _i64(m), _i64(n), _i64(k), al, _ptr(A),
                                                      _i64(self._ld(A)), _ptr(B), _i64(self._ld(B)), be, _ptr(C_),
                                                      _i64(self._ld(C_)), _int(n_moduli)))
        return C_

    def zgemm_oz2_3m_strided_batched(self, A, B, C_, n_moduli, alpha=1.0 + 0j, beta=0j):
        """complex128 CUDA tensors: A (batch, m, k) or (m, k), B (batch, k, n) or (k, n), C_ (batch, m, n)."""
        cvt = lambda z: (_dbl * 2)(complex(z).real, complex(z).imag)  # noqa: E731
        return self._batched(self._lib.emugemm_zgemm_oz2_3m_strided_batched, cvt, 16, A, B, C_, n_moduli, alpha, beta, OZ2_3M)

    # ---- pre-decomposed operands (emugemm_decompose / emugemm_gemm_pre) --------
    def decompose(self, scheme, role, X, pn, trans=False):
        """-> Operand for the left (role 0) or right (role 1) operand; X as in the _t calls."""
        torch = self._torch
        elem = self._elem(X)
        stored_rows, stored_cols = X.shape
        by_cols = bool(trans) if role == 0 else not trans
        rows, k = (stored_cols, stored_rows) if by_cols else (stored_rows, stored_cols)
        nbytes = int(self._lib.emugemm_operand_bytes(scheme, rows, k, pn))
        assert nbytes > 0, "invalid operand arguments"
        raw = torch.empty(nbytes + 1024, dtype=torch.uint8, device="cuda")
        if self._stream is not None:
            raw.record_stream(self._stream)  # written and read by kernels on the handle's stream
        off = (-raw.data_ptr()) % 1024
        if self._ws is None or self._ws.numel() < 8 * rows + 4096:
            self.reserve(max(8 * rows + 4096, 1 << 20))
        op = Operand()
        self._check(self._lib.emugemm_decompose(self._h, _int(scheme), _int(role), _int(int(trans)), _int(elem), _i64(rows), _i64(k),
                                                 _ptr(X), _i64(self._ld(X)), _int(pn), _vp(raw.data_ptr() + off), _sz(nbytes),
                                                 C.byref(op)))
        op.tensor = raw
        return op

    def gemm_pre(self, opA, opB, C_, alpha=1.0, beta=0.0):
        scheme_elem = {(OZ1, 4): 4, (OZ1, 8): 8, (OZ2, 4): 8, (OZ2, 8): 8, (OZ2_3M, 16): 16}[(opA.scheme, opA.elem)]
        self._reserve_for(opA.scheme, scheme_elem, opA.rows, opB.rows, opA.k, opA.pn)
        al = (_dbl * 2)(complex(alpha).real, complex(alpha).imag)
        be = (_dbl * 2)(complex(beta).real, complex(beta).imag)
        self._check(self._lib.emugemm_gemm_pre(self._h, C.byref(opA), C.byref(opB), al, be, _ptr(C_), _i64(self._ld(C_))))
        return C_

    # ---- test hooks -----------------------------------------------------------
    def _elem(self, X):
        torch = self._torch
        return {torch.float32: 4, torch.float64: 8, torch.complex128: 16}[X.dtype]

    def dbg_exponents(self, X, by_cols):
        torch = self._torch
        rows, k = (X.shape[1], X.shape[0]) if by_cols else X.shape
        self.reserve(max(8 * rows + 4096, 1 << 20))
        e = torch.empty(rows, dtype=torch.int32, device="cuda")
        self._check(self._lib.emugemm_dbg_exponents(self._h, _int(self._elem(X)), _int(int(by_cols)), _i64(rows), _i64(k),
                                                     _ptr(X), _i64(self._ld(X)), _ptr(e)))
        return e

    def dbg_oz1_slices(self, X, by_cols, p):
        torch = self._torch
        rows, k = (X.shape[1], X.shape[0]) if by_cols else X.shape
        kpad = (k + 127) // 128 * 128
        self.reserve(8 * rows + p * rows * kpad + (1 << 16))
        out = torch.empty((p, rows, k), dtype=torch.int8, device="cuda")
        e = torch.empty(rows, dtype=torch.int32, device="cuda")
        self._check(self._lib.emugemm_dbg_oz1_slices(self._h, _int(self._elem(X)), _int(int(by_cols)), _i64(rows), _i64(k),
                                                      _ptr(X), _i64(self._ld(X)), _int(p), _ptr(out), _ptr(e)))
        return out, e

    def dbg_oz1_accumulators(self, A, B, p, chunk_k=0):
        torch = self._torch
        m, k = A.shape
        n = B.shape[1]
        self._reserve_for(OZ1, self._elem(A), m, n, k, p)
        kpad = (k + 127) // 128 * 128
        ck = chunk_k if chunk_k > 0 else oz1_chunk_k(p, self.slice_bits)
        ck = min((ck + 127) // 128 * 128, oz1_chunk_k(p, self.slice_bits))
        nch = max(1, -(-kpad // ck))
        out = torch.empty((nch, p, m, n), dtype=torch.int32, device="cuda")
        got = _int(0)
        self._check(self._lib.emugemm_dbg_oz1_accumulators(self._h, _int(self._elem(A)), _i64(m), _i64(n), _i64(k), _ptr(A),
                                                            _i64(self._ld(A)), _ptr(B), _i64(self._ld(B)), _int(p), _i64(chunk_k),
                                                            _ptr(out), C.byref(got)))
        assert got.value == nch, (got.value, nch)
        return out

    def dbg_oz2_residues(self, X, by_cols, n_moduli, t_bits):
        torch = self._torch
        rows, k = (X.shape[1], X.shape[0]) if by_cols else X.shape
        kpad = (k + 127) // 128 * 128
        parts = 3 if X.dtype == torch.complex128 else 1
        self.reserve(8 * rows + parts * n_moduli * rows * kpad + (1 << 16))
        shape = (parts, n_moduli, rows, k) if parts == 3 else (n_moduli, rows, k)
        out = torch.empty(shape, dtype=torch.int8, device="cuda")
        e = torch.empty(rows, dtype=torch.int32, device="cuda")
        self._check(self._lib.emugemm_dbg_oz2_residues(self._h, _int(self._elem(X)), _int(int(by_cols)), _i64(rows), _i64(k),
                                                        _ptr(X), _i64(self._ld(X)), _int(n_moduli), _int(t_bits), _ptr(out), _ptr(e)))
        return out, e

    def dbg_oz2_modgemm(self, RA, RB, is3m=False):
        torch = self._torch
        N, m, k = RA.shape[-3:]
        n = RB.shape[-2]
        kpad = (k + 127) // 128 * 128
        parts = 3 if is3m else 1
        self.reserve(parts * N * (m + n) * kpad + (1 << 16))
        shape = (2, N, m, n) if is3m else (N, m, n)
        out = torch.empty(shape, dtype=torch.int8, device="cuda")
        self._check(self._lib.emugemm_dbg_oz2_modgemm(self._h, _int(int(is3m)), _i64(m), _i64(n), _i64(k), _int(N),
                                                       _ptr(RA.contiguous()), _ptr(RB.contiguous()), _ptr(out)))
        return out

    def dbg_oz2_crt(self, CR, eA, eB, tA, tB, C_, alpha=1.0, beta=0.0):
        N, m, n = CR.shape
        self._check(self._lib.emugemm_dbg_oz2_crt(self._h, _i64(m), _i64(n), _int(N), _ptr(CR), _ptr(eA), _ptr(eB), _int(tA),
                                                   _int(tB), _dbl(alpha), _dbl(beta), _ptr(C_), _i64(self._ld(C_))))
        return C_

    # ---- PROBES build only (EmuGemm(probes=True)) -------------------------------
    def dbg_set_flags(self, flags):
        """Timing experiments (include/emugemm.h): results become WRONG; exists only in libemugemm_probes.so."""
        self._check(self._lib.emugemm_dbg_set_flags(self._h, _int(flags)))

    def dbg_i8_probe(self, ops, iters=4000):
        """ops: list of (tmem_col, N, a_slot, b_row[, collector]).  -> (ms, Top/s, INT8 op / clk / SM from the SM cycle counter)."""
        ops = [tuple(op) + (0,) * (5 - len(op)) for op in ops]
        if self._ws is None:
            self.reserve(1 << 20)
        flat = (C.c_int * (5 * len(ops)))(*[int(x) for op in ops for x in op])
        ms, ctas, cyc = _flt(0), _int(0), C.c_longlong(0)
        self._check(self._lib.emugemm_dbg_i8_probe(self._h, _int(len(ops)), flat, _int(iters), C.byref(ms), C.byref(ctas),
                                                   C.byref(cyc)))
        per_cta = iters * sum(2.0 * 128 * op[1] * 32 for op in ops)
        return ms.value, per_cta * ctas.value / (ms.value * 1e-3) / 1e12, per_cta / max(cyc.value, 1)

    def dbg_oz1_issue_probe(self, p, use_collector=True, iters=2000):
        """-> (ms, Top/s, fraction of 16384 op/clk/SM) of the fused kernel's issue schedule on resident operands."""
        if self._ws is None:
            self.reserve(1 << 20)
        nt = {1: 256, 2: 256, 3: 160, 4: 128, 5: 96, 6: 80, 7: 64, 8: 64}[p]
        ms, ctas, cyc = _flt(0), _int(0), C.c_longlong(0)
        self._check(self._lib.emugemm_dbg_oz1_issue_probe(self._h, _int(p), _int(int(use_collector)), _int(iters), C.byref(ms),
                                                          C.byref(ctas), C.byref(cyc)))
        per_cta = iters * 4.0 * p * (p + 1) * 128 * nt * 32
        return ms.value, per_cta * ctas.value / (ms.value * 1e-3) / 1e12, per_cta / max(cyc.value, 1) / 16384.0

    def dbg_i8_peak_probe(self, n_mma=256, iters=20000):
        """uniform 128 x n_mma x 32 MMAs alternating between the two 256-column halves of TMEM."""
        return self.dbg_i8_probe([(0, n_mma, 0, 0), (256, n_mma, 0, 0)], iters // 2)
