/*
 * emugemm.h -- C ABI of the B200-native EmuGEMM hot path (arxiv/paper_2606_25453).
 *
 * High-precision GEMM  C = alpha*A*B + beta*C  emulated on INT8 tensor cores
 * (tcgen05.mma kind::i8, sm_100a only):
 *   Scheme I  (Eq. 1-3; fused kernel PAPER.md:171-209, Alg. 1)
 *   Scheme II (Eq. 4-8; fused mod-reduction PAPER.md:225-240)
 *   3M complex on Scheme II (Eq. 16-18)
 *
 * Conventions common to every call
 *   - Layout: row-major, no transposes.  A is m x k with row stride lda >= k,
 *     B is k x n with ldb >= n, C is m x n with ldc >= n; strides in elements
 *     (complex entry point: in complex elements, storage is (re, im) pairs).
 *   - m, n, k >= 0.  m*n == 0 is a no-op; k == 0 scales C by beta.  m, n < 2^31 - 256, k <= 8,388,480 (65535 * 128).
 *   - All matrix pointers are DEVICE pointers owned by the caller.  A and B are
 *     read-only.  C is read only when beta != 0 (BLAS rule: beta == 0 means C is
 *     not read, NaNs in C do not propagate) and is overwritten.
 *   - alpha / beta are host scalars passed by value (complex: host pointer to
 *     two doubles, read during the call).
 *   - Workspace is caller-owned device memory handed over with
 *     emugemm_set_workspace(); the library never allocates device memory on the
 *     hot path.  emugemm_workspace_bytes() says how much a call needs.
 *   - Calls are asynchronous on the handle's stream (emugemm_set_stream; default
 *     stream 0).  One handle per host thread.  The handle owns only host state.
 *   - Alignment: A, B, C base pointers 16-byte aligned, workspace 1024-byte.
 *   - Non-finite inputs: result unspecified, no fault.
 *   - Return value: EMUGEMM_OK (0) or a negative emugemm_status; no exceptions,
 *     no exit(), no stdout.  There is NO CPU fallback: on a device that is not
 *     sm_100 every compute call returns EMUGEMM_ERR_DEVICE.
 */
#ifndef EMUGEMM_H_
#define EMUGEMM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct emugemm_ctx *emugemm_handle_t;

enum emugemm_status {
  EMUGEMM_OK = 0,
  EMUGEMM_ERR_ARG = -1,       /* null pointer, negative size, ld too small, p / n_moduli out of range */
  EMUGEMM_ERR_ALIGNMENT = -2, /* A, B, C not 16-byte aligned or workspace not 1024-byte aligned */
  EMUGEMM_ERR_WORKSPACE = -3, /* workspace missing or smaller than emugemm_workspace_bytes() */
  EMUGEMM_ERR_PRECISION = -4, /* Scheme II: k too large for this n_moduli (bit budget T < 2) */
  EMUGEMM_ERR_DEVICE = -5,    /* no CUDA device or not compute capability 10.x */
  EMUGEMM_ERR_CUDA = -6,      /* a CUDA call failed; see emugemm_last_cuda_error() */
  EMUGEMM_ERR_STATIC_LIMIT = -7 /* emugemm_dgemm_oz1_static: the problem needs more than EMUGEMM_STATIC_WS_BYTES of scratch */
};

enum emugemm_scheme { EMUGEMM_OZ1 = 1, EMUGEMM_OZ2 = 2, EMUGEMM_OZ2_3M = 3, EMUGEMM_OZ1_4M = 4 };

/* ---- handle ------------------------------------------------------------- */
int emugemm_create(emugemm_handle_t *h);  /* host-only state; checks the device */
int emugemm_destroy(emugemm_handle_t h);
int emugemm_set_stream(emugemm_handle_t h, void *cuda_stream /* cudaStream_t */);
int emugemm_set_workspace(emugemm_handle_t h, void *dev_ptr, size_t bytes);
/* Scheme I digit format of this handle.  7 (default): digits of 7 bits in the form emugemm_set_slice_form
 * selects (two's-complement fields by default).  8 (R23; "slices of beta <= 8
 * bits"): balanced signed base-256 digits, d in [-128, 127], two guard bits under the row /
 * column exponent -- 8p - 2 bits per operand, so p = 7 reaches the accuracy of p = 8 at 7 bits
 * with 28 instead of 36 slice products.  Applies to dgemm_oz1, sgemm_oz1 and the Scheme I hooks. */
int emugemm_set_slice_bits(emugemm_handle_t h, int bits);
/* Digit FORM of the 7-bit Scheme I slices of this handle (all Scheme I calls, operand handles included).
 *   0 (default; R24; "a signed leading slice with unsigned remaining slices", here at beta = 7 so that
 *     every slice is an INT8 value): the two's-complement fields of X = trunc(x 2^(7p)): d_0 in [-128, 127], d_t in [0, 127]
 *     for t >= 1.  Seven of eight slices carry no sign bits, which the tensor pipe rewards with a higher clock under the
 *     power cap (profiles/r2_operand_sign_power.md: 8192^3 p = 8 74.5 -> 76.9 % of the nominal INT8 peak).
 *   1 (EMUGEMM_DIGITS_SIGN_MAGNITUDE; R1, the default of round 1): d_t = sign(x) * (7-bit field of |X|), all in
 *     [-127, 127].  The SAME integer X, same kernels, same weights; the results of the two forms differ only through the dropped
 *     slice pairs (t + u >= p).
 * Call after emugemm_set_slice_bits (which selects form 0); with 8-bit digits form 1 is EMUGEMM_ERR_ARG.
 * Overflow-safe chunk of a form: emugemm_oz1_chunk_k_bits(p, 7 | 8 | EMUGEMM_DIGITS_SIGN_MAGNITUDE).                          */
#define EMUGEMM_DIGITS_SIGN_MAGNITUDE 0x207
int emugemm_set_slice_form(emugemm_handle_t h, int form);
/* Scheme II real FP64 product (emugemm_dgemm_oz2 and its _t / strided-batched / pre-decomposed forms), SURVEY 8(f) item 4
 * (the paper keeps the CRT separate and pays the residue workspace): on = 1 runs the reconstruction
 * INSIDE the per-modulus GEMM kernel -- a work item is an output tile, the moduli are the inner loop, the tile's
 * residues wait in a per-CTA scratch of 2 x N x 32 KB (the [N][m][n] residue planes are never written), and the epilogue
 * warps run the exact FP64 CRT of the previous tile between the modulus epilogues of the current one.  Applies when
 * 7 <= n_moduli and the scratch (CTAs launched x 2 x N x 32 KB, at most 148 x 2 x N x 32 KB) fits in the workspace from
 * where the residue planes would have started: always for problems of at least two waves of 256 x 256 tiles, else when
 * the workspace has that much room beyond emugemm_workspace_bytes(); otherwise, and with on = 0, the separate CRT kernel
 * runs.  Both paths give bit-identical C.
 * DEFAULT: off -- measured on B200 the fused form is slower (8192^3, N = 16: 8.9 ms against 5.3 + 0.6 ms; the eight
 * epilogue warps cannot hide the FP64 reconstruction and the scratch competes with the operand panels for L2,
 * DESIGN.md 5.7): it is kept as the measured answer to "can Scheme II be fully fused on this machine".           */
int emugemm_set_oz2_fusion(emugemm_handle_t h, int on);
/* Bytes of workspace a call with these arguments needs.  elem = bytes per
 * matrix element: 4 (float), 8 (double), 16 (complex128).  p_or_nmoduli = p for
 * Scheme I, n_moduli for Scheme II / 3M.  Returns 0 for invalid arguments. */
size_t emugemm_workspace_bytes(int scheme, int elem, int64_t m, int64_t n, int64_t k, int p_or_nmoduli);
const char *emugemm_status_string(int status);
int emugemm_last_cuda_error(emugemm_handle_t h); /* cudaError_t of the last EMUGEMM_ERR_CUDA */
/* Non-finite inputs give an unspecified result and no fault (see above); the pre-pass of every one-shot compute call
 * raises a device-side flag when a row of A or a column of B holds an Inf or a NaN (it falls out of the exponent scan:
 * no extra pass).  *seen (HOST) = 1 if the LAST compute call of this handle saw one, else 0; synchronises the stream.
 * EMUGEMM_ERR_WORKSPACE before the first compute call or after the workspace was replaced.                    */
int emugemm_nonfinite_seen(emugemm_handle_t h, int *seen);

/* ---- Scheme I ------------------------------------------ *
 * C = alpha*A*B + beta*C with p signed INT8 slices of beta_bits = 7 bits each
 * under power-of-two row (A) / column (B) exponent scaling; the p(p+1)/2 slice
 * products with i + j < p are computed by ONE fused kernel into p INT32
 * accumulators kept in tensor memory, k is split into chunks that cannot
 * overflow INT32, the epilogue applies Eq. 3 and alpha/beta in FP64.
 * Range: double 1 <= p <= 8, float 1 <= p <= 4.                               */
int emugemm_dgemm_oz1(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, double alpha,
                      const double *A, int64_t lda, const double *B, int64_t ldb, double beta,
                      double *C, int64_t ldc, int p);
int emugemm_sgemm_oz1(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, float alpha,
                      const float *A, int64_t lda, const float *B, int64_t ldb, float beta,
                      float *C, int64_t ldc, int p);

/* Scheme I DGEMM for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): same arguments, same kernels and bit-identical results as emugemm_dgemm_oz1, but the scratch
 * (digit planes, exponents, diagnostics words) lives in a static device array inside the library image instead of a
 * workspace from emugemm_set_workspace -- no workspace is needed and none that is registered is touched.  The call
 * performs no cudaMalloc / cudaFree and calls no allocating library routine.
 *   Limit: emugemm_workspace_bytes(EMUGEMM_OZ1, 8, m, n, k, p) <= EMUGEMM_STATIC_WS_BYTES (32 MiB: e.g. 1024^3 with
 *     p = 8, 2048 x 2048 x 1024 with p = 3); beyond it the call returns EMUGEMM_ERR_STATIC_LIMIT and enqueues nothing.
 *     Every GPU that loads the library holds the array (32 MiB + 1 KiB) until the process exits.
 *   Sharing: ALL calls of this entry point on one device, from every handle, use the one array.  The call zeroes the
 *     words that must start at zero and rewrites every plane byte it reads, so back-to-back calls on ONE stream are
 *     safe; calls that overlap on the GPU (two streams, two handles, two host threads) RACE on the array and give
 *     wrong results -- serialise them, or use emugemm_dgemm_oz1 with one workspace per handle.
 *   A, B, C: device pointers, row-major, 16-byte aligned, owned by the caller; asynchronous on the handle's stream.
 *   Errors: as emugemm_dgemm_oz1 (ARG, ALIGNMENT, CUDA), plus STATIC_LIMIT; never ERR_WORKSPACE.                    */
#define EMUGEMM_STATIC_WS_BYTES (32u << 20)
size_t emugemm_static_workspace_limit(void); /* = EMUGEMM_STATIC_WS_BYTES of the loaded library */
int emugemm_dgemm_oz1_static(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, double alpha,
                             const double *A, int64_t lda, const double *B, int64_t ldb, double beta,
                             double *C, int64_t ldc, int p);

/* Strided batched Scheme I ("a batched implementation is possible through a
 * single interleaved tensor per batch entry"): C_b = alpha*A_b*B_b + beta*C_b for b = 0..batch-1, all of one
 * shape, X_b = X + b*strideX (strides in elements, >= 0; strideA / strideB = 0 shares one operand; the C_b must
 * not overlap: strideC >= (m-1)*ldc + n).  Row-major, no transposes.  Every entry is bit-identical to the
 * single call on it.  The digit planes of all entries are stacked entry-major and ONE fused launch walks
 * (entry, tile) work items, so many small products fill the machine; entries whose k needs several
 * overflow-safe chunks (k > emugemm_oz1_chunk_k) run one by one.  Workspace: emugemm_workspace_bytes(
 * EMUGEMM_OZ1, elem, batch*m, batch*n, k, p).  Limits: batch <= 65535, batch*m and batch*n < 2^31 - 256;
 * with batch > 1 every stride must keep the entries 16-byte aligned (EMUGEMM_ERR_ALIGNMENT).               */
int emugemm_dgemm_oz1_strided_batched(emugemm_handle_t h, int64_t batch, int64_t m, int64_t n, int64_t k,
                                      double alpha, const double *A, int64_t lda, int64_t strideA,
                                      const double *B, int64_t ldb, int64_t strideB, double beta, double *C,
                                      int64_t ldc, int64_t strideC, int p);
int emugemm_sgemm_oz1_strided_batched(emugemm_handle_t h, int64_t batch, int64_t m, int64_t n, int64_t k,
                                      float alpha, const float *A, int64_t lda, int64_t strideA,
                                      const float *B, int64_t ldb, int64_t strideB, float beta, float *C,
                                      int64_t ldc, int64_t strideC, int p);

/* Scheme I complex GEMM by the 4M formulation ("EmuGEMM-I uses the 4M formulation"; SURVEY 8(f)
 * item 3).  A, B, C hold complex128 as (re, im) pairs, strides in complex elements; alpha, beta point to HOST
 * {re, im}.  The four real products run as ONE fused Scheme I GEMM of size 2m x n x 2k on the real embedding
 * A' = [[Re A, -Im A], [Im A, Re A]], B' = [[Re B], [Im B]] (rows i and m + i share the exponent of row i of A).
 * Workspace: emugemm_workspace_bytes(EMUGEMM_OZ1_4M, 16, m, n, k, p).  1 <= p <= 8.                            */
int emugemm_zgemm_oz1_4m(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, const double alpha[2], const double *A,
                         int64_t lda, const double *B, int64_t ldb, const double beta[2], double *C, int64_t ldc, int p);

/* CGEMM: complex64 operands and result as (re, im) float pairs (PAPER.md:299 CGEMM by 4M), the
 * same kernels on 24-bit inputs, one more rounding to float at the end; alpha, beta HOST {re, im} doubles.
 * 1 <= p <= 4; 2 <= n_moduli <= 20 (8-11 cover FP32 accuracy).  Workspace as for the complex128 calls.        */
int emugemm_cgemm_oz1_4m(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, const double alpha[2], const float *A,
                         int64_t lda, const float *B, int64_t ldb, const double beta[2], float *C, int64_t ldc, int p);
int emugemm_cgemm_oz2_3m(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, const double alpha[2], const float *A,
                         int64_t lda, const float *B, int64_t ldb, const double beta[2], float *C, int64_t ldc,
                         int n_moduli);

/* ---- Scheme II ---------------------------------------- *
 * n_moduli pairwise-coprime moduli <= 256 (256, 255, 253, 251, 247, ... greedy
 * descending); symmetric INT8 residues; one INT8 GEMM per modulus with the
 * mod-reduction fused into its epilogue (Eq. 6-7); CRT (Eq. 8) and inverse
 * scaling in FP64.  Range: 2 <= n_moduli <= 20.
 * k: one launch covers one INT32-safe accumulation range (k 128^2 < 2^31, i.e. k <= 130,944 padded columns; R7).
 * A longer k is cut into equal chunks of at most that length: one GEMM launch per chunk, the output residues of the chunks
 * are added modulo m_l (the residues of a sum are the sums of the residues) and ONE reconstruction follows; the
 * workspace then holds a second set of output residue planes (emugemm_workspace_bytes accounts for it).  The bit budget
 * T (emugemm_oz2_budget) is taken for the whole k.  The strided batched entry points run such entries one by one.
 * The FP64 CRT is exact: for every residue vector the reconstructed integer is rounded once (R17), so the
 * 2-ulp bound of (|A||B|)_ij holds for every finite input, not only for well-scaled ones.                       */
int emugemm_dgemm_oz2(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, double alpha,
                      const double *A, int64_t lda, const double *B, int64_t ldb, double beta,
                      double *C, int64_t ldc, int n_moduli);

/* FP32 inputs and output ("EmuGEMM-II SGEMM (p8-p11)"): the same kernels on
 * 24-bit inputs; 8-11 moduli cover FP32 accuracy at k = 8192.                  */
int emugemm_sgemm_oz2(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, float alpha, const float *A, int64_t lda,
                      const float *B, int64_t ldb, float beta, float *C, int64_t ldc, int n_moduli);

/* Strided batched Scheme II, real: conventions, limits and alignment rule as
 * emugemm_dgemm_oz1_strided_batched.  Residue planes of all entries are stacked entry-major; ONE fused launch walks
 * (entry, modulus, tile) work items and ONE CRT launch covers the batch.  Every entry is bit-identical to the single
 * call on it.  Workspace: emugemm_workspace_bytes(EMUGEMM_OZ2 / EMUGEMM_OZ2_3M, elem, batch*m, batch*n, k,
 * n_moduli).                                                                                                */
int emugemm_dgemm_oz2_strided_batched(emugemm_handle_t h, int64_t batch, int64_t m, int64_t n, int64_t k,
                                      double alpha, const double *A, int64_t lda, int64_t strideA,
                                      const double *B, int64_t ldb, int64_t strideB, double beta, double *C,
                                      int64_t ldc, int64_t strideC, int n_moduli);
int emugemm_sgemm_oz2_strided_batched(emugemm_handle_t h, int64_t batch, int64_t m, int64_t n, int64_t k,
                                      float alpha, const float *A, int64_t lda, int64_t strideA,
                                      const float *B, int64_t ldb, int64_t strideB, float beta, float *C,
                                      int64_t ldc, int64_t strideC, int n_moduli);

/* complex128 by 3M, batched: strides in complex elements, alpha / beta point to HOST {re, im}.            */
int emugemm_zgemm_oz2_3m_strided_batched(emugemm_handle_t h, int64_t batch, int64_t m, int64_t n, int64_t k,
                                         const double alpha[2], const double *A, int64_t lda, int64_t strideA,
                                         const double *B, int64_t ldb, int64_t strideB, const double beta[2],
                                         double *C, int64_t ldc, int64_t strideC, int n_moduli);

/* ---- Scheme II complex via 3M ------------------------ *
 * A, B, C hold complex128 as (re, im) pairs; alpha, beta point to HOST {re, im}. */
int emugemm_zgemm_oz2_3m(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, const double alpha[2],
                         const double *A, int64_t lda, const double *B, int64_t ldb,
                         const double beta[2], double *C, int64_t ldc, int n_moduli);

/* ---- transposed operands (SURVEY 8(b) "NEXT": transposes / column-major) -- *
 * C = alpha op(A) op(B) + beta C with op(X) = X (trans = 0) or X^T (trans = 1, no
 * conjugation).  op(A) is m x k: A is stored m x k (lda >= k) or, transposed, k x m
 * (lda >= m); op(B) is k x n: B is stored k x n (ldb >= n) or n x k (ldb >= k).  All
 * row-major.  A column-major BLAS call C = A B is the row-major call C^T = B^T A^T on
 * the same buffers: swap the operands and m <-> n, every transposition flag keeps its
 * meaning.  The pre-pass reads a k-contiguous operand with its row kernel and a
 * k-strided one with its column (transposing) kernel; nothing else changes.        */
int emugemm_dgemm_oz1_t(emugemm_handle_t h, int transa, int transb, int64_t m, int64_t n, int64_t k, double alpha,
                        const double *A, int64_t lda, const double *B, int64_t ldb, double beta, double *C,
                        int64_t ldc, int p);
int emugemm_sgemm_oz1_t(emugemm_handle_t h, int transa, int transb, int64_t m, int64_t n, int64_t k, float alpha,
                        const float *A, int64_t lda, const float *B, int64_t ldb, float beta, float *C,
                        int64_t ldc, int p);
int emugemm_dgemm_oz2_t(emugemm_handle_t h, int transa, int transb, int64_t m, int64_t n, int64_t k, double alpha,
                        const double *A, int64_t lda, const double *B, int64_t ldb, double beta, double *C,
                        int64_t ldc, int n_moduli);
int emugemm_sgemm_oz2_t(emugemm_handle_t h, int transa, int transb, int64_t m, int64_t n, int64_t k, float alpha,
                        const float *A, int64_t lda, const float *B, int64_t ldb, float beta, float *C,
                        int64_t ldc, int n_moduli);
int emugemm_zgemm_oz2_3m_t(emugemm_handle_t h, int transa, int transb, int64_t m, int64_t n, int64_t k,
                           const double alpha[2], const double *A, int64_t lda, const double *B, int64_t ldb,
                           const double beta[2], double *C, int64_t ldc, int n_moduli);

/* ---- pre-decomposed operands ---------- *
 * An operand that takes part in several products is decomposed ONCE (slices or
 * residues + exponents, in the library's private layout, inside a caller-owned device
 * buffer) and then multiplied any number of times with emugemm_gemm_pre(), which
 * runs only the fused GEMM and the reconstruction.  Results are bit-identical to the
 * one-shot calls.  The struct is plain data owned by the caller; the buffer must
 * outlive its uses, be 1024-byte aligned and hold emugemm_operand_bytes() bytes.
 *   scheme : EMUGEMM_OZ1 (elem 4 / 8), EMUGEMM_OZ2 (elem 4 / 8), EMUGEMM_OZ2_3M (elem 16)
 *   role   : 0 = left operand op(A) (rows x k), 1 = right operand op(B) (k x rows)
 *   trans  : as in the _t calls (role 0: X stored k x rows; role 1: X stored rows x k)
 * Scheme II scales an operand with a bit budget that depends on k, n_moduli and the
 * role, so a handle is tied to them; Scheme I handles are tied to p and the digit
 * format of the handle at decomposition time.                                      */
typedef struct emugemm_operand {
  int scheme, role, elem, pn, slice_bits, t_bits;
  int64_t rows, k, kpad;
  void *buf;       /* device: int8 planes [planes][rows][kpad], then int32 exponents [rows] */
  size_t bytes;
} emugemm_operand_t;
size_t emugemm_operand_bytes(int scheme, int64_t rows, int64_t k, int p_or_nmoduli);
int emugemm_decompose(emugemm_handle_t h, int scheme, int role, int trans, int elem, int64_t rows, int64_t k,
                      const void *X, int64_t ldx, int p_or_nmoduli, void *dev_buf, size_t bytes,
                      emugemm_operand_t *out);
/* C (m x n, type by elem: float / double / complex128) = alpha A B + beta C; alpha, beta point to
 * HOST {re, im} (im ignored for real).  A->rows = m, B->rows = n, both with the same scheme, elem,
 * k, p / n_moduli (and digit format).  Needs the workspace of the corresponding one-shot call. */
int emugemm_gemm_pre(emugemm_handle_t h, const emugemm_operand_t *A, const emugemm_operand_t *B, const double alpha[2],
                     const double beta[2], void *C, int64_t ldc);

/* ---- per-stage timing of the last call (bench only) --------------------- *
 * When enabled, compute calls bracket their stages with CUDA events on the
 * handle's stream; emugemm_stage_ms() synchronises and returns milliseconds of
 * stage 0 = pre-pass, 1 = tensor-core GEMM kernel(s), 2 = reconstruction, and the
 * number of kernel launches of the last call in *launches (may be NULL).      */
int emugemm_enable_stage_timing(emugemm_handle_t h, int on);
/* SM cycles (SM clock domain, so independent of the clock frequency) that CTA 0 of
 * the fused tensor-core GEMM kernel(s) of the last compute call spent between its
 * set-up and its exit, summed over the call's GEMM launches; synchronises the
 * stream.  INT8 ops / (cycles * SM count) is the per-clock tensor efficiency
 * bench.py reports against 16384 op/clk/SM.  *cycles is a host pointer.        */
int emugemm_last_gemm_cycles(emugemm_handle_t h, unsigned long long *cycles);
int emugemm_stage_ms(emugemm_handle_t h, float ms[3], int *launches);

/* ---- test hooks (used only by tests/; canonical layouts, device pointers) -
 * They expose the integer intermediates the parity tests compare bit-exactly
 * without exposing the library's private operand layouts.
 * "Canonical slice view": int8 [planes][rows][k] with k contiguous; for operand
 * B the rows are the COLUMNS j of B.  elem = 4 / 8 / 16 as above (16: complex,
 * exponent shared by re and im).                                              */

/* Row (by_cols = 0: X is rows x k, ldx >= k) or column (by_cols = 1: X is
 * k x rows, ldx >= rows) max-exponent scan -> int32 e_out[rows].             */
int emugemm_dbg_exponents(emugemm_handle_t h, int elem, int by_cols, int64_t rows, int64_t k,
                          const void *X, int64_t ldx, int32_t *e_out);
/* Scheme I slices of one operand -> int8 out[p][rows][k], int32 e_out[rows]. */
int emugemm_dbg_oz1_slices(emugemm_handle_t h, int elem, int by_cols, int64_t rows, int64_t k,
                           const void *X, int64_t ldx, int p, int8_t *out, int32_t *e_out);
/* Fused Scheme I kernel with the INT32 accumulators of every k-chunk dumped:
 * out[chunk][p][m][n] (int32), *n_chunks_out chunks (host int).  chunk_k = 0
 * uses the library's overflow-safe chunk length, else that many k per chunk. */
int emugemm_dbg_oz1_accumulators(emugemm_handle_t h, int elem, int64_t m, int64_t n, int64_t k,
                                 const void *A, int64_t lda, const void *B, int64_t ldb, int p,
                                 int64_t chunk_k, int32_t *out, int *n_chunks_out);
/* Scheme II residues of one operand.  elem 8: out[N][rows][k]; elem 16 (3M):
 * out[3][N][rows][k] = re, im, Sigma planes.  t_bits = tA or tB.             */
int emugemm_dbg_oz2_residues(emugemm_handle_t h, int elem, int by_cols, int64_t rows, int64_t k,
                             const void *X, int64_t ldx, int n_moduli, int t_bits, int8_t *out,
                             int32_t *e_out);
/* Per-modulus products with fused reduction from canonical residue planes:
 * real: RA[N][m][k], RB[N][n][k] -> out[N][m][n];
 * is3m: RA[3][N][m][k], RB[3][N][n][k] -> out[2][N][m][n] (re, im).           */
int emugemm_dbg_oz2_modgemm(emugemm_handle_t h, int is3m, int64_t m, int64_t n, int64_t k,
                            int n_moduli, const int8_t *RA, const int8_t *RB, int8_t *out);
/* CRT + scaling alone: CR[N][m][n] int8 -> C (double, ldc), alpha/beta as in dgemm_oz2. */
int emugemm_dbg_oz2_crt(emugemm_handle_t h, int64_t m, int64_t n, int n_moduli, const int8_t *CR,
                        const int32_t *eA, const int32_t *eB, int tA, int tB, double alpha,
                        double beta, double *C, int64_t ldc);
/* Host-side helpers (no GPU): bit budget (returns T or < 0), overflow-safe chunk length. */
int emugemm_oz2_budget(int n_moduli, int64_t k, int is3m, int *tA, int *tB);
/* Host-side (no GPU): the integer constants of the exact FP64 CRT kernel for n_moduli (R17; PAPER.md:127-130
 * Eq. 8), so that a CPU test can check them against big integers.  Moduli are combined in pairs (2q, 2q+1), an odd
 * last one stays alone: *n_pairs = ceil(N/2).  Every pair weight W_q = (P/M_q)((P/M_q)^-1 mod M_q), M_q = m1 m2, and P
 * itself are written in *n_digits balanced base-2^(*digit_bits) digits: digits[q * n_digits + j], q < n_pairs, is
 * digit j of W_q, row q = n_pairs is P (sum_j digit_j 2^(j digit_bits), |digit| <= 2^(digit_bits-1)); pair[5q..5q+4] =
 * {M_q, K1, K2, C0, floor(2^32/M_q)}: x = (K1 c1 + K2 c2 + C0) mod M_q is the pair residue (K1 == 1 mod m1, == 0 mod
 * m2, K2 the other way round; C0 a multiple of M_q >= 2^24).  Caller arrays (HOST): digits >= 11 * 5 int64, pair >=
 * 10 * 5 uint32.  Returns 0, or EMUGEMM_ERR_ARG.                                                                  */
int emugemm_dbg_crt_constants(int n_moduli, int *n_pairs, int *n_digits, int *digit_bits, long long *digits, unsigned *pair);
int64_t emugemm_oz1_chunk_k(int p);                       /* 7-bit digits, default form */
int64_t emugemm_oz1_chunk_k_bits(int p, int code);   /* code 7 (default form) | 8 | EMUGEMM_DIGITS_SIGN_MAGNITUDE: the fullest accumulator stays below 2^31 */
/* ---- PROBES build only (libemugemm_probes.so, compiled with -DEMUGEMM_PROBES; bench.py loads it for its probe leg).
 * The shipped libemugemm.so exports none of the three calls below and carries no experiment switch in its kernels. */
#ifdef EMUGEMM_PROBES
/* Issue-bound tcgen05.mma kind::i8 probe (operands resident in shared memory, no
 * loads in the loop), one CTA per SM.  ops = HOST array of n_ops (<= 64) MMAs, five
 * ints each: {TMEM column of D, width N (multiple of 16, <= 256), A slot 0..7
 * (128 x 128 B tiles), first row of B (rows of 128 B), A collector hint 0 discard /
 * 1 fill / 2 use / 3 lastuse}; one iteration issues the
 * whole schedule, `iters` iterations run back to back.  INT8 ops per CTA =
 * iters * sum_o 2*128*N_o*32.  Returns milliseconds in *ms, the CTA count in *ctas
 * and (if not NULL) the SM cycles block 0 spent in *cycles (host pointers).  Needs a
 * workspace of >= 8 bytes.  bench.py uses it for the third INT8 denominator
 * (SURVEY 8(d)); DESIGN.md quotes its schedule measurements.                  */
int emugemm_dbg_i8_probe(emugemm_handle_t h, int n_ops, const int *ops, int iters, float *ms, int *ctas,
                         long long *cycles);

/* The MMA issue code of the fused Scheme I kernel for p slices, run `iters` times
 * (one iteration = one 128-byte k-block = 4 k32 steps) on operands resident in
 * shared memory (pseudo-random bytes), one CTA per SM: the tensor-pipe ceiling of
 * that schedule without TMA traffic.  INT8 ops per CTA = iters * 4 * p(p+1) * 128 *
 * NT(p) * 32.  use_collector bit 0 selects the A-operand collector hints, bit 1 the
 * one-MMA-per-product schedule (width NT) instead of the N-concatenated one.   */
int emugemm_dbg_oz1_issue_probe(emugemm_handle_t h, int p, int use_collector, int iters, float *ms, int *ctas,
                                long long *cycles);

/* Timing experiments on the fused kernels (results become WRONG, never set in
 * production): bit 0 = the TMA producer stops loading once its ring has been filled
 * once (barrier traffic unchanged), bit 1 = the epilogue skips its TMEM reads, math
 * and stores, bit 2 = only the stores are skipped, bit 3 = Scheme I with p <= 3 runs
 * the one-CTA N-concatenated kernel instead of the CTA-pair kernel, bit 4 = Scheme I
 * with p >= 4 runs without the 2-CTA multicast of A (A/B timing), bit 5 = the Scheme I
 * row pre-pass runs its two-phase form (row re-read) instead of the register-resident
 * single-read kernel; 0x40 = every CTA loads tile (0, 0) (no DRAM traffic, same L2 -> SM traffic), 0x80 = no serpentine k,
 * 0xFF00 = rasterisation group override, 0x10000 = wave barrier off, 0x20000 / 0x40000 = wave barrier forced on
 * (Scheme II real / Scheme I), 0x80000 / 0x100000 = fused Scheme II without the CRT arithmetic / the scratch loads,
 * 0x200000 / 0x400000 / 0x800000 = L2 eviction hints A EVICT_LAST / B EVICT_FIRST / B EVICT_LAST (results stay right),
 * 0x0F000000 = wave-barrier lead 2 (v - 1) k-blocks, 0x20000000 = set the device's persisting-L2 carve-out to its maximum
 * (device-wide and sticky: probe processes only).
 * Used to attribute tensor-pipe idle time and DRAM traffic (profiles/r2_wave_barrier.md).                  */
int emugemm_dbg_set_flags(emugemm_handle_t h, int flags);

#endif /* EMUGEMM_PROBES */

#ifdef __cplusplus
}
#endif
#endif /* EMUGEMM_H_ */
