// api.cu -- the C ABI of include/emugemm.h: handle, workspace carving, the
// per-call stage sequence (pre-pass -> fused tensor-core GEMM -> reconstruction)
// and the test hooks.  Host code only; every compute step runs in the kernels of
// prepass.cu / gemm_oz1.cu / gemm_oz2.cu / crt.cu.  There is no CPU fallback.
#include <cudaTypedefs.h>

#include <new>

#include "common.cuh"

using namespace emu;

namespace emu {

int encode_planes_tmap(emugemm_ctx *ctx, CUtensorMap *tm, const void *base, int64_t kpad, int64_t rows,
                       int64_t planes, int box_rows, int box_planes) {
  const cuuint64_t dims[3] = {static_cast<cuuint64_t>(kpad), static_cast<cuuint64_t>(rows),
                              static_cast<cuuint64_t>(planes)};
  const cuuint64_t strides[2] = {static_cast<cuuint64_t>(kpad), static_cast<cuuint64_t>(kpad) * static_cast<cuuint64_t>(rows)};
  const cuuint32_t box[3] = {static_cast<cuuint32_t>(kBlockK), static_cast<cuuint32_t>(box_rows),
                             static_cast<cuuint32_t>(box_planes)};
  const cuuint32_t estr[3] = {1, 1, 1};
  const CUresult r = ctx->encode(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void *>(base), dims, strides, box, estr,
                                 CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                 CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    ctx->last_cuda = static_cast<int>(r);
    return EMUGEMM_ERR_CUDA;
  }
  return EMUGEMM_OK;
}

// bump allocator over the caller's workspace (1024-byte granules)
struct Carver {
  uint8_t *p;
  size_t left;
  bool ok = true;
  Carver(void *base, size_t bytes) : p(static_cast<uint8_t *>(base)), left(bytes) {}
  template <typename T>
  T *take(size_t count) {
    const size_t bytes = static_cast<size_t>(round_up(static_cast<int64_t>(count * sizeof(T)), 1024));
    if (bytes > left) { ok = false; return nullptr; }
    T *r = reinterpret_cast<T *>(p);
    p += bytes;
    left -= bytes;
    return r;
  }
};
static size_t granule(size_t bytes) { return static_cast<size_t>(round_up(static_cast<int64_t>(bytes), 1024)); }

static int oz1_chunks(int p, int bits, int64_t kpad, int64_t chunk_override, int64_t *chunk_len) {
  int64_t c = chunk_override > 0 ? round_up(chunk_override, kBlockK) : oz1_chunk_k_host(p, bits);
  if (c > oz1_chunk_k_host(p, bits)) c = oz1_chunk_k_host(p, bits);
  int n = static_cast<int>((kpad + c - 1) / c);
  if (n < 1) n = 1;
  // equalise the chunks (same number, balanced length, still <= the safe bound)
  if (chunk_override <= 0) c = round_up((kpad + n - 1) / n, kBlockK);
  *chunk_len = c;
  return n;
}

// Chunk count of a one-shot / operand-handle Scheme I product: the overflow-safe minimum, or -- when k needs several
// chunks anyway and the output has so few tiles that whole waves of the persistent kernel would run partly empty -- up
// to twice as many, shorter chunks, chosen to minimise (waves of work items) x (chunk length + the per-item epilogue,
// ~250 columns' worth of MMA time).  1024 x 1024 x 65536 at p = 7: 64 cluster tiles x 4 chunks = 256 items on 74 workers
// = 4 waves of 16,384 columns; with 8 chunks 512 items = 7 waves of 8,192: 12 % less.  The partials are exact
// double-doubles, so the chunk count does not change the result (tests/test_gpu_full_size.py, k = 65,536).
static constexpr int64_t kChunkItemOverheadK = 256;
static bool oz1_chunks_may_balance(int nmin, int64_t tiles) { return nmin >= 2 && tiles * nmin < 8 * 128; }
static int oz1_chunks_balanced(int p, int bits, int64_t kpad, int64_t m, int64_t n, int num_sms, int64_t *chunk_len) {
  int64_t clen;
  const int nmin = oz1_chunks(p, bits, kpad, 0, &clen);
  *chunk_len = clen;
  const int64_t tiles = oz1_cluster_tiles_host(p, m, n), workers = num_sms / 2;
  if (!oz1_chunks_may_balance(nmin, tiles) || workers < 1 || tiles * nmin >= 8 * workers) return nmin;
  int best = nmin;
  int64_t best_cost = -1;
  for (int c = nmin; c <= 2 * nmin; ++c) {
    const int64_t len = round_up((kpad + c - 1) / c, kBlockK);
    const int nc = static_cast<int>((kpad + len - 1) / len);  // chunks actually needed at this length
    const int64_t waves = (tiles * nc + workers - 1) / workers;
    const int64_t cost = waves * (len + kChunkItemOverheadK);
    if (best_cost < 0 || cost < best_cost) { best_cost = cost; best = nc; *chunk_len = len; }
  }
  return best;
}

static size_t ws_common(int64_t m, int64_t n) {
  return 1024 /*diagnostics*/ + granule(8 * m) + granule(8 * n) + granule(4 * m) + granule(4 * n);
}

__global__ void scale_c_kernel(int64_t m, int64_t n, double br, double bi, void *C, int64_t ldc, int elem) {
  const int64_t idx = static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x;
  if (idx >= m * n) return;
  const int64_t i = idx / n, j = idx - i * n;
  if (elem == 8) {
    double *o = static_cast<double *>(C) + i * ldc + j;
    *o = (br == 0.0) ? 0.0 : br * *o;
  } else if (elem == 4) {
    float *o = static_cast<float *>(C) + i * ldc + j;
    *o = (br == 0.0) ? 0.0f : static_cast<float>(br) * *o;
  } else if (elem == 64) {  // complex64
    float *o = static_cast<float *>(C) + 2 * (i * ldc + j);
    const double re = o[0], im = o[1];
    if (br == 0.0 && bi == 0.0) { o[0] = 0.0f; o[1] = 0.0f; }
    else { o[0] = static_cast<float>(br * re - bi * im); o[1] = static_cast<float>(br * im + bi * re); }
  } else {
    double *o = static_cast<double *>(C) + 2 * (i * ldc + j);
    const double re = o[0], im = o[1];
    if (br == 0.0 && bi == 0.0) { o[0] = 0.0; o[1] = 0.0; }
    else { o[0] = br * re - bi * im; o[1] = br * im + bi * re; }
  }
}

// C = alpha (T[i][j] + i T[m + i][j]) + beta C: the complex combination of the 4M real embedding result T (2m x n)
template <typename TC /* double or float: component type of C */>
__global__ void zcombine_4m_kernel(int64_t m, int64_t n, const double *__restrict__ T, double ar, double ai, double br, double bi,
                                   TC *__restrict__ C, int64_t ldc) {
  const int64_t idx = static_cast<int64_t>(blockIdx.x) * 256 + threadIdx.x;
  if (idx >= m * n) return;
  const int64_t i = idx / n, j = idx - i * n;
  const double tr = T[idx], ti = T[idx + m * n];
  double re = ar * tr - ai * ti, im = ar * ti + ai * tr;
  TC *o = C + 2 * (i * ldc + j);
  if (br != 0.0 || bi != 0.0) {
    const double cr = o[0], ci = o[1];
    re += br * cr - bi * ci;
    im += br * ci + bi * cr;
  }
  o[0] = static_cast<TC>(re);
  o[1] = static_cast<TC>(im);
}

static int scale_c(emugemm_ctx *h, int64_t m, int64_t n, double br, double bi, void *C, int64_t ldc, int elem) {
  scale_c_kernel<<<static_cast<unsigned>((m * n + 255) / 256), 256, 0, h->stream>>>(m, n, br, bi, C, ldc, elem);
  h->launches++;
  EMU_CUDA(h, cudaGetLastError());
  return EMUGEMM_OK;
}

static int mark(emugemm_ctx *h, int i) {
  if (h->timing) EMU_CUDA(h, cudaEventRecord(h->ev[i], h->stream));
  return EMUGEMM_OK;
}

// degenerate calls (m n == 0) launch nothing: the stage events are still recorded so that emugemm_stage_ms stays valid
static int mark_all(emugemm_ctx *h) {
  for (int i = 0; i < 4; ++i) EMU_TRY(mark(h, i));
  return EMUGEMM_OK;
}

static int check_gemm_args(emugemm_ctx *h, int ta, int tb, int64_t m, int64_t n, int64_t k, const void *A, int64_t lda,
                           const void *B, int64_t ldb, const void *C, int64_t ldc) {
  if (!h) return EMUGEMM_ERR_ARG;
  if (m < 0 || n < 0 || k < 0 || (ta & ~1) || (tb & ~1)) return EMUGEMM_ERR_ARG;
  if (m == 0 || n == 0) return EMUGEMM_OK;
  if (!C || ldc < n) return EMUGEMM_ERR_ARG;
  // op(A) is m x k: stored m x k (lda >= k) or, transposed, k x m (lda >= m); op(B) is k x n likewise
  if (k > 0 && (!A || !B || lda < (ta ? m : k) || ldb < (tb ? k : n))) return EMUGEMM_ERR_ARG;
  if ((reinterpret_cast<uintptr_t>(A) | reinterpret_cast<uintptr_t>(B) | reinterpret_cast<uintptr_t>(C)) & 15)
    return EMUGEMM_ERR_ALIGNMENT;
  if (k >= (1LL << 31) - 256 || m >= (1LL << 31) - 256 || n >= (1LL << 31) - 256) return EMUGEMM_ERR_ARG;
  // the k-strided (column) pre-pass puts k / 128 in grid.y (<= 65535): a clean argument error instead of a launch failure
  // after part of the call has been enqueued; 8,388,480 is far beyond any workspace a B200 can hold anyway
  if (k > 65535LL * kBlockK) return EMUGEMM_ERR_ARG;
  return EMUGEMM_OK;
}

// Fused GEMM (one launch per overflow-safe k-chunk) + chunk reduction from sliced operands (shared by the one-shot
// calls and the pre-decomposed operand path).
static int oz1_gemm_phase(emugemm_ctx *h, int elem, int64_t m, int64_t n, int64_t kpad, int p, int bits, const int8_t *SA,
                          const int8_t *SB, const int32_t *eA, const int32_t *eB, double alpha, double beta, void *C,
                          int64_t ldc, int32_t *dump, int nch, int64_t clen, double *part, unsigned long long *diag,
                          int batch = 1, int64_t batch_stride_c = 0) {
  Oz1GemmArgs g;
  g.batch = batch; g.batch_stride_c = batch_stride_c;
  g.m = m; g.n = n; g.kpad = kpad; g.p = p; g.slice_bits = bits; g.SA = SA; g.SB = SB; g.eA = eA; g.eB = eB;
  g.alpha = alpha; g.beta = beta; g.C = C; g.ldc = ldc; g.cycles = diag;
  g.wave_ctr = diag ? diag + kDiagWaveCtr : nullptr;
  const int final_kind = (elem == kF32) ? 1 : 0;
  // ONE launch: with several overflow-safe k-chunks a work item of the persistent kernel is (chunk, tile), so short
  // chunks of a long-k problem still fill the machine
  g.k0 = 0; g.k1 = kpad; g.n_chunks = nch; g.chunk_k = clen;
  if (dump) { g.out_kind = 2; g.C = dump; g.chunk_stride = static_cast<int64_t>(p) * m * n * 4; }
  else if (nch == 1) { g.out_kind = final_kind; g.chunk_stride = 0; }
  else { g.out_kind = 3; g.C = part; g.chunk_stride = m * n * 16; }
  EMU_TRY(launch_oz1_gemm(h, g));
  EMU_TRY(mark(h, 2));
  if (nch > 1 && !dump) EMU_TRY(launch_oz1_chunk_reduce(h, m, n, nch, part, final_kind, alpha, beta, C, ldc));
  EMU_TRY(mark(h, 3));
  return EMUGEMM_OK;
}

// Scheme I call sequence; out_mode: 0 final, 2 = INT32 dump per chunk into `dump`
static int run_oz1(emugemm_ctx *h, int ta, int tb, int elem, int64_t m, int64_t n, int64_t k, double alpha, const void *A, int64_t lda,
                   const void *B, int64_t ldb, double beta, void *C, int64_t ldc, int p, int32_t *dump,
                   int64_t chunk_override, int *n_chunks_out) {
  EMU_TRY(check_gemm_args(h, ta, tb, m, n, k, A, lda, B, ldb, dump ? static_cast<const void *>(dump) : C, dump ? n : ldc));
  if (p < 1 || p > (elem == kF32 ? 4 : 8)) return EMUGEMM_ERR_ARG;
  h->launches = 0;
  if (m == 0 || n == 0) return mark_all(h);
  EMU_TRY(mark(h, 0));
  if (k == 0) {
    if (!dump) EMU_TRY(scale_c(h, m, n, beta, 0.0, C, ldc, elem));
    if (n_chunks_out) *n_chunks_out = 0;
    EMU_TRY(mark(h, 1)); EMU_TRY(mark(h, 2)); EMU_TRY(mark(h, 3));
    return EMUGEMM_OK;
  }
  const int64_t kpad = round_up(k, kBlockK);
  int64_t clen;
  const int bits = h->slice_bits;
  // the dump hook and an explicit chunk length keep the plain split; product calls may take more, shorter chunks
  const int nch = (dump || chunk_override > 0) ? oz1_chunks(p, bits, kpad, chunk_override, &clen)
                                               : oz1_chunks_balanced(p, bits, kpad, m, n, h->num_sms, &clen);
  if (!h->ws || (reinterpret_cast<uintptr_t>(h->ws) & 1023)) return h->ws ? EMUGEMM_ERR_ALIGNMENT : EMUGEMM_ERR_WORKSPACE;
  Carver cv(h->ws, h->ws_bytes);
  auto *diag = cv.take<unsigned long long>(1);
  auto *mbA = cv.take<unsigned long long>(m);
  auto *mbB = cv.take<unsigned long long>(n);
  auto *eA = cv.take<int32_t>(m);
  auto *eB = cv.take<int32_t>(n);
  auto *SA = cv.take<int8_t>(static_cast<size_t>(p) * m * kpad);
  auto *SB = cv.take<int8_t>(static_cast<size_t>(p) * n * kpad);
  double *part = (nch > 1 && !dump) ? cv.take<double>(static_cast<size_t>(nch) * m * n * 2) : nullptr;
  if (!cv.ok) return EMUGEMM_ERR_WORKSPACE;
  h->diag = diag;
  h->nf_flag = diag + kDiagNonFinite;
  EMU_CUDA(h, cudaMemsetAsync(diag, 0, kDiagBytes, h->stream));

  // planes are indexed [row of op(A)] / [column of op(B)] with k contiguous: a k-major stored operand (A^T stored
  // k x m, B stored k x n) goes through the column kernels, an operand whose k is contiguous through the row kernel
  EMU_TRY(launch_oz1_slice(h, elem, ta, m, k, kpad, A, lda, mbA, eA, p, bits, SA));
  EMU_TRY(launch_oz1_slice(h, elem, !tb, n, k, kpad, B, ldb, mbB, eB, p, bits, SB));
  EMU_TRY(mark(h, 1));
  EMU_TRY(oz1_gemm_phase(h, elem, m, n, kpad, p, bits, SA, SB, eA, eB, alpha, beta, C, ldc, dump, nch, clen, part, diag));
  if (n_chunks_out) *n_chunks_out = nch;
  return EMUGEMM_OK;
}

// Strided batched Scheme I: `batch` independent products of one shape.  The digit
// planes of all entries are stacked entry-major ([p][batch m][kpad], [p][batch n][kpad]), the pre-pass kernels take
// the entry from a grid dimension and ONE persistent fused launch walks (entry, tile) work items, so many small
// products fill the machine.  Entries whose k needs several overflow-safe chunks, and k = 0, run one by one.
static int run_oz1_batched(emugemm_ctx *h, int elem, int64_t batch, int64_t m, int64_t n, int64_t k, double alpha,
                           const void *A, int64_t lda, int64_t strideA, const void *B, int64_t ldb, int64_t strideB,
                           double beta, void *C, int64_t ldc, int64_t strideC, int p) {
  if (!h || batch < 0 || strideA < 0 || strideB < 0 || strideC < 0) return EMUGEMM_ERR_ARG;
  EMU_TRY(check_gemm_args(h, 0, 0, m, n, k, A, lda, B, ldb, C, ldc));
  if (p < 1 || p > (elem == kF32 ? 4 : 8)) return EMUGEMM_ERR_ARG;
  h->launches = 0;
  if (batch == 0 || m == 0 || n == 0) return mark_all(h);
  const int64_t es = (elem == kF32) ? 4 : 8;
  if (batch > 1) {
    if (((strideA * es) | (strideB * es) | (strideC * es)) & 15) return EMUGEMM_ERR_ALIGNMENT;
    if (strideC < (m - 1) * ldc + n) return EMUGEMM_ERR_ARG;  // the outputs must not overlap (inputs may: stride 0 shares one)
    if (batch > 65535 || batch * m >= (1LL << 31) - 256 || batch * n >= (1LL << 31) - 256) return EMUGEMM_ERR_ARG;
  }
  const int64_t kpad = round_up(k, kBlockK);
  int64_t clen = 0;
  const int bits = h->slice_bits;
  const int nch = k > 0 ? oz1_chunks(p, bits, kpad, 0, &clen) : 0;
  if (batch == 1 || k == 0 || nch > 1) {
    int launches = 0;
    for (int64_t b = 0; b < batch; ++b) {
      EMU_TRY(run_oz1(h, 0, 0, elem, m, n, k, alpha, static_cast<const char *>(A) + b * strideA * es, lda,
                      static_cast<const char *>(B) + b * strideB * es, ldb, beta, static_cast<char *>(C) + b * strideC * es, ldc, p,
                      nullptr, 0, nullptr));
      launches += h->launches;
    }
    h->launches = launches;
    return EMUGEMM_OK;
  }
  EMU_TRY(mark(h, 0));
  if (!h->ws || (reinterpret_cast<uintptr_t>(h->ws) & 1023)) return h->ws ? EMUGEMM_ERR_ALIGNMENT : EMUGEMM_ERR_WORKSPACE;
  const int64_t M = batch * m, N = batch * n;
  Carver cv(h->ws, h->ws_bytes);  // the layout of a single M x N x k call: emugemm_workspace_bytes(1, elem, batch m, batch n, k, p)
  auto *diag = cv.take<unsigned long long>(1);
  auto *mbA = cv.take<unsigned long long>(M);
  auto *mbB = cv.take<unsigned long long>(N);
  auto *eA = cv.take<int32_t>(M);
  auto *eB = cv.take<int32_t>(N);
  auto *SA = cv.take<int8_t>(static_cast<size_t>(p) * M * kpad);
  auto *SB = cv.take<int8_t>(static_cast<size_t>(p) * N * kpad);
  if (!cv.ok) return EMUGEMM_ERR_WORKSPACE;
  h->diag = diag;
  h->nf_flag = diag + kDiagNonFinite;
  EMU_CUDA(h, cudaMemsetAsync(diag, 0, kDiagBytes, h->stream));
  const int nb = static_cast<int>(batch);
  EMU_TRY(launch_oz1_slice(h, elem, 0, m, k, kpad, A, lda, mbA, eA, p, bits, SA, nb, strideA));
  EMU_TRY(launch_oz1_slice(h, elem, 1, n, k, kpad, B, ldb, mbB, eB, p, bits, SB, nb, strideB));
  EMU_TRY(mark(h, 1));
  return oz1_gemm_phase(h, elem, m, n, kpad, p, bits, SA, SB, eA, eB, alpha, beta, C, ldc, nullptr, 1, clen, nullptr, diag, nb,
                        strideC * es);
}

// Output residue planes of a Scheme II call: [parts_out][N][m][n] INT8; a k beyond one INT32-safe range (kOz2MaxChunkK) is cut
// into chunks whose output residues are added modulo m_l, which takes a second buffer of the same size right behind the first
static size_t oz2_cr_elems(int parts_out, int N, int64_t m, int64_t n, int64_t kpad) {
  const size_t one = granule(static_cast<size_t>(parts_out) * N * m * n);
  return kpad > kOz2MaxChunkK ? 2 * one : one;
}

// Per-modulus GEMMs with fused reduction + CRT from residue planes (one-shot calls and pre-decomposed operands).
static int oz2_gemm_phase(emugemm_ctx *h, int is3m, int64_t m, int64_t n, int64_t kpad, int N, const int8_t *RA,
                          const int8_t *RB, int8_t *CR, const int32_t *eA, const int32_t *eB, int tA, int tB,
                          const double alpha[2], const double beta[2], double *C, int64_t ldc, unsigned long long *diag,
                          int out_f32 = 0, int batch = 1, int64_t batch_stride_c = 0) {
  Oz2GemmArgs g;
  g.batch = batch;
  g.m = m; g.n = n; g.kpad = kpad; g.n_moduli = N; g.is3m = is3m; g.RA = RA; g.RB = RB; g.CR = CR; g.cycles = diag;
  g.wave_ctr = diag ? diag + kDiagWaveCtr : nullptr;
  Oz2CrtArgs c;
  c.m = m; c.n = n; c.n_moduli = N; c.CR = CR; c.eA = eA; c.eB = eB; c.tA = tA; c.tB = tB; c.is_complex = is3m; c.out_f32 = out_f32;
  c.alpha[0] = alpha[0]; c.alpha[1] = alpha[1]; c.beta[0] = beta[0]; c.beta[1] = beta[1];
  c.C = C; c.ldc = ldc; c.batch = batch; c.batch_stride_c = batch_stride_c;
  // Fused reconstruction (opt-in): real FP64 product, 7 <= N <= 20, and the per-CTA scratch (2 x N x
  // 32 KB for each of the <= num_sms CTAs) must fit in the workspace from where the residue planes would have started --
  // true for every problem of at least two waves of 256 x 256 tiles, or when the caller's workspace has that much room
  // beyond emugemm_workspace_bytes(); otherwise the separate CRT kernel runs.
  const int64_t tiles_out = ((m + 255) / 256) * ((n + 255) / 256) * batch;
  const int64_t ctas = 2 * (tiles_out < h->num_sms / 2 ? tiles_out : h->num_sms / 2);
  // CR is the last region carved from the workspace by every caller: the scratch may use everything from there on
  const size_t avail = static_cast<size_t>((static_cast<const uint8_t *>(h->ws) + h->ws_bytes) - reinterpret_cast<const uint8_t *>(CR));
  if (h->oz2_fusion && !is3m && !out_f32 && N >= 7 && kpad <= kOz2MaxChunkK && static_cast<size_t>(ctas) * 2 * N * 32768 <= avail) {
    g.fused = &c;
    g.scratch_bytes = avail;
    EMU_TRY(launch_oz2_gemm(h, g));
    EMU_TRY(mark(h, 2));
    EMU_TRY(mark(h, 3));
    return EMUGEMM_OK;
  }
  if (kpad > kOz2MaxChunkK) {
    // k-chunks of at most kOz2MaxChunkK columns (equalised): chunk 0 writes CR, every later chunk writes the second buffer
    // and is added modulo m_l (the residues of a sum are the sums of the residues)
    if (batch != 1) return EMUGEMM_ERR_ARG;  // the batched entry points run such entries one by one
    const int parts_out = is3m ? 2 : 1;
    const int nch = static_cast<int>((kpad + kOz2MaxChunkK - 1) / kOz2MaxChunkK);
    const int64_t clen = round_up((kpad + nch - 1) / nch, kBlockK);
    int8_t *CRtmp = CR + granule(static_cast<size_t>(parts_out) * N * m * n);
    for (int64_t k0 = 0; k0 < kpad; k0 += clen) {
      g.k0 = k0;
      g.k1 = k0 + clen < kpad ? k0 + clen : kpad;
      g.CR = k0 == 0 ? CR : CRtmp;
      if (k0 > 0 && g.wave_ctr) EMU_CUDA(h, cudaMemsetAsync(g.wave_ctr, 0, sizeof(unsigned long long), h->stream));
      EMU_TRY(launch_oz2_gemm(h, g));
      if (k0 > 0) EMU_TRY(launch_oz2_residue_add(h, CR, CRtmp, N, parts_out * N, m * n));
    }
  } else {
    EMU_TRY(launch_oz2_gemm(h, g));
  }
  EMU_TRY(mark(h, 2));
  EMU_TRY(launch_oz2_crt(h, c));
  EMU_TRY(mark(h, 3));
  return EMUGEMM_OK;
}

// Scheme II call sequence (real and 3M)
static int run_oz2(emugemm_ctx *h, int ta, int tb, int is3m, int64_t m, int64_t n, int64_t k, const double alpha[2], const void *A,
                   int64_t lda, const void *B, int64_t ldb, const double beta[2], double *C, int64_t ldc, int N, int f32 = 0) {
  EMU_TRY(check_gemm_args(h, ta, tb, m, n, k, A, lda, B, ldb, C, ldc));
  if (N < 2 || N > kMaxModuli) return EMUGEMM_ERR_ARG;
  h->launches = 0;
  if (m == 0 || n == 0) return mark_all(h);
  const int elem = is3m ? (f32 ? kC64 : kZ128) : (f32 ? kF32 : kF64);
  EMU_TRY(mark(h, 0));
  if (k == 0) {
    EMU_TRY(scale_c(h, m, n, beta[0], beta[1], C, ldc, elem));
    EMU_TRY(mark(h, 1)); EMU_TRY(mark(h, 2)); EMU_TRY(mark(h, 3));
    return EMUGEMM_OK;
  }
  int tA, tB;
  if (oz2_budget_host(N, k, is3m, &tA, &tB) < 2) return EMUGEMM_ERR_PRECISION;
  const int64_t kpad = round_up(k, kBlockK);  // k beyond one INT32-safe range (R7) is chunked inside oz2_gemm_phase
  const int parts_in = is3m ? 3 : 1, parts_out = is3m ? 2 : 1;
  if (!h->ws || (reinterpret_cast<uintptr_t>(h->ws) & 1023)) return h->ws ? EMUGEMM_ERR_ALIGNMENT : EMUGEMM_ERR_WORKSPACE;
  Carver cv(h->ws, h->ws_bytes);
  auto *diag = cv.take<unsigned long long>(1);
  auto *mbA = cv.take<unsigned long long>(m);
  auto *mbB = cv.take<unsigned long long>(n);
  auto *eA = cv.take<int32_t>(m);
  auto *eB = cv.take<int32_t>(n);
  auto *RA = cv.take<int8_t>(static_cast<size_t>(parts_in) * N * m * kpad);
  auto *RB = cv.take<int8_t>(static_cast<size_t>(parts_in) * N * n * kpad);
  auto *CR = cv.take<int8_t>(oz2_cr_elems(parts_out, N, m, n, kpad));
  if (!cv.ok) return EMUGEMM_ERR_WORKSPACE;
  h->diag = diag;
  h->nf_flag = diag + kDiagNonFinite;
  EMU_CUDA(h, cudaMemsetAsync(diag, 0, kDiagBytes, h->stream));

  EMU_TRY(launch_oz2_residues(h, elem, ta, m, k, kpad, A, lda, mbA, eA, N, tA, RA));
  EMU_TRY(launch_oz2_residues(h, elem, !tb, n, k, kpad, B, ldb, mbB, eB, N, tB, RB));
  EMU_TRY(mark(h, 1));
  return oz2_gemm_phase(h, is3m, m, n, kpad, N, RA, RB, CR, eA, eB, tA, tB, alpha, beta, C, ldc, diag, f32);
}

// Strided batched Scheme II (DGEMM / SGEMM / ZGEMM-3M): as run_oz1_batched -- residue planes of all entries stacked
// entry-major, the pre-pass kernels take the entry from a grid dimension, ONE persistent launch walks
// (entry, modulus, tile) work items, one CRT launch covers the batch (grid.y = entry).
static int run_oz2_batched(emugemm_ctx *h, int is3m, int f32, int64_t batch, int64_t m, int64_t n, int64_t k,
                           const double al[2], const void *A, int64_t lda, int64_t strideA, const void *B, int64_t ldb,
                           int64_t strideB, const double be[2], void *C, int64_t ldc, int64_t strideC, int N) {
  if (!h || batch < 0 || strideA < 0 || strideB < 0 || strideC < 0) return EMUGEMM_ERR_ARG;
  EMU_TRY(check_gemm_args(h, 0, 0, m, n, k, A, lda, B, ldb, C, ldc));
  if (N < 2 || N > kMaxModuli) return EMUGEMM_ERR_ARG;
  h->launches = 0;
  if (batch == 0 || m == 0 || n == 0) return mark_all(h);
  if (is3m && f32) return EMUGEMM_ERR_ARG;
  const int elem = is3m ? kZ128 : (f32 ? kF32 : kF64);
  const int64_t es = is3m ? 16 : (f32 ? 4 : 8);
  const int parts_in = is3m ? 3 : 1, parts_out = is3m ? 2 : 1;
  if (batch > 1) {
    if (((strideA * es) | (strideB * es) | (strideC * es)) & 15) return EMUGEMM_ERR_ALIGNMENT;
    if (strideC < (m - 1) * ldc + n) return EMUGEMM_ERR_ARG;
    if (batch > 65535 || batch * m >= (1LL << 31) - 256 || batch * n >= (1LL << 31) - 256) return EMUGEMM_ERR_ARG;
  }
  if (batch == 1 || k == 0 || round_up(k, kBlockK) > kOz2MaxChunkK) {  // k-chunked entries run one by one
    int launches = 0;
    for (int64_t b = 0; b < batch; ++b) {
      EMU_TRY(run_oz2(h, 0, 0, is3m, m, n, k, al, static_cast<const char *>(A) + b * strideA * es, lda,
                      static_cast<const char *>(B) + b * strideB * es, ldb, be,
                      reinterpret_cast<double *>(static_cast<char *>(C) + b * strideC * es), ldc, N, f32));
      launches += h->launches;
    }
    h->launches = launches;
    return EMUGEMM_OK;
  }
  int tA, tB;
  if (oz2_budget_host(N, k, is3m, &tA, &tB) < 2) return EMUGEMM_ERR_PRECISION;
  EMU_TRY(mark(h, 0));
  const int64_t kpad = round_up(k, kBlockK);
  if (!h->ws || (reinterpret_cast<uintptr_t>(h->ws) & 1023)) return h->ws ? EMUGEMM_ERR_ALIGNMENT : EMUGEMM_ERR_WORKSPACE;
  const int64_t M = batch * m, NN = batch * n;
  Carver cv(h->ws, h->ws_bytes);  // the layout of a single (batch m) x (batch n) x k call is an upper bound
  auto *diag = cv.take<unsigned long long>(1);
  auto *mbA = cv.take<unsigned long long>(M);
  auto *mbB = cv.take<unsigned long long>(NN);
  auto *eA = cv.take<int32_t>(M);
  auto *eB = cv.take<int32_t>(NN);
  auto *RA = cv.take<int8_t>(static_cast<size_t>(parts_in) * N * M * kpad);
  auto *RB = cv.take<int8_t>(static_cast<size_t>(parts_in) * N * NN * kpad);
  auto *CR = cv.take<int8_t>(static_cast<size_t>(parts_out) * N * M * n);
  if (!cv.ok) return EMUGEMM_ERR_WORKSPACE;
  h->diag = diag;
  h->nf_flag = diag + kDiagNonFinite;
  EMU_CUDA(h, cudaMemsetAsync(diag, 0, kDiagBytes, h->stream));
  const int nb = static_cast<int>(batch);
  EMU_TRY(launch_oz2_residues(h, elem, 0, m, k, kpad, A, lda, mbA, eA, N, tA, RA, nb, strideA));
  EMU_TRY(launch_oz2_residues(h, elem, 1, n, k, kpad, B, ldb, mbB, eB, N, tB, RB, nb, strideB));
  EMU_TRY(mark(h, 1));
  return oz2_gemm_phase(h, is3m, m, n, kpad, N, RA, RB, CR, eA, eB, tA, tB, al, be, static_cast<double *>(C), ldc, diag, f32, nb,
                        strideC);
}

}  // namespace emu

// =============================================================================
extern "C" {
#pragma GCC visibility push(default)

int emugemm_create(emugemm_handle_t *out) {
  if (!out) return EMUGEMM_ERR_ARG;
  *out = nullptr;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return EMUGEMM_ERR_DEVICE;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return EMUGEMM_ERR_DEVICE;
  if (prop.major != 10) return EMUGEMM_ERR_DEVICE;  // tcgen05 kind::i8 is sm_100a-only: no fallback
  emugemm_ctx *h = new (std::nothrow) emugemm_ctx();
  if (!h) return EMUGEMM_ERR_ARG;
  h->num_sms = prop.multiProcessorCount;
  void *fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) {
    delete h;
    return EMUGEMM_ERR_DEVICE;
  }
  h->encode = reinterpret_cast<PFN_cuTensorMapEncodeTiled_v12000>(fn);
  for (int i = 0; i < 4; ++i)
    if (cudaEventCreate(&h->ev[i]) != cudaSuccess) { delete h; return EMUGEMM_ERR_CUDA; }
  *out = h;
  return EMUGEMM_OK;
}

int emugemm_destroy(emugemm_handle_t h) {
  if (!h) return EMUGEMM_ERR_ARG;
  for (int i = 0; i < 4; ++i) if (h->ev[i]) cudaEventDestroy(h->ev[i]);
  delete h;
  return EMUGEMM_OK;
}

int emugemm_set_stream(emugemm_handle_t h, void *s) {
  if (!h) return EMUGEMM_ERR_ARG;
  h->stream = static_cast<cudaStream_t>(s);
  return EMUGEMM_OK;
}

// handle state: 7-bit digits are two's-complement fields (kDigitsTwos, R24) unless the sign-magnitude form (internal code 7,
// R1) was selected; 8 = balanced base 256 (R23)
int emugemm_set_slice_bits(emugemm_handle_t h, int bits) {
  if (!h || (bits != 7 && bits != 8)) return EMUGEMM_ERR_ARG;
  h->slice_bits = bits == 7 ? kDigitsTwos : 8;
  return EMUGEMM_OK;
}

int emugemm_set_slice_form(emugemm_handle_t h, int form) {
  if (!h || (form & ~1)) return EMUGEMM_ERR_ARG;
  if ((h->slice_bits & 0xFF) != 7) return form ? EMUGEMM_ERR_ARG : EMUGEMM_OK;  // the forms exist for 7-bit digits
  h->slice_bits = form ? 7 : kDigitsTwos;
  return EMUGEMM_OK;
}

int emugemm_set_oz2_fusion(emugemm_handle_t h, int on) {
  if (!h || (on & ~1)) return EMUGEMM_ERR_ARG;
  h->oz2_fusion = on;
  return EMUGEMM_OK;
}

int emugemm_set_workspace(emugemm_handle_t h, void *p, size_t bytes) {
  if (!h) return EMUGEMM_ERR_ARG;
  if (reinterpret_cast<uintptr_t>(p) & 1023) return EMUGEMM_ERR_ALIGNMENT;
  h->ws = p;
  h->ws_bytes = bytes;
  h->diag = nullptr;  // the diagnostics words lived in the previous workspace
  h->nf_flag = nullptr;
  return EMUGEMM_OK;
}

size_t emugemm_workspace_bytes(int scheme, int elem, int64_t m, int64_t n, int64_t k, int pn) {
  if (m < 0 || n < 0 || k < 0 || pn < 1) return 0;
  if (m == 0 || n == 0 || k == 0) return 1024;
  const int64_t kpad = round_up(k, kBlockK);
  size_t total = ws_common(m, n);
  if (scheme == EMUGEMM_OZ1) {
    if (pn > 8 || (elem != 4 && elem != 8)) return 0;
    total += granule(static_cast<size_t>(pn) * m * kpad) + granule(static_cast<size_t>(pn) * n * kpad);
    int64_t clen;
    // upper bound of the chunk count over both digit modes (the 8-bit mode has the shorter chunks), with room for the
    // balanced split where it may apply (few tiles: the partials are small)
    const int64_t tiles = oz1_cluster_tiles_host(pn, m, n);
    int nch = 1;
    for (int bits = 7; bits <= 8; ++bits) {
      const int nb = oz1_chunks(pn, bits, kpad, 0, &clen);
      const int ub = oz1_chunks_may_balance(nb, tiles) ? 2 * nb : nb;
      if (ub > nch) nch = ub;
    }
    if (nch > 1) total += granule(static_cast<size_t>(nch) * m * n * 16);
  } else if (scheme == EMUGEMM_OZ1_4M) {
    if (pn > 8 || elem != 16) return 0;
    const int64_t kk = 2 * kpad, mm = 2 * m;
    total += granule(4 * mm) + granule(static_cast<size_t>(pn) * mm * kk) + granule(static_cast<size_t>(pn) * n * kk) +
             granule(static_cast<size_t>(mm) * n * 8);
    int64_t clen;
    const int nch = oz1_chunks(pn, 8, kk, 0, &clen);
    if (nch > 1) total += granule(static_cast<size_t>(nch) * mm * n * 16);
  } else if (scheme == EMUGEMM_OZ2 || scheme == EMUGEMM_OZ2_3M) {
    if (pn > kMaxModuli) return 0;
    const size_t pi = scheme == EMUGEMM_OZ2_3M ? 3 : 1, po = scheme == EMUGEMM_OZ2_3M ? 2 : 1;
    total += granule(pi * pn * m * kpad) + granule(pi * pn * n * kpad) + oz2_cr_elems(static_cast<int>(po), pn, m, n, kpad);
  } else {
    return 0;
  }
  return total;
}

const char *emugemm_status_string(int s) {
  switch (s) {
    case EMUGEMM_OK: return "ok";
    case EMUGEMM_ERR_ARG: return "invalid argument";
    case EMUGEMM_ERR_ALIGNMENT: return "pointer not aligned";
    case EMUGEMM_ERR_WORKSPACE: return "workspace missing or too small";
    case EMUGEMM_ERR_PRECISION: return "k too large for this number of moduli";
    case EMUGEMM_ERR_DEVICE: return "no sm_100 CUDA device";
    case EMUGEMM_ERR_CUDA: return "CUDA error";
    case EMUGEMM_ERR_STATIC_LIMIT: return "problem exceeds the static scratch array (EMUGEMM_STATIC_WS_BYTES): use emugemm_dgemm_oz1 with a workspace";
    default: return "unknown status";
  }
}

int emugemm_last_cuda_error(emugemm_handle_t h) { return h ? h->last_cuda : 0; }

// Scheme I ZGEMM by 4M: one real Scheme I GEMM of size 2m x n x 2k on the real embedding
// A' = [[Re A, -Im A], [Im A, Re A]], B' = [[Re B], [Im B]], then the complex alpha / beta combination.
static int run_oz1_4m(emugemm_ctx *h, int elem, int64_t m, int64_t n, int64_t k, const double alpha[2], const void *A, int64_t lda,
                      const void *B, int64_t ldb, const double beta[2], void *C, int64_t ldc, int p) {
  if (!alpha || !beta) return EMUGEMM_ERR_ARG;
  EMU_TRY(check_gemm_args(h, 0, 0, m, n, k, A, lda, B, ldb, C, ldc));
  if (p < 1 || p > (elem == kC64 ? 4 : 8)) return EMUGEMM_ERR_ARG;
  h->launches = 0;
  if (m == 0 || n == 0) return mark_all(h);
  EMU_TRY(mark(h, 0));
  if (k == 0) {
    EMU_TRY(scale_c(h, m, n, beta[0], beta[1], C, ldc, elem));
    EMU_TRY(mark(h, 1)); EMU_TRY(mark(h, 2)); EMU_TRY(mark(h, 3));
    return EMUGEMM_OK;
  }
  const int64_t kpad = round_up(k, kBlockK), kk = 2 * kpad, mm = 2 * m;
  const int bits = h->slice_bits;
  int64_t clen;
  const int nch = oz1_chunks(p, bits, kk, 0, &clen);
  if (!h->ws || (reinterpret_cast<uintptr_t>(h->ws) & 1023)) return h->ws ? EMUGEMM_ERR_ALIGNMENT : EMUGEMM_ERR_WORKSPACE;
  Carver cv(h->ws, h->ws_bytes);
  auto *diag = cv.take<unsigned long long>(1);
  auto *mbB = cv.take<unsigned long long>(n);
  auto *eA = cv.take<int32_t>(mm);
  auto *eB = cv.take<int32_t>(n);
  auto *SA = cv.take<int8_t>(static_cast<size_t>(p) * mm * kk);
  auto *SB = cv.take<int8_t>(static_cast<size_t>(p) * n * kk);
  auto *T = cv.take<double>(static_cast<size_t>(mm) * n);
  double *part = nch > 1 ? cv.take<double>(static_cast<size_t>(nch) * mm * n * 2) : nullptr;
  if (!cv.ok) return EMUGEMM_ERR_WORKSPACE;
  h->diag = diag;
  h->nf_flag = diag + kDiagNonFinite;
  EMU_CUDA(h, cudaMemsetAsync(diag, 0, kDiagBytes, h->stream));
  EMU_TRY(launch_colmax(h, elem, n, k, B, ldb, mbB));
  EMU_TRY(launch_oz1_4m_slice(h, elem, 0, m, k, kpad, A, lda, nullptr, eA, p, bits, SA));
  EMU_TRY(launch_oz1_4m_slice(h, elem, 1, n, k, kpad, B, ldb, mbB, eB, p, bits, SB));
  EMU_TRY(mark(h, 1));
  EMU_TRY(oz1_gemm_phase(h, kF64, mm, n, kk, p, bits, SA, SB, eA, eB, 1.0, 0.0, T, n, nullptr, nch, clen, part, diag));
  const unsigned cgrid = static_cast<unsigned>((m * n + 255) / 256);
  if (elem == kC64)
    zcombine_4m_kernel<float><<<cgrid, 256, 0, h->stream>>>(m, n, T, alpha[0], alpha[1], beta[0], beta[1], static_cast<float *>(C), ldc);
  else
    zcombine_4m_kernel<double><<<cgrid, 256, 0, h->stream>>>(m, n, T, alpha[0], alpha[1], beta[0], beta[1], static_cast<double *>(C), ldc);
  h->launches++;
  EMU_CUDA(h, cudaGetLastError());
  EMU_TRY(mark(h, 3));
  return EMUGEMM_OK;
}

int emugemm_zgemm_oz1_4m(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, const double alpha[2], const double *A, int64_t lda,
                         const double *B, int64_t ldb, const double beta[2], double *C, int64_t ldc, int p) {
  return run_oz1_4m(h, kZ128, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, p);
}
// complex64 operands and result (CGEMM): alpha, beta stay HOST double pairs
int emugemm_cgemm_oz1_4m(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, const double alpha[2], const float *A, int64_t lda,
                         const float *B, int64_t ldb, const double beta[2], float *C, int64_t ldc, int p) {
  return run_oz1_4m(h, kC64, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, p);
}
int emugemm_cgemm_oz2_3m(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, const double alpha[2], const float *A, int64_t lda,
                         const float *B, int64_t ldb, const double beta[2], float *C, int64_t ldc, int n_moduli) {
  if (!alpha || !beta) return EMUGEMM_ERR_ARG;
  return run_oz2(h, 0, 0, 1, m, n, k, alpha, A, lda, B, ldb, beta, reinterpret_cast<double *>(C), ldc, n_moduli, 1);
}

int emugemm_dgemm_oz1_t(emugemm_handle_t h, int transa, int transb, int64_t m, int64_t n, int64_t k, double alpha,
                        const double *A, int64_t lda, const double *B, int64_t ldb, double beta, double *C, int64_t ldc, int p) {
  return run_oz1(h, transa, transb, kF64, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, p, nullptr, 0, nullptr);
}
int emugemm_sgemm_oz1_t(emugemm_handle_t h, int transa, int transb, int64_t m, int64_t n, int64_t k, float alpha,
                        const float *A, int64_t lda, const float *B, int64_t ldb, float beta, float *C, int64_t ldc, int p) {
  return run_oz1(h, transa, transb, kF32, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, p, nullptr, 0, nullptr);
}
int emugemm_dgemm_oz2_t(emugemm_handle_t h, int transa, int transb, int64_t m, int64_t n, int64_t k, double alpha,
                        const double *A, int64_t lda, const double *B, int64_t ldb, double beta, double *C, int64_t ldc,
                        int n_moduli) {
  const double al[2] = {alpha, 0.0}, be[2] = {beta, 0.0};
  return run_oz2(h, transa, transb, 0, m, n, k, al, A, lda, B, ldb, be, C, ldc, n_moduli);
}
int emugemm_sgemm_oz2_t(emugemm_handle_t h, int transa, int transb, int64_t m, int64_t n, int64_t k, float alpha,
                        const float *A, int64_t lda, const float *B, int64_t ldb, float beta, float *C, int64_t ldc,
                        int n_moduli) {
  const double al[2] = {alpha, 0.0}, be[2] = {beta, 0.0};
  return run_oz2(h, transa, transb, 0, m, n, k, al, A, lda, B, ldb, be, reinterpret_cast<double *>(C), ldc, n_moduli, 1);
}
int emugemm_sgemm_oz2(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, float alpha, const float *A, int64_t lda,
                      const float *B, int64_t ldb, float beta, float *C, int64_t ldc, int n_moduli) {
  return emugemm_sgemm_oz2_t(h, 0, 0, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, n_moduli);
}
int emugemm_zgemm_oz2_3m_t(emugemm_handle_t h, int transa, int transb, int64_t m, int64_t n, int64_t k, const double alpha[2],
                           const double *A, int64_t lda, const double *B, int64_t ldb, const double beta[2], double *C,
                           int64_t ldc, int n_moduli) {
  if (!alpha || !beta) return EMUGEMM_ERR_ARG;
  return run_oz2(h, transa, transb, 1, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, n_moduli);
}

int emugemm_dgemm_oz1(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, double alpha, const double *A, int64_t lda,
                      const double *B, int64_t ldb, double beta, double *C, int64_t ldc, int p) {
  return emugemm_dgemm_oz1_t(h, 0, 0, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, p);
}

int emugemm_sgemm_oz1(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, float alpha, const float *A, int64_t lda,
                      const float *B, int64_t ldb, float beta, float *C, int64_t ldc, int p) {
  return emugemm_sgemm_oz1_t(h, 0, 0, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, p);
}

int emugemm_dgemm_oz1_strided_batched(emugemm_handle_t h, int64_t batch, int64_t m, int64_t n, int64_t k, double alpha,
                                      const double *A, int64_t lda, int64_t strideA, const double *B, int64_t ldb,
                                      int64_t strideB, double beta, double *C, int64_t ldc, int64_t strideC, int p) {
  return run_oz1_batched(h, kF64, batch, m, n, k, alpha, A, lda, strideA, B, ldb, strideB, beta, C, ldc, strideC, p);
}
int emugemm_sgemm_oz1_strided_batched(emugemm_handle_t h, int64_t batch, int64_t m, int64_t n, int64_t k, float alpha,
                                      const float *A, int64_t lda, int64_t strideA, const float *B, int64_t ldb,
                                      int64_t strideB, float beta, float *C, int64_t ldc, int64_t strideC, int p) {
  return run_oz1_batched(h, kF32, batch, m, n, k, alpha, A, lda, strideA, B, ldb, strideB, beta, C, ldc, strideC, p);
}

int emugemm_dgemm_oz2_strided_batched(emugemm_handle_t h, int64_t batch, int64_t m, int64_t n, int64_t k, double alpha,
                                      const double *A, int64_t lda, int64_t strideA, const double *B, int64_t ldb,
                                      int64_t strideB, double beta, double *C, int64_t ldc, int64_t strideC, int n_moduli) {
  const double al[2] = {alpha, 0.0}, be[2] = {beta, 0.0};
  return run_oz2_batched(h, 0, 0, batch, m, n, k, al, A, lda, strideA, B, ldb, strideB, be, C, ldc, strideC, n_moduli);
}
int emugemm_sgemm_oz2_strided_batched(emugemm_handle_t h, int64_t batch, int64_t m, int64_t n, int64_t k, float alpha,
                                      const float *A, int64_t lda, int64_t strideA, const float *B, int64_t ldb,
                                      int64_t strideB, float beta, float *C, int64_t ldc, int64_t strideC, int n_moduli) {
  const double al[2] = {alpha, 0.0}, be[2] = {beta, 0.0};
  return run_oz2_batched(h, 0, 1, batch, m, n, k, al, A, lda, strideA, B, ldb, strideB, be, C, ldc, strideC, n_moduli);
}
int emugemm_zgemm_oz2_3m_strided_batched(emugemm_handle_t h, int64_t batch, int64_t m, int64_t n, int64_t k,
                                         const double alpha[2], const double *A, int64_t lda, int64_t strideA,
                                         const double *B, int64_t ldb, int64_t strideB, const double beta[2], double *C,
                                         int64_t ldc, int64_t strideC, int n_moduli) {
  if (!alpha || !beta) return EMUGEMM_ERR_ARG;
  return run_oz2_batched(h, 1, 0, batch, m, n, k, alpha, A, lda, strideA, B, ldb, strideB, beta, C, ldc, strideC, n_moduli);
}

int emugemm_dgemm_oz2(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, double alpha, const double *A, int64_t lda,
                      const double *B, int64_t ldb, double beta, double *C, int64_t ldc, int n_moduli) {
  return emugemm_dgemm_oz2_t(h, 0, 0, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, n_moduli);
}

int emugemm_zgemm_oz2_3m(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, const double alpha[2], const double *A,
                         int64_t lda, const double *B, int64_t ldb, const double beta[2], double *C, int64_t ldc,
                         int n_moduli) {
  return emugemm_zgemm_oz2_3m_t(h, 0, 0, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, n_moduli);
}

// ---- pre-decomposed operands ---------------------------------------------------
static int operand_planes(int scheme, int pn) { return scheme == EMUGEMM_OZ2_3M ? 3 * pn : pn; }

size_t emugemm_operand_bytes(int scheme, int64_t rows, int64_t k, int pn) {
  if (rows < 0 || k < 0 || pn < 1) return 0;
  if (scheme == EMUGEMM_OZ1 ? pn > 8 : (scheme == EMUGEMM_OZ2 || scheme == EMUGEMM_OZ2_3M) ? pn > kMaxModuli : true) return 0;
  const int64_t kpad = round_up(k, kBlockK);
  return granule(static_cast<size_t>(operand_planes(scheme, pn)) * rows * kpad) + granule(4 * static_cast<size_t>(rows)) + 1024;
}

int emugemm_decompose(emugemm_handle_t h, int scheme, int role, int trans, int elem, int64_t rows, int64_t k, const void *X,
                      int64_t ldx, int pn, void *dev_buf, size_t bytes, emugemm_operand_t *out) {
  if (!h || !out || !dev_buf || !X || rows <= 0 || k <= 0 || (role & ~1) || (trans & ~1)) return EMUGEMM_ERR_ARG;
  const bool oz1 = scheme == EMUGEMM_OZ1, oz2 = scheme == EMUGEMM_OZ2, z3m = scheme == EMUGEMM_OZ2_3M;
  if (!(oz1 || oz2 || z3m)) return EMUGEMM_ERR_ARG;
  if (oz1 ? !((elem == kF64 && pn >= 1 && pn <= 8) || (elem == kF32 && pn >= 1 && pn <= 4))
          : !((z3m ? elem == kZ128 : (elem == kF64 || elem == kF32)) && pn >= 2 && pn <= kMaxModuli))
    return EMUGEMM_ERR_ARG;
  const int by_cols = role == 0 ? trans : !trans;  // is k the strided dimension of the stored operand?
  if (ldx < (by_cols ? rows : k)) return EMUGEMM_ERR_ARG;
  if ((reinterpret_cast<uintptr_t>(X) & 15) || (reinterpret_cast<uintptr_t>(dev_buf) & 1023)) return EMUGEMM_ERR_ALIGNMENT;
  if (bytes < emugemm_operand_bytes(scheme, rows, k, pn)) return EMUGEMM_ERR_WORKSPACE;
  int t_bits = 0;
  if (!oz1) {
    int tA, tB;
    if (oz2_budget_host(pn, k, z3m, &tA, &tB) < 2) return EMUGEMM_ERR_PRECISION;
    t_bits = role == 0 ? tA : tB;
  }
  const int64_t kpad = round_up(k, kBlockK);
  Carver ob(dev_buf, bytes);
  auto *planes = ob.take<int8_t>(static_cast<size_t>(operand_planes(scheme, pn)) * rows * kpad);
  auto *e = ob.take<int32_t>(rows);
  unsigned long long *mb = nullptr;
  if (by_cols) {  // column maxima scratch comes from the handle's workspace
    if (!h->ws || (reinterpret_cast<uintptr_t>(h->ws) & 1023)) return h->ws ? EMUGEMM_ERR_ALIGNMENT : EMUGEMM_ERR_WORKSPACE;
    Carver cv(h->ws, h->ws_bytes);
    mb = cv.take<unsigned long long>(rows);
    if (!cv.ok) return EMUGEMM_ERR_WORKSPACE;
  }
  h->launches = 0;
  h->nf_flag = nullptr;  // the flag belongs to the one-shot calls (it lives in their workspace)
  if (oz1) EMU_TRY(launch_oz1_slice(h, elem, by_cols, rows, k, kpad, X, ldx, mb, e, pn, h->slice_bits, planes));
  else EMU_TRY(launch_oz2_residues(h, elem, by_cols, rows, k, kpad, X, ldx, mb, e, pn, t_bits, planes));
  out->scheme = scheme; out->role = role; out->elem = elem; out->pn = pn;
  out->slice_bits = oz1 ? h->slice_bits : 0; out->t_bits = t_bits;
  out->rows = rows; out->k = k; out->kpad = kpad; out->buf = dev_buf; out->bytes = bytes;
  return EMUGEMM_OK;
}

int emugemm_gemm_pre(emugemm_handle_t h, const emugemm_operand_t *A, const emugemm_operand_t *B, const double alpha[2],
                     const double beta[2], void *C, int64_t ldc) {
  if (!h || !A || !B || !alpha || !beta || !C) return EMUGEMM_ERR_ARG;
  if (A->role != 0 || B->role != 1 || A->scheme != B->scheme || A->elem != B->elem || A->pn != B->pn || A->k != B->k ||
      A->slice_bits != B->slice_bits || !A->buf || !B->buf || ldc < B->rows)
    return EMUGEMM_ERR_ARG;
  if (reinterpret_cast<uintptr_t>(C) & 15) return EMUGEMM_ERR_ALIGNMENT;
  const int64_t m = A->rows, n = B->rows, kpad = A->kpad;
  const int scheme = A->scheme, pn = A->pn, planes = operand_planes(scheme, pn);
  const int8_t *PA = static_cast<const int8_t *>(A->buf), *PB = static_cast<const int8_t *>(B->buf);
  const int32_t *eA = reinterpret_cast<const int32_t *>(PA + granule(static_cast<size_t>(planes) * m * kpad));
  const int32_t *eB = reinterpret_cast<const int32_t *>(PB + granule(static_cast<size_t>(planes) * n * kpad));
  if (!h->ws || (reinterpret_cast<uintptr_t>(h->ws) & 1023)) return h->ws ? EMUGEMM_ERR_ALIGNMENT : EMUGEMM_ERR_WORKSPACE;
  h->launches = 0;
  Carver cv(h->ws, h->ws_bytes);
  auto *diag = cv.take<unsigned long long>(1);
  EMU_TRY(mark(h, 0));
  EMU_TRY(mark(h, 1));
  if (scheme == EMUGEMM_OZ1) {
    int64_t clen;
    const int nch = oz1_chunks_balanced(pn, A->slice_bits, kpad, m, n, h->num_sms, &clen);  // as the one-shot call
    double *part = nch > 1 ? cv.take<double>(static_cast<size_t>(nch) * m * n * 2) : nullptr;
    if (!cv.ok) return EMUGEMM_ERR_WORKSPACE;
    h->diag = diag;
  h->nf_flag = diag + kDiagNonFinite;
    EMU_CUDA(h, cudaMemsetAsync(diag, 0, kDiagBytes, h->stream));
    return oz1_gemm_phase(h, A->elem, m, n, kpad, pn, A->slice_bits, PA, PB, eA, eB, alpha[0], beta[0], C, ldc, nullptr, nch,
                          clen, part, diag);
  }
  const int is3m = scheme == EMUGEMM_OZ2_3M;
  auto *CR = cv.take<int8_t>(oz2_cr_elems(is3m ? 2 : 1, pn, m, n, kpad));
  if (!cv.ok) return EMUGEMM_ERR_WORKSPACE;
  h->diag = diag;
  h->nf_flag = diag + kDiagNonFinite;
  EMU_CUDA(h, cudaMemsetAsync(diag, 0, kDiagBytes, h->stream));
  return oz2_gemm_phase(h, is3m, m, n, kpad, pn, PA, PB, CR, eA, eB, A->t_bits, B->t_bits, alpha, beta, static_cast<double *>(C),
                        ldc, diag, A->elem == kF32);
}

int emugemm_last_gemm_cycles(emugemm_handle_t h, unsigned long long *cycles) {
  if (!h || !cycles) return EMUGEMM_ERR_ARG;
  if (!h->diag) return EMUGEMM_ERR_WORKSPACE;
  EMU_CUDA(h, cudaStreamSynchronize(h->stream));
  EMU_CUDA(h, cudaMemcpy(cycles, h->diag, sizeof(unsigned long long), cudaMemcpyDeviceToHost));
  return EMUGEMM_OK;
}

int emugemm_nonfinite_seen(emugemm_handle_t h, int *seen) {
  if (!h || !seen) return EMUGEMM_ERR_ARG;
  if (!h->diag) return EMUGEMM_ERR_WORKSPACE;
  unsigned long long v = 0;
  EMU_CUDA(h, cudaStreamSynchronize(h->stream));
  EMU_CUDA(h, cudaMemcpy(&v, h->diag + kDiagNonFinite, sizeof(v), cudaMemcpyDeviceToHost));
  *seen = v != 0;
  return EMUGEMM_OK;
}

int emugemm_enable_stage_timing(emugemm_handle_t h, int on) {
  if (!h) return EMUGEMM_ERR_ARG;
  h->timing = on ? 1 : 0;
  return EMUGEMM_OK;
}

int emugemm_stage_ms(emugemm_handle_t h, float ms[3], int *launches) {
  if (!h || !ms) return EMUGEMM_ERR_ARG;
  if (!h->timing) return EMUGEMM_ERR_ARG;
  EMU_CUDA(h, cudaEventSynchronize(h->ev[3]));
  for (int i = 0; i < 3; ++i) EMU_CUDA(h, cudaEventElapsedTime(&ms[i], h->ev[i], h->ev[i + 1]));
  if (launches) *launches = h->launches;
  return EMUGEMM_OK;
}

// ---- test hooks --------------------------------------------------------------
static int unpad_planes(emugemm_ctx *h, int8_t *dst, const int8_t *src, int64_t planes_rows, int64_t k, int64_t kpad) {
  EMU_CUDA(h, cudaMemcpy2DAsync(dst, k, src, kpad, k, planes_rows, cudaMemcpyDeviceToDevice, h->stream));
  return EMUGEMM_OK;
}

int emugemm_dbg_exponents(emugemm_handle_t h, int elem, int by_cols, int64_t rows, int64_t k, const void *X, int64_t ldx,
                          int32_t *e_out) {
  if (!h || rows < 0 || k < 0 || !e_out) return EMUGEMM_ERR_ARG;
  if (!h->ws) return EMUGEMM_ERR_WORKSPACE;
  h->nf_flag = nullptr;  // the hooks carve the workspace from its start: no diagnostics words
  Carver cv(h->ws, h->ws_bytes);
  auto *mb = cv.take<unsigned long long>(rows);
  if (!cv.ok) return EMUGEMM_ERR_WORKSPACE;
  return launch_exponent_scan(h, elem, by_cols, rows, k, X, ldx, mb, e_out);
}

int emugemm_dbg_oz1_slices(emugemm_handle_t h, int elem, int by_cols, int64_t rows, int64_t k, const void *X, int64_t ldx,
                           int p, int8_t *out, int32_t *e_out) {
  if (!h || rows <= 0 || k <= 0 || !out || !e_out || p < 1 || p > 8) return EMUGEMM_ERR_ARG;
  if (!h->ws) return EMUGEMM_ERR_WORKSPACE;
  const int64_t kpad = round_up(k, kBlockK);
  h->nf_flag = nullptr;  // the hooks carve the workspace from its start: no diagnostics words
  Carver cv(h->ws, h->ws_bytes);
  auto *mb = cv.take<unsigned long long>(rows);
  auto *S = cv.take<int8_t>(static_cast<size_t>(p) * rows * kpad);
  if (!cv.ok) return EMUGEMM_ERR_WORKSPACE;
  EMU_TRY(launch_oz1_slice(h, elem, by_cols, rows, k, kpad, X, ldx, mb, e_out, p, h->slice_bits, S));
  return unpad_planes(h, out, S, static_cast<int64_t>(p) * rows, k, kpad);
}

int emugemm_dbg_oz1_accumulators(emugemm_handle_t h, int elem, int64_t m, int64_t n, int64_t k, const void *A, int64_t lda,
                                 const void *B, int64_t ldb, int p, int64_t chunk_k, int32_t *out, int *n_chunks_out) {
  if (!out) return EMUGEMM_ERR_ARG;
  return run_oz1(h, 0, 0, elem, m, n, k, 1.0, A, lda, B, ldb, 0.0, nullptr, n, p, out, chunk_k, n_chunks_out);
}

int emugemm_dbg_oz2_residues(emugemm_handle_t h, int elem, int by_cols, int64_t rows, int64_t k, const void *X, int64_t ldx,
                             int n_moduli, int t_bits, int8_t *out, int32_t *e_out) {
  if (!h || rows <= 0 || k <= 0 || !out || !e_out || n_moduli < 1 || n_moduli > kMaxModuli) return EMUGEMM_ERR_ARG;
  if (!h->ws) return EMUGEMM_ERR_WORKSPACE;
  const int64_t kpad = round_up(k, kBlockK);
  const int parts = (elem == kZ128) ? 3 : 1;
  h->nf_flag = nullptr;  // the hooks carve the workspace from its start: no diagnostics words
  Carver cv(h->ws, h->ws_bytes);
  auto *mb = cv.take<unsigned long long>(rows);
  auto *R = cv.take<int8_t>(static_cast<size_t>(parts) * n_moduli * rows * kpad);
  if (!cv.ok) return EMUGEMM_ERR_WORKSPACE;
  EMU_TRY(launch_oz2_residues(h, elem, by_cols, rows, k, kpad, X, ldx, mb, e_out, n_moduli, t_bits, R));
  return unpad_planes(h, out, R, static_cast<int64_t>(parts) * n_moduli * rows, k, kpad);
}

int emugemm_dbg_oz2_modgemm(emugemm_handle_t h, int is3m, int64_t m, int64_t n, int64_t k, int n_moduli, const int8_t *RA,
                            const int8_t *RB, int8_t *out) {
  if (!h || m <= 0 || n <= 0 || k <= 0 || !RA || !RB || !out || n_moduli < 1 || n_moduli > kMaxModuli) return EMUGEMM_ERR_ARG;
  if (!h->ws) return EMUGEMM_ERR_WORKSPACE;
  const int64_t kpad = round_up(k, kBlockK);
  const int parts = is3m ? 3 : 1;
  Oz2GemmArgs g;
  g.m = m; g.n = n; g.kpad = kpad; g.n_moduli = n_moduli; g.is3m = is3m; g.CR = out; g.cycles = nullptr;
  if (kpad == k) {
    g.RA = RA; g.RB = RB;
  } else {  // canonical planes are unpadded: stage zero-padded copies in the workspace
    Carver cv(h->ws, h->ws_bytes);
    auto *PA = cv.take<int8_t>(static_cast<size_t>(parts) * n_moduli * m * kpad);
    auto *PB = cv.take<int8_t>(static_cast<size_t>(parts) * n_moduli * n * kpad);
    if (!cv.ok) return EMUGEMM_ERR_WORKSPACE;
    EMU_CUDA(h, cudaMemsetAsync(PA, 0, static_cast<size_t>(parts) * n_moduli * m * kpad, h->stream));
    EMU_CUDA(h, cudaMemsetAsync(PB, 0, static_cast<size_t>(parts) * n_moduli * n * kpad, h->stream));
    EMU_CUDA(h, cudaMemcpy2DAsync(PA, kpad, RA, k, k, static_cast<size_t>(parts) * n_moduli * m, cudaMemcpyDeviceToDevice, h->stream));
    EMU_CUDA(h, cudaMemcpy2DAsync(PB, kpad, RB, k, k, static_cast<size_t>(parts) * n_moduli * n, cudaMemcpyDeviceToDevice, h->stream));
    g.RA = PA; g.RB = PB;
  }
  return launch_oz2_gemm(h, g);
}

int emugemm_dbg_oz2_crt(emugemm_handle_t h, int64_t m, int64_t n, int n_moduli, const int8_t *CR, const int32_t *eA,
                        const int32_t *eB, int tA, int tB, double alpha, double beta, double *C, int64_t ldc) {
  if (!h || m <= 0 || n <= 0 || !CR || !eA || !eB || !C || n_moduli < 2 || n_moduli > kMaxModuli) return EMUGEMM_ERR_ARG;
  Oz2CrtArgs c;
  c.m = m; c.n = n; c.n_moduli = n_moduli; c.CR = CR; c.eA = eA; c.eB = eB; c.tA = tA; c.tB = tB; c.is_complex = 0;
  c.alpha[0] = alpha; c.alpha[1] = 0; c.beta[0] = beta; c.beta[1] = 0; c.C = C; c.ldc = ldc;
  return launch_oz2_crt(h, c);
}

int emugemm_oz2_budget(int n_moduli, int64_t k, int is3m, int *tA, int *tB) {
  int a = 0, b = 0;
  const int T = oz2_budget_host(n_moduli, k, is3m, &a, &b);
  if (tA) *tA = a;
  if (tB) *tB = b;
  return T;
}

int emugemm_dbg_crt_constants(int n_moduli, int *n_pairs, int *n_digits, int *digit_bits, long long *digits, unsigned *pair) {
  if (!n_pairs || !n_digits || !digit_bits || !digits || !pair) return EMUGEMM_ERR_ARG;
  return crt_constants_dump(n_moduli, n_pairs, n_digits, digit_bits, digits, pair) ? EMUGEMM_ERR_ARG : EMUGEMM_OK;
}

int64_t emugemm_oz1_chunk_k(int p) { return (p >= 1 && p <= 8) ? oz1_chunk_k_host(p, kDigitsTwos) : 0; }  // default digit form
int64_t emugemm_oz1_chunk_k_bits(int p, int code) {  // public codes: 7 (default form), 8, EMUGEMM_DIGITS_SIGN_MAGNITUDE
  const int internal = code == 7 ? kDigitsTwos : code == 8 ? 8 : code == EMUGEMM_DIGITS_SIGN_MAGNITUDE ? 7 : 0;
  return (p >= 1 && p <= 8 && internal) ? oz1_chunk_k_host(p, internal) : 0;
}

#ifdef EMUGEMM_PROBES
int emugemm_dbg_i8_probe(emugemm_handle_t h, int n_ops, const int *ops, int iters, float *ms, int *ctas,
                         long long *cycles) {
  if (!h || !ms || !ctas) return EMUGEMM_ERR_ARG;
  return launch_i8_probe(h, n_ops, ops, iters, ms, ctas, cycles);
}

int emugemm_dbg_oz1_issue_probe(emugemm_handle_t h, int p, int use_collector, int iters, float *ms, int *ctas,
                                 long long *cycles) {
  if (!h || !ms || !ctas) return EMUGEMM_ERR_ARG;
  return launch_oz1_issue_probe(h, p, use_collector, iters, ms, ctas, cycles);
}

int emugemm_dbg_set_flags(emugemm_handle_t h, int flags) {
  if (!h) return EMUGEMM_ERR_ARG;
  h->dbg_flags = flags;
  return EMUGEMM_OK;
}

#endif  // EMUGEMM_PROBES

#pragma GCC visibility pop
}  // extern "C"
