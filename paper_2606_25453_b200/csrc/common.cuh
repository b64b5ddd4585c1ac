// common.cuh -- host-side context, error handling, TMA descriptor encoding and
// the internal interfaces between the stage drivers (pre-pass, fused GEMMs, CRT).
#pragma once
#include <cuda.h>
#include <cudaTypedefs.h>
#include <cuda_runtime.h>
#include <cstddef>
#include <cstdint>

#include "../../include/emugemm.h"

namespace emu {

constexpr int kBeta = 7;          // bits per signed slice (R1)
constexpr int kMaxModuli = 20;    // API range of n_moduli
// Scheme I digit formats as carried in slice_bits: 7 = sign-magnitude (R1), 8 = balanced base 256 (R23), kDigitsTwos = 7-bit
// two's-complement fields (R24): low byte = bits per slice, bit 8 = the form
constexpr int kDigitsTwos = 0x107;
constexpr int kTileM = 128;       // rows per CTA tile == tcgen05.mma M (PAPER.md:43 t_M = 128 on Blackwell)
constexpr int kBlockK = 128;      // bytes of k per pipeline block (one 128B swizzle row, 4 MMAs of K = 32)
// diagnostics words at the head of the workspace (zeroed per call): [0] SM cycles of the fused GEMM kernel (CTA 0),
// [1] wave-barrier counter of the fused Scheme I kernel, [2] non-finite-input flag raised by the pre-pass
constexpr int kDiagBytes = 64;
constexpr int kDiagWaveCtr = 1, kDiagNonFinite = 2;

struct StageTimer;

// Timing-experiment switches (emugemm_dbg_set_flags) and the tensor-pipe probe kernels exist only in the PROBES build
// (libemugemm_probes.so, -DEMUGEMM_PROBES, loaded by `bench.py` for its probe leg): the shipped library carries neither
// the flag tests in its hot loops nor an entry point that can make results wrong.
#ifdef EMUGEMM_PROBES
#define EMU_PROBE_FLAG(flags, bit) ((flags) & (bit))
#else
#define EMU_PROBE_FLAG(flags, bit) 0
#endif

}  // namespace emu

struct emugemm_ctx {
  cudaStream_t stream = nullptr;
  void *ws = nullptr;
  size_t ws_bytes = 0;
  int last_cuda = 0;
  int num_sms = 0;
  int timing = 0;
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
  int launches = 0;
  int dbg_flags = 0;
  int slice_bits = emu::kDigitsTwos;  // Scheme I digits: kDigitsTwos = 7-bit two's-complement fields (R24, default), 7 = 7-bit sign-magnitude (R1), 8 = balanced base 256 (R23)
  int oz2_fusion = 0;  // Scheme II real DGEMM: 1 = fused reconstruction when it applies (emugemm_set_oz2_fusion), 0 = separate CRT kernel
                       // (default: measured 8192^3 N = 16: 8.9 ms fused against 5.3 + 0.6 ms)
  unsigned long long *diag = nullptr;  // device: [0] = GEMM-kernel SM cycles of the last call (inside the workspace)
  unsigned long long *nf_flag = nullptr;  // device word the pre-pass ORs 1 into when an operand holds Inf / NaN (null: off)
  PFN_cuTensorMapEncodeTiled_v12000 encode = nullptr;
};

namespace emu {

#define EMU_CUDA(ctx, call)                     \
  do {                                          \
    cudaError_t _e = (call);                    \
    if (_e != cudaSuccess) {                    \
      (ctx)->last_cuda = static_cast<int>(_e);  \
      return EMUGEMM_ERR_CUDA;                  \
    }                                           \
  } while (0)

#define EMU_TRY(expr)            \
  do {                           \
    int _s = (expr);             \
    if (_s != EMUGEMM_OK) return _s; \
  } while (0)

inline int64_t round_up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }

// int8 tensor [planes][rows][kpad] (k contiguous), box {kBlockK, box_rows, box_planes},
// 128-byte swizzle, out-of-bounds rows / planes read as zero.
int encode_planes_tmap(emugemm_ctx *ctx, CUtensorMap *tm, const void *base, int64_t kpad, int64_t rows,
                       int64_t planes, int box_rows, int box_planes);

// ---- stage drivers (all asynchronous on ctx->stream) ------------------------
enum ElemKind { kF32 = 4, kF64 = 8, kZ128 = 16, kC64 = 64 /* complex64: internal id, not a byte count */ };

// Max-|x| bit pattern per row (by_cols = 0) or column (by_cols = 1) -> frexp exponent e_out[rows];
// maxbits is a rows x u64 scratch (zeroed inside).  For kZ128 the exponent covers re and im.
int launch_exponent_scan(emugemm_ctx *ctx, int elem, int by_cols, int64_t rows, int64_t k, const void *X,
                         int64_t ldx, unsigned long long *maxbits, int32_t *e_out);

// Column maxima (|x| bit patterns) of X (k x rows): the input of the by_cols = 1 plane kernels.
// batch > 1 (strided batched calls): entry b of X starts b * xstride elements further, its maxima are
// maxbits[b rows .. (b + 1) rows).
int launch_colmax(emugemm_ctx *ctx, int elem, int64_t rows, int64_t k, const void *X, int64_t ldx,
                  unsigned long long *maxbits, int batch = 1, int64_t xstride = 0);

// Scheme I slicing: out[p][rows][kpad] int8 (zero padded to kpad) AND the exponents e[rows] (output).
// by_cols = 0: one kernel scans each row and slices it (maxbits unused); by_cols = 1: maxbits is a scratch of
// batch * rows words: launch_colmax fills it, the column kernel derives and publishes the exponents and slices.
int launch_oz1_slice(emugemm_ctx *ctx, int elem, int by_cols, int64_t rows, int64_t k, int64_t kpad,
                     const void *X, int64_t ldx, unsigned long long *maxbits, int32_t *e, int p, int slice_bits,
                     int8_t *out, int batch = 1, int64_t xstride = 0);  // batch: out[p][batch rows][kpad], e[batch rows]

// Scheme II residues: elem 8: out[N][rows][kpad]; elem 16: out[3][N][rows][kpad] (re, im, Sigma); e as above.
int launch_oz2_residues(emugemm_ctx *ctx, int elem, int by_cols, int64_t rows, int64_t k, int64_t kpad,
                        const void *X, int64_t ldx, unsigned long long *maxbits, int32_t *e, int n_moduli,
                        int t_bits, int8_t *out, int batch = 1, int64_t xstride = 0);

// Scheme I complex by 4M: digit planes of the real embedding (prepass.cu) and the final complex combination.
int launch_oz1_4m_slice(emugemm_ctx *ctx, int elem /* kZ128 or kC64 */, int is_b, int64_t rows, int64_t k, int64_t kpad, const void *X, int64_t ldx,
                        const unsigned long long *maxbits, int32_t *e, int p, int slice_bits, int8_t *out);

struct Oz1GemmArgs {
  int64_t m, n, kpad;          // kpad: padded k of the slice planes (multiple of kBlockK)
  int64_t k0, k1;              // k range [k0, k1) handled by this launch (multiples of kBlockK)
  int n_chunks;                // > 1: the range is cut into overflow-safe chunks of chunk_k, one output per chunk
  int64_t chunk_k, chunk_stride;  // chunk length (multiple of kBlockK), bytes between the chunks' outputs
  int p;
  int slice_bits;              // 7 or 8 (weights 2^(bits (p-1-s)), scaling 2^(eA + eB - bits (p+1) [+ 4 guard bits]))
  const int8_t *SA, *SB;       // [p][m][kpad], [p][n][kpad]
  const int32_t *eA, *eB;
  int batch = 1;               // strided batched call: planes / exponents hold batch * m (n) rows, entry-major
  int64_t batch_stride_c = 0;  // bytes between the C matrices of consecutive entries
  int out_kind;                // 0: final FP64 C, 1: final FP32 C, 2: INT32 dump [p][m][n], 3: double-double partial [m][n][2]
  double alpha, beta;
  void *C;
  int64_t ldc;
  unsigned long long *cycles;  // device counter: += SM cycles CTA 0 spent in the kernel (diagnostic), may be null
  unsigned long long *wave_ctr = nullptr;  // zeroed device word for the wave barrier (null: no barrier)
};
int launch_oz1_gemm(emugemm_ctx *ctx, const Oz1GemmArgs &a);
// Sum n_chunks double-double partials part[c][m][n][2] and apply alpha/beta (out_kind 0 / 1 as above).
int launch_oz1_chunk_reduce(emugemm_ctx *ctx, int64_t m, int64_t n, int n_chunks, const double *part,
                            int out_kind, double alpha, double beta, void *C, int64_t ldc);

struct Oz2CrtArgs;
struct Oz2GemmArgs {
  int64_t m, n, kpad;
  int n_moduli;
  int is3m;
  const int8_t *RA, *RB;       // real: [N][rows][kpad]; 3M: [3][N][rows][kpad]
  int8_t *CR;                  // real: [N][m][n]; 3M: [2][N][m][n]
  unsigned long long *cycles;  // as in Oz1GemmArgs
  unsigned long long *wave_ctr = nullptr;  // as in Oz1GemmArgs
  int batch = 1;               // strided batched call: residue planes hold batch * m (n) rows entry-major, CR is [N][batch][m][n]
  int64_t k0 = 0, k1 = 0;      // k range [k0, k1) of this launch (multiples of kBlockK); k1 == 0: the whole kpad
  // Fused reconstruction (real product only): non-null = the kernel runs the CRT itself and writes C;
  // CR is then a scratch of scratch_bytes >= (CTAs launched) * N * 32 KB instead of the [N][m][n] planes.
  const Oz2CrtArgs *fused = nullptr;
  size_t scratch_bytes = 0;
};
int launch_oz2_gemm(emugemm_ctx *ctx, const Oz2GemmArgs &a);
// Longest k one launch may cover: INT32 accumulators of symmetric INT8 residues, k 128^2 < 2^31 (R7), in k-blocks
constexpr int64_t kOz2MaxChunkK = (131071 / kBlockK) * kBlockK;  // 130,944
// CR[plane][i] = sym((CR[plane][i] + T[plane][i]) mod m_(plane mod N)) for `planes` planes of `plane_elems` residues each:
// adds the output residues of one more k-chunk (Scheme II k-chunking: residues of chunks add modulo m_l)
int launch_oz2_residue_add(emugemm_ctx *ctx, int8_t *CR, const int8_t *T, int n_moduli, int planes, int64_t plane_elems);

struct Oz2CrtArgs {
  int64_t m, n;
  int n_moduli;
  const int8_t *CR;            // [N][m][n] (3M: second part at CR + N*m*n)
  const int32_t *eA, *eB;
  int tA, tB;
  int is_complex = 0;          // 0: real alpha/beta; 1: complex, C is (re, im) pairs
  int out_f32 = 0;               // C holds float (real: SGEMM) or float pairs (complex: CGEMM)
  double alpha[2], beta[2];
  double *C;
  int64_t ldc;
  int batch = 1;               // CR [N][batch][m][n], eA [batch m], eB [batch n], C_b = C + b * batch_stride_c elements
  int64_t batch_stride_c = 0;
};
int launch_oz2_crt(emugemm_ctx *ctx, const Oz2CrtArgs &a);
int crt_constants_dump(int N, int *NP, int *J, int *g, long long *digits, unsigned *pair);  // host only (test hook)

#ifdef EMUGEMM_PROBES
int launch_oz1_issue_probe(emugemm_ctx *ctx, int p, int coll, int iters, float *ms, int *ctas, long long *cycles);
int launch_i8_probe(emugemm_ctx *ctx, int n_ops, const int *ops, int iters, float *ms, int *ctas, long long *cycles);
#endif

// host helpers shared by api.cu and the drivers
int oz2_moduli_host(int n, int *mod);                  // greedy coprime list, descending from 256
int oz2_budget_host(int n, int64_t k, int is3m, int *tA, int *tB);
int64_t oz1_chunk_k_host(int p, int slice_bits = kDigitsTwos);
// Work items (cluster tiles) of one k-chunk of the fused Scheme I kernel for an m x n output with p slices; the
// kernel runs num_sms / 2 workers (CTA pairs) for every p (gemm_oz1.cu)
int64_t oz1_cluster_tiles_host(int p, int64_t m, int64_t n);

}  // namespace emu
