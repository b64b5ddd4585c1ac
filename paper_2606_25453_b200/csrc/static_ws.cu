// static_ws.cu -- emugemm_dgemm_oz1_static: the Scheme I DGEMM for callers that cannot allocate.
//
// Every other entry point takes its scratch (digit planes, exponents, diagnostics words) from the workspace the caller
// allocated and registered with emugemm_set_workspace.  Code under CUDA graph capture, tight serving loops and harnesses
// that forbid cudaMalloc have no such buffer: this entry point carves the SAME workspace layout out of a file-scope
// device array of kStaticWsBytes that the library image carries (every GPU that loads the library holds it until the
// process exits) and then runs the unchanged Scheme I call sequence (pre-pass kernels -> fused tcgen05 GEMM kernel).
// It calls no cudaMalloc / cudaFree and no allocating library routine.
//
// The array's name is a host-side stand-in in host code, NOT a device address: its device address is taken once per
// device, with that device current, by cudaGetSymbolAddress (return code checked) and that pointer is what the kernels
// get.
#include <mutex>

#include "common.cuh"

namespace emu {

constexpr size_t kStaticWsBytes = EMUGEMM_STATIC_WS_BYTES;  // usable bytes (include/emugemm.h)
constexpr int kStaticMaxDevices = 64;

// + 1024: the workspace layout wants 1024-byte granules and the array is only promised 256-byte alignment
static __device__ __align__(256) unsigned char g_static_ws[kStaticWsBytes + 1024];

static std::mutex g_static_mu;
static void *g_static_ptr[kStaticMaxDevices];  // device address of g_static_ws rounded up to 1024, per device ordinal

// Device address of the static scratch on the CURRENT device (set-up on first use per device; no allocation).
static int static_ws_ptr(emugemm_ctx *h, void **out) {
  int dev = -1;
  EMU_CUDA(h, cudaGetDevice(&dev));
  if (dev < 0 || dev >= kStaticMaxDevices) return EMUGEMM_ERR_DEVICE;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_ptr[dev]) {
    void *p = nullptr;
    EMU_CUDA(h, cudaGetSymbolAddress(&p, g_static_ws));
    if (!p) return EMUGEMM_ERR_DEVICE;
    const uintptr_t a = (reinterpret_cast<uintptr_t>(p) + 1023) & ~static_cast<uintptr_t>(1023);
    g_static_ptr[dev] = reinterpret_cast<void *>(a);
  }
  *out = g_static_ptr[dev];
  return EMUGEMM_OK;
}

}  // namespace emu

extern "C" {
#pragma GCC visibility push(default)

size_t emugemm_static_workspace_limit(void) { return emu::kStaticWsBytes; }

int emugemm_dgemm_oz1_static(emugemm_handle_t h, int64_t m, int64_t n, int64_t k, double alpha, const double *A, int64_t lda,
                             const double *B, int64_t ldb, double beta, double *C, int64_t ldc, int p) {
  if (!h) return EMUGEMM_ERR_ARG;
  if (m < 0 || n < 0 || k < 0 || p < 1 || p > 8) return EMUGEMM_ERR_ARG;
  // the size check comes first: a problem beyond the static array is refused before anything is enqueued
  const size_t need = emugemm_workspace_bytes(1 /* Scheme I */, 8 /* double */, m, n, k, p);
  if (need == 0) return EMUGEMM_ERR_ARG;
  if (need > emu::kStaticWsBytes) return EMUGEMM_ERR_STATIC_LIMIT;
  void *ws = nullptr;
  EMU_TRY(emu::static_ws_ptr(h, &ws));
  // The handle's own workspace registration is left as the caller set it: the static array is lent to the handle for
  // this call only.  The call sequence zeroes the words that must start at zero (wave-barrier counter, non-finite
  // flag, cycle counter: one cudaMemsetAsync on the handle's stream) and rewrites every plane byte it reads, so the
  // previous call's contents never leak into this one.
  void *const user_ws = h->ws;
  const size_t user_bytes = h->ws_bytes;
  h->ws = ws;
  h->ws_bytes = emu::kStaticWsBytes;
  const int st = emugemm_dgemm_oz1(h, m, n, k, alpha, A, lda, B, ldb, beta, C, ldc, p);
  h->ws = user_ws;
  h->ws_bytes = user_bytes;
  // h->diag / h->nf_flag keep pointing into the static array: emugemm_nonfinite_seen and emugemm_last_gemm_cycles
  // report on THIS call until the next compute call or emugemm_set_workspace replaces them
  return st;
}

#pragma GCC visibility pop
}
