// encode_static.cu -- hypic_segment_encode_static: segment encode (Eq. 8) for callers that cannot
// allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// hypic_segment_encode needs a caller-supplied workspace (chunk tables, the in-call fallback list and, for the per-channel
// gate, the prep records).  This variant keeps that scratch in a file-scope device array of this translation unit, of a
// stated, modest maximum size (kStaticScratchBytes = 4 MiB); every GPU that loads the library holds it until exit.  The
// caller passes inputs and outputs only; the call allocates nothing (no cudaMalloc / cudaFree / allocating library
// routine anywhere on its path -- the kernels below it never allocated either) and rejects problems whose workspace would
// not fit with HYPIC_ERR_STATIC_SCRATCH.
//
// The array is shared by every call on the device and keeps the last call's contents: what must start at zero (the
// fallback-list count and flags) is cleared by the call's own first kernel (chunk_offsets_kernel), every other table is
// written before it is read.  Two calls that overlap on the GPU (different streams, or different host threads without
// ordering between their streams) race on the array; calls on one stream are ordered and safe.
#include <mutex>

#include "common.cuh"

namespace hypic {
namespace {

constexpr size_t kStaticScratchBytes = 4u << 20;

// In host code this name is a host-side stand-in, not a device address: only cudaGetSymbolAddress gives the pointer a
// kernel may be handed.
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

constexpr int kMaxDevices = 64;
std::mutex g_static_mutex;
void* g_static_ptr[kMaxDevices] = {};  // per device ordinal; looked up once, with that device current

// the device address of the array on the CURRENT device (set-up once per device); returns a hypic status
int static_scratch_ptr(void** out) {
  int dev = 0;
  HYPIC_CUDA_OK(cudaGetDevice(&dev));
  if (dev >= 0 && dev < kMaxDevices) {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
      void* p = nullptr;
      HYPIC_CUDA_OK(cudaGetSymbolAddress(&p, g_static_scratch));
      g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return HYPIC_OK;
  }
  void* p = nullptr;  // beyond the cached ordinals: ask every time
  HYPIC_CUDA_OK(cudaGetSymbolAddress(&p, g_static_scratch));
  *out = p;
  return HYPIC_OK;
}

}  // namespace
}  // namespace hypic

using namespace hypic;

extern "C" {

size_t hypic_static_scratch_bytes(void) { return kStaticScratchBytes; }

int hypic_segment_encode_static(const void* k, const void* v, const float* g, const float* beta,
                                const int32_t* cu_seqlens, int32_t n_seg, int32_t t_total, int32_t H, int32_t dk,
                                int32_t dv, int kv_dtype, int gate, float* E, float* T, void* stream) {
  // size first: pure host arithmetic, the same figure hypic_segment_encode checks its workspace against (0 for an invalid
  // shape, which the call below then reports, and for the SIMT family, which uses no scratch)
  const size_t need = hypic_segment_encode_workspace(n_seg, t_total, H, dk, dv, kv_dtype, gate);
  if (need > kStaticScratchBytes) return HYPIC_ERR_STATIC_SCRATCH;
  void* ws = nullptr;
  const int st = static_scratch_ptr(&ws);
  if (st != HYPIC_OK) return st;
  return hypic_segment_encode(k, v, g, beta, cu_seqlens, n_seg, t_total, H, dk, dv, kv_dtype, gate, E, T, ws,
                              kStaticScratchBytes, stream);
}

}  // extern "C"
