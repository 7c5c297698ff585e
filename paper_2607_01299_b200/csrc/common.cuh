// common.cuh -- shared host/device helpers of libhypic (product code; nothing here is used by oracle/).
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

#include "../../include/hypic.h"

namespace hypic {

// Launch bookkeeping behind hypic_last_launch_count().
extern thread_local int g_launch_count;
inline void note_launch(int n = 1) { g_launch_count += n; }

// The CUDA error behind the most recent HYPIC_ERR_CUDA of this thread (hypic_last_cuda_error()).
extern thread_local int g_last_cuda_error;

#define HYPIC_CUDA_OK(expr)                        \
  do {                                             \
    cudaError_t _e = (expr);                       \
    if (_e != cudaSuccess) {                       \
      g_last_cuda_error = (int)_e;                 \
      return HYPIC_ERR_CUDA;                       \
    }                                              \
  } while (0)

struct EncodeArgs {
  const void* k;
  const void* v;
  const float* g;
  const float* beta;
  const int32_t* cu_seqlens;
  int32_t n_seg, t_total, H, dk, dv;
  int kv_dtype, gate;
  float* E;
  float* T;
  void* workspace;
  size_t workspace_bytes;
  cudaStream_t stream;
};

struct ComposeArgs {
  const float* S_in;
  const float* E_pool;
  const float* T_pool;
  const int32_t* seg_ids;
  const int32_t* cu_segs;
  int32_t R, P, total_steps, H, dk, dv;
  float* S_out;
  cudaStream_t stream;
};

struct ComposeF16Args {
  const float* S_in;
  const void* E_pool;  // fp16
  const void* T_pool;  // fp16
  const int32_t* seg_ids;
  const int32_t* cu_segs;
  int32_t R, P, total_steps, H, dk, dv;
  float* S_out;
  cudaStream_t stream;
};

struct SeamArgs {
  const void* q;
  const void* k;
  const void* v;
  const float* g;
  const float* beta;
  const int32_t* cu_tokens;
  int32_t R, t_total, H, dk, dv;
  int kv_dtype, gate;
  const float* S_in;
  float* S_out;
  float* o;
  float* T_out;  // NULL: seam-window step; else forward-encode mode (rows of T appended to the state)
  cudaStream_t stream;
};

struct DiagEncodeArgs {
  const void* k;
  const void* v;
  const float* g;
  const int32_t* cu_seqlens;
  int32_t n_seg, t_total, H, dk, dv;
  int kv_dtype, gate;
  float* E;
  float* tvec;
  cudaStream_t stream;
};

struct DiagComposeArgs {
  const float* S_in;
  const void* E_pool;  // fp32, or fp16 when e_f16
  const float* t_pool;
  const int32_t* seg_ids;
  const int32_t* cu_segs;
  int32_t R, P, total_steps, H, dk, dv;
  int gate;
  int e_f16;
  float* S_out;
  cudaStream_t stream;
};

struct RopeComposeArgs {
  const float* S_in;
  const void* E_pool;  // fp32, or fp16 when e_f16
  const float* t_pool;
  const int32_t* seg_ids;
  const int32_t* cu_segs;
  const int32_t* pos;
  const float* inv_freq;
  int32_t R, P, total_steps, H, dk, dv;
  float* S_out;
  void* workspace;
  int e_f16;
  cudaStream_t stream;
};

// Kernel families (each returns a hypic_status_t; UNSUPPORTED when the shape is outside its envelope).
int encode_simt(const EncodeArgs& a);
// the same kernel over a device-side list of units (s H + h), *unit_count entries; used as the in-call fp32 fallback
int encode_simt_list(const EncodeArgs& a, const int32_t* unit_list, const int32_t* unit_count);
int compose_simt(const ComposeArgs& a);
int seam_simt(const SeamArgs& a);
int diag_encode(const DiagEncodeArgs& a);
int diag_compose(const DiagComposeArgs& a);
size_t rope_compose_workspace(int32_t total_steps, int32_t dk);
int rope_compose(const RopeComposeArgs& a);
bool diag_encode_tensor_shape_ok(int32_t H, int32_t dk, int32_t dv, int kv_dtype, int gate);
int diag_encode_tensor(const DiagEncodeArgs& a);
bool encode_tensor_shape_ok(int32_t H, int32_t dk, int32_t dv, int kv_dtype, int gate);
inline bool encode_tensor_supported(const EncodeArgs& a) {
  return encode_tensor_shape_ok(a.H, a.dk, a.dv, a.kv_dtype, a.gate);
}
size_t encode_tensor_workspace(int32_t n_seg, int32_t t_total, int32_t H, int32_t dk, int32_t dv, int kv_dtype,
                               int gate);
int encode_tensor(const EncodeArgs& a);
bool compose_tensor_shape_ok(int32_t H, int32_t dk, int32_t dv);
inline bool compose_tensor_supported(const ComposeArgs& a) { return compose_tensor_shape_ok(a.H, a.dk, a.dv); }
int compose_tensor(const ComposeArgs& a);
bool compose_f16_shape_ok(int32_t H, int32_t dk, int32_t dv);
int compose_f16(const ComposeF16Args& a);
int pack_f16(const float* src, void* dst, size_t n, cudaStream_t stream);
unsigned int debug_timeout_count_compose_f16();
unsigned int debug_timeout_count_encode();
unsigned int envelope_violation_count_encode();
unsigned int debug_timeout_count();  // bounded-wait expiries in the tensor kernels since load (0 = healthy)

// Per-device one-time setup (cudaFuncSetAttribute is per device): `mask` holds one bit per device ordinal (< 64; beyond
// that the setup simply runs on every call).  Concurrent first calls may both run the setup, which is idempotent.
inline bool needs_device_setup(std::atomic<unsigned long long>& mask, int* dev_out) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) dev = 0;
  *dev_out = dev;
  return dev >= 64 || ((mask.load(std::memory_order_acquire) >> dev) & 1ull) == 0;
}
inline void device_setup_done(std::atomic<unsigned long long>& mask, int dev) {
  if (dev < 64) mask.fetch_or(1ull << dev, std::memory_order_release);
}

// Device properties of the CURRENT device, cached per device ordinal (SM count, opt-in shared memory).
struct DeviceInfo {
  int ok;  // 0 = not queried / failed
  int device;
  int sm_count;
  int cc_major, cc_minor;
  int max_smem_optin;
};
const DeviceInfo& device_info();

}  // namespace hypic
