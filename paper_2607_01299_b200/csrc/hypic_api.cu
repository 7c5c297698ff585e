// hypic_api.cu -- the C ABI of include/hypic.h: argument validation, kernel-family selection, launches.
// Validation of host-visible arguments happens before any CUDA call (see hypic.h "General rules").
#include <atomic>

#include "common.cuh"

namespace hypic {

thread_local int g_launch_count = 0;
thread_local int g_last_cuda_error = 0;
static std::atomic<int> g_impl{HYPIC_IMPL_AUTO};

const DeviceInfo& device_info() {
  static DeviceInfo infos[64];
  static std::atomic<unsigned long long> known{0};
  static thread_local DeviceInfo scratch;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) dev = 0;
  DeviceInfo* d = (dev >= 0 && dev < 64) ? &infos[dev] : &scratch;
  if (dev >= 0 && dev < 64 && ((known.load(std::memory_order_acquire) >> dev) & 1ull)) return *d;
  DeviceInfo t{};
  cudaDeviceProp p;
  if (cudaGetDeviceProperties(&p, dev) == cudaSuccess) {
    t.device = dev;
    t.sm_count = p.multiProcessorCount;
    t.cc_major = p.major;
    t.cc_minor = p.minor;
    t.max_smem_optin = (int)p.sharedMemPerBlockOptin;
    t.ok = 1;
  }
  *d = t;  // concurrent first calls write the same values
  if (dev >= 0 && dev < 64 && t.ok) known.fetch_or(1ull << dev, std::memory_order_release);
  return *d;
}

static bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

static int validate_encode_shape(int32_t n_seg, int32_t t_total, int32_t H, int32_t dk, int32_t dv, int kv_dtype,
                                 int gate) {
  if (n_seg < 0 || t_total < 0 || H <= 0 || dk <= 0 || dv <= 0) return HYPIC_ERR_INVALID_ARG;
  if (kv_dtype != HYPIC_DT_F32 && kv_dtype != HYPIC_DT_BF16) return HYPIC_ERR_INVALID_ARG;
  if (gate != HYPIC_GATE_SCALAR && gate != HYPIC_GATE_CHANNEL) return HYPIC_ERR_INVALID_ARG;
  if (n_seg == 0 && t_total != 0) return HYPIC_ERR_INVALID_ARG;
  if (dk != 64 && dk != 128) return HYPIC_ERR_UNSUPPORTED;
  if (dv > 1024) return HYPIC_ERR_UNSUPPORTED;
  return HYPIC_OK;
}

}  // namespace hypic

using namespace hypic;

extern "C" {

int hypic_set_impl(int impl) {
  if (impl != HYPIC_IMPL_AUTO && impl != HYPIC_IMPL_SIMT && impl != HYPIC_IMPL_TENSOR) return HYPIC_ERR_INVALID_ARG;
  g_impl.store(impl);
  return HYPIC_OK;
}

int hypic_get_impl(void) { return g_impl.load(); }

size_t hypic_segment_encode_workspace(int32_t n_seg, int32_t t_total, int32_t H, int32_t dk, int32_t dv,
                                      int kv_dtype, int gate) {
  if (validate_encode_shape(n_seg, t_total, H, dk, dv, kv_dtype, gate) != HYPIC_OK) return 0;
  if (g_impl.load() == HYPIC_IMPL_SIMT) return 0;
  return encode_tensor_workspace(n_seg, t_total, H, dk, dv, kv_dtype, gate);
}

int hypic_segment_encode(const void* k, const void* v, const float* g, const float* beta,
                         const int32_t* cu_seqlens, int32_t n_seg, int32_t t_total, int32_t H, int32_t dk,
                         int32_t dv, int kv_dtype, int gate, float* E, float* T, void* workspace,
                         size_t workspace_bytes, void* stream) {
  g_launch_count = 0;
  const int vs = validate_encode_shape(n_seg, t_total, H, dk, dv, kv_dtype, gate);
  if (vs != HYPIC_OK) return vs;
  if (!cu_seqlens) return HYPIC_ERR_INVALID_ARG;
  if (n_seg > 0 && (!E || !T)) return HYPIC_ERR_INVALID_ARG;
  if (t_total > 0 && (!k || !v || !g || !beta)) return HYPIC_ERR_INVALID_ARG;
  if (!aligned16(k) || !aligned16(v) || !aligned16(g) || !aligned16(beta) || !aligned16(E) || !aligned16(T) ||
      !aligned16(workspace))
    return HYPIC_ERR_INVALID_ARG;
  EncodeArgs a{k, v, g, beta, cu_seqlens, n_seg, t_total, H, dk, dv, kv_dtype, gate, E, T, workspace, workspace_bytes,
               (cudaStream_t)stream};
  const int impl = g_impl.load();
  const bool tensor_ok = encode_tensor_supported(a);
  if (impl == HYPIC_IMPL_TENSOR && !tensor_ok) return HYPIC_ERR_UNSUPPORTED;
  if (tensor_ok && impl != HYPIC_IMPL_SIMT) {
    const size_t need = encode_tensor_workspace(n_seg, t_total, H, dk, dv, kv_dtype, gate);
    if (need > 0 && (!workspace || workspace_bytes < need)) return HYPIC_ERR_WORKSPACE;
    return encode_tensor(a);
  }
  return encode_simt(a);
}

int hypic_compose(const float* S_in, const float* E_pool, const float* T_pool, const int32_t* seg_ids,
                  const int32_t* cu_segs, int32_t R, int32_t P, int32_t total_steps, int32_t H, int32_t dk,
                  int32_t dv, float* S_out, void* stream) {
  g_launch_count = 0;
  if (R < 0 || P < 0 || total_steps < 0 || H <= 0 || dk <= 0 || dv <= 0) return HYPIC_ERR_INVALID_ARG;
  if (!cu_segs) return HYPIC_ERR_INVALID_ARG;
  if (R > 0 && !S_out) return HYPIC_ERR_INVALID_ARG;
  if (total_steps > 0 && (!E_pool || !T_pool || !seg_ids || P == 0)) return HYPIC_ERR_INVALID_ARG;
  if (!aligned16(S_in) || !aligned16(E_pool) || !aligned16(T_pool) || !aligned16(S_out)) return HYPIC_ERR_INVALID_ARG;
  if (dk != 64 && dk != 128) return HYPIC_ERR_UNSUPPORTED;
  if (dv > 1024) return HYPIC_ERR_UNSUPPORTED;
  ComposeArgs a{S_in, E_pool, T_pool, seg_ids, cu_segs, R, P, total_steps, H, dk, dv, S_out, (cudaStream_t)stream};
  const int impl = g_impl.load();
  const bool tensor_ok = compose_tensor_supported(a);
  if (impl == HYPIC_IMPL_TENSOR && !tensor_ok) return HYPIC_ERR_UNSUPPORTED;
  if (tensor_ok && impl != HYPIC_IMPL_SIMT) return compose_tensor(a);
  return compose_simt(a);
}

int hypic_compose_f16(const float* S_in, const void* E_pool, const void* T_pool, const int32_t* seg_ids,
                      const int32_t* cu_segs, int32_t R, int32_t P, int32_t total_steps, int32_t H, int32_t dk, int32_t dv,
                      float* S_out, void* stream) {
  g_launch_count = 0;
  if (R < 0 || P < 0 || total_steps < 0 || H <= 0 || dk <= 0 || dv <= 0) return HYPIC_ERR_INVALID_ARG;
  if (!cu_segs) return HYPIC_ERR_INVALID_ARG;
  if (R > 0 && !S_out) return HYPIC_ERR_INVALID_ARG;
  if (total_steps > 0 && (!E_pool || !T_pool || !seg_ids || P == 0)) return HYPIC_ERR_INVALID_ARG;
  if (!aligned16(S_in) || !aligned16(E_pool) || !aligned16(T_pool) || !aligned16(S_out)) return HYPIC_ERR_INVALID_ARG;
  if (!compose_f16_shape_ok(H, dk, dv)) return HYPIC_ERR_UNSUPPORTED;
  ComposeF16Args a{S_in, E_pool, T_pool, seg_ids, cu_segs, R, P, total_steps, H, dk, dv, S_out, (cudaStream_t)stream};
  return compose_f16(a);
}

int hypic_tuple_pack_f16(const float* src, void* dst, size_t count, void* stream) {
  g_launch_count = 0;
  if (count > 0 && (!src || !dst)) return HYPIC_ERR_INVALID_ARG;
  if (!aligned16(src) || !aligned16(dst)) return HYPIC_ERR_INVALID_ARG;
  return pack_f16(src, dst, count, (cudaStream_t)stream);
}

int hypic_seam_window(const void* q, const void* k, const void* v, const float* g, const float* beta,
                      const int32_t* cu_tokens, int32_t R, int32_t t_total, int32_t H, int32_t dk, int32_t dv,
                      int kv_dtype, int gate, const float* S_in, float* S_out, float* o, void* stream) {
  g_launch_count = 0;
  if (R < 0 || t_total < 0 || H <= 0 || dk <= 0 || dv <= 0) return HYPIC_ERR_INVALID_ARG;
  if (kv_dtype != HYPIC_DT_F32 && kv_dtype != HYPIC_DT_BF16) return HYPIC_ERR_INVALID_ARG;
  if (gate != HYPIC_GATE_SCALAR && gate != HYPIC_GATE_CHANNEL) return HYPIC_ERR_INVALID_ARG;
  if (!cu_tokens) return HYPIC_ERR_INVALID_ARG;
  if (R > 0 && !S_out) return HYPIC_ERR_INVALID_ARG;
  if (t_total > 0 && (!q || !k || !v || !g || !beta || !o)) return HYPIC_ERR_INVALID_ARG;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(g) || !aligned16(beta) || !aligned16(S_in) ||
      !aligned16(S_out) || !aligned16(o))
    return HYPIC_ERR_INVALID_ARG;
  if (dk != 64 && dk != 128) return HYPIC_ERR_UNSUPPORTED;
  if (dv > 1024) return HYPIC_ERR_UNSUPPORTED;
  SeamArgs a{q, k, v, g, beta, cu_tokens, R, t_total, H, dk, dv, kv_dtype, gate, S_in, S_out, o, nullptr,
             (cudaStream_t)stream};
  return seam_simt(a);
}

int hypic_forward_encode(const void* q, const void* k, const void* v, const float* g, const float* beta,
                         const int32_t* cu_seqlens, int32_t n_seg, int32_t t_total, int32_t H, int32_t dk, int32_t dv,
                         int kv_dtype, int gate, float* o, float* E, float* T, void* stream) {
  g_launch_count = 0;
  const int vs = validate_encode_shape(n_seg, t_total, H, dk, dv, kv_dtype, gate);
  if (vs != HYPIC_OK) return vs;
  if (!cu_seqlens) return HYPIC_ERR_INVALID_ARG;
  if (n_seg > 0 && (!E || !T)) return HYPIC_ERR_INVALID_ARG;
  if (t_total > 0 && (!q || !k || !v || !g || !beta || !o)) return HYPIC_ERR_INVALID_ARG;
  if (!aligned16(q) || !aligned16(k) || !aligned16(v) || !aligned16(g) || !aligned16(beta) || !aligned16(o) ||
      !aligned16(E) || !aligned16(T))
    return HYPIC_ERR_INVALID_ARG;
  SeamArgs a{q, k, v, g, beta, cu_seqlens, n_seg, t_total, H, dk, dv, kv_dtype, gate, nullptr, E, o, T,
             (cudaStream_t)stream};
  return seam_simt(a);
}

int hypic_diag_encode(const void* k, const void* v, const float* g, const int32_t* cu_seqlens, int32_t n_seg,
                      int32_t t_total, int32_t H, int32_t dk, int32_t dv, int kv_dtype, int gate, float* E, float* tvec,
                      void* stream) {
  g_launch_count = 0;
  const int vs = validate_encode_shape(n_seg, t_total, H, dk, dv, kv_dtype, gate);
  if (vs != HYPIC_OK) return vs;
  if (!cu_seqlens) return HYPIC_ERR_INVALID_ARG;
  if (n_seg > 0 && (!E || !tvec)) return HYPIC_ERR_INVALID_ARG;
  if (t_total > 0 && (!k || !v || !g)) return HYPIC_ERR_INVALID_ARG;
  if (!aligned16(k) || !aligned16(v) || !aligned16(g) || !aligned16(E) || !aligned16(tvec)) return HYPIC_ERR_INVALID_ARG;
  DiagEncodeArgs a{k, v, g, cu_seqlens, n_seg, t_total, H, dk, dv, kv_dtype, gate, E, tvec, (cudaStream_t)stream};
  const int impl = g_impl.load();
  const bool tensor_ok = diag_encode_tensor_shape_ok(H, dk, dv, kv_dtype, gate);
  if (impl == HYPIC_IMPL_TENSOR && !tensor_ok) return HYPIC_ERR_UNSUPPORTED;
  if (tensor_ok && impl != HYPIC_IMPL_SIMT && t_total > 0) return diag_encode_tensor(a);
  return diag_encode(a);
}

int hypic_diag_encode_impl_for(int32_t H, int32_t dk, int32_t dv, int kv_dtype, int gate) {
  const int vs = validate_encode_shape(0, 0, H, dk, dv, kv_dtype, gate);
  if (vs != HYPIC_OK) return -vs;
  const int impl = g_impl.load();
  const bool tensor_ok = diag_encode_tensor_shape_ok(H, dk, dv, kv_dtype, gate);
  if (impl == HYPIC_IMPL_TENSOR) return tensor_ok ? HYPIC_IMPL_TENSOR : -HYPIC_ERR_UNSUPPORTED;
  if (impl == HYPIC_IMPL_SIMT) return HYPIC_IMPL_SIMT;
  return tensor_ok ? HYPIC_IMPL_TENSOR : HYPIC_IMPL_SIMT;
}

static int diag_compose_call(const float* S_in, const void* E_pool, int e_f16, const float* t_pool, const int32_t* seg_ids,
                             const int32_t* cu_segs, int32_t R, int32_t P, int32_t total_steps, int32_t H, int32_t dk,
                             int32_t dv, int gate, float* S_out, void* stream) {
  g_launch_count = 0;
  if (R < 0 || P < 0 || total_steps < 0 || H <= 0 || dk <= 0 || dv <= 0) return HYPIC_ERR_INVALID_ARG;
  if (gate != HYPIC_GATE_SCALAR && gate != HYPIC_GATE_CHANNEL) return HYPIC_ERR_INVALID_ARG;
  if (!cu_segs) return HYPIC_ERR_INVALID_ARG;
  if (R > 0 && !S_out) return HYPIC_ERR_INVALID_ARG;
  if (total_steps > 0 && (!E_pool || !t_pool || !seg_ids || P == 0)) return HYPIC_ERR_INVALID_ARG;
  if (!aligned16(S_in) || !aligned16(E_pool) || !aligned16(t_pool) || !aligned16(S_out)) return HYPIC_ERR_INVALID_ARG;
  if (dk % 4 != 0 || dk > 1024 || dv > 1024) return HYPIC_ERR_UNSUPPORTED;
  DiagComposeArgs a{S_in, E_pool, t_pool, seg_ids, cu_segs, R, P, total_steps, H, dk, dv, gate, e_f16, S_out,
                    (cudaStream_t)stream};
  return diag_compose(a);
}

int hypic_diag_compose(const float* S_in, const float* E_pool, const float* t_pool, const int32_t* seg_ids,
                       const int32_t* cu_segs, int32_t R, int32_t P, int32_t total_steps, int32_t H, int32_t dk,
                       int32_t dv, int gate, float* S_out, void* stream) {
  return diag_compose_call(S_in, E_pool, 0, t_pool, seg_ids, cu_segs, R, P, total_steps, H, dk, dv, gate, S_out, stream);
}

int hypic_diag_compose_f16(const float* S_in, const void* E_pool, const float* t_pool, const int32_t* seg_ids,
                           const int32_t* cu_segs, int32_t R, int32_t P, int32_t total_steps, int32_t H, int32_t dk,
                           int32_t dv, int gate, float* S_out, void* stream) {
  return diag_compose_call(S_in, E_pool, 1, t_pool, seg_ids, cu_segs, R, P, total_steps, H, dk, dv, gate, S_out, stream);
}

size_t hypic_rope_compose_workspace(int32_t total_steps, int32_t dk) {
  if (total_steps <= 0 || dk <= 0) return 0;
  return rope_compose_workspace(total_steps, dk);
}

static int rope_compose_call(const float* S_in, const void* E_pool, int e_f16, const float* t_pool,
                             const int32_t* seg_ids, const int32_t* cu_segs, const int32_t* pos, const float* inv_freq,
                             int32_t R, int32_t P, int32_t total_steps, int32_t H, int32_t dk, int32_t dv, float* S_out,
                             void* workspace, size_t workspace_bytes, void* stream) {
  g_launch_count = 0;
  if (R < 0 || P < 0 || total_steps < 0 || H <= 0 || dk <= 0 || dv <= 0) return HYPIC_ERR_INVALID_ARG;
  if (!cu_segs) return HYPIC_ERR_INVALID_ARG;
  if (R > 0 && !S_out) return HYPIC_ERR_INVALID_ARG;
  if (total_steps > 0 && (!E_pool || !t_pool || !seg_ids || !pos || !inv_freq || P == 0)) return HYPIC_ERR_INVALID_ARG;
  if (!aligned16(S_in) || !aligned16(E_pool) || !aligned16(S_out) || !aligned16(workspace)) return HYPIC_ERR_INVALID_ARG;
  if (dk % 8 != 0) return HYPIC_ERR_UNSUPPORTED;
  if (total_steps > 0 && (!workspace || workspace_bytes < rope_compose_workspace(total_steps, dk)))
    return HYPIC_ERR_WORKSPACE;
  RopeComposeArgs a{S_in, E_pool, t_pool, seg_ids, cu_segs, pos, inv_freq, R, P, total_steps, H, dk, dv, S_out,
                    workspace, e_f16, (cudaStream_t)stream};
  return rope_compose(a);
}

int hypic_rope_compose(const float* S_in, const float* E_pool, const float* t_pool, const int32_t* seg_ids,
                       const int32_t* cu_segs, const int32_t* pos, const float* inv_freq, int32_t R, int32_t P,
                       int32_t total_steps, int32_t H, int32_t dk, int32_t dv, float* S_out, void* workspace,
                       size_t workspace_bytes, void* stream) {
  return rope_compose_call(S_in, E_pool, 0, t_pool, seg_ids, cu_segs, pos, inv_freq, R, P, total_steps, H, dk, dv, S_out,
                           workspace, workspace_bytes, stream);
}

int hypic_rope_compose_f16(const float* S_in, const void* E_pool, const float* t_pool, const int32_t* seg_ids,
                           const int32_t* cu_segs, const int32_t* pos, const float* inv_freq, int32_t R, int32_t P,
                           int32_t total_steps, int32_t H, int32_t dk, int32_t dv, float* S_out, void* workspace,
                           size_t workspace_bytes, void* stream) {
  return rope_compose_call(S_in, E_pool, 1, t_pool, seg_ids, cu_segs, pos, inv_freq, R, P, total_steps, H, dk, dv, S_out,
                           workspace, workspace_bytes, stream);
}

int hypic_encode_impl_for(int32_t H, int32_t dk, int32_t dv, int kv_dtype, int gate) {
  const int vs = validate_encode_shape(0, 0, H, dk, dv, kv_dtype, gate);
  if (vs != HYPIC_OK) return -vs;
  const int impl = g_impl.load();
  const bool tensor_ok = encode_tensor_shape_ok(H, dk, dv, kv_dtype, gate);
  if (impl == HYPIC_IMPL_TENSOR) return tensor_ok ? HYPIC_IMPL_TENSOR : -HYPIC_ERR_UNSUPPORTED;
  if (impl == HYPIC_IMPL_SIMT) return HYPIC_IMPL_SIMT;
  return tensor_ok ? HYPIC_IMPL_TENSOR : HYPIC_IMPL_SIMT;
}

int hypic_compose_impl_for(int32_t H, int32_t dk, int32_t dv) {
  if (H <= 0 || dk <= 0 || dv <= 0) return -HYPIC_ERR_INVALID_ARG;
  if ((dk != 64 && dk != 128) || dv > 1024) return -HYPIC_ERR_UNSUPPORTED;
  const int impl = g_impl.load();
  const bool tensor_ok = compose_tensor_shape_ok(H, dk, dv);
  if (impl == HYPIC_IMPL_TENSOR) return tensor_ok ? HYPIC_IMPL_TENSOR : -HYPIC_ERR_UNSUPPORTED;
  if (impl == HYPIC_IMPL_SIMT) return HYPIC_IMPL_SIMT;
  return tensor_ok ? HYPIC_IMPL_TENSOR : HYPIC_IMPL_SIMT;
}

const char* hypic_status_string(int status) {
  switch (status) {
    case HYPIC_OK: return "ok";
    case HYPIC_ERR_INVALID_ARG: return "invalid argument";
    case HYPIC_ERR_UNSUPPORTED: return "unsupported shape or dtype";
    case HYPIC_ERR_WORKSPACE: return "workspace missing or too small";
    case HYPIC_ERR_CUDA: return "CUDA error";
    case HYPIC_ERR_STATIC_SCRATCH: return "problem needs more scratch than the built-in static array holds (hypic_static_scratch_bytes)";
    default: return "unknown status";
  }
}

int hypic_version(void) { return HYPIC_VERSION; }

unsigned int hypic_debug_timeout_count(void) { return debug_timeout_count(); }

unsigned int hypic_envelope_violation_count(void) { return envelope_violation_count_encode(); }

int hypic_last_launch_count(void) { return g_launch_count; }

int hypic_last_cuda_error(void) { return g_last_cuda_error; }

}  // extern "C"
