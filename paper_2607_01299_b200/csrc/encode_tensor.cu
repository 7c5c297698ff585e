// encode_tensor.cu -- tcgen05/TMEM segment encode: bf16 k/v, scalar gate, dk = dv = 128 (HYPIC_IMPL_TENSOR).
//
// Rows a0..a5 of SURVEY.md section 8(a), chunked (C = 64 tokens) WY/UT form of the token recurrence
// (Eq. 2, Table 1 GDN / KDA rows PAPER.md:61; T_C and S_{C|0} of PAPER.md:118-126).
//   Scalar gate (GDN): K0 chunk_offsets + ONE fused kernel, scan4_kernel (encode_scan4.cuh): the gate commutes with the
//     delta rule's factors, so the chunk algebra is gate-free and runs in the reverse (suffix-product) form.
//   Per-channel gate (KDA): K0 + K1 prep_kernel<1> (encode_prep.cuh: Gram, L, A = (I + L)^-1 by a blocked inverse, -W and
//     A_b as ready-made UMMA B tiles plus the gate record, in HBM) + K2 scan2_kernel<1> (encode_scan2.cuh: one CTA per
//     (segment, head), sequential over chunks, both row blocks of X = [E ; T] resident in TMEM).
//   Units the fp16 operands cannot carry go to a device-side list that the fp32 family recomputes inside the same call.
#include <cuda.h>
#include <cuda_fp16.h>
#include <stdlib.h>

#include "common.cuh"
#include "sm100_ptx.cuh"

namespace hypic {
namespace {
using namespace ptx;

constexpr int kC = 64;                  // chunk length (north_star)
constexpr int kD = 128;                 // dk = dv
constexpr int kTileB = kC * kC * 2;     // one 16-bit 64x64 tile: 8 KB
constexpr int kRecW = 0;                // record: -W (fp16, [token][dk], two 64-wide boxes) 16 KB
constexpr int kRecAb = 2 * kTileB;      //         A_b (fp16, [token][token]) 8 KB
constexpr int kRecBytes = 3 * kTileB;   // 24 KB per (chunk, head)
constexpr int kGateFloats = 72;         // d_j[64], gamma_C, pad (288 B = 18 x 16 B)
constexpr int kGateBytes = kGateFloats * 4;
// per-channel gate (KDA row of Table 1): the record also carries K~_j = k_j (.) (Gamma_C (/) Gamma_j) (fp16,
// laid out like a K tile) and the gate record is Gamma_C[128]
constexpr int kRecKt = 3 * kTileB;
constexpr int kRecBytesCh = 5 * kTileB;  // 40 KB per (chunk, head)
constexpr int kGateFloatsCh = 144;       // Gamma_C[128], pad (576 B = 36 x 16 B)
constexpr int kGateBytesCh = kGateFloatsCh * 4;

__host__ __device__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
// workspace: chunk_off int32[n_seg + 1], seg_order int32[n_seg] | fallback list int32[4 + 2 n_seg H] | chunk_meta int2[cap] |
//            records [cap][H][kRecBytes] | gate [cap][H][kGateFloats]
__host__ __device__ inline size_t chunk_cap(int32_t n_seg, int32_t t_total) { return (size_t)t_total / kC + n_seg; }
__host__ __device__ inline size_t ws_off_fb(int32_t n_seg) { return align_up(8 * ((size_t)n_seg + 1), 1024); }
__host__ __device__ inline size_t ws_off_meta(int32_t n_seg, int32_t H) {
  return ws_off_fb(n_seg) + align_up(4 * (4 + 2 * (size_t)n_seg * H), 1024);
}
__host__ __device__ inline size_t ws_off_rec(int32_t n_seg, int32_t H, size_t cap) {
  return ws_off_meta(n_seg, H) + align_up(8 * cap, 1024);
}

// ------------------------------------------------------------------------------------------------ K0
// chunk_meta[x] = (first token, number of valid tokens) of global chunk x, (0, 0) for the unused tail of the table:
// the prep CTAs read one entry instead of searching chunk_off (a chain of dependent global loads).
// seg_order = the segments by decreasing length (the paper's LPT rule, used here as the launch order of
// the scan CTAs so that the longest sequential scans start first); identity beyond 8192 segments.
__global__ void chunk_offsets_kernel(const int32_t* __restrict__ cu_seqlens, int n_seg, int32_t* __restrict__ chunk_off,
                                     int32_t* __restrict__ seg_order, int2* __restrict__ chunk_meta, int cap,
                                     int32_t* __restrict__ fb, long long n_units, int need_meta) {
  __shared__ int part[1024];
  const int tid = threadIdx.x;
  for (long long i = tid; i < 4 + n_units; i += 1024) fb[i] = 0;  // empty fallback list, no unit flagged
  const int per = (n_seg + 1023) / 1024;
  const int lo = min(n_seg, tid * per), hi = min(n_seg, lo + per);
  int sum = 0;
  for (int s = lo; s < hi; ++s) sum += (cu_seqlens[s + 1] - cu_seqlens[s] + kC - 1) / kC;
  {  // exclusive prefix sum of the 1,024 partial counts: warp scans, then a scan of the 32 warp totals
    const int lane = tid & 31, warp = tid >> 5;
    int incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int up = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += up;
    }
    __shared__ int wtot[32];
    if (lane == 31) wtot[warp] = incl;
    __syncthreads();
    if (warp == 0) {
      int w = wtot[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int up = __shfl_up_sync(0xffffffffu, w, o);
        if (lane >= o) w += up;
      }
      wtot[lane] = w;  // inclusive
      if (lane == 31) chunk_off[n_seg] = w;
    }
    __syncthreads();
    part[tid] = incl - sum + (warp > 0 ? wtot[warp - 1] : 0);
  }
  int run = part[tid];
  for (int s = lo; s < hi; ++s) {
    chunk_off[s] = run;
    const int b = cu_seqlens[s], e = cu_seqlens[s + 1];
    const int n = (e - b + kC - 1) / kC;
    if (need_meta)
      for (int c = 0; c < n; ++c) chunk_meta[run + c] = make_int2(b + c * kC, min(kC, e - b - c * kC));
    run += n;
  }
  __shared__ int total;
  if (tid == 1023) total = run;  // the last thread ends at the grand total
  __syncthreads();
  if (need_meta)
    for (int x = total + tid; x < cap; x += 1024) chunk_meta[x] = make_int2(0, 0);
  for (int sg = tid; sg < n_seg; sg += 1024) {
    int rank = sg;
    if (n_seg <= 8192) {
      const int len = cu_seqlens[sg + 1] - cu_seqlens[sg];
      rank = 0;
      for (int t = 0; t < n_seg; ++t) {
        const int lt = cu_seqlens[t + 1] - cu_seqlens[t];
        rank += (lt > len || (lt == len && t < sg)) ? 1 : 0;
      }
    }
    seg_order[rank] = sg;
  }
}

// ------------------------------------------------------------------------------------------------ K1, K2
__device__ unsigned int g_timeout_count_enc = 0;
__device__ unsigned int g_envelope_count_enc = 0;  // (chunk, head) pairs outside the fp16 envelope (hypic.h)

// The fallback list of a call (workspace): fb[0] = count, fb[4 .. 4 + n_units) = per-unit flags, then the list.  A unit
// (segment s, head h -> s H + h) is appended once; encode_simt's list kernel recomputes it in fp32 after the scan.
__device__ __forceinline__ void fb_append(int32_t* fb, int n_units, int unit) {
  if (atomicExch(&fb[4 + unit], 1) == 0) fb[4 + n_units + atomicAdd(&fb[0], 1)] = unit;
}

#include "encode_prep.cuh"

#include "encode_scan2.cuh"

#include "encode_scan4.cuh"

#include "diag_scan.cuh"

// k / v viewed as 3-D bf16 tensors [t_total][H][128]; box = 64 elements (128 B) x 1 head x 64 tokens, 128B swizzle:
// the box lands as one MN-major UMMA chunk (8-token atoms of 1 KB), two boxes per 64 x 128 tile.
typedef CUresult (*EncodeTiledFn3)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int make_kv_tensor_map(CUtensorMap* tm, const void* base, int32_t t_total, int32_t H) {
  static EncodeTiledFn3 fn = nullptr;
  if (fn == nullptr) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess || p == nullptr)
      return HYPIC_ERR_CUDA;
    fn = reinterpret_cast<EncodeTiledFn3>(p);
  }
  const cuuint64_t dims[3] = {(cuuint64_t)kD, (cuuint64_t)H, (cuuint64_t)t_total};
  const cuuint64_t strides[2] = {(cuuint64_t)kD * 2, (cuuint64_t)H * kD * 2};
  const cuuint32_t box[3] = {64, 1, 64};
  const cuuint32_t estr[3] = {1, 1, 1};
  const CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? HYPIC_OK : HYPIC_ERR_CUDA;
}

// E = 0, T = I for every (segment, head) when the call carries no tokens at all (no tensor map can be built).
__global__ void identity_fill_kernel(float* __restrict__ E, float* __restrict__ T, size_t n_units) {
  const size_t n = n_units * kD * kD;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    E[i] = 0.f;
    const size_t e = i % (kD * kD);
    T[i] = (e / kD == e % kD) ? 1.f : 0.f;
  }
}

}  // namespace

bool encode_tensor_shape_ok(int32_t, int32_t dk, int32_t dv, int kv_dtype, int gate) {
  return dk == kD && dv == kD && kv_dtype == HYPIC_DT_BF16 && (gate == HYPIC_GATE_SCALAR || gate == HYPIC_GATE_CHANNEL);
}

size_t encode_tensor_workspace(int32_t n_seg, int32_t t_total, int32_t H, int32_t dk, int32_t dv, int kv_dtype,
                               int gate) {
  if (!encode_tensor_shape_ok(H, dk, dv, kv_dtype, gate)) return 0;
  const size_t cap = chunk_cap(n_seg, t_total);
  // scalar gate: one fused kernel, nothing but the chunk tables and the fallback list; per-channel gate: prep records
  if (gate != HYPIC_GATE_CHANNEL) return ws_off_rec(n_seg, H, cap);
  return ws_off_rec(n_seg, H, cap) + cap * H * ((size_t)kRecBytesCh + kGateBytesCh);
}

int encode_tensor(const EncodeArgs& a) {
  if (!encode_tensor_supported(a)) return HYPIC_ERR_UNSUPPORTED;
  if (a.n_seg == 0) return HYPIC_OK;
  if (a.H > 65535 || a.n_seg > 65535 || (long long)a.H * a.n_seg > 0x3fffffffLL) return HYPIC_ERR_UNSUPPORTED;
  const size_t cap = chunk_cap(a.n_seg, a.t_total);
  if (cap > 0x7fffffffULL) return HYPIC_ERR_UNSUPPORTED;
  if (a.t_total == 0) {
    identity_fill_kernel<<<296, 256, 0, a.stream>>>(a.E, a.T, (size_t)a.n_seg * a.H);
    note_launch();
    HYPIC_CUDA_OK(cudaGetLastError());
    return HYPIC_OK;
  }
  uint8_t* ws = static_cast<uint8_t*>(a.workspace);
  int32_t* chunk_off = reinterpret_cast<int32_t*>(ws);
  int32_t* seg_order = chunk_off + a.n_seg + 1;
  int32_t* fb = reinterpret_cast<int32_t*>(ws + ws_off_fb(a.n_seg));
  const int n_units = a.n_seg * a.H;
  int2* chunk_meta = reinterpret_cast<int2*>(ws + ws_off_meta(a.n_seg, a.H));
  uint8_t* rec = ws + ws_off_rec(a.n_seg, a.H, cap);
  const bool ch = a.gate == HYPIC_GATE_CHANNEL;
  float* gate = reinterpret_cast<float*>(rec + cap * a.H * (size_t)(ch ? kRecBytesCh : kRecBytes));
  static std::atomic<unsigned long long> configured{0};
  int cfg_dev = 0;
  if (needs_device_setup(configured, &cfg_dev)) {
    HYPIC_CUDA_OK(cudaFuncSetAttribute(scan4_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kR_Smem));
    HYPIC_CUDA_OK(cudaFuncSetAttribute(scan2_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kS2Smem));
    device_setup_done(configured, cfg_dev);
  }
  const auto* kp = static_cast<const __nv_bfloat16*>(a.k);
  CUtensorMap tmK, tmV;
  int rc = make_kv_tensor_map(&tmK, a.k, a.t_total, a.H);
  if (rc == HYPIC_OK) rc = make_kv_tensor_map(&tmV, a.v, a.t_total, a.H);
  if (rc != HYPIC_OK) return rc;
  chunk_offsets_kernel<<<1, 1024, 0, a.stream>>>(a.cu_seqlens, a.n_seg, chunk_off, seg_order, chunk_meta, (int)cap, fb,
                                                 (long long)n_units, ch ? 1 : 0);  // the fused scalar-gate kernel needs no chunk table
  note_launch();
  const dim3 pgrid((unsigned)((cap + kPrepChunksPerCta - 1) / kPrepChunksPerCta), a.H), sgrid(a.H, a.n_seg);
  if (ch) {
    prep_kernel<true><<<pgrid, kPrepThreads, 0, a.stream>>>(kp, a.g, a.beta, chunk_meta, (int)cap, a.H, rec, gate, chunk_off,
                                                            a.n_seg, fb);
    note_launch();
    scan2_kernel<true><<<sgrid, kS2Threads, kS2Smem, a.stream>>>(tmK, tmV, a.cu_seqlens, chunk_off, seg_order, a.H, rec, gate,
                                                                 a.E, a.T, fb, n_units);
  } else {
    scan4_kernel<<<sgrid, kR_Threads, kR_Smem, a.stream>>>(tmK, tmV, a.g, a.beta, a.cu_seqlens, seg_order, a.H, a.E, a.T, fb,
                                                           n_units);
  }
  note_launch();
  HYPIC_CUDA_OK(cudaGetLastError());
  // Units the fp16 operands could not carry (a per-channel chunk decaying below e^-9, an operand beyond 65504, ...)
  // were put on the call's fallback list by the kernels above: the fp32 family recomputes exactly those, in the same
  // call and on the same stream, with a device-side list -- no work (a few idle CTAs) when the list is empty.
  return encode_simt_list(a, fb + 4 + n_units, fb);
}

bool diag_encode_tensor_shape_ok(int32_t, int32_t dk, int32_t dv, int kv_dtype, int gate) {
  return dk == kD && dv == kD && kv_dtype == HYPIC_DT_BF16 && (gate == HYPIC_GATE_SCALAR || gate == HYPIC_GATE_CHANNEL);
}

// Scalar family on the tensor cores (diag_scan.cuh).  t_total > 0 (the tensor maps need a non-empty tensor).
int diag_encode_tensor(const DiagEncodeArgs& a) {
  if (!diag_encode_tensor_shape_ok(a.H, a.dk, a.dv, a.kv_dtype, a.gate) || a.t_total <= 0) return HYPIC_ERR_UNSUPPORTED;
  if (a.n_seg == 0) return HYPIC_OK;
  if (a.H > 65535 || a.n_seg > 65535) return HYPIC_ERR_UNSUPPORTED;
  static std::atomic<unsigned long long> configured{0};
  int cfg_dev = 0;
  if (needs_device_setup(configured, &cfg_dev)) {
    HYPIC_CUDA_OK(cudaFuncSetAttribute(diag_scan_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kDtSmem));
    HYPIC_CUDA_OK(cudaFuncSetAttribute(diag_scan_split2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kDtSmem));
    HYPIC_CUDA_OK(cudaFuncSetAttribute(diag_scan_ch_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kDtChSmem));
    device_setup_done(configured, cfg_dev);
  }
  CUtensorMap tmK, tmV;
  int rc = make_kv_tensor_map(&tmK, a.k, a.t_total, a.H);
  if (rc == HYPIC_OK) rc = make_kv_tensor_map(&tmV, a.v, a.t_total, a.H);
  if (rc != HYPIC_OK) return rc;
  if (a.gate == HYPIC_GATE_CHANNEL)
    diag_scan_ch_kernel<<<dim3(a.H, a.n_seg), kDtThreads, kDtChSmem, a.stream>>>(tmK, tmV, a.g, a.cu_seqlens, a.H, a.E,
                                                                                a.tvec);
  else {
    // pair-split only while the split CTAs still fit one wave (few units: twice the parallelism, half the chain length).
    // With more units than that the split LOSES (measured on the cfg2-shaped layer, 640 units on 444 slots: 0.31 ms split
    // vs 0.25 ms unsplit -- the pipeline fill / drain and the E_1 round trip are paid twice, and the unsplit tail wave runs
    // faster than a full one anyway).
    const DeviceInfo& di = device_info();
    const long long slots = 3LL * (di.ok ? di.sm_count : 148), U = (long long)a.H * a.n_seg;
    const bool split = 2 * U <= slots;
    if (split)
      diag_scan_split2_kernel<<<dim3(a.H, a.n_seg, 2), kDtThreads, kDtSmem, a.stream>>>(tmK, tmV, a.g, a.cu_seqlens, a.H,
                                                                                       a.E, a.tvec);
    else
      diag_scan_kernel<<<dim3(a.H, a.n_seg), kDtThreads, kDtSmem, a.stream>>>(tmK, tmV, a.g, a.cu_seqlens, a.H, a.E,
                                                                             a.tvec);
  }
  note_launch();
  HYPIC_CUDA_OK(cudaGetLastError());
  return HYPIC_OK;
}

unsigned int envelope_violation_count_encode() {
  unsigned int v = 0;
  if (cudaDeviceSynchronize() != cudaSuccess) return 0xffffffffu;
  if (cudaMemcpyFromSymbol(&v, g_envelope_count_enc, sizeof(v)) != cudaSuccess) return 0xffffffffu;
  return v;
}

unsigned int debug_timeout_count_encode() {
  unsigned int v = 0;
  if (cudaMemcpyFromSymbol(&v, g_timeout_count_enc, sizeof(v)) != cudaSuccess) return 0xffffffffu;
  return v;
}

}  // namespace hypic
