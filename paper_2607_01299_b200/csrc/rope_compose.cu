// rope_compose.cu -- state RoPE re-rotation for the scalar family (Eq. 7): hypic_rope_compose.
//
//   S <- t_i S + E_i R(p_i)^T      over each request's ordered id list, p_i = the segment's global start position.
//
// T_i = t_i I commutes with every rotation, so a zero-start end-state cached at position 0 is moved to position p by
// rotating each of its rows like a key (row convention: keys run along the dk columns).  Pairing: column c < dk/2 with
// column c + dk/2, angle p * inv_freq[c] (reading R1).
//
// Two launches:
//   rope_table_kernel    cos / sin of every (list entry, pair): the angle p * inv_freq[c] is formed and reduced in fp64
//                        (in fp32 the product alone is off by p * 2^-24 rad: 5e-3 at p = 80,000), total_steps x dk/2
//                        values into the caller's workspace ([step][cos dk/2 | sin dk/2] fp32; it stays in L2)
//   rope_compose_kernel  the element-wise fold of diag_compose_kernel with the rotation in front: a thread owns 4 float4s
//                        of S for the whole chain; the partner column c +- dk/2 of the same row sits dk/8 lanes away in
//                        the same warp, so the pair is completed with one shuffle per float; E is streamed once
//                        (HBM-bound: 4 dv dk bytes per head-step).
#include <cuda_fp16.h>

#include "common.cuh"

namespace hypic {
namespace {

constexpr int kRcThreads = 256;
constexpr int kRcV4 = 4;

__global__ void rope_table_kernel(const int32_t* __restrict__ pos, const float* __restrict__ inv_freq, int total_steps,
                                  int half, float* __restrict__ table) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= total_steps * half) return;
  const int j = i / half, c = i % half;
  const double phi = (double)pos[j] * (double)inv_freq[c];
  double s, co;
  sincos(phi, &s, &co);
  table[(size_t)j * 2 * half + c] = (float)co;
  table[(size_t)j * 2 * half + half + c] = (float)s;
}

template <bool F16>  // F16: end-states stored in fp16 (the paper's cache precision), exact inputs
__global__ void __launch_bounds__(kRcThreads, 3)  // 3 CTAs per SM like diag_compose_kernel: bytes in flight set the rate
    rope_compose_kernel(const float* S_in /* may alias S_out */, const void* __restrict__ E_pool,
                        const float* __restrict__ t_pool, const int32_t* __restrict__ seg_ids,
                        const int32_t* __restrict__ cu_segs, const float* __restrict__ table, int H, int dk, int unit_v4,
                        float* S_out) {
  const int tid = threadIdx.x;
  const int h = blockIdx.y, r = blockIdx.z;
  const size_t unit = (size_t)r * H + h;
  const int dk4 = dk / 4, half = dk / 2, lane_xor = dk4 / 2;  // partner float4 of the same row: dk/8 lanes away
  int e4[kRcV4];
  bool live[kRcV4];
#pragma unroll
  for (int i = 0; i < kRcV4; ++i) {
    e4[i] = (blockIdx.x * kRcV4 + i) * kRcThreads + tid;
    live[i] = e4[i] < unit_v4;  // unit_v4 % dk4 == 0 and dk4 | 32: a pair is live or dead as a whole
  }
  // (blockIdx.x * kRcV4 + i) * kRcThreads is a multiple of dk4, so the column of every float4 this thread owns is the same
  const int c4 = tid % dk4;               // float4 column inside the row
  const bool upper = 4 * c4 >= half;      // second half of the pair: E' = E cos + partner sin; first: E cos - partner sin
  const int cpair = (4 * c4) % half;      // first of this float4's four pair indices
  const float sgn = upper ? 1.f : -1.f;
  float4 x[kRcV4];
#pragma unroll
  for (int i = 0; i < kRcV4; ++i) {
    x[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (live[i] && S_in) x[i] = *(reinterpret_cast<const float4*>(S_in) + unit * unit_v4 + e4[i]);  // plain load: S_out may alias S_in
  }
  const int j0 = cu_segs[r], j1 = cu_segs[r + 1];
  float4 e_nxt[kRcV4], cs_nxt, sn_nxt;
  float t_nxt = 1.f;
  auto fetch = [&](int j) {
    const size_t ph = (size_t)seg_ids[j] * H + h;
#pragma unroll
    for (int i = 0; i < kRcV4; ++i) {
      e_nxt[i] = make_float4(0.f, 0.f, 0.f, 0.f);
      if (live[i]) {
        if (F16) {
          const uint2 hv = __ldcs(reinterpret_cast<const uint2*>(E_pool) + ph * unit_v4 + e4[i]);
          const float2 lo = __half22float2(*reinterpret_cast<const __half2*>(&hv.x));
          const float2 hi = __half22float2(*reinterpret_cast<const __half2*>(&hv.y));
          e_nxt[i] = make_float4(lo.x, lo.y, hi.x, hi.y);
        } else {
          e_nxt[i] = __ldcs(reinterpret_cast<const float4*>(E_pool) + ph * unit_v4 + e4[i]);
        }
      }
    }
    t_nxt = __ldg(t_pool + ph);
    cs_nxt = __ldg(reinterpret_cast<const float4*>(table + (size_t)j * dk + cpair));
    sn_nxt = __ldg(reinterpret_cast<const float4*>(table + (size_t)j * dk + half + cpair));
  };
  if (j0 < j1) fetch(j0);
  for (int j = j0; j < j1; ++j) {
    float4 e_cur[kRcV4];
#pragma unroll
    for (int i = 0; i < kRcV4; ++i) e_cur[i] = e_nxt[i];
    const float t = t_nxt;
    const float4 cs = cs_nxt;
    const float4 sn = make_float4(sgn * sn_nxt.x, sgn * sn_nxt.y, sgn * sn_nxt.z, sgn * sn_nxt.w);
    if (j + 1 < j1) fetch(j + 1);
#pragma unroll
    for (int i = 0; i < kRcV4; ++i) {
      float4 p;  // the partner columns of the same row (all 32 lanes take part: dead float4s carry zeros)
      p.x = __shfl_xor_sync(0xffffffffu, e_cur[i].x, lane_xor);
      p.y = __shfl_xor_sync(0xffffffffu, e_cur[i].y, lane_xor);
      p.z = __shfl_xor_sync(0xffffffffu, e_cur[i].z, lane_xor);
      p.w = __shfl_xor_sync(0xffffffffu, e_cur[i].w, lane_xor);
      const float rx = fmaf(p.x, sn.x, e_cur[i].x * cs.x), ry = fmaf(p.y, sn.y, e_cur[i].y * cs.y);
      const float rz = fmaf(p.z, sn.z, e_cur[i].z * cs.z), rw = fmaf(p.w, sn.w, e_cur[i].w * cs.w);
      x[i].x = fmaf(x[i].x, t, rx);
      x[i].y = fmaf(x[i].y, t, ry);
      x[i].z = fmaf(x[i].z, t, rz);
      x[i].w = fmaf(x[i].w, t, rw);
    }
  }
#pragma unroll
  for (int i = 0; i < kRcV4; ++i)
    if (live[i]) __stcs(reinterpret_cast<float4*>(S_out) + unit * unit_v4 + e4[i], x[i]);
}

}  // namespace

size_t rope_compose_workspace(int32_t total_steps, int32_t dk) {
  return (size_t)(total_steps > 0 ? total_steps : 0) * (size_t)dk * sizeof(float);
}

int rope_compose(const RopeComposeArgs& a) {
  if (a.H > 65535 || a.R > 65535) return HYPIC_ERR_UNSUPPORTED;
  // pairs are completed by a warp shuffle: a row of dk/4 float4s must divide the warp, and must hold both halves
  if (a.dk != 8 && a.dk != 16 && a.dk != 32 && a.dk != 64 && a.dk != 128) return HYPIC_ERR_UNSUPPORTED;
  if (a.dv < 1 || a.dv > 1024) return HYPIC_ERR_UNSUPPORTED;
  if (a.R == 0) return HYPIC_OK;
  const int half = a.dk / 2;
  float* table = reinterpret_cast<float*>(a.workspace);
  if (a.total_steps > 0) {
    const int n = a.total_steps * half;
    rope_table_kernel<<<(n + 255) / 256, 256, 0, a.stream>>>(a.pos, a.inv_freq, a.total_steps, half, table);
    note_launch();
    HYPIC_CUDA_OK(cudaGetLastError());
  }
  const int unit_v4 = a.dv * a.dk / 4;
  dim3 grid((unit_v4 + kRcThreads * kRcV4 - 1) / (kRcThreads * kRcV4), a.H, a.R);
  auto kern = a.e_f16 ? rope_compose_kernel<true> : rope_compose_kernel<false>;
  kern<<<grid, kRcThreads, 0, a.stream>>>(a.S_in, a.E_pool, a.t_pool, a.seg_ids, a.cu_segs, table, a.H,
                                                         a.dk, unit_v4, a.S_out);
  note_launch();
  HYPIC_CUDA_OK(cudaGetLastError());
  return HYPIC_OK;
}

}  // namespace hypic
