// encode_simt.cu -- fp32 CUDA-core segment encode (kernel family HYPIC_IMPL_SIMT).
//
// Computes rows a0..a5 of SURVEY.md section 8(a) as the token recurrence itself (Eq. 2 with
// Table 1's GDN / KDA transitions), one thread per ROW of the stacked state X = [E; T]
// ((dv + dk) x dk).  Rows of X evolve independently of each other,
//     x <- x diag(a_t);   x <- x + beta_t (w_t - x.k_t) k_t^T,     w_t = v_t[i] for E rows, 0 for T rows,
// so a (segment, head) unit is split over ceil((dv+dk)/64) CTAs with no communication.  Each thread keeps
// its dk-wide row in registers; k_t / a_t / beta_t / w_t are staged per tile of TT tokens in shared memory
// and read as broadcasts.  This is the accurate path for fp32 inputs (cfg0, 1e-5) and the GPU-side second
// opinion for the tensor-core kernels; it is bound by the fp32 FMA pipe, not by HBM.
#include "common.cuh"

namespace hypic {
namespace {

constexpr int kRows = 64;  // threads (= rows of X) per CTA
constexpr int kTT = 16;    // tokens per staged tile

template <bool BF16>
__device__ __forceinline__ float load_kv(const void* p, size_t idx) {
  if (BF16) return __bfloat162float(reinterpret_cast<const __nv_bfloat16*>(p)[idx]);
  return reinterpret_cast<const float*>(p)[idx];
}

// One (segment s, head h, row block) unit of work; called by both kernels below.
template <int DK, bool BF16, bool CHANNEL>
__device__ __forceinline__ void encode_simt_unit(const void* __restrict__ k, const void* __restrict__ v,
                                                 const float* __restrict__ g, const float* __restrict__ beta,
                                                 const int32_t* __restrict__ cu_seqlens, int H, int dv,
                                                 float* __restrict__ E, float* __restrict__ T, int h, int s, int row0) {
  constexpr int AW = CHANNEL ? DK : 1;
  __shared__ __align__(16) float sk[2][kTT][DK];
  __shared__ __align__(16) float sa[2][kTT][AW];
  __shared__ float sw[2][kTT][kRows];
  __shared__ float sb[2][kTT];

  const int tid = threadIdx.x;
  const int row = row0 + tid;  // row of X = [E; T]
  const bool is_e = row < dv;
  const bool live = row < dv + DK;
  const int t_begin = cu_seqlens[s], t_end = cu_seqlens[s + 1];
  const int L = t_end - t_begin;

  float x[DK];
#pragma unroll
  for (int c = 0; c < DK; ++c) x[c] = 0.f;
  if (live && !is_e) {
#pragma unroll
    for (int c = 0; c < DK; ++c)
      if (c == row - dv) x[c] = 1.f;  // T starts at I (empty product)
  }

  auto stage = [&](int buf, int tile) {
    const int tbase = t_begin + tile * kTT;
    // k tile (and per-channel decay), converted to fp32 once per CTA
    for (int idx = tid; idx < kTT * DK; idx += kRows) {
      const int tok = idx / DK, c = idx % DK;
      const int t = tbase + tok;
      float kv = 0.f, av = 1.f;
      if (t < t_end) {
        const size_t th = (size_t)t * H + h;
        kv = load_kv<BF16>(k, th * DK + c);
        if (CHANNEL) av = expf(g[th * DK + c]);
      }
      sk[buf][tok][c] = kv;
      if (CHANNEL) sa[buf][tok][c] = av;
    }
    // this CTA's value entries w_t[i] (zero for T rows)
    for (int idx = tid; idx < kTT * kRows; idx += kRows) {
      const int tok = idx / kRows, j = idx % kRows;
      const int t = tbase + tok;
      float wv = 0.f;
      if (t < t_end && row0 + j < dv) wv = load_kv<BF16>(v, ((size_t)t * H + h) * dv + row0 + j);
      sw[buf][tok][j] = wv;
    }
    if (tid < kTT) {
      const int t = tbase + tid;
      float bv = 0.f, av = 1.f;
      if (t < t_end) {
        const size_t th = (size_t)t * H + h;
        bv = beta[th];
        if (!CHANNEL) av = expf(g[th]);
      }
      sb[buf][tid] = bv;
      if (!CHANNEL) sa[buf][tid][0] = av;
    }
  };

  const int n_tiles = (L + kTT - 1) / kTT;
  if (n_tiles > 0) stage(0, 0);
  __syncthreads();
  for (int tile = 0; tile < n_tiles; ++tile) {
    const int buf = tile & 1;
    if (tile + 1 < n_tiles) stage(buf ^ 1, tile + 1);
    const int n_tok = min(kTT, L - tile * kTT);
    for (int tok = 0; tok < n_tok; ++tok) {
      const float b = sb[buf][tok];
      const float w = sw[buf][tok][tid];
      const float4* k4 = reinterpret_cast<const float4*>(&sk[buf][tok][0]);
      float d0 = 0.f, d1 = 0.f, d2 = 0.f, d3 = 0.f;
      if (CHANNEL) {
        const float4* a4 = reinterpret_cast<const float4*>(&sa[buf][tok][0]);
#pragma unroll
        for (int c4 = 0; c4 < DK / 4; ++c4) {
          const float4 kk = k4[c4];
          const float4 aa = a4[c4];
          x[4 * c4 + 0] *= aa.x;
          x[4 * c4 + 1] *= aa.y;
          x[4 * c4 + 2] *= aa.z;
          x[4 * c4 + 3] *= aa.w;
          d0 = fmaf(x[4 * c4 + 0], kk.x, d0);
          d1 = fmaf(x[4 * c4 + 1], kk.y, d1);
          d2 = fmaf(x[4 * c4 + 2], kk.z, d2);
          d3 = fmaf(x[4 * c4 + 3], kk.w, d3);
        }
        const float coef = b * (w - ((d0 + d1) + (d2 + d3)));
#pragma unroll
        for (int c4 = 0; c4 < DK / 4; ++c4) {
          const float4 kk = k4[c4];
          x[4 * c4 + 0] = fmaf(coef, kk.x, x[4 * c4 + 0]);
          x[4 * c4 + 1] = fmaf(coef, kk.y, x[4 * c4 + 1]);
          x[4 * c4 + 2] = fmaf(coef, kk.z, x[4 * c4 + 2]);
          x[4 * c4 + 3] = fmaf(coef, kk.w, x[4 * c4 + 3]);
        }
      } else {
        const float a = sa[buf][tok][0];
#pragma unroll
        for (int c4 = 0; c4 < DK / 4; ++c4) {
          const float4 kk = k4[c4];
          d0 = fmaf(x[4 * c4 + 0], kk.x, d0);
          d1 = fmaf(x[4 * c4 + 1], kk.y, d1);
          d2 = fmaf(x[4 * c4 + 2], kk.z, d2);
          d3 = fmaf(x[4 * c4 + 3], kk.w, d3);
        }
        // decay first, then read the decayed state along k_t: (a x).k = a (x.k)
        const float coef = b * (w - a * ((d0 + d1) + (d2 + d3)));
#pragma unroll
        for (int c4 = 0; c4 < DK / 4; ++c4) {
          const float4 kk = k4[c4];
          x[4 * c4 + 0] = fmaf(coef, kk.x, a * x[4 * c4 + 0]);
          x[4 * c4 + 1] = fmaf(coef, kk.y, a * x[4 * c4 + 1]);
          x[4 * c4 + 2] = fmaf(coef, kk.z, a * x[4 * c4 + 2]);
          x[4 * c4 + 3] = fmaf(coef, kk.w, a * x[4 * c4 + 3]);
        }
      }
    }
    __syncthreads();
  }

  if (live) {
    float* dst = is_e ? E + (((size_t)s * H + h) * dv + row) * DK : T + (((size_t)s * H + h) * DK + (row - dv)) * DK;
    float4* d4 = reinterpret_cast<float4*>(dst);
#pragma unroll
    for (int c4 = 0; c4 < DK / 4; ++c4) d4[c4] = make_float4(x[4 * c4], x[4 * c4 + 1], x[4 * c4 + 2], x[4 * c4 + 3]);
  }
}

template <int DK, bool BF16, bool CHANNEL>
__global__ void __launch_bounds__(kRows) encode_simt_kernel(const void* __restrict__ k, const void* __restrict__ v,
                                                            const float* __restrict__ g,
                                                            const float* __restrict__ beta,
                                                            const int32_t* __restrict__ cu_seqlens, int H, int dv,
                                                            float* __restrict__ E, float* __restrict__ T) {
  encode_simt_unit<DK, BF16, CHANNEL>(k, v, g, beta, cu_seqlens, H, dv, E, T, blockIdx.y, blockIdx.z, blockIdx.x * kRows);
}

// The same work over a device-side list of units: CTA (x, y) takes row block x of list entries y, y + gridDim.y, ...
// An empty list costs one load per CTA.
template <int DK, bool BF16, bool CHANNEL>
__global__ void __launch_bounds__(kRows) encode_simt_list_kernel(const void* __restrict__ k, const void* __restrict__ v,
                                                                 const float* __restrict__ g,
                                                                 const float* __restrict__ beta,
                                                                 const int32_t* __restrict__ cu_seqlens, int H, int dv,
                                                                 float* __restrict__ E, float* __restrict__ T,
                                                                 const int32_t* __restrict__ unit_list,
                                                                 const int32_t* __restrict__ unit_count) {
  const int n = *unit_count;
  for (int i = blockIdx.y; i < n; i += gridDim.y) {
    const int u = unit_list[i];
    encode_simt_unit<DK, BF16, CHANNEL>(k, v, g, beta, cu_seqlens, H, dv, E, T, u % H, u / H, blockIdx.x * kRows);
    __syncthreads();  // the staging buffers are reused by the next unit
  }
}

template <int DK, bool BF16, bool CHANNEL>
int launch(const EncodeArgs& a) {
  dim3 grid((a.dv + DK + kRows - 1) / kRows, a.H, a.n_seg);
  encode_simt_kernel<DK, BF16, CHANNEL><<<grid, kRows, 0, a.stream>>>(a.k, a.v, a.g, a.beta, a.cu_seqlens, a.H, a.dv,
                                                                     a.E, a.T);
  note_launch();
  HYPIC_CUDA_OK(cudaGetLastError());
  return HYPIC_OK;
}

template <int DK>
int dispatch(const EncodeArgs& a) {
  const bool bf = a.kv_dtype == HYPIC_DT_BF16, ch = a.gate == HYPIC_GATE_CHANNEL;
  if (bf) return ch ? launch<DK, true, true>(a) : launch<DK, true, false>(a);
  return ch ? launch<DK, false, true>(a) : launch<DK, false, false>(a);
}

template <int DK, bool CHANNEL>
int launch_list(const EncodeArgs& a, const int32_t* unit_list, const int32_t* unit_count) {
  const long long units = (long long)a.n_seg * a.H;
  const dim3 grid((a.dv + DK + kRows - 1) / kRows, (unsigned)(units < 296 ? units : 296));
  encode_simt_list_kernel<DK, true, CHANNEL><<<grid, kRows, 0, a.stream>>>(a.k, a.v, a.g, a.beta, a.cu_seqlens, a.H, a.dv,
                                                                          a.E, a.T, unit_list, unit_count);
  note_launch();
  HYPIC_CUDA_OK(cudaGetLastError());
  return HYPIC_OK;
}

}  // namespace

int encode_simt_list(const EncodeArgs& a, const int32_t* unit_list, const int32_t* unit_count) {
  if (a.dk != 128 || a.kv_dtype != HYPIC_DT_BF16) return HYPIC_ERR_UNSUPPORTED;  // the tensor family's shapes
  if (a.n_seg == 0) return HYPIC_OK;
  return a.gate == HYPIC_GATE_CHANNEL ? launch_list<128, true>(a, unit_list, unit_count)
                                      : launch_list<128, false>(a, unit_list, unit_count);
}

int encode_simt(const EncodeArgs& a) {
  if (a.H > 65535 || a.n_seg > 65535) return HYPIC_ERR_UNSUPPORTED;
  if (a.dv < 1 || a.dv > 1024) return HYPIC_ERR_UNSUPPORTED;
  if (a.n_seg == 0) return HYPIC_OK;
  if (a.dk == 128) return dispatch<128>(a);
  if (a.dk == 64) return dispatch<64>(a);
  return HYPIC_ERR_UNSUPPORTED;
}

}  // namespace hypic
