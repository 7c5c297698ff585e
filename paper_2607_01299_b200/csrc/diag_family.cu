// diag_family.cu -- scalar and diagonal families of PAPER.md:57-61 (Table 1) with the compressed transitions of
// PAPER.md:188-200 (Table 3): T_i = a_i I (RetNet, Lightning-2, Mamba2) or diag(g_i) (GLA), u_i = k_i v_i^T.
// Row convention (state dv x dk):   S <- S diag(a_t) + v_t k_t^T,  a_t = exp(g_t);
//     encode:   E = end state from 0,  tvec = prod_t a_t   (one scalar, or a dk-vector, per (segment, head))
//     compose:  S <- S diag(tvec_i) + E_i                   (element-wise: "O(dk dv)" apply cost of Table 3)
//
// diag_encode_simt_kernel (fp32 CUDA cores; the accurate path for fp32 inputs and any dk in {64,128}, dv <= 1024):
//   one thread per row of E, dk-wide row in registers.  Tokens are staged in tiles of 16; inside a tile the keys are
//   pre-weighted once per CTA with the decay from their token to the END of the tile, k~_t = k_t * exp(G_end - G_t)
//   (a factor in (0, 1]: no overflow whatever the gate), so the row update is one FMA per element and token,
//   x += v_t[i] k~_t, and the state is decayed once per tile, x *= exp(G_end - G_start).  tvec is the exponential of
//   the log-decay summed in fp64 (4,096 fp32 terms would cost 1e-5 in fp32).
// diag_compose_kernel: the fold is element-wise, so every thread owns 4 float4s of S for the whole chain and streams
//   the E_i of its request through registers, one step prefetched ahead: bound by reading E_i from HBM.
#include <cuda_fp16.h>

#include "common.cuh"

namespace hypic {
namespace {

constexpr int kDgRows = 64;  // threads (= rows of E) per encode CTA
constexpr int kDgTT = 16;    // tokens per staged tile

template <bool BF16>
__device__ __forceinline__ float dg_load(const void* p, size_t idx) {
  if (BF16) return __bfloat162float(reinterpret_cast<const __nv_bfloat16*>(p)[idx]);
  return reinterpret_cast<const float*>(p)[idx];
}

template <int DK, bool BF16, bool CHANNEL>
__global__ void __launch_bounds__(kDgRows)
    diag_encode_simt_kernel(const void* __restrict__ k, const void* __restrict__ v, const float* __restrict__ g,
                            const int32_t* __restrict__ cu_seqlens, int H, int dv, float* __restrict__ E,
                            float* __restrict__ tvec) {
  constexpr int AW = CHANNEL ? DK : 1;
  __shared__ __align__(16) float sk[2][kDgTT][DK];   // pre-weighted keys of the tile
  __shared__ __align__(16) float sdec[2][AW];        // decay over the whole tile
  __shared__ float sw[2][kDgTT][kDgRows];            // this CTA's value entries v_t[i]
  __shared__ __align__(16) float sg[kDgTT][CHANNEL ? DK : 4];  // log-decays of the tile being staged

  const int tid = threadIdx.x;
  const int h = blockIdx.y, s = blockIdx.z;
  const int row0 = blockIdx.x * kDgRows;
  const int row = row0 + tid;
  const int t_begin = cu_seqlens[s], t_end = cu_seqlens[s + 1];
  const int L = t_end - t_begin;

  float x[DK];
#pragma unroll
  for (int c = 0; c < DK; ++c) x[c] = 0.f;

  // fp64 running sum of the log-decay: CTA 0 of the unit writes tvec.  Scalar gate: thread 0; channel gate: thread c
  // and c + 64.
  double gsum0 = 0.0, gsum1 = 0.0;

  // Staging of one tile: every global load of the tile is issued before anything waits (k stays in registers, raw,
  // across the suffix-sum phase), so a tile costs one global round trip, not one per element.
  constexpr int KV8 = kDgTT * DK / 8 / kDgRows;  // 8-channel groups of k per thread
  constexpr int GV4 = CHANNEL ? kDgTT * DK / 4 / kDgRows : 1;
  auto stage = [&](int buf, int tile) {
    const int tbase = t_begin + tile * kDgTT;
    const int n_tok = min(kDgTT, t_end - tbase);
    uint4 kraw[KV8][BF16 ? 1 : 2];
#pragma unroll
    for (int n = 0; n < KV8; ++n) {
      const int e8 = tid + n * kDgRows;
      const int tok = (e8 * 8) / DK, c0 = (e8 * 8) % DK;
#pragma unroll
      for (int u = 0; u < (BF16 ? 1 : 2); ++u) kraw[n][u] = make_uint4(0u, 0u, 0u, 0u);
      if (tok < n_tok) {
        const size_t e0 = ((size_t)(tbase + tok) * H + h) * DK + c0;
        if (BF16) {
          kraw[n][0] = __ldg(reinterpret_cast<const uint4*>(reinterpret_cast<const __nv_bfloat16*>(k) + e0));
        } else {
#pragma unroll
          for (int u = 0; u < (BF16 ? 1 : 2); ++u)
            kraw[n][u] = __ldg(reinterpret_cast<const uint4*>(reinterpret_cast<const float*>(k) + e0) + u);
        }
      }
    }
    float vraw[kDgTT];
#pragma unroll
    for (int tok = 0; tok < kDgTT; ++tok)
      vraw[tok] = (tok < n_tok && row < dv) ? dg_load<BF16>(v, ((size_t)(tbase + tok) * H + h) * dv + row) : 0.f;
    if (CHANNEL) {
      float4 graw[GV4];
#pragma unroll
      for (int n = 0; n < GV4; ++n) {
        const int e4 = tid + n * kDgRows;
        const int tok = (e4 * 4) / DK, c0 = (e4 * 4) % DK;
        graw[n] = tok < n_tok ? __ldg(reinterpret_cast<const float4*>(g + ((size_t)(tbase + tok) * H + h) * DK + c0))
                              : make_float4(0.f, 0.f, 0.f, 0.f);
      }
#pragma unroll
      for (int n = 0; n < GV4; ++n) {
        const int e4 = tid + n * kDgRows;
        *reinterpret_cast<float4*>(&sg[(e4 * 4) / DK][(e4 * 4) % DK]) = graw[n];
      }
    } else if (tid < kDgTT) {
      sg[tid][0] = tid < n_tok ? g[(size_t)(tbase + tid) * H + h] : 0.f;
    }
#pragma unroll
    for (int tok = 0; tok < kDgTT; ++tok) sw[buf][tok][tid] = vraw[tok];
    __syncthreads();
    // suffix sums inside the tile, one thread per channel (or thread 0): weight of token t = exp(sum_{s > t} g_s)
    for (int c = tid; c < AW; c += kDgRows) {
      float suf = 0.f;
      double acc = 0.0;
#pragma unroll
      for (int tok = kDgTT - 1; tok >= 0; --tok) {
        const float gv = sg[tok][c];
        sg[tok][c] = suf;  // in place: now the log-weight of token tok
        suf += gv;
        acc += (double)gv;
      }
      sdec[buf][c] = expf(suf);
      if (c < kDgRows) gsum0 += acc; else gsum1 += acc;
    }
    __syncthreads();
#pragma unroll
    for (int n = 0; n < KV8; ++n) {
      const int e8 = tid + n * kDgRows;
      const int tok = (e8 * 8) / DK, c0 = (e8 * 8) % DK;
      float kv[8];
      if (BF16) {
        const uint32_t w4[4] = {kraw[n][0].x, kraw[n][0].y, kraw[n][0].z, kraw[n][0].w};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          kv[2 * u] = __uint_as_float(w4[u] << 16);
          kv[2 * u + 1] = __uint_as_float(w4[u] & 0xffff0000u);
        }
      } else {
#pragma unroll
        for (int u = 0; u < (BF16 ? 1 : 2); ++u) {
          kv[4 * u] = __uint_as_float(kraw[n][u].x), kv[4 * u + 1] = __uint_as_float(kraw[n][u].y);
          kv[4 * u + 2] = __uint_as_float(kraw[n][u].z), kv[4 * u + 3] = __uint_as_float(kraw[n][u].w);
        }
      }
      float wt[8];
      if (CHANNEL) {
        const float4 l0 = *reinterpret_cast<const float4*>(&sg[tok][c0]);
        const float4 l1 = *reinterpret_cast<const float4*>(&sg[tok][c0 + 4]);
        wt[0] = expf(l0.x), wt[1] = expf(l0.y), wt[2] = expf(l0.z), wt[3] = expf(l0.w);
        wt[4] = expf(l1.x), wt[5] = expf(l1.y), wt[6] = expf(l1.z), wt[7] = expf(l1.w);
      } else {
        const float w1 = expf(sg[tok][0]);
#pragma unroll
        for (int u = 0; u < 8; ++u) wt[u] = w1;
      }
      float4* d4 = reinterpret_cast<float4*>(&sk[buf][tok][c0]);
      d4[0] = make_float4(kv[0] * wt[0], kv[1] * wt[1], kv[2] * wt[2], kv[3] * wt[3]);
      d4[1] = make_float4(kv[4] * wt[4], kv[5] * wt[5], kv[6] * wt[6], kv[7] * wt[7]);
    }
  };

  const int n_tiles = (L + kDgTT - 1) / kDgTT;
  if (n_tiles > 0) stage(0, 0);
  __syncthreads();
  for (int tile = 0; tile < n_tiles; ++tile) {
    const int buf = tile & 1;
    // decay of the state over this tile, then the tile's writes
    if (CHANNEL) {
      const float4* d4 = reinterpret_cast<const float4*>(&sdec[buf][0]);
#pragma unroll
      for (int c4 = 0; c4 < DK / 4; ++c4) {
        const float4 dd = d4[c4];
        x[4 * c4 + 0] *= dd.x;
        x[4 * c4 + 1] *= dd.y;
        x[4 * c4 + 2] *= dd.z;
        x[4 * c4 + 3] *= dd.w;
      }
    } else {
      const float dd = sdec[buf][0];
#pragma unroll
      for (int c = 0; c < DK; ++c) x[c] *= dd;
    }
    const int n_tok = min(kDgTT, L - tile * kDgTT);
    for (int tok = 0; tok < n_tok; ++tok) {
      const float w = sw[buf][tok][tid];
      const float4* k4 = reinterpret_cast<const float4*>(&sk[buf][tok][0]);
#pragma unroll
      for (int c4 = 0; c4 < DK / 4; ++c4) {
        const float4 kk = k4[c4];
        x[4 * c4 + 0] = fmaf(w, kk.x, x[4 * c4 + 0]);
        x[4 * c4 + 1] = fmaf(w, kk.y, x[4 * c4 + 1]);
        x[4 * c4 + 2] = fmaf(w, kk.z, x[4 * c4 + 2]);
        x[4 * c4 + 3] = fmaf(w, kk.w, x[4 * c4 + 3]);
      }
    }
    __syncthreads();  // everyone is done with sg (staging scratch) and with buffer buf ^ 1 of the tile before
    if (tile + 1 < n_tiles) stage(buf ^ 1, tile + 1);
    __syncthreads();
  }

  if (row < dv) {
    float4* d4 = reinterpret_cast<float4*>(E + (((size_t)s * H + h) * dv + row) * DK);
#pragma unroll
    for (int c4 = 0; c4 < DK / 4; ++c4) d4[c4] = make_float4(x[4 * c4], x[4 * c4 + 1], x[4 * c4 + 2], x[4 * c4 + 3]);
  }
  if (blockIdx.x == 0) {
    float* tv = tvec + ((size_t)s * H + h) * AW;
    if (tid < AW) tv[tid] = (float)exp(gsum0);
    if (CHANNEL && tid + kDgRows < AW) tv[tid + kDgRows] = (float)exp(gsum1);
  }
}

template <int DK, bool BF16, bool CHANNEL>
int dg_launch(const DiagEncodeArgs& a) {
  dim3 grid((a.dv + kDgRows - 1) / kDgRows, a.H, a.n_seg);
  diag_encode_simt_kernel<DK, BF16, CHANNEL><<<grid, kDgRows, 0, a.stream>>>(a.k, a.v, a.g, a.cu_seqlens, a.H, a.dv,
                                                                            a.E, a.tvec);
  note_launch();
  HYPIC_CUDA_OK(cudaGetLastError());
  return HYPIC_OK;
}

template <int DK>
int dg_dispatch(const DiagEncodeArgs& a) {
  const bool bf = a.kv_dtype == HYPIC_DT_BF16, ch = a.gate == HYPIC_GATE_CHANNEL;
  if (bf) return ch ? dg_launch<DK, true, true>(a) : dg_launch<DK, true, false>(a);
  return ch ? dg_launch<DK, false, true>(a) : dg_launch<DK, false, false>(a);
}

// ------------------------------------------------------------------------------------------------ compose
constexpr int kDcThreads = 256;
constexpr int kDcV4 = 4;  // float4s of S per thread: a CTA owns 4,096 consecutive elements of one (request, head)

// TSH (diagonal family): dk/4 divides the CTA width, so the four float4s a thread owns sit in the same columns and share
// ONE float4 of the decay vector per step (otherwise each float4 fetches its own).
template <bool CHANNEL, bool F16, bool TSH = false>
__global__ void __launch_bounds__(kDcThreads, (CHANNEL && !TSH) ? 2 : 3)
    diag_compose_kernel(const float* S_in /* may alias S_out */, const void* __restrict__ E_pool,
                        const float* __restrict__ t_pool, const int32_t* __restrict__ seg_ids,
                        const int32_t* __restrict__ cu_segs, int H, int dk, int unit_v4, float* S_out) {
  const int tid = threadIdx.x;
  const int h = blockIdx.y, r = blockIdx.z;
  const size_t unit = (size_t)r * H + h;
  int e4[kDcV4];  // float4 index inside the unit's dv x dk block
  bool live[kDcV4];
#pragma unroll
  for (int i = 0; i < kDcV4; ++i) {
    e4[i] = (blockIdx.x * kDcV4 + i) * kDcThreads + tid;
    live[i] = e4[i] < unit_v4;
  }
  float4 x[kDcV4];
#pragma unroll
  for (int i = 0; i < kDcV4; ++i) {
    x[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (live[i] && S_in) x[i] = *(reinterpret_cast<const float4*>(S_in) + unit * unit_v4 + e4[i]);  // plain load: S_out may alias S_in
  }
  const int dk4 = dk / 4;
  const int j0 = cu_segs[r], j1 = cu_segs[r + 1];
  constexpr int kTn = (CHANNEL && !TSH) ? kDcV4 : 1;
  float4 e_nxt[kDcV4], t_nxt[kTn];  // scalar family: one decay per step (t_nxt[0].x)
  const int tcol = tid % dk4;       // TSH: the float4 column all of this thread's float4s share
  auto fetch = [&](int j) {
    const size_t ph = (size_t)seg_ids[j] * H + h;
#pragma unroll
    for (int i = 0; i < kDcV4; ++i) {
      if (live[i]) {
        if (F16) {  // fp16-stored end-states (the paper's cache precision): exact inputs; kept raw in
                    // the prefetch registers and widened at use, so the load is not consumed one instruction later
          const uint2 hv = __ldcs(reinterpret_cast<const uint2*>(E_pool) + ph * unit_v4 + e4[i]);
          e_nxt[i] = make_float4(__uint_as_float(hv.x), __uint_as_float(hv.y), 0.f, 0.f);
        } else {
          e_nxt[i] = __ldcs(reinterpret_cast<const float4*>(E_pool) + ph * unit_v4 + e4[i]);
        }
        if (CHANNEL && !TSH) t_nxt[i] = __ldg(reinterpret_cast<const float4*>(t_pool + ph * dk) + e4[i] % dk4);
      }
    }
    if (!CHANNEL) t_nxt[0].x = __ldg(t_pool + ph);
    if (CHANNEL && TSH) t_nxt[0] = __ldg(reinterpret_cast<const float4*>(t_pool + ph * dk) + tcol);
  };
  if (j0 < j1) fetch(j0);
  for (int j = j0; j < j1; ++j) {
    float4 e_cur[kDcV4], t_cur[kDcV4];
#pragma unroll
    for (int i = 0; i < kDcV4; ++i) {
      e_cur[i] = e_nxt[i];
      t_cur[i] = CHANNEL ? t_nxt[kTn > 1 ? i : 0] : make_float4(t_nxt[0].x, t_nxt[0].x, t_nxt[0].x, t_nxt[0].x);
    }
    if (j + 1 < j1) fetch(j + 1);
#pragma unroll
    for (int i = 0; i < kDcV4; ++i) {
      if (F16) {
        const uint32_t w0 = __float_as_uint(e_cur[i].x), w1 = __float_as_uint(e_cur[i].y);
        const float2 lo = __half22float2(*reinterpret_cast<const __half2*>(&w0));
        const float2 hi = __half22float2(*reinterpret_cast<const __half2*>(&w1));
        e_cur[i] = make_float4(lo.x, lo.y, hi.x, hi.y);
      }
      x[i].x = fmaf(x[i].x, t_cur[i].x, e_cur[i].x);
      x[i].y = fmaf(x[i].y, t_cur[i].y, e_cur[i].y);
      x[i].z = fmaf(x[i].z, t_cur[i].z, e_cur[i].z);
      x[i].w = fmaf(x[i].w, t_cur[i].w, e_cur[i].w);
    }
  }
#pragma unroll
  for (int i = 0; i < kDcV4; ++i)
    if (live[i]) __stcs(reinterpret_cast<float4*>(S_out) + unit * unit_v4 + e4[i], x[i]);
}

}  // namespace

int diag_encode(const DiagEncodeArgs& a) {
  if (a.H > 65535 || a.n_seg > 65535) return HYPIC_ERR_UNSUPPORTED;
  if (a.dv < 1 || a.dv > 1024) return HYPIC_ERR_UNSUPPORTED;
  if (a.n_seg == 0) return HYPIC_OK;
  if (a.dk == 128) return dg_dispatch<128>(a);
  if (a.dk == 64) return dg_dispatch<64>(a);
  return HYPIC_ERR_UNSUPPORTED;
}

int diag_compose(const DiagComposeArgs& a) {
  if (a.H > 65535 || a.R > 65535) return HYPIC_ERR_UNSUPPORTED;
  if (a.dk % 4 != 0) return HYPIC_ERR_UNSUPPORTED;
  if (a.R == 0) return HYPIC_OK;
  const int unit_v4 = a.dv * a.dk / 4;
  dim3 grid((unit_v4 + kDcThreads * kDcV4 - 1) / (kDcThreads * kDcV4), a.H, a.R);
  const bool ch = a.gate == HYPIC_GATE_CHANNEL;
  const bool tsh = ch && kDcThreads % (a.dk / 4) == 0;
  auto kern = a.e_f16 ? (ch ? (tsh ? diag_compose_kernel<true, true, true> : diag_compose_kernel<true, true>)
                            : diag_compose_kernel<false, true>)
                      : (ch ? (tsh ? diag_compose_kernel<true, false, true> : diag_compose_kernel<true, false>)
                            : diag_compose_kernel<false, false>);
  kern<<<grid, kDcThreads, 0, a.stream>>>(a.S_in, a.E_pool, a.t_pool, a.seg_ids, a.cu_segs, a.H, a.dk, unit_v4, a.S_out);
  note_launch();
  HYPIC_CUDA_OK(cudaGetLastError());
  return HYPIC_OK;
}

}  // namespace hypic
