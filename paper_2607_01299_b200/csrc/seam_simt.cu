// seam_simt.cu -- seam-window step (Fig. 8).
//
// A handful of uncached tokens (w = 8 by default) are pushed through a linear-attention layer from
// the running state in front of them: per token one step of PAPER.md:84 Eq. 2 and the read-out of PAPER.md:86-90,
//     x <- x diag(a_t);   x <- x + beta_t (v_t[i] - x.k_t) k_t^T;   o_t[i] = x.q_t          (row i of S, row convention)
// With w = 8 the state is read and written once (8 dk bytes per row) for 4 w dk = 32 dk fp32 operations per row, which
// on B200 puts the HBM time, the FMA time and the shared-memory/shuffle (MIO) time within a factor 1.5 of each other,
// so the layout is chosen to keep all three low (measured unit costs: LDS.128 = 4 cycles per warp whatever the address
// pattern repeats, SHFL = 1 cycle per warp):
//   * a thread owns a 4-row x (dk/8)-column block of S: 8 adjacent lanes share 4 rows, lane l holding the float4s
//     l, l+8, .. of each.  Every warp load / store instruction covers 4 rows x 128 contiguous bytes (whole lines), and
//     a token's k_t / q_t slices are fetched from shared memory once per 4 rows;
//   * the 4 row sums x.k_t of a lane group are reduced by a 4-shuffle reduce-scatter (each lane ends with one row's
//     sum), the write coefficient beta (v - x.k) is formed once per row and gathered back with 4 indexed shuffles; the
//     read-outs x.q_t need only the reduce-scatter and sit off the recurrence's dependency chain;
//   * k, q, a, beta, v of a tile of 8 tokens are staged in shared memory (double-buffered, so longer windows stream)
//     and o is written back through shared memory as whole rows.
// One CTA = 128 threads = 64 rows of one (request, head) unit; grid = ceil(dv / 64) x H x R.
#include <algorithm>

#include "common.cuh"

namespace hypic {
namespace {

constexpr int kSeamLanes = 8;    // lanes sharing a row group
constexpr int kSeamRT = 4;       // rows per thread
constexpr int kSeamThreads = 128;
constexpr int kSeamRows = kSeamThreads / kSeamLanes * kSeamRT;  // 64 rows of S per CTA
constexpr int kSeamTT = 8;       // tokens per staged tile (= the default seam width)

template <bool BF16>
__device__ __forceinline__ float seam_load(const void* p, size_t idx) {
  if (BF16) return __bfloat162float(reinterpret_cast<const __nv_bfloat16*>(p)[idx]);
  return reinterpret_cast<const float*>(p)[idx];
}

// 8 consecutive elements starting at element index idx (a multiple of 8) -> fp32
template <bool BF16>
__device__ __forceinline__ void seam_load8(const void* p, size_t idx, float (&out)[8]) {
  if (BF16) {
    const uint4 u = __ldg(reinterpret_cast<const uint4*>(reinterpret_cast<const __nv_bfloat16*>(p) + idx));
    const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      out[2 * i] = __uint_as_float(w[i] << 16);
      out[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
    }
  } else {
    const float4* f = reinterpret_cast<const float4*>(reinterpret_cast<const float*>(p) + idx);
    const float4 a = __ldg(f), b = __ldg(f + 1);
    out[0] = a.x, out[1] = a.y, out[2] = a.z, out[3] = a.w;
    out[4] = b.x, out[5] = b.y, out[6] = b.z, out[7] = b.w;
  }
}

// Reduce-scatter of 4 per-lane values over a group of 8 lanes (bits b0 b1 b2 of the lane): returns the full sum of
// value rho = 2 b0 + b1 (lanes l and l ^ 4 hold the same row).  4 shuffles.
__device__ __forceinline__ float group8_reduce_scatter4(const float (&d)[4], bool b0, bool b1) {
  const float s0 = b0 ? d[0] : d[2], s1 = b0 ? d[1] : d[3];
  const float k0 = b0 ? d[2] : d[0], k1 = b0 ? d[3] : d[1];
  const float r0 = k0 + __shfl_xor_sync(0xffffffffu, s0, 1);  // rows {2 b0, 2 b0 + 1} over lane pairs
  const float r1 = k1 + __shfl_xor_sync(0xffffffffu, s1, 1);
  const float snd = b1 ? r0 : r1, kp = b1 ? r1 : r0;
  float r = kp + __shfl_xor_sync(0xffffffffu, snd, 2);        // row 2 b0 + b1 over 4 lanes
  r += __shfl_xor_sync(0xffffffffu, r, 4);
  return r;
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)),
               "l"(gmem_src)
               : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// Raw (unconverted) inputs of one staged tile of 8 tokens, as the registers of one thread: loaded one tile ahead of
// their use, so the global latency is covered by the arithmetic of the tile in front.
template <bool BF16, bool CHANNEL>
struct SeamRaw {
  uint4 k[BF16 ? 1 : 2], q[BF16 ? 1 : 2];
  float4 g[CHANNEL ? 2 : 1];
  float v[kSeamTT * kSeamRows / kSeamThreads];
  float b, gs;
};

template <int DK, bool BF16, bool CHANNEL>
__global__ void __launch_bounds__(kSeamThreads, 3)
    seam_simt_kernel(const void* __restrict__ q, const void* __restrict__ k, const void* __restrict__ v,
                     const float* __restrict__ g, const float* __restrict__ beta, const int32_t* __restrict__ cu_tokens,
                     int H, int dv, int n_blk, int n_items, const float* S_in, float* S_out, float* __restrict__ o) {
  constexpr int AW = CHANNEL ? DK : 1;
  constexpr int NJ = DK / 32;                   // float4s of a row owned by one lane
  constexpr int NS = kSeamRT * NJ;              // float4s of S owned by one thread
  constexpr int NV = kSeamTT * kSeamRows / kSeamThreads;
  constexpr int EPT = 8;                        // k / q channels per thread and staged tile
  static_assert(kSeamTT * DK / EPT <= kSeamThreads, "one staging pass");
  extern __shared__ __align__(16) uint8_t seam_smem[];
  float4* xs = reinterpret_cast<float4*>(seam_smem);  // [NS][kSeamThreads]: prefetched rows of the NEXT item
  __shared__ __align__(16) float sk[kSeamTT][DK];
  __shared__ __align__(16) float sq[kSeamTT][DK];
  __shared__ __align__(16) float sa[kSeamTT][AW];
  __shared__ float sv[kSeamTT][kSeamRows];
  __shared__ float sb[kSeamTT];
  __shared__ float so[kSeamTT][kSeamRows];

  const int tid = threadIdx.x;
  const int l = tid % kSeamLanes;
  const int rloc0 = (tid / kSeamLanes) * kSeamRT;  // first of this thread's 4 rows, within the item's 64
  const bool b0 = l & 1, b1 = l & 2;
  const int rho = 2 * (l & 1) + ((l >> 1) & 1);     // the row of the 4 this lane owns after a reduce-scatter
  const bool stager = tid < kSeamTT * DK / EPT;
  const int st_tok = (tid * EPT) / DK, st_c0 = (tid * EPT) % DK;

  // item = (request r, head h, block of 64 rows blk), blk fastest
  auto prefetch_rows = [&](int item) {
    if (!S_in) return;
    const int blk = item % n_blk, unit = item / n_blk;
#pragma unroll
    for (int i = 0; i < kSeamRT; ++i) {
      const int row = blk * kSeamRows + rloc0 + i;
      if (row < dv) {
        const float4* src = reinterpret_cast<const float4*>(S_in + ((size_t)unit * dv + row) * DK);
#pragma unroll
        for (int j = 0; j < NJ; ++j) cp_async16(&xs[(i * NJ + j) * kSeamThreads + tid], src + l + kSeamLanes * j);
      }
    }
    cp_async_commit();
  };

  auto load_raw = [&](SeamRaw<BF16, CHANNEL>& raw, int item, int tile, int t_begin, int t_end) {
    const int blk = item % n_blk, h = (item / n_blk) % H;
    const int tbase = t_begin + tile * kSeamTT;
    if (stager) {
      const int t = tbase + st_tok;
      if (t < t_end) {
        const size_t e0 = ((size_t)t * H + h) * DK + st_c0;
        if (BF16) {
          raw.k[0] = __ldg(reinterpret_cast<const uint4*>(reinterpret_cast<const __nv_bfloat16*>(k) + e0));
          raw.q[0] = __ldg(reinterpret_cast<const uint4*>(reinterpret_cast<const __nv_bfloat16*>(q) + e0));
        } else {
#pragma unroll
          for (int i = 0; i < (BF16 ? 1 : 2); ++i) {
            raw.k[i] = __ldg(reinterpret_cast<const uint4*>(reinterpret_cast<const float*>(k) + e0) + i);
            raw.q[i] = __ldg(reinterpret_cast<const uint4*>(reinterpret_cast<const float*>(q) + e0) + i);
          }
        }
        if (CHANNEL) {
#pragma unroll
          for (int i = 0; i < (CHANNEL ? 2 : 1); ++i) raw.g[i] = __ldg(reinterpret_cast<const float4*>(g + e0) + i);
        }
      } else {
#pragma unroll
        for (int i = 0; i < (BF16 ? 1 : 2); ++i) raw.k[i] = raw.q[i] = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
        for (int i = 0; i < (CHANNEL ? 2 : 1); ++i) raw.g[i] = make_float4(0.f, 0.f, 0.f, 0.f);
      }
    }
#pragma unroll
    for (int n = 0; n < NV; ++n) {
      const int idx = tid + n * kSeamThreads;
      const int tok = idx / kSeamRows, j = idx % kSeamRows;
      const int t = tbase + tok, row = blk * kSeamRows + j;
      raw.v[n] = (t < t_end && row < dv) ? seam_load<BF16>(v, ((size_t)t * H + h) * dv + row) : 0.f;
    }
    raw.b = 0.f, raw.gs = 0.f;
    if (tid < kSeamTT && tbase + tid < t_end) {
      const size_t th = (size_t)(tbase + tid) * H + h;
      raw.b = beta[th];
      if (!CHANNEL) raw.gs = g[th];
    }
  };

  auto store_raw = [&](const SeamRaw<BF16, CHANNEL>& raw) {
    if (stager) {
      float kv[EPT], qv[EPT];
      if (BF16) {
        const uint32_t wk[4] = {raw.k[0].x, raw.k[0].y, raw.k[0].z, raw.k[0].w};
        const uint32_t wq[4] = {raw.q[0].x, raw.q[0].y, raw.q[0].z, raw.q[0].w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          kv[2 * i] = __uint_as_float(wk[i] << 16), kv[2 * i + 1] = __uint_as_float(wk[i] & 0xffff0000u);
          qv[2 * i] = __uint_as_float(wq[i] << 16), qv[2 * i + 1] = __uint_as_float(wq[i] & 0xffff0000u);
        }
      } else {
#pragma unroll
        for (int i = 0; i < (BF16 ? 1 : 2); ++i) {
          kv[4 * i] = __uint_as_float(raw.k[i].x), kv[4 * i + 1] = __uint_as_float(raw.k[i].y);
          kv[4 * i + 2] = __uint_as_float(raw.k[i].z), kv[4 * i + 3] = __uint_as_float(raw.k[i].w);
          qv[4 * i] = __uint_as_float(raw.q[i].x), qv[4 * i + 1] = __uint_as_float(raw.q[i].y);
          qv[4 * i + 2] = __uint_as_float(raw.q[i].z), qv[4 * i + 3] = __uint_as_float(raw.q[i].w);
        }
      }
      float4* dk4 = reinterpret_cast<float4*>(&sk[st_tok][st_c0]);
      float4* dq4 = reinterpret_cast<float4*>(&sq[st_tok][st_c0]);
      dk4[0] = make_float4(kv[0], kv[1], kv[2], kv[3]);
      dk4[1] = make_float4(kv[4], kv[5], kv[6], kv[7]);
      dq4[0] = make_float4(qv[0], qv[1], qv[2], qv[3]);
      dq4[1] = make_float4(qv[4], qv[5], qv[6], qv[7]);
      if (CHANNEL) {
        float4* da4 = reinterpret_cast<float4*>(&sa[st_tok][st_c0]);
#pragma unroll
        for (int i = 0; i < (CHANNEL ? 2 : 1); ++i)
          da4[i] = make_float4(expf(raw.g[i].x), expf(raw.g[i].y), expf(raw.g[i].z), expf(raw.g[i].w));
      }
    }
#pragma unroll
    for (int n = 0; n < NV; ++n) {
      const int idx = tid + n * kSeamThreads;
      sv[idx / kSeamRows][idx % kSeamRows] = raw.v[n];
    }
    if (tid < kSeamTT) {
      sb[tid] = raw.b;
      if (!CHANNEL) sa[tid][0] = expf(raw.gs);
    }
  };

  int item = blockIdx.x;
  if (item >= n_items) return;
  int t_begin = cu_tokens[item / (n_blk * H)], t_end = cu_tokens[item / (n_blk * H) + 1];
  SeamRaw<BF16, CHANNEL> raw;
  prefetch_rows(item);
  load_raw(raw, item, 0, t_begin, t_end);

  while (item < n_items) {
    const int blk = item % n_blk, unit = item / n_blk, h = unit % H;
    const int row0 = blk * kSeamRows;
    const int L = t_end - t_begin;
    const int n_tiles = (L + kSeamTT - 1) / kSeamTT;
    const int next = item + gridDim.x;
    int nt_begin = 0, nt_end = 0;
    if (next < n_items) {
      nt_begin = cu_tokens[next / (n_blk * H)];
      nt_end = cu_tokens[next / (n_blk * H) + 1];
    }

    float4 x[kSeamRT][NJ];
    cp_async_wait_all();
#pragma unroll
    for (int i = 0; i < kSeamRT; ++i) {
      const bool have = S_in && row0 + rloc0 + i < dv;
#pragma unroll
      for (int j = 0; j < NJ; ++j)
        x[i][j] = have ? xs[(i * NJ + j) * kSeamThreads + tid] : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    if (next < n_items) prefetch_rows(next);  // every thread refills only the slots it has just read
    if (n_tiles == 0 && next < n_items) load_raw(raw, next, 0, nt_begin, nt_end);

    for (int tile = 0; tile < n_tiles; ++tile) {
      store_raw(raw);
      __syncthreads();
      if (tile + 1 < n_tiles)
        load_raw(raw, item, tile + 1, t_begin, t_end);
      else if (next < n_items)
        load_raw(raw, next, 0, nt_begin, nt_end);
      const int n_tok = min(kSeamTT, L - tile * kSeamTT);
#pragma unroll 1
      for (int tok = 0; tok < n_tok; ++tok) {
        const float b = sb[tok];
        const float w = sv[tok][rloc0 + rho];
        const float4* k4 = reinterpret_cast<const float4*>(&sk[tok][0]);
        const float4* q4 = reinterpret_cast<const float4*>(&sq[tok][0]);
        float4 kk[NJ], qq[NJ];
#pragma unroll
        for (int j = 0; j < NJ; ++j) kk[j] = k4[l + kSeamLanes * j];
#pragma unroll
        for (int j = 0; j < NJ; ++j) qq[j] = q4[l + kSeamLanes * j];
        float a = 1.f;
        if (CHANNEL) {
          const float4* a4 = reinterpret_cast<const float4*>(&sa[tok][0]);
#pragma unroll
          for (int j = 0; j < NJ; ++j) {
            const float4 aa = a4[l + kSeamLanes * j];
#pragma unroll
            for (int i = 0; i < kSeamRT; ++i) {
              x[i][j].x *= aa.x;
              x[i][j].y *= aa.y;
              x[i][j].z *= aa.z;
              x[i][j].w *= aa.w;
            }
          }
        } else {
          a = sa[tok][0];
        }
        float d[kSeamRT];
#pragma unroll
        for (int i = 0; i < kSeamRT; ++i) {
          float d0 = 0.f, d1 = 0.f;
#pragma unroll
          for (int j = 0; j < NJ; ++j) {
            d0 = fmaf(x[i][j].x, kk[j].x, d0);
            d1 = fmaf(x[i][j].y, kk[j].y, d1);
            d0 = fmaf(x[i][j].z, kk[j].z, d0);
            d1 = fmaf(x[i][j].w, kk[j].w, d1);
          }
          d[i] = d0 + d1;
        }
        // decay first, then read the decayed state along k_t: (a x).k = a (x.k)  (a = 1 on the per-channel path,
        // where the state was decayed above)
        const float coef_own = b * (w - a * group8_reduce_scatter4(d, b0, b1));
        float p[kSeamRT];
#pragma unroll
        for (int i = 0; i < kSeamRT; ++i) {
          const float coef = __shfl_sync(0xffffffffu, coef_own, (i >> 1) + 2 * (i & 1), kSeamLanes);
          float p0 = 0.f, p1 = 0.f;  // this lane's share of o_t[row] = S_t[row,:] . q_t, read AFTER token t's write
#pragma unroll
          for (int j = 0; j < NJ; ++j) {
            if (CHANNEL) {
              x[i][j].x = fmaf(coef, kk[j].x, x[i][j].x);
              x[i][j].y = fmaf(coef, kk[j].y, x[i][j].y);
              x[i][j].z = fmaf(coef, kk[j].z, x[i][j].z);
              x[i][j].w = fmaf(coef, kk[j].w, x[i][j].w);
            } else {
              x[i][j].x = fmaf(coef, kk[j].x, a * x[i][j].x);
              x[i][j].y = fmaf(coef, kk[j].y, a * x[i][j].y);
              x[i][j].z = fmaf(coef, kk[j].z, a * x[i][j].z);
              x[i][j].w = fmaf(coef, kk[j].w, a * x[i][j].w);
            }
            p0 = fmaf(x[i][j].x, qq[j].x, p0);
            p1 = fmaf(x[i][j].y, qq[j].y, p1);
            p0 = fmaf(x[i][j].z, qq[j].z, p0);
            p1 = fmaf(x[i][j].w, qq[j].w, p1);
          }
          p[i] = p0 + p1;
        }
        const float ot = group8_reduce_scatter4(p, b0, b1);
        if (l < 4) so[tok][rloc0 + rho] = ot;
      }
      __syncthreads();
#pragma unroll
      for (int n = 0; n < NV; ++n) {
        const int idx = tid + n * kSeamThreads;
        const int tok = idx / kSeamRows, j = idx % kSeamRows;
        if (tok < n_tok && row0 + j < dv)
          o[((size_t)(t_begin + tile * kSeamTT + tok) * H + h) * dv + row0 + j] = so[tok][j];
      }
    }

#pragma unroll
    for (int i = 0; i < kSeamRT; ++i) {
      const int row = row0 + rloc0 + i;
      if (row < dv) {
        float4* dst = reinterpret_cast<float4*>(S_out + ((size_t)unit * dv + row) * DK);
#pragma unroll
        for (int j = 0; j < NJ; ++j) __stcs(dst + l + kSeamLanes * j, x[i][j]);
      }
    }
    item = next;
    t_begin = nt_begin, t_end = nt_end;
  }
}

template <int DK, bool BF16, bool CHANNEL>
int seam_launch(const SeamArgs& a) {
  const int n_blk = (a.dv + kSeamRows - 1) / kSeamRows;
  const long long n_items = (long long)n_blk * a.H * a.R;
  if (n_items > 0x7fffffffLL) return HYPIC_ERR_UNSUPPORTED;
  const DeviceInfo& di = device_info();
  if (!di.ok) return HYPIC_ERR_CUDA;
  constexpr int kDyn = kSeamRT * (DK / 32) * kSeamThreads * 16;  // prefetch buffer for the next item's rows
  auto kern = seam_simt_kernel<DK, BF16, CHANNEL>;
  static bool attr_set = false;  // per instantiation
  if (!attr_set) {
    HYPIC_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kDyn));
    attr_set = true;
  }
  const int grid = (int)std::min<long long>(n_items, 3LL * di.sm_count);
  kern<<<grid, kSeamThreads, kDyn, a.stream>>>(a.q, a.k, a.v, a.g, a.beta, a.cu_tokens, a.H, a.dv, n_blk, (int)n_items,
                                               a.S_in, a.S_out, a.o);
  note_launch();
  HYPIC_CUDA_OK(cudaGetLastError());
  return HYPIC_OK;
}

template <int DK>
int seam_dispatch(const SeamArgs& a) {
  const bool bf = a.kv_dtype == HYPIC_DT_BF16, ch = a.gate == HYPIC_GATE_CHANNEL;
  if (bf) return ch ? seam_launch<DK, true, true>(a) : seam_launch<DK, true, false>(a);
  return ch ? seam_launch<DK, false, true>(a) : seam_launch<DK, false, false>(a);
}

}  // namespace

int seam_simt(const SeamArgs& a) {
  if (a.H > 65535 || a.R > 65535) return HYPIC_ERR_UNSUPPORTED;
  if (a.dv < 1 || a.dv > 1024) return HYPIC_ERR_UNSUPPORTED;
  if (a.R == 0) return HYPIC_OK;
  if (a.dk == 128) return seam_dispatch<128>(a);
  if (a.dk == 64) return seam_dispatch<64>(a);
  return HYPIC_ERR_UNSUPPORTED;
}

}  // namespace hypic
