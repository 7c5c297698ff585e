// seam_simt.cu -- seam-window step (Fig. 8).
//
// A handful of uncached tokens (w = 8 by default) are pushed through a linear-attention layer from
// the running state in front of them: per token one step of PAPER.md:84 Eq. 2 and the read-out of PAPER.md:86-90,
//     x <- x diag(a_t);   x <- x + beta_t (v_t[i] - x.k_t) k_t^T;   o_t[i] = x.q_t          (row i of S, row convention)
// With w = 8 the state is read and written once (8 dk bytes per row) for about 3 w dk = 24 dk fp32 multiply-adds per
// row, which on B200 puts the HBM time (83 us for the bench batch), the FMA-pipe time (~45 us) and the shared-memory /
// shuffle (MIO) time (~50 us) within a factor two of each other, so the layout keeps all three low and overlaps them
// (measured unit costs: LDS.128 = 4 cycles per warp whether or not quarter-warps repeat an address, SHFL = 1 cycle):
//   * a thread owns a 4-row x (dk/8)-column block of S: 8 adjacent lanes share 4 rows, lane l holding the float4s
//     l, l+8, .. of each.  Every warp load / store instruction covers 4 rows x 128 contiguous bytes (whole lines), and
//     a token's k_t / q_t slices are fetched from shared memory once per 4 rows;
//   * the 4 row sums x.k_t of a lane group are reduced by a 4-shuffle reduce-scatter (each lane ends with one row's
//     sum), the write coefficient beta (v - x.k) is formed once per row and gathered back with 4 indexed shuffles; the
//     read-outs x.q_t need only the reduce-scatter and sit off the recurrence's dependency chain;
//   * the arithmetic is packed fp32 (FFMA2 / FMUL2: two columns per instruction, half the issue slots); with a scalar
//     gate a tile of 8 tokens runs on y = x / gamma_t, which removes the per-token decay multiply (see FOLD below);
//   * persistent CTAs (3-4 per SM) walk the (request, head, 64-row block) items: the next item's rows of S_in are
//     prefetched into shared memory with cp.async while the current item computes (each thread refills only the slots
//     it reads itself, so no barrier guards them), the next tile's k, q, v, g, beta are loaded into registers one tile
//     ahead and converted / stored to shared memory when their turn comes, and o leaves through shared memory as
//     whole rows.
// One CTA = 128 threads; one item = 64 rows of one (request, head) unit.
//
// The same kernel is the fp32 "encode folded into the forward" pass (at cache
// time the segment's normal prefill also accumulates T_C): with T_out given, the rows of the stacked state [S ; T] are
// walked, T rows starting at the identity and taking no value term, so one pass over the tokens emits the per-token
// outputs o, the end-state E (= S_out from a zero start) and T.
#include <algorithm>
#include <type_traits>

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
  uint32_t v[kSeamTT * kSeamRows / kSeamThreads];  // bf16 bits or fp32 bits
  float b, gs;
};

template <int DK, bool BF16, bool CHANNEL, bool WITH_T>
__global__ void __launch_bounds__(kSeamThreads, CHANNEL ? 3 : 4)
    seam_simt_kernel(const void* __restrict__ q, const void* __restrict__ k, const void* __restrict__ v,
                     const float* __restrict__ g, const float* __restrict__ beta, const int32_t* __restrict__ cu_tokens,
                     int H, int dv, int n_blk, int n_items, const float* S_in, float* S_out, float* __restrict__ o,
                     float* __restrict__ T_out) {
  constexpr int AW = CHANNEL ? DK : 1;
  constexpr int NJ = DK / 32;                   // float4s of a row owned by one lane
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
  __shared__ float sgam[kSeamTT], sgi[kSeamTT];  // scalar gate: gamma_t since the tile's first token, and 1 / gamma_t
  __shared__ int s_fold;
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
      raw.v[n] = 0u;
      if (t < t_end && row < dv) {
        const size_t e = ((size_t)t * H + h) * dv + row;
        raw.v[n] = BF16 ? (uint32_t) reinterpret_cast<const uint16_t*>(v)[e] : reinterpret_cast<const uint32_t*>(v)[e];
      }
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
      sv[idx / kSeamRows][idx % kSeamRows] = __uint_as_float(BF16 ? raw.v[n] << 16 : raw.v[n]);
    }
    if (tid < kSeamTT) {
      sb[tid] = raw.b;
      if (!CHANNEL) {
        sa[tid][0] = expf(raw.gs);
        float G = raw.gs;  // inclusive prefix sum of the log-decay over the tile's tokens (lanes 0..7 of warp 0)
#pragma unroll
        for (int sft = 1; sft < kSeamTT; sft *= 2) {
          const float up = __shfl_up_sync((1u << kSeamTT) - 1u, G, sft);
          if (tid >= sft) G += up;
        }
        sgam[tid] = expf(G);
        sgi[tid] = expf(-G);
        const int ok = __all_sync((1u << kSeamTT) - 1u, fabsf(G) <= 40.f);  // false for NaN as well
        if (tid == 0) s_fold = ok;
      }
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
      const int row = row0 + rloc0 + i;
      const bool have = S_in && row < dv;
      // forward-encode mode (T_out != NULL): rows [dv, dv + dk) are the rows of T, which start at the identity
      const int m = (WITH_T && row >= dv) ? row - dv : -1;
#pragma unroll
      for (int j = 0; j < NJ; ++j) {
        const int c0 = 4 * (l + kSeamLanes * j);
        x[i][j] = have ? xs[(i * NJ + j) * kSeamThreads + tid]
                       : make_float4(m == c0 ? 1.f : 0.f, m == c0 + 1 ? 1.f : 0.f, m == c0 + 2 ? 1.f : 0.f,
                                     m == c0 + 3 ? 1.f : 0.f);
      }
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
      // FOLD (scalar gate only): the tile is run on y = x / gamma_t, gamma_t the decay accumulated since the tile's
      // first token, so the per-token decay of the state (one multiply per element) disappears:
      //     y += beta (v / gamma_t - y.k) k,   o_t = gamma_t (y.q),   x = gamma_8 y at the end of the tile.
      // Taken only while gamma_8 >= e^-40 (store_raw decides per tile); otherwise the plain form below runs.
      auto run_tokens = [&](auto fold_tag) {
        constexpr bool FOLD = decltype(fold_tag)::value;
#pragma unroll 2
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
                const float2 x01 = __fmul2_rn(make_float2(x[i][j].x, x[i][j].y), make_float2(aa.x, aa.y));
                const float2 x23 = __fmul2_rn(make_float2(x[i][j].z, x[i][j].w), make_float2(aa.z, aa.w));
                x[i][j] = make_float4(x01.x, x01.y, x23.x, x23.y);
              }
            }
          } else if (!FOLD) {
            a = sa[tok][0];
          }
          // packed fp32 (FFMA2): two columns per instruction, which halves the issue slots of the arithmetic
          float d[kSeamRT];
#pragma unroll
          for (int i = 0; i < kSeamRT; ++i) {
            float2 d01 = make_float2(0.f, 0.f), d23 = make_float2(0.f, 0.f);
#pragma unroll
            for (int j = 0; j < NJ; ++j) {
              d01 = __ffma2_rn(make_float2(x[i][j].x, x[i][j].y), make_float2(kk[j].x, kk[j].y), d01);
              d23 = __ffma2_rn(make_float2(x[i][j].z, x[i][j].w), make_float2(kk[j].z, kk[j].w), d23);
            }
            d[i] = (d01.x + d01.y) + (d23.x + d23.y);
          }
          // decay first, then read the decayed state along k_t: (a x).k = a (x.k)  (a = 1 on the per-channel path,
          // where the state was decayed above, and on the folded path, where v is divided by gamma_t instead)
          const float dsum = group8_reduce_scatter4(d, b0, b1);
          const float coef_own = FOLD ? b * (w * sgi[tok] - dsum) : b * (w - a * dsum);
          const float2 a2 = make_float2(a, a);
          float p[kSeamRT];
#pragma unroll
          for (int i = 0; i < kSeamRT; ++i) {
            const float coef = __shfl_sync(0xffffffffu, coef_own, (i >> 1) + 2 * (i & 1), kSeamLanes);
            const float2 c2 = make_float2(coef, coef);
            // this lane's share of o_t[row] = S_t[row,:] . q_t, read AFTER token t's write
            float2 p01 = make_float2(0.f, 0.f), p23 = make_float2(0.f, 0.f);
#pragma unroll
            for (int j = 0; j < NJ; ++j) {
              float2 x01 = make_float2(x[i][j].x, x[i][j].y), x23 = make_float2(x[i][j].z, x[i][j].w);
              if (!CHANNEL && !FOLD) {
                x01 = __fmul2_rn(a2, x01);
                x23 = __fmul2_rn(a2, x23);
              }
              x01 = __ffma2_rn(c2, make_float2(kk[j].x, kk[j].y), x01);
              x23 = __ffma2_rn(c2, make_float2(kk[j].z, kk[j].w), x23);
              p01 = __ffma2_rn(x01, make_float2(qq[j].x, qq[j].y), p01);
              p23 = __ffma2_rn(x23, make_float2(qq[j].z, qq[j].w), p23);
              x[i][j] = make_float4(x01.x, x01.y, x23.x, x23.y);
            }
            p[i] = (p01.x + p01.y) + (p23.x + p23.y);
          }
          float ot = group8_reduce_scatter4(p, b0, b1);
          if (FOLD) ot *= sgam[tok];
          if (l < 4) so[tok][rloc0 + rho] = ot;
        }
        if (FOLD) {
          const float gt = sgam[n_tok - 1];
          const float2 g2 = make_float2(gt, gt);
#pragma unroll
          for (int i = 0; i < kSeamRT; ++i)
#pragma unroll
            for (int j = 0; j < NJ; ++j) {
              const float2 x01 = __fmul2_rn(g2, make_float2(x[i][j].x, x[i][j].y));
              const float2 x23 = __fmul2_rn(g2, make_float2(x[i][j].z, x[i][j].w));
              x[i][j] = make_float4(x01.x, x01.y, x23.x, x23.y);
            }
        }
      };
      if (!CHANNEL && s_fold)
        run_tokens(std::true_type{});
      else
        run_tokens(std::false_type{});
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
      float* base = nullptr;
      if (row < dv)
        base = S_out + ((size_t)unit * dv + row) * DK;
      else if (WITH_T && row < dv + DK)
        base = T_out + ((size_t)unit * DK + (row - dv)) * DK;
      if (base) {
        float4* dst = reinterpret_cast<float4*>(base);
#pragma unroll
        for (int j = 0; j < NJ; ++j) __stcs(dst + l + kSeamLanes * j, x[i][j]);
      }
    }
    item = next;
    t_begin = nt_begin, t_end = nt_end;
  }
}

template <int DK, bool BF16, bool CHANNEL, bool WITH_T>
int seam_launch(const SeamArgs& a) {
  const int n_blk = (a.dv + (WITH_T ? DK : 0) + kSeamRows - 1) / kSeamRows;  // rows of [S ; T]
  const long long n_items = (long long)n_blk * a.H * a.R;
  if (n_items > 0x7fffffffLL) return HYPIC_ERR_UNSUPPORTED;
  const DeviceInfo& di = device_info();
  if (!di.ok) return HYPIC_ERR_CUDA;
  constexpr int kDyn = kSeamRT * (DK / 32) * kSeamThreads * 16;  // prefetch buffer for the next item's rows
  auto kern = seam_simt_kernel<DK, BF16, CHANNEL, WITH_T>;
  static bool attr_set = false;  // per instantiation
  if (!attr_set) {
    HYPIC_CUDA_OK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, kDyn));
    attr_set = true;
  }
  const int grid = (int)std::min<long long>(n_items, (CHANNEL ? 3LL : 4LL) * di.sm_count);
  kern<<<grid, kSeamThreads, kDyn, a.stream>>>(a.q, a.k, a.v, a.g, a.beta, a.cu_tokens, a.H, a.dv, n_blk, (int)n_items,
                                               a.S_in, a.S_out, a.o, a.T_out);
  note_launch();
  HYPIC_CUDA_OK(cudaGetLastError());
  return HYPIC_OK;
}

template <int DK, bool WITH_T>
int seam_dispatch(const SeamArgs& a) {
  const bool bf = a.kv_dtype == HYPIC_DT_BF16, ch = a.gate == HYPIC_GATE_CHANNEL;
  if (bf) return ch ? seam_launch<DK, true, true, WITH_T>(a) : seam_launch<DK, true, false, WITH_T>(a);
  return ch ? seam_launch<DK, false, true, WITH_T>(a) : seam_launch<DK, false, false, WITH_T>(a);
}

}  // namespace

int seam_simt(const SeamArgs& a) {
  if (a.H > 65535 || a.R > 65535) return HYPIC_ERR_UNSUPPORTED;
  if (a.dv < 1 || a.dv > 1024) return HYPIC_ERR_UNSUPPORTED;
  if (a.R == 0) return HYPIC_OK;
  if (a.dk == 128) return a.T_out ? seam_dispatch<128, true>(a) : seam_dispatch<128, false>(a);
  if (a.dk == 64) return a.T_out ? seam_dispatch<64, true>(a) : seam_dispatch<64, false>(a);
  return HYPIC_ERR_UNSUPPORTED;
}

}  // namespace hypic
