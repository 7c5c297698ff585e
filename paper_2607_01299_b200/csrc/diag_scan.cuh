// diag_scan.cuh -- scalar-family segment encode on the tensor cores (included by encode_tensor.cu, whose TMA / wait /
// packing helpers it shares).  PAPER.md:57-61 (Table 1, scalar family): S <- a_t S + v_t k_t^T, a_t = exp(g_t); per
// (segment, head) the zero-start end-state is ONE weighted contraction over the segment's tokens,
//     E = sum_t w_t v_t k_t^T = V^t diag(w) K,     w_t = prod_{s > t} a_s = exp(sum_{s > t} g_s)  in (0, 1],
// and T_C = (prod_t a_t) I is kept as the scalar tvec (Table 3).  There is no state-dependent step,
// so unlike the dense family nothing is sequential: the segment is streamed in chunks of 64 tokens, LAST chunk first,
// with the log-decay of all later tokens carried along (the weights are then known when a chunk arrives, never exceed 1,
// and tokens whose weight underflows fp16 contribute less than 6e-8 of the newest ones).  The arithmetic is 2 dk dv =
// 32,768 flop per token-head against 516 B of k, v, g: 64 flop/B, i.e. HBM-bound on B200 as long as the contraction
// runs on tcgen05 (the fp32 CUDA-core kernel of diag_family.cu is FMA-bound, six times slower).
//
// Roles of a CTA (320 threads, one (segment, head) unit, two CTAs per SM, 128 TMEM columns each):
//   warp 9      loader      TMA boxes of the bf16 K and V chunk tiles (64 tokens x 128 channels each), 3 stages, and the
//                           chunk's token weights (shuffle suffix scan of g, fp64 carry) -- up to 3 chunks ahead
//   warps 0-7   converters  in place: K~ = fp16(w_t k_t), V -> fp16, rows past the end of the segment zeroed; epilogue
//   warp 8      issuer      4 x tcgen05.mma (M = dv = 128, N = dk = 128, K = 16 tokens) per chunk, both operands
//                           MN-major straight from the swizzled boxes; accumulator E (fp32) stays in TMEM throughout
#pragma once

constexpr int kDtConvWarps = 8;
constexpr int kDtThreads = 32 * (kDtConvWarps + 2);  // converters, then the MMA issuer warp, then the loader warp
constexpr int kDtStages = 2;
constexpr int kDtStageBytes = 32768;  // K tile (2 boxes of 8 KB) + V tile
constexpr int kDtOffW = kDtStages * kDtStageBytes;        // per-stage token weights: float[kDtStages][64]
constexpr int kDtOffBar = kDtOffW + kDtStages * 64 * 4;
constexpr int kDtSmem = kDtOffBar + 128 + 1024;

struct DtBars {
  uint64_t full[kDtStages], conv[kDtStages], free_[kDtStages], done;
  double peer_g;  // split kernels: the peer CTA's total log-decay, written through distributed shared memory
  uint32_t tmem_base;
  int abort_flag;
};

__device__ __forceinline__ void cluster_arrive_release() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait_acquire() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
// store a double into the same shared-memory variable of CTA `rank` of this cluster
__device__ __forceinline__ void st_cluster_f64(double* local_smem_ptr, uint32_t rank, double v) {
  uint32_t remote;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(smem_u32(local_smem_ptr)), "r"(rank));
  asm volatile("st.shared::cluster.f64 [%0], %1;" ::"r"(remote), "d"(v) : "memory");
}

// Single-thread wait of the loader / issuer: mbarrier.try_wait already suspends the thread for a hardware-chosen time, so
// a plain retry loop reacts within tens of cycles; s2_wait's __nanosleep back-off (measured here: the loader woke up
// ~2,400 cycles after the stage had been freed, once per chunk) is only the bounded fallback.
__device__ __forceinline__ void dt_wait(uint64_t* bar, uint32_t parity, volatile int* abort_flag) {
#pragma unroll 1
  for (int i = 0; i < 4096; ++i)
    if (mbar_try_wait(bar, parity)) return;
  s2_wait(bar, parity, abort_flag);
}

// lds128 / sts128: encode_scan2.cuh

// Longest segments first (CTAs are handed out in index order, so the last ones set the tail of a launch with ragged
// segments): the segment of rank blockIdx.y by length, ties by index; every CTA ranks the n_seg <= 512 lengths itself in
// shared memory.  `scratch` (>= 2 KB + 4 B) is free until the pipeline starts; beyond 512 segments, index order.
__device__ __forceinline__ int dt_pick_segment(const int32_t* __restrict__ cu_seqlens, int n_seg, int* scratch) {
  int s = blockIdx.y;
  if (n_seg > 512) return s;
  int* s_len = scratch;
  int* s_pick = scratch + 512;
  for (int t = threadIdx.x; t < n_seg; t += blockDim.x) s_len[t] = cu_seqlens[t + 1] - cu_seqlens[t];
  __syncthreads();
  for (int t = threadIdx.x; t < n_seg; t += blockDim.x) {
    const int lt = s_len[t];
    int rank = 0;
    for (int j = 0; j < n_seg; ++j) {
      const int lj = s_len[j];
      rank += (lj > lt || (lj == lt && j < t)) ? 1 : 0;
    }
    if (rank == s) *s_pick = t;
  }
  __syncthreads();
  s = *s_pick;
  __syncthreads();
  return s;
}

// kSplit = 2: the unit is shared by a cluster of two CTAs (blockIdx.z = rank): rank 1 streams the later half of the chunks
// and writes its sum E_1 to the unit's place in E; rank 0 streams the earlier half with weights relative to ITS last
// token, learns rank 1's total log-decay G_1 through distributed shared memory, and after the cluster barrier writes
// E = exp(G_1) E_0 + E_1 in a fixed order (deterministic; no workspace, no atomics).  Twice the CTAs of half the length:
// 2.9 waves of 32 chunks instead of 1.44 waves of 64 on the cfg2-shaped layer, and twice the parallelism when units are few.
template <int kSplit>
__device__ __forceinline__ void diag_scan_body(const CUtensorMap& tmK, const CUtensorMap& tmV, const float* __restrict__ g,
                                               const int32_t* __restrict__ cu_seqlens, int H, float* E,
                                               float* __restrict__ tvec) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  DtBars* bars = reinterpret_cast<DtBars*>(smem + kDtOffBar);
  float* sw = reinterpret_cast<float*>(smem + kDtOffW);
  volatile int* abort_flag = &bars->abort_flag;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int h = blockIdx.x;
  const int s = dt_pick_segment(cu_seqlens, (int)gridDim.y, reinterpret_cast<int*>(smem));  // stage 0 is still empty
  const int seg_begin = cu_seqlens[s], seg_end = cu_seqlens[s + 1];
  const int nc_tot = (seg_end - seg_begin + kC - 1) / kC;
  const int rank = kSplit == 2 ? (int)blockIdx.z : 0;
  const int c_lo = (kSplit == 2 && rank == 1) ? nc_tot / 2 : 0;           // this CTA's chunks [c_lo, c_hi) of the segment
  const int c_hi = (kSplit == 2 && rank == 0) ? nc_tot / 2 : nc_tot;
  const int nc = c_hi - c_lo;
  float* Eu = E + ((size_t)s * H + h) * kD * kD;
  // (an empty range runs no pipeline iteration and contributes E = 0, log-decay 0; nobody returns before the cluster barrier)

  if (warp == kDtConvWarps) tmem_alloc(&bars->tmem_base, 128);
  if (tid == 0) {
    for (int i = 0; i < kDtStages; ++i) {
      mbar_init(&bars->full[i], 2);  // TMA bytes (expect_tx arrival) + the loader warp's weights
      mbar_init(&bars->conv[i], kDtConvWarps);
      mbar_init(&bars->free_[i], 1);
    }
    mbar_init(&bars->done, 1);
    bars->abort_flag = 0;
    fence_barrier_init();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  if (kSplit == 2) {  // both CTAs of the pair are running before either touches the other's shared memory
    cluster_arrive_release();
    cluster_wait_acquire();
  }
  const uint32_t tmem = bars->tmem_base;
  const uint32_t smem_base = smem_u32(smem);

  if (warp == kDtConvWarps + 1) {
    // ------------------------------------------------------------------------------- loader + token weights
    // Runs up to kDtStages chunks ahead of the converters, so neither the TMA latency nor the latency of the g loads
    // sits on anybody's critical path.  full[st] completes on the TMA bytes AND this warp's second arrival (weights).
    double carry = 0.0;   // log-decay of all tokens after the current chunk
    double lane_sum = 0.0;  // this lane's share of the segment's total log-decay, fp64 (tvec sums thousands of terms)
    // g of tokens 2 lane, 2 lane + 1 of a chunk, loaded two chunks ahead of its use
    auto load_g = [&](int i, float& ga, float& gb) {
      ga = gb = 0.f;
      if (i < nc) {
        const int ta = seg_begin + (c_hi - 1 - i) * kC + 2 * lane;
        if (ta < seg_end) ga = __ldg(g + (size_t)ta * H + h);
        if (ta + 1 < seg_end) gb = __ldg(g + (size_t)(ta + 1) * H + h);
      }
    };
    float ga0, gb0, ga1, gb1;
    load_g(0, ga0, gb0);
    load_g(1, ga1, gb1);
#pragma unroll 1
    for (int i = 0; i < nc; ++i) {
      const int st = i % kDtStages;
      const int t0 = seg_begin + (c_hi - 1 - i) * kC;  // last chunk first
      const int ta = t0 + 2 * lane, tb = ta + 1;
      const float ga = ga0, gb = gb0;
      ga0 = ga1, gb0 = gb1;
      load_g(i + 2, ga1, gb1);
      // envelope: the fp16 weights assume log-decays <= 0 (and finite); a chunk that breaks this is counted, like the dense
      // family's violations (hypic_envelope_violation_count), and should be re-run on the fp32 kernel
      if (__any_sync(0xffffffffu, !(ga <= 0.f) || !(gb <= 0.f)) && lane == 0) atomicAdd(&g_envelope_count_enc, 1u);
      if (i >= kDtStages) {
        if (lane == 0) dt_wait(&bars->free_[st], ((i / kDtStages) & 1) ^ 1, abort_flag);
        __syncwarp();
      }
      if (lane == 0) {
        const uint32_t sb = smem_base + st * kDtStageBytes;
        mbar_expect_tx(&bars->full[st], (uint32_t)kDtStageBytes);
        tma_load_3d(sb, &tmK, 0, h, t0, &bars->full[st]);
        tma_load_3d(sb + 8192, &tmK, 64, h, t0, &bars->full[st]);
        tma_load_3d(sb + 16384, &tmV, 0, h, t0, &bars->full[st]);
        tma_load_3d(sb + 24576, &tmV, 64, h, t0, &bars->full[st]);
      }
      // exclusive suffix sums of g inside the chunk by a shuffle scan over the lane pairs
      float suf = ga + gb;  // becomes the inclusive suffix sum over lanes >= lane
#pragma unroll
      for (int d = 1; d < 32; d *= 2) {
        const float up = __shfl_down_sync(0xffffffffu, suf, d);
        if (lane + d < 32) suf += up;
      }
      const float tot = __shfl_sync(0xffffffffu, suf, 0);
      const float excl = suf - (ga + gb);  // tokens of the lanes above
      const float cf = (float)carry;
      float* w = sw + st * 64;
      w[2 * lane + 1] = tb < seg_end ? __expf(cf + excl) : 0.f;
      w[2 * lane] = ta < seg_end ? __expf(cf + excl + gb) : 0.f;
      carry += (double)tot;
      lane_sum += (double)ga + (double)gb;
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars->full[st]);
    }
#pragma unroll
    for (int d = 16; d > 0; d /= 2) lane_sum += __shfl_xor_sync(0xffffffffu, lane_sum, d);
    if (kSplit == 1) {
      if (lane == 0) tvec[(size_t)s * H + h] = (float)exp(lane_sum);
    } else {
      if (rank == 1 && lane == 0) st_cluster_f64(&bars->peer_g, 0, lane_sum);  // into rank 0's shared memory
      cluster_arrive_release();
      cluster_wait_acquire();
      if (rank == 0 && lane == 0) tvec[(size_t)s * H + h] = (float)exp(lane_sum + bars->peer_g);
    }
  } else if (warp == kDtConvWarps) {
    // ----------------------------------------------------------------------------------------------- MMA issuer
    if (lane == 0) {
      constexpr uint32_t idesc = make_idesc(0u, 128, 128, 1, 1);  // fp16 x fp16 -> fp32, A (V tile) and B (K~ tile) MN-major
#pragma unroll 1
      for (int i = 0; i < nc; ++i) {
        const int st = i % kDtStages;
        dt_wait(&bars->conv[st], (i / kDtStages) & 1, abort_flag);
        tc_fence_after();
        const uint32_t sb = smem_base + st * kDtStageBytes;
#pragma unroll
        for (int ks = 0; ks < 4; ++ks)
          mma_f16_ss(tmem, make_desc(sb + 16384 + ks * 2048, 8192, 1024, 2), make_desc(sb + ks * 2048, 8192, 1024, 2),
                     idesc, (i > 0 || ks > 0) ? 1u : 0u);
        mma_commit(&bars->free_[st]);
      }
      if (nc > 0) mma_commit(&bars->done);
    }
    if (kSplit == 2) {
      cluster_arrive_release();
      cluster_wait_acquire();
    }
  } else {
    // ----------------------------------------------------------------------------------------------- converters
#pragma unroll 1
    for (int i = 0; i < nc; ++i) {
      const int st = i % kDtStages;
      const int t0 = seg_begin + (c_hi - 1 - i) * kC;
      s2_wait_warp(&bars->full[st], (i / kDtStages) & 1, abort_flag, lane);
      const float* w = sw + st * 64;
      const uint32_t tile = smem_base + st * kDtStageBytes;
      // 2,048 16-byte vectors: K boxes [0, 1024), V boxes [1024, 2048); vector idx of a box sits in token row (idx % 512) / 8
      constexpr int kConvThreads = 32 * kDtConvWarps;
#pragma unroll
      for (int it = 0; it < 2048 / kConvThreads; ++it) {
        const int idx = it * kConvThreads + tid;
        const int tok = (idx & 511) >> 3;
        const float m = it < 1024 / kConvThreads ? w[tok] : 1.f;
        uint4 x = lds128(tile + 16 * idx);
        x.x = pack_f16(m * __uint_as_float(x.x << 16), m * __uint_as_float(x.x & 0xffff0000u));
        x.y = pack_f16(m * __uint_as_float(x.y << 16), m * __uint_as_float(x.y & 0xffff0000u));
        x.z = pack_f16(m * __uint_as_float(x.z << 16), m * __uint_as_float(x.z & 0xffff0000u));
        x.w = pack_f16(m * __uint_as_float(x.w << 16), m * __uint_as_float(x.w & 0xffff0000u));
        if (t0 + tok >= seg_end) x = make_uint4(0u, 0u, 0u, 0u);  // rows past the segment hold other tokens' data
        sts128(tile + 16 * idx, x);
      }
      fence_proxy_async();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars->conv[st]);
    }
    // ----------------------------------------------------------------------------------------------- epilogue
    if (nc > 0) {
      s2_wait_warp(&bars->done, 0, abort_flag, lane);
      tc_fence_after();
    }
    const int q = warp & 3, hf = warp >> 2;  // TMEM lane quarter of this warp; column slice (two warps per quarter)
    const int row = 32 * q + lane;           // dv index = TMEM lane
    constexpr int kColsPerWarp = kD / (kDtConvWarps / 4);
    float4* dst = reinterpret_cast<float4*>(Eu + (size_t)row * kD + kColsPerWarp * hf);
    float scale = 1.f;
    if (kSplit == 2 && rank == 0) {
      cluster_arrive_release();
      cluster_wait_acquire();  // rank 1's E_1 is in global memory, its log-decay in bars->peer_g
      scale = expf((float)bars->peer_g);
    }
    const bool add_peer = kSplit == 2 && rank == 0;
    if (!(add_peer && nc == 0)) {  // (rank 0 with no chunks: E = E_1 is already in place)
#pragma unroll 1
      for (int cb = 0; cb < kColsPerWarp / 32; ++cb) {
        uint32_t x[32];
        if (nc > 0) {
          tmem_ld32(tmem + ((uint32_t)(32 * q) << 16) + kColsPerWarp * hf + 32 * cb, x);
          tmem_ld_wait();
        } else {
#pragma unroll
          for (int u = 0; u < 32; ++u) x[u] = 0u;
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) {
          float4 o4 = make_float4(__uint_as_float(x[4 * u]), __uint_as_float(x[4 * u + 1]), __uint_as_float(x[4 * u + 2]),
                                  __uint_as_float(x[4 * u + 3]));
          if (add_peer) {
            const float4 p4 = dst[8 * cb + u];  // plain load: written by the peer CTA during this kernel
            o4 = make_float4(fmaf(scale, o4.x, p4.x), fmaf(scale, o4.y, p4.y), fmaf(scale, o4.z, p4.z),
                             fmaf(scale, o4.w, p4.w));
          }
          dst[8 * cb + u] = o4;
        }
      }
    }
    if (kSplit == 2 && rank == 1) {
      cluster_arrive_release();  // E_1 written
      cluster_wait_acquire();
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kDtConvWarps) tmem_dealloc(tmem, 128);
}


__global__ void __launch_bounds__(kDtThreads, 3)
    diag_scan_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                     const float* __restrict__ g, const int32_t* __restrict__ cu_seqlens, int H, float* E,
                     float* __restrict__ tvec) {
  diag_scan_body<1>(tmK, tmV, g, cu_seqlens, H, E, tvec);
}

__global__ void __cluster_dims__(1, 1, 2) __launch_bounds__(kDtThreads, 3)
    diag_scan_split2_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                            const float* __restrict__ g, const int32_t* __restrict__ cu_seqlens, int H, float* E,
                            float* __restrict__ tvec) {
  diag_scan_body<2>(tmK, tmV, g, cu_seqlens, H, E, tvec);
}

// ------------------------------------------------------------------------------------------------------------------
// Diagonal family (GLA: T_i = diag(g_i)): the same reverse-streamed contraction with per-channel weights,
//     E[i, c] = sum_t v_t[i] k_t[c] w_t[c],   w_t[c] = exp(sum_{s > t} g_s[c]),   tvec[c] = exp(sum_t g_t[c]).
// The K / V tiles arrive by TMA as above; the 32 KB of fp32 log-decays per chunk are read straight from global memory by
// the converter threads, one chunk ahead, into registers: thread (pair p, range r) owns channels 2p, 2p+1 of tokens
// [16 r, 16 r + 16) of the chunk, scans its 16 tokens backwards, gets the totals of the later ranges through shared
// memory (one named barrier per chunk), and folds exp(.) into its 16 x 2 entries of the K tile with 32-bit accesses.
struct DtChShared {
  float2 tot[2][4][64];   // [chunk parity][token range][channel pair]: log-decay summed over the range
};
constexpr int kDtChOffX = kDtOffBar + 128;
constexpr int kDtChSmem = kDtChOffX + (int)sizeof(DtChShared) + 1024;

__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.b32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
// sts32: encode_scan4.cuh

__global__ void __launch_bounds__(kDtThreads, 3)
    diag_scan_ch_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                        const float* __restrict__ g, const int32_t* __restrict__ cu_seqlens, int H, float* __restrict__ E,
                        float* __restrict__ tvec) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  DtBars* bars = reinterpret_cast<DtBars*>(smem + kDtOffBar);
  DtChShared* xs = reinterpret_cast<DtChShared*>(smem + kDtChOffX);
  volatile int* abort_flag = &bars->abort_flag;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int h = blockIdx.x;
  const int s = dt_pick_segment(cu_seqlens, (int)gridDim.y, reinterpret_cast<int*>(smem));  // stage 0 is still empty
  const int seg_begin = cu_seqlens[s], seg_end = cu_seqlens[s + 1];
  const int nc = (seg_end - seg_begin + kC - 1) / kC;
  float* Eu = E + ((size_t)s * H + h) * kD * kD;
  float* tv = tvec + ((size_t)s * H + h) * kD;

  if (nc == 0) {  // empty segment: E = 0, tvec = 1
    for (int i = tid; i < kD * kD / 4; i += kDtThreads) reinterpret_cast<float4*>(Eu)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (tid < kD) tv[tid] = 1.f;
    return;
  }

  if (warp == kDtConvWarps) tmem_alloc(&bars->tmem_base, 128);
  if (tid == 0) {
    for (int i = 0; i < kDtStages; ++i) {
      mbar_init(&bars->full[i], 1);
      mbar_init(&bars->conv[i], kDtConvWarps);
      mbar_init(&bars->free_[i], 1);
    }
    mbar_init(&bars->done, 1);
    bars->abort_flag = 0;
    fence_barrier_init();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = bars->tmem_base;
  const uint32_t smem_base = smem_u32(smem);

  if (warp == kDtConvWarps + 1) {
    // ----------------------------------------------------------------------------------------------- loader
    if (lane == 0) {
#pragma unroll 1
      for (int i = 0; i < nc; ++i) {
        const int st = i % kDtStages;
        if (i >= kDtStages) dt_wait(&bars->free_[st], ((i / kDtStages) & 1) ^ 1, abort_flag);
        const uint32_t sb = smem_base + st * kDtStageBytes;
        const int t0 = seg_begin + (nc - 1 - i) * kC;  // last chunk first
        mbar_expect_tx(&bars->full[st], (uint32_t)kDtStageBytes);
        tma_load_3d(sb, &tmK, 0, h, t0, &bars->full[st]);
        tma_load_3d(sb + 8192, &tmK, 64, h, t0, &bars->full[st]);
        tma_load_3d(sb + 16384, &tmV, 0, h, t0, &bars->full[st]);
        tma_load_3d(sb + 24576, &tmV, 64, h, t0, &bars->full[st]);
      }
    }
  } else if (warp == kDtConvWarps) {
    // ----------------------------------------------------------------------------------------------- MMA issuer
    if (lane == 0) {
      constexpr uint32_t idesc = make_idesc(0u, 128, 128, 1, 1);
#pragma unroll 1
      for (int i = 0; i < nc; ++i) {
        const int st = i % kDtStages;
        dt_wait(&bars->conv[st], (i / kDtStages) & 1, abort_flag);
        tc_fence_after();
        const uint32_t sb = smem_base + st * kDtStageBytes;
#pragma unroll
        for (int ks = 0; ks < 4; ++ks)
          mma_f16_ss(tmem, make_desc(sb + 16384 + ks * 2048, 8192, 1024, 2), make_desc(sb + ks * 2048, 8192, 1024, 2),
                     idesc, (i > 0 || ks > 0) ? 1u : 0u);
        mma_commit(&bars->free_[st]);
      }
      mma_commit(&bars->done);
    }
  } else {
    // ----------------------------------------------------------------------------------------------- converters
    static_assert(kDtConvWarps == 8, "thread map below: 64 channel pairs x 4 token ranges");
    const int p = tid & 63, r = tid >> 6;
    double carry0 = 0.0, carry1 = 0.0;  // log-decay of all tokens after the current chunk, channels 2p and 2p + 1
    float2 gn[16];  // log-decays of this thread's 16 tokens x 2 channels of the current chunk; refilled in place, token
                    // by token, with the next chunk's as soon as each has been used (prefetch without a second array)
    auto load_g1 = [&](int i, int j) {
      const int t = seg_begin + (nc - 1 - i) * kC + 16 * r + j;
      return (i < nc && t < seg_end) ? __ldg(reinterpret_cast<const float2*>(g + ((size_t)t * H + h) * kD) + p)
                                     : make_float2(0.f, 0.f);
    };
#pragma unroll
    for (int j = 0; j < 16; ++j) gn[j] = load_g1(0, j);
    // K tile address of (token row 16 r + j, channel pair p): box p / 32, 128-byte rows, 16-byte chunks XOR-swizzled by row
    const uint32_t k_box = (uint32_t)(p >> 5) * 8192u, k_chunk = (uint32_t)((p & 31) >> 2), k_in = (uint32_t)(p & 3) * 4u;
#pragma unroll 1
    for (int i = 0; i < nc; ++i) {
      const int st = i % kDtStages;
      const int t0 = seg_begin + (nc - 1 - i) * kC;
      float s0 = 0.f, s1 = 0.f;
#pragma unroll
      for (int j = 0; j < 16; ++j) s0 += gn[j].x, s1 += gn[j].y;
      // envelope: log-decays <= 0 and finite (see the scalar kernel): a NaN / inf shows in the sums, a positive one in the
      // running maximum taken while the values are consumed below
      float gmax = (fabsf(s0) + fabsf(s1) < 3.0e38f) ? -1.f : 1.f;
      xs->tot[i & 1][r][p] = make_float2(s0, s1);
      asm volatile("bar.sync 1, 256;" ::: "memory");
      float later0 = 0.f, later1 = 0.f, all0 = 0.f, all1 = 0.f;
#pragma unroll
      for (int rr = 3; rr >= 0; --rr) {
        const float2 t = xs->tot[i & 1][rr][p];
        if (rr > r) later0 += t.x, later1 += t.y;
        all0 += t.x, all1 += t.y;
      }
      float run0 = (float)carry0 + later0, run1 = (float)carry1 + later1;  // log-weight of the range's LAST token
      carry0 += (double)all0, carry1 += (double)all1;
      s2_wait_warp(&bars->full[st], (i / kDtStages) & 1, abort_flag, lane);
      const uint32_t tile = smem_base + st * kDtStageBytes;
#pragma unroll
      for (int j = 15; j >= 0; --j) {
        const int tr = 16 * r + j;
        const uint32_t addr = tile + k_box + (uint32_t)tr * 128u + ((k_chunk ^ (uint32_t)(tr & 7)) << 4) + k_in;
        const uint32_t x = lds32(addr);
        uint32_t y = 0u;
        if (t0 + tr < seg_end)
          y = pack_f16(__uint_as_float(x << 16) * __expf(run0), __uint_as_float(x & 0xffff0000u) * __expf(run1));
        sts32(addr, y);
        run0 += gn[j].x, run1 += gn[j].y;  // weight of token j - 1: everything after it, token j included
        gmax = fmaxf(gmax, fmaxf(gn[j].x, gn[j].y));
        gn[j] = load_g1(i + 1, j);         // next chunk's log-decays: in flight during the rest of this conversion
      }
      if (__any_sync(0xffffffffu, gmax > 0.f) && lane == 0) atomicAdd(&g_envelope_count_enc, 1u);
      // V tile: bf16 -> fp16 in place, rows past the segment zeroed
#pragma unroll
      for (int it = 0; it < 4; ++it) {
        const int idx = 1024 + it * 256 + tid;
        const int tok = (idx & 511) >> 3;
        uint4 x = lds128(tile + 16 * idx);
        x.x = pack_f16(__uint_as_float(x.x << 16), __uint_as_float(x.x & 0xffff0000u));
        x.y = pack_f16(__uint_as_float(x.y << 16), __uint_as_float(x.y & 0xffff0000u));
        x.z = pack_f16(__uint_as_float(x.z << 16), __uint_as_float(x.z & 0xffff0000u));
        x.w = pack_f16(__uint_as_float(x.w << 16), __uint_as_float(x.w & 0xffff0000u));
        if (t0 + tok >= seg_end) x = make_uint4(0u, 0u, 0u, 0u);
        sts128(tile + 16 * idx, x);
      }
      fence_proxy_async();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars->conv[st]);
    }
    // tvec: the carry is now the log-decay of the whole segment (64-term fp32 chunk sums accumulated in fp64; the four
    // range-threads of a channel pair hold the same value)
    if (r == 0) *reinterpret_cast<float2*>(tv + 2 * p) = make_float2((float)exp(carry0), (float)exp(carry1));
    // ----------------------------------------------------------------------------------------------- epilogue
    s2_wait_warp(&bars->done, 0, abort_flag, lane);
    tc_fence_after();
    const int q = warp & 3, hf = warp >> 2;
    const int row = 32 * q + lane;
    constexpr int kColsPerWarp = kD / (kDtConvWarps / 4);
    float4* dst = reinterpret_cast<float4*>(Eu + (size_t)row * kD + kColsPerWarp * hf);
#pragma unroll 1
    for (int cb = 0; cb < kColsPerWarp / 32; ++cb) {
      uint32_t x[32];
      tmem_ld32(tmem + ((uint32_t)(32 * q) << 16) + kColsPerWarp * hf + 32 * cb, x);
      tmem_ld_wait();
#pragma unroll
      for (int u = 0; u < 8; ++u)
        dst[8 * cb + u] = make_float4(__uint_as_float(x[4 * u]), __uint_as_float(x[4 * u + 1]), __uint_as_float(x[4 * u + 2]),
                                      __uint_as_float(x[4 * u + 3]));
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kDtConvWarps) tmem_dealloc(tmem, 128);
}
