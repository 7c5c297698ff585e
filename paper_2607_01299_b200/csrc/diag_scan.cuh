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
// Roles of a CTA (192 threads, one (segment, head) unit, two CTAs per SM, 128 TMEM columns each):
//   warp 5      loader      TMA boxes of the bf16 K and V chunk tiles (64 tokens x 128 channels each), 3 stages
//   warps 0-3   converters  weights of the chunk (warp 0: shuffle suffix scan of g, fp64 carry), then in place:
//                           K~ = fp16(w_t k_t), V -> fp16, rows past the end of the segment zeroed; epilogue
//   warp 4      issuer      4 x tcgen05.mma (M = dv = 128, N = dk = 128, K = 16 tokens) per chunk, both operands
//                           MN-major straight from the swizzled boxes; accumulator E (fp32) stays in TMEM throughout
#pragma once

constexpr int kDtThreads = 192;
constexpr int kDtStages = 3;
constexpr int kDtStageBytes = 32768;  // K tile (2 boxes of 8 KB) + V tile
constexpr int kDtOffW = kDtStages * kDtStageBytes;        // per-stage token weights: float[kDtStages][64]
constexpr int kDtOffBar = kDtOffW + kDtStages * 64 * 4;
constexpr int kDtSmem = kDtOffBar + 128 + 1024;

struct DtBars {
  uint64_t full[kDtStages], conv[kDtStages], free_[kDtStages], done;
  uint32_t tmem_base;
  int abort_flag;
};

__device__ __forceinline__ void named_bar_sync128(int id) { asm volatile("bar.sync %0, 128;" ::"r"(id) : "memory"); }

__global__ void __launch_bounds__(kDtThreads, 2)
    diag_scan_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                     const float* __restrict__ g, const int32_t* __restrict__ cu_seqlens, int H, float* __restrict__ E,
                     float* __restrict__ tvec) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  DtBars* bars = reinterpret_cast<DtBars*>(smem + kDtOffBar);
  float* sw = reinterpret_cast<float*>(smem + kDtOffW);
  volatile int* abort_flag = &bars->abort_flag;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int h = blockIdx.x, s = blockIdx.y;
  const int seg_begin = cu_seqlens[s], seg_end = cu_seqlens[s + 1];
  const int nc = (seg_end - seg_begin + kC - 1) / kC;
  float* Eu = E + ((size_t)s * H + h) * kD * kD;

  if (nc == 0) {  // empty segment: E = 0, tvec = 1
    for (int i = tid; i < kD * kD / 4; i += kDtThreads) reinterpret_cast<float4*>(Eu)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (tid == 0) tvec[(size_t)s * H + h] = 1.f;
    return;
  }

  if (warp == 4) tmem_alloc(&bars->tmem_base, 128);
  if (tid == 0) {
    for (int i = 0; i < kDtStages; ++i) {
      mbar_init(&bars->full[i], 1);
      mbar_init(&bars->conv[i], 4);
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

  if (warp == 5) {
    // ----------------------------------------------------------------------------------------------- loader
    if (lane == 0) {
#pragma unroll 1
      for (int i = 0; i < nc; ++i) {
        const int st = i % kDtStages;
        if (i >= kDtStages) s2_wait(&bars->free_[st], ((i / kDtStages) & 1) ^ 1, abort_flag);
        const uint32_t sb = smem_base + st * kDtStageBytes;
        const int t0 = seg_begin + (nc - 1 - i) * kC;  // last chunk first
        mbar_expect_tx(&bars->full[st], (uint32_t)kDtStageBytes);
        tma_load_3d(sb, &tmK, 0, h, t0, &bars->full[st]);
        tma_load_3d(sb + 8192, &tmK, 64, h, t0, &bars->full[st]);
        tma_load_3d(sb + 16384, &tmV, 0, h, t0, &bars->full[st]);
        tma_load_3d(sb + 24576, &tmV, 64, h, t0, &bars->full[st]);
      }
    }
  } else if (warp == 4) {
    // ----------------------------------------------------------------------------------------------- MMA issuer
    if (lane == 0) {
      constexpr uint32_t idesc = make_idesc(0u, 128, 128, 1, 1);  // fp16 x fp16 -> fp32, A (V tile) and B (K~ tile) MN-major
#pragma unroll 1
      for (int i = 0; i < nc; ++i) {
        const int st = i % kDtStages;
        s2_wait(&bars->conv[st], (i / kDtStages) & 1, abort_flag);
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
    double carry = 0.0;  // warp 0: log-decay of all tokens after the current chunk (fp64: up to thousands of terms)
#pragma unroll 1
    for (int i = 0; i < nc; ++i) {
      const int st = i % kDtStages;
      const int t0 = seg_begin + (nc - 1 - i) * kC;
      float* w = sw + st * 64;
      if (warp == 0) {
        // tokens 2 lane, 2 lane + 1 of the chunk; exclusive suffix sums by a shuffle scan over the lane pairs
        const int ta = t0 + 2 * lane, tb = ta + 1;
        const float ga = ta < seg_end ? __ldg(g + (size_t)ta * H + h) : 0.f;
        const float gb = tb < seg_end ? __ldg(g + (size_t)tb * H + h) : 0.f;
        float suf = ga + gb;  // becomes the inclusive suffix sum over lanes >= lane
        double tot = (double)ga + (double)gb;
#pragma unroll
        for (int d = 1; d < 32; d *= 2) {
          const float up = __shfl_down_sync(0xffffffffu, suf, d);
          const double upd = __shfl_xor_sync(0xffffffffu, tot, d);
          if (lane + d < 32) suf += up;
          tot += upd;
        }
        const float excl = suf - (ga + gb);  // tokens of the lanes above
        const float cf = (float)carry;
        // the stage's weights were read by the conversion of chunk i - kDtStages, which this warp finished long ago
        w[2 * lane + 1] = tb < seg_end ? __expf(cf + excl) : 0.f;
        w[2 * lane] = ta < seg_end ? __expf(cf + excl + gb) : 0.f;
        carry += tot;
      }
      named_bar_sync128(1);
      s2_wait_warp(&bars->full[st], (i / kDtStages) & 1, abort_flag, lane);
      uint4* tile = reinterpret_cast<uint4*>(smem + st * kDtStageBytes);
      // 2,048 16-byte vectors: K boxes [0, 1024), V boxes [1024, 2048); vector idx of a box sits in token row (idx % 512) / 8
#pragma unroll 4
      for (int it = 0; it < 16; ++it) {
        const int idx = it * 128 + tid;
        const int tok = (idx & 511) >> 3;
        const float m = it < 8 ? w[tok] : 1.f;
        uint4 x = tile[idx];
        x.x = pack_f16(m * __uint_as_float(x.x << 16), m * __uint_as_float(x.x & 0xffff0000u));
        x.y = pack_f16(m * __uint_as_float(x.y << 16), m * __uint_as_float(x.y & 0xffff0000u));
        x.z = pack_f16(m * __uint_as_float(x.z << 16), m * __uint_as_float(x.z & 0xffff0000u));
        x.w = pack_f16(m * __uint_as_float(x.w << 16), m * __uint_as_float(x.w & 0xffff0000u));
        if (t0 + tok >= seg_end) x = make_uint4(0u, 0u, 0u, 0u);  // rows past the segment hold other tokens' data
        tile[idx] = x;
      }
      fence_proxy_async();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars->conv[st]);
      // w[st] is rewritten kDtStages chunks later, behind at least one more named barrier that every converter only
      // reaches after this conversion
    }
    // ----------------------------------------------------------------------------------------------- epilogue
    s2_wait_warp(&bars->done, 0, abort_flag, lane);
    tc_fence_after();
    const int row = 32 * warp + lane;  // dv index = TMEM lane
    float4* dst = reinterpret_cast<float4*>(Eu + (size_t)row * kD);
#pragma unroll 1
    for (int cb = 0; cb < 4; ++cb) {
      uint32_t x[32];
      tmem_ld32(tmem + ((uint32_t)(32 * warp) << 16) + 32 * cb, x);
      tmem_ld_wait();
#pragma unroll
      for (int u = 0; u < 8; ++u)
        dst[8 * cb + u] = make_float4(__uint_as_float(x[4 * u]), __uint_as_float(x[4 * u + 1]), __uint_as_float(x[4 * u + 2]),
                                      __uint_as_float(x[4 * u + 3]));
    }
    if (tid == 0) tvec[(size_t)s * H + h] = (float)exp(carry);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 4) tmem_dealloc(tmem, 128);
}
