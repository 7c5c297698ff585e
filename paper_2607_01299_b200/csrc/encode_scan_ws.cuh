// encode_scan_ws.cuh -- warp-specialised scan kernel (K2) of the tensor-family segment encode.
// Included by encode_tensor.cu inside namespace hypic::{anonymous}; uses its constants and helpers.
//
// One CTA per (row block b of X = [E; T], head, segment); 16 warps:
//   warp 0      loader      TMA tensor boxes for the K / V chunk tiles, bulk copies for the (A_b, A_b gamma) tiles
//                           and the gate record, two stages, one mbarrier per stage
//   warp 1      MMA issuer  one thread; per chunk c, in this order on the (in-order) tensor pipe:
//                             (3)_c   DY_c (+)= Xr (-W_c)^t           tf32, A from TMEM
//                             (2)_c+1 Wt = K^t A_bg^t                 bf16   (runs under the epilogue of c)
//                             (4)_c   X += U''_c K_c                  bf16
//                             (1)_c+1 DY_{c+1} = V^t A_b^t            bf16   (E block; runs under the pass of c+1)
//   warps 4-7   W group     Wt (TMEM) -> -rna_tf32 -> smem B tile of (3)
//   warps 8-15  state group pass: Xr = rna_tf32(X), X <- gamma_C X;  epilogue: DY * d_j -> bf16 hi/lo A tiles of (4)
// TMEM columns: X [0,128), Xr [128,256), DY [256,320) and [320,384) (double buffered), Wt [384,448).
#pragma once

constexpr int kWsThreads = 512;
constexpr int kWsStK = 0, kWsStV = 16384, kWsStAb = 32768, kWsStGate = 65536;
constexpr int kWsStageBytes = 65536 + 1024;
constexpr int kWsOffW = 2 * kWsStageBytes;
constexpr int kWsOffUhi = kWsOffW + 32768;
constexpr int kWsOffUlo = kWsOffUhi + 16384;
constexpr int kWsOffBar = kWsOffUlo + 16384;
constexpr int kWsSmem = kWsOffBar + 256 + 1024;

struct WsBars {
  uint64_t st_full[2], st_free[2], m2_done, wt_free, w_ready, w_free, xr_ready, m3_done, u_ready, m4_done;
  uint32_t tmem_base;
  int abort_flag;
};

__device__ __forceinline__ void tma_load_3d(uint32_t dst_smem, const CUtensorMap* tm, int c0, int c1, int c2,
                                            uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
          dst_smem),
      "l"(reinterpret_cast<uint64_t>(tm)), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
      : "memory");
}

__device__ __forceinline__ bool ws_wait(uint64_t* bar, uint32_t parity, volatile int* abort_flag) {
  for (uint32_t i = 0; i < 4000000u; ++i) {
    if (mbar_try_wait(bar, parity)) return true;
    if ((i & 1023u) == 1023u && *abort_flag) return false;
  }
  if (!*abort_flag) {
    *abort_flag = 1;
    atomicAdd(&g_timeout_count_enc, 1u);
  }
  return false;
}

__global__ void __launch_bounds__(kWsThreads, 1)
    scan_ws_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                   const int32_t* __restrict__ cu_seqlens, const int32_t* __restrict__ chunk_off, int H,
                   const uint8_t* __restrict__ ab, const float* __restrict__ gate, float* __restrict__ E,
                   float* __restrict__ T) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  WsBars* bars = reinterpret_cast<WsBars*>(smem + kWsOffBar);
  volatile int* abort_flag = &bars->abort_flag;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int blk = blockIdx.x, h = blockIdx.y, s = blockIdx.z;
  const bool is_e = (blk == 0);
  const int seg_begin = cu_seqlens[s], seg_end = cu_seqlens[s + 1];
  const int nc = (seg_end - seg_begin + kC - 1) / kC;
  const int chunk0 = chunk_off[s];

  if (warp == 2) tmem_alloc(&bars->tmem_base, 512);
  if (tid == 0) {
    for (int i = 0; i < 2; ++i) { mbar_init(&bars->st_full[i], 1); mbar_init(&bars->st_free[i], 1); }
    mbar_init(&bars->m2_done, 1);
    mbar_init(&bars->wt_free, 4);
    mbar_init(&bars->w_ready, 4);
    mbar_init(&bars->w_free, 1);
    mbar_init(&bars->xr_ready, 8);
    mbar_init(&bars->m3_done, 1);
    mbar_init(&bars->u_ready, 8);
    mbar_init(&bars->m4_done, 1);
    bars->abort_flag = 0;
    fence_barrier_init();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = bars->tmem_base;
  const uint32_t smem_base = smem_u32(smem);
  constexpr uint32_t cX = 0, cXr = 128, cDY = 256, cWt = 384;

  if (warp == 0) {
    // ------------------------------------------------------------------------------------------- loader
    if (lane == 0) {
      const uint32_t bytes = 16384u + (is_e ? 16384u : 0u) + (uint32_t)kAbBytes + (uint32_t)kGateBytes;
      for (int c = 0; c < nc; ++c) {
        const int st = c & 1;
        ws_wait(&bars->st_free[st], ((c >> 1) & 1) ^ 1, abort_flag);
        const uint32_t sb = smem_base + st * kWsStageBytes;
        const int t0 = seg_begin + c * kC;
        mbar_expect_tx(&bars->st_full[st], bytes);
        tma_load_3d(sb + kWsStK, &tmK, 0, h, t0, &bars->st_full[st]);
        tma_load_3d(sb + kWsStK + 8192, &tmK, 64, h, t0, &bars->st_full[st]);
        if (is_e) {
          tma_load_3d(sb + kWsStV, &tmV, 0, h, t0, &bars->st_full[st]);
          tma_load_3d(sb + kWsStV + 8192, &tmV, 64, h, t0, &bars->st_full[st]);
        }
        const size_t rec = (size_t)(chunk0 + c) * H + h;
        bulk_g2s(smem + st * kWsStageBytes + kWsStAb, ab + rec * kAbBytes, kAbBytes, &bars->st_full[st]);
        bulk_g2s(smem + st * kWsStageBytes + kWsStGate, gate + rec * kGateFloats, kGateBytes, &bars->st_full[st]);
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------------------------------------- MMA issuer
    if (lane == 0 && nc > 0) {
      constexpr uint32_t id12 = make_idesc(1u, 128, 64, 1, 0);   // bf16, A MN-major (K / V tile), B K-major
      constexpr uint32_t id3 = make_idesc(2u, 128, 64, 0, 1);    // tf32, A from TMEM, B MN-major
      constexpr uint32_t id4 = make_idesc(1u, 128, 128, 0, 1);   // bf16, A K-major (U''), B MN-major (K tile)
      auto issue2 = [&](int c) {  // Wt = K^t A_bg^t
        const int st = c & 1;
        ws_wait(&bars->st_full[st], (c >> 1) & 1, abort_flag);
        ws_wait(&bars->wt_free, (c & 1) ^ 1, abort_flag);
        tc_fence_after();
        const uint32_t sb = smem_base + st * kWsStageBytes;
#pragma unroll
        for (int hl = 0; hl < 2; ++hl)
#pragma unroll
          for (int ks = 0; ks < 4; ++ks)
            mma_f16_ss(tmem + cWt, make_desc(sb + kWsStK + ks * 2048, 8192, 1024, 2),
                       make_desc(sb + kWsStAb + (2 + hl) * kTileB + ks * 32, 16, 1024, 2), id12, (hl | ks) > 0);
        mma_commit(&bars->m2_done);
      };
      auto issue1 = [&](int c) {  // DY_c = V^t A_b^t (E block)
        if (!is_e) return;
        const uint32_t sb = smem_base + (c & 1) * kWsStageBytes;
#pragma unroll
        for (int hl = 0; hl < 2; ++hl)
#pragma unroll
          for (int ks = 0; ks < 4; ++ks)
            mma_f16_ss(tmem + cDY + 64 * (c & 1), make_desc(sb + kWsStV + ks * 2048, 8192, 1024, 2),
                       make_desc(sb + kWsStAb + hl * kTileB + ks * 32, 16, 1024, 2), id12, (hl | ks) > 0);
      };
      issue2(0);
      issue1(0);
      for (int c = 0; c < nc; ++c) {
        const uint32_t sb = smem_base + (c & 1) * kWsStageBytes;
        // (3)_c
        ws_wait(&bars->xr_ready, c & 1, abort_flag);
        ws_wait(&bars->w_ready, c & 1, abort_flag);
        tc_fence_after();
#pragma unroll
        for (int ks = 0; ks < 16; ++ks)
          mma_tf32_ts(tmem + cDY + 64 * (c & 1), tmem + cXr + ks * 8,
                      make_desc(smem_base + kWsOffW + ks * 1024, 16384, 512, 1), id3, (is_e || ks > 0) ? 1u : 0u);
        mma_commit(&bars->m3_done);
        mma_commit(&bars->w_free);
        // (2)_{c+1}
        if (c + 1 < nc) issue2(c + 1);
        // (4)_c
        ws_wait(&bars->u_ready, c & 1, abort_flag);
        tc_fence_after();
#pragma unroll
        for (int hl = 0; hl < 2; ++hl)
#pragma unroll
          for (int ks = 0; ks < 4; ++ks)
            mma_f16_ss(tmem + cX, make_desc(smem_base + (hl ? kWsOffUlo : kWsOffUhi) + ks * 32, 16, 1024, 2),
                       make_desc(sb + kWsStK + ks * 2048, 8192, 1024, 2), id4, 1u);
        mma_commit(&bars->m4_done);
        mma_commit(&bars->st_free[c & 1]);
        // (1)_{c+1}
        if (c + 1 < nc) issue1(c + 1);
      }
    }
  } else if (warp >= 4 && warp < 8) {
    // ------------------------------------------------------------------------------------------- W group
    const int q = warp & 3;
    const int row = 32 * q + lane;  // dk index = row of Wt
    const uint32_t tWt = tmem + cWt + ((uint32_t)(32 * q) << 16);
    uint8_t* base = smem + kWsOffW + (row >> 2) * 512 + (row & 3) * 128;
    for (int c = 0; c < nc; ++c) {
      ws_wait(&bars->m2_done, c & 1, abort_flag);
      tc_fence_after();
      uint32_t w0[32], w1[32];
      tmem_ld32(tWt, w0);
      tmem_ld32(tWt + 32, w1);
      tmem_ld_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars->wt_free);
      ws_wait(&bars->w_free, (c & 1) ^ 1, abort_flag);
#pragma unroll
      for (int nch = 0; nch < 2; ++nch) {
#pragma unroll
        for (int q8 = 0; q8 < 4; ++q8) {
          const uint32_t* w = nch ? w1 : w0;
          float4 lo4, hi4;
          lo4.x = -rna_tf32f(__uint_as_float(w[8 * q8 + 0])), lo4.y = -rna_tf32f(__uint_as_float(w[8 * q8 + 1]));
          lo4.z = -rna_tf32f(__uint_as_float(w[8 * q8 + 2])), lo4.w = -rna_tf32f(__uint_as_float(w[8 * q8 + 3]));
          hi4.x = -rna_tf32f(__uint_as_float(w[8 * q8 + 4])), hi4.y = -rna_tf32f(__uint_as_float(w[8 * q8 + 5]));
          hi4.z = -rna_tf32f(__uint_as_float(w[8 * q8 + 6])), hi4.w = -rna_tf32f(__uint_as_float(w[8 * q8 + 7]));
          uint8_t* p = base + nch * 16384 + ((q8 ^ (row & 3)) * 32);
          *reinterpret_cast<float4*>(p) = lo4;
          *reinterpret_cast<float4*>(p + 16) = hi4;
        }
      }
      fence_proxy_async();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars->w_ready);
    }
  } else if (warp >= 8) {
    // ------------------------------------------------------------------------------------------- state group
    const int q = warp & 3, hf = (warp - 8) >> 2;
    const int row = 32 * q + lane;
    const uint32_t lane_base = (uint32_t)(32 * q) << 16;
    uint8_t* uhi = smem + kWsOffUhi + (row >> 3) * 1024 + (row & 7) * 128;
    uint8_t* ulo = smem + kWsOffUlo + (row >> 3) * 1024 + (row & 7) * 128;
    for (int c = 0; c < nc; ++c) {
      const float* gt = reinterpret_cast<const float*>(smem + (c & 1) * kWsStageBytes + kWsStGate);
      // ---- pass: Xr = rna_tf32(X), X <- gamma_C X  (this warp: columns [64 hf, 64 hf + 64))
      ws_wait(&bars->st_full[c & 1], (c >> 1) & 1, abort_flag);
      ws_wait(&bars->m4_done, (c & 1) ^ 1, abort_flag);
      tc_fence_after();
      const float gC = gt[kC];
#pragma unroll
      for (int cb2 = 0; cb2 < 2; ++cb2) {
        const int col = 64 * hf + 32 * cb2;
        uint32_t x[32];
        if (c > 0) {
          tmem_ld32(tmem + cX + lane_base + col, x);
          tmem_ld_wait();
        } else {
#pragma unroll
          for (int i = 0; i < 32; ++i) x[i] = (!is_e && col + i == row) ? __float_as_uint(1.f) : 0u;
        }
        uint32_t xr[32];
#pragma unroll
        for (int i = 0; i < 32; ++i) {
          const float f = __uint_as_float(x[i]);
          xr[i] = __float_as_uint(rna_tf32f(f));
          x[i] = __float_as_uint(f * gC);
        }
        tmem_st32(tmem + cXr + lane_base + col, xr);
        tmem_st32(tmem + cX + lane_base + col, x);
      }
      tmem_st_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars->xr_ready);

      // ---- epilogue: U''[:, j] = DY[:, j] d_j for tokens j in [32 hf, 32 hf + 32) -> bf16 hi/lo, K-major 128B swizzle
      ws_wait(&bars->m3_done, c & 1, abort_flag);
      tc_fence_after();
      {
        uint32_t y[32];
        tmem_ld32(tmem + cDY + 64 * (c & 1) + lane_base + 32 * hf, y);
        tmem_ld_wait();
#pragma unroll
        for (int j8 = 0; j8 < 4; ++j8) {
          uint32_t hi[4], lo[4];
#pragma unroll
          for (int p = 0; p < 4; ++p) {
            const int j = 32 * hf + 8 * j8 + 2 * p;
            const float u0 = __uint_as_float(y[8 * j8 + 2 * p]) * gt[j];
            const float u1 = __uint_as_float(y[8 * j8 + 2 * p + 1]) * gt[j + 1];
            const float h0 = __bfloat162float(__float2bfloat16_rn(u0)), h1 = __bfloat162float(__float2bfloat16_rn(u1));
            hi[p] = pack_bf16(h0, h1);
            lo[p] = pack_bf16(u0 - h0, u1 - h1);
          }
          const uint32_t sw = (((4 * hf + j8) ^ (row & 7)) * 16);
          *reinterpret_cast<uint4*>(uhi + sw) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
          *reinterpret_cast<uint4*>(ulo + sw) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
        }
      }
      fence_proxy_async();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars->u_ready);
    }
    // ---- a5: write this warp's 64 columns of the block (thread = row)
    if (nc > 0) {
      ws_wait(&bars->m4_done, (nc - 1) & 1, abort_flag);
      tc_fence_after();
    }
    float* dst = (is_e ? E : T) + (((size_t)s * H + h) * kD + row) * kD;
#pragma unroll 1
    for (int cb2 = 0; cb2 < 2; ++cb2) {
      const int col = 64 * hf + 32 * cb2;
      uint32_t x[32];
      if (nc > 0) {
        tmem_ld32(tmem + cX + lane_base + col, x);
        tmem_ld_wait();
      } else {
#pragma unroll
        for (int i = 0; i < 32; ++i) x[i] = (!is_e && col + i == row) ? __float_as_uint(1.f) : 0u;
      }
      float4* d4 = reinterpret_cast<float4*>(dst + col);
#pragma unroll
      for (int u = 0; u < 8; ++u)
        d4[u] = make_float4(__uint_as_float(x[4 * u]), __uint_as_float(x[4 * u + 1]), __uint_as_float(x[4 * u + 2]),
                            __uint_as_float(x[4 * u + 3]));
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 2) tmem_dealloc(tmem, 512);
}
