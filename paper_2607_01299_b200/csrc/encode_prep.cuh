// encode_prep.cuh -- the prep kernel (K1) of the tensor-family segment encode: everything of a chunk that does not
// depend on the running state.  Included by encode_tensor.cu inside namespace hypic::{anonymous}.
//
// One CTA (4 warps) per (chunk, head).  Rows a1..a3 of SURVEY.md section 8(a).
// Scalar gate (GDN row of Table 1): alpha_t is a scalar, so it commutes with (I - beta k k^t) and the whole
// gate factors out of the chunk algebra: with Gamma(t) the decay from the segment start through
// token t, S_t / Gamma(t) obeys the UNGATED delta rule with values v_t / Gamma(t), and T_C = Gamma(L) prod (I - beta k k^t).
// The prep is therefore gate-free for the scalar gate:
//   a1  G_r = inclusive in-chunk cumulative log-decay (handed to the scan as the gate record; nothing here uses it)
//   a2  L_rj = beta_r (k_r.k_j) for j < r                          Gram by mma.sync (fp16 operands, fp32 accumulate)
//   a3  A = (I + L)^-1, blocked 4 x 4 in 16 x 16 blocks: the diagonal blocks by forward substitution in fp32 (one
//       column per lane), the off-diagonal ones by the 2 x 2 block inverse formula A21 = -A22 L21 A11 applied at block
//       sizes 16 and 32; their 16^3 products run on mma.sync, single pass on fp16 operands for the scalar gate (A only
//       feeds the fp16 tiles below; emulation: E 3.5e-4, T 1.0e-3 at 2,048 tokens either way), hi + lo split (three
//       passes, ~2^-22) for the per-channel gate
//   out -W = -(A diag(beta)) K  (mma.sync, fp16 out, K-major 128B-swizzled UMMA B tile of two 64-wide boxes),
//       A_b = A diag(beta) (fp16, K-major 128B-swizzled UMMA B tile), gate record G_r[64].
// Per-channel gate (KDA row): Gamma does not commute; L_rj = beta_r (k_r (.) Gamma_r).(k_j (/) Gamma_j), W = A_b (K (.) Gamma),
// K~ and Gamma_C go into the record (section 6.4).
// K is staged as fp16 (exact for bf16 values with |x| in [2^-14, 65504]; smaller magnitudes lose bits below 2^-24
// absolute), so that the Gram and W contractions run as f16 mma.sync with an 11-bit second operand.
#pragma once

constexpr int kPrepThreads = 128;
constexpr int kKsPitch = kD + 8;  // 16-bit elements per row of the staged K chunk (conflict-free ldmatrix rows)
constexpr int kLPitch = 68;       // floats per row of L / A
constexpr int kMPitch = 36;       // floats per row of the 32 x 32 temporary of the last merge

__device__ __forceinline__ void mma_f16_16816(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                              uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void ldmatrix_x4(uint32_t (&r)[4], uint32_t saddr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
               : "r"(saddr));
}
__device__ __forceinline__ void ldmatrix_x4_trans(uint32_t (&r)[4], uint32_t saddr) {
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3])
               : "r"(saddr));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 p = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&p);
}
__device__ __forceinline__ uint32_t pack_f16(float lo, float hi) {
  __half2 p = __floats2half2_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&p);
}
// (x0, x1) -> packed fp16 hi and packed fp16 lo = fp16(x - hi)
__device__ __forceinline__ void split_f16(float x0, float x1, uint32_t& hi, uint32_t& lo) {
  const __half2 h = __floats2half2_rn(x0, x1);
  const float2 hf = __half22float2(h);
  hi = *reinterpret_cast<const uint32_t*>(&h);
  lo = pack_f16(x0 - hf.x, x1 - hf.y);
}

// acc (16 x 16, two n-tiles of the m16n8 C fragment) += X Y with X = xs[0..16)[0..16), Y = ys[0..16)[0..16), both fp32
// row-major in shared memory with the given pitches; operands split in fp16 hi + lo, three passes (hh, lh, hl).
template <bool kSplit>
__device__ __forceinline__ void block_mma_16(float (&acc)[2][4], const float* xs, int xp, const float* ys, int yp,
                                             int lane) {
  const int gq = lane >> 2, tq = lane & 3;
  uint32_t ah[4], al[4];
  {
    const float2 p0 = *reinterpret_cast<const float2*>(xs + gq * xp + 2 * tq);
    const float2 p1 = *reinterpret_cast<const float2*>(xs + (gq + 8) * xp + 2 * tq);
    const float2 p2 = *reinterpret_cast<const float2*>(xs + gq * xp + 2 * tq + 8);
    const float2 p3 = *reinterpret_cast<const float2*>(xs + (gq + 8) * xp + 2 * tq + 8);
    split_f16(p0.x, p0.y, ah[0], al[0]);
    split_f16(p1.x, p1.y, ah[1], al[1]);
    split_f16(p2.x, p2.y, ah[2], al[2]);
    split_f16(p3.x, p3.y, ah[3], al[3]);
  }
#pragma unroll
  for (int nt = 0; nt < 2; ++nt) {
    const int n = 8 * nt + gq;
    uint32_t bh[2], bl[2];
    split_f16(ys[(2 * tq) * yp + n], ys[(2 * tq + 1) * yp + n], bh[0], bl[0]);
    split_f16(ys[(2 * tq + 8) * yp + n], ys[(2 * tq + 9) * yp + n], bh[1], bl[1]);
    mma_f16_16816(acc[nt], ah[0], ah[1], ah[2], ah[3], bh[0], bh[1]);
    if (kSplit) {
      mma_f16_16816(acc[nt], al[0], al[1], al[2], al[3], bh[0], bh[1]);
      mma_f16_16816(acc[nt], ah[0], ah[1], ah[2], ah[3], bl[0], bl[1]);
    }
  }
}
// store sign * acc as a 16 x 16 fp32 block
__device__ __forceinline__ void block_store_16(const float (&acc)[2][4], float sign, float* dst, int dp, int lane) {
  const int gq = lane >> 2, tq = lane & 3;
#pragma unroll
  for (int nt = 0; nt < 2; ++nt) {
    *reinterpret_cast<float2*>(dst + gq * dp + 8 * nt + 2 * tq) = make_float2(sign * acc[nt][0], sign * acc[nt][1]);
    *reinterpret_cast<float2*>(dst + (gq + 8) * dp + 8 * nt + 2 * tq) = make_float2(sign * acc[nt][2], sign * acc[nt][3]);
  }
}
__device__ __forceinline__ void block_zero(float (&acc)[2][4]) {
#pragma unroll
  for (int nt = 0; nt < 2; ++nt)
#pragma unroll
    for (int i = 0; i < 4; ++i) acc[nt][i] = 0.f;
}

// Each CTA works through kPrepChunksPerCta consecutive chunks of one head and keeps the next chunk's k rows, g and
// beta in flight in registers while it computes the current one: with one chunk per CTA 45 % of all stall samples
// sat on the first global loads (profiles/r01b), which 5 CTAs per SM cannot hide.
constexpr int kPrepChunksPerCta = 4;

template <bool kCh>
__global__ void __launch_bounds__(kPrepThreads, 4)
    prep_kernel(const __nv_bfloat16* __restrict__ k, const float* __restrict__ g, const float* __restrict__ beta,
                const int2* __restrict__ chunk_meta, int cap, int H,
                uint8_t* __restrict__ rec, float* __restrict__ gate, const int32_t* __restrict__ chunk_off, int n_seg,
                int32_t* __restrict__ fb) {
  __shared__ __align__(16) uint8_t s_k[kC * kKsPitch * 2];  // K chunk (fp16)
  __shared__ __align__(16) float s_a[kC * kLPitch];         // L, inverted in place to A (per-channel gate: first K (/) Gamma)
  uint8_t* s_k2 = reinterpret_cast<uint8_t*>(s_a);           // fp16 [64][kKsPitch]: exactly the size of s_a
  __shared__ __align__(16) float s_m[32 * kMPitch];         // temporaries of the block merges
  __shared__ __align__(16) float s_g[kCh ? kD : kC], s_b[kC];  // s_g: G_r per token (scalar) or G_C per channel
  __shared__ float s_wsum;
  __shared__ int s_viol;  // per-channel gate: this chunk breaks the fp16 envelope (a channel's log-decay outside [-9, 0])
  if (threadIdx.x == 0) s_viol = 0;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int gq = lane >> 2, tq = lane & 3;
  const int x0 = blockIdx.x * kPrepChunksPerCta, h = blockIdx.y;
  int2 metas[kPrepChunksPerCta];  // (first token, valid tokens); (0, 0) beyond the last chunk of the call
#pragma unroll
  for (int i = 0; i < kPrepChunksPerCta; ++i) metas[i] = (x0 + i < cap) ? chunk_meta[x0 + i] : make_int2(0, 0);
  uint4 kreg[kC * (kD / 8) / kPrepThreads];
  float greg = 0.f, breg = 0.f;
  auto prefetch = [&](int2 m) {  // rows >= valid are not read; their registers are ignored at the store
#pragma unroll
    for (int it = 0; it < kC * (kD / 8) / kPrepThreads; ++it) {
      const int idx = tid + it * kPrepThreads;
      const int r = idx / (kD / 8), c8 = idx % (kD / 8);
      if (r < m.y) kreg[it] = *reinterpret_cast<const uint4*>(k + ((size_t)(m.x + r) * H + h) * kD + c8 * 8);
    }
    greg = 0.f, breg = 0.f;
    if (tid < m.y) {
      if (!kCh) greg = g[(size_t)(m.x + tid) * H + h];
      breg = beta[(size_t)(m.x + tid) * H + h];
    }
  };
  if (metas[0].y > 0) prefetch(metas[0]);
  __half* ks = reinterpret_cast<__half*>(s_k);
  const uint32_t ks_base = smem_u32(s_k);

#pragma unroll 1
  for (int ci = 0; ci < kPrepChunksPerCta; ++ci) {
  const int x = x0 + ci;
  const int valid = metas[ci].y;
  if (valid == 0) break;
#pragma unroll
  for (int it = 0; it < kC * (kD / 8) / kPrepThreads; ++it) {
    const int idx = tid + it * kPrepThreads;
    const int r = idx / (kD / 8), c8 = idx % (kD / 8);
    uint4 val = make_uint4(0, 0, 0, 0);
    if (r < valid) {
      const uint4 raw = kreg[it];
      val.x = pack_f16(__uint_as_float(raw.x << 16), __uint_as_float(raw.x & 0xffff0000u));
      val.y = pack_f16(__uint_as_float(raw.y << 16), __uint_as_float(raw.y & 0xffff0000u));
      val.z = pack_f16(__uint_as_float(raw.z << 16), __uint_as_float(raw.z & 0xffff0000u));
      val.w = pack_f16(__uint_as_float(raw.w << 16), __uint_as_float(raw.w & 0xffff0000u));
    }
    *reinterpret_cast<uint4*>(ks + r * kKsPitch + c8 * 8) = val;
  }
  {  // a1: inclusive cumulative log-decay by a two-warp shuffle scan (warps 0 and 1 hold the 64 tokens)
    float gv = greg, bv = breg;
    if (!kCh && ci + 1 < kPrepChunksPerCta && metas[ci + 1].y > 0) prefetch(metas[ci + 1]);  // in flight during this chunk
    if (kCh) {
      // per-channel gate: thread = (channel pair 2p, 2p+1; token range [32 r, 32 r + 32)); G_j[c] = cumulative log-decay
      // down the chunk's tokens; the K chunk is rewritten as K (.) Gamma (s_k) and K (/) Gamma (s_k2), both fp16 (Gamma
      // in [e^-9, 1] inside the envelope).  All 32 log-decay loads of a thread are in flight together, and the two
      // fp16 tiles are touched with 32-bit accesses (the first version, one thread per channel walking 64 tokens with
      // four serialised load batches and 16-bit accesses, took 25,000 of the chunk's 35,000 cycles).
      if (tid < kC) s_b[tid] = bv;
      const int p = tid & 63, rg = tid >> 6;
      const int t0c = metas[ci].x;
      float2 gl[32];
#pragma unroll
      for (int i = 0; i < 32; ++i) {
        const int j = 32 * rg + i;
        gl[i] = (j < valid) ? __ldg(reinterpret_cast<const float2*>(g + ((size_t)(t0c + j) * H + h) * kD) + p)
                            : make_float2(0.f, 0.f);
      }
      float r0 = 0.f, r1 = 0.f;
#pragma unroll
      for (int i = 0; i < 32; ++i) {  // inclusive prefix inside the range, in place
        r0 += gl[i].x, r1 += gl[i].y;
        gl[i] = make_float2(r0, r1);
      }
      float2* s_gt = reinterpret_cast<float2*>(s_m);  // totals of range 0 (s_m is free until the block merges)
      if (rg == 0) s_gt[p] = make_float2(r0, r1);
      __syncthreads();  // the K chunk is in s_k; the totals of range 0 are visible
      const float2 base = rg ? s_gt[p] : make_float2(0.f, 0.f);
      __half2* ks2 = reinterpret_cast<__half2*>(s_k);
      __half2* k22 = reinterpret_cast<__half2*>(s_k2);
#pragma unroll 8
      for (int i = 0; i < 32; ++i) {
        const int idx = ((32 * rg + i) * kKsPitch) / 2 + p;
        const float2 kv = __half22float2(ks2[idx]);
        const float G0 = base.x + gl[i].x, G1 = base.y + gl[i].y;
        ks2[idx] = __floats2half2_rn(kv.x * __expf(G0), kv.y * __expf(G1));
        k22[idx] = __floats2half2_rn(kv.x * __expf(-G0), kv.y * __expf(-G1));
      }
      if (rg == 1) {
        s_g[2 * p] = base.x + r0;
        s_g[2 * p + 1] = base.y + r1;
      }
      if (ci + 1 < kPrepChunksPerCta && metas[ci + 1].y > 0) prefetch(metas[ci + 1]);  // in flight during the rest
    } else {
      if (warp < 2) {
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const float up = __shfl_up_sync(0xffffffffu, gv, o);
          if (lane >= o) gv += up;
        }
        if (tid == 31) s_wsum = gv;
      }
      __syncthreads();
      if (warp < 2) {
        if (warp == 1) gv += s_wsum;
        s_g[tid] = gv;
        s_b[tid] = bv;
      }
    }
  }
  __syncthreads();
  const uint32_t k2_base = smem_u32(kCh ? s_k2 : s_k);  // second Gram operand
  uint8_t* out = rec + ((size_t)x * H + h) * (kCh ? kRecBytesCh : kRecBytes);
  if (kCh) {
    // K~_j = k_j (.) (Gamma_C (/) Gamma_j) = (K (/) Gamma)_j (.) Gamma_C, fp16, laid out like a K tile ([token][dk], two
    // 64-wide boxes, 128B swizzle): the B operand of (4)
    const __half* k2 = reinterpret_cast<const __half*>(s_k2);
#pragma unroll
    for (int it = 0; it < kC * (kD / 8) / kPrepThreads; ++it) {
      const int idx = tid + it * kPrepThreads;
      const int j = idx / (kD / 8), c8 = idx % (kD / 8);
      uint32_t w[4];
#pragma unroll
      for (int p = 0; p < 4; ++p) {
        const int c = 8 * c8 + 2 * p;
        w[p] = pack_f16(__half2float(k2[j * kKsPitch + c]) * __expf(s_g[c]),
                        __half2float(k2[j * kKsPitch + c + 1]) * __expf(s_g[c + 1]));
      }
      const uint32_t off = (c8 >> 3) * 8192 + (j >> 3) * 1024 + (j & 7) * 128 + (((c8 & 7) ^ (j & 7)) * 16);
      *reinterpret_cast<uint4*>(out + kRecKt + off) = make_uint4(w[0], w[1], w[2], w[3]);
    }
  }
  // ---- a2: Gram K K^t, lower block triangle = 10 blocks of 16 x 16 (block row m, block column p <= m), dealt to the
  // warps as 3 + 2 + 3 + 2 so that no warp carries the whole last block row
  {
    // warp 0: (3,0) (3,1) (0,0)   warp 1: (3,2) (3,3)   warp 2: (2,0) (2,1) (2,2)   warp 3: (1,0) (1,1)
    const int m0 = (warp == 0 || warp == 1) ? 3 : (warp == 2 ? 2 : 1);  // block row of units 0 and 1
    const int p0 = (warp == 1) ? 2 : 0;                                 // block columns p0, p0 + 1
    const int nun = (warp & 1) ? 2 : 3;                                 // third unit: warp 0 -> (0,0), warp 2 -> (2,2)
    const int m2 = (warp == 0) ? 0 : 2, p2 = (warp == 0) ? 0 : 2;
    float acc[3][2][4];
#pragma unroll
    for (int u = 0; u < 3; ++u)
#pragma unroll
      for (int nt = 0; nt < 2; ++nt)
#pragma unroll
        for (int i = 0; i < 4; ++i) acc[u][nt][i] = 0.f;
    const int lrow = (lane & 7) + 8 * ((lane >> 3) & 1), lcol = 8 * (lane >> 4);  // A operand: ldmatrix lane -> (row, k)
    const int brow = (lane & 7) + 8 * (lane >> 4), bcol = 8 * ((lane >> 3) & 1);  // B operand
#pragma unroll
    for (int kk = 0; kk < kD / 16; ++kk) {
      uint32_t a[4], b[4];
      ldmatrix_x4(a, ks_base + (uint32_t)((16 * m0 + lrow) * kKsPitch + 16 * kk + lcol) * 2u);
      ldmatrix_x4(b, k2_base + (uint32_t)((16 * p0 + brow) * kKsPitch + 16 * kk + bcol) * 2u);
      mma_f16_16816(acc[0][0], a[0], a[1], a[2], a[3], b[0], b[1]);
      mma_f16_16816(acc[0][1], a[0], a[1], a[2], a[3], b[2], b[3]);
      ldmatrix_x4(b, k2_base + (uint32_t)((16 * (p0 + 1) + brow) * kKsPitch + 16 * kk + bcol) * 2u);
      mma_f16_16816(acc[1][0], a[0], a[1], a[2], a[3], b[0], b[1]);
      mma_f16_16816(acc[1][1], a[0], a[1], a[2], a[3], b[2], b[3]);
      if (nun == 3) {
        if (warp == 0) ldmatrix_x4(a, ks_base + (uint32_t)((16 * m2 + lrow) * kKsPitch + 16 * kk + lcol) * 2u);
        ldmatrix_x4(b, k2_base + (uint32_t)((16 * p2 + brow) * kKsPitch + 16 * kk + bcol) * 2u);
        mma_f16_16816(acc[2][0], a[0], a[1], a[2], a[3], b[0], b[1]);
        mma_f16_16816(acc[2][1], a[0], a[1], a[2], a[3], b[2], b[3]);
      }
    }
    if (kCh) __syncthreads();  // every warp is done with K (/) Gamma: L takes over its buffer
    // the strictly upper blocks are zero (the A_b tile reads them): 6 blocks of 16 x 16 = 384 float4
#pragma unroll
    for (int it = 0; it < 3; ++it) {
      const int idx = tid + it * kPrepThreads;       // 0..383
      const int blk = idx >> 6, e = idx & 63;        // block (i, j) with j > i, 64 float4 each
      const int bi = blk < 3 ? 0 : (blk < 5 ? 1 : 2), bj = blk < 3 ? blk + 1 : (blk < 5 ? blk - 1 : 3);
      *reinterpret_cast<float4*>(s_a + (16 * bi + (e >> 2)) * kLPitch + 16 * bj + 4 * (e & 3)) = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    // L_rj = beta_r (k_r.k_j) for j < r, else 0 (per-channel gate: the decay ratios already sit in the two Gram operands)
#pragma unroll
    for (int u = 0; u < 3; ++u) {
      if (u == 2 && nun < 3) continue;
      const int mm = (u < 2) ? m0 : m2, pp = (u < 2) ? p0 + u : p2;
#pragma unroll
      for (int hh = 0; hh < 2; ++hh) {
        const int r = 16 * mm + gq + 8 * hh;
        const float br = s_b[r];
#pragma unroll
        for (int nt = 0; nt < 2; ++nt) {
          const int j = 16 * pp + 8 * nt + 2 * tq;
          float v0 = 0.f, v1 = 0.f;
          if (j < r) v0 = br * acc[u][nt][2 * hh];
          if (j + 1 < r) v1 = br * acc[u][nt][2 * hh + 1];
          *reinterpret_cast<float2*>(s_a + r * kLPitch + j) = make_float2(v0, v1);
        }
      }
    }
  }
  __syncthreads();

  // ---- a3 (i): diagonal blocks D_w = (I + L_ww)^-1 in place, lane c < 16 = column c, row-oriented substitution
  {
    float* blk = s_a + (16 * warp) * kLPitch + 16 * warp;
    float a[16];
    const int c = lane & 15;
#pragma unroll
    for (int r = 0; r < 16; ++r) {
      float part[4] = {(r == c) ? 1.f : 0.f, 0.f, 0.f, 0.f};  // one partial sum per float4 of the row: short chains
#pragma unroll
      for (int j4 = 0; j4 < (r + 3) / 4; ++j4) {
        const float4 l = *reinterpret_cast<const float4*>(blk + r * kLPitch + 4 * j4);
        if (4 * j4 + 0 < r) part[j4] = fmaf(-l.x, a[4 * j4 + 0], part[j4]);
        if (4 * j4 + 1 < r) part[j4] = fmaf(-l.y, a[4 * j4 + 1], part[j4]);
        if (4 * j4 + 2 < r) part[j4] = fmaf(-l.z, a[4 * j4 + 2], part[j4]);
        if (4 * j4 + 3 < r) part[j4] = fmaf(-l.w, a[4 * j4 + 3], part[j4]);
      }
      const float sum = (part[0] + part[1]) + (part[2] + part[3]);
      a[r] = sum;
    }
    __syncwarp();
    if (lane < 16) {
#pragma unroll
      for (int r = 0; r < 16; ++r) blk[r * kLPitch + c] = a[r];
    }
  }
  __syncthreads();
  auto B = [&](int i, int j) { return s_a + (16 * i) * kLPitch + 16 * j; };

  // ---- a3 (ii): A10 = -D1 (L10 D0) (warp 0), A32 = -D3 (L32 D2) (warp 1)
  if (warp < 2) {
    const int i = 2 * warp + 1, j = 2 * warp;
    float* tmp = s_m + (16 * warp) * kMPitch;
    float acc[2][4];
    block_zero(acc);
    block_mma_16<kCh>(acc, B(i, j), kLPitch, B(j, j), kLPitch, lane);
    block_store_16(acc, 1.f, tmp, kMPitch, lane);
    __syncwarp();
    block_zero(acc);
    block_mma_16<kCh>(acc, B(i, i), kLPitch, tmp, kMPitch, lane);
    __syncwarp();
    block_store_16(acc, -1.f, B(i, j), kLPitch, lane);
  }
  __syncthreads();
  // ---- a3 (iii): the 32 x 32 block A[2:4, 0:2] = -A[2:4, 2:4] (L[2:4, 0:2] A[0:2, 0:2]); warp -> block (2 + w/2, w%2)
  {
    const int i = 2 + (warp >> 1), j = warp & 1;
    float acc[2][4];
    block_zero(acc);
    if (j == 0) block_mma_16<kCh>(acc, B(i, 0), kLPitch, B(0, 0), kLPitch, lane);
    block_mma_16<kCh>(acc, B(i, 1), kLPitch, B(1, j), kLPitch, lane);
    block_store_16(acc, 1.f, s_m + (16 * (i - 2)) * kMPitch + 16 * j, kMPitch, lane);
    __syncthreads();
    block_zero(acc);
    block_mma_16<kCh>(acc, B(i, 2), kLPitch, s_m + 16 * j, kMPitch, lane);
    if (i == 3) block_mma_16<kCh>(acc, B(3, 3), kLPitch, s_m + 16 * kMPitch + 16 * j, kMPitch, lane);
    block_store_16(acc, -1.f, B(i, j), kLPitch, lane);
  }
  __syncthreads();

  // ---- -W = -(A diag(beta)) K with mma.sync: warp w rows [16w, 16w+16), k-steps kk <= w (A is lower
  // triangular), in two halves of 64 columns; the fp16 fragments go straight to the record in its K-major
  // 128B-swizzled two-box layout (4-byte stores; each 16-byte chunk is completed by the four lanes of a quad)
#pragma unroll 1
  for (int nh = 0; nh < 2; ++nh) {
    float wacc[8][4];
#pragma unroll
    for (int nt = 0; nt < 8; ++nt)
#pragma unroll
      for (int i = 0; i < 4; ++i) wacc[nt][i] = 0.f;
#pragma unroll
    for (int kk = 0; kk < 4; ++kk) {
      if (kk > warp) continue;
      uint32_t a[4];
      {
        const int r0 = 16 * warp + gq, c0 = 16 * kk + 2 * tq;
        const float* sc = s_b;  // per-channel gate: Gamma already sits in the K (.) Gamma operand
        const float g0 = sc[c0], g1 = sc[c0 + 1], g8 = sc[c0 + 8], g9 = sc[c0 + 9];
        const float2 p0 = *reinterpret_cast<const float2*>(s_a + r0 * kLPitch + c0);
        const float2 p1 = *reinterpret_cast<const float2*>(s_a + (r0 + 8) * kLPitch + c0);
        const float2 p2 = *reinterpret_cast<const float2*>(s_a + r0 * kLPitch + c0 + 8);
        const float2 p3 = *reinterpret_cast<const float2*>(s_a + (r0 + 8) * kLPitch + c0 + 8);
        a[0] = pack_f16(p0.x * g0, p0.y * g1);
        a[1] = pack_f16(p1.x * g0, p1.y * g1);
        a[2] = pack_f16(p2.x * g8, p2.y * g9);
        a[3] = pack_f16(p3.x * g8, p3.y * g9);
      }
      // B fragments (k = token, n = dk) by transposing ldmatrix over the [token][dk] tile, two n-tiles at a time
      const int tok = 16 * kk + (lane & 7) + ((lane >> 3) & 1) * 8;
#pragma unroll
      for (int np = 0; np < 4; ++np) {
        uint32_t b[4];
        ldmatrix_x4_trans(b, ks_base + (uint32_t)(tok * kKsPitch + 64 * nh + 8 * (2 * np + (lane >> 4))) * 2u);
        mma_f16_16816(wacc[2 * np], a[0], a[1], a[2], a[3], b[0], b[1]);
        mma_f16_16816(wacc[2 * np + 1], a[0], a[1], a[2], a[3], b[2], b[3]);
      }
    }
#pragma unroll
    for (int nt = 0; nt < 8; ++nt)
#pragma unroll
      for (int hh = 0; hh < 2; ++hh) {
        const int r = 16 * warp + gq + 8 * hh;
        const uint32_t off = nh * 8192 + (r >> 3) * 1024 + (r & 7) * 128 + ((nt ^ (r & 7)) * 16) + tq * 4;
        *reinterpret_cast<uint32_t*>(out + kRecW + off) = pack_f16(-wacc[nt][2 * hh], -wacc[nt][2 * hh + 1]);
      }
  }
  // ---- A_b = A diag(beta) as an fp16 B tile (K-major, 128B swizzle: row r, 16-byte chunk j8 at ((j8 ^ (r & 7)) * 16))
#pragma unroll
  for (int it = 0; it < kC * 8 / kPrepThreads; ++it) {
    const int idx = tid + it * kPrepThreads;
    const int r = idx >> 3, j8 = idx & 7;
    const float4 v0 = *reinterpret_cast<const float4*>(s_a + r * kLPitch + 8 * j8);
    const float4 v1 = *reinterpret_cast<const float4*>(s_a + r * kLPitch + 8 * j8 + 4);
    const float4 b0 = *reinterpret_cast<const float4*>(s_b + 8 * j8);
    const float4 b1 = *reinterpret_cast<const float4*>(s_b + 8 * j8 + 4);
    const uint32_t off = (r >> 3) * 1024 + (r & 7) * 128 + ((j8 ^ (r & 7)) * 16);
    *reinterpret_cast<uint4*>(out + kRecAb + off) =
        make_uint4(pack_f16(v0.x * b0.x, v0.y * b0.y), pack_f16(v0.z * b0.z, v0.w * b0.w),
                   pack_f16(v1.x * b1.x, v1.y * b1.y), pack_f16(v1.z * b1.z, v1.w * b1.w));
  }
  if (kCh) {
    float* go = gate + ((size_t)x * H + h) * kGateFloatsCh;
    const float gc = s_g[tid];
    go[tid] = expf(gc);
    if (tid < kGateFloatsCh - kD) go[kD + tid] = 0.f;
    if (!(gc >= -9.f && gc <= 0.f)) s_viol = 1;  // also NaN
  } else {
    float* go = gate + ((size_t)x * H + h) * kGateFloats;  // the scan turns G_r into the value weights (lazy decay)
    if (tid < kGateFloats) go[tid] = (tid < kC) ? s_g[tid] : 0.f;
  }
  __syncthreads();  // s_k, s_a, s_g are free for the next chunk
  if (kCh && tid == 0 && s_viol) {
    // the unit of this chunk is recomputed by the fp32 family inside the same call (no host involvement): find its
    // segment in chunk_off and put (segment, head) on the call's fallback list
    s_viol = 0;
    atomicAdd(&g_envelope_count_enc, 1u);  // diagnostic counter (hypic_envelope_violation_count)
    int lo = 0, hi = n_seg;                // chunk_off[lo] <= x < chunk_off[hi]
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (chunk_off[mid] <= x) lo = mid; else hi = mid;
    }
    fb_append(fb, n_seg * H, lo * H + h);
  }
  }
}
