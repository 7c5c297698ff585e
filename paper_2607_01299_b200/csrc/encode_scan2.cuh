// encode_scan2.cuh -- the scan kernel (K2) of the tensor-family segment encode.
// Included by encode_tensor.cu inside namespace hypic::{anonymous}; uses its constants and helpers.
//
// One CTA per (segment, head), sequential over the segment's 64-token chunks; both row blocks of the stacked state
// X = [E ; T] (128 rows each) stay in TMEM as fp32 for the whole segment.  Every contraction is a single-pass
// tcgen05.mma kind::f16 on fp16 operands (11 significant bits, like tf32, at the full 16-bit rate):
//     (1)_c  DY_E  = V^t A_b^t              A = the V tile (MN-major), B = A_b from the prep record   (E block only)
//     (3)_c  DY_b += Xh_b (-W)^t            A = Xh_b = fp16(X_b) read from TMEM, B = -W from the prep record
//     (4)_c  X_b  += U''_b K                A = U''_b = fp16(DY_b d_j) read from TMEM (it takes over the columns of
//                                           Xh_b, dead once (3)_c has completed), B = the K tile (MN-major)
// fp16 has a narrow exponent range, so the T block is held row-normalised: row r of the TMEM copy is T_r 2^s_r with
// s_r re-chosen in every pass so that the row maximum sits in [2^14, 2^15); since (3) and (4) are linear in the row
// the factor never has to be undone before the final write-out.  E rows live on the scale of v and stay unscaled.
// k / v arrive as bf16 and are converted to fp16 in place in shared memory (exact for |x| in [2^-14, 65504]).
//
// 19 warps:
// (the warp scheduler favours the highest warp id of an SM sub-partition, so the latency-critical single-thread
// roles sit at the top):
//   warps 0-7     E chain     thread = (row of E, 64-column half): pass  Xh = fp16(X), X <- gamma_C X;
//                             epilogue  U'' = fp16(DY d_j)
//   warps 8-15    T chain     same for T plus the row re-normalisation
//   warps 16-17   converters  K (warp 16) and V (warp 17) tile bf16 -> fp16 in place; warp 16 also owns TMEM alloc;
//                             warp 17 issues (1) for the tile it has just converted
//   warp 18       loader      TMA tensor boxes for the K / V chunk tiles, bulk copies for the prep record (-W, A_b)
//                             and the gate record; three stages
// There is no separate MMA-issuer role: after a chain-wide named barrier, one elected thread of the chain issues the
// chain's next batch itself (a dedicated issuer thread that polled both chains reacted 450-800 cycles late per batch,
// starved by the busy chain warps of its SM sub-partition) and commits it to the mbarrier the chain then waits on.
// The two chains only share read-only operands, so while one is in its element-wise phase the tensor pipe runs the
// other one's MMAs.  TMEM columns: X_E [0,128), X_T [128,256), Xh_E [256,320), Xh_T [320,384), DY_E [384,448),
// DY_T [448,512).  All waits are bounded; a protocol error bumps g_timeout_count_enc instead of hanging the GPU.
#pragma once

constexpr int kS2Threads = 640;
constexpr int kS2Stages = 3;
constexpr int kS2StK = 0, kS2StV = 16384, kS2StRec = 32768, kS2StGate = 32768 + kRecBytes;
constexpr int kS2StageBytes = 32768 + kRecBytes + 1024;
constexpr int kS2OffXch = kS2Stages * kS2StageBytes;  // T chain: row maxima of the two column halves
constexpr int kS2OffBar = kS2OffXch + 1024;
constexpr int kS2Smem = kS2OffBar + 256 + 1024;

struct S2Bars {
  uint64_t st_full[kS2Stages], st_free[kS2Stages];
  uint64_t st_ready[kS2Stages];     // converters -> chains, (1) issuer: the stage's K and V tiles are fp16 (2 arrivals)
  uint64_t m3_done[2], m4_done[2];  // [block]: 0 = E, 1 = T
  uint64_t dy_free;                 // E chain -> V converter (which issues (1)): DY_E may be overwritten
  // Progress counters read with plain acquire loads: an mbarrier probe costs ~380 cycles in this kernel even when the
  // phase completed long ago, and these two sit on the chains' critical path once per chunk.
  int fin_flag;                     // 1 once the V converter has posted p_final / g_total
  int issued1_cnt;                  // chunks whose (1) is in the tensor pipe
  uint32_t tmem_base;
  int abort_flag;
  // scalar gate (lazy decay of the E block): written by the V converter, read by the chains
  float resc[kS2Stages];            // factor the E chain applies to X_E in the pass of the stage's chunk (1 = none)
  float p_final;                    // E = X_E exp(p_final) at write-out
  double g_total;                   // the segment's total log-decay: T = That exp(g_total)
  int bad;                          // a chain saw a non-finite result: the unit goes to the fp32 fallback list
  float fac[1][kC];                 // V converter scratch: this chunk's value weights
};
constexpr float kLazyP = 4.1588831f;  // ln 64: the stored E block runs at most 64x above / below its true scale

__device__ __forceinline__ void tma_load_3d(uint32_t dst_smem, const CUtensorMap* tm, int c0, int c1, int c2,
                                            uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
          dst_smem),
      "l"(reinterpret_cast<uint64_t>(tm)), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
      : "memory");
}

__device__ __noinline__ bool s2_wait(uint64_t* bar, uint32_t parity, volatile int* abort_flag) {
#pragma unroll 1
  for (uint32_t i = 0; i < 4000000u; ++i) {
    if (mbar_try_wait(bar, parity)) return true;
    __nanosleep(20);  // back off: a tight try_wait loop floods the shared-memory pipeline the working warps need
    if ((i & 1023u) == 1023u && *abort_flag) return false;
  }
  if (!*abort_flag) {
    *abort_flag = 1;
    atomicAdd(&g_timeout_count_enc, 1u);
  }
  return false;
}

// single-thread roles (loader, (1) issuer): retry try_wait for a long while before the sleeping fallback -- a thread
// that has gone into s2_wait's __nanosleep loop wakes up thousands of cycles after its barrier completed
__device__ __forceinline__ void s2_wait_spin(uint64_t* bar, uint32_t parity, volatile int* abort_flag) {
#pragma unroll 1
  for (int i = 0; i < 256; ++i)
    if (mbar_try_wait_hint(bar, parity, 20000u)) return;  // suspended in hardware until the phase completes (or 20 us)
  s2_wait(bar, parity, abort_flag);
}

__device__ __forceinline__ void s2_wait_warp(uint64_t* bar, uint32_t parity, volatile int* abort_flag, int) {
  // the chains' waits: try_wait with a suspend-time hint, so that a waiting warp sleeps in hardware until the phase
  // completes instead of re-issuing the probe -- 16 chain warps polling st_ready in a tight loop flooded the
  // shared-memory pipeline and slowed the two converter warps they were waiting for to ~4,000 cycles per tile
  if (mbar_test_wait(bar, parity)) return;  // already complete: the plain probe is cheaper than a suspending one
#pragma unroll 1
  for (int i = 0; i < 64; ++i)
    if (mbar_try_wait_hint(bar, parity, 100000u)) return;
  s2_wait(bar, parity, abort_flag);
}

__device__ __forceinline__ void flag_release(int* p, int v) {
  asm volatile("st.release.cta.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}
__device__ __forceinline__ int flag_acquire(const int* p) {
  int v;
  asm volatile("ld.acquire.cta.shared::cta.b32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
  return v;
}
// bounded spin until *p > c
__device__ __forceinline__ void s2_wait_count(const int* p, int c, volatile int* abort_flag) {
#pragma unroll 1
  for (uint32_t i = 0; i < 40000000u; ++i) {
    if (flag_acquire(p) > c) return;
    if ((i & 4095u) == 4095u && *abort_flag) return;
  }
  if (!*abort_flag) {
    *abort_flag = 1;
    atomicAdd(&g_timeout_count_enc, 1u);
  }
}

// 32 lanes x 16 columns
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t* r) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(taddr),
      "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),
      "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
      : "memory");
}
// (a, b) <- (a, b) * (s0, s1)  as one packed fp32x2 multiply
__device__ __forceinline__ void mul2v(uint32_t& a, uint32_t& b, float s0, float s1) {
  asm("{\n\t.reg .b64 t, u;\n\tmov.b64 t, {%0, %1};\n\tmov.b64 u, {%2, %3};\n\tmul.rn.f32x2 t, t, u;\n\tmov.b64 {%0, %1}, t;\n\t}"
      : "+r"(a), "+r"(b)
      : "r"(__float_as_uint(s0)), "r"(__float_as_uint(s1)));
}
__device__ __forceinline__ void mul2(uint32_t& a, uint32_t& b, float s) { mul2v(a, b, s, s); }
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ float pow2i(int e) { return __uint_as_float((uint32_t)(127 + e) << 23); }  // e in [-126, 127]

// explicit shared-space 128-bit accesses by 32-bit shared address: through a generic pointer derived from the aligned
// dynamic-smem base ptxas emits LD.E / ST.E (generic), which cost the converters ~160 cycles per dependent round trip
__device__ __forceinline__ uint4 lds128(uint32_t a) {
  uint4 v;
  asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ void sts128(uint32_t a, const uint4& v) {
  asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ float lds32f(uint32_t a) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
  return v;
}
// eight bf16 (one 16-byte piece of a TMA box) -> eight fp16 scaled by f
__device__ __forceinline__ uint4 cvt8_bf16_f16(uint4 w, float f) {
  uint32_t a0 = w.x << 16, a1 = w.x & 0xffff0000u, b0 = w.y << 16, b1 = w.y & 0xffff0000u;
  uint32_t c0 = w.z << 16, c1 = w.z & 0xffff0000u, d0 = w.w << 16, d1 = w.w & 0xffff0000u;
  mul2(a0, a1, f);
  mul2(b0, b1, f);
  mul2(c0, c1, f);
  mul2(d0, d1, f);
  return make_uint4(pack_f16(__uint_as_float(a0), __uint_as_float(a1)), pack_f16(__uint_as_float(b0), __uint_as_float(b1)),
                    pack_f16(__uint_as_float(c0), __uint_as_float(c1)), pack_f16(__uint_as_float(d0), __uint_as_float(d1)));
}
__device__ __forceinline__ uint4 cvt8_bf16_f16(uint4 w) {
  return make_uint4(pack_f16(__uint_as_float(w.x << 16), __uint_as_float(w.x & 0xffff0000u)),
                    pack_f16(__uint_as_float(w.y << 16), __uint_as_float(w.y & 0xffff0000u)),
                    pack_f16(__uint_as_float(w.z << 16), __uint_as_float(w.z & 0xffff0000u)),
                    pack_f16(__uint_as_float(w.w << 16), __uint_as_float(w.w & 0xffff0000u)));
}

// MMA batches of one chunk; each is issued by one elected thread of the chain that produced its operands.
__device__ __forceinline__ void s2_issue1(uint32_t tmem, uint32_t sb) {  // DY_E = V^t A_b^t
  constexpr uint32_t id1 = make_idesc(0u, 128, 64, 1, 0);  // fp16, A MN-major (V tile), B K-major (A_b)
#pragma unroll
  for (int ks = 0; ks < 4; ++ks)
    mma_f16_ss(tmem + 384, make_desc(sb + kS2StV + ks * 2048, 8192, 1024, 2),
               make_desc(sb + kS2StRec + kRecAb + ks * 32, 16, 1024, 2), id1, ks > 0);
}
__device__ __forceinline__ void s2_issue3(uint32_t tmem, uint32_t sb, int b) {  // DY_b (+)= Xh_b (-W)^t
  constexpr uint32_t id3 = make_idesc(0u, 128, 64, 0, 0);  // fp16, A from TMEM, B K-major (-W)
#pragma unroll
  for (int ks = 0; ks < 8; ++ks)
    mma_f16_ts(tmem + 384 + 64 * b, tmem + 256 + 64 * b + 8 * ks,
               make_desc(sb + kS2StRec + kRecW + (ks >> 2) * 8192 + (ks & 3) * 32, 16, 1024, 2), id3,
               (b == 0 || ks > 0) ? 1u : 0u);
}
__device__ __forceinline__ void s2_issue4(uint32_t tmem, uint32_t sb, int b) {  // X_b += U''_b K
  constexpr uint32_t id4 = make_idesc(0u, 128, 128, 0, 1);  // fp16, A from TMEM (U''), B MN-major (K tile)
#pragma unroll
  for (int ks = 0; ks < 4; ++ks)
    mma_f16_ts(tmem + 128 * b, tmem + 256 + 64 * b + 8 * ks, make_desc(sb + kS2StK + ks * 2048, 8192, 1024, 2), id4, 1u);
}

template <bool kIsT, bool kCh>
__device__ __forceinline__ void s2_chain(uint8_t* smem, S2Bars* bars, volatile int* abort_flag, uint32_t tmem, int cw,
                                         int lane, int nc, float* __restrict__ dst_block) {
  constexpr int b = kIsT ? 1 : 0;
  constexpr uint32_t cX = kIsT ? 128 : 0, cH = kIsT ? 320 : 256, cD = kIsT ? 448 : 384;
  const int q = cw & 3, hf = cw >> 2;  // TMEM lane quarter; column half
  const int row = 32 * q + lane;
  const uint32_t lane_base = (uint32_t)(32 * q) << 16;
  const uint32_t tX = tmem + cX + lane_base + 64 * hf, tH = tmem + cH + lane_base + 32 * hf,
                 tD = tmem + cD + lane_base + 32 * hf;
  float* xch = reinterpret_cast<float*>(smem + kS2OffXch);
  int s_exp = 0;  // T chain: the TMEM copy of this row is T_row * 2^s_exp

  // X_0 = [0 ; I]
#pragma unroll
  for (int cb = 0; cb < 2; ++cb) {
    uint32_t x[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) x[i] = (kIsT && 64 * hf + 32 * cb + i == row) ? __float_as_uint(1.f) : 0u;
    tmem_st32(tX + 32 * cb, x);
  }
  tmem_st_wait();
  const uint32_t smem_base = smem_u32(smem);
  const bool issuer = (cw == 0 && lane == 0);  // this chain's MMA-issuing thread

#pragma unroll 1
  for (int c = 0; c < nc; ++c) {
    const int st = c % kS2Stages;
    const float* gt = reinterpret_cast<const float*>(smem + st * kS2StageBytes + kS2StGate);
    // converted, hence also landed.  A hardware-suspended mbarrier wait: the chains often arrive first, and a spinning
    // chain (16 warps polling a counter) starved the three converter warps of issue slots (profiles/r02a)
    s2_wait_warp(&bars->st_ready[st], (c / kS2Stages) & 1, abort_flag, lane);
    if (c > 0) s2_wait_warp(&bars->m4_done[b], (c - 1) & 1, abort_flag, lane);
    tc_fence_after();
    const float gC = kCh ? 1.f : gt[kC];  // scalar gate: gamma_C; per-channel gate: Gamma_C[col] = gt[col], applied below
    // ---- pass: Xh = fp16(X) (A operand of (3)), X <- gamma_C X; T rows are re-normalised on the way
    {
      uint32_t x0[32], x1[32];
      tmem_ld32(tX, x0);
      tmem_ld32(tX + 32, x1);
      tmem_ld_wait();
      float f = gC;
      if (kIsT) {
        float m = 0.f;
#pragma unroll
        for (int i = 0; i < 32; ++i) m = fmaxf(m, fmaxf(fabsf(__uint_as_float(x0[i])), fabsf(__uint_as_float(x1[i]))));
        xch[2 * row + hf] = m;
        named_bar_sync(1 + q, 64);
        m = fmaxf(m, xch[2 * row + (hf ^ 1)]);
        // row maximum in [2^(e-127), 2^(e-126)): move it to [2^14, 2^15) -- in place, the row stays normalised
        const int e = (int)(__float_as_uint(m) >> 23);
        int dlt = (e == 0) ? 0 : 141 - e;
        dlt = max(-100, min(100, dlt));
        s_exp += dlt;
        const float sc = pow2i(dlt);
        f = gC * sc;
        if (kCh) {  // per-channel gate: normalise in place, the per-column decay follows below
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            mul2(x0[2 * j], x0[2 * j + 1], sc);
            mul2(x1[2 * j], x1[2 * j + 1], sc);
          }
        } else {    // scalar gate: Xh from x sc, then one multiply by gamma_C sc below
          uint32_t hh[16];
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            uint32_t a0 = x0[2 * j], a1 = x0[2 * j + 1];
            mul2(a0, a1, sc);
            hh[j] = pack_f16(__uint_as_float(a0), __uint_as_float(a1));
          }
          tmem_st16(tH, hh);
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            uint32_t a0 = x1[2 * j], a1 = x1[2 * j + 1];
            mul2(a0, a1, sc);
            hh[j] = pack_f16(__uint_as_float(a0), __uint_as_float(a1));
          }
          tmem_st16(tH + 16, hh);
        }
      }
      if (!kIsT || kCh) {
        uint32_t hh[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) hh[j] = pack_f16(__uint_as_float(x0[2 * j]), __uint_as_float(x0[2 * j + 1]));
        tmem_st16(tH, hh);
#pragma unroll
        for (int j = 0; j < 16; ++j) hh[j] = pack_f16(__uint_as_float(x1[2 * j]), __uint_as_float(x1[2 * j + 1]));
        tmem_st16(tH + 16, hh);
      }
      tmem_st_wait();  // Xh is in TMEM; the decayed X follows while (3) runs (only (4) needs it)
      tc_fence_before();
      named_bar_sync(5 + b, 256);  // the whole chain has written Xh
      if (issuer) {
        if (!kIsT) s2_wait_count(&bars->issued1_cnt, c, abort_flag);  // (1)_c is ahead of (3)_c in the tensor pipe
        tc_fence_after();
        s2_issue3(tmem, smem_base + st * kS2StageBytes, b);
        mma_commit(&bars->m3_done[b]);
      }
      __syncwarp();
      if (kCh) {
        const float4* gv = reinterpret_cast<const float4*>(gt + 64 * hf);
#pragma unroll
        for (int j4 = 0; j4 < 8; ++j4) {
          const float4 a = gv[j4], b4 = gv[8 + j4];
          mul2v(x0[4 * j4], x0[4 * j4 + 1], a.x, a.y);
          mul2v(x0[4 * j4 + 2], x0[4 * j4 + 3], a.z, a.w);
          mul2v(x1[4 * j4], x1[4 * j4 + 1], b4.x, b4.y);
          mul2v(x1[4 * j4 + 2], x1[4 * j4 + 3], b4.z, b4.w);
        }
      } else {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          mul2(x0[2 * j], x0[2 * j + 1], f);
          mul2(x1[2 * j], x1[2 * j + 1], f);
        }
      }
      tmem_st32(tX, x0);
      tmem_st32(tX + 32, x1);
      tmem_st_wait();
    }

    // ---- epilogue: U''[:, j] = fp16(DY[:, j] d_j) -> TMEM (A operand of (4)); this thread: tokens [32 hf, 32 hf + 32)
    s2_wait_warp(&bars->m3_done[b], c & 1, abort_flag, lane);
    tc_fence_after();
    {
      uint32_t y[32];
      tmem_ld32(tD, y);
      tmem_ld_wait();
#pragma unroll
      for (int j8 = 0; j8 < 4; ++j8) {
        float4 d0 = make_float4(1.f, 1.f, 1.f, 1.f), d1 = d0;  // per-channel gate: the decay ratios sit in the K~ tile
        if (!kCh) {
          d0 = *reinterpret_cast<const float4*>(gt + 32 * hf + 8 * j8);
          d1 = *reinterpret_cast<const float4*>(gt + 32 * hf + 8 * j8 + 4);
        }
        const float dd[8] = {d0.x, d0.y, d0.z, d0.w, d1.x, d1.y, d1.z, d1.w};
#pragma unroll
        for (int p = 0; p < 4; ++p) {
          uint32_t u0 = y[8 * j8 + 2 * p], u1 = y[8 * j8 + 2 * p + 1];
          if (!kCh) mul2v(u0, u1, dd[2 * p], dd[2 * p + 1]);
          y[4 * j8 + p] = pack_f16(__uint_as_float(u0), __uint_as_float(u1));  // packed in place: slot 4 j8 + p < 8 j8 + 2 p
        }
      }
      tmem_st16(tH - 16 * hf, y);  // columns [16 hf, 16 hf + 16) of the (dead) Xh region: tokens [32 hf, 32 hf + 32)
      tmem_st_wait();
    }
    tc_fence_before();
    named_bar_sync(5 + b, 256);  // the whole chain has written U''
    if (issuer) {
      if (!kIsT) mbar_arrive(&bars->dy_free);  // DY_E has been read: the V converter may issue (1) of the next chunk
      tc_fence_after();
      s2_issue4(tmem, smem_base + st * kS2StageBytes, b);
      mma_commit(&bars->m4_done[b]);
      mma_commit(&bars->st_free[st]);  // count 2: released when both chains' (4) of this chunk have completed
    }
    __syncwarp();
  }

  // ---- a5: write this thread's 64 columns of its row (T: undo the row normalisation, in two exact steps)
  if (nc > 0) {
    s2_wait_warp(&bars->m4_done[b], (nc - 1) & 1, abort_flag, lane);
    tc_fence_after();
  }
  const int se = max(-250, min(250, s_exp));
  const float f0 = pow2i(-(se / 2)), f1 = pow2i(-(se - se / 2));
  float* dst = dst_block + (size_t)row * kD + 64 * hf;
  bool bad = false;
#pragma unroll 1
  for (int cb = 0; cb < 2; ++cb) {
    uint32_t x[32];
    tmem_ld32(tX + 32 * cb, x);
    tmem_ld_wait();
    float4* d4 = reinterpret_cast<float4*>(dst + 32 * cb);
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      float4 o = make_float4(__uint_as_float(x[4 * u]), __uint_as_float(x[4 * u + 1]), __uint_as_float(x[4 * u + 2]),
                             __uint_as_float(x[4 * u + 3]));
      if (kIsT) {
        o.x = o.x * f0 * f1;
        o.y = o.y * f0 * f1;
        o.z = o.z * f0 * f1;
        o.w = o.w * f0 * f1;
      }
      bad |= !(fabsf(o.x) <= 3.0e38f) | !(fabsf(o.y) <= 3.0e38f) | !(fabsf(o.z) <= 3.0e38f) | !(fabsf(o.w) <= 3.0e38f);
      d4[u] = o;
    }
  }
  if (bad) bars->bad = 1;  // an fp16 operand overflowed somewhere: the unit goes to the fp32 fallback list
}


// (The scalar gate no longer runs through this kernel: encode_scan4.cuh.  scan2_kernel is instantiated for the
// per-channel gate only.)
template <bool kCh>
__global__ void __launch_bounds__(kS2Threads, 1)
    scan2_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                 const int32_t* __restrict__ cu_seqlens, const int32_t* __restrict__ chunk_off,
                 const int32_t* __restrict__ seg_order, int H, const uint8_t* __restrict__ rec, const float* __restrict__ gate, float* __restrict__ E,
                 float* __restrict__ T, int32_t* __restrict__ fb, int n_units) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  S2Bars* bars = reinterpret_cast<S2Bars*>(smem + kS2OffBar);
  volatile int* abort_flag = &bars->abort_flag;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int h = blockIdx.x, s = seg_order[blockIdx.y];  // longest segments first
  const int seg_begin = cu_seqlens[s], seg_end = cu_seqlens[s + 1];
  const int nc = (seg_end - seg_begin + kC - 1) / kC;
  const int chunk0 = chunk_off[s];

  if (warp == 16) tmem_alloc(&bars->tmem_base, 512);
  if (tid == 0) {
    for (int i = 0; i < kS2Stages; ++i) {
      mbar_init(&bars->st_full[i], 1);
      if (i == 0) mbar_init(&bars->dy_free, 1);
      mbar_init(&bars->st_free[i], 2);
      mbar_init(&bars->st_ready[i], 2);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(&bars->m3_done[i], 1);
      mbar_init(&bars->m4_done[i], 1);
    }
    bars->abort_flag = 0;
    bars->bad = 0;
    bars->p_final = 0.f;
    bars->g_total = 0.0;
    bars->fin_flag = bars->issued1_cnt = 0;
    fence_barrier_init();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = bars->tmem_base;
  const uint32_t smem_base = smem_u32(smem);

  if (warp == 18) {
    // ------------------------------------------------------------------------------------------- loader
    if (lane == 0) {
      constexpr uint32_t bytes = 32768u + (uint32_t)kRecBytes + (uint32_t)(kCh ? kGateBytesCh : kGateBytes);
#pragma unroll 1
      for (int c = 0; c < nc; ++c) {
        const int st = c % kS2Stages;
        s2_wait_spin(&bars->st_free[st], ((c / kS2Stages) & 1) ^ 1, abort_flag);
        const uint32_t sb = smem_base + st * kS2StageBytes;
        const int t0 = seg_begin + c * kC;
        mbar_expect_tx(&bars->st_full[st], bytes);
        const size_t r = (size_t)(chunk0 + c) * H + h;
        if (kCh) {  // the K~ tile of the prep record (fp16, same layout as a K tile) takes the K slot
          bulk_g2s(smem + st * kS2StageBytes + kS2StK, rec + r * kRecBytesCh + kRecKt, 2 * kTileB, &bars->st_full[st]);
        } else {
          tma_load_3d(sb + kS2StK, &tmK, 0, h, t0, &bars->st_full[st]);
          tma_load_3d(sb + kS2StK + 8192, &tmK, 64, h, t0, &bars->st_full[st]);
        }
        tma_load_3d(sb + kS2StV, &tmV, 0, h, t0, &bars->st_full[st]);
        tma_load_3d(sb + kS2StV + 8192, &tmV, 64, h, t0, &bars->st_full[st]);
        bulk_g2s(smem + st * kS2StageBytes + kS2StRec, rec + r * (kCh ? kRecBytesCh : kRecBytes), kRecBytes,
                 &bars->st_full[st]);
        bulk_g2s(smem + st * kS2StageBytes + kS2StGate, gate + r * (kCh ? kGateFloatsCh : kGateFloats),
                 kCh ? kGateBytesCh : kGateBytes, &bars->st_full[st]);
      }
    }
  } else if (warp == 19) {
    // ------------------------------------------------------------------------------------------- (1) issuer
    // (1)_c = V^t A_b^t goes to the tensor pipe as soon as the V tile is converted and DY_E is free (the E chain has
    // read it for chunk c - 1) -- a role of its own, so that neither the converters nor the E chain ever wait for it.
    if (lane == 0) {
#pragma unroll 1
      for (int c = 0; c < nc; ++c) {
        const int st = c % kS2Stages;
        s2_wait_spin(&bars->st_ready[st], (c / kS2Stages) & 1, abort_flag);
        if (c > 0) s2_wait_spin(&bars->dy_free, (c - 1) & 1, abort_flag);
        tc_fence_after();
        s2_issue1(tmem, smem_base + st * kS2StageBytes);
        tc_fence_before();
        flag_release(&bars->issued1_cnt, c + 1);
      }
    }
  } else if (warp >= 16) {
    // ------------------------------------------------------------------------------------------- converters
    // bf16 -> fp16 in place (element-wise on 16-bit lanes, so the 128B swizzle of the TMA boxes is untouched): warp 16
    // the K tile, warp 17 the V tile.  Rows at or beyond the segment's end belong to the next segment (or lie past the
    // tensor): they are zeroed, so that nothing of a neighbour -- not even an Inf or NaN -- reaches this unit through
    // 0 x garbage.  Scalar gate: the V converter also runs the lazy-decay automaton of the E block (s2_chain_sc) and
    // folds the value weights into the tile.
    const int role = warp == 16 ? 0 : 1;
    float p_lazy = 0.f;
    double g_tot = 0.0;
    const int seg_len = seg_end - seg_begin;
#pragma unroll 1
    for (int c = 0; c < nc; ++c) {
      const int st = c % kS2Stages;
      s2_wait_warp(&bars->st_full[st], (c / kS2Stages) & 1, abort_flag, lane);
      const int valid = min(kC, seg_len - c * kC);
      const bool weigh = !kCh && role != 0;
      float* fac = bars->fac[0];
      if (weigh) {
        const float* gt = reinterpret_cast<const float*>(smem + st * kS2StageBytes + kS2StGate);  // G_r, inclusive
        const float GC = gt[kC - 1], g0 = gt[lane], g1 = gt[lane + 32];
        const bool rs = !(fabsf(p_lazy + GC) <= kLazyP);  // also NaN
        fac[lane] = rs ? expf(GC - g0) : expf(-(p_lazy + g0));
        fac[lane + 32] = rs ? expf(GC - g1) : expf(-(p_lazy + g1));
        if (role == 1 && lane == 0) bars->resc[st] = rs ? expf(p_lazy + GC) : 1.f;
        p_lazy = rs ? 0.f : p_lazy + GC;
        g_tot += (double)GC;
        __syncwarp();
      }
      const uint32_t tile = smem_base + st * kS2StageBytes + (role == 0 ? kS2StK : kS2StV) + 16 * lane;
      const uint32_t fac_s = smem_u32(fac) + 4 * (lane >> 3);
      if (!(kCh && role == 0)) {  // the K~ tile of the per-channel gate arrives as fp16 (rows past the end are zero)
        // 16-byte piece it * 32 + lane of a box belongs to token 4 (it % 16) + lane / 8; four pieces in flight per lane
#pragma unroll 1
        for (int i0 = 0; i0 < 32; i0 += 4) {
          uint4 w[4];
          float f[4];
#pragma unroll
          for (int j = 0; j < 4; ++j) w[j] = lds128(tile + 512 * (i0 + j));
          if (weigh) {
#pragma unroll
            for (int j = 0; j < 4; ++j) f[j] = lds32f(fac_s + 16 * ((i0 + j) & 15));
          }
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const int tok = 4 * ((i0 + j) & 15) + (lane >> 3);
            uint4 o = weigh ? cvt8_bf16_f16(w[j], f[j]) : cvt8_bf16_f16(w[j]);
            if (tok >= valid) o = make_uint4(0u, 0u, 0u, 0u);
            sts128(tile + 512 * (i0 + j), o);
          }
        }
      }
      fence_proxy_async();
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars->st_ready[st]);
      __syncwarp();
    }
    if (role == 1 && lane == 0) {
      bars->p_final = p_lazy;
      bars->g_total = g_tot;
    }
    if (role == 1 && lane == 0) flag_release(&bars->fin_flag, 1);
  } else if (warp < 8) {
    s2_chain<false, true>(smem, bars, abort_flag, tmem, warp, lane, nc, E + ((size_t)s * H + h) * kD * kD);
  } else {
    s2_chain<true, true>(smem, bars, abort_flag, tmem, warp - 8, lane, nc, T + ((size_t)s * H + h) * kD * kD);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 16) tmem_dealloc(tmem, 512);
  if (tid == 0 && bars->bad) fb_append(fb, n_units, s * H + h);
}
