// encode_scan3.cuh -- the fused segment-encode kernel of the tensor family, scalar gate (GDN row of Table 1).
// Included by encode_tensor.cu inside namespace hypic::{anonymous}; uses the helpers of encode_prep.cuh / encode_scan2.cuh.
//
// One CTA per (segment, head) does rows a0..a5 of SURVEY.md section 8(a) for all of the segment's 64-token chunks: the
// state-independent half of the chunk algebra (Gram, UT solve, W) runs in producer warps two chunks ahead of the
// sequential half, and what it produces (W, A_b) never leaves shared memory -- no prep record in HBM, K read once.
//
// Algebra.  The scalar gate commutes with (I - beta k k^t), so with Gamma(t) the decay from the segment
// start through token t, S_t / Gamma(t) obeys the UNGATED delta rule with values v_t / Gamma(t) and
// T_C = Gamma(L) prod (I - beta k k^t).  Per chunk, all gate-free:
//     (G) Gram = K K^t                     tcgen05, 64 x 64 of a 128-row accumulator (rows 64.. are don't-care)
//         L_rj = beta_r Gram_rj (j < r),  A = (I + L)^-1 (warp-level blocked solve),  A_b = A diag(beta)
//     (W) W^t  = K^t A_b^t                 tcgen05: [dk][token], written out as the MN-major B tile of (3)
//     (1) DY_E  = V^t (A_b diag(f))^t      f_j = the chunk's value weights (lazy decay of the E block, below)
//     (3) DY_b -= Xh_b W^t                 Xh_b = fp16(X_b) read from TMEM
//     (4) X_b  += U''_b K                  U'' = fp16(DY_b) read from TMEM
// for the stacked state X = [E ; T] (two 128-row blocks resident in TMEM as fp32 for the whole segment).
//   T block: rows held as That_r 2^s_r, s_r re-chosen every 8th chunk (row maximum to [2^11, 2^12)); T = exp(sum g) That.
//   E block: stored X_E = E exp(-p), p = pending log-decay; the chunk's values enter with f_j = exp(-(p + G_j)) (G_j the
//            inclusive in-chunk cumulative log-decay).  When |p + G_C| would exceed ln 64 the pass multiplies X_E by
//            exp(p + G_C), f_j = exp(G_C - G_j) <= 1 and p restarts at 0.
// Operands: K is converted bf16 -> fp16 in place by the producer warps; V is used as it arrives (bf16, no conversion
// pass): A_b diag(f) goes to (1) as a bf16 hi + lo pair (16 significant bits), eight kind::f16 MMAs on bf16 operands.
// Legacy mma.sync runs at about an eighth of the tcgen05 rate on this part (measured: ~32 cycles per m16n8k16 and
// sub-partition), which made the Gram and W contractions the bottleneck of both the stand-alone prep kernel and a first
// fused version; they are on tcgen05 here, and only the 16 x 16 merges of the inverse stay on mma.sync.
//
// TMEM columns: X_E [0,128), X_T [128,256), Xh_E [256,320), Xh_T [320,384), DY [384,448) shared by the two chains in
// turn (E's (1) + (3) and epilogue, then T's (3) and epilogue), ACC [448,512) the producers' accumulator (Gram, W^t),
// taken in turn by the two producer groups under a lock.
//
// 19 warps (608 threads, 96 registers each); roles by urgency:
//   warp 0       loader     TMA boxes of K (4-deep ring, two chunks ahead of V) and V (2-deep ring)
//   warp 1       gate       the chunk's g / beta, its cumulative log-decay and the lazy-decay automaton (a ring of 8
//                           gate records)
//   warp 2       V helper   zeroes the rows of a ragged last V tile that belong to the next segment, releases V to (1)
//   warps 3-6    E chain    thread = row of E: pass Xh = fp16(X) (and the lazy rescale), epilogue U'' = fp16(DY);
//                           one elected thread issues the chain's MMA batches (3), (4)
//   warps 7-10   T chain    same for T, plus the row re-normalisation every 8th chunk
//   warps 11-14  producer group 0 (even chunks), warps 15-18 producer group 1 (odd chunks)
#pragma once

constexpr int kF_Threads = 608;
// warp roles.  The warp scheduler of a sub-partition serves its eligible warps lowest warp id first (measured here: as
// warp 16 the loader issued one instruction per ~90 cycles behind the producers' dense mma.sync code), so the roles sit
// in order of urgency: the single-thread roles, the two chains (the critical path), the producers (background work).
constexpr int kF_WLoader = 0, kF_WGate = 1, kF_WIssuer = 2, kF_WChainE = 3, kF_WChainT = 7, kF_WProd = 11;
constexpr int kF_KStages = 4, kF_VStages = 2, kF_Slots = 2, kF_GateSlots = 8;
constexpr int kF_OffK = 0;                                   // 4 x 16 KB: K tile, two 64-column boxes [token][64]
constexpr int kF_OffV = kF_OffK + kF_KStages * 2 * kTileB;   // 2 x 16 KB: V tile (bf16 as it arrives)
constexpr int kF_OffOut = kF_OffV + kF_VStages * 2 * kTileB; // 2 x 32 KB: -W (16 KB), A_b f hi (8 KB), A_b f lo (8 KB)
constexpr int kF_OutW = 0, kF_OutHi = 2 * kTileB, kF_OutLo = 3 * kTileB, kF_OutBytes = 4 * kTileB;
constexpr int kF_OffScr = kF_OffOut + kF_Slots * kF_OutBytes;  // 2 x producer scratch
constexpr int kF_ScrA = 0;                                   // fp32 [64][68]: L, inverted in place to A
constexpr int kF_ScrM = kC * kLPitch * 4;                    // fp32 [32][36]: temporaries of the block merges
constexpr int kF_ScrB = kF_ScrM + 32 * kMPitch * 4;          // fp32 [64] beta, [64] beta f
constexpr int kF_ScrBytes = kF_ScrB + 512;
constexpr int kF_OffGate = kF_OffScr + 2 * kF_ScrBytes;      // 8 x gate record: G_j[64], beta_j[64], p_old, resc, G_C, rs
constexpr int kF_GateFloats = 2 * kC + 4;
constexpr int kF_OffBar = kF_OffGate + kF_GateSlots * kF_GateFloats * 4;
constexpr int kF_Smem = kF_OffBar + 512 + 1024;

struct F_Bars {
  uint64_t k_full[kF_KStages], k_free[kF_KStages];  // TMA landed / both chains' (4) of the stage's chunk completed
  uint64_t k_ready[kF_KStages];                     // the stage's K tile has been converted to fp16 (and a ragged tail zeroed)
  uint64_t v_full[kF_VStages], v_free[kF_VStages];  // TMA landed / (1) of the stage's chunk completed
  uint64_t out_full[kF_Slots], out_free[kF_Slots];  // producer group done (4 warps) / (1) and both (3) completed
  uint64_t gate_full[kF_GateSlots];                 // loader wrote the chunk's gate record
  uint64_t m3_done[2], m4_done[2];                  // [block]: 0 = E, 1 = T
  uint64_t dy_for_t, dy_for_e;                      // the shared DY columns: E's epilogue has read them / T's has (128 arrivals)
  uint64_t v_ok[kF_VStages];                        // the V tile has landed and a ragged tail is zeroed
  uint64_t acc_done[2];                             // [producer group]: its MMAs into ACC have completed
  int acc_lock;                                     // ACC is taken (one producer group at a time)
  int fin_flag;                                     // the loader has posted p_final / g_total
  uint32_t tmem_base;
  int abort_flag;
  int bad;
  float p_final;
  double g_total;
};

// byte offset of element (row = token, col = dk) inside a K / V tile: box col / 64, 128-byte rows, 128B swizzle
__device__ __forceinline__ uint32_t f_tile_off(int row, int col) {
  return (uint32_t)((col >> 6) * 8192 + row * 128 + ((((col & 63) >> 3) ^ (row & 7)) << 4) + (col & 7) * 2);
}
__device__ __forceinline__ void sts32(uint32_t a, uint32_t v) { asm volatile("st.shared.b32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ uint32_t pack_bf16_rn(float lo, float hi) {
  __nv_bfloat162 p = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&p);
}

// Waits of the background roles (producers, loader, gate, V helper): they run chunks ahead of the chains, so a late
// wake-up costs nothing, while a tight probe loop takes issue slots from the warps on the critical path (ncu: half of
// all executed instructions were mbarrier probes).
__device__ __forceinline__ void f_wait_lazy(uint64_t* bar, uint32_t parity, volatile int* abort_flag) {
#pragma unroll 1
  for (int i = 0; i < 200000; ++i) {
    if (mbar_try_wait(bar, parity)) return;
    __nanosleep(500);
  }
  s2_wait(bar, parity, abort_flag);
}

constexpr uint32_t kF_DY = 384, kF_ACC = 448;
// ---- MMA bursts.  Each is ONE asm block executed by a whole converged warp (warp-uniform control flow): one elected lane
// issues, descriptors and TMEM addresses advance inside the block, and the commits ride along.  Issued from a
// lane-divergent branch (`if (lane == 0)`), ptxas wraps every tcgen05.mma in an ELECT / R2UR.BROADCAST x 5 / branch
// loop of ~21 dependent instructions -- ~100 cycles of issue time per MMA, 44 MMAs per chunk; in this form the
// UTCHMMAs come out back to back on the uniform datapath.
// Descriptor arithmetic: the low 14 bits hold (address >> 4); steps used: 16 rows of a 128-byte-row tile = 2048 B =
// +128, 32 B inside a row = +2, the next 64-column box = 8192 B = +512.
#define F_MMA_TS "@P tcgen05.mma.cta_group::1.kind::f16 [%0], [at], bd, %3, Q;\n\t"
#define F_MMA_SS "@P tcgen05.mma.cta_group::1.kind::f16 [%0], ad, bd, %3, Q;\n\t"
#define F_COMMIT(n) "@P tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%" #n "];\n\t"
// (3): DY (+)= Xh_b (-W)^t -- A = Xh from TMEM (8 columns per k-step), B = the slot's W^t tile (MN-major, negated by the
// instruction descriptor); then commits to m3_done and to the slot's out_free, and to v_free for the E chain.
__device__ __forceinline__ void f_issue3(uint32_t d_tmem, uint32_t a_tmem, uint32_t w_tile, uint32_t acc_first,
                                         uint64_t* bar0, uint64_t* bar1, uint64_t* bar2) {
  constexpr uint32_t id3 = make_idesc(0u, 128, 64, 0, 1, 0, 1);
  const uint64_t bd0 = make_desc(w_tile, 8192, 1024, 2);
  const uint32_t b2 = bar2 ? smem_u32(bar2) : 0u;
  asm volatile(
      "{\n\t.reg .pred P, Q, R;\n\t.reg .b64 bd;\n\t.reg .b32 at;\n\t"
      "elect.sync _|P, 0xffffffff;\n\t"
      "setp.ne.b32 Q, %4, 0;\n\tsetp.ne.b32 R, %7, 0;\n\tand.pred R, R, P;\n\t"
      "mov.b64 bd, %2;\n\tmov.b32 at, %1;\n\t" F_MMA_TS
      "setp.ne.b32 Q, 1, 0;\n\t"
      "add.s64 bd, bd, 128;\n\tadd.s32 at, at, 8;\n\t" F_MMA_TS
      "add.s64 bd, bd, 128;\n\tadd.s32 at, at, 8;\n\t" F_MMA_TS
      "add.s64 bd, bd, 128;\n\tadd.s32 at, at, 8;\n\t" F_MMA_TS
      "add.s64 bd, bd, 128;\n\tadd.s32 at, at, 8;\n\t" F_MMA_TS
      "add.s64 bd, bd, 128;\n\tadd.s32 at, at, 8;\n\t" F_MMA_TS
      "add.s64 bd, bd, 128;\n\tadd.s32 at, at, 8;\n\t" F_MMA_TS
      "add.s64 bd, bd, 128;\n\tadd.s32 at, at, 8;\n\t" F_MMA_TS
      F_COMMIT(5) F_COMMIT(6)
      "@R tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%7];\n\t"
      "}" ::"r"(d_tmem), "r"(a_tmem), "l"(bd0), "r"(id3), "r"(acc_first), "r"(smem_u32(bar0)), "r"(smem_u32(bar1)), "r"(b2)
      : "memory");
}
// (4): X_b += U''_b K -- A = U'' from TMEM, B = the K tile (MN-major, two 64-column boxes); commits to m4_done, k_free
__device__ __forceinline__ void f_issue4(uint32_t d_tmem, uint32_t a_tmem, uint32_t k_tile, uint64_t* bar0, uint64_t* bar1) {
  constexpr uint32_t id4 = make_idesc(0u, 128, 128, 0, 1);
  const uint64_t bd0 = make_desc(k_tile, 8192, 1024, 2);
  asm volatile(
      "{\n\t.reg .pred P, Q;\n\t.reg .b64 bd;\n\t.reg .b32 at;\n\t"
      "elect.sync _|P, 0xffffffff;\n\t"
      "setp.ne.b32 Q, 1, 0;\n\t"
      "mov.b64 bd, %2;\n\tmov.b32 at, %1;\n\t" F_MMA_TS
      "add.s64 bd, bd, 128;\n\tadd.s32 at, at, 8;\n\t" F_MMA_TS
      "add.s64 bd, bd, 128;\n\tadd.s32 at, at, 8;\n\t" F_MMA_TS
      "add.s64 bd, bd, 128;\n\tadd.s32 at, at, 8;\n\t" F_MMA_TS
      F_COMMIT(4) F_COMMIT(5)
      "}" ::"r"(d_tmem), "r"(a_tmem), "l"(bd0), "r"(id4), "r"(smem_u32(bar0)), "r"(smem_u32(bar1))
      : "memory");
}
// (1): DY = V^t (A_b f)^t on bf16 operands -- A = the V tile (MN-major, +128 per 16 tokens), B = the hi tile then the lo
// tile of A_b diag(f) (K-major, +2 per 16 tokens; lo = hi + 8192 B); no commit: (3) of the same chunk follows
__device__ __forceinline__ void f_issue1(uint32_t d_tmem, uint32_t v_tile, uint32_t hi_tile) {
  constexpr uint32_t id1 = make_idesc(1u, 128, 64, 1, 0);
  const uint64_t ad0 = make_desc(v_tile, 8192, 1024, 2), bd0 = make_desc(hi_tile, 16, 1024, 2);
  asm volatile(
      "{\n\t.reg .pred P, Q;\n\t.reg .b64 ad, bd;\n\t"
      "elect.sync _|P, 0xffffffff;\n\t"
      "setp.ne.b32 Q, 0, 0;\n\t"
      "mov.b64 ad, %1;\n\tmov.b64 bd, %2;\n\t" F_MMA_SS
      "setp.ne.b32 Q, 1, 0;\n\t"
      "add.s64 ad, ad, 128;\n\tadd.s64 bd, bd, 2;\n\t" F_MMA_SS
      "add.s64 ad, ad, 128;\n\tadd.s64 bd, bd, 2;\n\t" F_MMA_SS
      "add.s64 ad, ad, 128;\n\tadd.s64 bd, bd, 2;\n\t" F_MMA_SS
      "mov.b64 ad, %1;\n\tadd.s64 bd, bd, 506;\n\t" F_MMA_SS
      "add.s64 ad, ad, 128;\n\tadd.s64 bd, bd, 2;\n\t" F_MMA_SS
      "add.s64 ad, ad, 128;\n\tadd.s64 bd, bd, 2;\n\t" F_MMA_SS
      "add.s64 ad, ad, 128;\n\tadd.s64 bd, bd, 2;\n\t" F_MMA_SS
      "}" ::"r"(d_tmem), "l"(ad0), "l"(bd0), "r"(id1)
      : "memory");
}
// (G): ACC[0:64, 0:64] = K K^t -- A = B = the fp16 K tile, K-major, two 64-column boxes.  M = 128: the A rows 64..127 run
// on into whatever follows the 64-row box (valid shared memory); their results land in TMEM lanes 64..127 and are never
// read.  An M = 64 instruction costs the same tensor time.  Commits to the group's acc_done.
__device__ __forceinline__ void f_issue_gram(uint32_t d_tmem, uint32_t k_tile, uint64_t* bar0) {
  constexpr uint32_t idg = make_idesc(0u, 128, 64, 0, 0);
  const uint64_t d0 = make_desc(k_tile, 16, 1024, 2);
  asm volatile(
      "{\n\t.reg .pred P, Q;\n\t.reg .b64 ad, bd;\n\t"
      "elect.sync _|P, 0xffffffff;\n\t"
      "setp.ne.b32 Q, 0, 0;\n\t"
      "mov.b64 ad, %1;\n\tmov.b64 bd, %1;\n\t" F_MMA_SS
      "setp.ne.b32 Q, 1, 0;\n\t"
      "add.s64 ad, ad, 2;\n\tmov.b64 bd, ad;\n\t" F_MMA_SS
      "add.s64 ad, ad, 2;\n\tmov.b64 bd, ad;\n\t" F_MMA_SS
      "add.s64 ad, ad, 2;\n\tmov.b64 bd, ad;\n\t" F_MMA_SS
      "add.s64 ad, ad, 506;\n\tmov.b64 bd, ad;\n\t" F_MMA_SS
      "add.s64 ad, ad, 2;\n\tmov.b64 bd, ad;\n\t" F_MMA_SS
      "add.s64 ad, ad, 2;\n\tmov.b64 bd, ad;\n\t" F_MMA_SS
      "add.s64 ad, ad, 2;\n\tmov.b64 bd, ad;\n\t" F_MMA_SS
      F_COMMIT(2)
      "}" ::"r"(d_tmem), "l"(d0), "r"(smem_u32(bar0)), "r"(idg)
      : "memory");
}
// (W): ACC = K^t A_b^t = W^t -- A = the K tile MN-major (+128 per 16 tokens), B = the A_b tile K-major (+2); commits to
// the group's acc_done
__device__ __forceinline__ void f_issue_w(uint32_t d_tmem, uint32_t k_tile, uint32_t ab_tile, uint64_t* bar0) {
  constexpr uint32_t idw = make_idesc(0u, 128, 64, 1, 0);
  const uint64_t ad0 = make_desc(k_tile, 8192, 1024, 2), bd0 = make_desc(ab_tile, 16, 1024, 2);
  asm volatile(
      "{\n\t.reg .pred P, Q;\n\t.reg .b64 ad, bd;\n\t"
      "elect.sync _|P, 0xffffffff;\n\t"
      "setp.ne.b32 Q, 0, 0;\n\t"
      "mov.b64 ad, %1;\n\tmov.b64 bd, %2;\n\t" F_MMA_SS
      "setp.ne.b32 Q, 1, 0;\n\t"
      "add.s64 ad, ad, 128;\n\tadd.s64 bd, bd, 2;\n\t" F_MMA_SS
      "add.s64 ad, ad, 128;\n\tadd.s64 bd, bd, 2;\n\t" F_MMA_SS
      "add.s64 ad, ad, 128;\n\tadd.s64 bd, bd, 2;\n\t" F_MMA_SS
      F_COMMIT(4)
      "}" ::"r"(d_tmem), "l"(ad0), "l"(bd0), "r"(idw), "r"(smem_u32(bar0))
      : "memory");
}
// ACC lock (one thread per producer group)
__device__ __forceinline__ void f_acc_acquire(int* lock) {
  const uint32_t a = smem_u32(lock);
  uint32_t old;
#pragma unroll 1
  for (int i = 0; i < 4000000; ++i) {
    asm volatile("atom.acquire.cta.shared::cta.cas.b32 %0, [%1], 0, 1;" : "=r"(old) : "r"(a) : "memory");
    if (old == 0u) return;
    __nanosleep(64);
  }
}
__device__ __forceinline__ void f_acc_release(int* lock) { flag_release(lock, 0); }

// ---------------------------------------------------------------------------------------------------- chains
// One body for both chains (kIsT is a run-time flag): the 19 warps of this kernel run six different roles, and with the
// two chains instantiated separately the hot code no longer fitted the instruction caches (ncu: 3.7 warps per issue
// stalled on "no instruction").
__device__ __noinline__ void f_chain(const bool kIsT, uint8_t* smem, F_Bars* bars, volatile int* abort_flag, uint32_t tmem,
                                     int cw, int lane, int nc, float* __restrict__ dst_block) {
  const int b = kIsT ? 1 : 0;
  const uint32_t cX = kIsT ? 128 : 0, cH = kIsT ? 320 : 256, cD = kF_DY;
  const int wq = cw & 3;           // a warp reaches the TMEM lane quarter warp id % 4; a chain's four warps cover all four
  const int row = 32 * wq + lane;
  const uint32_t lane_base = (uint32_t)(32 * wq) << 16;
  const uint32_t tX = tmem + cX + lane_base, tH = tmem + cH + lane_base, tD = tmem + cD + lane_base;
  const uint32_t smem_base = smem_u32(smem);
  const float* gate_ring = reinterpret_cast<const float*>(smem + kF_OffGate);
  int s_exp = 0;  // T chain: the TMEM copy of this row is That_row * 2^s_exp
  const bool issue_warp = (cw == (kIsT ? kF_WChainT : kF_WChainE));  // warp-uniform: the bursts elect their lane

  // X_0 = [0 ; I]
#pragma unroll
  for (int cb = 0; cb < 4; ++cb) {
    uint32_t x[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) x[i] = (kIsT && 32 * cb + i == row) ? __float_as_uint(1.f) : 0u;
    tmem_st32(tX + 32 * cb, x);
  }
  tmem_st_wait();

#pragma unroll 1
  for (int c = 0; c < nc; ++c) {
    const int slot = c & 1, kst = c % kF_KStages;
    const uint32_t out = smem_base + kF_OffOut + slot * kF_OutBytes;
    s2_wait_warp(&bars->out_full[slot], (c >> 1) & 1, abort_flag, lane);  // -W, A_b and the fp16 K tile are in place
    if (c > 0) s2_wait_warp(&bars->m4_done[b], (c - 1) & 1, abort_flag, lane);
    tc_fence_after();
    // ---- pass: Xh = fp16(X), 32 columns at a time; X itself is only rewritten on a rescale
    {
      float f = 1.f;
      bool rewrite;
      if (kIsT) {
        rewrite = (c & 7) == 0;
        if (rewrite) {  // the whole row lives in this thread: row maximum -> power-of-two scale
          float m = 0.f;
#pragma unroll 1
          for (int cb = 0; cb < 4; ++cb) {
            uint32_t x[32];
            tmem_ld32(tX + 32 * cb, x);
            tmem_ld_wait();
#pragma unroll
            for (int i = 0; i < 32; ++i) m = fmaxf(m, fabsf(__uint_as_float(x[i])));
          }
          const int e = (int)((__float_as_uint(m) >> 23) & 0xffu);  // row maximum in [2^(e-127), 2^(e-126))
          int dlt = (e == 0 || e == 255) ? 0 : 138 - e;             // -> [2^11, 2^12)
          dlt = max(-100, min(100, dlt));
          s_exp += dlt;
          f = pow2i(dlt);
        }
      } else {
        f = gate_ring[(c & (kF_GateSlots - 1)) * kF_GateFloats + 2 * kC + 1];
        rewrite = (f != 1.f);
      }
      {
        uint32_t xa[32], xb[32], hh[16];
        tmem_ld32(tX, xa);
#pragma unroll
        for (int cb = 0; cb < 4; cb += 2) {  // the next 32 columns are in flight while these are converted
          tmem_ld_wait();
          tmem_ld32(tX + 32 * (cb + 1), xb);
          if (rewrite) {
#pragma unroll
            for (int j = 0; j < 16; ++j) mul2(xa[2 * j], xa[2 * j + 1], f);
            tmem_st32(tX + 32 * cb, xa);  // (3) reads Xh alone; (4) of this chunk is issued after the chain barrier below
          }
#pragma unroll
          for (int j = 0; j < 16; ++j) hh[j] = pack_f16(__uint_as_float(xa[2 * j]), __uint_as_float(xa[2 * j + 1]));
          tmem_st16(tH + 16 * cb, hh);
          tmem_ld_wait();
          if (cb + 2 < 4) tmem_ld32(tX + 32 * (cb + 2), xa);
          if (rewrite) {
#pragma unroll
            for (int j = 0; j < 16; ++j) mul2(xb[2 * j], xb[2 * j + 1], f);
            tmem_st32(tX + 32 * (cb + 1), xb);
          }
#pragma unroll
          for (int j = 0; j < 16; ++j) hh[j] = pack_f16(__uint_as_float(xb[2 * j]), __uint_as_float(xb[2 * j + 1]));
          tmem_st16(tH + 16 * (cb + 1), hh);
        }
      }
      tmem_st_wait();
      tc_fence_before();
      named_bar_sync(1 + b, 128);  // the whole chain has written Xh
      if (issue_warp) {
        // The DY columns are shared by the two chains in turn.  E: (1) and (3) of this chunk go to the tensor pipe in one
        // burst once T's epilogue of the previous chunk has read DY; T: (3) follows E's epilogue of this chunk.
        if (!kIsT) {
          if (c > 0) s2_wait_warp(&bars->dy_for_e, (c - 1) & 1, abort_flag, lane);
          s2_wait_warp(&bars->v_ok[slot], (c >> 1) & 1, abort_flag, lane);
          tc_fence_after();
          f_issue1(tmem + kF_DY, smem_base + kF_OffV + slot * 2 * kTileB, out + kF_OutHi);
        } else {
          s2_wait_warp(&bars->dy_for_t, c & 1, abort_flag, lane);
          tc_fence_after();
        }
        // commits: m3_done; out_free (count 2: both chains' (3) -- and with E's, (1) -- have read the slot); E: v_free
        f_issue3(tmem + kF_DY, tmem + cH, out + kF_OutW, kIsT ? 0u : 1u, &bars->m3_done[b], &bars->out_free[slot],
                 kIsT ? nullptr : &bars->v_free[slot]);
      }
    }
    // ---- epilogue: U'' = fp16(DY) -> TMEM (A operand of (4)), tokens [32 cb, 32 cb + 32) -> columns [16 cb, 16 cb + 16).
    // DY is handed to the other chain as soon as this thread's loads have completed (128 arrivals), before the conversion.
    s2_wait_warp(&bars->m3_done[b], c & 1, abort_flag, lane);
    tc_fence_after();
    {
      uint32_t y0[32], y1[32];
      tmem_ld32(tD, y0);
      tmem_ld32(tD + 32, y1);
      tmem_ld_wait();
      tc_fence_before();
      mbar_arrive(kIsT ? &bars->dy_for_e : &bars->dy_for_t);
#pragma unroll
      for (int j = 0; j < 16; ++j) y0[j] = pack_f16(__uint_as_float(y0[2 * j]), __uint_as_float(y0[2 * j + 1]));  // slot j <= 2 j
      tmem_st16(tH, y0);
#pragma unroll
      for (int j = 0; j < 16; ++j) y1[j] = pack_f16(__uint_as_float(y1[2 * j]), __uint_as_float(y1[2 * j + 1]));
      tmem_st16(tH + 16, y1);
    }
    tmem_st_wait();
    tc_fence_before();
    named_bar_sync(1 + b, 128);  // the whole chain has written U''
    if (issue_warp) {
      tc_fence_after();
      // commits: m4_done; k_free (count 2: both chains' (4) of this chunk have completed)
      f_issue4(tmem + cX, tmem + cH, smem_base + kF_OffK + kst * 2 * kTileB, &bars->m4_done[b], &bars->k_free[kst]);
    }
  }

  // ---- a5: write this thread's row; the gate (and T's row scale) is applied here, in fp64, so that a T that underflows
  // fp32 underflows exactly like the correctly rounded result
  s2_wait_count(&bars->fin_flag, 0, abort_flag);  // the loader has posted p_final and g_total
  if (nc > 0) {
    s2_wait_warp(&bars->m4_done[b], (nc - 1) & 1, abort_flag, lane);
    tc_fence_after();
  }
  const double sc = kIsT ? exp(bars->g_total - 0.6931471805599453 * (double)s_exp) : (double)expf(bars->p_final);
  float* dst = dst_block + (size_t)row * kD;
  bool bad = false;
#pragma unroll 1
  for (int cb = 0; cb < 4; ++cb) {
    uint32_t x[32];
    tmem_ld32(tX + 32 * cb, x);
    tmem_ld_wait();
    float4* d4 = reinterpret_cast<float4*>(dst + 32 * cb);
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      float4 o;
      o.x = (float)((double)__uint_as_float(x[4 * u]) * sc);
      o.y = (float)((double)__uint_as_float(x[4 * u + 1]) * sc);
      o.z = (float)((double)__uint_as_float(x[4 * u + 2]) * sc);
      o.w = (float)((double)__uint_as_float(x[4 * u + 3]) * sc);
      bad |= !(fabsf(o.x) <= 3.0e38f) | !(fabsf(o.y) <= 3.0e38f) | !(fabsf(o.z) <= 3.0e38f) | !(fabsf(o.w) <= 3.0e38f);
      d4[u] = o;
    }
  }
  if (bad) bars->bad = 1;  // an fp16 operand overflowed somewhere: the unit goes to the fp32 fallback list
}

// ---------------------------------------------------------------------------------------------------- producers
// One chunk of the state-independent half, by one group of four warps (gtid = 0..127; `wq` = the TMEM lane quarter the
// warp can reach): the chunk's K tile `kt` (shared address, bf16 as TMA delivered it) is converted to fp16 in place, then
// Gram (tcgen05) -> L -> A = (I + L)^-1 -> A_b, A_b f -> W^t (tcgen05) -> the MN-major W tile of (3).
__device__ __forceinline__ void f_produce(uint8_t* smem, F_Bars* bars, volatile int* abort_flag, uint32_t tmem, int gi,
                                          int gtid, int wq, int c, int valid, uint32_t kt, uint32_t out) {
  const int warp = gtid >> 5, lane = gtid & 31;
  uint8_t* scr = smem + kF_OffScr + gi * kF_ScrBytes;
  float* s_a = reinterpret_cast<float*>(scr + kF_ScrA);
  float* s_m = reinterpret_cast<float*>(scr + kF_ScrM);
  float* s_b = reinterpret_cast<float*>(scr + kF_ScrB);
  float* s_bf = s_b + kC;
  const float* gr = reinterpret_cast<const float*>(smem + kF_OffGate) + (c & (kF_GateSlots - 1)) * kF_GateFloats;
  const uint32_t acc_t = tmem + kF_ACC + ((uint32_t)(32 * wq) << 16);
  const int it = c >> 1;  // this group's chunk counter: phase of acc_done is 2 it (Gram), 2 it + 1 (W)

  if (gtid < kC) {  // beta and the value weights f_j of the lazy decay
    const float bj = gr[kC + gtid], Gj = gr[gtid];
    const float p_old = gr[2 * kC], GC = gr[2 * kC + 2], rs = gr[2 * kC + 3];
    s_b[gtid] = bj;
    s_bf[gtid] = bj * (rs != 0.f ? expf(GC - Gj) : expf(-(p_old + Gj)));
  }
  named_bar_sync(3 + gi, 128);

  // ---- a2: Gram on the tensor pipe, then L_rj = beta_r Gram_rj (j < r) into s_a (the upper triangle as zeros)
  if (wq == 0) {
    if (lane == 0) f_acc_acquire(&bars->acc_lock);
    __syncwarp();
    tc_fence_after();
    f_issue_gram(tmem + kF_ACC, kt, &bars->acc_done[gi]);
  }
  if (wq < 2) {  // Gram rows 0..63 sit in TMEM lanes 0..63: the two warps of the group that reach them
    s2_wait_warp(&bars->acc_done[gi], (2 * it) & 1, abort_flag, lane);
    tc_fence_after();
    const int r = 32 * wq + lane;
    const float br = s_b[r];
#pragma unroll 1
    for (int cb = 0; cb < 2; ++cb) {
      uint32_t x[32];
      tmem_ld32(acc_t + 32 * cb, x);
      tmem_ld_wait();
#pragma unroll
      for (int j4 = 0; j4 < 8; ++j4) {
        float4 o;
        const int j = 32 * cb + 4 * j4;
        o.x = (j + 0 < r) ? br * __uint_as_float(x[4 * j4 + 0]) : 0.f;
        o.y = (j + 1 < r) ? br * __uint_as_float(x[4 * j4 + 1]) : 0.f;
        o.z = (j + 2 < r) ? br * __uint_as_float(x[4 * j4 + 2]) : 0.f;
        o.w = (j + 3 < r) ? br * __uint_as_float(x[4 * j4 + 3]) : 0.f;
        *reinterpret_cast<float4*>(s_a + r * kLPitch + j) = o;
      }
    }
    tc_fence_before();
  }
  named_bar_sync(3 + gi, 128);
  if (gtid == 0) f_acc_release(&bars->acc_lock);

  // ---- a3 (i): diagonal blocks D_w = (I + L_ww)^-1 in place, lane c < 16 = column c, row-oriented substitution
  {
    float* blk = s_a + (16 * warp) * kLPitch + 16 * warp;
    float a[16];
    const int cc = lane & 15;
#pragma unroll
    for (int r = 0; r < 16; ++r) {
      float part[4] = {(r == cc) ? 1.f : 0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int j4 = 0; j4 < (r + 3) / 4; ++j4) {
        const float4 l = *reinterpret_cast<const float4*>(blk + r * kLPitch + 4 * j4);
        if (4 * j4 + 0 < r) part[j4] = fmaf(-l.x, a[4 * j4 + 0], part[j4]);
        if (4 * j4 + 1 < r) part[j4] = fmaf(-l.y, a[4 * j4 + 1], part[j4]);
        if (4 * j4 + 2 < r) part[j4] = fmaf(-l.z, a[4 * j4 + 2], part[j4]);
        if (4 * j4 + 3 < r) part[j4] = fmaf(-l.w, a[4 * j4 + 3], part[j4]);
      }
      a[r] = (part[0] + part[1]) + (part[2] + part[3]);
    }
    __syncwarp();
    if (lane < 16) {
#pragma unroll
      for (int r = 0; r < 16; ++r) blk[r * kLPitch + cc] = a[r];
    }
  }
  named_bar_sync(3 + gi, 128);
  auto B = [&](int i, int j) { return s_a + (16 * i) * kLPitch + 16 * j; };
  // ---- a3 (ii): A10 = -D1 (L10 D0) (warp 0), A32 = -D3 (L32 D2) (warp 1); single-pass fp16 products on mma.sync (A only
  // feeds the 16-bit tiles below; emulation: no change in E / T error against fp32-quality merges)
  if (warp < 2) {
    const int i = 2 * warp + 1, j = 2 * warp;
    float* tmp = s_m + (16 * warp) * kMPitch;
    const float* xs[2] = {B(i, j), B(i, i)};
    const float* ys[2] = {B(j, j), tmp};
    const int yp[2] = {kLPitch, kMPitch};
#pragma unroll 1
    for (int st = 0; st < 2; ++st) {  // tmp = L10 D0, then A10 = -D1 tmp (one inlined product: code size)
      float acc[2][4];
      block_zero(acc);
      block_mma_16<false>(acc, xs[st], kLPitch, ys[st], yp[st], lane);
      __syncwarp();
      block_store_16(acc, st == 0 ? 1.f : -1.f, st == 0 ? tmp : B(i, j), st == 0 ? kMPitch : kLPitch, lane);
      __syncwarp();
    }
  }
  named_bar_sync(3 + gi, 128);
  // ---- a3 (iii): the 32 x 32 block A[2:4, 0:2] = -A[2:4, 2:4] (L[2:4, 0:2] A[0:2, 0:2]); warp -> block (2 + w/2, w%2)
  {
    const int i = 2 + (warp >> 1), j = warp & 1;
#pragma unroll 1
    for (int st = 0; st < 2; ++st) {
      // st 0: tmp_ij = L_i0 A_0j (j = 0 only) + L_i1 A_1j;  st 1: A_ij = -(A_i2 tmp_0j + A_i3 tmp_1j (i = 3 only))
      float acc[2][4];
      block_zero(acc);
#pragma unroll 1
      for (int t = 0; t < 2; ++t) {
        const bool use = st == 0 ? (t == 1 || j == 0) : (t == 0 || i == 3);
        if (!use) continue;
        const float* x = st == 0 ? B(i, t) : B(i, 2 + t);
        const float* y = st == 0 ? B(t, j) : s_m + (16 * t) * kMPitch + 16 * j;
        block_mma_16<false>(acc, x, kLPitch, y, st == 0 ? kLPitch : kMPitch, lane);
      }
      if (st == 0) {
        block_store_16(acc, 1.f, s_m + (16 * (i - 2)) * kMPitch + 16 * j, kMPitch, lane);
        named_bar_sync(3 + gi, 128);
      } else {
        block_store_16(acc, -1.f, B(i, j), kLPitch, lane);
      }
    }
  }
  named_bar_sync(3 + gi, 128);

  // the output slot is free once (1) and both (3) of chunk c - 2 have completed
  if (c >= kF_Slots) f_wait_lazy(&bars->out_free[c & 1], ((c >> 1) - 1) & 1, abort_flag);

  // ---- A_b = A diag(beta) as an fp16 B tile (the B operand of the W contraction; it borrows the upper half of the
  // slot's W tile, which is only written once that contraction has completed) and A_b f = A diag(beta f) as a bf16
  // hi + lo pair of B tiles for (1).  All K-major, 128B swizzle: row r, 16-byte piece j8 at ((j8 ^ (r & 7)) * 16).
  // Columns of tokens past the segment's end carry beta = 0.
  const uint32_t ab_tile = out + kF_OutW + 8192;
#pragma unroll 1
  for (int i0 = 0; i0 < kC * 8 / 128; ++i0) {
    const int idx = gtid + i0 * 128;
    const int r = idx >> 3, j8 = idx & 7;
    const float4 v0 = *reinterpret_cast<const float4*>(s_a + r * kLPitch + 8 * j8);
    const float4 v1 = *reinterpret_cast<const float4*>(s_a + r * kLPitch + 8 * j8 + 4);
    const float av[8] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w};
    uint32_t hi[4], lo[4], ab[4];
#pragma unroll
    for (int p2 = 0; p2 < 4; ++p2) {
      const float2 bb = *reinterpret_cast<const float2*>(s_b + 8 * j8 + 2 * p2);
      const float2 bf = *reinterpret_cast<const float2*>(s_bf + 8 * j8 + 2 * p2);
      ab[p2] = pack_f16(av[2 * p2] * bb.x, av[2 * p2 + 1] * bb.y);
      const float x0 = av[2 * p2] * bf.x, x1 = av[2 * p2 + 1] * bf.y;
      const __nv_bfloat162 h2 = __floats2bfloat162_rn(x0, x1);
      const float2 hf = __bfloat1622float2(h2);
      hi[p2] = *reinterpret_cast<const uint32_t*>(&h2);
      lo[p2] = pack_bf16_rn(x0 - hf.x, x1 - hf.y);
    }
    const uint32_t off = (r >> 3) * 1024 + (r & 7) * 128 + ((j8 ^ (r & 7)) * 16);
    sts128(ab_tile + off, make_uint4(ab[0], ab[1], ab[2], ab[3]));
    sts128(out + kF_OutHi + off, make_uint4(hi[0], hi[1], hi[2], hi[3]));
    sts128(out + kF_OutLo + off, make_uint4(lo[0], lo[1], lo[2], lo[3]));
  }
  fence_proxy_async();
  named_bar_sync(3 + gi, 128);

  // ---- W^t = K^t A_b^t on the tensor pipe: thread = dk index c' holds W[0..63][c']; packed as token pairs into row c'
  // of the slot's W tile ([dk][token], 128-byte rows, 128B swizzle: the MN-major B operand of (3))
  if (wq == 0) {
    if (lane == 0) f_acc_acquire(&bars->acc_lock);
    __syncwarp();
    tc_fence_after();
    f_issue_w(tmem + kF_ACC, kt, ab_tile, &bars->acc_done[gi]);
  }
  s2_wait_warp(&bars->acc_done[gi], (2 * it + 1) & 1, abort_flag, lane);
  tc_fence_after();
  {
    const int cr = 32 * wq + lane;  // dk index = TMEM lane
    const uint32_t wrow = out + kF_OutW + (cr >> 3) * 1024 + (cr & 7) * 128;
#pragma unroll 1
    for (int cb = 0; cb < 2; ++cb) {
      uint32_t x[32];
      tmem_ld32(acc_t + 32 * cb, x);
      tmem_ld_wait();
#pragma unroll
      for (int p8 = 0; p8 < 4; ++p8) {  // tokens 32 cb + 8 p8 .. + 7 -> 16-byte piece 4 cb + p8 of the row
        const uint4 o = make_uint4(pack_f16(__uint_as_float(x[8 * p8 + 0]), __uint_as_float(x[8 * p8 + 1])),
                                   pack_f16(__uint_as_float(x[8 * p8 + 2]), __uint_as_float(x[8 * p8 + 3])),
                                   pack_f16(__uint_as_float(x[8 * p8 + 4]), __uint_as_float(x[8 * p8 + 5])),
                                   pack_f16(__uint_as_float(x[8 * p8 + 6]), __uint_as_float(x[8 * p8 + 7])));
        sts128(wrow + (((4 * cb + p8) ^ (cr & 7)) << 4), o);
      }
    }
  }
  tc_fence_before();
  fence_proxy_async();
  named_bar_sync(3 + gi, 128);  // every TMEM read of ACC is done; also: the scratch is rewritten by the group's next chunk
  if (gtid == 0) f_acc_release(&bars->acc_lock);
  if (lane == 0) mbar_arrive(&bars->out_full[c & 1]);  // count 4: one arrival per warp of the group
}

// ---------------------------------------------------------------------------------------------------- kernel
__global__ void __launch_bounds__(kF_Threads, 1)  // 18 warps = 5 on two of the four sub-partitions (16 K registers each): 96 per thread
    scan3_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                 const float* __restrict__ g, const float* __restrict__ beta, const int32_t* __restrict__ cu_seqlens,
                 const int32_t* __restrict__ seg_order, int H, float* __restrict__ E, float* __restrict__ T,
                 int32_t* __restrict__ fb, int n_units) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  F_Bars* bars = reinterpret_cast<F_Bars*>(smem + kF_OffBar);
  volatile int* abort_flag = &bars->abort_flag;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int h = blockIdx.x, s = seg_order[blockIdx.y];  // longest segments first
  const int seg_begin = cu_seqlens[s], seg_end = cu_seqlens[s + 1];
  const int seg_len = seg_end - seg_begin;
  const int nc = (seg_len + kC - 1) / kC;

  if (warp == kF_WLoader) tmem_alloc(&bars->tmem_base, 512);
  if (tid == 0) {
    for (int i = 0; i < kF_KStages; ++i) {
      mbar_init(&bars->k_full[i], 1);
      mbar_init(&bars->k_free[i], 2);
      mbar_init(&bars->k_ready[i], 1);
    }
    for (int i = 0; i < kF_VStages; ++i) {
      mbar_init(&bars->v_full[i], 1);
      mbar_init(&bars->v_free[i], 1);
    }
    for (int i = 0; i < kF_Slots; ++i) {
      mbar_init(&bars->out_full[i], 4);
      mbar_init(&bars->out_free[i], 2);
    }
    for (int i = 0; i < kF_GateSlots; ++i) mbar_init(&bars->gate_full[i], 1);
    for (int i = 0; i < 2; ++i) {
      mbar_init(&bars->m3_done[i], 1);
      mbar_init(&bars->m4_done[i], 1);
    }
    mbar_init(&bars->dy_for_t, 128);
    mbar_init(&bars->dy_for_e, 128);
    mbar_init(&bars->v_ok[0], 1);
    mbar_init(&bars->v_ok[1], 1);
    mbar_init(&bars->acc_done[0], 1);
    mbar_init(&bars->acc_done[1], 1);
    bars->acc_lock = 0;
    bars->abort_flag = 0;
    bars->bad = 0;
    bars->p_final = 0.f;
    bars->g_total = 0.0;
    bars->fin_flag = 0;
    fence_barrier_init();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = bars->tmem_base;
  const uint32_t smem_base = smem_u32(smem);

  if (warp == kF_WLoader) {
    // ------------------------------------------------------------------------------------------- loader
    // Iteration c: the K tile of chunk c, then the V tile of chunk c - 2.  K runs two chunks ahead of V because the
    // producers need it two chunks before (1) needs V, and the 2-deep V ring would otherwise hold the K loads back (a V
    // slot is free only when (1) of the chunk two back has completed).  One lane, nothing but waits and TMA issues.
    if (lane == 0) {
#pragma unroll 1
      for (int c = 0; c < nc + 2; ++c) {
        if (c < nc) {
          const int kst = c % kF_KStages;
          const int t0 = seg_begin + c * kC;
          if (c >= kF_KStages) f_wait_lazy(&bars->k_free[kst], ((c / kF_KStages) - 1) & 1, abort_flag);
          mbar_expect_tx(&bars->k_full[kst], 2 * kTileB);
          tma_load_3d(smem_base + kF_OffK + kst * 2 * kTileB, &tmK, 0, h, t0, &bars->k_full[kst]);
          tma_load_3d(smem_base + kF_OffK + kst * 2 * kTileB + 8192, &tmK, 64, h, t0, &bars->k_full[kst]);
        }
        const int cv = c - 2;
        if (cv >= 0) {
          const int vst = cv & 1;
          const int t0 = seg_begin + cv * kC;
          if (cv >= kF_VStages) f_wait_lazy(&bars->v_free[vst], ((cv >> 1) - 1) & 1, abort_flag);
          mbar_expect_tx(&bars->v_full[vst], 2 * kTileB);
          tma_load_3d(smem_base + kF_OffV + vst * 2 * kTileB, &tmV, 0, h, t0, &bars->v_full[vst]);
          tma_load_3d(smem_base + kF_OffV + vst * 2 * kTileB + 8192, &tmV, 64, h, t0, &bars->v_full[vst]);
        }
      }
    }
  } else if (warp == kF_WGate) {
    // ------------------------------------------------------------------------------------------- gate
    // All 32 lanes, always converged (a warp whose lane 0 also span on mbarriers ran these shuffles on ptxas'
    // divergent-warp fallback path and needed ~7,000 cycles per chunk).  Lanes t, t + 32 own tokens t, t + 32 of the
    // chunk; the next chunk's g / beta are in flight while this one is scanned.  Paced by the chunk's K tile landing, so
    // it never runs more than kF_KStages chunks ahead of the chains and the 8-slot gate ring cannot be lapped.
    float* gate_ring = reinterpret_cast<float*>(smem + kF_OffGate);
    float p_lazy = 0.f;
    double g_tot = 0.0;
    float gn0 = 0.f, gn1 = 0.f, bn0 = 0.f, bn1 = 0.f;
    auto fetch = [&](int c) {
      const int t0 = seg_begin + c * kC, valid = min(kC, seg_len - c * kC);
      gn0 = gn1 = bn0 = bn1 = 0.f;  // tokens past the segment's end: g = 0, beta = 0 (exact no-ops)
      if (lane < valid) {
        gn0 = g[(size_t)(t0 + lane) * H + h];
        bn0 = beta[(size_t)(t0 + lane) * H + h];
      }
      if (lane + 32 < valid) {
        gn1 = g[(size_t)(t0 + lane + 32) * H + h];
        bn1 = beta[(size_t)(t0 + lane + 32) * H + h];
      }
    };
    if (nc > 0) fetch(0);
#pragma unroll 1
    for (int c = 0; c < nc; ++c) {
      float g0 = gn0, g1 = gn1;
      const float b0 = bn0, b1 = bn1;
      if (c + 1 < nc) fetch(c + 1);
      f_wait_lazy(&bars->k_full[c % kF_KStages], (c / kF_KStages) & 1, abort_flag);  // pacing only
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {  // inclusive scans of the two token halves
        const float u0 = __shfl_up_sync(0xffffffffu, g0, o), u1 = __shfl_up_sync(0xffffffffu, g1, o);
        if (lane >= o) g0 += u0, g1 += u1;
      }
      g1 += __shfl_sync(0xffffffffu, g0, 31);
      const float GC = __shfl_sync(0xffffffffu, g1, 31);
      const bool rs = !(fabsf(p_lazy + GC) <= kLazyP);  // also NaN
      float* gr = gate_ring + (c & (kF_GateSlots - 1)) * kF_GateFloats;
      gr[lane] = g0;
      gr[lane + 32] = g1;
      gr[kC + lane] = b0;
      gr[kC + lane + 32] = b1;
      if (lane == 0) {
        gr[2 * kC] = p_lazy;
        gr[2 * kC + 1] = rs ? expf(p_lazy + GC) : 1.f;
        gr[2 * kC + 2] = GC;
        gr[2 * kC + 3] = rs ? 1.f : 0.f;
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&bars->gate_full[c & (kF_GateSlots - 1)]);
      p_lazy = rs ? 0.f : p_lazy + GC;
      g_tot += (double)GC;
    }
    if (lane == 0) {
      bars->p_final = p_lazy;
      bars->g_total = g_tot;
      flag_release(&bars->fin_flag, 1);
    }
  } else if (warp == kF_WIssuer) {
    // ------------------------------------------------------------------------------------------- converter
    // Walks the tiles in the loader's order (K of chunk c, then V of chunk c - 2; every phase of k_full / v_full is waited
    // for: a parity wait must never skip one).  K: bf16 -> fp16 in place (element-wise on 16-bit lanes, so the 128B swizzle
    // of the TMA boxes is untouched), two chunks ahead of the producers' need.  V stays bf16.  The ragged last chunk's
    // boxes also hold tokens of the next segment: those rows are zeroed in both tiles, so that nothing of a neighbour --
    // not even an Inf or NaN -- reaches the unit through 0 x garbage.
#pragma unroll 1
    for (int c = 0; c < nc + 2; ++c) {
      if (c < nc) {
        const int kst = c % kF_KStages;
        const int valid = min(kC, seg_len - c * kC);
        const uint32_t kt = smem_base + kF_OffK + kst * 2 * kTileB;
        f_wait_lazy(&bars->k_full[kst], (c / kF_KStages) & 1, abort_flag);
#pragma unroll 1
        for (int i0 = 0; i0 < 32; i0 += 8) {  // 16-byte piece p of the tile: token (p % 512) / 8
          uint4 w[8];
#pragma unroll
          for (int j = 0; j < 8; ++j) w[j] = lds128(kt + 16 * (lane + 32 * (i0 + j)));
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const int p = lane + 32 * (i0 + j);
            uint4 o = cvt8_bf16_f16(w[j]);
            if (((p & 511) >> 3) >= valid) o = make_uint4(0u, 0u, 0u, 0u);
            sts128(kt + 16 * p, o);
          }
        }
        fence_proxy_async();  // the fp16 K tile must be visible to the tensor pipe's reads
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars->k_ready[kst]);
        __syncwarp();
      }
      const int cv = c - 2;
      if (cv >= 0) {
        const int slot = cv & 1;
        const int valid = min(kC, seg_len - cv * kC);
        const uint32_t vt = smem_base + kF_OffV + slot * 2 * kTileB;
        f_wait_lazy(&bars->v_full[slot], (cv >> 1) & 1, abort_flag);
        if (valid < kC) {
#pragma unroll 1
          for (int p = lane; p < 1024; p += 32)
            if (((p & 511) >> 3) >= valid) sts128(vt + 16 * p, make_uint4(0u, 0u, 0u, 0u));
          fence_proxy_async();
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars->v_ok[slot]);
        __syncwarp();
      }
    }
  } else if (warp >= kF_WProd) {
    // ------------------------------------------------------------------------------------------- producers
    const int gi = (warp - kF_WProd) >> 2, gtid = tid - 32 * kF_WProd - 128 * gi;
#pragma unroll 1
    for (int c = gi; c < nc; c += 2) {
      const int kst = c % kF_KStages;
      f_wait_lazy(&bars->gate_full[c & (kF_GateSlots - 1)], (c / kF_GateSlots) & 1, abort_flag);
      f_wait_lazy(&bars->k_ready[kst], (c / kF_KStages) & 1, abort_flag);
      f_produce(smem, bars, abort_flag, tmem, gi, gtid, warp & 3, c, min(kC, seg_len - c * kC),
                smem_base + kF_OffK + kst * 2 * kTileB, smem_base + kF_OffOut + (c & 1) * kF_OutBytes);
    }
  } else if (warp < kF_WChainT) {
    f_chain(false, smem, bars, abort_flag, tmem, warp, lane, nc, E + ((size_t)s * H + h) * kD * kD);
  } else {
    f_chain(true, smem, bars, abort_flag, tmem, warp, lane, nc, T + ((size_t)s * H + h) * kD * kD);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == kF_WLoader) tmem_dealloc(tmem, 512);
  if (tid == 0 && bars->bad) fb_append(fb, n_units, s * H + h);
}
