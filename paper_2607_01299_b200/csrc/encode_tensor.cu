// encode_tensor.cu -- tcgen05/TMEM segment encode: bf16 k/v, scalar gate, dk = dv = 128 (HYPIC_IMPL_TENSOR).
//
// Rows a0..a5 of SURVEY.md section 8(a), chunked (C = 64 tokens) WY/UT form of the token recurrence
// (Eq. 2, Table 1 GDN row PAPER.md:61; T_C and S_{C|0} of PAPER.md:118-126).  Per chunk, with
// G_r the in-chunk inclusive cumulative log-decay, gamma_r = exp(G_r), d_j = exp(G_C - G_j):
//     L_rj = beta_r exp(G_r - G_j) (k_r.k_j)  (j < r),   A = (I + L)^-1,   A_b = A diag(beta),
//     W = A_b diag(gamma) K  (C x dk),   U^ = A_b V  (C x dv),
//     X <- gamma_C X + ([U^t ; 0] - X W^t) diag(d) K          for the stacked state X = [E ; T].
// Three launches:
//   K0 chunk_offsets : prefix sum of ceil(L_s / 64) (cu_seqlens lives on the device; no host sync).
//   K1 prep          : per (chunk, head), state-independent: Gram (mma.sync bf16), L, A by forward substitution
//                      (fp32), then A_b and A_b diag(gamma) split into bf16 hi + lo and stored as ready-made
//                      K-major 128B-swizzled UMMA B tiles, plus the gate record (d_j, gamma_C).
//   K2 scan          : one CTA per (segment, head, row block of X), sequential over chunks; every contraction is
//                      a tcgen05.mma with the state block resident in TMEM (see the kernel's comment).
#include <cuda.h>
#include <stdlib.h>

#include "common.cuh"
#include "sm100_ptx.cuh"

namespace hypic {
namespace {
using namespace ptx;

constexpr int kC = 64;                  // chunk length (north_star)
constexpr int kD = 128;                 // dk = dv
constexpr int kTileB = kC * kC * 2;     // one bf16 64x64 B tile: 8 KB
constexpr int kAbBytes = 4 * kTileB;    // A_b hi, A_b lo, A_bg hi, A_bg lo
constexpr int kGateFloats = 72;         // d_j[64], gamma_C, pad (288 B = 18 x 16 B)
constexpr int kGateBytes = kGateFloats * 4;

__host__ __device__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct Workspace {
  int32_t* chunk_off;  // [n_seg + 1]
  uint8_t* ab;         // [n_chunk_cap][H][kAbBytes]
  float* gate;         // [n_chunk_cap][H][kGateFloats]
};
__host__ __device__ inline size_t ws_off_ab(int32_t n_seg) { return align_up(4 * ((size_t)n_seg + 1), 1024); }
__host__ __device__ inline size_t chunk_cap(int32_t n_seg, int32_t t_total) { return (size_t)t_total / kC + n_seg; }

// ------------------------------------------------------------------------------------------------ K0
__global__ void chunk_offsets_kernel(const int32_t* __restrict__ cu_seqlens, int n_seg, int32_t* __restrict__ chunk_off) {
  __shared__ int part[1024];
  const int tid = threadIdx.x;
  const int per = (n_seg + 1023) / 1024;
  const int lo = min(n_seg, tid * per), hi = min(n_seg, lo + per);
  int sum = 0;
  for (int s = lo; s < hi; ++s) sum += (cu_seqlens[s + 1] - cu_seqlens[s] + kC - 1) / kC;
  part[tid] = sum;
  __syncthreads();
  if (tid == 0) {
    int run = 0;
    for (int i = 0; i < 1024; ++i) {
      const int v = part[i];
      part[i] = run;
      run += v;
    }
    chunk_off[n_seg] = run;
  }
  __syncthreads();
  int run = part[tid];
  for (int s = lo; s < hi; ++s) {
    chunk_off[s] = run;
    run += (cu_seqlens[s + 1] - cu_seqlens[s] + kC - 1) / kC;
  }
}

// ------------------------------------------------------------------------------------------------ K1
constexpr int kPrepThreads = 64;
constexpr int kKsPitch = kD + 8;  // bf16 elements per row of the staged K chunk (conflict-free fragment loads)
constexpr int kLPitch = 68;       // floats per row of L / A

__device__ __forceinline__ void mma_bf16_16816(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                               uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 p = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&p);
}

__global__ void __launch_bounds__(kPrepThreads)
    prep_kernel(const __nv_bfloat16* __restrict__ k, const float* __restrict__ g, const float* __restrict__ beta,
                const int32_t* __restrict__ cu_seqlens, const int32_t* __restrict__ chunk_off, int n_seg, int H,
                uint8_t* __restrict__ ab, float* __restrict__ gate) {
  __shared__ __align__(16) uint8_t s_k[kC * kKsPitch * 2];  // K chunk (bf16), later reused for A (fp32)
  __shared__ __align__(16) float s_l[kC * kLPitch];
  __shared__ float s_g[kC], s_b[kC];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int x = blockIdx.x, h = blockIdx.y;
  if (x >= chunk_off[n_seg]) return;
  // segment of this chunk: last s with chunk_off[s] <= x
  int lo = 0, hi = n_seg - 1;
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (chunk_off[mid] <= x) lo = mid; else hi = mid - 1;
  }
  const int s = lo;
  const int t0 = cu_seqlens[s] + (x - chunk_off[s]) * kC;
  const int valid = min(kC, cu_seqlens[s + 1] - t0);

  __nv_bfloat16* ks = reinterpret_cast<__nv_bfloat16*>(s_k);
  for (int idx = tid; idx < kC * (kD / 8); idx += kPrepThreads) {
    const int r = idx / (kD / 8), c8 = idx % (kD / 8);
    uint4 val = make_uint4(0, 0, 0, 0);
    if (r < valid) val = *reinterpret_cast<const uint4*>(k + ((size_t)(t0 + r) * H + h) * kD + c8 * 8);
    *reinterpret_cast<uint4*>(ks + r * kKsPitch + c8 * 8) = val;
  }
  {
    const bool ok = tid < valid;
    s_g[tid] = ok ? g[(size_t)(t0 + tid) * H + h] : 0.f;
    s_b[tid] = ok ? beta[(size_t)(t0 + tid) * H + h] : 0.f;
  }
  __syncthreads();
  if (tid == 0) {  // inclusive cumulative log-decay (a1)
    float run = 0.f;
    for (int r = 0; r < kC; ++r) {
      run += s_g[r];
      s_g[r] = run;
    }
  }
  __syncthreads();

  // ---- a2: Gram K K^t with mma.sync (bf16 in, fp32 accumulate); warp w owns rows [32w, 32w+32)
  {
    const int gq = lane >> 2, tq = lane & 3;
    float acc[2][8][4];
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
      for (int nt = 0; nt < 8; ++nt)
#pragma unroll
        for (int i = 0; i < 4; ++i) acc[mt][nt][i] = 0.f;
    const uint32_t* kw = reinterpret_cast<const uint32_t*>(s_k);
    constexpr int pw = kKsPitch / 2;  // 32-bit words per row
#pragma unroll
    for (int kk = 0; kk < kD / 16; ++kk) {
      uint32_t a[2][4];
#pragma unroll
      for (int mt = 0; mt < 2; ++mt) {
        const int r0 = 32 * warp + 16 * mt + gq;
        a[mt][0] = kw[r0 * pw + 8 * kk + tq];
        a[mt][1] = kw[(r0 + 8) * pw + 8 * kk + tq];
        a[mt][2] = kw[r0 * pw + 8 * kk + 4 + tq];
        a[mt][3] = kw[(r0 + 8) * pw + 8 * kk + 4 + tq];
      }
#pragma unroll
      for (int nt = 0; nt < 8; ++nt) {
        const int n0 = 8 * nt + gq;
        const uint32_t b0 = kw[n0 * pw + 8 * kk + tq], b1 = kw[n0 * pw + 8 * kk + 4 + tq];
        mma_bf16_16816(acc[0][nt], a[0][0], a[0][1], a[0][2], a[0][3], b0, b1);
        mma_bf16_16816(acc[1][nt], a[1][0], a[1][1], a[1][2], a[1][3], b0, b1);
      }
    }
    // L_rj = beta_r exp(G_r - G_j) (k_r.k_j) for j < r, else 0
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
      for (int nt = 0; nt < 8; ++nt)
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const int r = 32 * warp + 16 * mt + gq + ((i >> 1) ? 8 : 0);
          const int j = 8 * nt + 2 * tq + (i & 1);
          float v = 0.f;
          if (j < r) v = s_b[r] * expf(s_g[r] - s_g[j]) * acc[mt][nt][i];
          s_l[j * kLPitch + r] = v;  // stored transposed: Lt[j][r]
        }
  }
  __syncthreads();

  // ---- a3: A = (I + L)^-1, column c per thread, right-looking (column-oriented) forward substitution in fp32:
  // a_j = t_j is final once columns < j have been applied; then t_r -= L_rj a_j for r > j (independent FMAs).
  // Column c of A is zero above row c, so a warp skips the steps below its first column.
  float a[kC];
  {
    const int c = tid;
#pragma unroll
    for (int r = 0; r < kC; ++r) a[r] = (r == c) ? 1.f : 0.f;
#pragma unroll
    for (int j = 0; j < kC - 1; ++j) {
      if (j >= 32 * warp) {
        const float aj = a[j];
        const float4* lcol = reinterpret_cast<const float4*>(s_l + j * kLPitch);
#pragma unroll
        for (int r4 = (j + 1) / 4; r4 < kC / 4; ++r4) {
          const float4 l = lcol[r4];
          if (4 * r4 + 0 > j) a[4 * r4 + 0] = fmaf(-l.x, aj, a[4 * r4 + 0]);
          if (4 * r4 + 1 > j) a[4 * r4 + 1] = fmaf(-l.y, aj, a[4 * r4 + 1]);
          if (4 * r4 + 2 > j) a[4 * r4 + 2] = fmaf(-l.z, aj, a[4 * r4 + 2]);
          if (4 * r4 + 3 > j) a[4 * r4 + 3] = fmaf(-l.w, aj, a[4 * r4 + 3]);
        }
      }
    }
  }
  // A_b = A diag(beta) staged as fp32 [r][c] in the (now dead) K buffer
  float* s_a = reinterpret_cast<float*>(s_k);
  {
    const float bc = s_b[tid];
#pragma unroll
    for (int r = 0; r < kC; ++r) s_a[r * kLPitch + tid] = a[r] * bc;
  }
  __syncthreads();

  // ---- emit the four bf16 B tiles (K-major, 128B swizzle: row r, 16-byte chunk j8 at ((j8 ^ (r & 7)) * 16))
  uint8_t* out = ab + ((size_t)x * H + h) * kAbBytes;
  for (int idx = tid; idx < kC * 8; idx += kPrepThreads) {
    const int r = idx >> 3, j8 = idx & 7;
    float v[8], vg[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      v[i] = s_a[r * kLPitch + 8 * j8 + i];
      vg[i] = v[i] * expf(s_g[8 * j8 + i]);
    }
    uint32_t hi[4], lo[4], ghi[4], glo[4];
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      const float h0 = __bfloat162float(__float2bfloat16_rn(v[2 * p])), h1 = __bfloat162float(__float2bfloat16_rn(v[2 * p + 1]));
      hi[p] = pack_bf16(h0, h1);
      lo[p] = pack_bf16(v[2 * p] - h0, v[2 * p + 1] - h1);
      const float q0 = __bfloat162float(__float2bfloat16_rn(vg[2 * p])), q1 = __bfloat162float(__float2bfloat16_rn(vg[2 * p + 1]));
      ghi[p] = pack_bf16(q0, q1);
      glo[p] = pack_bf16(vg[2 * p] - q0, vg[2 * p + 1] - q1);
    }
    const uint32_t off = (r >> 3) * 1024 + (r & 7) * 128 + ((j8 ^ (r & 7)) * 16);
    *reinterpret_cast<uint4*>(out + 0 * kTileB + off) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
    *reinterpret_cast<uint4*>(out + 1 * kTileB + off) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
    *reinterpret_cast<uint4*>(out + 2 * kTileB + off) = make_uint4(ghi[0], ghi[1], ghi[2], ghi[3]);
    *reinterpret_cast<uint4*>(out + 3 * kTileB + off) = make_uint4(glo[0], glo[1], glo[2], glo[3]);
  }
  float* go = gate + ((size_t)x * H + h) * kGateFloats;
  go[tid] = expf(s_g[kC - 1] - s_g[tid]);
  if (tid < kGateFloats - kC) go[kC + tid] = (tid == 0) ? expf(s_g[kC - 1]) : 0.f;
}

// ------------------------------------------------------------------------------------------------ K2
// One CTA per (row block b of X, head, segment): b = 0 is E (dv = 128 rows), b = 1 is T (dk = 128 rows); rows of
// X evolve independently given the chunk operators, so the two blocks share nothing but their inputs.
// TMEM columns: X [0,128) fp32 state block (pre-scaled by gamma_C before the chunk's update), Xr [128,256) =
// rna_tf32(X) (the hardware truncates tf32 operands), DY [256,320), Wt [320,384).  Per chunk:
//   (2) Wt  = K^t  A_bg^t        bf16, A = K tile (MN-major), B = A_bg hi/lo tiles           -> TMEM
//   (1) DY  = V^t  A_b^t         bf16 (E block only)                                          -> TMEM
//       Wt -> registers -> -rna_tf32 -> smem as the MN-major (32B-base swizzle) B tile of (3)
//   (3) DY += Xr (-W)^t          tf32, A = Xr from TMEM
//       DY -> registers -> * d_j -> bf16 hi/lo -> smem K-major A tiles of (4)
//   (4) X  += U'' K              bf16, B = K tile (MN-major)
constexpr int kScanThreads = 128;
constexpr int kStK = 0, kStV = 16384, kStAb = 32768, kStGate = 65536;
constexpr int kStageBytes = 65536 + 1024;
constexpr int kOffW = 2 * kStageBytes;
constexpr int kOffUhi = kOffW + 32768;
constexpr int kOffUlo = kOffUhi + 16384;
constexpr int kOffBar = kOffUlo + 16384;
constexpr int kScanSmem = kOffBar + 64 + 1024;

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, bool valid) {
  const int sz = valid ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

__device__ __forceinline__ float rna_tf32f(float x) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return __uint_as_float(r);
}

__device__ unsigned int g_timeout_count_enc = 0;

__global__ void __launch_bounds__(kScanThreads, 1)
    scan_kernel(const __nv_bfloat16* __restrict__ k, const __nv_bfloat16* __restrict__ v,
                const int32_t* __restrict__ cu_seqlens, const int32_t* __restrict__ chunk_off, int H,
                const uint8_t* __restrict__ ab, const float* __restrict__ gate, float* __restrict__ E,
                float* __restrict__ T) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint64_t* mbar = reinterpret_cast<uint64_t*>(smem + kOffBar);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + kOffBar + 16);
  const int tid = threadIdx.x, warp = tid >> 5;
  const int blk = blockIdx.x, h = blockIdx.y, s = blockIdx.z;
  const bool is_e = (blk == 0);
  const int seg_begin = cu_seqlens[s], seg_end = cu_seqlens[s + 1];
  const int nc = (seg_end - seg_begin + kC - 1) / kC;
  const int chunk0 = chunk_off[s];

  if (warp == 0) tmem_alloc(tmem_slot, 512);
  if (tid == 32) {
    mbar_init(mbar, 1);
    fence_barrier_init();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;
  const uint32_t lane_base = (uint32_t)(32 * warp) << 16;
  const uint32_t tX = tmem + lane_base, tXr = tmem + 128 + lane_base, tDY = tmem + 256 + lane_base,
                 tWt = tmem + 320 + lane_base;
  const uint32_t smem_base = smem_u32(smem);
  const int row = tid;  // row of the state block (and dk index in the Wt conversion)

  auto load_stage = [&](int c, int st) {
    const int t0 = seg_begin + c * kC;
    const int valid = min(kC, seg_end - t0);
    const uint32_t sb = smem_base + st * kStageBytes;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const int idx = tid + kScanThreads * i;
      const int r = idx >> 4, c16 = idx & 15;
      const uint32_t off = (c16 >> 3) * 8192 + (r >> 3) * 1024 + (r & 7) * 128 + (((c16 & 7) ^ (r & 7)) * 16);
      const bool ok = r < valid;
      const size_t goff = ((size_t)(t0 + (ok ? r : 0)) * H + h) * kD + c16 * 8;
      cp_async16(sb + kStK + off, k + goff, ok);
      if (is_e) cp_async16(sb + kStV + off, v + goff, ok);
    }
    const uint8_t* abg = ab + ((size_t)(chunk0 + c) * H + h) * kAbBytes;
#pragma unroll
    for (int i = 0; i < kAbBytes / 16 / kScanThreads; ++i) {
      const int idx = tid + kScanThreads * i;
      cp_async16(sb + kStAb + idx * 16, abg + (size_t)idx * 16, true);
    }
    if (tid < kGateBytes / 16)
      cp_async16(sb + kStGate + tid * 16, gate + ((size_t)(chunk0 + c) * H + h) * kGateFloats + tid * 4, true);
    cp_async_commit();
  };

  uint32_t ph = 0;
  bool dead = false;
  auto wait_mma = [&]() {
    if (!dead && !mbar_wait(mbar, ph & 1, 4000000u)) {
      dead = true;
      if (tid == 0) atomicAdd(&g_timeout_count_enc, 1u);
    }
    ++ph;
    tc_fence_after();
  };

  if (nc > 0) load_stage(0, 0);
  for (int c = 0; c < nc; ++c) {
    const int st = c & 1;
    if (c + 1 < nc) {
      load_stage(c + 1, st ^ 1);
      cp_async_wait<1>();
    } else {
      cp_async_wait<0>();
    }
    fence_proxy_async();
    __syncthreads();
    const uint8_t* stg = smem + st * kStageBytes;
    const float* gt = reinterpret_cast<const float*>(stg + kStGate);
    const uint32_t sb = smem_base + st * kStageBytes;

    // ---- pass: Xr = rna_tf32(X); X <- gamma_C X  (c = 0: X is its initial value, 0 or I)
    {
      const float gC = gt[kC];
#pragma unroll 1
      for (int cb = 0; cb < 4; ++cb) {
        uint32_t x[32];
        if (c > 0) {
          tmem_ld32(tX + 32 * cb, x);
          tmem_ld_wait();
        } else {
#pragma unroll
          for (int i = 0; i < 32; ++i) x[i] = (!is_e && 32 * cb + i == row) ? __float_as_uint(1.f) : 0u;
        }
        uint32_t xr[32], xs[32];
#pragma unroll
        for (int i = 0; i < 32; ++i) {
          const float f = __uint_as_float(x[i]);
          xr[i] = __float_as_uint(rna_tf32f(f));
          xs[i] = __float_as_uint(f * gC);
        }
        tmem_st32(tXr + 32 * cb, xr);
        tmem_st32(tX + 32 * cb, xs);
      }
      tmem_st_wait();
    }
    tc_fence_before();
    __syncthreads();

    // ---- (2) Wt = K^t A_bg^t, (1) DY = V^t A_b^t
    if (tid == 0) {
      tc_fence_after();
      constexpr uint32_t id12 = make_idesc(1u, 128, 64, 1, 0);
#pragma unroll
      for (int hl = 0; hl < 2; ++hl)
#pragma unroll
        for (int ks = 0; ks < 4; ++ks) {
          const uint64_t ad = make_desc(sb + kStK + ks * 2048, 8192, 1024, 2);
          const uint64_t bd = make_desc(sb + kStAb + (2 + hl) * kTileB + ks * 32, 16, 1024, 2);
          mma_f16_ss(tmem + 320, ad, bd, id12, (hl | ks) > 0);
        }
      if (is_e) {
#pragma unroll
        for (int hl = 0; hl < 2; ++hl)
#pragma unroll
          for (int ks = 0; ks < 4; ++ks) {
            const uint64_t ad = make_desc(sb + kStV + ks * 2048, 8192, 1024, 2);
            const uint64_t bd = make_desc(sb + kStAb + hl * kTileB + ks * 32, 16, 1024, 2);
            mma_f16_ss(tmem + 256, ad, bd, id12, (hl | ks) > 0);
          }
      }
      mma_commit(mbar);
    }
    __syncthreads();
    wait_mma();

    // ---- Wt -> -rna_tf32 -> smem B tile of (3): [k = dk row][n = token], 32-bit MN-major, 32B-base swizzle
    {
      uint8_t* wt = smem + kOffW;
#pragma unroll 1
      for (int nch = 0; nch < 2; ++nch) {
        uint32_t w[32];
        tmem_ld32(tWt + 32 * nch, w);
        tmem_ld_wait();
        uint8_t* base = wt + nch * 16384 + (row >> 2) * 512 + (row & 3) * 128;
#pragma unroll
        for (int q8 = 0; q8 < 4; ++q8) {
          float4 lo4, hi4;
          lo4.x = -rna_tf32f(__uint_as_float(w[8 * q8 + 0])), lo4.y = -rna_tf32f(__uint_as_float(w[8 * q8 + 1]));
          lo4.z = -rna_tf32f(__uint_as_float(w[8 * q8 + 2])), lo4.w = -rna_tf32f(__uint_as_float(w[8 * q8 + 3]));
          hi4.x = -rna_tf32f(__uint_as_float(w[8 * q8 + 4])), hi4.y = -rna_tf32f(__uint_as_float(w[8 * q8 + 5]));
          hi4.z = -rna_tf32f(__uint_as_float(w[8 * q8 + 6])), hi4.w = -rna_tf32f(__uint_as_float(w[8 * q8 + 7]));
          uint8_t* p = base + ((q8 ^ (row & 3)) * 32);
          *reinterpret_cast<float4*>(p) = lo4;
          *reinterpret_cast<float4*>(p + 16) = hi4;
        }
      }
    }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();

    // ---- (3) DY (+)= Xr (-W)^t
    if (tid == 0) {
      tc_fence_after();
      constexpr uint32_t id3 = make_idesc(2u, 128, 64, 0, 1);
#pragma unroll
      for (int ks = 0; ks < 16; ++ks) {
        const uint64_t bd = make_desc(smem_base + kOffW + ks * 1024, 16384, 512, 1);
        mma_tf32_ts(tmem + 256, tmem + 128 + ks * 8, bd, id3, (is_e || ks > 0) ? 1u : 0u);
      }
      mma_commit(mbar);
    }
    __syncthreads();
    wait_mma();

    // ---- DY * d_j -> bf16 hi/lo -> K-major A tiles of (4)
    {
      uint8_t* uhi = smem + kOffUhi + (row >> 3) * 1024 + (row & 7) * 128;
      uint8_t* ulo = smem + kOffUlo + (row >> 3) * 1024 + (row & 7) * 128;
#pragma unroll 1
      for (int half = 0; half < 2; ++half) {
        uint32_t y[32];
        tmem_ld32(tDY + 32 * half, y);
        tmem_ld_wait();
#pragma unroll
        for (int j8 = 0; j8 < 4; ++j8) {
          uint32_t hi[4], lo[4];
#pragma unroll
          for (int p = 0; p < 4; ++p) {
            const int j = 32 * half + 8 * j8 + 2 * p;
            const float u0 = __uint_as_float(y[8 * j8 + 2 * p]) * gt[j];
            const float u1 = __uint_as_float(y[8 * j8 + 2 * p + 1]) * gt[j + 1];
            const float h0 = __bfloat162float(__float2bfloat16_rn(u0)), h1 = __bfloat162float(__float2bfloat16_rn(u1));
            hi[p] = pack_bf16(h0, h1);
            lo[p] = pack_bf16(u0 - h0, u1 - h1);
          }
          const int chunk = 4 * half + j8;
          const uint32_t sw = ((chunk ^ (row & 7)) * 16);
          *reinterpret_cast<uint4*>(uhi + sw) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
          *reinterpret_cast<uint4*>(ulo + sw) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
        }
      }
    }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();

    // ---- (4) X += U'' K
    if (tid == 0) {
      tc_fence_after();
      constexpr uint32_t id4 = make_idesc(1u, 128, 128, 0, 1);
#pragma unroll
      for (int hl = 0; hl < 2; ++hl)
#pragma unroll
        for (int ks = 0; ks < 4; ++ks) {
          const uint64_t ad = make_desc(smem_base + (hl ? kOffUlo : kOffUhi) + ks * 32, 16, 1024, 2);
          const uint64_t bd = make_desc(sb + kStK + ks * 2048, 8192, 1024, 2);
          mma_f16_ss(tmem, ad, bd, id4, 1u);
        }
      mma_commit(mbar);
    }
    __syncthreads();
    wait_mma();
  }

  // ---- a5: write the block out (thread = row)
  {
    float* dst = (is_e ? E : T) + (((size_t)s * H + h) * kD + row) * kD;
#pragma unroll 1
    for (int cb = 0; cb < 4; ++cb) {
      uint32_t x[32];
      if (nc > 0) {
        tmem_ld32(tX + 32 * cb, x);
        tmem_ld_wait();
      } else {
#pragma unroll
        for (int i = 0; i < 32; ++i) x[i] = (!is_e && 32 * cb + i == row) ? __float_as_uint(1.f) : 0u;
      }
      float4* d4 = reinterpret_cast<float4*>(dst + 32 * cb);
#pragma unroll
      for (int u = 0; u < 8; ++u)
        d4[u] = make_float4(__uint_as_float(x[4 * u]), __uint_as_float(x[4 * u + 1]), __uint_as_float(x[4 * u + 2]),
                            __uint_as_float(x[4 * u + 3]));
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, 512);
}

#include "encode_scan_ws.cuh"

// k / v viewed as 3-D bf16 tensors [t_total][H][128]; box = 64 elements (128 B) x 1 head x 64 tokens, 128B swizzle:
// the box lands as one MN-major UMMA chunk (8-token atoms of 1 KB), two boxes per 64 x 128 tile.
typedef CUresult (*EncodeTiledFn3)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                   const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int make_kv_tensor_map(CUtensorMap* tm, const void* base, int32_t t_total, int32_t H) {
  static EncodeTiledFn3 fn = nullptr;
  if (fn == nullptr) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess || p == nullptr)
      return HYPIC_ERR_CUDA;
    fn = reinterpret_cast<EncodeTiledFn3>(p);
  }
  const cuuint64_t dims[3] = {(cuuint64_t)kD, (cuuint64_t)H, (cuuint64_t)t_total};
  const cuuint64_t strides[2] = {(cuuint64_t)kD * 2, (cuuint64_t)H * kD * 2};
  const cuuint32_t box[3] = {64, 1, 64};
  const cuuint32_t estr[3] = {1, 1, 1};
  const CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? HYPIC_OK : HYPIC_ERR_CUDA;
}

}  // namespace

bool encode_tensor_shape_ok(int32_t, int32_t dk, int32_t dv, int kv_dtype, int gate) {
  return dk == kD && dv == kD && kv_dtype == HYPIC_DT_BF16 && gate == HYPIC_GATE_SCALAR;
}

size_t encode_tensor_workspace(int32_t n_seg, int32_t t_total, int32_t H, int32_t dk, int32_t dv, int kv_dtype,
                               int gate) {
  if (!encode_tensor_shape_ok(H, dk, dv, kv_dtype, gate)) return 0;
  const size_t cap = chunk_cap(n_seg, t_total);
  return ws_off_ab(n_seg) + cap * H * ((size_t)kAbBytes + kGateBytes);
}

int encode_tensor(const EncodeArgs& a) {
  if (!encode_tensor_supported(a)) return HYPIC_ERR_UNSUPPORTED;
  if (a.n_seg == 0) return HYPIC_OK;
  if (a.H > 65535 || a.n_seg > 65535) return HYPIC_ERR_UNSUPPORTED;
  const size_t cap = chunk_cap(a.n_seg, a.t_total);
  if (cap > 0x7fffffffULL) return HYPIC_ERR_UNSUPPORTED;
  uint8_t* ws = static_cast<uint8_t*>(a.workspace);
  int32_t* chunk_off = reinterpret_cast<int32_t*>(ws);
  uint8_t* ab = ws + ws_off_ab(a.n_seg);
  float* gate = reinterpret_cast<float*>(ab + cap * a.H * (size_t)kAbBytes);
  static bool configured = false;
  if (!configured) {
    HYPIC_CUDA_OK(cudaFuncSetAttribute(scan_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kScanSmem));
    configured = true;
  }
  const auto* kp = static_cast<const __nv_bfloat16*>(a.k);
  const auto* vp = static_cast<const __nv_bfloat16*>(a.v);
  chunk_offsets_kernel<<<1, 1024, 0, a.stream>>>(a.cu_seqlens, a.n_seg, chunk_off);
  note_launch();
  if (cap > 0) {
    prep_kernel<<<dim3((unsigned)cap, a.H), kPrepThreads, 0, a.stream>>>(kp, a.g, a.beta, a.cu_seqlens, chunk_off,
                                                                         a.n_seg, a.H, ab, gate);
    note_launch();
  }
  static const bool use_v1 = [] {
    const char* e = getenv("HYPIC_SCAN_V1");  // diagnostics: the lock-step 128-thread scan kernel
    return e != nullptr && e[0] == '1';
  }();
  if (use_v1 || a.t_total == 0) {
    scan_kernel<<<dim3(2, a.H, a.n_seg), kScanThreads, kScanSmem, a.stream>>>(kp, vp, a.cu_seqlens, chunk_off, a.H, ab,
                                                                              gate, a.E, a.T);
  } else {
    static bool configured_ws = false;
    if (!configured_ws) {
      HYPIC_CUDA_OK(cudaFuncSetAttribute(scan_ws_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kWsSmem));
      configured_ws = true;
    }
    CUtensorMap tmK, tmV;
    int rc = make_kv_tensor_map(&tmK, a.k, a.t_total, a.H);
    if (rc == HYPIC_OK) rc = make_kv_tensor_map(&tmV, a.v, a.t_total, a.H);
    if (rc != HYPIC_OK) return rc;
    scan_ws_kernel<<<dim3(2, a.H, a.n_seg), kWsThreads, kWsSmem, a.stream>>>(tmK, tmV, a.cu_seqlens, chunk_off, a.H, ab,
                                                                            gate, a.E, a.T);
  }
  note_launch();
  HYPIC_CUDA_OK(cudaGetLastError());
  return HYPIC_OK;
}

unsigned int debug_timeout_count_encode() {
  unsigned int v = 0;
  if (cudaMemcpyFromSymbol(&v, g_timeout_count_enc, sizeof(v)) != cudaSuccess) return 0xffffffffu;
  return v;
}

}  // namespace hypic
