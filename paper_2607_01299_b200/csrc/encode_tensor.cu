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
//   K1 prep          : per (chunk, head), state-independent: Gram (mma.sync), L, A by forward substitution (fp32),
//                      -W (mma.sync, fp16 out) and A_b (fp16), stored as ready-made K-major 128B-swizzled
//                      UMMA B tiles, plus the gate record (d_j, gamma_C).
//   K2 scan          : one CTA per (segment, head), sequential over chunks, both row blocks of X resident in TMEM;
//                      every state contraction is a tcgen05.mma (see encode_scan2.cuh).
#include <cuda.h>
#include <cuda_fp16.h>
#include <stdlib.h>

#include "common.cuh"
#include "sm100_ptx.cuh"

namespace hypic {
namespace {
using namespace ptx;

constexpr int kC = 64;                  // chunk length (north_star)
constexpr int kD = 128;                 // dk = dv
constexpr int kTileB = kC * kC * 2;     // one 16-bit 64x64 tile: 8 KB
constexpr int kRecW = 0;                // record: -W (fp16, [token][dk], two 64-wide boxes) 16 KB
constexpr int kRecAb = 2 * kTileB;      //         A_b (fp16, [token][token]) 8 KB
constexpr int kRecBytes = 3 * kTileB;   // 24 KB per (chunk, head)
constexpr int kGateFloats = 72;         // d_j[64], gamma_C, pad (288 B = 18 x 16 B)
constexpr int kGateBytes = kGateFloats * 4;

__host__ __device__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
__host__ __device__ inline size_t ws_off_rec(int32_t n_seg) { return align_up(4 * ((size_t)n_seg + 1), 1024); }
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
constexpr int kKsPitch = kD + 8;  // 16-bit elements per row of the staged K chunk (conflict-free fragment loads)
constexpr int kLPitch = 68;       // floats per row of L / A

__device__ __forceinline__ void mma_f16_16816(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                              uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
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

// K is staged as fp16 (exact for bf16 values with |x| in [2^-14, 65504]; smaller magnitudes lose bits below
// 2^-24 absolute), so that the Gram and W contractions run as f16 mma.sync with an 11-bit A operand.
__global__ void __launch_bounds__(kPrepThreads)
    prep_kernel(const __nv_bfloat16* __restrict__ k, const float* __restrict__ g, const float* __restrict__ beta,
                const int32_t* __restrict__ cu_seqlens, const int32_t* __restrict__ chunk_off, int n_seg, int H,
                uint8_t* __restrict__ rec, float* __restrict__ gate) {
  __shared__ __align__(16) uint8_t s_k[kC * kKsPitch * 2];  // K chunk (fp16); later the staged W tile
  __shared__ __align__(16) float s_l[kC * kLPitch];         // L^t; later A_b
  __shared__ float s_g[kC], s_b[kC], s_gam[kC];
  __shared__ float s_wsum;
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

  __half* ks = reinterpret_cast<__half*>(s_k);
  for (int idx = tid; idx < kC * (kD / 8); idx += kPrepThreads) {
    const int r = idx / (kD / 8), c8 = idx % (kD / 8);
    uint4 val = make_uint4(0, 0, 0, 0);
    if (r < valid) {
      const uint4 raw = *reinterpret_cast<const uint4*>(k + ((size_t)(t0 + r) * H + h) * kD + c8 * 8);
      const uint32_t w[4] = {raw.x, raw.y, raw.z, raw.w};
      uint32_t o[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) o[i] = pack_f16(__uint_as_float(w[i] << 16), __uint_as_float(w[i] & 0xffff0000u));
      val = make_uint4(o[0], o[1], o[2], o[3]);
    }
    *reinterpret_cast<uint4*>(ks + r * kKsPitch + c8 * 8) = val;
  }
  {  // a1: inclusive cumulative log-decay by a two-warp shuffle scan
    const bool ok = tid < valid;
    float gv = ok ? g[(size_t)(t0 + tid) * H + h] : 0.f;
    s_b[tid] = ok ? beta[(size_t)(t0 + tid) * H + h] : 0.f;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const float up = __shfl_up_sync(0xffffffffu, gv, o);
      if (lane >= o) gv += up;
    }
    if (tid == 31) s_wsum = gv;
    __syncthreads();
    if (warp == 1) gv += s_wsum;
    s_g[tid] = gv;
    s_gam[tid] = expf(gv);
  }
  __syncthreads();

  // ---- a2: Gram K K^t with mma.sync (fp16 in, fp32 accumulate); warp w owns rows [32w, 32w+32)
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
        if (nt > 4 * warp + 3) continue;  // strictly above the diagonal for every row of this warp
        const int n0 = 8 * nt + gq;
        const uint32_t b0 = kw[n0 * pw + 8 * kk + tq], b1 = kw[n0 * pw + 8 * kk + 4 + tq];
        mma_f16_16816(acc[0][nt], a[0][0], a[0][1], a[0][2], a[0][3], b0, b1);
        mma_f16_16816(acc[1][nt], a[1][0], a[1][1], a[1][2], a[1][3], b0, b1);
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
          if (j < r) v = s_b[r] * __expf(s_g[r] - s_g[j]) * acc[mt][nt][i];
          s_l[j * kLPitch + r] = v;  // stored transposed: Lt[j][r]
        }
  }
  __syncthreads();

  // ---- a3: A = (I + L)^-1, column c per thread, right-looking (column-oriented) forward substitution in fp32:
  // a_j = t_j is final once columns < j have been applied; then t_r -= L_rj a_j for r > j (independent FMAs).
  // Column c of A is zero above row c, so a warp skips the steps below its first column.
  {
    float a[kC];
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
    __syncthreads();  // every column is done reading L
    // A_b = A diag(beta) as fp32 [r][c] in the (now dead) L buffer
    const float bc = s_b[tid];
#pragma unroll
    for (int r = 0; r < kC; ++r) s_l[r * kLPitch + tid] = a[r] * bc;
  }
  __syncthreads();
  const float* s_a = s_l;

  // ---- W = (A_b diag(gamma)) K with mma.sync: M = 64 tokens (warp w: rows [32w, 32w+32)), N = 128, K = 64 tokens
  float wacc[2][16][4];
  {
    const int gq = lane >> 2, tq = lane & 3;
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
      for (int nt = 0; nt < 16; ++nt)
#pragma unroll
        for (int i = 0; i < 4; ++i) wacc[mt][nt][i] = 0.f;
    const uint32_t ks_base = smem_u32(s_k);
#pragma unroll
    for (int kk = 0; kk < kC / 16; ++kk) {
      if (kk > 2 * warp + 1) continue;  // A_b is lower triangular: rows < 32(w+1) have no columns >= 32(w+1)
      uint32_t a[2][4];
      const int c0 = 16 * kk + 2 * tq;
      const float g0 = s_gam[c0], g1 = s_gam[c0 + 1], g8 = s_gam[c0 + 8], g9 = s_gam[c0 + 9];
#pragma unroll
      for (int mt = 0; mt < 2; ++mt) {
        const int r0 = 32 * warp + 16 * mt + gq;
        const float2 p0 = *reinterpret_cast<const float2*>(s_a + r0 * kLPitch + c0);
        const float2 p1 = *reinterpret_cast<const float2*>(s_a + (r0 + 8) * kLPitch + c0);
        const float2 p2 = *reinterpret_cast<const float2*>(s_a + r0 * kLPitch + c0 + 8);
        const float2 p3 = *reinterpret_cast<const float2*>(s_a + (r0 + 8) * kLPitch + c0 + 8);
        a[mt][0] = pack_f16(p0.x * g0, p0.y * g1);
        a[mt][1] = pack_f16(p1.x * g0, p1.y * g1);
        a[mt][2] = pack_f16(p2.x * g8, p2.y * g9);
        a[mt][3] = pack_f16(p3.x * g8, p3.y * g9);
      }
      // B fragments (k = token, n = dk) by transposing ldmatrix over the [token][dk] tile, two n-tiles at a time
      const int tok = 16 * kk + (lane & 7) + ((lane >> 3) & 1) * 8;
#pragma unroll
      for (int np = 0; np < 8; ++np) {
        uint32_t b[4];
        ldmatrix_x4_trans(b, ks_base + (uint32_t)(tok * kKsPitch + 8 * (2 * np + (lane >> 4))) * 2u);
        mma_f16_16816(wacc[0][2 * np], a[0][0], a[0][1], a[0][2], a[0][3], b[0], b[1]);
        mma_f16_16816(wacc[1][2 * np], a[1][0], a[1][1], a[1][2], a[1][3], b[0], b[1]);
        mma_f16_16816(wacc[0][2 * np + 1], a[0][0], a[0][1], a[0][2], a[0][3], b[2], b[3]);
        mma_f16_16816(wacc[1][2 * np + 1], a[1][0], a[1][1], a[1][2], a[1][3], b[2], b[3]);
      }
    }
  }
  __syncthreads();  // K is dead: stage W over it, already in the K-major 128B-swizzled two-box layout
  {
    const int gq = lane >> 2, tq = lane & 3;
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
      for (int nt = 0; nt < 16; ++nt)
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
          const int r = 32 * warp + 16 * mt + gq + 8 * hh;
          const int col = 8 * nt + 2 * tq;
          const uint32_t off = (col >> 6) * 8192 + (r >> 3) * 1024 + (r & 7) * 128 + ((((col & 63) >> 3) ^ (r & 7)) * 16) +
                               (col & 7) * 2;
          *reinterpret_cast<uint32_t*>(s_k + off) = pack_f16(-wacc[mt][nt][2 * hh], -wacc[mt][nt][2 * hh + 1]);  // -W
        }
  }
  __syncthreads();
  uint8_t* out = rec + ((size_t)x * H + h) * kRecBytes;
  for (int idx = tid; idx < 2 * kTileB / 16; idx += kPrepThreads)
    *reinterpret_cast<uint4*>(out + kRecW + idx * 16) = *reinterpret_cast<const uint4*>(s_k + idx * 16);

  // ---- A_b as an fp16 B tile (K-major, 128B swizzle: row r, 16-byte chunk j8 at ((j8 ^ (r & 7)) * 16))
  for (int idx = tid; idx < kC * 8; idx += kPrepThreads) {
    const int r = idx >> 3, j8 = idx & 7;
    const float4 v0 = *reinterpret_cast<const float4*>(s_a + r * kLPitch + 8 * j8);
    const float4 v1 = *reinterpret_cast<const float4*>(s_a + r * kLPitch + 8 * j8 + 4);
    const uint32_t off = (r >> 3) * 1024 + (r & 7) * 128 + ((j8 ^ (r & 7)) * 16);
    *reinterpret_cast<uint4*>(out + kRecAb + off) =
        make_uint4(pack_f16(v0.x, v0.y), pack_f16(v0.z, v0.w), pack_f16(v1.x, v1.y), pack_f16(v1.z, v1.w));
  }
  float* go = gate + ((size_t)x * H + h) * kGateFloats;
  go[tid] = expf(s_g[kC - 1] - s_g[tid]);
  if (tid < kGateFloats - kC) go[kC + tid] = (tid == 0) ? s_gam[kC - 1] : 0.f;
}

__device__ unsigned int g_timeout_count_enc = 0;

#include "encode_scan2.cuh"

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

// E = 0, T = I for every (segment, head) when the call carries no tokens at all (no tensor map can be built).
__global__ void identity_fill_kernel(float* __restrict__ E, float* __restrict__ T, size_t n_units) {
  const size_t n = n_units * kD * kD;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    E[i] = 0.f;
    const size_t e = i % (kD * kD);
    T[i] = (e / kD == e % kD) ? 1.f : 0.f;
  }
}

}  // namespace

bool encode_tensor_shape_ok(int32_t, int32_t dk, int32_t dv, int kv_dtype, int gate) {
  return dk == kD && dv == kD && kv_dtype == HYPIC_DT_BF16 && gate == HYPIC_GATE_SCALAR;
}

size_t encode_tensor_workspace(int32_t n_seg, int32_t t_total, int32_t H, int32_t dk, int32_t dv, int kv_dtype,
                               int gate) {
  if (!encode_tensor_shape_ok(H, dk, dv, kv_dtype, gate)) return 0;
  const size_t cap = chunk_cap(n_seg, t_total);
  return ws_off_rec(n_seg) + cap * H * ((size_t)kRecBytes + kGateBytes);
}

int encode_tensor(const EncodeArgs& a) {
  if (!encode_tensor_supported(a)) return HYPIC_ERR_UNSUPPORTED;
  if (a.n_seg == 0) return HYPIC_OK;
  if (a.H > 65535 || a.n_seg > 65535) return HYPIC_ERR_UNSUPPORTED;
  const size_t cap = chunk_cap(a.n_seg, a.t_total);
  if (cap > 0x7fffffffULL) return HYPIC_ERR_UNSUPPORTED;
  if (a.t_total == 0) {
    identity_fill_kernel<<<296, 256, 0, a.stream>>>(a.E, a.T, (size_t)a.n_seg * a.H);
    note_launch();
    HYPIC_CUDA_OK(cudaGetLastError());
    return HYPIC_OK;
  }
  uint8_t* ws = static_cast<uint8_t*>(a.workspace);
  int32_t* chunk_off = reinterpret_cast<int32_t*>(ws);
  uint8_t* rec = ws + ws_off_rec(a.n_seg);
  float* gate = reinterpret_cast<float*>(rec + cap * a.H * (size_t)kRecBytes);
  static bool configured = false;
  if (!configured) {
    HYPIC_CUDA_OK(cudaFuncSetAttribute(scan2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kS2Smem));
    configured = true;
  }
  const auto* kp = static_cast<const __nv_bfloat16*>(a.k);
  CUtensorMap tmK, tmV;
  int rc = make_kv_tensor_map(&tmK, a.k, a.t_total, a.H);
  if (rc == HYPIC_OK) rc = make_kv_tensor_map(&tmV, a.v, a.t_total, a.H);
  if (rc != HYPIC_OK) return rc;
  chunk_offsets_kernel<<<1, 1024, 0, a.stream>>>(a.cu_seqlens, a.n_seg, chunk_off);
  note_launch();
  prep_kernel<<<dim3((unsigned)cap, a.H), kPrepThreads, 0, a.stream>>>(kp, a.g, a.beta, a.cu_seqlens, chunk_off,
                                                                       a.n_seg, a.H, rec, gate);
  note_launch();
  scan2_kernel<<<dim3(a.H, a.n_seg), kS2Threads, kS2Smem, a.stream>>>(tmK, tmV, a.cu_seqlens, chunk_off, a.H, rec, gate,
                                                                     a.E, a.T);
  note_launch();
  HYPIC_CUDA_OK(cudaGetLastError());
  return HYPIC_OK;
}

#ifdef HYPIC_TIMELINE
extern "C" int hypic_debug_timeline(long long* out, int n) {
  return cudaMemcpyFromSymbol(out, g_s2_timeline, sizeof(long long) * (size_t)n) == cudaSuccess ? 0 : 1;
}
#endif

unsigned int debug_timeout_count_encode() {
  unsigned int v = 0;
  if (cudaMemcpyFromSymbol(&v, g_timeout_count_enc, sizeof(v)) != cudaSuccess) return 0xffffffffu;
  return v;
}

}  // namespace hypic
