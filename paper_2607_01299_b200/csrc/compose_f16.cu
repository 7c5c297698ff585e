// compose_f16.cu -- composition over fp16-stored tuples (the paper keeps (T_C, S_{C|0}) in
// fp16, 32 KB per T at dk = dv = 128: PAPER.md:196-198), dk = dv = 128, plus the pack kernel that produces such pools.
//
//   S <- S T_i + E_i   (Eq. 6 as the chain of Eq. 4 steps), S in fp32, T_i and E_i stored in fp16.
// One CTA per (request, head) chain; 64 KB of (T_i, E_i) per step instead of 128 KB, so twice the steps per HBM byte.
//   * T_i needs no conversion at all: TMA tensor boxes (64 columns x 32 rows, 128B swizzle) land each 32-row slab
//     directly in the 16-bit MN-major B-operand layout of tcgen05.mma kind::f16; a stored fp16 value is an exact operand.
//   * S lives in TMEM as a two-term fp16 split of the row-normalised state (row maximum in [2^13, 2^14)):
//     D = S_hi T + S_lo T, 22 significant bits of S against exact T, fp32 accumulation in TMEM.
//   * round-trip warps read D (tcgen05.ld), undo the row scale in fp32, add E_i (fp16 tile staged by TMA boxes of
//     32 rows x 128 B, conflict-free row-per-thread reads) and write the next S_hi / S_lo, or S_out after the last step.
// S_in is read straight from global memory (fp32).  All waits are bounded (hypic_debug_timeout_count).
#include <cuda.h>
#include <cuda_fp16.h>
#include <string.h>

#include "common.cuh"
#include "sm100_ptx.cuh"

namespace hypic {

__device__ unsigned int g_timeout_count_f16 = 0;

namespace {
using namespace ptx;

constexpr int kD = 128;
constexpr int kTSlab = 32 * kD * 2;   // 32 rows of T in fp16: 8 KB = two boxes of 4 KB
constexpr int kTMat = 4 * kTSlab;     // one T matrix: 32 KB
constexpr int kNT = 3;                // T matrices in flight (one mbarrier probe per step: a probe costs ~380 cycles)
constexpr int kEQuarter = 32 * kD * 2;  // 32 rows of E in fp16: 8 KB = two boxes
constexpr int kNE = 8;                // E quarter slots: two buffers x 4 TMEM lane quarters
constexpr int kThreads = 608;         // warp 0 T producer, 1 MMA issuer, 2 E producer, 3-18 round trip

constexpr int kOffT = 0;
constexpr int kOffE = kOffT + kNT * kTMat;
constexpr int kOffXch = kOffE + kNE * kEQuarter;
constexpr int kOffBar = kOffXch + 4096;  // row maxima: one 2 KB exchange buffer per interleaved head
constexpr int kSmemBytes = kOffBar + 512 + 1024;

struct Bars {
  uint64_t t_full[kNT], t_empty[kNT], e_full[kNE], e_empty[kNE], d_full[2], a_ready[2];  // [head of the pair]
  uint32_t tmem_base;
  int abort_flag;
  int req_pick;  // LPT order: the request this CTA folds
};

__device__ __forceinline__ bool wait_or_abort(uint64_t* bar, uint32_t parity, volatile int* abort_flag) {
  for (uint32_t i = 0; i < 4000000u; ++i) {
    if (mbar_try_wait(bar, parity)) return true;
    if ((i & 1023u) == 1023u && *abort_flag) return false;
  }
  if (!*abort_flag) {
    *abort_flag = 1;
    atomicAdd(&g_timeout_count_f16, 1u);
  }
  return false;
}
__device__ __forceinline__ void split_f16(float x0, float x1, uint32_t& hi, uint32_t& lo) {
  const __half2 h = __floats2half2_rn(x0, x1);
  const float2 hf = __half22float2(h);
  const __half2 l = __floats2half2_rn(x0 - hf.x, x1 - hf.y);
  hi = *reinterpret_cast<const uint32_t*>(&h);
  lo = *reinterpret_cast<const uint32_t*>(&l);
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t* r) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(taddr),
      "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),
      "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
      : "memory");
}
__device__ __forceinline__ void tma_load_2d(void* dst_smem, const CUtensorMap* tm, int c0, int c1, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
          smem_u32(dst_smem)),
      "l"(reinterpret_cast<uint64_t>(tm)), "r"(c0), "r"(c1), "r"(smem_u32(bar))
      : "memory");
}

// [rows][128] fp16 row-major viewed as a 2-D tensor; box = 64 columns (128 B) x 32 rows, 128B swizzle.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int make_rows_tensor_map_f16(CUtensorMap* tm, const void* base, uint64_t rows) {
  static EncodeTiledFn fn = nullptr;
  if (fn == nullptr) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess || p == nullptr)
      return HYPIC_ERR_CUDA;
    fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  const cuuint64_t dims[2] = {(cuuint64_t)kD, (cuuint64_t)rows};
  const cuuint64_t strides[1] = {(cuuint64_t)kD * 2};
  const cuuint32_t box[2] = {64, 32};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? HYPIC_OK : HYPIC_ERR_CUDA;
}

// kHeads = 2: the CTA folds heads h0, h0 + 1 of one request as two interleaved chains (they share the step list): while the
// round-trip warps rewrite one head's state the tensor pipe multiplies the other's, instead of the strict
// MMAs -> commit -> round trip -> barrier sequence of a single chain.  TMEM: 256 columns per head.
template <int kHeads>
__global__ void __launch_bounds__(kThreads, 1)
    compose_f16_kernel(const __grid_constant__ CUtensorMap tmE, const __grid_constant__ CUtensorMap tmT,
                       const float* S_in /* may alias S_out */, const int32_t* __restrict__ seg_ids,
                       const int32_t* __restrict__ cu_segs, int R, int H, float* S_out) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  Bars* bars = reinterpret_cast<Bars*>(smem + kOffBar);
  volatile int* abort_flag = &bars->abort_flag;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int hp = H / kHeads;  // CTAs per request
  // Longest lists first (the hardware hands out CTAs in index order, so the last CTAs set the tail of the launch): the
  // request this CTA folds is the one whose list length has rank blockIdx.x / hp, ties by index.  Each CTA ranks the
  // R <= 512 lengths itself from shared memory (a microsecond); beyond that, index order.
  int r = blockIdx.x / hp;
  if (R <= 512) {
    int* s_len = reinterpret_cast<int*>(smem + kOffXch);  // free until the first round trip
    int* s_pick = &bars->req_pick;
    for (int t = threadIdx.x; t < R; t += kThreads) s_len[t] = cu_segs[t + 1] - cu_segs[t];
    __syncthreads();
    for (int t = threadIdx.x; t < R; t += kThreads) {
      const int lt = s_len[t];
      int rank = 0;
      for (int j = 0; j < R; ++j) {
        const int lj = s_len[j];
        rank += (lj > lt || (lj == lt && j < t)) ? 1 : 0;
      }
      if (rank == r) *s_pick = t;
    }
    __syncthreads();
    r = *s_pick;
    __syncthreads();  // s_len is the exchange buffer of the round trip from here on
  }
  const int h0 = (blockIdx.x % hp) * kHeads;
  const int seg_begin = cu_segs[r];
  const int n = cu_segs[r + 1] - seg_begin;
  const size_t mat = (size_t)kD * kD;

  if (warp == 0) tmem_alloc(&bars->tmem_base, 256 * kHeads);
  if (tid == 32) {
    for (int i = 0; i < kNT; ++i) { mbar_init(&bars->t_full[i], 1); mbar_init(&bars->t_empty[i], 1); }
    for (int i = 0; i < kNE; ++i) { mbar_init(&bars->e_full[i], 1); mbar_init(&bars->e_empty[i], 4); }
    for (int u = 0; u < 2; ++u) {
      mbar_init(&bars->d_full[u], 1);
      mbar_init(&bars->a_ready[u], 16);
    }
    bars->abort_flag = 0;
    fence_barrier_init();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = bars->tmem_base;
  // per head u: D fp32 at columns [256 u, 256 u + 128); S_hi, S_lo fp16 at + 128, + 192 (64 columns each)

  if (warp == 0) {
    // ---------------------------------------------------------------- T producer: 32-row slabs, two boxes each
    if (lane == 0) {
      uint32_t it = 0;
      for (int i = 0; i < n * kHeads; ++i) {
        const int row0 = (seg_ids[seg_begin + i / kHeads] * H + h0 + i % kHeads) * kD;
        const uint32_t slot = it % kNT, ph = (it / kNT) & 1;
        wait_or_abort(&bars->t_empty[slot], ph ^ 1, abort_flag);
        mbar_expect_tx(&bars->t_full[slot], kTMat);
        for (int j = 0; j < 4; ++j) {
          uint8_t* dst = smem + kOffT + slot * kTMat + j * kTSlab;
          tma_load_2d(dst, &tmT, 0, row0 + 32 * j, &bars->t_full[slot]);
          tma_load_2d(dst + kTSlab / 2, &tmT, 64, row0 + 32 * j, &bars->t_full[slot]);
        }
        ++it;
      }
    }
  } else if (warp == 1) {
    // ---------------------------------------------------------------- MMA issuer (one thread)
    if (lane == 0) {
      constexpr uint32_t idesc = make_idesc(0u, 128, 128, 0, 1);  // fp16, M = N = 128, A from TMEM, B MN-major
      uint32_t it = 0;
      for (int v = 0; v < n * kHeads; ++v) {
        const int i = v / kHeads, u = v % kHeads;
        const uint32_t tD = tmem + 256 * u, tAhi = tD + 128, tAlo = tD + 192;
        const uint32_t slot = it % kNT, ph = (it / kNT) & 1;
        wait_or_abort(&bars->t_full[slot], ph, abort_flag);  // T runs ahead of the state: probe it first
        wait_or_abort(&bars->a_ready[u], i & 1, abort_flag);
        tc_fence_after();
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const uint32_t t_addr = smem_u32(smem + kOffT + slot * kTMat + j * kTSlab);
#pragma unroll
          for (int ks = 0; ks < 2; ++ks) {
            // 16 rows of T per instruction = two 8-row atoms of 1 KB; the two 64-column boxes are 4 KB apart
            const uint64_t bd = make_desc(t_addr + ks * 2048, 4096, 1024, 2);
            const uint32_t acol = j * 16 + ks * 8;
            mma_f16_ts(tD, tAhi + acol, bd, idesc, (j | ks) > 0);
            mma_f16_ts(tD, tAlo + acol, bd, idesc, 1);
          }
        }
        mma_commit(&bars->t_empty[slot]);
        ++it;
        mma_commit(&bars->d_full[u]);
      }
    }
  } else if (warp == 2) {
    // ---------------------------------------------------------------- E producer: per TMEM lane quarter, two boxes
    if (lane == 0) {
      uint32_t it = 0;
      for (int i = 0; i < n * kHeads; ++i) {
        const int row0 = (seg_ids[seg_begin + i / kHeads] * H + h0 + i % kHeads) * kD;
        for (int q = 0; q < 4; ++q, ++it) {
          const uint32_t slot = it % kNE, ph = (it / kNE) & 1;
          wait_or_abort(&bars->e_empty[slot], ph ^ 1, abort_flag);
          mbar_expect_tx(&bars->e_full[slot], kEQuarter);
          tma_load_2d(smem + kOffE + slot * kEQuarter, &tmE, 0, row0 + 32 * q, &bars->e_full[slot]);
          tma_load_2d(smem + kOffE + slot * kEQuarter + kEQuarter / 2, &tmE, 64, row0 + 32 * q, &bars->e_full[slot]);
        }
      }
    }
  } else {
    // ---------------------------------------------------------------- round trip: D (+E) -> next S_hi/S_lo or S_out
    const int q = warp & 3;            // TMEM lane quarter this warp may touch
    const int part = (warp - 3) >> 2;  // which 32 columns of the quarter this warp handles (4 warps per quarter)
    const uint32_t lane_base = (uint32_t)(32 * q) << 16;
    const int row = 32 * q + lane;
    float unscale_u[kHeads];  // D of step s holds 2^-r_m (S T): r_m = this row's normalisation chosen after step s - 1
#pragma unroll
    for (int u = 0; u < kHeads; ++u) unscale_u[u] = 1.f;
    for (int s = -1; s < n; ++s) {
#pragma unroll
     for (int u = 0; u < kHeads; ++u) {
      const size_t unit = (size_t)r * H + h0 + u;
      const uint32_t tD = tmem + 256 * u, tAhi = tD + 128, tAlo = tD + 192;
      float* out_row = S_out + unit * mat + (size_t)row * kD + 32 * part;
      float* xch = reinterpret_cast<float*>(smem + kOffXch + 2048 * u);
      float unscale = unscale_u[u];
      const bool last = (s == n - 1);
      float xv[32];
      if (s >= 0) {
        const uint32_t ev = (uint32_t)(4 * (kHeads * s + u) + q);
        const uint32_t eslot = ev % kNE, eph = (ev / kNE) & 1;
        wait_or_abort(&bars->e_full[eslot], eph, abort_flag);  // E runs ahead: its probe overlaps the MMAs
        wait_or_abort(&bars->d_full[u], s & 1, abort_flag);
        tc_fence_after();
        const uint8_t* eb = smem + kOffE + eslot * kEQuarter + (part >> 1) * (kEQuarter / 2) + lane * 128;
        uint32_t d[32];
        tmem_ld32(tD + lane_base + 32 * part, d);
        tmem_ld_wait();
#pragma unroll
        for (int u = 0; u < 4; ++u) {  // 8 columns per 16-byte chunk
          const uint4 e = *reinterpret_cast<const uint4*>(eb + (((4 * (part & 1) + u) ^ (lane & 7)) * 16));
          const uint32_t ew[4] = {e.x, e.y, e.z, e.w};
#pragma unroll
          for (int p = 0; p < 4; ++p) {
            const float2 ef = __half22float2(*reinterpret_cast<const __half2*>(&ew[p]));
            xv[8 * u + 2 * p] = fmaf(__uint_as_float(d[8 * u + 2 * p]), unscale, ef.x);
            xv[8 * u + 2 * p + 1] = fmaf(__uint_as_float(d[8 * u + 2 * p + 1]), unscale, ef.y);
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars->e_empty[eslot]);
      } else {
        const float4* src = reinterpret_cast<const float4*>(S_in + unit * mat + (size_t)row * kD + 32 * part);
#pragma unroll
        for (int u = 0; u < 8; ++u) {
          const float4 v = (S_in != nullptr) ? src[u] : make_float4(0.f, 0.f, 0.f, 0.f);
          xv[4 * u] = v.x, xv[4 * u + 1] = v.y, xv[4 * u + 2] = v.z, xv[4 * u + 3] = v.w;
        }
      }
      if (last) {
        float4* o4 = reinterpret_cast<float4*>(out_row);
#pragma unroll
        for (int u = 0; u < 8; ++u) o4[u] = make_float4(xv[4 * u], xv[4 * u + 1], xv[4 * u + 2], xv[4 * u + 3]);
      } else {
        // row normalisation: maximum of the whole row (all four column parts) into [2^13, 2^14)
        float m = 0.f;
#pragma unroll
        for (int c = 0; c < 32; c += 2) m = fmaxf(m, fmaxf(fabsf(xv[c]), fabsf(xv[c + 1])));
        xch[4 * row + part] = m;
        named_bar_sync(1 + q, 128);
        const float4 mm = *reinterpret_cast<const float4*>(xch + 4 * row);
        m = fmaxf(fmaxf(mm.x, mm.y), fmaxf(mm.z, mm.w));
        const int e = (int)(__float_as_uint(m) >> 23);
        int rs = (e == 0) ? 0 : e - 140;  // max in [2^(e-127), 2^(e-126)) -> 2^-rs max in [2^13, 2^14)
        rs = max(-100, min(100, rs));
        const float sc = __uint_as_float((uint32_t)(127 - rs) << 23);
        unscale_u[u] = __uint_as_float((uint32_t)(127 + rs) << 23);
        uint32_t hi[16], lo[16];
#pragma unroll
        for (int c = 0; c < 16; ++c) split_f16(xv[2 * c] * sc, xv[2 * c + 1] * sc, hi[c], lo[c]);
        tmem_st16(tAhi + lane_base + 16 * part, hi);
        tmem_st16(tAlo + lane_base + 16 * part, lo);
        tmem_st_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars->a_ready[u]);
      }
     }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, 256 * kHeads);
}

__global__ void pack_f16_kernel(const float* __restrict__ src, __half* __restrict__ dst, size_t n) {
  const size_t i4 = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) * 4;
  if (i4 + 3 < n) {
    const float4 v = *reinterpret_cast<const float4*>(src + i4);
    const __half2 a = __floats2half2_rn(v.x, v.y), b = __floats2half2_rn(v.z, v.w);
    *reinterpret_cast<uint2*>(dst + i4) = make_uint2(*reinterpret_cast<const uint32_t*>(&a), *reinterpret_cast<const uint32_t*>(&b));
  } else {
    for (size_t i = i4; i < n; ++i) dst[i] = __float2half_rn(src[i]);
  }
}

}  // namespace

bool compose_f16_shape_ok(int32_t, int32_t dk, int32_t dv) { return dk == kD && dv == kD; }

int compose_f16(const ComposeF16Args& a) {
  if (!compose_f16_shape_ok(a.H, a.dk, a.dv)) return HYPIC_ERR_UNSUPPORTED;
  if (a.R == 0) return HYPIC_OK;
  static std::atomic<unsigned long long> configured{0};
  int cfg_dev = 0;
  if (needs_device_setup(configured, &cfg_dev)) {
    HYPIC_CUDA_OK(cudaFuncSetAttribute(compose_f16_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes));
    HYPIC_CUDA_OK(cudaFuncSetAttribute(compose_f16_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes));
    device_setup_done(configured, cfg_dev);
  }
  const long long units = (long long)a.R * a.H;
  if (units > 0x7fffffffLL) return HYPIC_ERR_UNSUPPORTED;
  CUtensorMap tmE, tmT;
  if (a.total_steps > 0) {
    int rc = make_rows_tensor_map_f16(&tmE, a.E_pool, (uint64_t)a.P * a.H * kD);
    if (rc == HYPIC_OK) rc = make_rows_tensor_map_f16(&tmT, a.T_pool, (uint64_t)a.P * a.H * kD);
    if (rc != HYPIC_OK) return rc;
  } else {
    memset(&tmE, 0, sizeof(tmE));
    memset(&tmT, 0, sizeof(tmT));
  }
  // heads h, h + 1 of a request as two interleaved chains of one CTA -- once there are enough units to keep every SM busy
  // that way; with fewer (cfg2: 32 chains) one chain per CTA on twice the SMs is the faster schedule (0.076 vs 0.113 ms)
  const DeviceInfo& di = device_info();
  if (a.H % 2 == 0 && units >= 2LL * (di.ok ? di.sm_count : 148))
    compose_f16_kernel<2><<<(unsigned)(units / 2), kThreads, kSmemBytes, a.stream>>>(tmE, tmT, a.S_in, a.seg_ids,
                                                                                    a.cu_segs, a.R, a.H, a.S_out);
  else
    compose_f16_kernel<1><<<(unsigned)units, kThreads, kSmemBytes, a.stream>>>(tmE, tmT, a.S_in, a.seg_ids, a.cu_segs,
                                                                              a.R, a.H, a.S_out);
  note_launch();
  HYPIC_CUDA_OK(cudaGetLastError());
  return HYPIC_OK;
}

int pack_f16(const float* src, void* dst, size_t n, cudaStream_t stream) {
  if (n == 0) return HYPIC_OK;
  const size_t threads = (n + 3) / 4;
  const size_t blocks = (threads + 255) / 256;
  if (blocks > 0x7fffffffULL) return HYPIC_ERR_UNSUPPORTED;
  pack_f16_kernel<<<(unsigned)blocks, 256, 0, stream>>>(src, static_cast<__half*>(dst), n);
  note_launch();
  HYPIC_CUDA_OK(cudaGetLastError());
  return HYPIC_OK;
}

unsigned int debug_timeout_count_compose_f16() {
  unsigned int v = 0;
  if (cudaMemcpyFromSymbol(&v, g_timeout_count_f16, sizeof(v)) != cudaSuccess) return 0xffffffffu;
  return v;
}

}  // namespace hypic
