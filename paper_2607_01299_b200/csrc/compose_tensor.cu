// compose_tensor.cu -- tcgen05/TMEM composition, dk = dv = 128 (kernel family HYPIC_IMPL_TENSOR).
//
// Row a6 of SURVEY.md section 8(a):  S <- S T_i + E_i  (Eq. 6 as the chain of Eq. 4 steps) for one
// (request, head) chain per CTA.  The chain is HBM-bound (128 KB of (T_i, E_i) per 4.2 MFLOP step), so the kernel
// is a streaming pipeline; tensor cores only keep the fp32-accurate GEMM off the critical path:
//   * S lives in TMEM for the whole chain as two tf32 operands S_hi = rna_tf32(S), S_lo = S - S_hi
//     (A operand of tcgen05.mma kind::tf32 read from TMEM: lane = row of S, column = k);
//   * T_i streams HBM -> smem in 32-row slabs (1-D bulk async copies on mbarriers), converter warps split
//     each slab into T_hi / T_lo in the 32-bit MN-major "128B swizzle, 32B base" layout (B operand);
//   * 3xTF32:  D = S_hi T_hi + S_lo T_hi + S_hi T_lo  (fp32 accumulate in TMEM; the hardware truncates tf32
//     operands, which is why hi is rounded in software and lo carries the remainder);
//   * round-trip warps (two per TMEM lane quarter) read D (tcgen05.ld), add E_i (staged by TMA tensor boxes of
//     32 rows x 128 B with the 128B swizzle, so that row-per-thread reads are bank-conflict free; per-row bulk
//     copies were measured to cost ~46 cycles of TMA issue each and dominated the step), and write the next
//     S_hi / S_lo (tcgen05.st), or S_out after the last step.
// S_in enters as "step -1" (D = 0, E = S_in).  All waits are bounded: a protocol error raises the timeout
// counter (hypic_debug_timeout_count) instead of hanging the GPU.
#include <cuda.h>
#include <string.h>

#include "common.cuh"
#include "sm100_ptx.cuh"

namespace hypic {

__device__ unsigned int g_timeout_count = 0;

namespace {
using namespace ptx;

constexpr int kD = 128;
constexpr int kSlabBytes = 32 * kD * 4;  // 32 rows of T (or E): 16 KB
constexpr int kNRaw = 3;                 // raw T slabs in flight
constexpr int kNHl = 3;                  // converted (hi, lo) slab pairs
constexpr int kESlotBytes = kSlabBytes;  // 4 TMA boxes of 32 rows x 128 B (128B swizzle: conflict-free row reads)
constexpr int kThreads = 480;            // warp 0 T producer, 1 MMA, 2 E producer, 3-6 converters, 7-14 round trip

constexpr int kOffHl = 0;
constexpr int kOffRaw = kOffHl + kNHl * 2 * kSlabBytes;
constexpr int kOffE = kOffRaw + kNRaw * kSlabBytes;
constexpr int kOffBar = kOffE + 4 * kESlotBytes;
constexpr int kSmemBytes = kOffBar + 256 + 1024;  // + barriers + alignment slack

struct Bars {
  uint64_t raw_full[kNRaw], raw_empty[kNRaw], hl_full[kNHl], hl_empty[kNHl], e_full[4], e_empty[4], d_full, a_ready;
  uint32_t tmem_base;
  int abort_flag;
};

__device__ __forceinline__ bool wait_or_abort(uint64_t* bar, uint32_t parity, volatile int* abort_flag) {
  for (uint32_t i = 0; i < 4000000u; ++i) {
    if (mbar_try_wait(bar, parity)) return true;
    if ((i & 1023u) == 1023u && *abort_flag) return false;
  }
  if (!*abort_flag) {
    *abort_flag = 1;
    atomicAdd(&g_timeout_count, 1u);
  }
  return false;
}

__device__ __forceinline__ float rna_tf32(float x) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return __uint_as_float(r);
}

__device__ __forceinline__ void tma_load_2d(void* dst_smem, const CUtensorMap* tm, int c0, int c1, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
          smem_u32(dst_smem)),
      "l"(reinterpret_cast<uint64_t>(tm)), "r"(c0), "r"(c1), "r"(smem_u32(bar))
      : "memory");
}

// [rows][128] fp32 row-major viewed as a 2-D tensor; box = 32 columns (128 B) x 32 rows, 128B swizzle.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int make_rows_tensor_map(CUtensorMap* tm, const float* base, uint64_t rows) {
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
  const cuuint64_t strides[1] = {(cuuint64_t)kD * 4};
  const cuuint32_t box[2] = {32, 32};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float*>(base), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? HYPIC_OK : HYPIC_ERR_CUDA;
}

__global__ void __launch_bounds__(kThreads, 1)
    compose_tensor_kernel(const __grid_constant__ CUtensorMap tmE, const __grid_constant__ CUtensorMap tmS,
                          const float* __restrict__ S_in, const float* __restrict__ T_pool, const int32_t* __restrict__ seg_ids,
                          const int32_t* __restrict__ cu_segs, int H, float* __restrict__ S_out) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  Bars* bars = reinterpret_cast<Bars*>(smem + kOffBar);
  volatile int* abort_flag = &bars->abort_flag;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int unit = blockIdx.x;
  const int r = unit / H, h = unit % H;
  const int seg_begin = cu_segs[r];
  const int n = cu_segs[r + 1] - seg_begin;
  const size_t mat = (size_t)kD * kD;

  if (warp == 0) tmem_alloc(&bars->tmem_base, 512);
  if (tid == 32) {
    for (int i = 0; i < kNRaw; ++i) { mbar_init(&bars->raw_full[i], 1); mbar_init(&bars->raw_empty[i], 4); }
    for (int i = 0; i < kNHl; ++i) { mbar_init(&bars->hl_full[i], 4); mbar_init(&bars->hl_empty[i], 1); }
    for (int i = 0; i < 4; ++i) { mbar_init(&bars->e_full[i], 1); mbar_init(&bars->e_empty[i], 2); }
    mbar_init(&bars->d_full, 1);
    mbar_init(&bars->a_ready, 8);
    bars->abort_flag = 0;
    fence_barrier_init();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = bars->tmem_base;
  const uint32_t tD = tmem, tAhi = tmem + 128, tAlo = tmem + 256;

  if (warp == 0) {
    // ---------------------------------------------------------------- T producer: 16 KB slabs into the raw ring
    if (lane == 0) {
      uint32_t it = 0;
      for (int i = 0; i < n; ++i) {
        const int id = seg_ids[seg_begin + i];
        const float* Tg = T_pool + ((size_t)id * H + h) * mat;
        for (int j = 0; j < 4; ++j, ++it) {
          const uint32_t slot = it % kNRaw, ph = (it / kNRaw) & 1;
          wait_or_abort(&bars->raw_empty[slot], ph ^ 1, abort_flag);
          mbar_expect_tx(&bars->raw_full[slot], kSlabBytes);
          bulk_g2s(smem + kOffRaw + slot * kSlabBytes, Tg + (size_t)j * 32 * kD, kSlabBytes, &bars->raw_full[slot]);
        }
      }
    }
  } else if (warp == 1) {
    // ---------------------------------------------------------------- MMA issuer (one thread)
    if (lane == 0) {
      constexpr uint32_t idesc = make_idesc(2u, 128, 128, 0, 1);  // tf32, M = N = 128, B MN-major
      uint32_t it = 0;
      for (int i = 0; i < n; ++i) {
        wait_or_abort(&bars->a_ready, i & 1, abort_flag);
        tc_fence_after();
        for (int j = 0; j < 4; ++j, ++it) {
          const uint32_t slot = it % kNHl, ph = (it / kNHl) & 1;
          wait_or_abort(&bars->hl_full[slot], ph, abort_flag);
          tc_fence_after();
          const uint32_t hi_addr = smem_u32(smem + kOffHl + slot * 2 * kSlabBytes);
          const uint32_t lo_addr = hi_addr + kSlabBytes;
#pragma unroll
          for (int ks = 0; ks < 4; ++ks) {
            // 8 rows of T per instruction = two 4-row atoms of 512 B; 32-column chunks are 4 KB apart
            const uint64_t bhi = make_desc(hi_addr + ks * 1024, 4096, 512, 1);
            const uint64_t blo = make_desc(lo_addr + ks * 1024, 4096, 512, 1);
            const uint32_t acol = j * 32 + ks * 8;
            mma_tf32_ts(tD, tAhi + acol, bhi, idesc, (j | ks) > 0);
            mma_tf32_ts(tD, tAlo + acol, bhi, idesc, 1);
            mma_tf32_ts(tD, tAhi + acol, blo, idesc, 1);
          }
          mma_commit(&bars->hl_empty[slot]);
        }
        mma_commit(&bars->d_full);
      }
    }
  } else if (warp == 2) {
    // ---------------------------------------------------------------- E producer: 4 TMA boxes (32 x 32 fp32) per slab
    if (lane < 4) {
      uint32_t ecount = 0;
      for (int s = -1; s < n; ++s) {
        const CUtensorMap* tm;
        int row0;
        if (s < 0) {
          if (S_in == nullptr) continue;
          tm = &tmS;
          row0 = unit * kD;
        } else {
          tm = &tmE;
          row0 = (seg_ids[seg_begin + s] * H + h) * kD;
        }
        for (int q = 0; q < 4; ++q) {
          wait_or_abort(&bars->e_empty[q], (ecount & 1) ^ 1, abort_flag);
          if (lane == 0) mbar_expect_tx(&bars->e_full[q], kSlabBytes);
          __syncwarp(0xf);
          tma_load_2d(smem + kOffE + q * kESlotBytes + lane * 4096, tm, 32 * lane, row0 + 32 * q, &bars->e_full[q]);
        }
        ++ecount;
      }
    }
  } else if (warp < 7) {
    // ---------------------------------------------------------------- converters: raw slab -> (hi, lo) tiles
    const int ctid = tid - 96;
    uint32_t it = 0;
    for (int i = 0; i < n; ++i) {
      for (int j = 0; j < 4; ++j, ++it) {
        const uint32_t rslot = it % kNRaw, rph = (it / kNRaw) & 1;
        const uint32_t hslot = it % kNHl, hph = (it / kNHl) & 1;
        wait_or_abort(&bars->raw_full[rslot], rph, abort_flag);
        const float4* raw = reinterpret_cast<const float4*>(smem + kOffRaw + rslot * kSlabBytes);
        float4 x[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) x[u] = raw[ctid + 128 * u];
        wait_or_abort(&bars->hl_empty[hslot], hph ^ 1, abort_flag);
        uint8_t* hi_t = smem + kOffHl + hslot * 2 * kSlabBytes;
        uint8_t* lo_t = hi_t + kSlabBytes;
#pragma unroll
        for (int u = 0; u < 8; ++u) {
          const int idx = ctid + 128 * u;
          const int k = idx >> 5, n0 = (idx & 31) * 4;  // row of the slab, first of 4 columns
          const uint32_t off = (n0 >> 5) * 4096 + (k >> 2) * 512 + (k & 3) * 128 +
                               ((((n0 & 31) >> 3) ^ (k & 3)) * 32) + ((n0 & 7) * 4);
          float4 hi, lo;
          hi.x = rna_tf32(x[u].x), hi.y = rna_tf32(x[u].y), hi.z = rna_tf32(x[u].z), hi.w = rna_tf32(x[u].w);
          lo.x = x[u].x - hi.x, lo.y = x[u].y - hi.y, lo.z = x[u].z - hi.z, lo.w = x[u].w - hi.w;
          *reinterpret_cast<float4*>(hi_t + off) = hi;
          *reinterpret_cast<float4*>(lo_t + off) = lo;
        }
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) {
          mbar_arrive(&bars->hl_full[hslot]);
          mbar_arrive(&bars->raw_empty[rslot]);
        }
      }
    }
  } else {
    // ---------------------------------------------------------------- round trip: D (+E) -> next S_hi/S_lo or S_out
    const int q = warp & 3;            // TMEM lane quarter this warp may touch
    const int half = (warp - 7) >> 2;  // which 64 columns of the quarter this warp handles
    const uint32_t lane_base = (uint32_t)(32 * q) << 16;
    const int row = 32 * q + lane;
    const uint8_t* erow = smem + kOffE + q * kESlotBytes + lane * 128;
    float* out_row = S_out + (size_t)unit * mat + (size_t)row * kD;
    uint32_t ecount = 0;
    for (int s = -1; s < n; ++s) {
      const bool have_e = (s >= 0) || (S_in != nullptr);
      const bool last = (s == n - 1);
      if (s >= 0) {
        wait_or_abort(&bars->d_full, s & 1, abort_flag);
        tc_fence_after();
      }
      if (have_e) wait_or_abort(&bars->e_full[q], ecount & 1, abort_flag);
#pragma unroll 1
      for (int cb = 2 * half; cb < 2 * half + 2; ++cb) {
        uint32_t d[32];
        if (s >= 0) {
          tmem_ld32(tD + lane_base + 32 * cb, d);
          tmem_ld_wait();
        } else {
#pragma unroll
          for (int c = 0; c < 32; ++c) d[c] = 0u;
        }
        float xv[32];
#pragma unroll
        for (int c = 0; c < 32; ++c) xv[c] = __uint_as_float(d[c]);
        if (have_e) {
          const uint8_t* eb = erow + cb * 4096;
#pragma unroll
          for (int u = 0; u < 8; ++u) {
            const float4 e = *reinterpret_cast<const float4*>(eb + ((u ^ (lane & 7)) * 16));
            xv[4 * u] += e.x, xv[4 * u + 1] += e.y, xv[4 * u + 2] += e.z, xv[4 * u + 3] += e.w;
          }
        }
        if (last) {
          float4* o4 = reinterpret_cast<float4*>(out_row + 32 * cb);
#pragma unroll
          for (int u = 0; u < 8; ++u) o4[u] = make_float4(xv[4 * u], xv[4 * u + 1], xv[4 * u + 2], xv[4 * u + 3]);
        } else {
          uint32_t hi[32], lo[32];
#pragma unroll
          for (int c = 0; c < 32; ++c) {
            const float hf = rna_tf32(xv[c]);
            hi[c] = __float_as_uint(hf);
            lo[c] = __float_as_uint(xv[c] - hf);
          }
          tmem_st32(tAhi + lane_base + 32 * cb, hi);
          tmem_st32(tAlo + lane_base + 32 * cb, lo);
        }
      }
      if (have_e) {
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars->e_empty[q]);
        ++ecount;
      }
      if (!last) {
        tmem_st_wait();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&bars->a_ready);
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 0) tmem_dealloc(tmem, 512);
}

}  // namespace

bool compose_tensor_shape_ok(int32_t, int32_t dk, int32_t dv) { return dk == kD && dv == kD; }

int compose_tensor(const ComposeArgs& a) {
  if (!compose_tensor_shape_ok(a.H, a.dk, a.dv)) return HYPIC_ERR_UNSUPPORTED;
  if (a.R == 0) return HYPIC_OK;
  static bool configured = false;
  if (!configured) {
    HYPIC_CUDA_OK(cudaFuncSetAttribute(compose_tensor_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemBytes));
    configured = true;
  }
  const long long units = (long long)a.R * a.H;
  if (units > 0x7fffffffLL) return HYPIC_ERR_UNSUPPORTED;
  CUtensorMap tmE, tmS;
  if (a.total_steps > 0 || a.S_in != nullptr) {
    const int rc = make_rows_tensor_map(&tmE, a.total_steps > 0 ? a.E_pool : a.S_in,
                                        a.total_steps > 0 ? (uint64_t)a.P * a.H * kD : (uint64_t)units * kD);
    if (rc != HYPIC_OK) return rc;
  } else {
    memset(&tmE, 0, sizeof(tmE));
  }
  tmS = tmE;
  if (a.S_in != nullptr) {
    const int rc = make_rows_tensor_map(&tmS, a.S_in, (uint64_t)units * kD);
    if (rc != HYPIC_OK) return rc;
  }
  compose_tensor_kernel<<<(unsigned)units, kThreads, kSmemBytes, a.stream>>>(tmE, tmS, a.S_in, a.T_pool, a.seg_ids,
                                                                            a.cu_segs, a.H, a.S_out);
  note_launch();
  HYPIC_CUDA_OK(cudaGetLastError());
  return HYPIC_OK;
}

unsigned int debug_timeout_count() {
  unsigned int v = 0;
  if (cudaMemcpyFromSymbol(&v, g_timeout_count, sizeof(v)) != cudaSuccess) return 0xffffffffu;
  const unsigned int e = debug_timeout_count_encode();
  return e == 0xffffffffu ? e : v + e;
}

}  // namespace hypic
