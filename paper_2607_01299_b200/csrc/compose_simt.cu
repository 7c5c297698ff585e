// compose_simt.cu -- fp32 CUDA-core composition (kernel family HYPIC_IMPL_SIMT).
//
// Row a6 of SURVEY.md section 8(a): for each (request, head) fold S <- S T_i + E_i (Eq. 6 as the
// chain of Eq. 4 steps) over the request's ordered id list.  Rows of S are independent, so a CTA owns a block
// of up to 128 rows of one (request, head); S stays in shared memory (stored transposed) for the whole
// chain, T_i streams through shared memory in 16-row k-slabs, E_i is read straight from global memory into
// the accumulators.  Plain FFMA, fp32 accumulation in list order: the accurate (1e-5 class) path; bound by
// the fp32 pipe, not by HBM -- the tensor-core family (compose_tensor.cu) is the HBM-bound one.
#include "common.cuh"

namespace hypic {
namespace {

constexpr int kThreads = 256;  // 16 x 16 threads, each an 8 x (DK/16) micro-tile
constexpr int kBM = 128;       // rows of S per CTA
constexpr int kSlab = 16;      // rows of T per staged slab

template <int DK>
__global__ void __launch_bounds__(kThreads) compose_simt_kernel(const float* S_in,  /* may alias S_out: no __restrict__, no read-only path */
                                                                const float* __restrict__ E_pool,
                                                                const float* __restrict__ T_pool,
                                                                const int32_t* __restrict__ seg_ids,
                                                                const int32_t* __restrict__ cu_segs, int H, int dv,
                                                                float* S_out) {
  constexpr int NJ = DK / 16;     // output columns per thread
  constexpr int LDS_ = kBM + 4;   // padded leading dimension of the transposed state
  extern __shared__ __align__(16) float smem[];
  float* St = smem;                    // [DK][LDS_]   St[c][i] = S[i][c]
  float* Ts = smem + DK * LDS_;        // [2][kSlab][DK]

  const int tid = threadIdx.x;
  const int tx = tid % 16, ty = tid / 16;
  const int h = blockIdx.y, r = blockIdx.z;
  const int row0 = blockIdx.x * kBM;
  const int n_rows = min(kBM, dv - row0);
  const int j0 = tx * NJ, i0 = ty * 8;

  // load S_in rows (or zeros) transposed into shared memory
  const size_t s_off = (((size_t)r * H + h) * dv + row0) * DK;
  for (int idx = tid; idx < kBM * DK; idx += kThreads) {
    const int i = idx / DK, c = idx % DK;
    float val = 0.f;
    if (S_in != nullptr && i < n_rows) val = S_in[s_off + (size_t)i * DK + c];
    St[c * LDS_ + i] = val;
  }
  __syncthreads();

  const int seg_begin = cu_segs[r], seg_end = cu_segs[r + 1];
  for (int sidx = seg_begin; sidx < seg_end; ++sidx) {
    const int id = seg_ids[sidx];
    const float* Tg = T_pool + ((size_t)id * H + h) * DK * DK;
    const float* Eg = E_pool + (((size_t)id * H + h) * dv + row0) * DK;

    float acc[8][NJ];
#pragma unroll
    for (int ii = 0; ii < 8; ++ii) {
      if (i0 + ii < n_rows) {
#pragma unroll
        for (int jj = 0; jj < NJ; jj += 4) {
          const float4 e = *reinterpret_cast<const float4*>(Eg + (size_t)(i0 + ii) * DK + j0 + jj);
          acc[ii][jj] = e.x, acc[ii][jj + 1] = e.y, acc[ii][jj + 2] = e.z, acc[ii][jj + 3] = e.w;
        }
      } else {
#pragma unroll
        for (int jj = 0; jj < NJ; ++jj) acc[ii][jj] = 0.f;
      }
    }

    constexpr int kSlabElems = kSlab * DK;
    auto stage = [&](int buf, int slab) {
      const float4* src = reinterpret_cast<const float4*>(Tg + (size_t)slab * kSlabElems);
      float4* dst = reinterpret_cast<float4*>(Ts + buf * kSlabElems);
      for (int idx = tid; idx < kSlabElems / 4; idx += kThreads) dst[idx] = src[idx];
    };
    stage(0, 0);
    __syncthreads();
    constexpr int n_slabs = DK / kSlab;
    for (int slab = 0; slab < n_slabs; ++slab) {
      const int buf = slab & 1;
      if (slab + 1 < n_slabs) stage(buf ^ 1, slab + 1);
      const float* Tb = Ts + buf * kSlabElems;
#pragma unroll
      for (int kk = 0; kk < kSlab; ++kk) {
        const int c = slab * kSlab + kk;
        const float4 a0 = *reinterpret_cast<const float4*>(St + c * LDS_ + i0);
        const float4 a1 = *reinterpret_cast<const float4*>(St + c * LDS_ + i0 + 4);
        const float av[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
        float bv[NJ];
#pragma unroll
        for (int jj = 0; jj < NJ; jj += 4) {
          const float4 b4 = *reinterpret_cast<const float4*>(Tb + kk * DK + j0 + jj);
          bv[jj] = b4.x, bv[jj + 1] = b4.y, bv[jj + 2] = b4.z, bv[jj + 3] = b4.w;
        }
#pragma unroll
        for (int ii = 0; ii < 8; ++ii)
#pragma unroll
          for (int jj = 0; jj < NJ; ++jj) acc[ii][jj] = fmaf(av[ii], bv[jj], acc[ii][jj]);
      }
      __syncthreads();
    }
    // every thread has finished reading St (last barrier above): write the new state back, transposed
#pragma unroll
    for (int jj = 0; jj < NJ; ++jj) {
      float4* d = reinterpret_cast<float4*>(St + (j0 + jj) * LDS_ + i0);
      d[0] = make_float4(acc[0][jj], acc[1][jj], acc[2][jj], acc[3][jj]);
      d[1] = make_float4(acc[4][jj], acc[5][jj], acc[6][jj], acc[7][jj]);
    }
    __syncthreads();
  }

  float* out = S_out + s_off;
  for (int idx = tid; idx < kBM * DK; idx += kThreads) {
    const int i = idx / DK, c = idx % DK;
    if (i < n_rows) out[(size_t)i * DK + c] = St[c * LDS_ + i];
  }
}

template <int DK>
int launch(const ComposeArgs& a) {
  const size_t smem = (size_t)(DK * (kBM + 4) + 2 * kSlab * DK) * sizeof(float);
  static std::atomic<unsigned long long> configured{0};
  int cfg_dev = 0;
  if (needs_device_setup(configured, &cfg_dev)) {
    HYPIC_CUDA_OK(cudaFuncSetAttribute(compose_simt_kernel<DK>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)smem));
    device_setup_done(configured, cfg_dev);
  }
  dim3 grid((a.dv + kBM - 1) / kBM, a.H, a.R);
  compose_simt_kernel<DK><<<grid, kThreads, smem, a.stream>>>(a.S_in, a.E_pool, a.T_pool, a.seg_ids, a.cu_segs, a.H,
                                                              a.dv, a.S_out);
  note_launch();
  HYPIC_CUDA_OK(cudaGetLastError());
  return HYPIC_OK;
}

}  // namespace

int compose_simt(const ComposeArgs& a) {
  if (a.H > 65535 || a.R > 65535) return HYPIC_ERR_UNSUPPORTED;
  if (a.dv < 1 || a.dv > 1024) return HYPIC_ERR_UNSUPPORTED;
  if (a.R == 0) return HYPIC_OK;
  if (a.dk == 128) return launch<128>(a);
  if (a.dk == 64) return launch<64>(a);
  return HYPIC_ERR_UNSUPPORTED;
}

}  // namespace hypic
