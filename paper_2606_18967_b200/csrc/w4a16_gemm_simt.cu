// w4a16_gemm_simt.cu -- er_w4a16_gemm_simt: plain CUDA-core W4A16 linear (debug / cross-check aid for the
// tcgen05 kernel in w4a16_gemm.cu; same contract, include/er.h).  One warp per output column n, lanes
// stride over packed words, 8 batch rows per pass; per-group fp32 partial sums scaled by the group scale.
#include "er_common.cuh"

namespace {

constexpr int kMC = 8;  // batch rows per pass

__global__ void __launch_bounds__(128) w4a16_simt_kernel(const __nv_bfloat16* __restrict__ x, int M, int K,
                                                         int64_t ldx, const uint32_t* __restrict__ qw,
                                                         const __nv_bfloat16* __restrict__ scales, int N, void* y,
                                                         int64_t ldy, int y_f32) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int n = blockIdx.x * 4 + warp;
  if (n >= N) return;
  const int words = K >> 3, groups = K >> 7;
  for (int m0 = blockIdx.y * kMC; m0 < M; m0 += gridDim.y * kMC) {
    float acc[kMC];
#pragma unroll
    for (int i = 0; i < kMC; ++i) acc[i] = 0.f;
    for (int g = 0; g < groups; ++g) {
      float part[kMC];
#pragma unroll
      for (int i = 0; i < kMC; ++i) part[i] = 0.f;
      if (lane < 16) {  // 16 words per group
        const int j = g * 16 + lane;
        const uint32_t wd = qw[er::packed_word_index(n, j, groups)];
#pragma unroll
        for (int t = 0; t < 4; ++t) {
          const float q0 = (float)((int)((wd >> (4 * t)) & 0xF) - 8);       // k = 8 j + 2 t
          const float q1 = (float)((int)((wd >> (4 * t + 16)) & 0xF) - 8);  // k = 8 j + 2 t + 1
          const int k = 8 * j + 2 * t;
#pragma unroll
          for (int i = 0; i < kMC; ++i) {
            if (m0 + i < M) {
              const __nv_bfloat162 xv = *reinterpret_cast<const __nv_bfloat162*>(x + (size_t)(m0 + i) * ldx + k);
              part[i] = fmaf(__bfloat162float(xv.x), q0, part[i]);
              part[i] = fmaf(__bfloat162float(xv.y), q1, part[i]);
            }
          }
        }
      }
      const float s = __bfloat162float(scales[(size_t)g * N + n]);
#pragma unroll
      for (int i = 0; i < kMC; ++i) {
        float p = part[i];
#pragma unroll
        for (int o = 8; o > 0; o >>= 1) p += __shfl_xor_sync(0xffffffffu, p, o);
        acc[i] = fmaf(s, p, acc[i]);
      }
    }
    if (lane == 0) {
#pragma unroll
      for (int i = 0; i < kMC; ++i) {
        if (m0 + i < M) {
          if (y_f32) reinterpret_cast<float*>(y)[(size_t)(m0 + i) * ldy + n] = acc[i];
          else reinterpret_cast<__nv_bfloat16*>(y)[(size_t)(m0 + i) * ldy + n] = __float2bfloat16_rn(acc[i]);
        }
      }
    }
  }
}

}  // namespace

extern "C" int er_w4a16_gemm_simt(const void* x_bf16, int64_t M, int64_t K, int64_t ldx_elems, const void* qweight,
                                  const void* scales, int64_t N, int group, void* y, int64_t ldy_elems, int y_dtype,
                                  void* stream) {
  if (!x_bf16 || !qweight || !scales || !y) return ER_ERR_NULL;
  if (group != ER_GROUP || M < 1 || N < 128 || N % 128 != 0 || K < ER_GROUP || K % ER_GROUP != 0 || ldx_elems < K || ldy_elems < N ||
      M > (1 << 20) || N > (1 << 24) || K > (1 << 24))
    return ER_ERR_SHAPE;
  if (y_dtype != ER_BF16 && y_dtype != ER_F32) return ER_ERR_DTYPE;
  if ((reinterpret_cast<uintptr_t>(x_bf16) & 3u) || (ldx_elems & 1) || (reinterpret_cast<uintptr_t>(qweight) & 3u))
    return ER_ERR_ALIGN;
  int st = er::check_arch();
  if (st != ER_OK) return st;
  dim3 grid((unsigned)((N + 3) / 4), (unsigned)((M + kMC - 1) / kMC > 32 ? 32 : (M + kMC - 1) / kMC));
  w4a16_simt_kernel<<<grid, 128, 0, (cudaStream_t)stream>>>(
      reinterpret_cast<const __nv_bfloat16*>(x_bf16), (int)M, (int)K, ldx_elems,
      reinterpret_cast<const uint32_t*>(qweight), reinterpret_cast<const __nv_bfloat16*>(scales), (int)N, y, ldy_elems,
      y_dtype == ER_F32);
  ER_CUDA_TRY(cudaGetLastError());
  return ER_OK;
}
