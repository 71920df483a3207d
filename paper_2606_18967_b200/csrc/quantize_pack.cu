// quantize_pack.cu -- er_quantize_pack: the per-RL-step drafter refresh ("lightweight RTN
// quantization to the FFN and QKVO projection layers", L150 Alg. 1 line 3) and er_unpack_codes.
//
// HBM-bound streaming kernel: 2 B read + 0.5 B + 2/128 B written per element.
// One CTA quantizes a tile of 32 rows x 512 k.  A lane owns 8 consecutive k (one 128-bit load, one 32-bit
// packed word out); 16 lanes cover one 128-element group, so the group max is 4 shuffle-xor steps.  All 8
// loads of a thread are issued before any arithmetic (128 B in flight per thread).  The 4 x 32 scales of
// the tile are transposed through shared memory so that they leave as 64-byte runs along N.
#include "er_common.cuh"

namespace {

constexpr int kTileRows = 32;
constexpr int kTileK = 512;
constexpr int kThreads = 256;
constexpr int kIters = 8;  // (row, 256-wide half) pairs per warp: 4 rows x 2 halves

__device__ __forceinline__ uint4 ld_stream(const uint4* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}

// q = clamp(rint(w / s), -8, 7) + 8 with IEEE-division semantics at the ties that matter (Q6):
// t = w * r (r = rn(1/s)) is refined by one exact-residual Newton step, which returns k + 1/2 exactly
// whenever w / s is exactly k + 1/2, and is otherwise within ~1e-6 of w / s while every non-tie quotient
// of two 8-bit significands is >= 1/1020 away from a tie.
__device__ __forceinline__ uint32_t code_of(float w, float s, float r) {
  float t = w * r;
  float e = __fmaf_rn(-t, s, w);
  t = __fmaf_rn(e, r, t);
  float q = rintf(t);
  q = fminf(fmaxf(q, -8.0f), 7.0f);
  return (uint32_t)(__float2int_rn(q) + 8);
}
__device__ __forceinline__ uint32_t code_of_div(float w, float s) {
  float q = rintf(__fdiv_rn(w, s));
  q = fminf(fmaxf(q, -8.0f), 7.0f);
  return (uint32_t)(__float2int_rn(q) + 8);
}

__global__ void __launch_bounds__(kThreads) quantize_pack_kernel(const uint16_t* __restrict__ w, int64_t N,
                                                                 int64_t K, int64_t ldw,
                                                                 uint32_t* __restrict__ qweight,
                                                                 uint16_t* __restrict__ scales) {
  __shared__ uint16_t s_scales[kTileK / ER_GROUP][kTileRows];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t n0 = (int64_t)blockIdx.y * kTileRows;
  const int64_t k0 = (int64_t)blockIdx.x * kTileK;

  uint4 v[kIters];
  bool ok[kIters];
#pragma unroll
  for (int it = 0; it < kIters; ++it) {
    const int r = warp * 4 + (it >> 1);
    const int64_t n = n0 + r;
    const int64_t k = k0 + (it & 1) * 256 + lane * 8;
    ok[it] = (n < N) && (k < K);
    v[it] = make_uint4(0, 0, 0, 0);
    if (ok[it]) v[it] = ld_stream(reinterpret_cast<const uint4*>(w + n * ldw + k));
  }

#pragma unroll
  for (int it = 0; it < kIters; ++it) {
    const int r = warp * 4 + (it >> 1);
    const uint32_t raw[4] = {v[it].x, v[it].y, v[it].z, v[it].w};
    float f[8];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      f[2 * i] = __uint_as_float(raw[i] << 16);
      f[2 * i + 1] = __uint_as_float(raw[i] & 0xFFFF0000u);
    }
    float amax = 0.0f;
#pragma unroll
    for (int i = 0; i < 8; ++i) amax = fmaxf(amax, fabsf(f[i]));
#pragma unroll
    for (int off = 1; off < 16; off <<= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, off));

    const __nv_bfloat16 sb = __float2bfloat16_rn(__fdiv_rn(amax, 7.0f));
    const float s = __bfloat162float(sb);
    uint32_t word = 0x88888888u;  // all q = 0 (s == 0, Q8)
    if (s > 0.0f) {
      word = 0;
      if (s >= 1e-30f) {
        const float rcp = __frcp_rn(s);
#pragma unroll
        for (int i = 0; i < 8; ++i) word |= code_of(f[i], s, rcp) << (4 * ((i >> 1) + 4 * (i & 1)));
      } else {  // 1/s would overflow: plain IEEE division
#pragma unroll
        for (int i = 0; i < 8; ++i) word |= code_of_div(f[i], s) << (4 * ((i >> 1) + 4 * (i & 1)));
      }
    }
    if (ok[it]) {
      const int64_t n = n0 + r;
      const int64_t k = k0 + (it & 1) * 256 + lane * 8;
      qweight[n * (K >> 3) + (k >> 3)] = word;
    }
    if ((lane & 15) == 0) s_scales[(it & 1) * 2 + (lane >> 4)][r] = (s > 0.0f) ? __bfloat16_as_ushort(sb) : 0;
  }
  __syncthreads();
  if (threadIdx.x < (kTileK / ER_GROUP) * kTileRows) {
    const int g = threadIdx.x >> 5, r = threadIdx.x & 31;
    const int64_t gg = (k0 >> 7) + g, n = n0 + r;
    if (n < N && gg < (K >> 7)) scales[gg * N + n] = s_scales[g][r];
  }
}

__global__ void unpack_codes_kernel(const uint32_t* __restrict__ qweight, int64_t words, int8_t* __restrict__ codes) {
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= words) return;
  const uint32_t wd = qweight[j];
  uint32_t lo = 0, hi = 0;  // 8 int8 codes of logical k = 8 j + 0..7
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    const uint32_t even = ((wd >> (4 * t)) & 0xFu) - 8u;        // k = 2 t
    const uint32_t odd = ((wd >> (4 * t + 16)) & 0xFu) - 8u;    // k = 2 t + 1
    const uint32_t pair = (even & 0xFFu) | ((odd & 0xFFu) << 8);
    if (t < 2) lo |= pair << (16 * t);
    else hi |= pair << (16 * (t - 2));
  }
  reinterpret_cast<uint2*>(codes)[j] = make_uint2(lo, hi);
}

}  // namespace

extern "C" {

int er_quantize_pack(const void* w_bf16, int64_t N, int64_t K, int64_t ldw_elems, int group, void* qweight_out,
                     void* scales_out, void* stream) {
  if (!w_bf16 || !qweight_out || !scales_out) return ER_ERR_NULL;
  if (group != ER_GROUP || N < 1 || K < ER_GROUP || K % ER_GROUP != 0 || ldw_elems < K) return ER_ERR_SHAPE;
  if (!er::aligned16(w_bf16) || !er::aligned16(qweight_out) || (ldw_elems % 8) != 0 ||
      (reinterpret_cast<uintptr_t>(scales_out) & 1u))
    return ER_ERR_ALIGN;
  int st = er::check_arch();
  if (st != ER_OK) return st;
  // grid.x = k tiles (fastest) so that consecutive CTAs stream consecutive bytes of the same rows
  dim3 grid((unsigned)((K + kTileK - 1) / kTileK), (unsigned)((N + kTileRows - 1) / kTileRows));
  if (grid.y > 65535u) return ER_ERR_SHAPE;  // N > 2,097,120 rows: split the call
  quantize_pack_kernel<<<grid, kThreads, 0, (cudaStream_t)stream>>>(
      reinterpret_cast<const uint16_t*>(w_bf16), N, K, ldw_elems, reinterpret_cast<uint32_t*>(qweight_out),
      reinterpret_cast<uint16_t*>(scales_out));
  ER_CUDA_TRY(cudaGetLastError());
  return ER_OK;
}

int er_unpack_codes(const void* qweight, int64_t N, int64_t K, int8_t* codes_out, void* stream) {
  if (!qweight || !codes_out) return ER_ERR_NULL;
  if (N < 1 || K < 8 || K % 8 != 0) return ER_ERR_SHAPE;
  if ((reinterpret_cast<uintptr_t>(qweight) & 3u) || (reinterpret_cast<uintptr_t>(codes_out) & 7u)) return ER_ERR_ALIGN;
  int st = er::check_arch();
  if (st != ER_OK) return st;
  const int64_t words = N * (K >> 3);
  const int64_t blocks = (words + 255) / 256;
  if (blocks > 0x7FFFFFFFll) return ER_ERR_SHAPE;
  unpack_codes_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(reinterpret_cast<const uint32_t*>(qweight),
                                                                         words, codes_out);
  ER_CUDA_TRY(cudaGetLastError());
  return ER_OK;
}

}  // extern "C"
