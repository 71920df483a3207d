// quantize_pack8.cu -- er_quantize_pack8: the W8 variant of the drafter refresh (Table 4 "RTN W8";
// SURVEY.md 8(f) f3).  RTN int8, symmetric, group 128 along K, s = bf16_rne(amax / 127), q = clamp(rint(w / s), -127,
// 127) with IEEE division.  The codes leave as TWO NIBBLE PLANES in the W4 layout (ER_PACK_V2 over 2 K columns): group g
// becomes groups 2g (high nibbles a, scale 16 s) and 2g + 1 (low nibbles b, scale s), q + 128 = 16 a + b -- so the W4
// GEMM kernels contract a W8 matrix as they stand (er_w8a16_gemm).  Same tiling as quantize_pack.cu: a CTA takes 32 rows
// x 512 k, a lane 16 consecutive k (one 256-bit load), 8 lanes a group; 2 B read + 1 B + 4/128 B written per element.
#include <cuda_bf16.h>
#include "er_common.cuh"

namespace {

constexpr int kTileRows = 32;
constexpr int kTileK = 512;
constexpr int kThreads = 256;
constexpr int kIters = 4;  // rows per warp

struct U8 { uint32_t v[8]; };

__device__ __forceinline__ uint32_t absmax2(uint32_t a, uint32_t b) {
  uint32_t d;
  asm("max.xorsign.abs.bf16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
  return d;
}

constexpr float kMagic8 = 12582912.0f + 128.0f;   // 1.5 * 2^23 + 128: bits(t + kMagic8) = 0x4B400000 + rint(t) + 128

// bits whose low byte is the stored code u = clamp(rint(w / s), -127, 127) + 128.  r ~ 1 / s (MUFU.RCP) and one
// exact-residual Newton step, as in quantize_pack.cu: the result is the IEEE quotient wherever that matters -- exact at
// ties (k + 1/2 is representable), and a non-tie quotient of two 8-bit significands with |w / s| >= 1/2 is at least
// 1/1020 away from a tie, against an error of t below 2e-5.  kDiv: plain IEEE division (denormal scales, 1 / s overflows).
template <bool kDiv>
__device__ __forceinline__ uint32_t code8(float w, float s, float r) {
  float t;
  if (kDiv) {
    t = __fdiv_rn(w, s);
  } else {
    t = w * r;
    const float e = __fmaf_rn(-t, s, w);
    t = __fmaf_rn(e, r, t);
  }
  return __float_as_uint(fminf(fmaxf(t, -127.0f), 127.0f) + kMagic8);
}

// The two plane words of 8 consecutive k (4 raw words of bf16 pairs): logical k = 2 t + h sits in nibble t + 4 h.
template <bool kDiv>
__device__ __forceinline__ void planes8(const uint32_t* raw, float s, float r, uint32_t& hi, uint32_t& lo) {
  uint32_t a = 0, b = 0;
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    const uint32_t u0 = code8<kDiv>(__uint_as_float(raw[t] << 16), s, r);
    const uint32_t u1 = code8<kDiv>(__uint_as_float(raw[t] & 0xFFFF0000u), s, r);
    a |= ((u0 >> 4) & 15u) << (4 * t);
    a |= ((u1 >> 4) & 15u) << (4 * t + 16);
    b |= (u0 & 15u) << (4 * t);
    b |= (u1 & 15u) << (4 * t + 16);
  }
  hi = a;
  lo = b;
}

__global__ void __launch_bounds__(kThreads) quantize_pack8_kernel(const uint16_t* __restrict__ w, int64_t N, int64_t K,
                                                                  int64_t ldw, uint32_t* __restrict__ qweight,
                                                                  uint16_t* __restrict__ scales) {
  __shared__ uint16_t s_scales[kTileK / ER_GROUP][kTileRows];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t n0 = (int64_t)blockIdx.y * kTileRows;
  const int64_t k = (int64_t)blockIdx.x * kTileK + lane * 16;

  U8 v[kIters];
  bool ok[kIters];
#pragma unroll
  for (int it = 0; it < kIters; ++it) {
    const int64_t n = n0 + warp * kIters + it;
    ok[it] = (n < N) && (k < K);
#pragma unroll
    for (int i = 0; i < 8; ++i) v[it].v[i] = 0;
    if (ok[it]) {
      const uint4* src = reinterpret_cast<const uint4*>(w + n * ldw + k);
      const uint4 a = __ldg(src), b = __ldg(src + 1);
      v[it].v[0] = a.x; v[it].v[1] = a.y; v[it].v[2] = a.z; v[it].v[3] = a.w;
      v[it].v[4] = b.x; v[it].v[5] = b.y; v[it].v[6] = b.z; v[it].v[7] = b.w;
    }
  }

#pragma unroll
  for (int it = 0; it < kIters; ++it) {
    const int r_in_tile = warp * kIters + it;
    const uint32_t* raw = v[it].v;
    uint32_t m2 = absmax2(absmax2(absmax2(raw[0], raw[1]), absmax2(raw[2], raw[3])),
                          absmax2(absmax2(raw[4], raw[5]), absmax2(raw[6], raw[7])));
#pragma unroll
    for (int off = 1; off < 8; off <<= 1) m2 = absmax2(m2, __shfl_xor_sync(0xffffffffu, m2, off));
    const float amax = fmaxf(fabsf(__uint_as_float(m2 << 16)), fabsf(__uint_as_float(m2 & 0xFFFF0000u)));
    const __nv_bfloat16 sb = __float2bfloat16_rn(__fdiv_rn(amax, 127.0f));
    const float s = __bfloat162float(sb);
    // plane words: the 8 codes of a word sit at nibble t + 4 h for logical k = 2 t + h (as in the W4 layout)
    uint32_t hi[2] = {0x88888888u, 0x88888888u}, lo[2] = {0u, 0u};    // s == 0: q = 0 -> u = 128 = (8, 0)
    if (s >= 1e-30f) {
      float r;
      asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(s));
      planes8<false>(raw, s, r, hi[0], lo[0]);
      planes8<false>(raw + 4, s, r, hi[1], lo[1]);
    } else if (s > 0.0f) {
      planes8<true>(raw, s, 0.f, hi[0], lo[0]);
      planes8<true>(raw + 4, s, 0.f, hi[1], lo[1]);
    }
    if (ok[it]) {
      const int64_t n = n0 + r_in_tile;
      const int64_t g = k >> 7, kin = k & 127;                 // k is a multiple of 16: an aligned pair of words
      const int64_t ka = (2 * g) * ER_GROUP + kin;             // column of the two-plane matrix (2 K columns)
      *reinterpret_cast<uint2*>(qweight + er::packed_word_index(n, ka >> 3, K >> 6)) = make_uint2(hi[0], hi[1]);
      *reinterpret_cast<uint2*>(qweight + er::packed_word_index(n, (ka + ER_GROUP) >> 3, K >> 6)) = make_uint2(lo[0], lo[1]);
    }
    if ((lane & 7) == 0) s_scales[lane >> 3][r_in_tile] = (s > 0.0f) ? __bfloat16_as_ushort(sb) : 0;
  }
  __syncthreads();
  if (threadIdx.x < (kTileK / ER_GROUP) * kTileRows) {
    const int g = threadIdx.x >> 5, r = threadIdx.x & 31;
    const int64_t gg = ((int64_t)blockIdx.x * kTileK >> 7) + g, n = n0 + r;
    if (n < N && gg < (K >> 7)) {
      const uint16_t sb = s_scales[g][r];
      const float s16 = __bfloat162float(__ushort_as_bfloat16(sb)) * 16.0f;     // exact unless it overflows
      scales[(2 * gg) * N + n] = __bfloat16_as_ushort(__float2bfloat16_rn(s16));
      scales[(2 * gg + 1) * N + n] = sb;
    }
  }
}

}  // namespace

extern "C" int er_quantize_pack8(const void* w_bf16, int64_t N, int64_t K, int64_t ldw_elems, int group,
                                 void* qweight_out, void* scales_out, void* stream) {
  if (!w_bf16 || !qweight_out || !scales_out) return ER_ERR_NULL;
  if (group != ER_GROUP || N < 128 || N % 128 != 0 || K < ER_GROUP || K % ER_GROUP != 0 || ldw_elems < K)
    return ER_ERR_SHAPE;
  if (!er::aligned16(w_bf16) || !er::aligned16(qweight_out) || (ldw_elems % 8) != 0 ||
      (reinterpret_cast<uintptr_t>(scales_out) & 1u))
    return ER_ERR_ALIGN;
  int st = er::check_arch();
  if (st != ER_OK) return st;
  dim3 grid((unsigned)((K + kTileK - 1) / kTileK), (unsigned)((N + kTileRows - 1) / kTileRows));
  if (grid.y > 65535u) return ER_ERR_SHAPE;
  quantize_pack8_kernel<<<grid, kThreads, 0, (cudaStream_t)stream>>>(
      reinterpret_cast<const uint16_t*>(w_bf16), N, K, ldw_elems, reinterpret_cast<uint32_t*>(qweight_out),
      reinterpret_cast<uint16_t*>(scales_out));
  ER_CUDA_TRY(cudaGetLastError());
  return ER_OK;
}
