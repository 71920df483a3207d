// quantize_pack.cu -- er_quantize_pack: the per-RL-step drafter refresh ("lightweight RTN
// quantization to the FFN and QKVO projection layers", L150 Alg. 1 line 3) and er_unpack_codes.
//
// HBM-bound streaming kernel: 2 B read + 0.5 B + 2/128 B written per element.  The first
// version was instruction-bound (ncu: issue 75 %, DRAM 35 %), so the arithmetic is cut to ~7 instructions per
// element:
//   - a lane owns 16 consecutive k (ONE 256-bit load, two packed words out); 8 lanes cover a 128-element group,
//     so the group max is 3 shuffle-xor steps, taken on packed bf16x2 |w| (half the compares);
//   - scale s = bf16_rne(amax * (1/7)): identical to the IEEE division for every bf16 amax (Q4: a/7 is
//     never within 2^-12 relative of a bf16 rounding boundary);
//   - q = rint(w / s) with IEEE-division semantics AT TIES (Q6): t = w * r with r ~ 1/s (MUFU.RCP),
//     one exact-residual Newton step (returns k + 1/2 exactly whenever w / s is exactly k + 1/2; every non-tie
//     quotient of two 8-bit significands is >= 1/1020 from a tie, far above the 1e-6 error of t);
//   - rounding + offset in one FADD: bits(t + (1.5 * 2^23 + 8)) = 0x4B400000 + (q + 8), RNE on the integer grid;
//   - nibble placement by integer multiply-add of those bits (the constant upper bits are removed once per word).
// A CTA quantizes a tile of 32 rows x 512 k; a warp takes 4 rows, all 4 loads issued before any arithmetic.  The
// 4 x 32 scales of the tile are transposed through shared memory so that they leave as 64-byte runs along N.
#include <cuda_bf16.h>
#include "er_common.cuh"

namespace {

constexpr int kTileRows = 32;
constexpr int kTileK = 512;
constexpr int kThreads = 256;
constexpr int kIters = 4;  // rows per warp

struct U8 { uint32_t v[8]; };

__device__ __forceinline__ U8 ld_stream256(const void* p) {
  U8 r;
  asm volatile("ld.global.nc.L1::no_allocate.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(r.v[0]), "=r"(r.v[1]), "=r"(r.v[2]), "=r"(r.v[3]), "=r"(r.v[4]), "=r"(r.v[5]), "=r"(r.v[6]),
                 "=r"(r.v[7])
               : "l"(p));
  return r;
}
__device__ __forceinline__ uint4 ld_stream128(const void* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}

// packed bf16x2 max(|a|, |b|) in ONE instruction; the result's sign bits are xor-of-signs garbage, which the
// next absmax2 (or the final mask) discards.
__device__ __forceinline__ uint32_t absmax2(uint32_t a, uint32_t b) {
  uint32_t d;
  asm("max.xorsign.abs.bf16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
  return d;
}

constexpr float kMagic = 12582912.0f + 8.0f;  // 1.5 * 2^23 + 8: bits(t + kMagic) = 0x4B400000 + rint(t) + 8

// bits whose low nibble is the stored code u = rint(w / s) + 8 (upper 28 bits = 0x4B40000)
__device__ __forceinline__ uint32_t code_bits(float w, float s, float r) {
  float t = w * r;
  const float e = __fmaf_rn(-t, s, w);
  t = __fmaf_rn(e, r, t);
  return __float_as_uint(t + kMagic);
}
__device__ __forceinline__ uint32_t code_bits_div(float w, float s) {  // denormal scales: plain IEEE division
  // a bf16 scale below 2^-126 has fewer than 8 significant bits, so amax / s can reach 8 (e.g. amax = 8 ulp, s = 1 ulp):
  // the clamp of DESIGN.md Q7 is needed here, and only here (rint(clamp(t)) == clamp(rint(t)) for these bounds)
  return __float_as_uint(fminf(fmaxf(__fdiv_rn(w, s), -8.0f), 7.0f) + kMagic);
}

// Packs the 8 codes of 4 raw words (k = 0..7 of the word) into one packed word (ER_PACK_V2 keeps this intra-word order): logical k = 2 t + h sits in
// nibble t + 4 h.  `sum of (0x4B400000 << 4 i)` over i = 0..7 (mod 2^32) is the constant removed at the end.
template <bool kDiv>
__device__ __forceinline__ uint32_t pack8(const uint32_t* raw, float s, float r) {
  uint32_t acc = 0;
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    const float lo = __uint_as_float(raw[t] << 16);
    const float hi = __uint_as_float(raw[t] & 0xFFFF0000u);
    const uint32_t bl = kDiv ? code_bits_div(lo, s) : code_bits(lo, s, r);
    const uint32_t bh = kDiv ? code_bits_div(hi, s) : code_bits(hi, s, r);
    acc += bl << (4 * t);
    acc += bh << (4 * t + 16);
  }
  constexpr uint32_t kConst = 0x4B400000u * 0x11111111u;  // sum_i 0x4B400000 << 4 i  (mod 2^32)
  return acc - kConst;
}

// cold path (denormal scale: 1/s would overflow), kept out of line; reloads its 16 elements so that the hot
// path's registers never need an address
__device__ __noinline__ uint2 pack16_div(const uint16_t* src, float s) {
  const uint4 a = *reinterpret_cast<const uint4*>(src), b = *reinterpret_cast<const uint4*>(src + 8);
  const uint32_t r0[4] = {a.x, a.y, a.z, a.w}, r1[4] = {b.x, b.y, b.z, b.w};
  return make_uint2(pack8<true>(r0, s, 0.f), pack8<true>(r1, s, 0.f));
}

// One CTA quantizes the tile (bx: 512-k tile, by: 32-row tile) of one weight matrix.
__device__ __forceinline__ void quantize_tile(const uint16_t* __restrict__ w, int64_t N, int64_t K, int64_t ldw,
                                              uint32_t* __restrict__ qweight, uint16_t* __restrict__ scales,
                                              int vec256, unsigned bx, unsigned by) {
  __shared__ uint16_t s_scales[kTileK / ER_GROUP][kTileRows];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t n0 = (int64_t)by * kTileRows;
  const int64_t k = (int64_t)bx * kTileK + lane * 16;

  U8 v[kIters];
  bool ok[kIters];
#pragma unroll
  for (int it = 0; it < kIters; ++it) {
    const int64_t n = n0 + warp * kIters + it;
    ok[it] = (n < N) && (k < K);
#pragma unroll
    for (int i = 0; i < 8; ++i) v[it].v[i] = 0;
    if (ok[it]) {
      const uint16_t* src = w + n * ldw + k;
      if (vec256) {
        v[it] = ld_stream256(src);
      } else {  // rows only 16-byte aligned
        const uint4 a = ld_stream128(src), b = ld_stream128(src + 8);
        v[it].v[0] = a.x; v[it].v[1] = a.y; v[it].v[2] = a.z; v[it].v[3] = a.w;
        v[it].v[4] = b.x; v[it].v[5] = b.y; v[it].v[6] = b.z; v[it].v[7] = b.w;
      }
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
    const __nv_bfloat16 sb = __float2bfloat16_rn(amax * 0.142857149f);
    const float s = __bfloat162float(sb);
    uint32_t w0, w1;
    if (s >= 1e-30f) {
      float r;
      asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(s));
      w0 = pack8<false>(raw, s, r);
      w1 = pack8<false>(raw + 4, s, r);
    } else if (s > 0.0f) {
      const uint2 pd = pack16_div(w + (n0 + r_in_tile) * ldw + k, s);
      w0 = pd.x; w1 = pd.y;
    } else {
      w0 = w1 = 0x88888888u;  // all q = 0 (s == 0, Q8)
    }
    if (ok[it]) {
      const int64_t n = n0 + r_in_tile;
      // k is a multiple of 16: the two words are an aligned pair inside one 16-byte chunk of the block row
      *reinterpret_cast<uint2*>(qweight + er::packed_word_index(n, k >> 3, K >> 7)) = make_uint2(w0, w1);
    }
    if ((lane & 7) == 0) s_scales[lane >> 3][r_in_tile] = (s > 0.0f) ? __bfloat16_as_ushort(sb) : 0;
  }
  __syncthreads();
  if (threadIdx.x < (kTileK / ER_GROUP) * kTileRows) {
    const int g = threadIdx.x >> 5, r = threadIdx.x & 31;
    const int64_t gg = ((int64_t)bx * kTileK >> 7) + g, n = n0 + r;
    if (n < N && gg < (K >> 7)) scales[gg * N + n] = s_scales[g][r];
  }
}

__global__ void __launch_bounds__(kThreads) quantize_pack_kernel(const uint16_t* __restrict__ w, int64_t N,
                                                                 int64_t K, int64_t ldw,
                                                                 uint32_t* __restrict__ qweight,
                                                                 uint16_t* __restrict__ scales, int vec256) {
  quantize_tile(w, N, K, ldw, qweight, scales, vec256, blockIdx.x, blockIdx.y);
}

// Several weight matrices in one launch (the refresh of a whole decoder layer / model): a 1-D grid over the tiles of
// all of them, so that the tails of the small matrices overlap with the large ones instead of each paying its own
// launch and drain.
constexpr int kMaxBatch = 8;
struct BatchParams {
  const uint16_t* w[kMaxBatch];
  uint32_t* qweight[kMaxBatch];
  uint16_t* scales[kMaxBatch];
  int64_t N[kMaxBatch], K[kMaxBatch], ldw[kMaxBatch];
  unsigned kt[kMaxBatch];          // 512-k tiles per row tile
  unsigned first[kMaxBatch + 1];   // first CTA of every matrix
  int vec256[kMaxBatch];
  int count;
};
__global__ void __launch_bounds__(kThreads) quantize_pack_batched_kernel(const __grid_constant__ BatchParams bp) {
  int t = 0;
  while (t + 1 < bp.count && blockIdx.x >= bp.first[t + 1]) ++t;
  const unsigned local = blockIdx.x - bp.first[t];
  // k tiles fastest, as in the single-matrix grid: consecutive CTAs stream consecutive bytes of the same rows
  quantize_tile(bp.w[t], bp.N[t], bp.K[t], bp.ldw[t], bp.qweight[t], bp.scales[t], bp.vec256[t], local % bp.kt[t],
                local / bp.kt[t]);
}

__global__ void unpack_codes_kernel(const uint32_t* __restrict__ qweight, int64_t words, int64_t K,
                                    int8_t* __restrict__ codes) {
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;  // logical word: row n = j / (K/8), octet jj
  if (j >= words) return;
  const int64_t n = j / (K >> 3), jj = j % (K >> 3);
  const uint32_t wd = qweight[er::packed_word_index(n, jj, K >> 7)];
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
  if (group != ER_GROUP || N < 128 || N % 128 != 0 || K < ER_GROUP || K % ER_GROUP != 0 || ldw_elems < K)
    return ER_ERR_SHAPE;
  if (!er::aligned16(w_bf16) || !er::aligned16(qweight_out) || (ldw_elems % 8) != 0 ||
      (reinterpret_cast<uintptr_t>(scales_out) & 1u))
    return ER_ERR_ALIGN;
  int st = er::check_arch();
  if (st != ER_OK) return st;
  // grid.x = k tiles (fastest) so that consecutive CTAs stream consecutive bytes of the same rows
  dim3 grid((unsigned)((K + kTileK - 1) / kTileK), (unsigned)((N + kTileRows - 1) / kTileRows));
  if (grid.y > 65535u) return ER_ERR_SHAPE;  // N > 2,097,120 rows: split the call
  const int vec256 = ((reinterpret_cast<uintptr_t>(w_bf16) & 31u) == 0 && (ldw_elems % 16) == 0) ? 1 : 0;
  quantize_pack_kernel<<<grid, kThreads, 0, (cudaStream_t)stream>>>(
      reinterpret_cast<const uint16_t*>(w_bf16), N, K, ldw_elems, reinterpret_cast<uint32_t*>(qweight_out),
      reinterpret_cast<uint16_t*>(scales_out), vec256);
  ER_CUDA_TRY(cudaGetLastError());
  return ER_OK;
}

int er_quantize_pack_batched(const er_linear_desc* descs, int count, int group, void* stream) {
  if (count < 0) return ER_ERR_SHAPE;
  if (count == 0) return ER_OK;
  if (!descs) return ER_ERR_NULL;
  for (int i = 0; i < count; ++i) {           // validate everything before anything is launched
    const er_linear_desc& d = descs[i];
    if (!d.w || !d.qweight || !d.scales) return ER_ERR_NULL;
    if (group != ER_GROUP || d.N < 128 || d.N % 128 != 0 || d.K < ER_GROUP || d.K % ER_GROUP != 0 || d.ldw < d.K)
      return ER_ERR_SHAPE;
    if ((d.N + kTileRows - 1) / kTileRows > 65535) return ER_ERR_SHAPE;
    if (!er::aligned16(d.w) || !er::aligned16(d.qweight) || (d.ldw % 8) != 0 ||
        (reinterpret_cast<uintptr_t>(d.scales) & 1u))
      return ER_ERR_ALIGN;
  }
  int st = er::check_arch();
  if (st != ER_OK) return st;
  for (int base = 0; base < count; base += kMaxBatch) {
    BatchParams bp;
    bp.count = count - base < kMaxBatch ? count - base : kMaxBatch;
    unsigned long long total = 0;
    for (int i = 0; i < bp.count; ++i) {
      const er_linear_desc& d = descs[base + i];
      bp.w[i] = reinterpret_cast<const uint16_t*>(d.w);
      bp.qweight[i] = reinterpret_cast<uint32_t*>(d.qweight);
      bp.scales[i] = reinterpret_cast<uint16_t*>(d.scales);
      bp.N[i] = d.N; bp.K[i] = d.K; bp.ldw[i] = d.ldw;
      bp.kt[i] = (unsigned)((d.K + kTileK - 1) / kTileK);
      bp.vec256[i] = ((reinterpret_cast<uintptr_t>(d.w) & 31u) == 0 && (d.ldw % 16) == 0) ? 1 : 0;
      bp.first[i] = (unsigned)total;
      total += (unsigned long long)bp.kt[i] * (unsigned long long)((d.N + kTileRows - 1) / kTileRows);
      if (total > 0x7FFFFFFFull) return ER_ERR_SHAPE;
    }
    for (int i = bp.count; i <= kMaxBatch; ++i) bp.first[i] = (unsigned)total;
    quantize_pack_batched_kernel<<<(unsigned)total, kThreads, 0, (cudaStream_t)stream>>>(bp);
    ER_CUDA_TRY(cudaGetLastError());
  }
  return ER_OK;
}

int er_unpack_codes(const void* qweight, int64_t N, int64_t K, int8_t* codes_out, void* stream) {
  if (!qweight || !codes_out) return ER_ERR_NULL;
  if (N < 128 || N % 128 != 0 || K < ER_GROUP || K % ER_GROUP != 0) return ER_ERR_SHAPE;
  if ((reinterpret_cast<uintptr_t>(qweight) & 3u) || (reinterpret_cast<uintptr_t>(codes_out) & 7u)) return ER_ERR_ALIGN;
  int st = er::check_arch();
  if (st != ER_OK) return st;
  const int64_t words = N * (K >> 3);
  const int64_t blocks = (words + 255) / 256;
  if (blocks > 0x7FFFFFFFll) return ER_ERR_SHAPE;
  unpack_codes_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(reinterpret_cast<const uint32_t*>(qweight),
                                                                         words, K, codes_out);
  ER_CUDA_TRY(cudaGetLastError());
  return ER_OK;
}

}  // extern "C"
