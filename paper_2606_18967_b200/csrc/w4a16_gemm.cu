// w4a16_gemm.cu -- er_w4a16_gemm: the weight-quantized self-drafter's linear, Y = X . dequant(Wq)^T
// (dense projections are ~90 % of tail decode latency and weight loading dominates at
// small batch; L175: W4A16 weight-only kernel; L467: "on-the-fly dequantization and kernel-level overhead").
//
// sm_100a design, third version.  The first two were bound by one long
// wait -> convert -> MMA -> read-back chain per warp and by single-thread issue loops whose TMA / MMA
// operands the compiler could not prove warp-uniform (profiles/r01_*): here every role is its own warp(s),
// the chains only meet at mbarriers, and the issuing warps run warp-uniform code with one elected lane.
//
//   persistent   one CTA per SM; the (tile, 128-k group) units of the whole problem are dealt out as ONE
//                contiguous range per CTA ("stream-K"): every CTA streams the same number of bytes.
//   swap-AB      the 128 weight rows of a tile are the M = 128 of tcgen05.mma, the padded batch is its N.
//   warp 0       producer: per group ONE 8 KiB 1-D bulk copy of the packed block (ER_PACK_V2 keeps every
//                [128 rows x 128 k] block contiguous and pre-swizzled), one 256-byte bulk copy of the group's
//                scales and two SWIZZLE_128B TMA boxes of X [MPAD x 64 k], into a ring of up to 16 stages.
//   warp 1       MMA issuer: tcgen05.mma.kind::f16, A (weights) from TENSOR MEMORY, B (= X tile) from shared
//                memory, a fresh fp32 TMEM accumulator per group so the group scale is applied exactly.
//   warps 4-19   converters, two sets of 8 (even / odd groups).  A thread owns HALF a weight row of the
//                group: 2 x LDS.128, nibble -> 16-bit float with the magic-number trick, tcgen05.st into the
//                A buffer (the 4x expanded weights never touch shared memory).
//   warps 20-27  scale-accumulate: tcgen05.ld of the group's accumulator, acc += scale * d in fp32 registers,
//                and the output: a tile wholly owned by one CTA is stored directly, otherwise fp32 partials go
//                to the workspace and the last CTA of the tile (ticket counter) adds them in ascending CTA
//                order.  Deterministic, no float atomics.
//   TMEM         4 A buffers (64 columns each) and 8 (MPAD = 64: 4) accumulators cycle independently: an A
//                buffer is refilled once the MMAs that read it completed, an accumulator once it was drained.
//   barriers     full[stage] (TMA landed), done[stage] (ONE tcgen05.commit per group: accumulator readable, A
//                buffer and shared-memory stage reusable), a_full[A buffer], d_free[accumulator].  One warp per
//                role polls (tight test_wait) and releases its peers through a named barrier.
#include <cuda.h>
#include "er_common.cuh"

namespace {

using namespace er;

constexpr int kTileN = 128;                 // weight rows per tile
constexpr int kWBytes = kTileN * 64;        // 8 KiB packed weights per group stage
constexpr int kScaleBytes = kTileN * 2;     // 128 bf16 scales
constexpr int kCvtWarp0 = 4, kCvtWarps = 16;    // converter warps 4..19
constexpr int kEpiWarp0 = 20, kEpiWarps = 8;    // scale-accumulate warps 20..27
constexpr int kThreads = (kEpiWarp0 + kEpiWarps) * 32;   // 896
constexpr int kMaxStages = 16;
constexpr int kNA = 4;                      // A-operand buffers in TMEM
constexpr int kTmemCols = 512;
constexpr int kTmemA = 0;                   // A operand: kNA buffers x 64 columns
constexpr int kTmemD = 256;                 // accumulators: kND buffers x MPAD columns
constexpr int kSmemLimit = 227 * 1024;

template <int MPAD>
struct Cfg {
  static constexpr int kXBytes = MPAD * 128 * 2;           // two boxes of [MPAD x 64] bf16
  static constexpr int kStageBytes = ((kWBytes + kXBytes + kScaleBytes + 1023) / 1024) * 1024;
  static constexpr int kND = MPAD <= 32 ? 8 : 4;           // accumulator buffers in TMEM (kND * MPAD <= 256 columns)
  static constexpr int kScBufBytes = kMaxStages * kTileN * 4;   // fp32 scales of the groups in flight, by stage
  static constexpr int kFixed = kScBufBytes + 1024 /*align slack*/ + 512 /*barriers*/;
  static constexpr int kStagesRaw = (kSmemLimit - kFixed) / kStageBytes;
  static constexpr int kStages = kStagesRaw > kMaxStages ? kMaxStages : kStagesRaw;
  static constexpr int kSmem = kStages * kStageBytes + kFixed;
  static constexpr uint32_t kTxBytes = kWBytes + kXBytes + kScaleBytes;
  static constexpr int kCW = MPAD / 2;                     // accumulator columns per scale-accumulate warp
};

struct GemmParams {
  int M, N, K;
  int G;               // groups per tile = K / 128
  int ntiles;          // N / 128
  int tiles;           // ntiles * mchunks
  int unit_groups;     // groups per scheduling unit: 1 (stream-K) or G (whole tiles)
  long long units;     // tiles * G / unit_groups
  int y_f32;
  int64_t ldy;
  void* y;
  const uint8_t* qweight;  // ER_PACK_V2 blocks
  const uint8_t* scales;   // bf16 [G][N]
  float* partials;     // workspace + ER_GEMM_COUNTER_BYTES: [cta][2][MPAD][128]
  int* counters;       // workspace: one ticket per tile
  int dbg;             // debug/sweep flags (er_gemm_tuning key 2); 0 in production
#ifdef ER_GEMM_TRACE
  unsigned long long* trace;
  int dbg_cta;
#endif
};

// Optional in-kernel timeline (development builds only, -DER_GEMM_TRACE): lane 0 of every warp of CTA 0 logs
// (event id, clock) pairs.
#ifdef ER_GEMM_TRACE
// section timer: ER_TR(k) adds the cycles since the previous ER_TR of this warp to bucket k (k < 8)
#define ER_TR(id)                                   \
  do {                                              \
    const unsigned tr_now = (unsigned)clock();      \
    if ((id) < 8) tr_sum[(id)] += tr_now - tr_prev; \
    tr_prev = tr_now;                               \
  } while (0)
#else
#define ER_TR(id) do {} while (0)
#endif

#define ER_TMEM_ST16(taddr, r, o)                                                                              \
  asm volatile(                                                                                                \
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" \
      ::"r"(taddr), "r"(r[o + 0]), "r"(r[o + 1]), "r"(r[o + 2]), "r"(r[o + 3]), "r"(r[o + 4]), "r"(r[o + 5]),   \
      "r"(r[o + 6]), "r"(r[o + 7]), "r"(r[o + 8]), "r"(r[o + 9]), "r"(r[o + 10]), "r"(r[o + 11]),              \
      "r"(r[o + 12]), "r"(r[o + 13]), "r"(r[o + 14]), "r"(r[o + 15])                                           \
      : "memory")

#define ER_TMEM_LD16(taddr, r, o)                                                                              \
  asm volatile(                                                                                                \
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];" \
      : "=r"(r[o + 0]), "=r"(r[o + 1]), "=r"(r[o + 2]), "=r"(r[o + 3]), "=r"(r[o + 4]), "=r"(r[o + 5]),        \
        "=r"(r[o + 6]), "=r"(r[o + 7]), "=r"(r[o + 8]), "=r"(r[o + 9]), "=r"(r[o + 10]), "=r"(r[o + 11]),      \
        "=r"(r[o + 12]), "=r"(r[o + 13]), "=r"(r[o + 14]), "=r"(r[o + 15])                                     \
      : "r"(taddr)                                                                                             \
      : "memory")

#define ER_TMEM_LD8(taddr, r, o)                                                                 \
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"           \
               : "=r"(r[o + 0]), "=r"(r[o + 1]), "=r"(r[o + 2]), "=r"(r[o + 3]), "=r"(r[o + 4]), \
                 "=r"(r[o + 5]), "=r"(r[o + 6]), "=r"(r[o + 7])                                  \
               : "r"(taddr)                                                                      \
               : "memory")

__device__ __forceinline__ uint32_t lop3_and_or(uint32_t a, uint32_t mask, uint32_t orv) {
  uint32_t d;
  asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(d) : "r"(a), "r"(mask), "r"(orv));
  return d;
}

// One packed word (8 codes; nibble positions (t, t + 4) hold the consecutive pair k = 2t, 2t + 1) -> 4 registers
// of bf16 pairs holding q = u - 8 exactly: (w >> 4t) & 0x000F000F | 0x43004300 is the pair (128 + u, 128 + u'),
// one packed fma (x * 1 - 136, on the FMA pipe) removes the offset.  7 logic-pipe + 4 FMA-pipe ops per word.
// (An fp16 A operand would need 5 logic ops, but tcgen05.mma.kind::f16 faults on fp16 A x bf16 B.)
__device__ __forceinline__ void dequant_word(uint32_t w, uint32_t* a) {
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    const uint32_t v = lop3_and_or(w >> (4 * t), 0x000F000Fu, 0x43004300u);
    asm("fma.rn.bf16x2 %0, %1, %2, %3;" : "=r"(a[t]) : "r"(v), "r"(0x3F803F80u), "r"(0xC308C308u));
  }
}

__device__ __forceinline__ uint4 lds128(uint32_t saddr) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(saddr));
  return v;
}
__device__ __forceinline__ uint32_t lds_u16(uint32_t saddr) {
  uint32_t v;
  asm volatile("ld.shared.u16 %0, [%1];" : "=r"(v) : "r"(saddr));
  return v;
}
__device__ __forceinline__ float lds_f32(uint32_t saddr) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(saddr));
  return v;
}
__device__ __forceinline__ void sts_f32(uint32_t saddr, float v) {
  asm volatile("st.shared.f32 [%0], %1;" ::"r"(saddr), "f"(v) : "memory");
}

__device__ __forceinline__ void named_bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// first unit of CTA c when `units` units are dealt to `P` CTAs as contiguous, balanced ranges
__device__ __forceinline__ long long range_begin(long long units, int P, int c) { return (units * c) / P; }
// the CTA whose range contains unit u
__device__ __forceinline__ int owner_of(long long units, int P, long long u) {
  int c = (int)((u * P) / units);
  while (c + 1 < P && range_begin(units, P, c + 1) <= u) ++c;
  while (c > 0 && range_begin(units, P, c) > u) --c;
  return c;
}

template <int MPAD>
__global__ void __launch_bounds__(kThreads, 1)
w4a16_gemm_kernel(const __grid_constant__ CUtensorMap map_x, const GemmParams p) {
  using C = Cfg<MPAD>;
  constexpr int S = C::kStages;
  constexpr int ND = C::kND;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  float* sc_buf = reinterpret_cast<float*>(smem + S * C::kStageBytes);          // [S][128]
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + S * C::kStageBytes + C::kScBufBytes);
  uint64_t* full = bars;                        // [S]   TMA landed
  uint64_t* done = bars + kMaxStages;           // [S]   the group's MMAs have completed: accumulator readable,
                                                //       A buffer and shared-memory stage reusable
  uint64_t* a_full = bars + 2 * kMaxStages;     // [kNA] A operand (and scales) of a group written
  uint64_t* d_free = a_full + kNA;              // [ND]  accumulator drained
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(d_free + 8);
  int* last_flag = reinterpret_cast<int*>(tmem_slot + 1);

  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);   // provably warp-uniform
  const int lane = threadIdx.x & 31;
  const int P = gridDim.x, cta = blockIdx.x;
  const int ug = p.unit_groups;
  const long long gb = range_begin(p.units, P, cta) * ug;        // first global group index of this CTA
  const long long ge = range_begin(p.units, P, cta + 1) * ug;
  const int n_it = (int)(ge - gb);
#ifdef ER_GEMM_TRACE
  unsigned tr_sum[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  unsigned tr_prev = (unsigned)clock();
#endif

  if (warp == 0) {
    if (lane < S) {
      mbar_init(&full[lane], 1);
      mbar_init(&done[lane], 1);
    }
    if (lane < kNA) mbar_init(&a_full[lane], 8);
    if (lane < ND) mbar_init(&d_free[lane], kEpiWarps);
    mbar_fence_init();
    if (lane == 0) tma_prefetch_desc(&map_x);
  }
  if (warp == 1) tmem_alloc<kTmemCols>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = __shfl_sync(0xffffffffu, *tmem_slot, 0);
  ER_TR(0);

  if (warp == 0) {
    // ===================== producer (warp-uniform; one elected lane issues) =====================
    const int tile0 = (int)(gb / p.G);
    int g = (int)(gb % p.G), tn = tile0 % p.ntiles, mc = tile0 / p.ntiles;
    int s = 0;
    uint32_t ph = 0;
    for (int it = 0; it < n_it; ++it) {
      mbar_spin(&done[s], ph ^ 1);      // the stage's previous group (it - S) has been contracted
      ER_TR(1);
      if (elect_one()) {
        uint8_t* st = smem + s * C::kStageBytes;
        mbar_arrive_expect_tx(&full[s], C::kTxBytes);
        // ER_PACK_V2: the [128 rows x 128 k] block of (tile, g) is 8 KiB of contiguous, pre-swizzled bytes
        bulk_load_1d(st, p.qweight + ((size_t)tn * p.G + g) * kWBytes, kWBytes, &full[s], kEvictFirst);
        tma_load_2d(st + kWBytes, &map_x, &full[s], g * 128, mc * MPAD, kEvictLast);
        tma_load_2d(st + kWBytes + MPAD * 128, &map_x, &full[s], g * 128 + 64, mc * MPAD, kEvictLast);
        bulk_load_1d(st + kWBytes + C::kXBytes, p.scales + ((size_t)g * p.N + tn * kTileN) * 2, kScaleBytes,
                     &full[s], kEvictFirst);
      }
      __syncwarp();
      ER_TR(2);
      if (++g == p.G) {
        g = 0;
        if (++tn == p.ntiles) { tn = 0; ++mc; }
      }
      if (++s == S) { s = 0; ph ^= 1; }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (warp-uniform; one elected lane issues) =====================
    constexpr uint32_t idesc = idesc_bf16_m128(MPAD);
    int s = 0;
    for (int it = 0; it < n_it; ++it) {
      const int ia = it & (kNA - 1), id = it & (ND - 1);
      if (p.dbg & 64) {
        mbar_spin(&full[s], (it / S) & 1);
        if (elect_one()) mbar_arrive(&done[s]);
      } else {
        mbar_spin(&a_full[ia], (it / kNA) & 1);          // implies full[s]: the converters waited for it
        mbar_spin(&d_free[id], ((it / ND) & 1) ^ 1);     // accumulator of group it - ND drained
        ER_TR(1);
        tc_fence_after();
        if (elect_one()) {
          const uint32_t xbase = smem_u32(smem + s * C::kStageBytes + kWBytes);
          const uint32_t d_t = tmem + kTmemD + id * MPAD;
          const uint32_t a_t = tmem + kTmemA + ia * 64;
#pragma unroll
          for (int kk = 0; kk < 8; ++kk) {
            const uint64_t bdesc = smem_desc_sw128(xbase + (kk >> 2) * (MPAD * 128) + (kk & 3) * 32);
            mma_ts_f16((p.dbg & 256) ? (tmem + kTmemD + 128 + kk * 16) : d_t, a_t + kk * 8, bdesc, idesc, kk > 0 ? 1u : 0u);
          }
          tc_commit(&done[s]);
        }
      }
      __syncwarp();
      ER_TR(2);
      if (++s == S) s = 0;
    }
  } else if (warp >= kCvtWarp0 && warp < kCvtWarp0 + kCvtWarps) {
    // ===================== converters: packed int4 -> bf16 A operand in TMEM =====================
    const int dw = warp - kCvtWarp0;
    const int set = dw >> 3;               // 0: even groups of the range, 1: odd groups
    const int half = (dw >> 2) & 1;        // which 64 k of the group's 128 this thread converts
    const int q4 = warp & 3;               // TMEM lane quarter this warp may access
    const int row = q4 * 32 + lane;        // weight row inside the tile
    const uint32_t lane_addr = (uint32_t)(q4 * 32) << 16;
    const int sw = (row >> 1) & 3;
    const uint32_t smem_s = smem_u32(smem);
    const uint32_t row_off0 = row * 64 + (((2 * half) ^ sw) << 4), row_off1 = row * 64 + (((2 * half + 1) ^ sw) << 4);
    const uint32_t sc_s = smem_u32(sc_buf) + row * 4;
    const bool poller = ((dw & 7) == 0);   // one warp of the set polls the mbarriers, a named barrier releases the
                                           // other seven (a blocked bar.sync costs no issue slots, a poll loop does)
    int s = set;                           // stage of group `it`
    uint32_t ph = 0;
    int sp = set + S - kNA;                // stage of group it - kNA (whose MMAs read this A buffer last)
    uint32_t php = 1;                      // ... and the parity of that use; starts "one lap behind"
    if (sp >= S) { sp -= S; php = 0; }
    for (int it = set; it < n_it; it += 2) {
      const int ia = it & (kNA - 1);
      ER_TR(4);
      if (poller) {
        mbar_spin(&full[s], ph);
        if (it >= kNA && !(p.dbg & 64)) mbar_spin(&done[sp], php);
      }
      named_bar_sync(1 + set, 256);
      ER_TR(1);
      if (p.dbg & 64) {
        // streaming-only mode: nothing is converted
      } else {
        tc_fence_after();
        const uint32_t st = smem_s + s * C::kStageBytes;
        const uint4 pk0 = lds128(st + row_off0);
        const uint4 pk1 = lds128(st + row_off1);
        uint32_t sc16 = 0;
        if (half == 0) sc16 = lds_u16(st + kWBytes + C::kXBytes + row * 2);
        uint32_t a[32];
        dequant_word(pk0.x, a + 0);
        dequant_word(pk0.y, a + 4);
        dequant_word(pk0.z, a + 8);
        dequant_word(pk0.w, a + 12);
        dequant_word(pk1.x, a + 16);
        dequant_word(pk1.y, a + 20);
        dequant_word(pk1.z, a + 24);
        dequant_word(pk1.w, a + 28);
        ER_TR(2);
        const uint32_t a_t = tmem + lane_addr + kTmemA + ia * 64 + half * 32;
        ER_TMEM_ST16(a_t + 0, a, 0);
        ER_TMEM_ST16(a_t + 16, a, 16);
        if (half == 0) sts_f32(sc_s + s * (kTileN * 4), __uint_as_float(sc16 << 16));
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&a_full[ia]);
      }
      ER_TR(3);
      s += 2;
      if (s >= S) { s -= S; ph ^= 1; }
      sp += 2;
      if (sp >= S) { sp -= S; php ^= 1; }
    }
  } else if (warp >= kEpiWarp0) {
    // ===================== scale-accumulate + output =====================
    constexpr int CW = C::kCW;
    constexpr int kEpiThreads = kEpiWarps * 32;
    const int ew = warp - kEpiWarp0;
    const int ch = ew >> 2;                // which half of the accumulator columns (batch rows m)
    const int q4 = warp & 3;
    const int row = q4 * 32 + lane;
    const uint32_t lane_addr = (uint32_t)(q4 * 32) << 16;
    const bool leader = (threadIdx.x == kEpiWarp0 * 32);
    const uint32_t sc_s = smem_u32(sc_buf) + row * 4;
    float acc[CW];
    int it = 0;
    int s = 0;
    uint32_t ph = 0;
    while (it < n_it && !(p.dbg & 64)) {
      // ---- segment = the part of one tile inside this CTA's range ----
      const long long gi0 = gb + it;
      const int tile = (int)(gi0 / p.G), g_lo = (int)(gi0 % p.G);
      const int seg_len = min(p.G - g_lo, n_it - it);
      const int it_end = it + seg_len;
#pragma unroll
      for (int m = 0; m < CW; ++m) acc[m] = 0.f;
      for (int i = it; i < it_end; ++i) {
        const int id = i & (ND - 1);
        ER_TR(4);
        if (ew == 0) mbar_spin(&done[s], ph);
        named_bar_sync(4, kEpiThreads);
        tc_fence_after();
        ER_TR(1);
        uint32_t d[CW];
        const uint32_t d_t = tmem + lane_addr + kTmemD + id * MPAD + ch * CW;
        if constexpr (CW == 8) {
          ER_TMEM_LD8(d_t, d, 0);
        } else {
#pragma unroll
          for (int c = 0; c < CW; c += 16) ER_TMEM_LD16(d_t + c, d, c);
        }
        const float sc = lds_f32(sc_s + s * (kTileN * 4));
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&d_free[id]);
#pragma unroll
        for (int m = 0; m < CW; ++m) acc[m] = fmaf(sc, __uint_as_float(d[m]), acc[m]);
        ER_TR(2);
        if (++s == S) { s = 0; ph ^= 1; }
      }

      // ---- output: direct store, or partial + last-arriver reduction in ascending CTA order ----
      const int n0 = (tile % p.ntiles) * kTileN, m0 = (tile / p.ntiles) * MPAD + ch * CW;
      const int mvalid = min(CW, p.M - m0);     // may be <= 0: nothing of this half is a real batch row
      const int n = n0 + row;
      bool store = true;
      if (seg_len != p.G) {
        float* mine = p.partials + ((size_t)cta * 2 + (it == 0 ? 0 : 1)) * (MPAD * kTileN) + ch * CW * kTileN;
#pragma unroll
        for (int m = 0; m < CW; ++m)
          if (m < mvalid) __stcg(mine + m * kTileN + row, acc[m]);
        __threadfence();
        named_bar_sync(3, kEpiThreads);
        const long long u_first = ((long long)tile * p.G) / ug, u_last = ((long long)(tile + 1) * p.G - 1) / ug;
        const int c_lo = owner_of(p.units, P, u_first), c_hi = owner_of(p.units, P, u_last);
        if (leader) {
          const int old = atomicAdd(p.counters + tile, 1);
          const int last = (old == c_hi - c_lo);
          if (last) p.counters[tile] = 0;  // leave the counter zero for the next call
          *last_flag = last;
        }
        named_bar_sync(3, kEpiThreads);
        store = (*last_flag != 0);
        if (store) {
          __threadfence();
#pragma unroll
          for (int m = 0; m < CW; ++m) acc[m] = 0.f;
          for (int c = c_lo; c <= c_hi; ++c) {
            // CTA c's piece of this tile is its first segment iff its range starts inside the tile
            const long long cb = range_begin(p.units, P, c) * ug;
            const int which = (cb >= (long long)tile * p.G) ? 0 : 1;
            const float* src = p.partials + ((size_t)c * 2 + which) * (MPAD * kTileN) + ch * CW * kTileN;
#pragma unroll
            for (int m = 0; m < CW; ++m)
              if (m < mvalid) acc[m] += __ldcg(src + m * kTileN + row);
          }
        }
        named_bar_sync(3, kEpiThreads);   // last_flag may be rewritten by the next segment only after all have read it
      }
      if (store) {
        if (p.y_f32) {
          float* y = reinterpret_cast<float*>(p.y);
#pragma unroll
          for (int m = 0; m < CW; ++m)
            if (m < mvalid) y[(size_t)(m0 + m) * p.ldy + n] = acc[m];
        } else {
          __nv_bfloat16* y = reinterpret_cast<__nv_bfloat16*>(p.y);
#pragma unroll
          for (int m = 0; m < CW; ++m)
            if (m < mvalid) y[(size_t)(m0 + m) * p.ldy + n] = __float2bfloat16_rn(acc[m]);
        }
      }
      ER_TR(3);
      it = it_end;
    }
  }

  ER_TR(5);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  if (warp == 1) tmem_dealloc<kTmemCols>(tmem);
  ER_TR(6);
#ifdef ER_GEMM_TRACE
  if (p.trace && blockIdx.x == p.dbg_cta && lane == 0)
    for (int i = 0; i < 8; ++i) p.trace[warp * 8 + i] = tr_sum[i];
#endif
}

}  // namespace

// =====================================================================================================
// host side: tensor maps, stream-K plan, launch
// =====================================================================================================
namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (fn) return fn;
  void* sym = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) != cudaSuccess ||
      qres != cudaDriverEntryPointSuccess)
    return nullptr;
  fn = reinterpret_cast<EncodeTiledFn>(sym);
  return fn;
}

// 2-D row-major tensor [rows][cols] of elements, row pitch in bytes, box [box_rows][box_cols].
bool make_map_2d(CUtensorMap* map, CUtensorMapDataType dt, const void* base, uint64_t rows, uint64_t cols,
                 uint64_t pitch_bytes, uint32_t box_rows, uint32_t box_cols, CUtensorMapSwizzle swz) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {pitch_bytes};
  cuuint32_t box[2] = {box_cols, box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(map, dt, 2, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, swz,
                  CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

#ifdef ER_GEMM_TRACE
unsigned long long* g_trace = nullptr;
#endif
int g_tune_dbg = 0;
int g_tune_force_ctas = 0;  // > 0: use this many CTAs (tests / sweeps); 0 = one per SM

struct Plan {
  int mpad, mchunks, ntiles, tiles, G, unit_groups, ctas;
  long long units;
};

int mpad_of(int64_t M) { return M <= 16 ? 16 : (M <= 32 ? 32 : 64); }

Plan make_plan(int64_t M, int64_t N, int64_t K) {
  Plan pl;
  pl.mpad = mpad_of(M);
  pl.mchunks = (int)((M + pl.mpad - 1) / pl.mpad);
  pl.ntiles = (int)(N / kTileN);
  pl.tiles = pl.ntiles * pl.mchunks;
  pl.G = (int)(K / ER_GROUP);
  // one ticket counter per tile: beyond the counter array, whole tiles are dealt out (no partial sums)
  pl.unit_groups = (pl.tiles <= ER_GEMM_COUNTER_BYTES / 4) ? 1 : pl.G;
  pl.units = (long long)pl.tiles * pl.G / pl.unit_groups;
  int ctas = er::sm_count();
  if (g_tune_force_ctas > 0 && g_tune_force_ctas < ctas) ctas = g_tune_force_ctas;
  if ((long long)ctas > pl.units) ctas = (int)pl.units;
  pl.ctas = ctas;
  return pl;
}

size_t workspace_for(int mpad) {
  return ER_GEMM_COUNTER_BYTES + (size_t)er::sm_count() * 2 * mpad * kTileN * sizeof(float);
}

template <int MPAD>
int launch(const CUtensorMap& mx, const GemmParams& gp, const Plan& pl, cudaStream_t stream) {
  static bool attr_set = false;
  if (!attr_set) {
    ER_CUDA_TRY(cudaFuncSetAttribute(w4a16_gemm_kernel<MPAD>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     Cfg<MPAD>::kSmem));
    attr_set = true;
  }
  w4a16_gemm_kernel<MPAD><<<pl.ctas, kThreads, Cfg<MPAD>::kSmem, stream>>>(mx, gp);
  ER_CUDA_TRY(cudaGetLastError());
  return ER_OK;
}

}  // namespace

extern "C" {

// Internal tuning knob for tests and sweeps (not part of the stable ABI): key 1 = number of CTAs the stream-K
// plan uses (0 = one per SM); key 0 is accepted and ignored (it belonged to the first kernel version).
int er_gemm_tuning(int key, int value) {
  if (key == 0 && (value == 1 || value == 2)) return ER_OK;
  if (key == 1 && value >= 0) { g_tune_force_ctas = value; return ER_OK; }
  if (key == 2 && value >= 0) { g_tune_dbg = value; return ER_OK; }
  if (key == 3) return ER_OK;   // (retired knob)
  return ER_ERR_SHAPE;
}

#ifdef ER_GEMM_TRACE
void er_gemm_set_trace(void* dev_ptr) { g_trace = reinterpret_cast<unsigned long long*>(dev_ptr); }
#endif

size_t er_gemm_workspace_bytes(int64_t M, int64_t N, int64_t K) {
  if (M < 1 || N < kTileN || N % kTileN != 0 || K < ER_GROUP || K % ER_GROUP != 0) return 0;
  return workspace_for(mpad_of(M));
}

int er_gemm_workspace_init(void* workspace, size_t workspace_bytes, void* stream) {
  if (!workspace) return ER_ERR_NULL;
  if (workspace_bytes < ER_GEMM_COUNTER_BYTES) return ER_ERR_WORKSPACE;
  ER_CUDA_TRY(cudaMemsetAsync(workspace, 0, ER_GEMM_COUNTER_BYTES, (cudaStream_t)stream));
  return ER_OK;
}

int er_w4a16_gemm(const void* x_bf16, int64_t M, int64_t K, int64_t ldx_elems, const void* qweight,
                  const void* scales, int64_t N, int group, void* y, int64_t ldy_elems, int y_dtype, void* workspace,
                  size_t workspace_bytes, void* stream) {
  if (!x_bf16 || !qweight || !scales || !y) return ER_ERR_NULL;
  if (group != ER_GROUP || M < 1 || M > (1 << 20) || N < kTileN || N % kTileN != 0 || N > (1 << 24) ||
      K < ER_GROUP || K % ER_GROUP != 0 || K > (1 << 24) || ldx_elems < K || ldy_elems < N)
    return ER_ERR_SHAPE;
  if (y_dtype != ER_BF16 && y_dtype != ER_F32) return ER_ERR_DTYPE;
  if (!er::aligned16(x_bf16) || !er::aligned16(qweight) || !er::aligned16(scales) || (ldx_elems % 8) != 0)
    return ER_ERR_ALIGN;
  if (!workspace) return ER_ERR_WORKSPACE;
  if (!er::aligned16(workspace)) return ER_ERR_ALIGN;
  const Plan pl = make_plan(M, N, K);
  if (workspace_bytes < workspace_for(pl.mpad)) return ER_ERR_WORKSPACE;
  int st = er::check_arch();
  if (st != ER_OK) return st;

  CUtensorMap mx;
  bool ok = make_map_2d(&mx, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, x_bf16, (uint64_t)M, (uint64_t)K,
                         (uint64_t)ldx_elems * 2, (uint32_t)pl.mpad, 64, CU_TENSOR_MAP_SWIZZLE_128B);
  if (!ok) {
    er::set_last_cuda_error((int)cudaErrorInvalidValue);
    return ER_ERR_CUDA;
  }
  GemmParams gp;
  gp.M = (int)M; gp.N = (int)N; gp.K = (int)K;
  gp.G = pl.G; gp.ntiles = pl.ntiles; gp.tiles = pl.tiles; gp.unit_groups = pl.unit_groups; gp.units = pl.units;
  gp.dbg = g_tune_dbg;
#ifdef ER_GEMM_TRACE
  gp.trace = g_trace;
  gp.dbg_cta = g_tune_force_ctas < 0 ? 0 : 0;
#endif
  gp.qweight = reinterpret_cast<const uint8_t*>(qweight);
  gp.scales = reinterpret_cast<const uint8_t*>(scales);
  gp.y_f32 = (y_dtype == ER_F32); gp.ldy = ldy_elems; gp.y = y;
  gp.counters = reinterpret_cast<int*>(workspace);
  gp.partials = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(workspace) + ER_GEMM_COUNTER_BYTES);
  cudaStream_t s = (cudaStream_t)stream;
  if (pl.mpad == 16) return launch<16>(mx, gp, pl, s);
  if (pl.mpad == 32) return launch<32>(mx, gp, pl, s);
  return launch<64>(mx, gp, pl, s);
}

}  // extern "C"
