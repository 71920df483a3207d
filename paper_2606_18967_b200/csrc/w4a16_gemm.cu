// w4a16_gemm.cu -- er_w4a16_gemm: the weight-quantized self-drafter's linear, Y = X . dequant(Wq)^T
// (dense projections are ~90 % of tail decode latency and weight loading dominates at
// small batch; L175: W4A16 weight-only kernel; L467: "on-the-fly dequantization and kernel-level overhead").
// This file: the host entry point (validation, work plan, dispatch to the three kernels) and the tcgen05 kernel with
// one fp32 accumulator per 128-k group (exact group scale), which serves M <= 16 -- except M <= 8 on plans without a
// cluster (w4a16_gemm_small.cu) -- and every M > 16 (M > 64 in chunks of 64 batch rows).  Instantiated a second time
// (kPlanes) for er_w8a16_gemm: a W8 matrix stored as two nibble planes per group (quantize_pack8.cu) is a W4 matrix with
// 2 K columns whose groups 2g, 2g + 1 contract the same 128 columns of X; the high plane carries no offset, the low plane
// all of it (M <= 16: constant tile -2304; above: -136 / -128 in the workers).
//
// What the earlier versions taught (profiles/r01_*, r02_gemm.md): TMA / MMA issue must be warp-uniform code with one
// elected lane; a closed ring of few TMEM buffers between separate converter / MMA / read-back roles is bound by the
// round-trip latency of its mbarriers; the nibble -> bf16 conversion (7 logic-pipe operations per packed word, the
// logic pipe runs at half rate) is the largest cost, ~224 cycles per 128-k group and SM sub-partition.
//
//   persistent   one CTA per SM; the (tile, 128-k group) units of the whole problem are dealt out as ONE
//                contiguous range per CTA (stream-K / tile split / thread-block cluster: w4a16_plan.cuh).
//   swap-AB      the 128 weight rows of a tile are the M = 128 of tcgen05.mma, the padded batch is its N.
//   warp 24      producer: per group ONE 8 KiB 1-D bulk copy of the packed block (ER_PACK_V2 keeps every
//                [128 rows x 128 k] block contiguous and pre-swizzled), one 256-byte bulk copy of the group's
//                scales and two SWIZZLE_128B TMA boxes of X [MPAD x 64 k], into a ring of up to 16 stages.
//   warps 25-26  MMA issuers: tcgen05.mma.kind::f16, A (weights) from TENSOR MEMORY, B (= X tile) from shared
//                memory, a fresh fp32 TMEM accumulator per group so the group scale is applied exactly; at M <= 16
//                eight more MMAs per group with a constant -136 tile remove the stored nibble's offset.
//   warps 0-23   three self-paced worker sets of 8 warps; set j owns the groups j, j+3, ... of the CTA's range and
//                its own (A operand, accumulator) buffers in TMEM (two pairs at M <= 16).  A thread owns HALF a
//                weight row of the group.  Per group: wait for the stage (every warp on the mbarrier itself),
//                2 x LDS.128, nibble -> bf16 ((w >> 4t) & 0x000F000F | 0x43004300 = the pair 128 + u; above M = 16
//                one packed fma removes the 136), the scale-accumulate of the set's previous group (tcgen05.ld +
//                fma: its MMAs had the whole conversion to finish), tcgen05.st of the new A operand (the 4x
//                expanded weights never touch shared memory) and an arrival on the set's a_full barrier.
//   output       at the end of a tile segment sets 1-2 hand their partial sums to set 0 through shared memory;
//                a tile wholly owned by one CTA is stored directly; in cluster mode the CTAs of a tile add their
//                sums through distributed shared memory; otherwise fp32 partials go to the workspace and the last
//                CTA of the tile (ticket counter) adds them in ascending CTA order.  Deterministic.
#include "w4a16_plan.cuh"

namespace {

using namespace er;

constexpr int kSets = 3;                    // worker sets
constexpr int kSetWarp0 = 0;                // worker warps 0..23, 8 per set
constexpr int kSetThreads = 256;
constexpr int kWorkerThreads = kSets * kSetThreads;      // 768
// The role warps sit ABOVE the workers: the warp arbiter of an SM sub-partition prefers the highest warp id, and the
// producer / MMA issuers are few-instruction, latency-critical warps that must not queue behind 6 converting warps.
constexpr int kProdWarp = kSets * 8;        // 24
constexpr int kMmaWarp0 = kProdWarp + 1;    // 25, 26
constexpr int kThreads = (kProdWarp + 4) * 32;           // 896 (warp 27 idles)
constexpr int kMaxStages = 16;
constexpr int kTmemCols = 512;
constexpr int kTmemA = 0;                   // A operand: kBuf 64-column buffers per set

template <int MPAD>
struct Cfg {
  static constexpr int kXBytes = MPAD * 128 * 2;           // two boxes of [MPAD x 64] bf16
  static constexpr int kStageBytes = ((kWBytes + kXBytes + kScaleBytes + 1023) / 1024) * 1024;
  static constexpr int kRedBytes = (kSets - 1) * MPAD * kTileN * 4;   // partial sums of sets 1.. handed to set 0
  // cluster mode (M <= 32): up to 3 [MPAD x 128] fp32 slots that the other CTAs of the cluster write into rank 0;
  // a region of their own, so the writers need not wait for rank 0's pipeline to drain (the ring depth is not
  // critical: 8 and 16 stages measure the same)
  static constexpr int kSlotBytes = (MPAD <= 32) ? 3 * MPAD * kTileN * 4 : 0;
  static constexpr int kFixed = kRedBytes + kSlotBytes + 1024 /*align slack*/ + 512 /*barriers*/;
  static constexpr int kStagesRaw = (kSmemLimit - kFixed) / kStageBytes;
  static constexpr int kStages = kStagesRaw > kMaxStages ? kMaxStages : kStagesRaw;
  static constexpr int kSmem = kStages * kStageBytes + kFixed;
  static constexpr uint32_t kTxBytes = kWBytes + kXBytes + kScaleBytes;
  static constexpr int kCW = MPAD / 2;                     // accumulator columns per thread (half of the batch rows)
  static constexpr bool kSubInWorkers = (MPAD > 16);      // see dequant_word
  static constexpr bool kEpiFirst = (MPAD > 32);           // register pressure: read back before converting
  // TMEM: every set owns kBuf (A operand, accumulator) pairs.  Two pairs (M <= 16, where the columns allow it)
  // let a set convert group i + 1 while the MMAs of group i are still in flight.
  static constexpr int kBuf = (MPAD == 16) ? 2 : 1;
  static constexpr int kTmemConst = kSets * kBuf * 64;     // per set 8 columns of bf16 pairs (-136, -136): the constant A tile
  static constexpr int kTmemD = (kTmemConst + 8 * kSets + MPAD - 1) / MPAD * MPAD;   // accumulators, MPAD columns each
  static_assert(kTmemD + kSets * kBuf * MPAD <= kTmemCols, "TMEM columns");
};

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
// of bf16 pairs (128 + u, 128 + u'): (w >> 4t) & 0x000F000F | 0x43004300, i.e. 3 shifts + 4 lop3 per word, all
// on the half-rate logic pipe.  The stored nibble is u = q + 8, so the A operand is q + 136; the -136 is NOT
// removed here (one packed fma per pair would cost as many issue cycles again) but folded into the
// contraction: eight more MMAs per group with a constant A tile of -136 add -136 * sum_k x to the accumulator.
// (An fp16 A operand would need 5 logic ops, but tcgen05.mma.kind::f16 faults on fp16 A x bf16 B.)
// kSub: remove the 136 here with one packed fma per pair (used where the tensor pipe, not the logic pipe, is the
// busier one: at N >= 32 the eight constant-tile MMAs per group cost more than the subtracts, which issue on the
// FMA pipe beside the logic-pipe shifts and lop3s).
template <bool kSub>
__device__ __forceinline__ void dequant_word(uint32_t w, uint32_t* a, uint32_t off2) {
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    const uint32_t v = lop3_and_or(w >> (4 * t), 0x000F000Fu, 0x43004300u);
    if (kSub) asm("fma.rn.bf16x2 %0, %1, %2, %3;" : "=r"(a[t]) : "r"(v), "r"(0x3F803F80u), "r"(off2));
    else a[t] = v;
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

__device__ __forceinline__ void named_bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

template <int MPAD, bool kClusterMode, bool kPlanes = false>
__global__ void __launch_bounds__(kThreads, 1)
w4a16_gemm_kernel(const __grid_constant__ CUtensorMap map_x, const GemmParams p) {
  using C = Cfg<MPAD>;
  constexpr int S = C::kStages;
  constexpr int kBuf = C::kBuf;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  float* red = reinterpret_cast<float*>(smem + S * C::kStageBytes);             // [kSets-1][MPAD][128]
  uint8_t* slots_base = smem + S * C::kStageBytes + C::kRedBytes;               // cluster slots (see Cfg)
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + S * C::kStageBytes + C::kRedBytes + C::kSlotBytes);
  uint64_t* full = bars;                        // [S]     TMA landed
  uint64_t* empty = bars + kMaxStages;          // [S]     the group's MMAs completed: the stage may be refilled
  uint64_t* a_full = bars + 2 * kMaxStages;     // [kSets][kBuf] the A operand is written, its accumulator drained
  uint64_t* done = a_full + 8;                  // [kSets][kBuf] the MMAs completed: accumulator readable, A free
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(done + 8);
  int* last_flag = reinterpret_cast<int*>(tmem_slot + 1);

  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);   // provably warp-uniform
  const int lane = threadIdx.x & 31;
  const int P = gridDim.x, cta = blockIdx.x;
  const int ug = p.unit_groups;
  const int gb = range_begin(p.uq, p.ur, p.split, cta) * ug;        // first global group index of this CTA
  const int ge = range_begin(p.uq, p.ur, p.split, cta + 1) * ug;
  const int n_it = (int)(ge - gb);
  static_assert(!kClusterMode || MPAD <= 32, "the host only uses clusters at M <= 32");
  float cl_acc[kClusterMode ? C::kCW : 1];      // cluster mode: set 0's sum over this CTA's part of its tile ...
  int cl_tile = -1;                     // ... and the tile

  if (warp == kProdWarp) {
    if (lane < S) {
      mbar_init(&full[lane], 1);
      mbar_init(&empty[lane], 1);
    }
    if (lane < kSets * C::kBuf) {
      mbar_init(&a_full[lane], 8);
      mbar_init(&done[lane], 1);
    }
    mbar_fence_init();
    if (lane == 0) tma_prefetch_desc(&map_x);
    // the producer does not wait for the TENSOR-MEMORY allocation: it arrives on the prologue barrier and goes on to
    // griddepcontrol.wait and its first loads (the ~0.3 us of the prologue are otherwise serialised behind the previous
    // kernel's exit in every launch)
    named_bar_arrive(15, kThreads);
  } else {
    if (warp == kMmaWarp0) tmem_alloc<kTmemCols>(tmem_slot);
    tc_fence_before();
    named_bar_sync(15, kThreads);
    tc_fence_after();
  }
  const uint32_t tmem = (warp == kProdWarp) ? 0u : __shfl_sync(0xffffffffu, *tmem_slot, 0);
  if constexpr (kClusterMode) {   // "I have started": waited for before the first remote shared-memory access
    if (p.cluster > 1) asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory");
  }
  // Programmatic dependent launch: everything above touched no global memory, so it may overlap the tail of the
  // previous kernel in the stream; from here on its results (X, the workspace) are needed.  The next kernel may be
  // scheduled as soon as SMs free up (it waits at its own griddepcontrol.wait).  (Issuing the first ring stages of
  // weights BEFORE the wait was measured and does not pay here: with one CTA per SM the next kernel's CTAs only
  // become resident when this kernel's exit, so there is nothing to overlap with -- profiles/r02_gemm.md.)
  // The producer first asks L2 for the beginning of this CTA's weight stream (a contiguous byte range of ER_PACK_V2):
  // safe even right behind a refresh, because L2 is the point of coherence and a prefetched line cannot be stale.
  if (warp == kProdWarp && elect_one()) {
    // 64 KB per SM: deeper prefetches measured slower (profiles/r02_gemm.md).  Only with one batch chunk (M <= 64): with
    // several, the tiles of chunk mc > 0 re-use the weight blocks of chunk 0 and gb is no position in the weight stream
    // (a prefetch of gb * 8 KiB reached beyond the matrix and cost the M > 64 launches a factor of two)
    const int npf = p.mchunks == 1 ? (n_it < 8 ? n_it : 8) : 0;
    const int wb = gb;
    if (npf > 0) bulk_prefetch_l2(p.qweight + (size_t)wb * kWBytes, (uint32_t)npf * kWBytes);
  }
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  if (warp == kProdWarp) {
    // ===================== producer (warp-uniform; one elected lane issues) =====================
    const int tile0 = (int)(gb / p.G);
    int g = (int)(gb % p.G), tn = tile0 % p.ntiles, mc = tile0 / p.ntiles;
    int s = 0;
    uint32_t ph = 0;
    for (int it = 0; it < n_it; ++it) {
      mbar_wait(&empty[s], ph ^ 1);      // the stage's previous group (it - S) has been contracted
      if (elect_one()) {
        uint8_t* st = smem + s * C::kStageBytes;
        mbar_arrive_expect_tx(&full[s], C::kTxBytes);
        // ER_PACK_V2: the [128 rows x 128 k] block of (tile, g) is 8 KiB of contiguous, pre-swizzled bytes
        bulk_load_1d(st, p.qweight + ((size_t)tn * p.G + g) * kWBytes, kWBytes, &full[s], kEvictFirst);
        const int xk = (g >> (kPlanes ? 1 : 0)) * 128;      // two-plane W8: both planes of a group contract the same X columns
        tma_load_2d(st + kWBytes, &map_x, &full[s], xk, mc * MPAD, kEvictLast);
        tma_load_2d(st + kWBytes + MPAD * 128, &map_x, &full[s], xk + 64, mc * MPAD, kEvictLast);
        bulk_load_1d(st + kWBytes + C::kXBytes, p.scales + ((size_t)g * p.N + tn * kTileN) * 2, kScaleBytes,
                     &full[s], kEvictFirst);
      }
      __syncwarp();
      if (++g == p.G) {
        g = 0;
        if (++tn == p.ntiles) { tn = 0; ++mc; }
      }
      if (++s == S) { s = 0; ph ^= 1; }
    }
  } else if (warp == kMmaWarp0 || warp == kMmaWarp0 + 1) {
    // ===================== MMA issuers (warp-uniform; one elected lane issues) =====================
    // Two issuers, on different SM sub-partitions (the worker warps keep the issue slots busy: one issuer alone is
    // too slow).  An a_full barrier must always be served by the same issuer, which then sees every one of its
    // phases: with two buffers per set warp 1 takes the even groups of the range and warp 2 the odd ones (a
    // (set, buffer) pair has a fixed group parity); with one buffer per set warp 1 serves sets 0 and 2, warp 2
    // serves set 1.
    constexpr uint32_t idesc = idesc_bf16_m128(MPAD);
    int s = 0, set = 0, i = 0;           // stage, set and the set's group count of group `it`
    uint32_t ph = 0;                     // parity of full[s] (streaming-only mode)
    for (int it = 0; it < n_it; ++it) {
      const bool mine = (kBuf == 2) ? ((it & 1) == warp - kMmaWarp0) : ((set == 1) == (warp == kMmaWarp0 + 1));
      if (mine) {
        {
          const int bi = set * kBuf + (i % kBuf);
          mbar_wait(&a_full[bi], (i / kBuf) & 1);            // implies full[s] (the set waited for it)
          tc_fence_after();
          if (elect_one()) {
            const uint32_t xbase = smem_u32(smem + s * C::kStageBytes + kWBytes);
            const uint32_t d_t = tmem + C::kTmemD + bi * MPAD;
            const uint32_t a_t = tmem + kTmemA + bi * 64;
#pragma unroll
            for (int kk = 0; kk < 8; ++kk) {
              const uint64_t bdesc = smem_desc_sw128(xbase + (kk >> 2) * (MPAD * 128) + (kk & 3) * 32);
              mma_ts_f16(d_t, a_t + kk * 8, bdesc, idesc, kk > 0 ? 1u : 0u);
            }
            // - 136 * sum_k x[m][k]: the stored nibble's offset.  Two-plane W8: the high-nibble plane (even groups; G is
            // even, so the parity of gb + it is the plane) carries none, the low-nibble plane all of it (- 2304, see the
            // constant tile)
            if (!C::kSubInWorkers && !(kPlanes && !((gb + it) & 1))) {
#pragma unroll
              for (int kk = 0; kk < 8; ++kk) {
                const uint64_t bdesc = smem_desc_sw128(xbase + (kk >> 2) * (MPAD * 128) + (kk & 3) * 32);
                mma_ts_f16(d_t, tmem + C::kTmemConst + set * 8, bdesc, idesc, 1u);
              }
            }
            tc_commit(&done[bi]);
            tc_commit(&empty[s]);
          }
        }
        __syncwarp();
      }
      if (++s == S) { s = 0; ph ^= 1; }
      if (++set == kSets) { set = 0; ++i; }
    }
  } else if (warp < kProdWarp) {
    // ===================== worker sets: convert, scale-accumulate, output =====================
    constexpr int CW = C::kCW;
    const int dw = warp - kSetWarp0;
    const int set = dw >> 3;               // groups set, set + 3, ... of the CTA's range
    const int half = (dw >> 2) & 1;        // which 64 k of a group this thread converts / which half of the batch rows
    const int q4 = warp & 3;               // TMEM lane quarter this warp may access
    const int row = q4 * 32 + lane;        // weight row inside the tile
    const uint32_t lane_addr = (uint32_t)(q4 * 32) << 16;
    const int sw = (row >> 1) & 3;
    // loop invariants, pinned in registers (otherwise the compiler rematerialises the shared-window arithmetic
    // in every iteration)
    uint32_t w_addr0, w_addr1, sc_addr;
    asm volatile("mov.u32 %0, %1;" : "=r"(w_addr0) : "r"(smem_u32(smem) + row * 64 + (((2 * half) ^ sw) << 4)));
    asm volatile("mov.u32 %0, %1;" : "=r"(w_addr1) : "r"(smem_u32(smem) + row * 64 + (((2 * half + 1) ^ sw) << 4)));
    asm volatile("mov.u32 %0, %1;" : "=r"(sc_addr) : "r"(smem_u32(smem) + kWBytes + C::kXBytes + row * 2));
    uint32_t full_addr, done_addr, afull_addr;
    asm volatile("mov.u32 %0, %1;" : "=r"(full_addr) : "r"(smem_u32(full)));
    asm volatile("mov.u32 %0, %1;" : "=r"(done_addr) : "r"(smem_u32(&done[set * kBuf])));
    asm volatile("mov.u32 %0, %1;" : "=r"(afull_addr) : "r"(smem_u32(&a_full[set * kBuf])));
    // every warp waits on the mbarriers itself (try_wait suspends the warp in hardware): measured 1 % faster than one
    // polling warp per set + a named barrier, and the warps of a set no longer wait for their slowest sibling
    const bool leader = (threadIdx.x == kSetWarp0 * 32);
    uint32_t a_t, d_t;
    asm volatile("mov.u32 %0, %1;" : "=r"(a_t) : "r"(tmem + lane_addr + kTmemA + set * kBuf * 64 + half * 32));
    asm volatile("mov.u32 %0, %1;" : "=r"(d_t) : "r"(tmem + lane_addr + C::kTmemD + set * kBuf * MPAD + half * CW));

    if (half == 0) {                       // the set's constant A tile (-136, -136), one lane quarter per warp; ordered
                                           // before the set's first MMA by its first a_full arrival
      // (-136, -136); two-plane W8: (-2304, -2304) = -(16 * 128 + 128 + 128), exact in bf16: with scales (16 s, s) the
      // planes then sum to s * sum_k x (16 a + b - 128) = s * sum_k x q
      const uint32_t c = kPlanes ? 0xC510C510u : 0xC308C308u;
      asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%1,%1,%1,%1,%1,%1,%1};" ::"r"(
                       tmem + lane_addr + C::kTmemConst + set * 8), "r"(c) : "memory");
      asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
      tc_fence_before();
    }

    float acc[CW];
    float sc_old = 0.f, sc_new = 0.f;      // scales of the (up to kBuf) groups whose MMAs are in flight
    int npend = 0;                         // how many
    uint32_t pd = 0;                       // bit b: parity of done[set][b] for its next read-back
    int wbuf = 0, rbuf = 0;                // buffer the next group is written to / read back from
    int my = set;                          // this set's next group (index into the CTA's range)
    int s = set % S;                       // its stage ...
    uint32_t ph = 0;                       // ... and the parity of full[s]
    int it = 0, seg = 0;

    // scale-accumulate of the set's pending group: acc += scale * (sum over its 128 k of x * q)
    auto read_back = [&]() {
      mbar_wait_addr(done_addr + rbuf * 8, (pd >> rbuf) & 1);
      pd ^= 1u << rbuf;
      tc_fence_after();
      uint32_t d[CW];
      const uint32_t dt = d_t + rbuf * MPAD;
      if constexpr (CW == 8) {
        ER_TMEM_LD8(dt, d, 0);
      } else {
#pragma unroll
        for (int c = 0; c < CW; c += 16) ER_TMEM_LD16(dt + c, d, c);
      }
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
      for (int m = 0; m < CW; ++m) acc[m] = fmaf(sc_old, __uint_as_float(d[m]), acc[m]);
      sc_old = sc_new;
      --npend;
      if (kBuf == 2) rbuf ^= 1;
    };

    int pend_tile[2] = {-1, -1};           // partial tiles of this CTA (head / tail segment of its range)
    auto store_tile = [&](int tile, const float (&v)[CW]) {
      const int n = (tile % p.ntiles) * kTileN + row, m0 = (tile / p.ntiles) * MPAD + half * CW;
      const int mvalid = min(CW, p.M - m0);     // may be <= 0: nothing of this half is a real batch row
      if (p.y_f32) {
        float* y = reinterpret_cast<float*>(p.y);
#pragma unroll
        for (int m = 0; m < CW; ++m)
          if (m < mvalid) y[(size_t)(m0 + m) * p.ldy + n] = v[m];
      } else {
        __nv_bfloat16* y = reinterpret_cast<__nv_bfloat16*>(p.y);
#pragma unroll
        for (int m = 0; m < CW; ++m)
          if (m < mvalid) y[(size_t)(m0 + m) * p.ldy + n] = __float2bfloat16_rn(v[m]);
      }
    };

    while (it < n_it) {
      // ---- segment = the part of one tile inside this CTA's range ----
      const int gi0 = gb + it;
      const int tile = (int)(gi0 / p.G), g_lo = (int)(gi0 % p.G);
      const int seg_len = min(p.G - g_lo, n_it - it);
      const int it_end = it + seg_len;
      const bool last_seg = (it_end == n_it);
#pragma unroll
      for (int m = 0; m < CW; ++m) acc[m] = 0.f;
      for (; my < it_end; my += kSets) {
        mbar_wait_addr(full_addr + s * 8, ph);
        {
          const uint32_t st = s * C::kStageBytes;
          if (C::kEpiFirst && npend == kBuf) read_back();
          const uint4 pk0 = lds128(st + w_addr0);
          const uint4 pk1 = lds128(st + w_addr1);
          const uint32_t sc16 = lds_u16(st + sc_addr);
          // (-136, -136) as bf16 pair; two-plane W8: the low-nibble plane (odd groups) takes (-128, -128): b - 0
          const uint32_t off2 = (kPlanes && ((gb + my) & 1)) ? 0xC300C300u : 0xC308C308u;
          uint32_t a[32];
          dequant_word<C::kSubInWorkers>(pk0.x, a + 0, off2);
          dequant_word<C::kSubInWorkers>(pk0.y, a + 4, off2);
          dequant_word<C::kSubInWorkers>(pk0.z, a + 8, off2);
          dequant_word<C::kSubInWorkers>(pk0.w, a + 12, off2);
          dequant_word<C::kSubInWorkers>(pk1.x, a + 16, off2);
          dequant_word<C::kSubInWorkers>(pk1.y, a + 20, off2);
          dequant_word<C::kSubInWorkers>(pk1.z, a + 24, off2);
          dequant_word<C::kSubInWorkers>(pk1.w, a + 28, off2);
          // the set's previous group: its MMAs had this whole conversion to finish; after this the A buffer
          // (read by those MMAs) and the accumulator are free again
          if (!C::kEpiFirst && npend == kBuf) read_back();
          ER_TMEM_ST16(a_t + wbuf * 64 + 0, a, 0);
          ER_TMEM_ST16(a_t + wbuf * 64 + 16, a, 16);
          asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive_addr(afull_addr + wbuf * 8);
          if (npend == 0) sc_old = __uint_as_float(sc16 << 16);
          else sc_new = __uint_as_float(sc16 << 16);
          ++npend;
          if (kBuf == 2) wbuf ^= 1;
        }
        s += kSets;
        if (s >= S) { s -= S; ph ^= 1; }
      }
      while (npend > 0) read_back();

      // ---- combine the three sets' partial sums in a fixed order (set 0 + set 1 + set 2), in set 0 ----
      if (set != 0) {
        if (seg > 0) named_bar_sync(5, kWorkerThreads);   // set 0 has read the previous segment's `red`
        float* mine = red + ((set - 1) * MPAD + half * CW) * kTileN + row;
#pragma unroll
        for (int m = 0; m < CW; ++m) mine[m * kTileN] = acc[m];
        named_bar_arrive(6, kWorkerThreads);
      } else {
        named_bar_sync(6, kWorkerThreads);
#pragma unroll
        for (int j = 0; j < kSets - 1; ++j) {
          const float* theirs = red + (j * MPAD + half * CW) * kTileN + row;
#pragma unroll
          for (int m = 0; m < CW; ++m) acc[m] += theirs[m * kTileN];
        }
        if (!last_seg) named_bar_arrive(5, kWorkerThreads);

        // ---- output: a whole tile is stored directly; a partial one goes to the workspace as fp32 and is
        //      finished after the main loop (the reduction's round trips would otherwise stall the pipeline) ----
        if (seg_len == p.G) {
          store_tile(tile, acc);
        } else if (kClusterMode && p.cluster > 1) {   // reduced over the cluster at the end of the kernel (one segment
                                                      // per CTA)
          if constexpr (kClusterMode) {
#pragma unroll
            for (int m = 0; m < CW; ++m) cl_acc[m] = acc[m];
          }
          cl_tile = tile;
        } else {
          const int k = (it == 0 ? 0 : 1);
          const int m0 = (tile / p.ntiles) * MPAD + half * CW;
          const int mvalid = min(CW, p.M - m0);
          float* mine = p.partials + ((size_t)cta * 2 + k) * (MPAD * kTileN) + half * CW * kTileN;
#pragma unroll
          for (int m = 0; m < CW; ++m)
            if (m < mvalid) __stcg(mine + m * kTileN + row, acc[m]);
          pend_tile[k] = tile;
        }
      }
      it = it_end;
      ++seg;
    }

    // ---- partial tiles: ticket per tile; the last CTA to arrive adds all partials in ascending CTA order ----
    // Ordering: partial stores (all threads) -> bar.sync -> the leader's acq_rel ticket (release is cumulative over
    // what the barrier made visible to the leader); last arriver: acq_rel ticket -> bar.sync -> ld.cg of the others'
    // partials.  No per-thread __threadfence on either side.
    if (set == 0 && (pend_tile[0] >= 0 || pend_tile[1] >= 0)) {
      named_bar_sync(7, kSetThreads);
      int c_lo[2] = {0, 0}, c_hi[2] = {-1, -1};
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        if (pend_tile[k] < 0) continue;
        const int u_first = (pend_tile[k] * p.G) / ug;
        const int u_last = ((pend_tile[k] + 1) * p.G - 1) / ug;
        c_lo[k] = owner_of(p.uq, p.ur, p.split, u_first);
        c_hi[k] = owner_of(p.uq, p.ur, p.split, u_last);
      }
      if (leader) {
        int old[2] = {0, 0};
#pragma unroll
        for (int k = 0; k < 2; ++k)
          if (pend_tile[k] >= 0)   // two independent round trips
            asm volatile("atom.acq_rel.gpu.global.add.s32 %0, [%1], 1;" : "=r"(old[k]) : "l"(p.counters + pend_tile[k]) : "memory");
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          const int last = (pend_tile[k] >= 0 && old[k] == c_hi[k] - c_lo[k]);
          if (last) p.counters[pend_tile[k]] = 0;  // leave the counter zero for the next call
          last_flag[k] = last;
        }
      }
      named_bar_sync(7, kSetThreads);
      constexpr int kChunk = CW <= 8 ? 6 : (CW <= 16 ? 3 : 1);   // contributors whose loads are in flight together
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        if (pend_tile[k] < 0 || last_flag[k] == 0) continue;
        const int tile = pend_tile[k];
        const int m0 = (tile / p.ntiles) * MPAD + half * CW;
        const int mvalid = min(CW, p.M - m0);
#pragma unroll
        for (int m = 0; m < CW; ++m) acc[m] = 0.f;
        for (int c0 = c_lo[k]; c0 <= c_hi[k]; c0 += kChunk) {
          float v[kChunk][CW];
#pragma unroll
          for (int j = 0; j < kChunk; ++j) {
            const int c = min(c0 + j, c_hi[k]);
            // CTA c's piece of this tile is its first segment iff its range starts inside the tile
            const int cb = range_begin(p.uq, p.ur, p.split, c) * ug;
            const int which = (cb >= tile * p.G) ? 0 : 1;
            const float* src = p.partials + ((size_t)c * 2 + which) * (MPAD * kTileN) + half * CW * kTileN;
#pragma unroll
            for (int m = 0; m < CW; ++m) v[j][m] = (m < mvalid && c0 + j <= c_hi[k]) ? __ldcg(src + m * kTileN + row) : 0.f;
          }
#pragma unroll
          for (int j = 0; j < kChunk; ++j)
#pragma unroll
            for (int m = 0; m < CW; ++m)
              if (c0 + j <= c_hi[k]) acc[m] += v[j][m];
        }
        store_tile(tile, acc);
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  if (warp == kMmaWarp0) tmem_dealloc<kTmemCols>(tmem);

  // ---- cluster mode: the k CTAs of a tile add their sums through distributed shared memory (an L2 ticket plus
  //      partial loads costs two ~1 us round trips; here it is remote shared-memory stores and one cluster barrier).
  //      Rank r > 0 writes its [MPAD x 128] fp32 tile into slot r - 1 of rank 0's slot region; rank 0
  //      adds the slots in rank order and stores the tile.  Deterministic. ----
  if constexpr (kClusterMode) if (p.cluster > 1) {
    uint32_t rank;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
    asm volatile("barrier.cluster.wait.aligned;" ::: "memory");   // every CTA of the cluster has started (long ago)
    const bool set0 = (warp < 8);
    const int row = (warp & 3) * 32 + lane, hf = ((warp - kSetWarp0) >> 2) & 1;
    if (set0 && rank != 0 && cl_tile >= 0) {
      uint32_t remote;
      asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(smem_u32(slots_base)), "r"(0));
      remote += (((rank - 1) * MPAD + hf * C::kCW) * kTileN + row) * 4;
#pragma unroll
      for (int m = 0; m < C::kCW; ++m)
        asm volatile("st.shared::cluster.f32 [%0], %1;" ::"r"(remote + m * kTileN * 4), "f"(cl_acc[m]) : "memory");
    }
    // one cluster barrier: the remote stores are visible to rank 0 (rank 0's slot region is never touched by its own
    // pipeline, so the writers did not have to wait for it)
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
    if (set0 && rank == 0 && cl_tile >= 0) {
      const float* slots = reinterpret_cast<const float*>(slots_base);
      for (int r = 1; r < p.cluster; ++r)
#pragma unroll
        for (int m = 0; m < C::kCW; ++m) cl_acc[m] += slots[((r - 1) * MPAD + hf * C::kCW + m) * kTileN + row];
      const int n = (cl_tile % p.ntiles) * kTileN + row, m0 = (cl_tile / p.ntiles) * MPAD + hf * C::kCW;
      const int mvalid = min(C::kCW, p.M - m0);
      if (p.y_f32) {
        float* y = reinterpret_cast<float*>(p.y);
#pragma unroll
        for (int m = 0; m < C::kCW; ++m)
          if (m < mvalid) y[(size_t)(m0 + m) * p.ldy + n] = cl_acc[m];
      } else {
        __nv_bfloat16* y = reinterpret_cast<__nv_bfloat16*>(p.y);
#pragma unroll
        for (int m = 0; m < C::kCW; ++m)
          if (m < mvalid) y[(size_t)(m0 + m) * p.ldy + n] = __float2bfloat16_rn(cl_acc[m]);
      }
    }
  }
}

}  // namespace


// =====================================================================================================
// host side: tensor maps, work plan, launch
// =====================================================================================================
namespace er {

#ifdef ER_DEV
Tuning g_tune = {1, 1, 1, 0, 1, 0, 1, 0};
#endif

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
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

}  // namespace er

namespace {


int max_active_clusters16(int c);

int mpad_of(int64_t M) { return M <= 16 ? 16 : (M <= 32 ? 32 : 64); }

// M > 64: which kernel (64-row chunks here, or the 128-row kernel of w4a16_gemm_wide.cu) and which partition (whole tiles,
// or stream-K ranges whose partial tiles go through the workspace).  Estimated microseconds from measured constants
// (profiles/r02_gemm.md section 10): 0.40 / 0.54 us per 128-k group and SM for a tile of 64 / 128 batch rows, 22 / 14 us for
// the partial-tile traffic and reduction of a stream-K plan (partials of 32 / 64 KB written and re-read at the end of the
// launch, by all CTAs at once).
struct PlanAbove64 { bool wide, whole_wide, whole_narrow; int split_wide; };
PlanAbove64 plan_above_64(int64_t M, int64_t N, int64_t K, bool planes) {
  const Tuning& tn = er::g_tune;
  const long long sms = er::sm_count(), G = K / ER_GROUP, ntiles = N / kTileN;
  const long long tn_ = ntiles * ((M + 63) / 64), tw_ = ntiles * ((M + 127) / 128);
  const double whole_n = (double)((tn_ + sms - 1) / sms) * G * 0.40, sk_n = (double)((tn_ * G + sms - 1) / sms) * 0.40 + 22.0;
  const double whole_w = (double)((tw_ + sms - 1) / sms) * G * 0.54, sk_w = (double)((tw_ * G + sms - 1) / sms) * 0.54 + 14.0;
  // wide kernel, tile split: k parts per tile, one partial tile per CTA instead of two (measured: ~6 us + the share of the
  // stream-K figure that the number of partial tiles makes up)
  const long long ks = tw_ > 0 ? sms / tw_ : 0;
  const double split_w = (ks >= 2 && ks <= G && tn.split) ? (double)((G + ks - 1) / ks) * 0.54 + 6.0 + 14.0 * (double)(tw_ * ks) / (2.0 * sms)
                                                          : 1e30;
  PlanAbove64 r;
  r.split_wide = (tn.units == 0 && split_w < fmin(whole_w, sk_w)) ? (int)ks : 0;
  (void)planes;   // the two-plane W8 matrix is a W4 matrix with 2 K columns for this purpose
  r.wide = tn.wide != 0 && (tn.wide == 2 || fmin(fmin(whole_w, sk_w), split_w) < fmin(whole_n, sk_n));
  r.whole_wide = tn.units == 1 || (tn.units == 0 && whole_w <= sk_w);
  r.whole_narrow = tn.units == 1 || (tn.units == 0 && whole_n <= sk_n);
  return r;
}

Plan make_plan(int64_t M, int64_t N, int64_t K) {
  const Tuning& tn = er::g_tune;
  Plan pl;
  pl.mpad = mpad_of(M);
  pl.mchunks = (int)((M + pl.mpad - 1) / pl.mpad);
  pl.ntiles = (int)(N / kTileN);
  pl.tiles = pl.ntiles * pl.mchunks;
  pl.G = (int)(K / ER_GROUP);
  // one ticket counter per tile: beyond the counter array, whole tiles are dealt out (no partial sums)
  pl.unit_groups = (pl.tiles <= ER_GEMM_COUNTER_BYTES / 4) ? 1 : pl.G;
  int ctas = er::sm_count();
  if (tn.force_ctas > 0 && tn.force_ctas < ctas) ctas = tn.force_ctas;
  // M > 64 (several chunks of 64 batch rows, every (chunk, weight tile) a tile of its own): whole tiles where the cost
  // model prefers them to stream-K ranges (plan_above_64)
  if (M > 64 && tn.force_ctas == 0 && plan_above_64(M, N, K, true).whole_narrow) pl.unit_groups = pl.G;
  pl.units = (long long)pl.tiles * pl.G / pl.unit_groups;
  if ((long long)ctas > pl.units) ctas = (int)pl.units;
  pl.ctas = ctas;
  // tile split: when k >= 2 parts per tile fill at least 90 % of the CTAs, no CTA has to straddle two tiles
  pl.split = 0;
  if (tn.split && pl.unit_groups == 1 && tn.force_ctas == 0) {
    const int k = ctas / pl.tiles;
    if (k >= 2 && k <= pl.G && pl.tiles * k * 10 >= ctas * 9) {
      pl.split = k;
      pl.ctas = pl.tiles * k;
    }
  }
  // cluster mode (M <= 32): the parts of a tile are one thread-block cluster and reduce through distributed shared
  // memory.  The cluster size is limited by how many clusters of one-CTA-per-SM footprint the GPCs can hold at once.
  pl.cluster = 1;
  if (tn.cluster && pl.mpad <= 32 && pl.unit_groups == 1 && tn.force_ctas == 0 && pl.mchunks == 1) {
    for (int c = 4; c >= 2; --c) {
      if (c <= pl.G && max_active_clusters16(c) >= pl.tiles && pl.tiles * c * 10 >= ctas * 7) {
        pl.cluster = c;
        pl.split = c;
        pl.ctas = pl.tiles * c;
        break;
      }
    }
  }
  return pl;
}

size_t workspace_for(int mpad) {
  return ER_GEMM_COUNTER_BYTES + (size_t)er::sm_count() * 2 * mpad * kTileN * sizeof(float);
}


template <int MPAD, bool kCl, bool kPlanes = false>
int launch(const CUtensorMap& mx, const GemmParams& gp, const Plan& pl, cudaStream_t stream) {
  static bool attr_set[er::kMaxDevices] = {};
  const int dev = er::current_device();
  if (dev < 0 || dev >= er::kMaxDevices || !attr_set[dev]) {
    ER_CUDA_TRY(cudaFuncSetAttribute(w4a16_gemm_kernel<MPAD, kCl, kPlanes>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     Cfg<MPAD>::kSmem));
    if (dev >= 0 && dev < er::kMaxDevices) attr_set[dev] = true;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)pl.ctas);
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = Cfg<MPAD>::kSmem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = er::g_tune.pdl;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if (pl.cluster > 1) {
    attr[1].id = cudaLaunchAttributeClusterDimension;
    attr[1].val.clusterDim.x = (unsigned)pl.cluster;
    attr[1].val.clusterDim.y = 1;
    attr[1].val.clusterDim.z = 1;
    cfg.numAttrs = 2;
  }
  ER_CUDA_TRY(cudaLaunchKernelEx(&cfg, w4a16_gemm_kernel<MPAD, kCl, kPlanes>, mx, gp));
  return ER_OK;
}

// how many clusters of c CTAs of the tcgen05 M <= 16 kernel (one CTA per SM) can be resident at once; per device
int max_active_clusters16(int c) {
  static int cache[er::kMaxDevices][9] = {};
  if (c < 2 || c > 8) return 0;
  const int dev = er::current_device();
  const bool cacheable = dev >= 0 && dev < er::kMaxDevices;
  if (cacheable && cache[dev][c] != 0) return cache[dev][c] < 0 ? 0 : cache[dev][c];
  cudaFuncSetAttribute(w4a16_gemm_kernel<16, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg<16>::kSmem);
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(c * 64));
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = Cfg<16>::kSmem;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)c;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  int n = 0;
  if (cudaOccupancyMaxActiveClusters(&n, w4a16_gemm_kernel<16, true>, &cfg) != cudaSuccess) {
    (void)cudaGetLastError();
    n = 0;
  }
  if (cacheable) cache[dev][c] = n > 0 ? n : -1;
  return n;
}

}  // namespace

extern "C" {

#ifdef ER_DEV
// Development library only (csrc/er_dev.h; never part of liber_b200.so): partition / launch-mode knobs for the tests
// that compare every mode against the oracle.  key 1 = number of CTAs (0 = one per SM), 3 = programmatic dependent
// launch, 4 = tile split, 5 = cluster mode, 6 = M <= 16 through the warp-MMA kernel (1) or the tcgen05 kernel (0).
int er_dev_gemm_tuning(int key, int value) {
  if (key == 1 && value >= 0) { er::g_tune.force_ctas = value; return ER_OK; }
  if (key == 3 && (value == 0 || value == 1)) { er::g_tune.pdl = value; return ER_OK; }
  if (key == 4 && (value == 0 || value == 1)) { er::g_tune.split = value; return ER_OK; }
  if (key == 5 && (value == 0 || value == 1)) { er::g_tune.cluster = value; return ER_OK; }
  if (key == 6 && (value == 0 || value == 1)) { er::g_tune.small_mma = value; return ER_OK; }
  if (key == 7 && value >= 0 && value <= 2) { er::g_tune.large = value; return ER_OK; }
  if (key == 8 && value >= 0 && value <= 2) { er::g_tune.wide = value; return ER_OK; }
  if (key == 9 && value >= 0 && value <= 2) { er::g_tune.units = value; return ER_OK; }
  return ER_ERR_SHAPE;
}
#endif


size_t er_gemm_workspace_bytes(int64_t M, int64_t N, int64_t K) {
  if (M < 1 || N < kTileN || N % kTileN != 0 || K < ER_GROUP || K % ER_GROUP != 0) return 0;
  size_t exact = workspace_for(mpad_of(M));
  if (M > 64) {   // the 128-row kernel's partial tiles (w4a16_gemm_wide.cu)
    const size_t wide = er::wide_workspace_bytes();
    if (wide > exact) exact = wide;
  }
#ifdef ER_DEV   // the development library can switch to the pre-scaled large-batch kernel (w4a16_gemm_large.cu)
  const size_t large = M > 16 ? er::large_workspace_bytes(M, N, K) : 0;
  return exact > large ? exact : large;
#else
  return exact;
#endif
}

int er_gemm_workspace_init(void* workspace, size_t workspace_bytes, void* stream) {
  if (!workspace) return ER_ERR_NULL;
  if (workspace_bytes < ER_GEMM_COUNTER_BYTES) return ER_ERR_WORKSPACE;
  ER_CUDA_TRY(cudaMemsetAsync(workspace, 0, ER_GEMM_COUNTER_BYTES, (cudaStream_t)stream));
  return ER_OK;
}

// `planes` = 1: W8 stored as two nibble planes (er_w8a16_gemm): the packed matrix has 2 K columns (2 K / 128 groups), X has K.
static int gemm_impl(const void* x_bf16, int64_t M, int64_t K, int64_t ldx_elems, const void* qweight,
                     const void* scales, int64_t N, int group, void* y, int64_t ldy_elems, int y_dtype, void* workspace,
                     size_t workspace_bytes, void* stream, int planes) {
  if (!x_bf16 || !qweight || !scales || !y) return ER_ERR_NULL;
  if (group != ER_GROUP || M < 1 || M > (1 << 20) || N < kTileN || N % kTileN != 0 || N > (1 << 24) ||
      K < ER_GROUP || K % ER_GROUP != 0 || K > (1 << 24) || ldx_elems < K || ldy_elems < N)
    return ER_ERR_SHAPE;
  if (y_dtype != ER_BF16 && y_dtype != ER_F32) return ER_ERR_DTYPE;
  if (!er::aligned16(x_bf16) || !er::aligned16(qweight) || !er::aligned16(scales) || (ldx_elems % 8) != 0)
    return ER_ERR_ALIGN;
  if (!workspace) return ER_ERR_WORKSPACE;
  if (!er::aligned16(workspace)) return ER_ERR_ALIGN;
  const int64_t Kw = planes ? 2 * K : K;           // columns of the packed matrix
  const Plan pl = make_plan(M, N, Kw);
  if ((long long)pl.tiles * pl.G >= (1ll << 31)) return ER_ERR_SHAPE;
  if (workspace_bytes < er_gemm_workspace_bytes(M, N, Kw)) return ER_ERR_WORKSPACE;
  int st = er::check_arch();
  if (st != ER_OK) return st;

  GemmParams gp;
  gp.M = (int)M; gp.N = (int)N; gp.K = (int)Kw; gp.planes = planes;
  gp.G = pl.G; gp.ntiles = pl.ntiles; gp.mchunks = pl.mchunks; gp.tiles = pl.tiles; gp.unit_groups = pl.unit_groups; gp.units = (int)pl.units;
  gp.uq = (int)(pl.units / pl.ctas); gp.ur = (int)(pl.units % pl.ctas);
  gp.split = pl.split;
  gp.cluster = pl.cluster;
  if (pl.split > 0) { gp.uq = pl.G; gp.ur = 0; }
  gp.qweight = reinterpret_cast<const uint8_t*>(qweight);
  gp.scales = reinterpret_cast<const uint8_t*>(scales);
  gp.y_f32 = (y_dtype == ER_F32); gp.ldy = ldy_elems; gp.y = y;
  gp.counters = reinterpret_cast<int*>(workspace);
  gp.partials = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(workspace) + ER_GEMM_COUNTER_BYTES);
  cudaStream_t s = (cudaStream_t)stream;
#ifdef ER_DEV
  // development library only: the pre-scaled large-batch kernel (w4a16_gemm_large.cu says why it is not shipped)
  if (!planes && M > 16 && (er::g_tune.large == 2 || (er::g_tune.large == 1 && er::large_preferred(M, N, K))))
    return er::launch_large(x_bf16, M, N, K, ldx_elems, gp, s);
#endif
  // M > 64: a batch tile of 128 rows, the weights converted once per tile (w4a16_gemm_wide.cu)
  if (M > 64) {
    const PlanAbove64 pa = plan_above_64(M, N, Kw, planes != 0);
    if (pa.wide) return er::launch_wide(x_bf16, M, N, Kw, ldx_elems, gp, pa.whole_wide, pa.split_wide, s);
  }
  // M <= 8 on a plan without a cluster (the large-N linears: gate/up): the warp-level-MMA kernel streams them faster
  // (w4a16_gemm_small.cu; measured in profiles/r02_gemm.md)
  if (!planes && M <= 8 && pl.cluster == 1 && er::g_tune.small_mma) return er::launch_small(x_bf16, M, K, ldx_elems, gp, pl, s);

  CUtensorMap mx;
  bool ok = er::make_map_2d(&mx, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, x_bf16, (uint64_t)M, (uint64_t)K,
                            (uint64_t)ldx_elems * 2, (uint32_t)pl.mpad, 64, CU_TENSOR_MAP_SWIZZLE_128B);
  if (!ok) {
    er::set_last_cuda_error((int)cudaErrorInvalidValue);
    return ER_ERR_CUDA;
  }
  if (planes) {     // the two-plane W8 instantiations (er_w8a16_gemm)
    if (pl.mpad == 16) return pl.cluster > 1 ? launch<16, true, true>(mx, gp, pl, s) : launch<16, false, true>(mx, gp, pl, s);
    if (pl.mpad == 32) return pl.cluster > 1 ? launch<32, true, true>(mx, gp, pl, s) : launch<32, false, true>(mx, gp, pl, s);
    return launch<64, false, true>(mx, gp, pl, s);
  }
  if (pl.mpad == 16) return pl.cluster > 1 ? launch<16, true>(mx, gp, pl, s) : launch<16, false>(mx, gp, pl, s);
  if (pl.mpad == 32) return pl.cluster > 1 ? launch<32, true>(mx, gp, pl, s) : launch<32, false>(mx, gp, pl, s);
  return launch<64, false>(mx, gp, pl, s);
}

int er_w4a16_gemm(const void* x_bf16, int64_t M, int64_t K, int64_t ldx_elems, const void* qweight,
                  const void* scales, int64_t N, int group, void* y, int64_t ldy_elems, int y_dtype, void* workspace,
                  size_t workspace_bytes, void* stream) {
  return gemm_impl(x_bf16, M, K, ldx_elems, qweight, scales, N, group, y, ldy_elems, y_dtype, workspace, workspace_bytes,
                   stream, 0);
}

size_t er_w8_gemm_workspace_bytes(int64_t M, int64_t N, int64_t K) { return er_gemm_workspace_bytes(M, N, 2 * K); }

int er_w8a16_gemm(const void* x_bf16, int64_t M, int64_t K, int64_t ldx_elems, const void* qweight,
                  const void* scales, int64_t N, int group, void* y, int64_t ldy_elems, int y_dtype, void* workspace,
                  size_t workspace_bytes, void* stream) {
  return gemm_impl(x_bf16, M, K, ldx_elems, qweight, scales, N, group, y, ldy_elems, y_dtype, workspace, workspace_bytes,
                   stream, 1);
}

// ---- er_w4a16_gemm_static: the M <= 16 drafter linear for callers that may not allocate (include/er.h) ----
// The tile counters and split-K partial tiles live in THIS array instead of a caller-provided workspace: 16 KiB of
// counters + 2 x 16 x 128 fp32 per CTA for up to 192 CTAs.  Every GPU that loads the library holds it until exit.  In
// host code `g_static_scratch` is only a stand-in for the symbol: its device address is asked for once per device, with
// that device current, and that pointer is what the kernel gets.
constexpr size_t kStaticScratchBytes = ER_GEMM_COUNTER_BYTES + (size_t)192 * 2 * ER_STATIC_GEMM_MAX_M * kTileN * sizeof(float);
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

int er_w4a16_gemm_static(const void* x_bf16, int64_t M, int64_t K, int64_t ldx_elems, const void* qweight,
                         const void* scales, int64_t N, int group, void* y, int64_t ldy_elems, int y_dtype,
                         void* stream) {
  if (M > ER_STATIC_GEMM_MAX_M) return ER_ERR_SHAPE;                 // beyond what the static scratch is sized for
  if (M >= 1 && N >= kTileN && N % kTileN == 0 && K >= ER_GROUP && K % ER_GROUP == 0 &&
      er_gemm_workspace_bytes(M, N, K) > kStaticScratchBytes)
    return ER_ERR_WORKSPACE;                                         // a device with more than 192 SMs
  static void* ptr[er::kMaxDevices];                                 // device address of the array, per device
  const int dev = er::current_device();
  if (dev < 0 || dev >= er::kMaxDevices) return ER_ERR_CUDA;
  if (!ptr[dev]) {
    void* q = nullptr;
    ER_CUDA_TRY(cudaGetSymbolAddress(&q, g_static_scratch));
    if (!q) return ER_ERR_CUDA;
    ptr[dev] = q;
  }
  // The array keeps the last call's contents.  The partial tiles are always written before they are read; the counters
  // must start at zero: a completed call leaves them so, this memset covers a call that did not complete.
  ER_CUDA_TRY(cudaMemsetAsync(ptr[dev], 0, ER_GEMM_COUNTER_BYTES, (cudaStream_t)stream));
  return gemm_impl(x_bf16, M, K, ldx_elems, qweight, scales, N, group, y, ldy_elems, y_dtype, ptr[dev],
                   kStaticScratchBytes, stream, 0);
}

}  // extern "C"
