// w4a16_gemm_small.cu -- er_w4a16_gemm at M <= 8 on plans without a thread-block cluster (the large-N linears, e.g.
// gate/up): the most memory-bound corner of the weight-quantized self-drafter ("weight loading dominates"
// small-batch decode; L175 W4A16 weight-only kernel; L467 "on-the-fly dequantization and kernel-level overhead" is
// what eta_D pays on top of the bytes).
//
// What bounds this regime on sm_100a is not the contraction (2 * 8 * 128 * 128 flop per 8 KiB of weights) but the
// nibble -> bf16 conversion -- 7 half-rate logic-pipe operations per packed word = 224 ALU cycles per [128 rows x 128
// k] block and SM sub-partition against 370 cycles of HBM time -- and whatever the warps have to wait for.  The
// tcgen05 kernel (w4a16_gemm.cu) needs a CTA-wide rendezvous per 128-k group twice (all 128 rows of the A operand in
// TENSOR MEMORY before the MMA, the accumulator read back after it for the exact per-group scale).  Here every warp
// is on its own; measured on gate/up at M <= 8: 16.9 us against 18.5-19.0 us (profiles/r02_gemm.md, which also has
// the experiments behind every choice below).
//
//   persistent   one CTA per SM; the (tile, 128-k group) units are dealt out as one contiguous range per CTA
//                (stream-K / tile split, w4a16_plan.cuh), as in the tcgen05 kernel.
//   two rings    packed weights (8 KiB stages, up to 20) and X + scales + x sums (3 KiB stages, 10).  A weight stage
//                is handed back as soon as its words sit in registers, at the START of a group's contraction, so the
//                weight ring is almost entirely bytes in flight.
//   warp 20      weight producer: one 8 KiB 1-D bulk copy per group (ER_PACK_V2 keeps the block contiguous and
//                pre-swizzled).  (Letting it start BEFORE griddepcontrol.wait -- the weights never depend on the
//                previous GEMM -- was measured and buys nothing: with one CTA per SM this kernel's CTAs only become
//                resident when the previous kernel's exit; a half-SM variant that does co-reside lost more in the
//                main loop than it gained.  So the usual stream order holds for every operand.)
//   warps 21-25  one X warp per worker set: loads the X boxes and the scales of the set's groups and, when they have
//                landed, sums x[m][k] over the group's 128 k with the tensor cores (A = ones) -- the 136 * sum that
//                the stored nibble's offset adds to every output of the group (one helper warp for all groups was the
//                bottleneck of an earlier version: ~350 cycles of dependent latency per group).
//   warps 0-19   five sets of four warps; set j takes the groups j, j + 5, ... of the CTA's range.  A warp owns 32
//                weight rows of the group (two 16-row blocks) and all 128 k: 4 x LDS.128 of packed words, nibble
//                -> bf16 in registers ((w >> 4t) & 0x000F000F | 0x43004300 = 128 + u), and mma.sync.m16n8k16 (bf16 x
//                bf16 -> fp32) with the weights as the A fragment and X as the B fragment: the swap-AB of the tcgen05
//                kernel at warp level.  The k index of an MMA is only a label: thread t of a quad takes the k = 32 t
//                .. 32 t + 31 of a row, i.e. exactly one 16-byte chunk of ER_PACK_V2, and reads the matching 64 bytes
//                of X.  The group's fp32 sum, minus 136 * sum x, is multiplied by the group scale and added to the
//                running sum (no rounding of q * s).  No warp waits for another one inside the main loop.
//   output       at the end of a tile segment the five sets add their sums in set order through one shared-memory
//                tile; whole tiles are stored directly, partial ones go through the workspace (ticket per tile,
//                ascending CTA order).  Deterministic.
#include "w4a16_plan.cuh"

namespace {

using namespace er;

constexpr int kSets = 5;
constexpr int kSetWarps = 4;
constexpr int kSetThreads = kSetWarps * 32;          // 128
constexpr int kWorkerWarps = kSets * kSetWarps;      // 20
constexpr int kProdWarp = kWorkerWarps;              // 20: the weight producer; warps 21 .. 25: one X warp per set
constexpr int kThreads = (kWorkerWarps + 1 + kSets) * 32;   // 832
constexpr int kXStages = 10;                         // ring of X / scale stages: two per set
constexpr int kMaxWStages = 20;                      // ring of packed-weight stages: as deep as shared memory allows
constexpr int kPrefetchGroups = 12;                  // 96 KB of weights asked from L2 before griddepcontrol.wait
constexpr int kRedLd = 132;                          // row pitch of the shared reduction tile (bank-conflict free)

template <int MB>
struct SCfg {
  static constexpr int MPAD = 8 * MB;
  // TWO rings.  A packed-weight stage (8 KiB) is handed back as soon as its words sit in registers, at the START of
  // a group's contraction, so that nearly the whole weight ring is bytes in flight: the HBM stream needs about 100
  // KB outstanding per SM (6.4 TB/s x 2.3 us / 148), and a single ring whose stages stay occupied until the group is
  // contracted never gets there.  X, the scales and the x sums of a group live in the small second ring until the
  // group is finished.
  // X of a group: k 0..63 as a box of MPAD rows, k 64..127 as a box of MPAD + 2 rows that starts two rows EARLIER
  // (rows -2, -1 are out of bounds and arrive as zeros): the 128-byte swizzle then differs between the boxes by 2,
  // and the eight lanes of a quarter-warp (rows g, g + 1, four 64-byte column blocks) hit eight different 16-byte
  // bank groups.
  static constexpr int kX0Bytes = MPAD * 128;
  static constexpr int kX1Bytes = (MPAD + 2) * 128;
  static constexpr int kOffX0 = 0;
  static constexpr int kOffX1 = kX0Bytes;                       // MPAD * 128 is a multiple of 1024
  static constexpr int kOffScale = kOffX1 + kX1Bytes;
  static constexpr int kOffXs = kOffScale + kScaleBytes;        // fp32 [MPAD]: sum over the group's 128 k of x[m][k]
  static constexpr int kXStageBytes = ((kOffXs + MPAD * 4 + 1023) / 1024) * 1024;
  static constexpr uint32_t kXTxBytes = kX0Bytes + kX1Bytes + kScaleBytes;
  static constexpr int kRedBytes = MPAD * kRedLd * 4;
  static constexpr int kFixed = kXStages * kXStageBytes + kRedBytes + 1024 /*align slack*/ + 1024 /*barriers*/;
  static constexpr int kWStagesRaw = (kSmemLimit - kFixed) / kWBytes;
  // a multiple of kSets (like kXStages): a stage is then always read by the same set, whose waits on its phases are
  // in program order
  static constexpr int kWStages = (kWStagesRaw > kMaxWStages ? kMaxWStages : kWStagesRaw) / kSets * kSets;
  static constexpr int kSmem = kWStages * kWBytes + kFixed;
  static_assert(kX0Bytes % 1024 == 0, "box alignment");
  static_assert(kWStages >= 2 * kSets && kXStages % kSets == 0, "rings");
};

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
__device__ __forceinline__ void named_bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void named_bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// One packed word (nibble positions (t, t + 4) hold the consecutive pair k = 8 j + 2 t, + 1) -> 4 registers of bf16
// pairs (128 + u, 128 + u'): (w >> 4t) & 0x000F000F | 0x43004300, i.e. 3 shifts + 4 lop3 on the half-rate logic pipe.
// The stored nibble is u = q + 8, so the MMA contracts q + 136; the 136 * sum_k x[m][k] that this adds to every
// output of a group is removed on the fp32 sum (a packed bf16 fma per register here would run on the datapath the
// MMAs use: measured + 20 % on the whole loop).
__device__ __forceinline__ void dequant_word(uint32_t w, uint32_t* a) {
#pragma unroll
  for (int t = 0; t < 4; ++t)
    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(a[t]) : "r"(w >> (4 * t)), "r"(0x000F000Fu), "r"(0x43004300u));
}

// D += A (16 x 16, row) * B (16 x 8, col), bf16 x bf16 -> fp32
__device__ __forceinline__ void mma16816(float* c, uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0,
                                         uint32_t b1) {
  asm("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}

template <int MB>
__global__ void __launch_bounds__(kThreads, 1)
w4a16_small_kernel(const __grid_constant__ CUtensorMap map_x0, const __grid_constant__ CUtensorMap map_x1,
                   const GemmParams p) {
  using C = SCfg<MB>;
  constexpr int SW = C::kWStages, SX = kXStages;
  constexpr int MPAD = C::MPAD;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* xring = smem + SW * kWBytes;                                          // [SX] X / scale / x-sum stages
  float* red = reinterpret_cast<float*>(xring + SX * C::kXStageBytes);           // [MPAD][kRedLd]
  uint64_t* bars = reinterpret_cast<uint64_t*>(reinterpret_cast<uint8_t*>(red) + C::kRedBytes);
  uint64_t* wfull = bars;                       // [SW] packed weights landed
  uint64_t* wempty = wfull + kMaxWStages;       // [SW] the four warps of the group's set hold the words in registers
  uint64_t* xfull = wempty + kMaxWStages;       // [SX] X and scales landed
  uint64_t* xs_full = xfull + kXStages;         // [SX] the helpers have written the group's x sums
  uint64_t* xempty = xs_full + kXStages;        // [SX] the set and the helpers are done with the stage
  int* last_flag = reinterpret_cast<int*>(xempty + kXStages);

  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);   // provably warp-uniform
  const int lane = threadIdx.x & 31;
  const int cta = blockIdx.x;
  const int ug = p.unit_groups;
  const int gb = range_begin(p.uq, p.ur, p.split, cta) * ug;        // first global group index of this CTA
  const int ge = range_begin(p.uq, p.ur, p.split, cta + 1) * ug;
  const int n_it = ge - gb;

  if (warp == kProdWarp) {
    if (lane < SW) {
      mbar_init(&wfull[lane], 1);
      mbar_init(&wempty[lane], kSetWarps);
    }
    if (lane < SX) {
      mbar_init(&xfull[lane], 1);
      mbar_init(&xs_full[lane], 1);
      mbar_init(&xempty[lane], kSetWarps + 1);
    }
    mbar_fence_init();
    if (lane == 0) {
      tma_prefetch_desc(&map_x0);
      tma_prefetch_desc(&map_x1);
    }
    named_bar_arrive(15, kThreads);   // the producer goes straight on to its first loads
  } else {
    named_bar_sync(15, kThreads);     // the barriers are initialised
  }
  // Programmatic dependent launch: the prologue above touched no global memory and may overlap the tail of the
  // previous kernel in the stream; from here on its results (X, the workspace) are needed.  The next kernel may be
  // scheduled as soon as SMs free up (it waits at its own griddepcontrol.wait).
  // ... except that the weight producer first asks L2 for the beginning of this CTA's weight stream (a contiguous
  // byte range of ER_PACK_V2): that hides part of the first DRAM round trip under the previous kernel's tail, and it is
  // safe even right behind a refresh -- L2 is the point of coherence, a prefetched line cannot be stale.
  if (warp == kProdWarp && elect_one()) {
    const int npf = n_it < kPrefetchGroups ? n_it : kPrefetchGroups;
    bulk_prefetch_l2(p.qweight + (size_t)gb * kWBytes, (uint32_t)npf * kWBytes);
  }
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  float tot[2][MB][4];                  // a worker's running sums [row block][n8 block][fragment element]

  if (warp == kProdWarp) {
    // ===================== weight producer (warp-uniform; one elected lane issues) =====================
    int g = gb % p.G, tn = (gb / p.G) % p.ntiles;
    int s = 0;
    uint32_t ph = 0;
    for (int it = 0; it < n_it; ++it) {
      mbar_wait(&wempty[s], ph ^ 1);     // the stage's previous group (it - SW) sits in registers
      if (elect_one()) {
        mbar_arrive_expect_tx(&wfull[s], kWBytes);
        // ER_PACK_V2: the [128 rows x 128 k] block of (tile, g) is 8 KiB of contiguous, pre-swizzled bytes
        bulk_load_1d(smem + s * kWBytes, p.qweight + ((size_t)tn * p.G + g) * kWBytes, kWBytes, &wfull[s], kEvictFirst);
      }
      __syncwarp();
      if (++g == p.G) {
        g = 0;
        if (++tn == p.ntiles) tn = 0;
      }
      if (++s == SW) { s = 0; ph ^= 1; }
    }
  } else if (warp > kProdWarp) {
    // ===================== X warps: warp kProdWarp + 1 + j serves worker set j -- it loads X and the scales of the
    // set's groups (two TMA boxes + 256 bytes, kXStages / kSets stages ahead) and, once they have landed, sums x[m][k]
    // over the group's 128 k for every batch row with the tensor cores (A = ones: every row of the product is that
    // sum, in fp32): the 136 * sum the stored nibble's offset adds to every output of the group =====================
    const int j = warp - kProdWarp - 1;
    if (j < kSets) {
      const int g = lane >> 2, t = lane & 3;
      const uint32_t sbase = smem_u32(xring);
      const int xsw = (t < 2) ? g : ((g + 2) & 7);
      const uint32_t xrow = sbase + ((t < 2) ? (C::kOffX0 + g * 128) : (C::kOffX1 + (g + 2) * 128));
      const int q0 = ((t & 1) * 4) ^ xsw;
      // issue side: group `iss` of the CTA's range = (tile tn_i, group g_i), into stage isl
      int iss = j, isl = j;
      uint32_t iph = 0;
      int g_i = (gb + j) % p.G, tn_i = ((gb + j) / p.G) % p.ntiles;
      auto issue = [&]() {
        mbar_wait(&xempty[isl], iph ^ 1);  // the set (and this warp) are done with the stage's previous group
        if (elect_one()) {
          uint8_t* st = xring + isl * C::kXStageBytes;
          mbar_arrive_expect_tx(&xfull[isl], C::kXTxBytes);
          tma_load_2d(st + C::kOffX0, &map_x0, &xfull[isl], g_i * 128, 0, kEvictLast);
          tma_load_2d(st + C::kOffX1, &map_x1, &xfull[isl], g_i * 128 + 64, -2, kEvictLast);
          bulk_load_1d(st + C::kOffScale, p.scales + ((size_t)g_i * p.N + tn_i * kTileN) * 2, kScaleBytes, &xfull[isl],
                       kEvictFirst);
        }
        __syncwarp();
        iss += kSets;
        isl += kSets;
        if (isl >= SX) { isl -= SX; iph ^= 1; }
        g_i += kSets;
        while (g_i >= p.G) {
          g_i -= p.G;
          if (++tn_i == p.ntiles) tn_i = 0;
        }
      };
#pragma unroll 1
      for (int d = 0; d < SX / kSets && iss < n_it; ++d) issue();
      int psl = j;
      uint32_t pph = 0;
      for (int prc = j; prc < n_it; prc += kSets) {
        mbar_wait(&xfull[psl], pph);
        const uint32_t st = psl * C::kXStageBytes;
        constexpr uint32_t one2 = 0x3F803F80u;
#pragma unroll
        for (int nb = 0; nb < MB; ++nb) {
          float c0[4] = {0.f, 0.f, 0.f, 0.f}, c1[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const uint4 xb = lds128(st + xrow + nb * 1024 + ((q0 ^ i) << 4));
            mma16816(c0, one2, one2, one2, one2, xb.x, xb.y);
            mma16816(c1, one2, one2, one2, one2, xb.z, xb.w);
          }
          if (g == 0)
            asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(sbase + st + C::kOffXs + (8 * nb + 2 * t) * 4),
                         "f"(c0[0] + c1[0]), "f"(c0[1] + c1[1]) : "memory");
        }
        __syncwarp();
        if (lane == 0) {
          mbar_arrive(&xs_full[psl]);
          mbar_arrive(&xempty[psl]);
        }
        psl += kSets;
        if (psl >= SX) { psl -= SX; pph ^= 1; }
        if (iss < n_it) issue();
      }
    }
  } else {
    // ===================== worker sets =====================
    const int set = warp >> 2;             // groups set, set + kSets, ... of the CTA's range
    const int wq = warp & 3;               // rows 32 wq .. 32 wq + 31 of the tile
    const int g = lane >> 2, t = lane & 3; // MMA fragment coordinates
    const uint32_t wbase = smem_u32(smem), xbase = smem_u32(xring);
    // packed words: row r = 32 wq + 16 rb + 8 h + g keeps its 64 bytes at r * 64, its logical 16-byte chunk t (k = 32 t
    // .. 32 t + 31) sits at chunk t ^ ((r >> 1) & 3) -- the same for the four rows of this thread
    const uint32_t w_off = wbase + (32 * wq + g) * 64 + ((t ^ ((g >> 1) & 3)) << 4);
    const uint32_t sc_off = xbase + C::kOffScale + (32 * wq + g) * 2;
    // X: batch row m = 8 nb + g, bytes 64 t .. 64 t + 63 of its 256: box (t >> 1), 16-byte chunk (t & 1) * 4 + i,
    // swizzled with the row's position in its box (box 1 starts two rows early)
    const int xs = (t < 2) ? g : ((g + 2) & 7);
    const uint32_t xrow = xbase + ((t < 2) ? (C::kOffX0 + g * 128) : (C::kOffX1 + (g + 2) * 128));
    const int q0 = ((t & 1) * 4) ^ xs;
    // loop invariants, pinned in registers (otherwise the compiler rematerialises this arithmetic in every iteration,
    // on the logic pipe the conversion needs)
    uint32_t xo[4], w_addr, sc_addr, xs_addr, wfull_addr, wempty_addr, xfull_addr, xempty_addr, xsf_addr;
#pragma unroll
    for (int i = 0; i < 4; ++i) asm volatile("mov.u32 %0, %1;" : "=r"(xo[i]) : "r"(xrow + ((q0 ^ i) << 4)));
    asm volatile("mov.u32 %0, %1;" : "=r"(w_addr) : "r"(w_off));
    asm volatile("mov.u32 %0, %1;" : "=r"(sc_addr) : "r"(sc_off));
    asm volatile("mov.u32 %0, %1;" : "=r"(xs_addr) : "r"(xbase + C::kOffXs + 8 * t));
    asm volatile("mov.u32 %0, %1;" : "=r"(wfull_addr) : "r"(smem_u32(wfull)));
    asm volatile("mov.u32 %0, %1;" : "=r"(wempty_addr) : "r"(smem_u32(wempty)));
    asm volatile("mov.u32 %0, %1;" : "=r"(xfull_addr) : "r"(smem_u32(xfull)));
    asm volatile("mov.u32 %0, %1;" : "=r"(xempty_addr) : "r"(smem_u32(xempty)));
    asm volatile("mov.u32 %0, %1;" : "=r"(xsf_addr) : "r"(smem_u32(xs_full)));
    uint32_t rt_zero;                      // 0 at run time (M < 2^20), unknown at compile time
    asm volatile("mov.u32 %0, %1;" : "=r"(rt_zero) : "r"((uint32_t)p.M >> 24));
    const bool last_set = (set == kSets - 1);
    const bool leader = (threadIdx.x == (kSets - 1) * kSetThreads);

    int my = set;                          // this set's next group (index into the CTA's range)
    int ws = set, xs_i = set;              // its weight / X stage (kSets <= SX <= SW) ...
    uint32_t wph = 0, xph = 0;             // ... and the parities of wfull[ws] / xfull[xs_i]
    int it = 0, seg = 0;
    int pend_tile[2] = {-1, -1};           // partial tiles of this CTA (head / tail segment of its range)

    // element e = (rb, nb, j) of a thread's sums: weight row and batch row
    auto row_of = [&](int rb, int j) { return 32 * wq + 16 * rb + g + 8 * (j >> 1); };
    auto m_of = [&](int nb, int j) { return 8 * nb + 2 * t + (j & 1); };
    auto store_tile = [&](int tile, const float (&v)[2][MB][4]) {
      const int n0 = tile * kTileN;
#pragma unroll
      for (int rb = 0; rb < 2; ++rb)
#pragma unroll
        for (int nb = 0; nb < MB; ++nb)
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const int m = m_of(nb, j);
            if (m < p.M) {
              const size_t idx = (size_t)m * p.ldy + n0 + row_of(rb, j);
              if (p.y_f32) reinterpret_cast<float*>(p.y)[idx] = v[rb][nb][j];
              else reinterpret_cast<__nv_bfloat16*>(p.y)[idx] = __float2bfloat16_rn(v[rb][nb][j]);
            }
          }
    };

    while (it < n_it) {
      // ---- segment = the part of one tile inside this CTA's range ----
      const int gi0 = gb + it;
      const int tile = gi0 / p.G, g_lo = gi0 % p.G;
      const int seg_len = min(p.G - g_lo, n_it - it);
      const int it_end = it + seg_len;
      const bool last_seg = (it_end == n_it);
#pragma unroll
      for (int rb = 0; rb < 2; ++rb)
#pragma unroll
        for (int nb = 0; nb < MB; ++nb)
#pragma unroll
          for (int j = 0; j < 4; ++j) tot[rb][nb][j] = 0.f;

      for (; my < it_end; my += kSets) {
        mbar_wait_addr(wfull_addr + ws * 8, wph);
        uint32_t w[2][2][4];                 // [row block][row g / g + 8][word i]: k = 32 t + 8 i .. + 7
#pragma unroll
        for (int rb = 0; rb < 2; ++rb)
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const uint4 v = lds128(ws * kWBytes + w_addr + rb * 1024 + h * 512);
            w[rb][h][0] = v.x; w[rb][h][1] = v.y; w[rb][h][2] = v.z; w[rb][h][3] = v.w;
          }
        mbar_wait_addr(xfull_addr + xs_i * 8, xph);
        const uint32_t st = xs_i * C::kXStageBytes;
        uint32_t sc16[2][2];
#pragma unroll
        for (int rb = 0; rb < 2; ++rb)
#pragma unroll
          for (int h = 0; h < 2; ++h) sc16[rb][h] = lds_u16(st + sc_addr + rb * 32 + h * 16);
        float c[2][MB][4];
#pragma unroll
        for (int rb = 0; rb < 2; ++rb)
#pragma unroll
          for (int nb = 0; nb < MB; ++nb)
#pragma unroll
            for (int j = 0; j < 4; ++j) c[rb][nb][j] = 0.f;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          uint4 xb[MB];                      // X[m][32 t + 8 i .. + 7]: B fragments of the MMA steps 2 i and 2 i + 1
#pragma unroll
          for (int nb = 0; nb < MB; ++nb) xb[nb] = lds128(st + xo[i] + nb * 1024);
          uint32_t a[2][2][4];
#pragma unroll
          for (int rb = 0; rb < 2; ++rb)
#pragma unroll
            for (int h = 0; h < 2; ++h) dequant_word(w[rb][h][i], a[rb][h]);
          if (i == 0) {
            // The packed words are in registers: hand the weight stage back.  The arrive must not issue before the
            // four LDS.128 have returned, so its address is made to depend on one register of each (two lop3 whose
            // result is zero, which the assembler cannot know).
            uint32_t dep;
            asm volatile("lop3.b32 %0, %1, %2, %3, 0x80;" : "=r"(dep) : "r"(w[0][0][3]), "r"(w[0][1][3]), "r"(w[1][0][3]));
            asm volatile("lop3.b32 %0, %1, %2, %3, 0x80;" : "=r"(dep) : "r"(dep), "r"(w[1][1][3]), "r"(rt_zero));
            __syncwarp();
            if (lane == 0) mbar_arrive_addr(wempty_addr + ws * 8 + dep);
          }
#pragma unroll
          for (int rb = 0; rb < 2; ++rb)
#pragma unroll
            for (int nb = 0; nb < MB; ++nb)
              mma16816(c[rb][nb], a[rb][0][0], a[rb][1][0], a[rb][0][1], a[rb][1][1], xb[nb].x, xb[nb].y);
#pragma unroll
          for (int rb = 0; rb < 2; ++rb)
#pragma unroll
            for (int nb = 0; nb < MB; ++nb)
              mma16816(c[rb][nb], a[rb][0][2], a[rb][1][2], a[rb][0][3], a[rb][1][3], xb[nb].z, xb[nb].w);
        }
        // the helpers' sums of x over this group (they had the whole conversion to get there)
        mbar_wait_addr(xsf_addr + xs_i * 8, xph);
        float xsum[MB][2];
#pragma unroll
        for (int nb = 0; nb < MB; ++nb)
          asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(xsum[nb][0]), "=f"(xsum[nb][1]) : "r"(st + xs_addr + nb * 32));
        // the group's exact scale on the fp32 sum, the nibble offset removed: s * (c - 136 * sum_k x)
#pragma unroll
        for (int rb = 0; rb < 2; ++rb) {
          const float s0 = __uint_as_float(sc16[rb][0] << 16), s1 = __uint_as_float(sc16[rb][1] << 16);
#pragma unroll
          for (int nb = 0; nb < MB; ++nb) {
            tot[rb][nb][0] = fmaf(s0, fmaf(-136.f, xsum[nb][0], c[rb][nb][0]), tot[rb][nb][0]);
            tot[rb][nb][1] = fmaf(s0, fmaf(-136.f, xsum[nb][1], c[rb][nb][1]), tot[rb][nb][1]);
            tot[rb][nb][2] = fmaf(s1, fmaf(-136.f, xsum[nb][0], c[rb][nb][2]), tot[rb][nb][2]);
            tot[rb][nb][3] = fmaf(s1, fmaf(-136.f, xsum[nb][1], c[rb][nb][3]), tot[rb][nb][3]);
          }
        }
        // every shared-memory read of the stage has returned (the arithmetic above consumed them): hand it back
        __syncwarp();
        if (lane == 0) mbar_arrive_addr(xempty_addr + xs_i * 8);
        ws += kSets;
        if (ws >= SW) { ws -= SW; wph ^= 1; }
        xs_i += kSets;
        if (xs_i >= SX) { xs_i -= SX; xph ^= 1; }
      }

      // ---- the sets add their sums in set order through the shared tile: set 0 writes, sets 1 .. kSets-2 add, the last
      //      set ends with the total in registers.  Barrier k (1 .. kSets-1) hands the tile from set k-1 to set k,
      //      barrier kSets hands it back to set 0 for the next segment. ----
      if (set == 0) {
        if (seg > 0) named_bar_sync(kSets, 2 * kSetThreads);
      } else {
        named_bar_sync(set, 2 * kSetThreads);
      }
#pragma unroll
      for (int rb = 0; rb < 2; ++rb)
#pragma unroll
        for (int nb = 0; nb < MB; ++nb)
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            float* q = red + m_of(nb, j) * kRedLd + row_of(rb, j);
            if (set > 0) tot[rb][nb][j] += *q;
            if (!last_set) *q = tot[rb][nb][j];
          }
      if (!last_set) {
        named_bar_arrive(set + 1, 2 * kSetThreads);
      } else {
        if (!last_seg) named_bar_arrive(kSets, 2 * kSetThreads);
        // ---- output: a whole tile is stored directly; a partial one goes to the workspace as fp32 and is finished
        //      after the main loop, or (cluster mode) is reduced over the cluster at the end of the kernel ----
        if (seg_len == p.G) {
          store_tile(tile, tot);
        } else {
          const int k = (it == 0 ? 0 : 1);
          float* mine = p.partials + ((size_t)cta * 2 + k) * (MPAD * kTileN);
#pragma unroll
          for (int rb = 0; rb < 2; ++rb)
#pragma unroll
            for (int nb = 0; nb < MB; ++nb)
#pragma unroll
              for (int j = 0; j < 4; ++j)
                if (m_of(nb, j) < p.M) __stcg(mine + m_of(nb, j) * kTileN + row_of(rb, j), tot[rb][nb][j]);
          pend_tile[k] = tile;
        }
      }
      it = it_end;
      ++seg;
    }

    // ---- partial tiles: ticket per tile; the last CTA to arrive adds all partials in ascending CTA order ----
    // Ordering: partial stores (all threads of the last set) -> bar.sync -> the leader's acq_rel ticket (release is
    // cumulative over what the barrier made visible to the leader); last arriver: acq_rel ticket -> bar.sync ->
    // ld.cg of the others' partials.
    if (last_set && (pend_tile[0] >= 0 || pend_tile[1] >= 0)) {
      named_bar_sync(kSets + 1, kSetThreads);
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
      named_bar_sync(kSets + 1, kSetThreads);
      constexpr int kChunk = 4;   // contributors whose loads are in flight together
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        if (pend_tile[k] < 0 || last_flag[k] == 0) continue;
        const int tile = pend_tile[k];
#pragma unroll
        for (int rb = 0; rb < 2; ++rb)
#pragma unroll
          for (int nb = 0; nb < MB; ++nb)
#pragma unroll
            for (int j = 0; j < 4; ++j) tot[rb][nb][j] = 0.f;
        for (int c0 = c_lo[k]; c0 <= c_hi[k]; c0 += kChunk) {
          float v[kChunk][2][MB][4];
#pragma unroll
          for (int q = 0; q < kChunk; ++q) {
            const int c = min(c0 + q, c_hi[k]);
            // CTA c's piece of this tile is its first segment iff its range starts inside the tile
            const int cb = range_begin(p.uq, p.ur, p.split, c) * ug;
            const int which = (cb >= tile * p.G) ? 0 : 1;
            const float* src = p.partials + ((size_t)c * 2 + which) * (MPAD * kTileN);
#pragma unroll
            for (int rb = 0; rb < 2; ++rb)
#pragma unroll
              for (int nb = 0; nb < MB; ++nb)
#pragma unroll
                for (int j = 0; j < 4; ++j)
                  v[q][rb][nb][j] = (m_of(nb, j) < p.M && c0 + q <= c_hi[k])
                                        ? __ldcg(src + m_of(nb, j) * kTileN + row_of(rb, j)) : 0.f;
          }
#pragma unroll
          for (int q = 0; q < kChunk; ++q)
#pragma unroll
            for (int rb = 0; rb < 2; ++rb)
#pragma unroll
              for (int nb = 0; nb < MB; ++nb)
#pragma unroll
                for (int j = 0; j < 4; ++j)
                  if (c0 + q <= c_hi[k]) tot[rb][nb][j] += v[q][rb][nb][j];
        }
        store_tile(tile, tot);
      }
    }
  }

}

template <int MB>
int launch(const CUtensorMap& m0, const CUtensorMap& m1, const GemmParams& gp, const Plan& pl, cudaStream_t stream) {
  static bool attr_set[er::kMaxDevices] = {};
  const int dev = er::current_device();
  if (dev < 0 || dev >= er::kMaxDevices || !attr_set[dev]) {
    ER_CUDA_TRY(cudaFuncSetAttribute(w4a16_small_kernel<MB>, cudaFuncAttributeMaxDynamicSharedMemorySize, SCfg<MB>::kSmem));
    if (dev >= 0 && dev < er::kMaxDevices) attr_set[dev] = true;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)pl.ctas);
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = SCfg<MB>::kSmem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = er::g_tune.pdl;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  ER_CUDA_TRY(cudaLaunchKernelEx(&cfg, w4a16_small_kernel<MB>, m0, m1, gp));
  return ER_OK;
}

}  // namespace

namespace er {

// M <= 8, plans without a thread-block cluster (the large-N linears): see er_w4a16_gemm in w4a16_gemm.cu
int launch_small(const void* x, int64_t M, int64_t K, int64_t ldx, GemmParams gp, const Plan& pl, cudaStream_t stream) {
  if (M > 8 || pl.cluster > 1) return ER_ERR_SHAPE;
  CUtensorMap m0, m1;
  const bool ok = make_map_2d(&m0, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, x, (uint64_t)M, (uint64_t)K, (uint64_t)ldx * 2, 8,
                              64, CU_TENSOR_MAP_SWIZZLE_128B) &&
                  make_map_2d(&m1, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, x, (uint64_t)M, (uint64_t)K, (uint64_t)ldx * 2, 10,
                              64, CU_TENSOR_MAP_SWIZZLE_128B);
  if (!ok) {
    set_last_cuda_error((int)cudaErrorInvalidValue);
    return ER_ERR_CUDA;
  }
  return launch<1>(m0, m1, gp, pl, stream);
}

}  // namespace er
