// w4a16_gemm_wide.cu -- er_w4a16_gemm at M > 64: the exact per-group arithmetic of w4a16_gemm.cu (a fresh fp32 accumulator
// per 128-k group, the fp32 group scale applied to it, q * s never rounded) with a batch tile of 128 rows, so that a weight
// tile is converted ONCE per 128 batch rows instead of once per 64 (the conversion, not the tensor pipe, bounds the
// narrower kernel there).  What makes 128 accumulator columns fit: ONE worker set of 16 warps -- a thread converts a
// QUARTER of a weight row per group (one LDS.128 = 32 k) and owns a quarter of the batch columns of the accumulator (32
// fp32 registers, as in the 64-row kernel) -- with two (A operand, accumulator) pairs in TENSOR MEMORY, so the set
// converts group i + 1 while the MMAs of group i run and reads group i - 1 back.  No cross-set hand-off is left.
//
//   persistent   one CTA per SM over (tile, 128-k group) units as in w4a16_plan.cuh; tile = (chunk of 128 batch rows,
//                128 weight rows); whole tiles where they keep the CTAs busy, else stream-K ranges whose partial tiles go
//                through the workspace (ticket per tile, ascending CTA order).  Deterministic.
//   warps 0-15   workers: warp w converts k-quarter (w >> 2) of the rows of lane quarter (w & 3) and reads back batch
//                columns 32 (w >> 2) ... + 31 of those rows
//   warp 16      producer: 8 KiB bulk copy of the packed block + 256 B of scales + two SWIZZLE_128B boxes of X
//                [128 x 64 k] per group into a ring of 5 stages
//   warps 17-18  MMA issuers (even / odd groups): 8 x tcgen05.mma.kind::f16 (M = 128, N = 128, K = 16) per group, A
//                from TENSOR MEMORY, B = X from shared memory, a fresh accumulator per group
#include "w4a16_plan.cuh"

namespace {

using namespace er;

constexpr int kMP = 128;                     // batch rows per tile
constexpr int kWorkerWarps = 16;
constexpr int kWorkerThreads = kWorkerWarps * 32;
constexpr int kProdWarp = kWorkerWarps;      // 16
constexpr int kMmaWarp0 = kProdWarp + 1;     // 17, 18
constexpr int kThreads = (kMmaWarp0 + 2) * 32;   // 608
constexpr int kCW = kMP / 4;                 // accumulator columns per thread
constexpr int kXBytes = kMP * 128 * 2;       // two boxes of [128 x 64] bf16
constexpr int kStageBytes = ((kWBytes + kXBytes + kScaleBytes + 1023) / 1024) * 1024;
constexpr int kStages = 5;
constexpr int kSmem = kStages * kStageBytes + 1024 /*align slack*/ + 512 /*barriers*/;
constexpr uint32_t kTxBytes = kWBytes + kXBytes + kScaleBytes;
constexpr int kTmemCols = 512;
constexpr int kTmemA = 0;                    // two A operands of 64 columns
constexpr int kTmemD = 128;                  // two accumulators of 128 columns
static_assert(kSmem <= kSmemLimit, "shared memory");

#define ERW_TMEM_ST16(taddr, r)                                                                                \
  asm volatile(                                                                                                \
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" \
      ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),     \
      "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])             \
      : "memory")

#define ERW_TMEM_LD16(taddr, r, o)                                                                             \
  asm volatile(                                                                                                \
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];" \
      : "=r"(r[o + 0]), "=r"(r[o + 1]), "=r"(r[o + 2]), "=r"(r[o + 3]), "=r"(r[o + 4]), "=r"(r[o + 5]),        \
        "=r"(r[o + 6]), "=r"(r[o + 7]), "=r"(r[o + 8]), "=r"(r[o + 9]), "=r"(r[o + 10]), "=r"(r[o + 11]),      \
        "=r"(r[o + 12]), "=r"(r[o + 13]), "=r"(r[o + 14]), "=r"(r[o + 15])                                     \
      : "r"(taddr)                                                                                             \
      : "memory")

// One packed word -> 4 registers of bf16 pairs (q, q'): (w >> 4t) & 0x000F000F | 0x43004300 = (128 + u, 128 + u'), then
// one packed fma removes the 136 exactly (u = q + 8).
__device__ __forceinline__ void dequant_word(uint32_t w, uint32_t* a, uint32_t off2) {
#pragma unroll
  for (int t = 0; t < 4; ++t) {
    uint32_t v;
    asm("lop3.b32 %0, %1, %2, %3, 0xEA;" : "=r"(v) : "r"(w >> (4 * t)), "r"(0x000F000Fu), "r"(0x43004300u));
    asm("fma.rn.bf16x2 %0, %1, %2, %3;" : "=r"(a[t]) : "r"(v), "r"(0x3F803F80u), "r"(off2));
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
__device__ __forceinline__ void named_bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }

__device__ __forceinline__ void named_bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

// kPlanes: the two-plane W8 instantiation (er_w8a16_gemm; w4a16_gemm.cu): groups 2g, 2g + 1 of the packed matrix contract
// the same 128 columns of X; the high-nibble plane (even groups; G is even) takes -136 per widened nibble, the low one -128.
template <bool kPlanes>
__global__ void __launch_bounds__(kThreads, 1)
w4a16_wide_kernel(const __grid_constant__ CUtensorMap map_x, const GemmParams p) {
  constexpr int S = kStages;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + S * kStageBytes);
  uint64_t* full = bars;                        // [S] TMA landed
  uint64_t* empty = bars + 8;                   // [S] the group's MMAs completed: the stage may be refilled
  uint64_t* a_full = bars + 16;                 // [2] the A operand is written, its accumulator drained
  uint64_t* done = bars + 18;                   // [2] the MMAs completed: accumulator readable, A free
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 20);
  int* last_flag = reinterpret_cast<int*>(tmem_slot + 1);

  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
  const int lane = threadIdx.x & 31;
  const int cta = blockIdx.x;
  const int ug = p.unit_groups;
  const int gb = range_begin(p.uq, p.ur, p.split, cta) * ug;        // first global group index of this CTA
  const int ge = range_begin(p.uq, p.ur, p.split, cta + 1) * ug;
  const int n_it = ge - gb;

  if (warp == kProdWarp) {
    if (lane < S) {
      mbar_init(&full[lane], 1);
      mbar_init(&empty[lane], 1);
    }
    if (lane < 2) {
      mbar_init(&a_full[lane], kWorkerWarps);
      mbar_init(&done[lane], 1);
    }
    mbar_fence_init();
    if (lane == 0) tma_prefetch_desc(&map_x);
    named_bar_arrive(15, kThreads);
  } else {
    if (warp == kMmaWarp0) tmem_alloc<kTmemCols>(tmem_slot);
    tc_fence_before();
    named_bar_sync(15, kThreads);
    tc_fence_after();
  }
  const uint32_t tmem = (warp == kProdWarp) ? 0u : __shfl_sync(0xffffffffu, *tmem_slot, 0);
  // programmatic dependent launch: nothing above touched global memory (w4a16_gemm.cu)
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  if (warp == kProdWarp) {
    // ===================== producer =====================
    const int tile0 = gb / p.G;
    int g = gb % p.G, tn = tile0 % p.ntiles, mc = tile0 / p.ntiles;
    int s = 0;
    uint32_t ph = 0;
    for (int it = 0; it < n_it; ++it) {
      mbar_wait(&empty[s], ph ^ 1);
      if (elect_one()) {
        uint8_t* st = smem + s * kStageBytes;
        mbar_arrive_expect_tx(&full[s], kTxBytes);
        bulk_load_1d(st, p.qweight + ((size_t)tn * p.G + g) * kWBytes, kWBytes, &full[s], kEvictFirst);
        const int xk = (g >> (kPlanes ? 1 : 0)) * 128;
        tma_load_2d(st + kWBytes, &map_x, &full[s], xk, mc * kMP, kEvictLast);
        tma_load_2d(st + kWBytes + kMP * 128, &map_x, &full[s], xk + 64, mc * kMP, kEvictLast);
        bulk_load_1d(st + kWBytes + kXBytes, p.scales + ((size_t)g * p.N + tn * kTileN) * 2, kScaleBytes, &full[s],
                     kEvictFirst);
      }
      __syncwarp();
      if (++g == p.G) {
        g = 0;
        if (++tn == p.ntiles) { tn = 0; ++mc; }
      }
      if (++s == S) { s = 0; ph ^= 1; }
    }
  } else if (warp == kMmaWarp0 || warp == kMmaWarp0 + 1) {
    // ===================== MMA issuers: warp 17 the even groups of the range, warp 18 the odd ones =====================
    // (buffer = group parity, so an a_full barrier is always served by the same issuer, which sees each of its phases)
    constexpr uint32_t idesc = idesc_bf16_m128(kMP);
    const int b = warp - kMmaWarp0;
    int s = 0;
    for (int it = 0; it < n_it; ++it) {
      if ((it & 1) == b) {
        mbar_wait(&a_full[b], (it >> 1) & 1);            // implies full[s]: the workers waited for it
        tc_fence_after();
        if (elect_one()) {
          const uint32_t xbase = smem_u32(smem + s * kStageBytes + kWBytes);
          const uint32_t d_t = tmem + kTmemD + b * kMP;
          const uint32_t a_t = tmem + kTmemA + b * 64;
#pragma unroll
          for (int kk = 0; kk < 8; ++kk) {
            const uint64_t bdesc = smem_desc_sw128(xbase + (kk >> 2) * (kMP * 128) + (kk & 3) * 32);
            mma_ts_f16(d_t, a_t + kk * 8, bdesc, idesc, kk > 0 ? 1u : 0u);
          }
          tc_commit(&done[b]);
          tc_commit(&empty[s]);
        }
        __syncwarp();
      }
      if (++s == S) s = 0;
    }
  } else {
    // ===================== workers: convert, scale-accumulate, output =====================
    const int part = warp >> 2;             // k-quarter converted / batch-column quarter read back
    const int q4 = warp & 3;                // TMEM lane quarter this warp may access
    const int row = q4 * 32 + lane;         // weight row inside the tile
    const uint32_t lane_addr = (uint32_t)(q4 * 32) << 16;
    const int sw = (row >> 1) & 3;
    const uint32_t w_addr = smem_u32(smem) + row * 64 + ((part ^ sw) << 4);
    const uint32_t sc_addr = smem_u32(smem) + kWBytes + kXBytes + row * 2;
    const uint32_t a_t = tmem + lane_addr + kTmemA + part * 16;
    const uint32_t d_t = tmem + lane_addr + kTmemD + part * kCW;
    const bool leader = (threadIdx.x == 0);

    float acc[kCW];
    float sc_old = 0.f, sc_new = 0.f;      // scales of the (up to two) groups whose MMAs are in flight
    int npend = 0;
    uint32_t pd = 0;                       // bit b: parity of done[b] for its next read-back
    int wbuf = 0, rbuf = 0;
    int s = 0;
    uint32_t ph = 0;
    int it = 0;
    int pend_tile[2] = {-1, -1};

    // scale-accumulate of the oldest group in flight, in two halves so that other work can sit between the tcgen05.ld and
    // its use: read_back_issue() waits for the group's MMAs and starts the loads, read_back_finish() consumes them
    uint32_t d[kCW];
    auto read_back_issue = [&]() {
      mbar_wait(&done[rbuf], (pd >> rbuf) & 1);
      pd ^= 1u << rbuf;
      tc_fence_after();
      ERW_TMEM_LD16(d_t + rbuf * kMP, d, 0);
      ERW_TMEM_LD16(d_t + rbuf * kMP + 16, d, 16);
    };
    auto read_back_finish = [&]() {
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
      for (int m = 0; m < kCW; ++m) acc[m] = fmaf(sc_old, __uint_as_float(d[m]), acc[m]);
      sc_old = sc_new;
      --npend;
      rbuf ^= 1;
    };

    while (it < n_it) {
      // ---- segment = the part of one tile inside this CTA's range ----
      const int gi0 = gb + it;
      const int tile = gi0 / p.G, g_lo = gi0 % p.G;
      const int seg_len = min(p.G - g_lo, n_it - it);
      const int it_end = it + seg_len;
#pragma unroll
      for (int m = 0; m < kCW; ++m) acc[m] = 0.f;
      for (; it < it_end; ++it) {
        mbar_wait(&full[s], ph);
        const uint32_t st = s * kStageBytes;
        const uint4 pk = lds128(st + w_addr);
        const uint32_t sc16 = lds_u16(st + sc_addr);
        // the group before last frees the A buffer and the accumulator written next; its TENSOR-MEMORY loads are in flight
        // while this group is converted, and their use hides the latency of the A operand's store
        const bool drain = (npend == 2);
        if (drain) read_back_issue();
        const uint32_t off2 = (kPlanes && ((gb + it) & 1)) ? 0xC300C300u : 0xC308C308u;   // (-128, -128) : (-136, -136)
        uint32_t a[16];
        dequant_word(pk.x, a + 0, off2);
        dequant_word(pk.y, a + 4, off2);
        dequant_word(pk.z, a + 8, off2);
        dequant_word(pk.w, a + 12, off2);
        ERW_TMEM_ST16(a_t + wbuf * 64, a);
        if (drain) read_back_finish();
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(&a_full[wbuf]);
        if (npend == 0) sc_old = __uint_as_float(sc16 << 16);
        else sc_new = __uint_as_float(sc16 << 16);
        ++npend;
        wbuf ^= 1;
        if (++s == S) { s = 0; ph ^= 1; }
      }
      while (npend > 0) { read_back_issue(); read_back_finish(); }

      // ---- output: a whole tile is stored directly; a partial one goes to the workspace as fp32 ----
      const int n = (tile % p.ntiles) * kTileN + row, m0 = (tile / p.ntiles) * kMP + part * kCW;
      const int mvalid = min(kCW, p.M - m0);   // may be <= 0
      if (seg_len == p.G) {
        if (p.y_f32) {
          float* y = reinterpret_cast<float*>(p.y);
#pragma unroll
          for (int m = 0; m < kCW; ++m)
            if (m < mvalid) y[(size_t)(m0 + m) * p.ldy + n] = acc[m];
        } else {
          __nv_bfloat16* y = reinterpret_cast<__nv_bfloat16*>(p.y);
#pragma unroll
          for (int m = 0; m < kCW; ++m)
            if (m < mvalid) y[(size_t)(m0 + m) * p.ldy + n] = __float2bfloat16_rn(acc[m]);
        }
      } else {
        const int k = (it_end - seg_len == 0) ? 0 : 1;      // head segment of this CTA's range, or its tail
        float* mine = p.partials + ((size_t)cta * 2 + k) * (kMP * kTileN) + part * kCW * kTileN;
#pragma unroll
        for (int m = 0; m < kCW; ++m)
          if (m < mvalid) __stcg(mine + m * kTileN + row, acc[m]);
        pend_tile[k] = tile;
      }
    }

    // ---- partial tiles: ticket per tile; the last CTA to arrive adds all partials in ascending CTA order ----
    // Ordering: partial stores (all threads) -> bar.sync -> the leader's acq_rel ticket (release is cumulative over what the
    // barrier made visible to the leader); last arriver: acq_rel ticket -> bar.sync -> ld.cg of the others' partials.
    if (pend_tile[0] >= 0 || pend_tile[1] >= 0) {       // uniform over the CTA's workers
      named_bar_sync(7, kWorkerThreads);
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
          if (pend_tile[k] >= 0)
            asm volatile("atom.acq_rel.gpu.global.add.s32 %0, [%1], 1;" : "=r"(old[k]) : "l"(p.counters + pend_tile[k]) : "memory");
#pragma unroll
        for (int k = 0; k < 2; ++k) {
          const int last = (pend_tile[k] >= 0 && old[k] == c_hi[k] - c_lo[k]);
          if (last) p.counters[pend_tile[k]] = 0;  // leave the counter zero for the next call
          last_flag[k] = last;
        }
      }
      named_bar_sync(7, kWorkerThreads);
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        if (pend_tile[k] < 0 || last_flag[k] == 0) continue;
        const int tile = pend_tile[k];
        const int n = (tile % p.ntiles) * kTileN + row, m0 = (tile / p.ntiles) * kMP + part * kCW;
        const int mvalid = min(kCW, p.M - m0);
#pragma unroll
        for (int m = 0; m < kCW; ++m) acc[m] = 0.f;
        for (int c = c_lo[k]; c <= c_hi[k]; ++c) {
          // CTA c's piece of this tile is its first segment iff its range starts inside the tile
          const int cb = range_begin(p.uq, p.ur, p.split, c) * ug;
          const int which = (cb >= tile * p.G) ? 0 : 1;
          const float* src = p.partials + ((size_t)c * 2 + which) * (kMP * kTileN) + part * kCW * kTileN;
          float v[kCW];
#pragma unroll
          for (int m = 0; m < kCW; ++m) v[m] = (m < mvalid) ? __ldcg(src + m * kTileN + row) : 0.f;
#pragma unroll
          for (int m = 0; m < kCW; ++m) acc[m] += v[m];
        }
        if (p.y_f32) {
          float* y = reinterpret_cast<float*>(p.y);
#pragma unroll
          for (int m = 0; m < kCW; ++m)
            if (m < mvalid) y[(size_t)(m0 + m) * p.ldy + n] = acc[m];
        } else {
          __nv_bfloat16* y = reinterpret_cast<__nv_bfloat16*>(p.y);
#pragma unroll
          for (int m = 0; m < kCW; ++m)
            if (m < mvalid) y[(size_t)(m0 + m) * p.ldy + n] = __float2bfloat16_rn(acc[m]);
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  if (warp == kMmaWarp0) tmem_dealloc<kTmemCols>(tmem);
}

}  // namespace

namespace er {

size_t wide_workspace_bytes() { return ER_GEMM_COUNTER_BYTES + (size_t)sm_count() * 2 * kMP * kTileN * sizeof(float); }

// M > 64: `gp` arrives with the problem, the output and the workspace filled in; the partition is made here.
int launch_wide(const void* x, int64_t M, int64_t N, int64_t K, int64_t ldx, GemmParams gp, bool whole, int split,
                cudaStream_t stream) {   // K = columns of the PACKED matrix (2 x the columns of X for two-plane W8: gp.planes)
  const bool planes = gp.planes != 0;
  const int mchunks = (int)((M + kMP - 1) / kMP), ntiles = (int)(N / kTileN), G = (int)(K / ER_GROUP);
  const long long tiles = (long long)ntiles * mchunks;
  if (tiles * G >= (1ll << 31)) return ER_ERR_SHAPE;
  int ctas = sm_count();
  if (g_tune.force_ctas > 0 && g_tune.force_ctas < ctas) ctas = g_tune.force_ctas;
  // whole tiles or stream-K ranges: decided by the caller's cost model (w4a16_gemm.cu, plan_above_64); always whole tiles
  // beyond the counter array
  int unit_groups = (whole || tiles > ER_GEMM_COUNTER_BYTES / 4) ? G : 1;
  if (g_tune.force_ctas > 0 && tiles <= ER_GEMM_COUNTER_BYTES / 4) unit_groups = 1;
  const long long units = tiles * G / unit_groups;
  if ((long long)ctas > units) ctas = (int)units;
  gp.G = G; gp.ntiles = ntiles; gp.mchunks = mchunks; gp.tiles = (int)tiles; gp.unit_groups = unit_groups;
  gp.units = (int)units; gp.uq = (int)(units / ctas); gp.ur = (int)(units % ctas);
  gp.split = 0; gp.cluster = 1;
  if (split >= 2 && unit_groups == 1 && g_tune.force_ctas == 0 && tiles * split <= sm_count()) {
    // tile split: CTA c owns part c % split of tile c / split (w4a16_plan.cuh): one segment and one partial tile per CTA
    gp.split = split; gp.uq = G; gp.ur = 0;
    ctas = (int)(tiles * split);
  }
  CUtensorMap mx;
  if (!make_map_2d(&mx, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, x, (uint64_t)M, (uint64_t)(planes ? K / 2 : K), (uint64_t)ldx * 2, (uint32_t)kMP, 64,
                   CU_TENSOR_MAP_SWIZZLE_128B)) {
    set_last_cuda_error((int)cudaErrorInvalidValue);
    return ER_ERR_CUDA;
  }
  static bool attr_set[kMaxDevices] = {};
  const int dev = current_device();
  if (dev < 0 || dev >= kMaxDevices || !attr_set[dev]) {
    ER_CUDA_TRY(cudaFuncSetAttribute(w4a16_wide_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem));
    ER_CUDA_TRY(cudaFuncSetAttribute(w4a16_wide_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmem));
    if (dev >= 0 && dev < kMaxDevices) attr_set[dev] = true;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)ctas);
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = kSmem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = g_tune.pdl;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  if (planes) ER_CUDA_TRY(cudaLaunchKernelEx(&cfg, w4a16_wide_kernel<true>, mx, gp));
  else ER_CUDA_TRY(cudaLaunchKernelEx(&cfg, w4a16_wide_kernel<false>, mx, gp));
  return ER_OK;
}

}  // namespace er
