// w4a16_gemm.cu -- er_w4a16_gemm: the weight-quantized self-drafter's linear, Y = X . dequant(Wq)^T
// (dense projections are ~90 % of tail decode latency and weight loading dominates at
// small batch; L175: W4A16 weight-only kernel; L467: "on-the-fly dequantization and kernel-level overhead").
//
// sm_100a design:
//   swap-AB: the 128 weight rows of a tile are the M = 128 of tcgen05.mma, the (padded) batch is its N.
//   warp 0      TMA producer: per 256-k block one SWIZZLE_128B box of packed int4 [128 rows x 128 B], the
//               matching X boxes [MPAD x 64 k] x 4 and the 2 x 128 group scales, into a ring of stages.
//   warps 2-5   workers, one thread per weight row: LDS.128 of the packed row, nibble -> bf16 in registers
//               ((w >> 4t) & 0x000F000F | 0x43004300 is the pair 128+u; minus 136 is q exactly), tcgen05.st
//               of the bf16 A operand straight into TENSOR MEMORY (no shared-memory round trip of the 4x
//               expanded weights), then the fp32 scale-accumulate of the previous group's TMEM partial sum.
//   warp 1      one thread issues tcgen05.mma.kind::f16 with A from TMEM, B (= X tile) from shared memory,
//               one fresh fp32 TMEM accumulator per 128-k group (so the group scale is applied exactly, in
//               fp32, after the contraction), and commits to mbarriers.
//   split-K     partial [MPAD x 128] fp32 tiles go to the workspace; the last CTA of a tile (atomic ticket)
//               adds them in ascending split order and stores Y.  Deterministic.
#include <cuda.h>
#include "er_common.cuh"

namespace {

using namespace er;

constexpr int kBlockK = 256;                 // k per pipeline stage (= 128 packed bytes per row = one swizzle row)
constexpr int kTileN = 128;                  // weight rows per CTA tile
constexpr int kWBytes = kTileN * 128;        // 16 KiB packed weights per stage
constexpr int kScaleBytes = 2 * kTileN * 2;  // 2 groups x 128 bf16
constexpr int kThreads = 192;
constexpr int kTmemCols = 256;
constexpr int kTmemA = 0;    // A operand ring: 2 buffers x 64 columns (128 k of bf16 pairs)
constexpr int kTmemD = 128;  // accumulator ring: 2 buffers x MPAD columns

template <int MPAD>
struct Cfg {
  static constexpr int kXBytes = MPAD * kBlockK * 2;  // 4 boxes of [MPAD x 64] bf16
  static constexpr int kStageBytes = kWBytes + kXBytes + 1024;
  static constexpr int kStages = (MPAD == 16) ? 4 : (MPAD == 32 ? 3 : 4);
  static constexpr int kMinBlocks = (MPAD <= 32) ? 2 : 1;
  static constexpr int kSmem = kStages * kStageBytes + 1024 /*align slack*/ + 256 /*barriers*/;
  static constexpr uint32_t kTxBytes = kWBytes + kXBytes + kScaleBytes;
};

struct GemmParams {
  int M, N, K;
  int kblocks;         // ceil(K / 256)
  int splits;          // K splits per tile
  int y_f32;
  int64_t ldy;
  void* y;
  const void* scales;  // unused by the kernel (TMA), kept for debugging
  float* partials;     // workspace + ER_GEMM_COUNTER_BYTES
  int* counters;       // workspace
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

// 4 packed words (32 codes) -> 16 registers of bf16 pairs (k, k+1), exact.
__device__ __forceinline__ void dequant4(const uint4& p, uint32_t (&a)[64], int base) {
  const uint32_t w[4] = {p.x, p.y, p.z, p.w};
  const __nv_bfloat162 off = __floats2bfloat162_rn(136.0f, 136.0f);
#pragma unroll
  for (int i = 0; i < 4; ++i) {
#pragma unroll
    for (int t = 0; t < 4; ++t) {
      uint32_t v = ((w[i] >> (4 * t)) & 0x000F000Fu) | 0x43004300u;  // bf16 pair (128 + u_k, 128 + u_{k+1})
      __nv_bfloat162 h = __hsub2(*reinterpret_cast<__nv_bfloat162*>(&v), off);
      a[base + 4 * i + t] = *reinterpret_cast<uint32_t*>(&h);
    }
  }
}

template <int MPAD>
__global__ void __launch_bounds__(kThreads, Cfg<MPAD>::kMinBlocks)
w4a16_gemm_kernel(const __grid_constant__ CUtensorMap map_w, const __grid_constant__ CUtensorMap map_x,
                  const __grid_constant__ CUtensorMap map_s, const GemmParams p) {
  using C = Cfg<MPAD>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + C::kStages * C::kStageBytes);
  uint64_t* full = bars;                    // [kStages] TMA landed
  uint64_t* empty = bars + C::kStages;      // [kStages] workers (128) + MMA commit (1) released the stage
  uint64_t* a_full = bars + 2 * C::kStages; // [2] A operand of a group written to TMEM by 128 workers
  uint64_t* mma_done = a_full + 2;          // [2] MMAs of a group complete: D readable, A buffer reusable
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(mma_done + 2);
  int* last_flag = reinterpret_cast<int*>(tmem_slot + 1);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int split = blockIdx.x, ntile = blockIdx.y, mchunk = blockIdx.z;
  const int n0 = ntile * kTileN, m0 = mchunk * 64;
  // k-block range of this split (balanced)
  const int kb_begin = (int)(((int64_t)p.kblocks * split) / p.splits);
  const int kb_end = (int)(((int64_t)p.kblocks * (split + 1)) / p.splits);
  const int nkb = kb_end - kb_begin;
  const int ngroups = 2 * nkb;

  if (threadIdx.x == 0) {
    tma_prefetch_desc(&map_w);
    tma_prefetch_desc(&map_x);
    tma_prefetch_desc(&map_s);
    for (int s = 0; s < C::kStages; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], 129);
    }
    for (int j = 0; j < 2; ++j) {
      mbar_init(&a_full[j], 128);
      mbar_init(&mma_done[j], 1);
    }
    mbar_fence_init();
  }
  if (warp == 1) tmem_alloc<kTmemCols>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *tmem_slot;

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      for (int i = 0; i < nkb; ++i) {
        const int s = i % C::kStages;
        mbar_wait(&empty[s], ((i / C::kStages) & 1) ^ 1);
        uint8_t* st = smem + s * C::kStageBytes;
        const int kb = kb_begin + i;
        mbar_arrive_expect_tx(&full[s], C::kTxBytes);
        tma_load_2d(st, &map_w, &full[s], kb * 128, n0, kEvictFirst);
#pragma unroll
        for (int bx = 0; bx < 4; ++bx)
          tma_load_2d(st + kWBytes + bx * (MPAD * 128), &map_x, &full[s], kb * kBlockK + bx * 64, m0, kEvictLast);
        tma_load_2d(st + kWBytes + C::kXBytes, &map_s, &full[s], n0, kb * 2, kEvictFirst);
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    if (lane == 0) {
      constexpr uint32_t idesc = idesc_bf16_m128(MPAD);
      for (int g = 0; g < ngroups; ++g) {
        const int i = g >> 1, h = g & 1, s = i % C::kStages, j = g & 1;
        if (h == 0) mbar_wait(&full[s], (i / C::kStages) & 1);
        mbar_wait(&a_full[j], (g >> 1) & 1);
        tc_fence_after();
        const uint32_t xbase = smem_u32(smem + s * C::kStageBytes + kWBytes);
        const uint32_t d_t = tmem + kTmemD + j * MPAD;
        const uint32_t a_t = tmem + kTmemA + j * 64;
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
          const int koff = h * 128 + kk * 16;  // k offset inside the stage
          const uint64_t bdesc = smem_desc_sw128(xbase + (koff >> 6) * (MPAD * 128) + (koff & 63) * 2);
          mma_ts_f16(d_t, a_t + kk * 8, bdesc, idesc, kk > 0 ? 1u : 0u);
        }
        tc_commit(&mma_done[j]);
        if (h == 1) tc_commit(&empty[s]);
      }
    }
  } else {
    // ===================== workers: dequant -> TMEM, scale-accumulate =====================
    const int q4 = warp & 3;               // TMEM lane quarter this warp may access
    const int row = q4 * 32 + lane;        // weight row inside the tile
    const uint32_t lane_addr = (uint32_t)(q4 * 32) << 16;
    float acc[MPAD];
#pragma unroll
    for (int m = 0; m < MPAD; ++m) acc[m] = 0.f;
    float sc_prev = 0.f;

    auto epilogue_group = [&](int hgrp, float sc) {
      const int j = hgrp & 1;
      mbar_wait(&mma_done[j], (hgrp >> 1) & 1);
      tc_fence_after();
      uint32_t d[MPAD];
#pragma unroll
      for (int c = 0; c < MPAD; c += 16) ER_TMEM_LD16(tmem + lane_addr + kTmemD + j * MPAD + c, d, c);
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
      for (int m = 0; m < MPAD; ++m) acc[m] = fmaf(sc, __uint_as_float(d[m]), acc[m]);
    };

    for (int g = 0; g < ngroups; ++g) {
      const int i = g >> 1, h = g & 1, s = i % C::kStages, j = g & 1;
      if (h == 0) mbar_wait(&full[s], (i / C::kStages) & 1);
      const uint8_t* st = smem + s * C::kStageBytes;
      const uint8_t* wrow = st + row * 128;
      uint4 pk[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) pk[c] = *reinterpret_cast<const uint4*>(wrow + (((4 * h + c) ^ (row & 7)) << 4));
      const float sc = __bfloat162float(
          *reinterpret_cast<const __nv_bfloat16*>(st + kWBytes + C::kXBytes + h * 256 + row * 2));
      uint32_t a[64];
#pragma unroll
      for (int c = 0; c < 4; ++c) dequant4(pk[c], a, 16 * c);
      // A buffer j is free: mma_done of group g-2 was waited for in the previous iteration's epilogue
      const uint32_t a_t = tmem + lane_addr + kTmemA + j * 64;
      ER_TMEM_ST16(a_t + 0, a, 0);
      ER_TMEM_ST16(a_t + 16, a, 16);
      ER_TMEM_ST16(a_t + 32, a, 32);
      ER_TMEM_ST16(a_t + 48, a, 48);
      asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
      tc_fence_before();
      if (h == 1) mbar_arrive(&empty[s]);
      mbar_arrive(&a_full[j]);
      if (g > 0) epilogue_group(g - 1, sc_prev);
      sc_prev = sc;
    }
    if (ngroups > 0) epilogue_group(ngroups - 1, sc_prev);

    // ---- output: direct store, or split-K partial + last-arriver reduction ----
    const int mvalid = min(MPAD, p.M - m0);
    const int n = n0 + row;
    bool store = true;
    if (p.splits > 1) {
      const int tile_id = mchunk * gridDim.y + ntile;
      float* mine = p.partials + ((size_t)tile_id * p.splits + split) * (MPAD * kTileN);
#pragma unroll
      for (int m = 0; m < MPAD; ++m)
        if (m < mvalid) __stcg(mine + m * kTileN + row, acc[m]);
      __threadfence();
      asm volatile("bar.sync 1, 128;" ::: "memory");
      if (threadIdx.x == 64) {
        const int old = atomicAdd(p.counters + tile_id, 1);
        const int last = (old == p.splits - 1);
        if (last) p.counters[tile_id] = 0;  // leave the counter zero for the next call
        *last_flag = last;
      }
      asm volatile("bar.sync 1, 128;" ::: "memory");
      store = (*last_flag != 0);
      if (store) {
        __threadfence();
        const float* base = p.partials + (size_t)tile_id * p.splits * (MPAD * kTileN);
#pragma unroll
        for (int m = 0; m < MPAD; ++m) {
          if (m < mvalid) {
            float sum = 0.f;
            for (int sp = 0; sp < p.splits; ++sp) sum += __ldcg(base + (size_t)sp * (MPAD * kTileN) + m * kTileN + row);
            acc[m] = sum;
          }
        }
      }
    }
    if (store) {
      if (p.y_f32) {
        float* y = reinterpret_cast<float*>(p.y);
#pragma unroll
        for (int m = 0; m < MPAD; ++m)
          if (m < mvalid) y[(size_t)(m0 + m) * p.ldy + n] = acc[m];
      } else {
        __nv_bfloat16* y = reinterpret_cast<__nv_bfloat16*>(p.y);
#pragma unroll
        for (int m = 0; m < MPAD; ++m)
          if (m < mvalid) y[(size_t)(m0 + m) * p.ldy + n] = __float2bfloat16_rn(acc[m]);
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  if (warp == 1) tmem_dealloc<kTmemCols>(tmem);
}

}  // namespace

// =====================================================================================================
// host side: tensor maps, split-K plan, launch
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

// 2-D row-major tensor [rows][cols] of `esize`-byte elements, row pitch in bytes, box [box_rows][box_cols].
bool make_map_2d(CUtensorMap* map, CUtensorMapDataType dt, int esize, const void* base, uint64_t rows, uint64_t cols,
                 uint64_t pitch_bytes, uint32_t box_rows, uint32_t box_cols, CUtensorMapSwizzle swz) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {cols, rows};
  cuuint64_t strides[1] = {pitch_bytes};
  cuuint32_t box[2] = {box_cols, box_rows};
  cuuint32_t estr[2] = {1, 1};
  (void)esize;
  CUresult r = fn(map, dt, 2, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, swz,
                  CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

int g_tune_ctas_per_sm = 2;   // split-K target: resident CTAs per SM to fill (MPAD <= 32)
int g_tune_force_splits = 0;  // > 0: force this many K splits (tests / sweeps)

struct Plan {
  int mpad, mchunks, ntiles, kblocks, splits;
};

Plan make_plan(int64_t M, int64_t N, int64_t K) {
  Plan pl;
  pl.mpad = M <= 16 ? 16 : (M <= 32 ? 32 : 64);
  pl.mchunks = (int)((M + 63) / 64);
  pl.ntiles = (int)(N / kTileN);
  pl.kblocks = (int)((K + kBlockK - 1) / kBlockK);
  const int tiles = pl.ntiles * pl.mchunks;
  const int resident = er::sm_count() * (pl.mpad <= 32 ? g_tune_ctas_per_sm : 1);
  int splits = 1;
  if (tiles < resident) {
    splits = resident / tiles;
    if (splits > pl.kblocks) splits = pl.kblocks;
    if (splits < 1) splits = 1;
  }
  if (g_tune_force_splits > 0) splits = g_tune_force_splits < pl.kblocks ? g_tune_force_splits : pl.kblocks;
  if (tiles > ER_GEMM_COUNTER_BYTES / 4) splits = 1;  // counters cover 4096 tiles
  if (splits > 65535) splits = 65535;
  pl.splits = splits;
  return pl;
}

size_t plan_workspace(const Plan& pl) {
  size_t partial = 0;
  if (pl.splits > 1) partial = (size_t)pl.ntiles * pl.mchunks * pl.splits * pl.mpad * kTileN * sizeof(float);
  return ER_GEMM_COUNTER_BYTES + partial;
}

template <int MPAD>
int launch(const CUtensorMap& mw, const CUtensorMap& mx, const CUtensorMap& ms, const GemmParams& gp, const Plan& pl,
           cudaStream_t stream) {
  static bool attr_set = false;
  if (!attr_set) {
    ER_CUDA_TRY(cudaFuncSetAttribute(w4a16_gemm_kernel<MPAD>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     Cfg<MPAD>::kSmem));
    attr_set = true;
  }
  dim3 grid((unsigned)pl.splits, (unsigned)pl.ntiles, (unsigned)pl.mchunks);
  w4a16_gemm_kernel<MPAD><<<grid, kThreads, Cfg<MPAD>::kSmem, stream>>>(mw, mx, ms, gp);
  ER_CUDA_TRY(cudaGetLastError());
  return ER_OK;
}

}  // namespace

extern "C" {

// Internal tuning knob for sweeps (not part of the stable ABI): key 0 = CTAs per SM targeted by the
// split-K planner (1 or 2), key 1 = forced split count (0 = planner).
int er_gemm_tuning(int key, int value) {
  if (key == 0 && (value == 1 || value == 2)) { g_tune_ctas_per_sm = value; return ER_OK; }
  if (key == 1 && value >= 0) { g_tune_force_splits = value; return ER_OK; }
  return ER_ERR_SHAPE;
}

size_t er_gemm_workspace_bytes(int64_t M, int64_t N, int64_t K) {
  if (M < 1 || N < kTileN || N % kTileN != 0 || K < ER_GROUP || K % ER_GROUP != 0) return 0;
  // independent of tuning knobs: the largest split count the planner can pick for this shape
  Plan pl = make_plan(M, N, K);
  Plan worst = pl;
  const int tiles = pl.ntiles * pl.mchunks;
  if (tiles <= ER_GEMM_COUNTER_BYTES / 4) {
    int s = (2 * er::sm_count()) / tiles;
    if (s < 1) s = 1;
    if (s > pl.kblocks) s = pl.kblocks;
    if (g_tune_force_splits > s) s = g_tune_force_splits < pl.kblocks ? g_tune_force_splits : pl.kblocks;
    if (s > worst.splits) worst.splits = s;
  }
  return plan_workspace(worst);
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
  if (pl.mchunks > 65535 || pl.ntiles > 65535) return ER_ERR_SHAPE;
  if (workspace_bytes < plan_workspace(pl)) return ER_ERR_WORKSPACE;
  int st = er::check_arch();
  if (st != ER_OK) return st;

  CUtensorMap mw, mx, ms;
  bool ok = make_map_2d(&mw, CU_TENSOR_MAP_DATA_TYPE_UINT8, 1, qweight, (uint64_t)N, (uint64_t)(K / 2),
                        (uint64_t)(K / 2), kTileN, 128, CU_TENSOR_MAP_SWIZZLE_128B);
  ok = ok && make_map_2d(&mx, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, x_bf16, (uint64_t)M, (uint64_t)K,
                         (uint64_t)ldx_elems * 2, (uint32_t)pl.mpad, 64, CU_TENSOR_MAP_SWIZZLE_128B);
  ok = ok && make_map_2d(&ms, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, scales, (uint64_t)(K / ER_GROUP), (uint64_t)N,
                         (uint64_t)N * 2, 2, kTileN, CU_TENSOR_MAP_SWIZZLE_NONE);
  if (!ok) {
    er::set_last_cuda_error((int)cudaErrorInvalidValue);
    return ER_ERR_CUDA;
  }
  GemmParams gp;
  gp.M = (int)M; gp.N = (int)N; gp.K = (int)K;
  gp.kblocks = pl.kblocks; gp.splits = pl.splits;
  gp.y_f32 = (y_dtype == ER_F32); gp.ldy = ldy_elems; gp.y = y; gp.scales = scales;
  gp.counters = reinterpret_cast<int*>(workspace);
  gp.partials = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(workspace) + ER_GEMM_COUNTER_BYTES);
  cudaStream_t s = (cudaStream_t)stream;
  if (pl.mpad == 16) return launch<16>(mw, mx, ms, gp, pl, s);
  if (pl.mpad == 32) return launch<32>(mw, mx, ms, gp, pl, s);
  return launch<64>(mw, mx, ms, gp, pl, s);
}

}  // extern "C"
