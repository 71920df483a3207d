// bf16_gemm.cu -- er_bf16_gemm: Y = X . W^T with bf16 weights, the streaming GEMM of everything the drafter keeps in
// higher precision and of the target model itself:
//   - the drafter's lm_head ("embedding, LM head, norms ... higher precision", PAPER.md:L455 sec. D.2; L101 sec. 4.1
//     quantizes only the FFN and QKVO projections): 152064 x 3584 bf16 = 1.09 GB of the 4.46 GB a drafter step streams;
//   - the target-side linears behind T_p (one autoregressive step) and T_V(gamma) (verifying gamma + 1 positions of
//     every sequence at once) in the paper's speedup model  tau * T_p / (gamma * T_q + T_V)  (Eq. 1,
//     L488-L492 Eq. 5).
// The same skeleton as the W4A16 kernel (w4a16_gemm.cu) minus the dequantisation: persistent, one CTA per SM, the
// (tile, k unit) work dealt out as one contiguous range per CTA (stream-K, w4a16_plan.cuh); swap-AB -- the 128 weight
// rows of a tile are the M of tcgen05.mma.kind::f16, the padded batch (16 ... 256) is its N; both operands come
// straight from shared memory (SWIZZLE_128B TMA boxes), the fp32 accumulator lives in TENSOR MEMORY for a whole tile
// segment and is double-buffered, so the epilogue of one segment runs under the MMAs of the next.
//   warp 4      producer: per k unit the W boxes [128 rows x 64 k] and the X boxes [MPAD x 64 k] into a ring
//   warp 5      MMA issuer (one elected lane): UK / 16 MMAs per unit, tcgen05.commit frees the stage; at the end of a
//               segment a commit tells the epilogue that the accumulator is complete
//   warps 0-3   epilogue: tcgen05.ld of the accumulator (a thread owns one weight row), then a direct store of a whole
//               tile, or fp32 partials to the workspace -- the last CTA of a tile (ticket) adds them in ascending CTA
//               order.  Deterministic, no float atomics.
#include "w4a16_plan.cuh"

namespace {

using namespace er;

constexpr int kThreads = 192;
constexpr int kMaxStages = 8;

template <int MPAD>
struct BCfg {
  static constexpr int UK = (MPAD <= 64) ? 128 : 64;          // k per ring stage
  static constexpr int kBoxes = UK / 64;
  static constexpr int kWBox = kTileN * 128;                  // [128 rows x 64 k] bf16
  static constexpr int kXBox = MPAD * 128;
  static constexpr int kStageBytes = kBoxes * (kWBox + kXBox);
  static constexpr uint32_t kTxBytes = kStageBytes;
  static constexpr int kFixed = 1024 /*align slack*/ + 512 /*barriers*/;
  static constexpr int kStagesRaw = (kSmemLimit - kFixed) / kStageBytes;
  static constexpr int kStages = kStagesRaw > kMaxStages ? kMaxStages : kStagesRaw;
  static constexpr int kSmem = kStages * kStageBytes + kFixed;
  static constexpr int kTmemCols = (2 * MPAD <= 32) ? 32 : (2 * MPAD <= 64 ? 64 : (2 * MPAD <= 128 ? 128 : (2 * MPAD <= 256 ? 256 : 512)));
  static_assert(kStages >= 2 && kStageBytes % 1024 == 0, "ring");
};

#define ER_TMEM_LD16(taddr, r)                                                                                 \
  asm volatile(                                                                                                \
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];" \
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),        \
        "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])   \
      : "r"(taddr)                                                                                             \
      : "memory")

__device__ __forceinline__ void named_bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }

template <int MPAD>
__global__ void __launch_bounds__(kThreads, 1)
bf16_gemm_kernel(const __grid_constant__ CUtensorMap map_w, const __grid_constant__ CUtensorMap map_x,
                 const GemmParams p) {
  using C = BCfg<MPAD>;
  constexpr int S = C::kStages;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + S * C::kStageBytes);
  uint64_t* full = bars;                        // [S] TMA landed
  uint64_t* empty = bars + kMaxStages;          // [S] the unit's MMAs completed
  uint64_t* acc_full = bars + 2 * kMaxStages;   // [2] the segment's MMAs completed: accumulator readable
  uint64_t* acc_free = acc_full + 2;            // [2] the epilogue has read the accumulator
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(acc_free + 2);
  int* last_flag = reinterpret_cast<int*>(tmem_slot + 1);

  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
  const int lane = threadIdx.x & 31;
  const int cta = blockIdx.x;
  const int ug = p.unit_groups;                 // units (of UK k) per scheduling unit
  const int gb = range_begin(p.uq, p.ur, p.split, cta) * ug;
  const int ge = range_begin(p.uq, p.ur, p.split, cta + 1) * ug;
  const int n_it = ge - gb;

  if (warp == 4) {
    if (lane < S) {
      mbar_init(&full[lane], 1);
      mbar_init(&empty[lane], 1);
    }
    if (lane < 2) {
      mbar_init(&acc_full[lane], 1);
      mbar_init(&acc_free[lane], 4);
    }
    mbar_fence_init();
    if (lane == 0) {
      tma_prefetch_desc(&map_w);
      tma_prefetch_desc(&map_x);
    }
  }
  if (warp == 5) tmem_alloc<C::kTmemCols>(tmem_slot);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = __shfl_sync(0xffffffffu, *tmem_slot, 0);
  // programmatic dependent launch: see w4a16_gemm.cu
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  if (warp == 4) {
    // ===================== producer =====================
    const int tile0 = gb / p.G;
    int g = gb % p.G, tn = tile0 % p.ntiles, mc = tile0 / p.ntiles;
    int s = 0;
    uint32_t ph = 0;
    for (int it = 0; it < n_it; ++it) {
      mbar_wait(&empty[s], ph ^ 1);
      if (elect_one()) {
        uint8_t* st = smem + s * C::kStageBytes;
        mbar_arrive_expect_tx(&full[s], C::kTxBytes);
#pragma unroll
        for (int b = 0; b < C::kBoxes; ++b) {
          tma_load_2d(st + b * C::kWBox, &map_w, &full[s], g * C::UK + b * 64, tn * kTileN, kEvictFirst);
          tma_load_2d(st + C::kBoxes * C::kWBox + b * C::kXBox, &map_x, &full[s], g * C::UK + b * 64, mc * MPAD,
                      kEvictLast);
        }
      }
      __syncwarp();
      if (++g == p.G) {
        g = 0;
        if (++tn == p.ntiles) { tn = 0; ++mc; }
      }
      if (++s == S) { s = 0; ph ^= 1; }
    }
  } else if (warp == 5) {
    // ===================== MMA issuer =====================
    constexpr uint32_t idesc = idesc_bf16_m128(MPAD);
    int s = 0;
    uint32_t ph = 0;
    int it = 0, seg = 0;
    while (it < n_it) {
      const int g_lo = (gb + it) % p.G;
      const int seg_len = min(p.G - g_lo, n_it - it);
      const int buf = seg & 1;
      if (seg >= 2) mbar_wait(&acc_free[buf], ((seg >> 1) - 1) & 1);   // the epilogue of segment seg - 2 has drained it
      tc_fence_after();
      const uint32_t d_t = tmem + buf * MPAD;
      for (int u = 0; u < seg_len; ++u) {
        mbar_wait(&full[s], ph);
        tc_fence_after();
        if (elect_one()) {
          const uint32_t wbase = smem_u32(smem + s * C::kStageBytes);
          const uint32_t xbase = wbase + C::kBoxes * C::kWBox;
#pragma unroll
          for (int kk = 0; kk < C::UK / 16; ++kk) {
            const uint64_t adesc = smem_desc_sw128(wbase + (kk >> 2) * C::kWBox + (kk & 3) * 32);
            const uint64_t bdesc = smem_desc_sw128(xbase + (kk >> 2) * C::kXBox + (kk & 3) * 32);
            mma_ss_f16(d_t, adesc, bdesc, idesc, (u > 0 || kk > 0) ? 1u : 0u);
          }
          tc_commit(&empty[s]);
          if (u == seg_len - 1) tc_commit(&acc_full[buf]);
        }
        __syncwarp();
        if (++s == S) { s = 0; ph ^= 1; }
      }
      it += seg_len;
      ++seg;
    }
  } else {
    // ===================== epilogue (warps 0-3: TMEM lane quarter = warp) =====================
    const int row = warp * 32 + lane;
    const uint32_t lane_addr = (uint32_t)(warp * 32) << 16;
    const bool leader = (threadIdx.x == 0);
    int it = 0, seg = 0;
    int pend_tile[2] = {-1, -1};
    while (it < n_it) {
      const int gi0 = gb + it;
      const int tile = gi0 / p.G, g_lo = gi0 % p.G;
      const int seg_len = min(p.G - g_lo, n_it - it);
      const int buf = seg & 1;
      mbar_wait(&acc_full[buf], (seg >> 1) & 1);
      tc_fence_after();
      const int n = (tile % p.ntiles) * kTileN + row, m_base = (tile / p.ntiles) * MPAD;
      const bool whole = (seg_len == p.G);
      const int k = (it == 0 ? 0 : 1);
      float* mine = p.partials + ((size_t)cta * 2 + k) * (MPAD * kTileN);
#pragma unroll 1
      for (int c0 = 0; c0 < MPAD; c0 += 16) {
        if (m_base + c0 >= p.M) break;             // rows >= M are never written (uniform over the CTA)
        uint32_t v[16];
        ER_TMEM_LD16(tmem + lane_addr + buf * MPAD + c0, v);
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          const int m = m_base + c0 + j;
          if (m < p.M) {
            if (whole) {
              if (p.y_f32) reinterpret_cast<float*>(p.y)[(size_t)m * p.ldy + n] = __uint_as_float(v[j]);
              else reinterpret_cast<__nv_bfloat16*>(p.y)[(size_t)m * p.ldy + n] = __float2bfloat16_rn(__uint_as_float(v[j]));
            } else {
              __stcg(mine + (c0 + j) * kTileN + row, __uint_as_float(v[j]));
            }
          }
        }
      }
      if (!whole) pend_tile[k] = tile;
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&acc_free[buf]);
      it += seg_len;
      ++seg;
    }

    // ---- partial tiles: ticket per tile; the last CTA to arrive adds all partials in ascending CTA order ----
    if (pend_tile[0] >= 0 || pend_tile[1] >= 0) {
      named_bar_sync(1, 128);
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
      named_bar_sync(1, 128);
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        if (pend_tile[k] < 0 || last_flag[k] == 0) continue;
        const int tile = pend_tile[k];
        const int n0 = (tile % p.ntiles) * kTileN, m_base = (tile / p.ntiles) * MPAD;
        // a partial tile is [MPAD][128] fp32: the 128 threads walk it as float4 (thread t: batch row 4 i + t / 32, four
        // consecutive n from (t % 32) * 4), kI rows of loads in flight per partial, partials added in ascending CTA order
        const int t = threadIdx.x, col4 = (t & 31) * 4;
        constexpr int kI = 8;
#pragma unroll 1
        for (int i0 = 0; i0 < MPAD / 4; i0 += kI) {
          if (m_base + 4 * i0 >= p.M) break;
          float4 acc[kI];
#pragma unroll
          for (int i = 0; i < kI; ++i) acc[i] = make_float4(0.f, 0.f, 0.f, 0.f);
          for (int c = c_lo[k]; c <= c_hi[k]; ++c) {
            // CTA c's piece of this tile is its first segment iff its range starts inside the tile
            const int cb = range_begin(p.uq, p.ur, p.split, c) * ug;
            const int which = (cb >= tile * p.G) ? 0 : 1;
            const float* src = p.partials + ((size_t)c * 2 + which) * (MPAD * kTileN);
            float4 v[kI];
#pragma unroll
            for (int i = 0; i < kI; ++i) {
              const int m = 4 * (i0 + i) + (t >> 5);
              v[i] = (i0 + i < MPAD / 4 && m_base + m < p.M) ? __ldcg(reinterpret_cast<const float4*>(src + m * kTileN + col4))
                                                            : make_float4(0.f, 0.f, 0.f, 0.f);
            }
#pragma unroll
            for (int i = 0; i < kI; ++i) { acc[i].x += v[i].x; acc[i].y += v[i].y; acc[i].z += v[i].z; acc[i].w += v[i].w; }
          }
#pragma unroll
          for (int i = 0; i < kI; ++i) {
            const int m = m_base + 4 * (i0 + i) + (t >> 5);
            if (i0 + i < MPAD / 4 && m < p.M) {
              const size_t o = (size_t)m * p.ldy + n0 + col4;
              if (p.y_f32) {
                float* y = reinterpret_cast<float*>(p.y) + o;      // ldy is not necessarily a multiple of 4: scalar stores
                y[0] = acc[i].x; y[1] = acc[i].y; y[2] = acc[i].z; y[3] = acc[i].w;
              } else {
                __nv_bfloat16* y = reinterpret_cast<__nv_bfloat16*>(p.y) + o;
                y[0] = __float2bfloat16_rn(acc[i].x); y[1] = __float2bfloat16_rn(acc[i].y);
                y[2] = __float2bfloat16_rn(acc[i].z); y[3] = __float2bfloat16_rn(acc[i].w);
              }
            }
          }
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  if (warp == 5) tmem_dealloc<C::kTmemCols>(tmem);
}

int mpad_of(int64_t M) { return M <= 16 ? 16 : (M <= 32 ? 32 : (M <= 64 ? 64 : (M <= 128 ? 128 : 256))); }
int uk_of(int mpad) { return mpad <= 64 ? 128 : 64; }

size_t workspace_for(int mpad) {
  return ER_GEMM_COUNTER_BYTES + (size_t)er::sm_count() * 2 * mpad * kTileN * sizeof(float);
}

template <int MPAD>
int launch(const CUtensorMap& mw, const CUtensorMap& mx, const GemmParams& gp, int ctas, cudaStream_t stream) {
  static bool attr_set[er::kMaxDevices] = {};
  const int dev = er::current_device();
  if (dev < 0 || dev >= er::kMaxDevices || !attr_set[dev]) {
    ER_CUDA_TRY(cudaFuncSetAttribute(bf16_gemm_kernel<MPAD>, cudaFuncAttributeMaxDynamicSharedMemorySize, BCfg<MPAD>::kSmem));
    if (dev >= 0 && dev < er::kMaxDevices) attr_set[dev] = true;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)ctas);
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = BCfg<MPAD>::kSmem;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = er::g_tune.pdl;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  ER_CUDA_TRY(cudaLaunchKernelEx(&cfg, bf16_gemm_kernel<MPAD>, mw, mx, gp));
  return ER_OK;
}

// Plan: the padded batch MPAD (the N of the MMA) may be SMALLER than M -- the batch is then cut into chunks, every (chunk,
// 128-row weight tile) is a tile of its own, and a tile's weights are read once per chunk (from L2 after the first).
// That buys whole tiles for most SMs on the small linears, where stream-K would leave partial tiles of MPAD x 128 fp32
// for the last CTA of a tile to add up (128 threads: ~12 bytes per clock).  Costs per 128-k group in SM cycles, fitted
// to the lm_head timings (profiles/r02_gemm.md section 7): 800 + 4.9 MPAD with the weights in L2 (the X box is re-read
// for every tile), 1440 when the weights stream from HBM at the measured peak.
struct BPlan { int mpad, whole, ctas; double cycles; };
BPlan bf16_plan(int64_t M, int64_t N, int64_t K) {
  const int sms = er::sm_count();
  const int cap = (er::g_tune.force_ctas > 0 && er::g_tune.force_ctas < sms) ? er::g_tune.force_ctas : sms;
  const int ntiles = (int)(N / kTileN);
  const double G128 = (double)K / 128.0;
  const double hbm = (double)N * (double)K * 2.0 / 22.7 / sms;   // cycles to stream all weights once: 22.7 B / clock / SM
  BPlan best = {mpad_of(M), 0, 1, 1e300};
  for (int mpad = mpad_of(M); mpad >= 16; mpad >>= 1) {
    const long long tiles = (long long)ntiles * ((M + mpad - 1) / mpad);
    const double per_group = 800.0 + 4.9 * mpad;
    if (er::g_tune.force_ctas == 0) {   // whole tiles
      const int c = (int)(tiles < cap ? tiles : cap);
      const double cyc = fmax((double)((tiles + c - 1) / c) * G128 * per_group, hbm) + 3000.0;
      if (cyc < best.cycles) best = {mpad, 1, c, cyc};
    }
    if (tiles <= ER_GEMM_COUNTER_BYTES / 4) {   // stream-K: units of uk k, partial tiles through the workspace
      const int uk = uk_of(mpad);
      const long long upt = K / uk, units = tiles * upt;
      const int c = (int)(units < cap ? units : cap);
      const double per_unit = per_group * uk / 128.0;
      const bool aligned = units % c == 0 && (units / c) % upt == 0;            // every CTA gets whole tiles anyway
      const double parts = fmin((double)c / (double)tiles + 1.0, (double)c);     // partial tiles the last CTA adds
      const double cyc = fmax((double)((units + c - 1) / c) * per_unit, hbm) + (aligned ? 0.0 : parts * mpad * 512.0 / 12.0) +
                         6000.0;
      if (cyc < best.cycles) best = {mpad, 0, c, cyc};
    }
  }
  return best;
}

}  // namespace

extern "C" {

size_t er_bf16_gemm_workspace_bytes(int64_t M, int64_t N, int64_t K) {
  if (M < 1 || N < kTileN || N % kTileN != 0 || K < ER_GROUP || K % ER_GROUP != 0) return 0;
  return workspace_for(mpad_of(M));
}

int er_bf16_gemm(const void* x_bf16, int64_t M, int64_t K, int64_t ldx_elems, const void* w_bf16, int64_t N,
                 int64_t ldw_elems, void* y, int64_t ldy_elems, int y_dtype, void* workspace, size_t workspace_bytes,
                 void* stream) {
  if (!x_bf16 || !w_bf16 || !y) return ER_ERR_NULL;
  if (M < 1 || M > (1 << 20) || N < kTileN || N % kTileN != 0 || N > (1 << 24) || K < ER_GROUP || K % ER_GROUP != 0 ||
      K > (1 << 24) || ldx_elems < K || ldw_elems < K || ldy_elems < N)
    return ER_ERR_SHAPE;
  if (y_dtype != ER_BF16 && y_dtype != ER_F32) return ER_ERR_DTYPE;
  if (!er::aligned16(x_bf16) || !er::aligned16(w_bf16) || (ldx_elems % 8) != 0 || (ldw_elems % 8) != 0) return ER_ERR_ALIGN;
  if (!workspace) return ER_ERR_WORKSPACE;
  if (!er::aligned16(workspace)) return ER_ERR_ALIGN;
  if (workspace_bytes < workspace_for(mpad_of(M))) return ER_ERR_WORKSPACE;
  int st = er::check_arch();
  if (st != ER_OK) return st;
  const BPlan pl = bf16_plan(M, N, K);
  const int mpad = pl.mpad, uk = uk_of(mpad);
  const int mchunks = (int)((M + mpad - 1) / mpad), ntiles = (int)(N / kTileN);
  const long long tiles = (long long)ntiles * mchunks;
  const int G = (int)(K / uk);
  if (tiles * G >= (1ll << 31)) return ER_ERR_SHAPE;
  const int unit_groups = pl.whole ? G : 1;
  const long long units = tiles * G / unit_groups;
  const int ctas = pl.ctas;

  CUtensorMap mw, mx;
  const bool ok = er::make_map_2d(&mw, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, w_bf16, (uint64_t)N, (uint64_t)K,
                                  (uint64_t)ldw_elems * 2, kTileN, 64, CU_TENSOR_MAP_SWIZZLE_128B) &&
                  er::make_map_2d(&mx, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, x_bf16, (uint64_t)M, (uint64_t)K,
                                  (uint64_t)ldx_elems * 2, (uint32_t)mpad, 64, CU_TENSOR_MAP_SWIZZLE_128B);
  if (!ok) {
    er::set_last_cuda_error((int)cudaErrorInvalidValue);
    return ER_ERR_CUDA;
  }
  GemmParams gp = {};
  gp.M = (int)M; gp.N = (int)N; gp.K = (int)K;
  gp.G = G; gp.ntiles = ntiles; gp.tiles = (int)tiles; gp.unit_groups = unit_groups; gp.units = (int)units;
  gp.uq = (int)(units / ctas); gp.ur = (int)(units % ctas);
  gp.split = 0; gp.cluster = 1;
  gp.y_f32 = (y_dtype == ER_F32); gp.ldy = ldy_elems; gp.y = y;
  gp.qweight = nullptr; gp.scales = nullptr;
  gp.counters = reinterpret_cast<int*>(workspace);
  gp.partials = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(workspace) + ER_GEMM_COUNTER_BYTES);
  cudaStream_t s = (cudaStream_t)stream;
  switch (mpad) {
    case 16: return launch<16>(mw, mx, gp, ctas, s);
    case 32: return launch<32>(mw, mx, gp, ctas, s);
    case 64: return launch<64>(mw, mx, gp, ctas, s);
    case 128: return launch<128>(mw, mx, gp, ctas, s);
    default: return launch<256>(mw, mx, gp, ctas, s);
  }
}

}  // extern "C"
