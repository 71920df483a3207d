// w4a16_plan.cuh -- what the two W4A16 GEMM kernels (w4a16_gemm_small.cu: M <= 16, warp-level MMA;
// w4a16_gemm.cu: M > 16, tcgen05 / TMEM) share: the kernel parameter block, the work partition and the
// host-side plan.  Product path only (the CPU oracle shares nothing with this).
#pragma once
#include <cuda.h>
#include "er_common.cuh"

namespace er {

constexpr int kTileN = 128;                 // weight rows per tile
constexpr int kWBytes = kTileN * 64;        // 8 KiB packed weights per (tile, group) block
constexpr int kScaleBytes = kTileN * 2;     // 128 bf16 scales
constexpr int kSmemLimit = 227 * 1024;

struct GemmParams {
  int M, N, K;
  int G;               // groups per tile = K / 128
  int ntiles;          // N / 128
  int tiles;           // ntiles * mchunks
  int mchunks;         // chunks of MPAD batch rows (tile t = chunk t / ntiles of weight tile t % ntiles)
  int unit_groups;     // groups per scheduling unit: 1 (stream-K) or G (whole tiles)
  int units;           // tiles * G / unit_groups (< 2^31, checked on the host)
  int uq, ur;          // units / CTAs and units % CTAs: CTA c owns units [c*uq + min(c, ur), ...)
  int split;           // > 0: tile split (see range_begin); uq = groups per tile
  int cluster;         // > 1: the `split` CTAs of a tile form one thread-block cluster and reduce through DSMEM
  int planes;          // 1: W8 stored as two nibble planes (er_w8a16_gemm): groups 2g, 2g + 1 share the X of group g,
                       // the even (high-nibble) plane carries no offset, the odd one the whole of it (w4a16_gemm.cu)
  int y_f32;
  int64_t ldy;
  void* y;
  const uint8_t* qweight;  // ER_PACK_V2 blocks
  const uint8_t* scales;   // bf16 [G][N]
  float* partials;     // workspace + ER_GEMM_COUNTER_BYTES: [cta][2][MPAD][128]
  int* counters;       // workspace: one ticket per tile
};

// Work partition (32-bit arithmetic only).  split == 0 ("stream-K"): the units are dealt to the CTAs as contiguous,
// balanced ranges -- the first `ur` CTAs get uq + 1 units, the others uq.  split == k > 0 ("tile split", chosen when
// tiles * k CTAs fit the SMs): CTA c owns part c % k of tile c / k, so no CTA straddles two tiles (one segment, one
// partial sum, one ticket per CTA) -- only for unit_groups == 1; uq then holds the groups per tile.
__host__ __device__ __forceinline__ int range_begin(int uq, int ur, int split, int c) {
  if (split > 0) {
    const int t = c / split, j = c - t * split;
    return t * uq + (j * uq) / split;
  }
  return c * uq + (c < ur ? c : ur);
}
// the CTA whose range contains unit u
__host__ __device__ __forceinline__ int owner_of(int uq, int ur, int split, int u) {
  if (split > 0) {
    const int t = u / uq, g = u - t * uq;
    int j = (g * split) / uq;                        // close; fix up against the exact boundaries
    while (j + 1 < split && ((j + 1) * uq) / split <= g) ++j;
    while (j > 0 && (j * uq) / split > g) --j;
    return t * split + j;
  }
  const int big = ur * (uq + 1);
  return u < big ? u / (uq + 1) : ur + (u - big) / uq;
}

struct Plan {
  int mpad, mchunks, ntiles, tiles, G, unit_groups, ctas, split, cluster;
  long long units;
};

// Development knobs: constants in the shipped library; variables (set through er_dev.h) only in the
// development build (-DER_DEV, liber_b200_dev.so), which the partition / launch-mode tests load explicitly.
struct Tuning {
  int pdl;          // programmatic dependent launch
  int split;        // tile split where it applies
  int cluster;      // cluster mode where it applies
  int force_ctas;   // > 0: use this many CTAs; 0 = one per SM
  int small_mma;    // M <= 8 without a cluster through the warp-level-MMA kernel (0: through the tcgen05 kernel)
  int large;        // 1: the pre-scaled large-batch kernel where it is preferred (M > 64, whole tiles); 0: never;
                    // 2: for every M > 16 (tests)
  int wide;         // M > 64 through the 128-row kernel (w4a16_gemm_wide.cu): 1 where the plan prefers it, 2 always;
                    // 0: in chunks of 64 rows (w4a16_gemm.cu)
  int units;        // M > 64: 0 = plan's choice, 1 = whole tiles, 2 = stream-K ranges (tests / measurements)
};
#ifdef ER_DEV
extern Tuning g_tune;
#else
constexpr Tuning g_tune = {1, 1, 1, 0, 1, 0, 1, 0};
#endif

// 2-D row-major tensor [rows][cols] of elements, row pitch in bytes, box [box_rows][box_cols].
bool make_map_2d(CUtensorMap* map, CUtensorMapDataType dt, const void* base, uint64_t rows, uint64_t cols,
                 uint64_t pitch_bytes, uint32_t box_rows, uint32_t box_cols, CUtensorMapSwizzle swz);

// M <= 8, no cluster: w4a16_gemm_small.cu
int launch_small(const void* x, int64_t M, int64_t K, int64_t ldx, GemmParams gp, const Plan& pl, cudaStream_t stream);

// M > 64: w4a16_gemm_wide.cu
size_t wide_workspace_bytes();
int launch_wide(const void* x, int64_t M, int64_t N, int64_t K, int64_t ldx, GemmParams gp, bool whole, int split,
                cudaStream_t stream);

// M > 16, development library only: w4a16_gemm_large.cu
int large_mpad_of(int64_t M);
size_t large_workspace_bytes(int64_t M, int64_t N, int64_t K);
bool large_preferred(int64_t M, int64_t N, int64_t K);
int launch_large(const void* x, int64_t M, int64_t N, int64_t K, int64_t ldx, GemmParams gp, cudaStream_t stream);

}  // namespace er
