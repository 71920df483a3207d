// spec_verify.cu -- er_spec_verify: speculative-decoding verification by rejection sampling
// (sec. 2.2; L445 sec. D.1: accept drafted tokens, resample at the first rejection "from the
// adjusted target distribution", bonus token when everything is accepted; L544: needs the full
// distribution at the rejected position).
//
// One thread-block CLUSTER (up to 8 CTAs of 256 threads) per sequence: with one CTA per sequence only B of
// the 148 SMs pull bytes (9 % DRAM throughput measured at B = 64, profiles/r01_baseline_ncu.md).  Every CTA
// owns a contiguous range of 2048-token tiles of the vocabulary; rows are streamed with 128-bit loads (8
// consecutive elements per thread).  Per-row softmax normalisers and residual masses are reduced inside the
// CTA, exchanged through distributed shared memory and combined in rank order by every CTA, so all CTAs of
// a cluster take the same decisions.  The statistics of all gamma + 1 positions are computed in ONE sweep with
// one cluster exchange (a lazy scan, stopping at the first rejection, reads less when acceptance is low but
// pays a cluster barrier and a DRAM round trip per position; with the paper's acceptance of ~0.98 every row is
// needed anyway).  The residual draw is a multi-level inverse CDF: per-warp segment sums (256 consecutive
// tokens) -> per-CTA totals, exchanged -> the CTA whose range holds the threshold does an fp64 prefix over
// its segments and a warp scan inside the one segment that contains the threshold.
#include <cooperative_groups.h>
#include "er_common.cuh"

namespace cg = cooperative_groups;

namespace {

constexpr int kThreads = 256;
constexpr int kMaxCluster = 8;
constexpr int kWarps = kThreads / 32;
constexpr int kPerThread = 8;
constexpr int kTile = kThreads * kPerThread;  // 2048 tokens
constexpr int kMaxV = 1 << 20;
constexpr float kNegInf = -3.0e38f;

// ---- 8 consecutive elements starting at token v0 (clipped to V): raw load, then widening to fp32 ----
// (split in two so that the loads of several tiles can be in flight before the first one is consumed)
template <typename T>
struct Load8;
template <>
struct Load8<float> {
  struct Raw { float4 a, b; };
  static constexpr int kBatch = 2;   // tiles whose loads are issued together
  static __device__ __forceinline__ Raw load(const float* row, int v0, int V, bool vec, float fill) {
    Raw r;
    if (vec && v0 + 8 <= V) {
      r.a = *reinterpret_cast<const float4*>(row + v0);
      r.b = *reinterpret_cast<const float4*>(row + v0 + 4);
    } else {
      float f[8];
#pragma unroll
      for (int i = 0; i < 8; ++i) f[i] = (v0 + i < V) ? row[v0 + i] : fill;
      r.a = make_float4(f[0], f[1], f[2], f[3]);
      r.b = make_float4(f[4], f[5], f[6], f[7]);
    }
    return r;
  }
  static __device__ __forceinline__ void expand(const Raw& r, float (&f)[8]) {
    f[0] = r.a.x; f[1] = r.a.y; f[2] = r.a.z; f[3] = r.a.w;
    f[4] = r.b.x; f[5] = r.b.y; f[6] = r.b.z; f[7] = r.b.w;
  }
  static __device__ __forceinline__ float one(const float* row, int v) { return row[v]; }
};
template <>
struct Load8<__nv_bfloat16> {
  struct Raw { uint4 a; };
  static constexpr int kBatch = 4;
  static __device__ __forceinline__ Raw load(const __nv_bfloat16* row, int v0, int V, bool vec, float fill) {
    Raw r;
    if (vec && v0 + 8 <= V) {
      r.a = *reinterpret_cast<const uint4*>(row + v0);
    } else {
      uint32_t h[8];
      const uint32_t fb = __float_as_uint(fill) >> 16;   // the fills used (0, -3e38) survive truncation to bf16
#pragma unroll
      for (int i = 0; i < 8; ++i)
        h[i] = (v0 + i < V) ? (uint32_t)__bfloat16_as_ushort(row[v0 + i]) : fb;
      r.a = make_uint4(h[0] | (h[1] << 16), h[2] | (h[3] << 16), h[4] | (h[5] << 16), h[6] | (h[7] << 16));
    }
    return r;
  }
  static __device__ __forceinline__ void expand(const Raw& r, float (&f)[8]) {
    const uint32_t w[4] = {r.a.x, r.a.y, r.a.z, r.a.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      f[2 * i] = __uint_as_float(w[i] << 16);
      f[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
    }
  }
  static __device__ __forceinline__ float one(const __nv_bfloat16* row, int v) { return __bfloat162float(row[v]); }
};
template <typename T>
__device__ __forceinline__ void load8(const T* row, int v0, int V, bool vec, float fill, float (&f)[8]) {
  Load8<T>::expand(Load8<T>::load(row, v0, V, vec, fill), f);
}

// 2^x by the special-function unit alone (relative error about 2^-22; no range-reduction code around it)
__device__ __forceinline__ float ex2_fast(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

__device__ __forceinline__ float warp_max(float x) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) x = fmaxf(x, __shfl_xor_sync(0xffffffffu, x, o));
  return x;
}
__device__ __forceinline__ float warp_sum(float x) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
  return x;
}

struct RowStats {
  float max;      // max logit of the row
  float inv_sum;  // 1 / sum_v exp((l - max) / T)
};

struct Shared {
  double xmass[2][kMaxCluster];    // [parity][rank]: residual mass of every CTA's range
  float4 wstat[17][kWarps];        // [position][warp]: per-warp (max_t, sum_t, max_d, sum_d) of this CTA's range
  float4 xall[kMaxCluster][17];    // [rank][position]: per-CTA statistics of every CTA of the cluster
  float4 stat[17];                 // [position]: (max_t, 1/sum_t, max_d, 1/sum_d) over the whole vocabulary
  float px[16], qx[16], ua[16];    // target / draft value at the drafted token and the uniform, per position
  int seg;
  int token;
  int flag;
  double thr_local;
};

struct ClusterCtx {
  int rank, size;      // this CTA's rank in the cluster, CTAs per cluster
  int tile_lo, tile_hi;  // its range of kTile-token tiles
  int xpar;            // parity of the next exchange buffer
  bool started;        // the "every CTA of the cluster has started" handshake has been waited for
};

// A CTA's shared memory may be written remotely only once that CTA has started executing: every CTA arrives
// (relaxed) on the cluster barrier at kernel entry, and all threads wait for that phase here, right before the
// first remote store.  Uniform over the CTA; a no-op for clusters of one.
__device__ __forceinline__ void cluster_started(ClusterCtx& cx) {
  if (cx.size > 1 && !cx.started) asm volatile("barrier.cluster.wait.aligned;" ::: "memory");
  cx.started = true;
}

// Softmax statistics (online max / sum of exponentials) of one target row and (optionally) one draft row over
// this CTA's tile range, reduced to one entry per warp in sh.wstat[pos].
template <typename T>
__device__ void row_stats(const T* trow, const T* drow, const T* next_t, const T* next_d, int V, bool vec, float scale,
                          Shared& sh, ClusterCtx& cx, int pos) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  float mt = kNegInf, st_ = 0.f, md = kNegInf, sd_ = 0.f;
  constexpr int NB = Load8<T>::kBatch;
  for (int t0 = cx.tile_lo; t0 < cx.tile_hi; t0 += NB) {
    typename Load8<T>::Raw rt[NB], rd[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) {           // all loads of the batch first: they overlap in flight
      const int v0 = (t0 + j) * kTile + tid * kPerThread;
      if (t0 + j < cx.tile_hi && v0 < V) {
        rt[j] = Load8<T>::load(trow, v0, V, vec, kNegInf);
        if (drow) rd[j] = Load8<T>::load(drow, v0, V, vec, kNegInf);
        // the same tile of the NEXT position goes to L2 now: one position (~80 KB per CTA) of run-ahead, so
        // only the very first batch of the sweep pays a DRAM round trip per warp
        if (next_t) prefetch_l2(next_t + v0);
        if (next_d) prefetch_l2(next_d + v0);
      }
    }
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      const int v0 = (t0 + j) * kTile + tid * kPerThread;
      if (t0 + j < cx.tile_hi && v0 < V) {
        float f[8];
        Load8<T>::expand(rt[j], f);
        float cm = f[0];
#pragma unroll
        for (int i = 1; i < 8; ++i) cm = fmaxf(cm, f[i]);
        if (cm > mt) { st_ *= exp2f((mt - cm) * scale); mt = cm; }
        if (mt > kNegInf) {   // a chunk of masked (-inf) logits before any finite one adds nothing (and -mt * scale
                              // would overflow: fma(-inf, scale, +inf) is NaN)
          const float nt = -mt * scale;
#pragma unroll
          for (int i = 0; i < 8; ++i) st_ += ex2_fast(fmaf(f[i], scale, nt));
        }
        if (drow) {
          Load8<T>::expand(rd[j], f);
          cm = f[0];
#pragma unroll
          for (int i = 1; i < 8; ++i) cm = fmaxf(cm, f[i]);
          if (cm > md) { sd_ *= exp2f((md - cm) * scale); md = cm; }
          if (md > kNegInf) {
            const float nd = -md * scale;
#pragma unroll
            for (int i = 0; i < 8; ++i) sd_ += ex2_fast(fmaf(f[i], scale, nd));
          }
        }
      }
    }
  }
  // warp level only (no CTA barrier per position): max, then the sum of the rescaled partial sums
  const float wm_t = warp_max(mt), wm_d = warp_max(md);
  st_ = (mt > kNegInf) ? st_ * exp2f((mt - wm_t) * scale) : 0.f;
  sd_ = (md > kNegInf) ? sd_ * exp2f((md - wm_d) * scale) : 0.f;
  const float ws_t = warp_sum(st_), ws_d = warp_sum(sd_);
  if (lane == 0) sh.wstat[pos][warp] = make_float4(wm_t, ws_t, wm_d, ws_d);
}

// (max, sum) pairs a and b of two disjoint parts of a row -> the pair of their union
__device__ __forceinline__ void merge_stat(float& m, float& s, float m2, float s2, float scale) {
  const float mm = fmaxf(m, m2);
  const float a = (m > kNegInf) ? s * exp2f((m - mm) * scale) : 0.f;
  const float b = (m2 > kNegInf) ? s2 * exp2f((m2 - mm) * scale) : 0.f;
  m = mm;
  s = a + b;
}

// After row_stats of positions 0..npos-1: combine warps (in order), exchange over the cluster through
// distributed shared memory, combine ranks (in order).  Every CTA ends with the same sh.stat[].
__device__ void combine_stats(int npos, float scale, Shared& sh, ClusterCtx& cx) {
  const int tid = threadIdx.x;
  cg::cluster_group cluster = cg::this_cluster();
  cluster_started(cx);
  __syncthreads();
  if (tid < npos) {
    float mt = kNegInf, st = 0.f, md = kNegInf, sd = 0.f;
    for (int w = 0; w < kWarps; ++w) {
      const float4 v = sh.wstat[tid][w];
      merge_stat(mt, st, v.x, v.y, scale);
      merge_stat(md, sd, v.z, v.w, scale);
    }
    const float4 mine = make_float4(mt, st, md, sd);
    for (int c = 0; c < cx.size; ++c) *cluster.map_shared_rank(&sh.xall[cx.rank][tid], c) = mine;
  }
  cluster.sync();
  if (tid < npos) {
    float mt = kNegInf, st = 0.f, md = kNegInf, sd = 0.f;
    for (int c = 0; c < cx.size; ++c) {
      const float4 v = sh.xall[c][tid];
      merge_stat(mt, st, v.x, v.y, scale);
      merge_stat(md, sd, v.z, v.w, scale);
    }
    sh.stat[tid] = make_float4(mt, __fdiv_rn(1.0f, st), md, sd > 0.f ? __fdiv_rn(1.0f, sd) : 0.f);
  }
  __syncthreads();
}

// The 8 residual weights of one thread chunk from its raw loads.  use_q == false: w = p (bonus token /
// degenerate residual).
template <typename T, bool kLogits>
__device__ __forceinline__ void weights8_raw(const typename Load8<T>::Raw& rp, const typename Load8<T>::Raw& rq,
                                             float scale, const RowStats& st, const RowStats& sd, bool use_q,
                                             float (&w)[8]) {
  float p[8];
  Load8<T>::expand(rp, p);
  if (kLogits) {
#pragma unroll
    const float nt = -st.max * scale;
#pragma unroll
    for (int i = 0; i < 8; ++i) p[i] = ex2_fast(fmaf(p[i], scale, nt)) * st.inv_sum;
  }
  if (use_q) {
    float q[8];
    Load8<T>::expand(rq, q);
    if (kLogits) {
#pragma unroll
      const float nd = -sd.max * scale;
#pragma unroll
      for (int i = 0; i < 8; ++i) q[i] = ex2_fast(fmaf(q[i], scale, nd)) * sd.inv_sum;
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) w[i] = fmaxf(0.f, p[i] - q[i]);
  } else {
#pragma unroll
    for (int i = 0; i < 8; ++i) w[i] = p[i];
  }
}
template <typename T, bool kLogits>
__device__ __forceinline__ void weights8(const T* trow, const T* drow, int v0, int V, bool vec, float scale,
                                         const RowStats& st, const RowStats& sd, bool use_q, float (&w)[8]) {
  const float fill = kLogits ? kNegInf : 0.f;
  typename Load8<T>::Raw rp = Load8<T>::load(trow, v0, V, vec, fill), rq = rp;
  if (use_q) rq = Load8<T>::load(drow, v0, V, vec, fill);
  weights8_raw<T, kLogits>(rp, rq, scale, st, sd, use_q, w);
}

// Inverse-CDF draw over w in vocab order: token = min{v : C(v) > r R}.  Returns -1 in every CTA of the cluster
// if R == 0; otherwise the token in the CTA whose tile range holds the threshold and -2 in the others.
template <typename T, bool kLogits>
__device__ int draw_token(const T* trow, const T* drow, int V, bool vec, float scale, const RowStats& st,
                          const RowStats& sd, bool use_q, float r, Shared& sh, ClusterCtx& cx, float* seg_sums) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int ntile = cx.tile_hi - cx.tile_lo;
  // level 1: sums of 256-token segments (one warp, one tile each) of this CTA's range
  constexpr int NB = Load8<T>::kBatch;
  const float fill = kLogits ? kNegInf : 0.f;
  for (int t0 = 0; t0 < ntile; t0 += NB) {
    typename Load8<T>::Raw rp[NB], rq[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) {           // all loads of the batch first: they overlap in flight
      const int v0 = (cx.tile_lo + t0 + j) * kTile + tid * kPerThread;
      if (t0 + j < ntile && v0 < V) {
        rp[j] = Load8<T>::load(trow, v0, V, vec, fill);
        if (use_q) rq[j] = Load8<T>::load(drow, v0, V, vec, fill);
      }
    }
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      if (t0 + j < ntile) {                  // uniform over the CTA
        const int v0 = (cx.tile_lo + t0 + j) * kTile + tid * kPerThread;
        float s = 0.f;
        if (v0 < V) {
          float w[8];
          weights8_raw<T, kLogits>(rp[j], use_q ? rq[j] : rp[j], scale, st, sd, use_q, w);
          s = ((w[0] + w[1]) + (w[2] + w[3])) + ((w[4] + w[5]) + (w[6] + w[7]));
        }
        s = warp_sum(s);
        if (lane == 0) seg_sums[(t0 + j) * kWarps + warp] = s;
      }
    }
  }
  __syncthreads();
  // level 2a: this CTA's mass (fp64, vocab order), published to the whole cluster
  cg::cluster_group cluster = cg::this_cluster();
  const int par = cx.xpar;
  cx.xpar ^= 1;
  const int nseg = ntile * kWarps;
  cluster_started(cx);
  if (warp == 0) {
    double mine = 0.0;                       // lane-strided partial sums, then a butterfly: the same value in
    for (int i = lane; i < nseg; i += 32) mine += (double)seg_sums[i];   // every lane, in a fixed order
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mine += __shfl_xor_sync(0xffffffffu, mine, o);
    if (lane < cx.size) *cluster.map_shared_rank(&sh.xmass[par][cx.rank], lane) = mine;
  }
  cluster.sync();
  // level 2b: every CTA finds, identically, the rank whose range holds the threshold
  double R = 0.0;
  for (int c = 0; c < cx.size; ++c) R += sh.xmass[par][c];
  if (!(R > 0.0)) return -1;
  const double thr = (double)r * R;
  int owner = cx.size - 1;
  double before = 0.0;
  {
    double c0 = 0.0;
    for (int c = 0; c < cx.size; ++c) {
      const double nc = c0 + sh.xmass[par][c];
      if (nc > thr) { owner = c; break; }
      c0 = nc;
    }
    // if rounding left no rank (cannot happen for r < 1), fall to the last rank with mass
    while (owner > 0 && !(sh.xmass[par][owner] > 0.0)) --owner;
    for (int c = 0; c < owner; ++c) before += sh.xmass[par][c];
  }
  if (owner != cx.rank) return -2;
  // level 2c (owner only): fp64 prefix over its segments in vocab order by one thread
  if (tid == 0) {
    const double thr_cta = thr - before;
    double c = 0.0;
    int seg = -1;
    for (int i = 0; i < nseg; ++i) {
      const double nc = c + (double)seg_sums[i];
      if (nc > thr_cta) { seg = i; break; }
      c = nc;
    }
    if (seg < 0) {      // rounding left no segment (the rank was chosen from a differently ordered sum): take
      seg = nseg - 1;   // the last segment with mass and recompute its exclusive prefix
      while (seg > 0 && !(seg_sums[seg] > 0.f)) --seg;
      c = 0.0;
      for (int i = 0; i < seg; ++i) c += (double)seg_sums[i];
    }
    sh.thr_local = thr_cta - c;
    sh.seg = seg;
    sh.token = -1;
  }
  __syncthreads();
  const int seg = sh.seg;
  // level 3: warp scan inside the chosen 256-token segment
  if (warp == 0) {
    const int v0 = (cx.tile_lo + seg / kWarps) * kTile + (seg % kWarps) * 256 + lane * kPerThread;
    float w[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) w[i] = 0.f;
    if (v0 < V) weights8<T, kLogits>(trow, drow, v0, V, vec, scale, st, sd, use_q, w);
    float incl[8];
    float run = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) { run += w[i]; incl[i] = run; }
    float pre = run;  // inclusive scan of lane totals
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const float up = __shfl_up_sync(0xffffffffu, pre, o);
      if (lane >= o) pre += up;
    }
    const float excl = pre - run;
    const float thr = (float)sh.thr_local;
    int first = 8;
#pragma unroll
    for (int i = 7; i >= 0; --i)
      if (excl + incl[i] > thr && w[i] > 0.f) first = i;
    const unsigned hit = __ballot_sync(0xffffffffu, first < 8);
    int last_pos = -1;  // last element with mass, for the rounding fallback
#pragma unroll
    for (int i = 0; i < 8; ++i)
      if (w[i] > 0.f) last_pos = v0 + i;
    int tok;
    if (hit) {
      const int src = __ffs(hit) - 1;
      tok = __shfl_sync(0xffffffffu, v0 + first, src);
    } else {
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) last_pos = max(last_pos, __shfl_xor_sync(0xffffffffu, last_pos, o));
      tok = last_pos;
    }
    if (lane == 0) sh.token = tok;
  }
  __syncthreads();
  return sh.token;
}

template <typename T, bool kLogits>
__global__ void __launch_bounds__(kThreads, 4)
spec_verify_kernel(const T* __restrict__ target, const T* __restrict__ draft, float scale,
                   const int32_t* __restrict__ draft_tokens, const float* __restrict__ u_accept,
                   const float* __restrict__ u_sample, int gamma, int V, int32_t* __restrict__ accept_count,
                   int32_t* __restrict__ out_tokens) {
  extern __shared__ float seg_sums[];
  __shared__ Shared sh;
  cg::cluster_group cluster = cg::this_cluster();
  ClusterCtx cx;
  cx.size = (int)cluster.num_blocks();
  cx.rank = (int)cluster.block_rank();
  cx.xpar = 0;
  cx.started = false;
  if (cx.size > 1) asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory");   // "I have started"
  const int tiles = (V + kTile - 1) / kTile;
  const int per = (tiles + cx.size - 1) / cx.size;
  cx.tile_lo = min(cx.rank * per, tiles);
  cx.tile_hi = min(cx.tile_lo + per, tiles);
  const int b = blockIdx.x / cx.size, tid = threadIdx.x;
  const bool vec = ((size_t)V * sizeof(T)) % 16 == 0;
  const T* tgt = target + (size_t)b * (gamma + 1) * V;
  const T* drf = draft + (size_t)b * gamma * V;
  const int32_t* xs = draft_tokens + (size_t)b * gamma;

  if (tid < gamma) {           // everything the accept tests read, fetched once, off the per-position critical path
    const int x = min(max(xs[tid], 0), V - 1);
    sh.px[tid] = Load8<T>::one(tgt + (size_t)tid * V, x);
    sh.qx[tid] = Load8<T>::one(drf + (size_t)tid * V, x);
    sh.ua[tid] = u_accept[(size_t)b * gamma + tid];
  }
  __syncthreads();

  // Statistics of ALL gamma + 1 positions in one sweep and one cluster exchange.  (A lazy scan would skip the rows
  // behind the first rejection, but costs a cluster barrier and a DRAM round trip per position; in the paper's
  // regime nearly every drafted token is accepted, so those rows are needed anyway.)
  if (kLogits) {
    for (int t = cx.tile_lo; t < cx.tile_hi; ++t) {     // position 0: everything behind the first batch to L2
      const int v0 = t * kTile + tid * kPerThread;
      if (v0 < V) { prefetch_l2(tgt + v0); prefetch_l2(drf + v0); }
    }
    for (int i = 0; i <= gamma; ++i)
      row_stats<T>(tgt + (size_t)i * V, i < gamma ? drf + (size_t)i * V : nullptr,
                   i < gamma ? tgt + (size_t)(i + 1) * V : nullptr, i + 1 < gamma ? drf + (size_t)(i + 1) * V : nullptr,
                   V, vec, scale, sh, cx, i);
    combine_stats(gamma + 1, scale, sh, cx);
  }
  if (tid == 0) {              // every CTA of the cluster takes the same decisions from the same numbers
    int k = 0;
    for (; k < gamma; ++k) {
      float p = sh.px[k], q = sh.qx[k];
      if (kLogits) {
        const float4 v = sh.stat[k];
        p = exp2f((p - v.x) * scale) * v.y;
        q = exp2f((q - v.z) * scale) * v.w;
      }
      const float lhs = __fmul_rn(sh.ua[k], q);
      if (!(lhs < p)) break;
    }
    sh.flag = k;
  }
  __syncthreads();
  const int n = sh.flag;
  RowStats st{0.f, 1.f}, sd{0.f, 1.f};
  if (kLogits) {
    const float4 v = sh.stat[n];
    st.max = v.x; st.inv_sum = v.y; sd.max = v.z; sd.inv_sum = v.w;
  }
  const T* trow = tgt + (size_t)n * V;
  const T* drow = (n < gamma) ? drf + (size_t)n * V : nullptr;
  const float r = u_sample[b];
  int tok = draw_token<T, kLogits>(trow, drow, V, vec, scale, st, sd, n < gamma, r, sh, cx, seg_sums);
  if (tok == -1) tok = draw_token<T, kLogits>(trow, nullptr, V, vec, scale, st, sd, false, r, sh, cx, seg_sums);
  if (tok == -1) tok = (cx.rank == 0) ? V - 1 : -2;  // all-zero target row: outside the contract, stay memory-safe
  if (tok == -2) return;                             // another CTA of the cluster owns the draw and the outputs
  if (tid == 0) accept_count[b] = n;
  if (tid <= gamma) {
    int32_t o = -1;
    if (tid < n) o = xs[tid];
    else if (tid == n) o = tok;
    out_tokens[(size_t)b * (gamma + 1) + tid] = o;
  }
}

template <typename T, bool kLogits>
int launch_verify(int cluster_size, size_t smem, cudaStream_t s, const T* target, const T* draft, float scale,
                  const int32_t* draft_tokens, const float* u_accept, const float* u_sample, int B, int gamma, int V,
                  int32_t* accept_count, int32_t* out_tokens) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(B * cluster_size));
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)cluster_size;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  ER_CUDA_TRY(cudaLaunchKernelEx(&cfg, spec_verify_kernel<T, kLogits>, target, draft, scale, draft_tokens, u_accept,
                                 u_sample, gamma, V, accept_count, out_tokens));
  return ER_OK;
}

#ifdef ER_DEV
int g_force_cluster = 0;   // development library only (er_dev.h): 0 = automatic
#else
constexpr int g_force_cluster = 0;
#endif

}  // namespace

#ifdef ER_DEV
extern "C" int er_dev_verify_cluster(int cluster) {
  if (cluster != 0 && cluster != 1 && cluster != 2 && cluster != 4 && cluster != 8) return ER_ERR_SHAPE;
  g_force_cluster = cluster;
  return ER_OK;
}
#endif

extern "C" int er_spec_verify(const void* target, const void* draft, int in_dtype, int inputs_are_logits,
                              float temperature, const int32_t* draft_tokens, const float* u_accept,
                              const float* u_sample, int32_t B, int32_t gamma, int32_t V, int32_t* accept_count,
                              int32_t* out_tokens, void* stream) {
  if (B < 0 || gamma < 1 || gamma > 16 || V < 1 || V > kMaxV) return ER_ERR_SHAPE;
  if (in_dtype != ER_BF16 && in_dtype != ER_F32) return ER_ERR_DTYPE;
  if (in_dtype == ER_BF16 && !inputs_are_logits) return ER_ERR_DTYPE;
  if (inputs_are_logits && !(temperature > 0.0f)) return ER_ERR_SHAPE;
  if (B == 0) return ER_OK;
  if (!target || !draft || !draft_tokens || !u_accept || !u_sample || !accept_count || !out_tokens) return ER_ERR_NULL;
  if (!er::aligned16(target) || !er::aligned16(draft)) return ER_ERR_ALIGN;
  int st = er::check_arch();
  if (st != ER_OK) return st;
  const int tiles = (V + kTile - 1) / kTile;
  int cluster = tiles >= 8 ? 8 : (tiles >= 4 ? 4 : (tiles >= 2 ? 2 : 1));   // CTAs per sequence
  if (g_force_cluster > 0 && g_force_cluster <= cluster) cluster = g_force_cluster;
  const int per = (tiles + cluster - 1) / cluster;
  const size_t smem = (size_t)per * kWarps * sizeof(float);
  const float scale = (float)(1.4426950408889634 / (double)temperature);
  cudaStream_t s = (cudaStream_t)stream;
  int rc;
  if (in_dtype == ER_F32 && !inputs_are_logits) {
    rc = launch_verify<float, false>(cluster, smem, s, (const float*)target, (const float*)draft, scale, draft_tokens,
                                     u_accept, u_sample, B, gamma, V, accept_count, out_tokens);
  } else if (in_dtype == ER_F32) {
    rc = launch_verify<float, true>(cluster, smem, s, (const float*)target, (const float*)draft, scale, draft_tokens,
                                    u_accept, u_sample, B, gamma, V, accept_count, out_tokens);
  } else {
    rc = launch_verify<__nv_bfloat16, true>(cluster, smem, s, (const __nv_bfloat16*)target,
                                            (const __nv_bfloat16*)draft, scale, draft_tokens, u_accept, u_sample, B,
                                            gamma, V, accept_count, out_tokens);
  }
  if (rc != ER_OK) return rc;
  ER_CUDA_TRY(cudaGetLastError());
  return ER_OK;
}
