// spec_verify.cu -- er_spec_verify: speculative-decoding verification by rejection sampling
// (sec. 2.2; L445 sec. D.1: accept drafted tokens, resample at the first rejection "from the
// adjusted target distribution", bonus token when everything is accepted; L544: needs the full
// distribution at the rejected position).
//
// One thread-block CLUSTER of 1024-thread CTAs per sequence, ONE CTA PER SM: the vocabulary is split into 256-token
// segments (one 128-bit load per lane of a warp) and every CTA of the cluster owns a contiguous, balanced range of
// them.  The cluster size (1, 2, 4 or 8) is the one that keeps the most SMs busy for the given B (B = 64: clusters
// of 2 -> 128 CTAs, one wave, every SM the same 1.37 MB; round 1 used clusters of 8 x 256 threads, four per SM at
// most, which left some SMs with twice the work of others: profiles/r02_ncu.md).  Per-row softmax normalisers and
// residual masses are reduced inside the CTA, exchanged through distributed shared memory and combined in rank
// order by every CTA, so all CTAs of a cluster take the same decisions.  The statistics of all gamma + 1
// positions are computed in ONE sweep with one cluster exchange (a lazy scan, stopping at the first rejection,
// reads less when acceptance is low but pays a cluster barrier and a DRAM round trip per position; with the
// paper's acceptance of ~0.98 every row is needed anyway).  The sweep is bound by the special-function unit
// (one ex2 per logit, 16 per clock and SM) and by HBM about equally, so everything else in its loop is kept
// small: the running maximum of a bf16 row is tracked on the packed words (4 max.bf16x2 per 8 logits, no
// unpacking), and the segments of consecutive rows are dealt to the warps in rotation so that no warp carries
// the ragged tail of every row.  The residual draw is a multi-level inverse CDF: per-warp segment sums ->
// per-CTA totals, exchanged -> the CTA whose range holds the threshold does an fp64 blocked prefix over its
// segments (one warp) and a warp scan inside the one segment that contains the threshold.
#include <cooperative_groups.h>
#include <cuda_bf16.h>
#include "er_common.cuh"

namespace cg = cooperative_groups;

namespace {

#ifndef ER_VERIFY_THREADS
#define ER_VERIFY_THREADS 1024
#endif
constexpr int kThreads = ER_VERIFY_THREADS;
constexpr int kMaxCluster = 8;
constexpr int kWarps = kThreads / 32;
constexpr int kPerThread = 8;
constexpr int kSeg = 32 * kPerThread;         // 256 tokens: what one warp loads at once
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
  int token;
  int flag;
};

struct ClusterCtx {
  int rank, size;      // this CTA's rank in the cluster, CTAs per cluster
  int seg_lo, seg_hi;  // its range of kSeg-token segments
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

// Online softmax statistics of one lane: running maximum m, sum s of 2^((l - m) * scale), nm = -m * scale.
// run2 (bf16 rows only) is the running maximum on the packed words, lane-wise over the two halves.
struct Acc {
  float m, s, nm;
  uint32_t run2;
  __device__ __forceinline__ void init() { m = kNegInf; s = 0.f; nm = 0.f; run2 = 0xFF80FF80u; }   // (-inf, -inf)
  __device__ __forceinline__ void raise(float cm, float scale) {
    if (cm > m) { s *= ex2_fast((m - cm) * scale); m = cm; nm = -cm * scale; }
  }
};

__device__ __forceinline__ uint32_t max_bf16x2(uint32_t a, uint32_t b) {
  uint32_t d;
  asm("max.bf16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
  return d;
}

template <typename T>
struct Accum;
template <>
struct Accum<float> {
  static __device__ __forceinline__ void add(const Load8<float>::Raw& r, Acc& a, float scale) {
    float f[8];
    Load8<float>::expand(r, f);
    float cm = fmaxf(fmaxf(fmaxf(f[0], f[1]), fmaxf(f[2], f[3])), fmaxf(fmaxf(f[4], f[5]), fmaxf(f[6], f[7])));
    a.raise(cm, scale);
    if (a.m > kNegInf) {   // masked (-inf) logits before any finite one add nothing (and -m * scale would
                           // overflow: fma(-inf, scale, +inf) is NaN)
      float s0 = 0.f, s1 = 0.f;
#pragma unroll
      for (int i = 0; i < 8; i += 2) {
        s0 += ex2_fast(fmaf(f[i], scale, a.nm));
        s1 += ex2_fast(fmaf(f[i + 1], scale, a.nm));
      }
      a.s += s0 + s1;
    }
  }
};
template <>
struct Accum<__nv_bfloat16> {
  static __device__ __forceinline__ void add(const Load8<__nv_bfloat16>::Raw& r, Acc& a, float scale) {
    const uint32_t n2 = max_bf16x2(max_bf16x2(max_bf16x2(r.a.x, r.a.y), max_bf16x2(r.a.z, r.a.w)), a.run2);
    if (n2 != a.run2) {    // rare after the first few segments
      a.run2 = n2;
      a.raise(fmaxf(__uint_as_float(n2 << 16), __uint_as_float(n2 & 0xFFFF0000u)), scale);
    }
    if (a.m > kNegInf) {
      const uint32_t w[4] = {r.a.x, r.a.y, r.a.z, r.a.w};
      float s0 = 0.f, s1 = 0.f;
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        s0 += ex2_fast(fmaf(__uint_as_float(w[i] << 16), scale, a.nm));
        s1 += ex2_fast(fmaf(__uint_as_float(w[i] & 0xFFFF0000u), scale, a.nm));
      }
      a.s += s0 + s1;
    }
  }
};

// Softmax statistics of one target row and (optionally) one draft row over this CTA's segment range, reduced to
// one entry per warp in sh.wstat[pos].  Warp w takes the local segments (w - rot) mod kWarps, + kWarps, ...;
// rot advances with the position by the size of the ragged remainder, so the extra segment of a row goes to
// different warps in consecutive rows.
template <typename T>
__device__ void row_stats(const T* trow, const T* drow, int V, bool vec, float scale, Shared& sh,
                          const ClusterCtx& cx, int pos) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nloc = cx.seg_hi - cx.seg_lo;
  const int rot = (pos * (nloc % kWarps)) % kWarps;
  int first = warp - rot;
  if (first < 0) first += kWarps;
  Acc at, ad;
  at.init();
  ad.init();
  constexpr int NB = Load8<T>::kBatch;
  for (int s0 = first; s0 < nloc; s0 += NB * kWarps) {
    typename Load8<T>::Raw rt[NB], rd[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) {           // all loads of the batch first: they overlap in flight
      const int v0 = (cx.seg_lo + s0 + j * kWarps) * kSeg + lane * kPerThread;
      if (s0 + j * kWarps < nloc && v0 < V) {
        rt[j] = Load8<T>::load(trow, v0, V, vec, kNegInf);
        if (drow) rd[j] = Load8<T>::load(drow, v0, V, vec, kNegInf);
      }
    }
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      const int v0 = (cx.seg_lo + s0 + j * kWarps) * kSeg + lane * kPerThread;
      if (s0 + j * kWarps < nloc && v0 < V) {
        Accum<T>::add(rt[j], at, scale);
        if (drow) Accum<T>::add(rd[j], ad, scale);
      }
    }
  }
  // warp level only (no CTA barrier per position): max, then the sum of the rescaled partial sums
  const float wm_t = warp_max(at.m), wm_d = warp_max(ad.m);
  const float st_ = (at.m > kNegInf) ? at.s * ex2_fast((at.m - wm_t) * scale) : 0.f;
  const float sd_ = (ad.m > kNegInf) ? ad.s * ex2_fast((ad.m - wm_d) * scale) : 0.f;
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

// After row_stats of positions 0..npos-1: combine the warps of a position (one warp per position, a fixed
// shuffle tree), exchange over the cluster through distributed shared memory, combine ranks (in order).  Every
// CTA ends with the same sh.stat[].
__device__ void combine_stats(int npos, float scale, Shared& sh, ClusterCtx& cx) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  cg::cluster_group cluster = cg::this_cluster();
  cluster_started(cx);
  __syncthreads();
  for (int p = warp; p < npos; p += kWarps) {
    const float4 v = (lane < kWarps) ? sh.wstat[p][lane] : make_float4(kNegInf, 0.f, kNegInf, 0.f);
    const float mt = warp_max(v.x), md = warp_max(v.z);
    const float st = warp_sum(v.x > kNegInf ? v.y * exp2f((v.x - mt) * scale) : 0.f);
    const float sd = warp_sum(v.z > kNegInf ? v.w * exp2f((v.z - md) * scale) : 0.f);
    if (lane < cx.size) *cluster.map_shared_rank(&sh.xall[cx.rank][p], lane) = make_float4(mt, st, md, sd);
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
    const float nt = -st.max * scale;
#pragma unroll
    for (int i = 0; i < 8; ++i) p[i] = ex2_fast(fmaf(p[i], scale, nt)) * st.inv_sum;
  }
  if (use_q) {
    float q[8];
    Load8<T>::expand(rq, q);
    if (kLogits) {
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
// if R == 0; otherwise the token in the CTA whose segment range holds the threshold and -2 in the others.
template <typename T, bool kLogits>
__device__ int draw_token(const T* trow, const T* drow, int V, bool vec, float scale, const RowStats& st,
                          const RowStats& sd, bool use_q, float r, Shared& sh, ClusterCtx& cx, float* seg_sums) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nloc = cx.seg_hi - cx.seg_lo;
  // level 1: sums of this CTA's 256-token segments, one warp each
  constexpr int NB = Load8<T>::kBatch;
  const float fill = kLogits ? kNegInf : 0.f;
  for (int s0 = warp; s0 < nloc; s0 += NB * kWarps) {
    typename Load8<T>::Raw rp[NB], rq[NB];
#pragma unroll
    for (int j = 0; j < NB; ++j) {           // all loads of the batch first: they overlap in flight
      const int v0 = (cx.seg_lo + s0 + j * kWarps) * kSeg + lane * kPerThread;
      if (s0 + j * kWarps < nloc && v0 < V) {
        rp[j] = Load8<T>::load(trow, v0, V, vec, fill);
        if (use_q) rq[j] = Load8<T>::load(drow, v0, V, vec, fill);
      }
    }
#pragma unroll
    for (int j = 0; j < NB; ++j) {
      if (s0 + j * kWarps < nloc) {          // uniform over the warp
        const int v0 = (cx.seg_lo + s0 + j * kWarps) * kSeg + lane * kPerThread;
        float s = 0.f;
        if (v0 < V) {
          float w[8];
          weights8_raw<T, kLogits>(rp[j], use_q ? rq[j] : rp[j], scale, st, sd, use_q, w);
          s = ((w[0] + w[1]) + (w[2] + w[3])) + ((w[4] + w[5]) + (w[6] + w[7]));
        }
        s = warp_sum(s);
        if (lane == 0) seg_sums[s0 + j * kWarps] = s;
      }
    }
  }
  __syncthreads();
  // level 2a (warp 0): fp64 prefix over the segments in vocab order -- lane l sums the block [l blk, (l+1) blk)
  // sequentially, then an inclusive scan over the lanes; the last lane's value is this CTA's mass, published to
  // the whole cluster
  cg::cluster_group cluster = cg::this_cluster();
  const int par = cx.xpar;
  cx.xpar ^= 1;
  cluster_started(cx);
  const int blk = (nloc + 31) / 32;
  const int i_lo = min(lane * blk, nloc), i_hi = min(i_lo + blk, nloc);
  double incl = 0.0, excl = 0.0;
  if (warp == 0) {
    double mine = 0.0;
    for (int i = i_lo; i < i_hi; ++i) mine += (double)seg_sums[i];
    incl = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const double up = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += up;
    }
    excl = __shfl_up_sync(0xffffffffu, incl, 1);
    if (lane == 0) excl = 0.0;
    const double total = __shfl_sync(0xffffffffu, incl, 31);
    if (lane < cx.size) *cluster.map_shared_rank(&sh.xmass[par][cx.rank], lane) = total;
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
  if (warp == 0) {
    // level 2c (owner only): the lane whose block holds the threshold walks its block
    const double thr_cta = thr - before;
    const unsigned holds = __ballot_sync(0xffffffffu, incl > thr_cta && i_hi > i_lo);
    const unsigned has_mass = __ballot_sync(0xffffffffu, incl > excl);
    // rounding may leave no lane (the rank was chosen from a differently ordered sum): the last lane with mass
    const int src = holds ? __ffs(holds) - 1 : (has_mass ? 31 - __clz(has_mass) : 0);
    int seg = -1;
    double c = excl;
    if (lane == src) {
      for (int i = i_lo; i < i_hi; ++i) {
        const double nc = c + (double)seg_sums[i];
        if (nc > thr_cta) { seg = i; break; }
        c = nc;
      }
      if (seg < 0) {      // same rounding case inside the block: its last segment with mass, prefix recomputed
        seg = max(i_hi - 1, i_lo);
        while (seg > i_lo && !(seg_sums[seg] > 0.f)) --seg;
        c = excl;
        for (int i = i_lo; i < seg; ++i) c += (double)seg_sums[i];
      }
    }
    seg = __shfl_sync(0xffffffffu, seg, src);
    const float thr_seg = (float)(thr_cta - __shfl_sync(0xffffffffu, c, src));
    // level 3: warp scan inside the chosen 256-token segment
    const int v0 = (cx.seg_lo + seg) * kSeg + lane * kPerThread;
    float w[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) w[i] = 0.f;
    if (v0 < V) weights8<T, kLogits>(trow, drow, v0, V, vec, scale, st, sd, use_q, w);
    float incl8[8];
    float run = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) { run += w[i]; incl8[i] = run; }
    float pre = run;  // inclusive scan of lane totals
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const float up = __shfl_up_sync(0xffffffffu, pre, o);
      if (lane >= o) pre += up;
    }
    const float excl8 = pre - run;
    int first = 8;
#pragma unroll
    for (int i = 7; i >= 0; --i)
      if (excl8 + incl8[i] > thr_seg && w[i] > 0.f) first = i;
    const unsigned hit = __ballot_sync(0xffffffffu, first < 8);
    int last_pos = -1;  // last element with mass, for the rounding fallback
#pragma unroll
    for (int i = 0; i < 8; ++i)
      if (w[i] > 0.f) last_pos = v0 + i;
    int tok;
    if (hit) {
      tok = __shfl_sync(0xffffffffu, v0 + first, __ffs(hit) - 1);
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
__global__ void __launch_bounds__(kThreads, 1)
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
  const int nseg = (V + kSeg - 1) / kSeg;
  cx.seg_lo = (int)(((long long)nseg * cx.rank) / cx.size);         // balanced to one segment
  cx.seg_hi = (int)(((long long)nseg * (cx.rank + 1)) / cx.size);
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
    for (int i = 0; i <= gamma; ++i)
      row_stats<T>(tgt + (size_t)i * V, i < gamma ? drf + (size_t)i * V : nullptr, V, vec, scale, sh, cx, i);
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

// CTAs that can be resident at once when launched in clusters of c (one 1024-thread CTA per SM; clusters of 4 / 8
// cannot use every SM of every GPC).  Cached per device.
int resident_ctas(int c) {
  static int cache[er::kMaxDevices][kMaxCluster + 1];
  if (c <= 1) return er::sm_count();
  const int dev = er::current_device();
  const bool cacheable = dev >= 0 && dev < er::kMaxDevices;
  if (cacheable && cache[dev][c] != 0) return cache[dev][c];
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(c * 64));
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = 0;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)c;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  int n = 0;
  if (cudaOccupancyMaxActiveClusters(&n, spec_verify_kernel<__nv_bfloat16, true>, &cfg) != cudaSuccess) {
    (void)cudaGetLastError();
    n = 0;
  }
  n = n > 0 ? n * c : er::sm_count() / c * c;
  if (cacheable) cache[dev][c] = n;
  return n;
}

// CTAs per sequence: the power of two (at most 8, every CTA with at least one segment per warp) that needs the
// fewest waves of resident CTAs per unit of work; ties go to the smaller cluster (less to exchange).
int pick_cluster(int B, int nseg) {
  int best = 1;
  double best_cost = 0.0;
  for (int c = 1; c <= kMaxCluster; c *= 2) {
    if (c > 1 && nseg / c < kWarps) break;
    const int slots = resident_ctas(c);
    const long long ctas = (long long)B * c;
    const double waves = (double)((ctas + slots - 1) / slots);
    const double cost = waves / c + 0.004 * c;   // + the exchange, a little dearer for larger clusters
    if (c == 1 || cost < best_cost) { best = c; best_cost = cost; }
  }
  return best;
}

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
  const int nseg = (V + kSeg - 1) / kSeg;
  int cluster = pick_cluster(B, nseg);
  if (g_force_cluster > 0 && g_force_cluster <= nseg) cluster = g_force_cluster;
  const size_t smem = (size_t)((nseg + cluster - 1) / cluster) * sizeof(float);   // one sum per local segment
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
