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
// small: the maximum of a chunk of bf16 logits is taken on the packed words (max.bf16x2) and compared with one
// setp against a threshold (the softmax reference of a lane is raised lazily, see Acc), and the segments of
// consecutive rows are dealt to the warps in rotation so that no warp carries the ragged tail of every row.
// The residual draw is a multi-level inverse CDF: per-warp segment sums -> per-CTA totals, exchanged -> the
// CTA whose range holds the threshold does an fp64 blocked prefix over its segments (one warp) and a warp scan
// inside the one segment that contains the threshold.
//
// Two kernels share that decomposition: spec_verify_ring_kernel (logits whose rows are 16-byte multiples: every
// paper-shaped workload) streams the rows through a shared-memory ring filled by one producer lane with
// cp.async.bulk; spec_verify_kernel reads them with ld.global batches into registers (probability inputs, rows
// that are not 16-byte multiples).
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
constexpr float kNegInf = -3.0e38f;         // "no finite logit seen yet": the initial reference of the statistics
// Logit positions beyond V are filled with a true -inf (probability 0), never with a finite sentinel: a finite fill would
// become the reference of a lane whose real logits are all masked (-inf) and overflow -m * scale
#define ER_LOGIT_FILL (__uint_as_float(0xFF800000u))

// ---- 8 consecutive elements starting at token v0 (clipped to V): raw load, then widening to fp32 ----
// (split in two so that the loads of several segments can be in flight before the first one is consumed)
template <typename T>
struct Load8;
template <>
struct Load8<float> {
  struct Raw { float4 a, b; };
  static constexpr int kBatch = 2;   // segments whose loads are issued together (register path)
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
      const uint32_t fb = __float_as_uint(fill) >> 16;   // the fills used (0, -inf) are exact in bf16
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

// A row's softmax as one fma and one ex2 per logit: p(v) = 2^(l_v * scale + bias), bias = -m * scale - log2(sum_v
// 2^((l_v - m) * scale)) for the row's reference m.  (Probability inputs do not use it.)
struct RowStats {
  float bias;
};
__device__ __forceinline__ RowStats row_stats_of(float m, float inv_sum, float scale) {
  return RowStats{fmaf(-m, scale, log2f(inv_sum))};
}

constexpr int kMaxRows = 33;         // gamma <= 16: rows t_0, d_0, t_1, d_1, ..., t_gamma
constexpr int kMaxDepth = 12;        // stages of the shared-memory ring (ring kernel)

struct Shared {
  double xmass[2][kMaxCluster];      // [parity][rank]: residual mass of every CTA's range
  float2 wstat[kMaxRows][32];        // [row][warp]: per-warp (max, sum) of this CTA's range of the row
  float2 xall[kMaxCluster][kMaxRows];  // [rank][row]: per-CTA statistics of every CTA of the cluster
  float4 stat[17];                   // [position]: (max_t, 1/sum_t, max_d, 1/sum_d) over the whole vocabulary
  float px[16], qx[16], ua[16];      // target / draft value at the drafted token and the uniform, per position
  uint64_t full[kMaxDepth], empty[kMaxDepth];   // ring kernel: stage landed / stage consumed
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

// Online softmax statistics of one lane: a REFERENCE logit m (the maximum of some chunk seen so far), four partial
// sums s[] of 2^((l - m) * scale) and nm = -m * scale.  The reference is raised lazily (the trick of recent
// attention kernels): only when a chunk holds a logit above thr = m + kMargin / scale, i.e. when a term would
// exceed 2^kMargin -- with fp32 sums of at most 2^20 terms that is far from overflow, and the result is the same
// (reference, sum) pair algebra as an exact running maximum.  After the first chunk of a row the raise is
// practically never taken, so the loop is: maximum of the chunk on the packed words, one compare, then
// unpack / fma / ex2 / add per logit.
constexpr float kMargin = 32.f;

struct Acc {
  float m, nm, s[4];
  float thr;          // float rows: raise when a logit exceeds this
  uint32_t thr2;      // bf16 rows: the same as packed bf16x2 (rounded down)
  __device__ __forceinline__ void init() {
    m = kNegInf; nm = 0.f; thr = __uint_as_float(0xFF800000u); thr2 = 0xFF80FF80u;   // -inf: the first finite chunk raises
#pragma unroll
    for (int i = 0; i < 4; ++i) s[i] = 0.f;
  }
  __device__ __forceinline__ float sum() const { return (s[0] + s[1]) + (s[2] + s[3]); }
  // cm = the maximum of the chunk that tripped the threshold: it becomes the reference
  __device__ __forceinline__ void raise(float cm, float scale) {
    const float f = ex2_fast((m - cm) * scale);     // m = -3e38 at first: f = 0 and the sums are 0 anyway
#pragma unroll
    for (int i = 0; i < 4; ++i) s[i] *= f;
    m = cm;
    nm = -cm * scale;
    thr = cm + kMargin / scale;
    uint32_t b = __float_as_uint(thr);              // bf16 not above thr: truncation rounds a negative value up,
    uint32_t h = b >> 16;                           // so step one further down there
    if ((b & 0x80000000u) && (b & 0xFFFFu)) h += 1;
    if ((b & 0x7F800000u) == 0x7F800000u) h = 0x7F7Fu;   // thr overflowed (tiny scale): largest finite bf16
    thr2 = h | (h << 16);
  }
};

__device__ __forceinline__ uint32_t max_bf16x2(uint32_t a, uint32_t b) {
  uint32_t d;
  asm("max.bf16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b));
  return d;
}
// true if either half of a exceeds the same half of b
__device__ __forceinline__ bool any_gt_bf16x2(uint32_t a, uint32_t b) {
  uint32_t r;
  asm("{\n\t.reg .pred p, q;\n\t"
      "setp.gt.bf16x2 p|q, %1, %2;\n\t"
      "or.pred p, p, q;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t}\n"
      : "=r"(r)
      : "r"(a), "r"(b));
  return r != 0;
}

// N chunks of 8 logits of one row -> the lane's statistics.  A chunk that does not exist is passed as all -inf:
// it never trips the threshold, and its terms are 2^(-inf) = 0 (nm is finite, so no inf - inf).
template <typename T>
struct Accum;
template <>
struct Accum<float> {
  static __device__ __forceinline__ Load8<float>::Raw neg_inf() {
    const float x = __uint_as_float(0xFF800000u);
    Load8<float>::Raw r;
    r.a = make_float4(x, x, x, x);
    r.b = r.a;
    return r;
  }
  template <int N>
  static __device__ __forceinline__ void add(const Load8<float>::Raw (&r)[N], Acc& a, float scale) {
    float cm = __uint_as_float(0xFF800000u);
#pragma unroll
    for (int j = 0; j < N; ++j)
      cm = fmaxf(cm, fmaxf(fmaxf(fmaxf(r[j].a.x, r[j].a.y), fmaxf(r[j].a.z, r[j].a.w)),
                           fmaxf(fmaxf(r[j].b.x, r[j].b.y), fmaxf(r[j].b.z, r[j].b.w))));
    if (cm > a.thr) a.raise(cm, scale);
#pragma unroll
    for (int j = 0; j < N; ++j) {
      a.s[0] += ex2_fast(fmaf(r[j].a.x, scale, a.nm)) + ex2_fast(fmaf(r[j].b.x, scale, a.nm));
      a.s[1] += ex2_fast(fmaf(r[j].a.y, scale, a.nm)) + ex2_fast(fmaf(r[j].b.y, scale, a.nm));
      a.s[2] += ex2_fast(fmaf(r[j].a.z, scale, a.nm)) + ex2_fast(fmaf(r[j].b.z, scale, a.nm));
      a.s[3] += ex2_fast(fmaf(r[j].a.w, scale, a.nm)) + ex2_fast(fmaf(r[j].b.w, scale, a.nm));
    }
  }
};
template <>
struct Accum<__nv_bfloat16> {
  static __device__ __forceinline__ Load8<__nv_bfloat16>::Raw neg_inf() {
    Load8<__nv_bfloat16>::Raw r;
    r.a = make_uint4(0xFF80FF80u, 0xFF80FF80u, 0xFF80FF80u, 0xFF80FF80u);
    return r;
  }
  template <int N>
  static __device__ __forceinline__ void add(const Load8<__nv_bfloat16>::Raw (&r)[N], Acc& a, float scale) {
    uint32_t n2 = max_bf16x2(max_bf16x2(r[0].a.x, r[0].a.y), max_bf16x2(r[0].a.z, r[0].a.w));
#pragma unroll
    for (int j = 1; j < N; ++j)
      n2 = max_bf16x2(n2, max_bf16x2(max_bf16x2(r[j].a.x, r[j].a.y), max_bf16x2(r[j].a.z, r[j].a.w)));
    if (any_gt_bf16x2(n2, a.thr2))
      a.raise(fmaxf(__uint_as_float(n2 << 16), __uint_as_float(n2 & 0xFFFF0000u)), scale);
#pragma unroll
    for (int j = 0; j < N; ++j) {
      a.s[0] += ex2_fast(fmaf(__uint_as_float(r[j].a.x << 16), scale, a.nm));
      a.s[1] += ex2_fast(fmaf(__uint_as_float(r[j].a.x & 0xFFFF0000u), scale, a.nm));
      a.s[2] += ex2_fast(fmaf(__uint_as_float(r[j].a.y << 16), scale, a.nm));
      a.s[3] += ex2_fast(fmaf(__uint_as_float(r[j].a.y & 0xFFFF0000u), scale, a.nm));
      a.s[0] += ex2_fast(fmaf(__uint_as_float(r[j].a.z << 16), scale, a.nm));
      a.s[1] += ex2_fast(fmaf(__uint_as_float(r[j].a.z & 0xFFFF0000u), scale, a.nm));
      a.s[2] += ex2_fast(fmaf(__uint_as_float(r[j].a.w << 16), scale, a.nm));
      a.s[3] += ex2_fast(fmaf(__uint_as_float(r[j].a.w & 0xFFFF0000u), scale, a.nm));
    }
  }
};

// The lanes' statistics of one row -> one (reference, sum) of the warp (no CTA barrier per row): the largest
// reference, then the sum of the rescaled sums.
__device__ __forceinline__ void warp_row_stat(const Acc& a, float scale, float2& out) {
  const float wm = warp_max(a.m);
  const float ws = warp_sum((a.m > kNegInf) ? a.sum() * ex2_fast((a.m - wm) * scale) : 0.f);
  if ((threadIdx.x & 31) == 0) out = make_float2(wm, ws);
}

// Softmax statistics of one target row and (optionally) one draft row over this CTA's segment range, reduced to
// one entry per warp in sh.wstat[2 pos] and sh.wstat[2 pos + 1].  Warp w takes the local segments (w - rot) mod kWarps, + kWarps, ...;
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
      rt[j] = Accum<T>::neg_inf();
      rd[j] = rt[j];
      if (s0 + j * kWarps < nloc && v0 < V) {
        rt[j] = Load8<T>::load(trow, v0, V, vec, ER_LOGIT_FILL);
        if (drow) rd[j] = Load8<T>::load(drow, v0, V, vec, ER_LOGIT_FILL);
      }
    }
    Accum<T>::add(rt, at, scale);
    if (drow) Accum<T>::add(rd, ad, scale);
  }
  warp_row_stat(at, scale, sh.wstat[2 * pos][warp]);
  if (drow) warp_row_stat(ad, scale, sh.wstat[2 * pos + 1][warp]);
}

// (max, sum) pairs a and b of two disjoint parts of a row -> the pair of their union
__device__ __forceinline__ void merge_stat(float& m, float& s, float m2, float s2, float scale) {
  const float mm = fmaxf(m, m2);
  const float a = (m > kNegInf) ? s * exp2f((m - mm) * scale) : 0.f;
  const float b = (m2 > kNegInf) ? s2 * exp2f((m2 - mm) * scale) : 0.f;
  m = mm;
  s = a + b;
}

// After the statistics of rows 0 .. 2 gamma: combine the nw warps that wrote a row (one warp per row, a fixed
// shuffle tree), exchange over the cluster through distributed shared memory, combine ranks (in order).  Every
// CTA ends with the same sh.stat[].
__device__ void combine_stats(int gamma, int nw, float scale, Shared& sh, ClusterCtx& cx) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nrows = 2 * gamma + 1, warps = (int)(blockDim.x >> 5);
  cg::cluster_group cluster = cg::this_cluster();
  cluster_started(cx);
  __syncthreads();
  for (int r = warp; r < nrows; r += warps) {
    const float2 v = (lane < nw) ? sh.wstat[r][lane] : make_float2(kNegInf, 0.f);
    const float m = warp_max(v.x);
    const float sm = warp_sum(v.x > kNegInf ? v.y * exp2f((v.x - m) * scale) : 0.f);
    if (lane < cx.size) *cluster.map_shared_rank(&sh.xall[cx.rank][r], lane) = make_float2(m, sm);
  }
  cluster.sync();
  if (tid <= gamma) {
    float mt = kNegInf, st = 0.f, md = kNegInf, sd = 0.f;
    for (int c = 0; c < cx.size; ++c) {
      const float2 v = sh.xall[c][2 * tid];
      merge_stat(mt, st, v.x, v.y, scale);
      if (tid < gamma) {
        const float2 u = sh.xall[c][2 * tid + 1];
        merge_stat(md, sd, u.x, u.y, scale);
      }
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
    for (int i = 0; i < 8; ++i) p[i] = ex2_fast(fmaf(p[i], scale, st.bias));
  }
  if (use_q) {
    float q[8];
    Load8<T>::expand(rq, q);
    if (kLogits) {
#pragma unroll
      for (int i = 0; i < 8; ++i) q[i] = ex2_fast(fmaf(q[i], scale, sd.bias));
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
  const float fill = kLogits ? ER_LOGIT_FILL : 0.f;
  typename Load8<T>::Raw rp = Load8<T>::load(trow, v0, V, vec, fill), rq = rp;
  if (use_q) rq = Load8<T>::load(drow, v0, V, vec, fill);
  weights8_raw<T, kLogits>(rp, rq, scale, st, sd, use_q, w);
}

// Inverse-CDF draw over w in vocab order, level 1: the sums of this CTA's 256-token segments, one warp each.
template <typename T, bool kLogits>
__device__ void draw_segment_sums(const T* trow, const T* drow, int V, bool vec, float scale, const RowStats& st,
                                  const RowStats& sd, bool use_q, const ClusterCtx& cx, float* seg_sums) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nloc = cx.seg_hi - cx.seg_lo;
  constexpr int NB = Load8<T>::kBatch;
  const float fill = kLogits ? ER_LOGIT_FILL : 0.f;
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
}

// Levels 2 and 3 of the draw, once seg_sums holds this CTA's segment sums: token = min{v : C(v) > r R}.  Returns -1
// in every CTA of the cluster if R == 0; otherwise the token in the CTA whose segment range holds the threshold
// and -2 in the others.
template <typename T, bool kLogits>
__device__ int draw_finish(const T* trow, const T* drow, int V, bool vec, float scale, const RowStats& st,
                           const RowStats& sd, bool use_q, float r, Shared& sh, ClusterCtx& cx,
                           const float* seg_sums) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nloc = cx.seg_hi - cx.seg_lo;
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

// The accept tests: n = number of drafted tokens accepted before the first rejection, decided by
// one thread from sh.px / qx / ua (and sh.stat for logits); every CTA of the cluster takes the same decisions from
// the same numbers.  u q < p is evaluated in fp32 (V3).
template <bool kLogits>
__device__ int accept_prefix(int gamma, float scale, Shared& sh) {
  if (threadIdx.x == 0) {
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
  return sh.flag;
}

// accept_count[b] and out_tokens[b][0 .. gamma], by the CTA that owns the draw (tok >= 0).
__device__ void write_outputs(int tok, int n, int b, int gamma, int V, const int32_t* xs, const ClusterCtx& cx,
                              int32_t* accept_count, int32_t* out_tokens) {
  if (tok == -1) tok = (cx.rank == 0) ? V - 1 : -2;  // all-zero target row: outside the contract, stay memory-safe
  if (tok == -2) return;                             // another CTA of the cluster owns the draw and the outputs
  const int tid = threadIdx.x;
  if (tid == 0) accept_count[b] = n;
  if (tid <= gamma) {
    int32_t o = -1;
    if (tid < n) o = xs[tid];
    else if (tid == n) o = tok;
    out_tokens[(size_t)b * (gamma + 1) + tid] = o;
  }
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
    combine_stats(gamma, kWarps, scale, sh, cx);
  }
  const int n = accept_prefix<kLogits>(gamma, scale, sh);
  RowStats st{0.f}, sd{0.f};
  if (kLogits) {
    const float4 v = sh.stat[n];
    st = row_stats_of(v.x, v.y, scale);
    if (n < gamma) sd = row_stats_of(v.z, v.w, scale);
  }
  const T* trow = tgt + (size_t)n * V;
  const T* drow = (n < gamma) ? drf + (size_t)n * V : nullptr;
  const float r = u_sample[b];
  draw_segment_sums<T, kLogits>(trow, drow, V, vec, scale, st, sd, n < gamma, cx, seg_sums);
  int tok = draw_finish<T, kLogits>(trow, drow, V, vec, scale, st, sd, n < gamma, r, sh, cx, seg_sums);
  if (tok == -1) {   // no residual mass: draw from the target row itself
    draw_segment_sums<T, kLogits>(trow, nullptr, V, vec, scale, st, sd, false, cx, seg_sums);
    tok = draw_finish<T, kLogits>(trow, nullptr, V, vec, scale, st, sd, false, r, sh, cx, seg_sums);
  }
  write_outputs(tok, n, b, gamma, V, xs, cx, accept_count, out_tokens);
}

// ---------------------------------------------------------------------------------------------------------------
// Ring kernel (logits whose rows are 16-byte multiples: every paper-shaped workload).  The loads of the sweep are
// taken off the compute warps: one producer lane streams the CTA's slice of row after row through a 192 KB ring
// of shared-memory stages with cp.async.bulk (a stage = 32 consecutive segments of one row), kCons consumer warps
// take two segments of every stage each.  The ring never drains at a row boundary, so the special-function unit
// and HBM overlap instead of taking turns (the register path above waits for a DRAM round trip per batch of
// loads).  The draw pass goes through the same ring, a stage = 16 segments of the target row + the same 16 of the
// draft row.
constexpr int kCons = 31;                       // consumer warps
constexpr int kRingThreads = (kCons + 1) * 32;  // + the producer warp
constexpr int kSPW = 2;                         // segments per consumer warp and sweep stage
constexpr int kStageSegs = kCons * kSPW;
constexpr int kRingBytes = 192 * 1024;

template <typename T>
struct Ring {
  static constexpr int kSegBytes = kSeg * (int)sizeof(T);
  static constexpr int kStageBytes = kStageSegs * kSegBytes;
  static constexpr int kDepth = kRingBytes / kStageBytes;
  static_assert(kDepth >= 2 && kDepth <= kMaxDepth, "ring depth");
  static_assert(kStageBytes % 32 == 0, "the two halves of a draw stage are 16-byte aligned");
};

// Position in the ring, stepped identically by the producer lane and by every consumer warp: slot and the parity
// of the slot's current use.  A consumer waits on full[slot] with `phase`; the producer waits on empty[slot] with
// phase ^ 1 (on a fresh barrier that is the already-completed "previous" phase, so the first round passes).
template <int kDepth>
struct Pipe {
  uint32_t slot = 0, phase = 0;
  __device__ __forceinline__ void step() {
    if (++slot == kDepth) { slot = 0; phase ^= 1; }
  }
};

__device__ __forceinline__ void bulk_load_plain(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   er::smem_u32(smem_dst)),
               "l"(gsrc), "r"(bytes), "r"(er::smem_u32(bar))
               : "memory");
}

// the lanes of a float row's last chunk that lie beyond V were not copied: give them the fill value
__device__ __forceinline__ void clip_tail(Load8<float>::Raw& r, int v0, int V, float fill) {
  if (v0 + 8 > V) {
    float* f = reinterpret_cast<float*>(&r);
#pragma unroll
    for (int i = 0; i < 8; ++i)
      if (v0 + i >= V) f[i] = fill;
  }
}
__device__ __forceinline__ void clip_tail(Load8<__nv_bfloat16>::Raw&, int, int, float) {}   // V % 8 == 0 here

// Producer lane: the bytes [seg_lo kSeg, min(seg_hi kSeg, V)) of row_a -- and, if row_b is given, the same bytes of
// row_b -- in stages of `segs` segments into consecutive ring slots: row_a into the first half of a slot
// (or all of it), row_b into the second half.  A slot is refilled once every consumer warp has released it.
template <typename T>
__device__ __forceinline__ void produce_rows(unsigned char* ring, Shared& sh, Pipe<Ring<T>::kDepth>& pp,
                                             const T* row_a, const T* row_b, int V, const ClusterCtx& cx, int segs) {
  using R = Ring<T>;
  const long long lo = (long long)cx.seg_lo * kSeg;
  const long long hi = min((long long)cx.seg_hi * kSeg, (long long)V);
  const long long total = (hi - lo) * (long long)sizeof(T);
  const long long step = (long long)segs * R::kSegBytes;
  const unsigned char* src_a = reinterpret_cast<const unsigned char*>(row_a + lo);
  const unsigned char* src_b = reinterpret_cast<const unsigned char*>(row_b + lo);
  for (long long off = 0; off < total; off += step, pp.step()) {
    er::mbar_wait(&sh.empty[pp.slot], pp.phase ^ 1);
    const uint32_t bytes = (uint32_t)min(step, total - off);
    unsigned char* dst = ring + (size_t)pp.slot * R::kStageBytes;
    er::mbar_arrive_expect_tx(&sh.full[pp.slot], row_b ? 2 * bytes : bytes);
    bulk_load_plain(dst, src_a + off, bytes, &sh.full[pp.slot]);
    if (row_b) bulk_load_plain(dst + R::kStageBytes / 2, src_b + off, bytes, &sh.full[pp.slot]);
  }
}

// Consumer warps: online statistics of one row from the ring; sh.wstat[row][warp].  The segments of a stage are
// dealt to the warps in a rotation that advances with the row by the size of the ragged last stage.
template <typename T>
__device__ __forceinline__ void consume_row_stats(const unsigned char* ring, Shared& sh, Pipe<Ring<T>::kDepth>& pp,
                                                  int row, int V, float scale, const ClusterCtx& cx) {
  using R = Ring<T>;
  using Raw = typename Load8<T>::Raw;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nloc = cx.seg_hi - cx.seg_lo;
  const int nst = (nloc + kStageSegs - 1) / kStageSegs;
  // stages in which every segment exists and lies wholly below V: no validity tests there
  const int nfull = (int)min((long long)nloc, (long long)V / kSeg - cx.seg_lo) / kStageSegs;
  const int rot = (row * (nloc % kStageSegs)) % kStageSegs;
  int jj[kSPW];
  uint32_t off[kSPW];
#pragma unroll
  for (int j = 0; j < kSPW; ++j) {
    jj[j] = warp * kSPW + j + rot;
    if (jj[j] >= kStageSegs) jj[j] -= kStageSegs;
    off[j] = (uint32_t)(jj[j] * R::kSegBytes + lane * kPerThread * (int)sizeof(T));
  }
  Acc a;
  a.init();
  for (int k = 0; k < nst; ++k, pp.step()) {
    er::mbar_wait(&sh.full[pp.slot], pp.phase);
    const unsigned char* stage = ring + (size_t)pp.slot * R::kStageBytes;
    Raw r[kSPW];
    if (k < nfull) {
#pragma unroll
      for (int j = 0; j < kSPW; ++j) r[j] = *reinterpret_cast<const Raw*>(stage + off[j]);
    } else {
#pragma unroll
      for (int j = 0; j < kSPW; ++j) {
        const int sg = k * kStageSegs + jj[j];
        const int v0 = (cx.seg_lo + sg) * kSeg + lane * kPerThread;
        r[j] = Accum<T>::neg_inf();
        if (sg < nloc && v0 < V) {
          r[j] = *reinterpret_cast<const Raw*>(stage + off[j]);
          clip_tail(r[j], v0, V, ER_LOGIT_FILL);
        }
      }
    }
    Accum<T>::add(r, a, scale);
    __syncwarp();
    if (lane == 0) er::mbar_arrive(&sh.empty[pp.slot]);
  }
  warp_row_stat(a, scale, sh.wstat[row][warp]);
}

// Consumer warps: level 1 of the draw from the ring (stage = 16 segments of the target row in the first half of a
// slot and, if use_q, the same 16 of the draft row in the second half).
template <typename T>
__device__ __forceinline__ void consume_segment_sums(const unsigned char* ring, Shared& sh,
                                                     Pipe<Ring<T>::kDepth>& pp, int V, float scale, const RowStats& st, const RowStats& sd, bool use_q,
                                                     const ClusterCtx& cx, float* seg_sums) {
  using R = Ring<T>;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nloc = cx.seg_hi - cx.seg_lo;
  const int nst = (nloc + kCons - 1) / kCons;
  for (int k = 0; k < nst; ++k, pp.step()) {
    er::mbar_wait(&sh.full[pp.slot], pp.phase);
    const unsigned char* stage = ring + (size_t)pp.slot * R::kStageBytes;
    const int sg = k * kCons + warp;
    if (sg < nloc) {
      const int v0 = (cx.seg_lo + sg) * kSeg + lane * kPerThread;
      float s = 0.f;
      if (v0 < V) {
        const size_t o = (size_t)warp * R::kSegBytes + (size_t)lane * kPerThread * sizeof(T);
        typename Load8<T>::Raw rp = *reinterpret_cast<const typename Load8<T>::Raw*>(stage + o), rq = rp;
        clip_tail(rp, v0, V, ER_LOGIT_FILL);
        if (use_q) {
          rq = *reinterpret_cast<const typename Load8<T>::Raw*>(stage + R::kStageBytes / 2 + o);
          clip_tail(rq, v0, V, ER_LOGIT_FILL);
        }
        float w[8];
        weights8_raw<T, true>(rp, rq, scale, st, sd, use_q, w);
        s = ((w[0] + w[1]) + (w[2] + w[3])) + ((w[4] + w[5]) + (w[6] + w[7]));
      }
      s = warp_sum(s);
      if (lane == 0) seg_sums[sg] = s;
    }
    __syncwarp();
    if (lane == 0) er::mbar_arrive(&sh.empty[pp.slot]);
  }
}

template <typename T>
__global__ void __launch_bounds__(kRingThreads, 1)
spec_verify_ring_kernel(const T* __restrict__ target, const T* __restrict__ draft, float scale,
                        const int32_t* __restrict__ draft_tokens, const float* __restrict__ u_accept,
                        const float* __restrict__ u_sample, int gamma, int V, int32_t* __restrict__ accept_count,
                        int32_t* __restrict__ out_tokens) {
  using R = Ring<T>;
  extern __shared__ __align__(128) unsigned char dyn[];
  unsigned char* ring = dyn;
  float* seg_sums = reinterpret_cast<float*>(dyn + kRingBytes);
  __shared__ Shared sh;
  cg::cluster_group cluster = cg::this_cluster();
  ClusterCtx cx;
  cx.size = (int)cluster.num_blocks();
  cx.rank = (int)cluster.block_rank();
  cx.xpar = 0;
  cx.started = false;
  if (cx.size > 1) asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory");   // "I have started"
  const int nseg = (V + kSeg - 1) / kSeg;
  cx.seg_lo = (int)(((long long)nseg * cx.rank) / cx.size);
  cx.seg_hi = (int)(((long long)nseg * (cx.rank + 1)) / cx.size);
  const int b = blockIdx.x / cx.size, tid = threadIdx.x, warp = tid >> 5;
  const T* tgt = target + (size_t)b * (gamma + 1) * V;
  const T* drf = draft + (size_t)b * gamma * V;
  const int32_t* xs = draft_tokens + (size_t)b * gamma;
  if (tid == 0) {
    for (int i = 0; i < R::kDepth; ++i) {
      er::mbar_init(&sh.full[i], 1);
      er::mbar_init(&sh.empty[i], kCons);
    }
    er::mbar_fence_init();
  }
  __syncthreads();

  // ---- the sweep: rows t_0, d_0, t_1, d_1, ..., t_gamma ----
  const int nrows = 2 * gamma + 1;
  Pipe<R::kDepth> pp;     // the producer lane's, or this consumer warp's
  if (warp == kCons) {
    const int lane = tid & 31;
    if (lane == 0) {
      for (int row = 0; row < nrows; ++row)
        produce_rows<T>(ring, sh, pp, (row & 1) ? drf + (size_t)(row >> 1) * V : tgt + (size_t)(row >> 1) * V,
                        (const T*)nullptr, V, cx, kStageSegs);
    } else if (lane <= gamma) {   // everything the accept tests read, fetched by the producer warp's idle lanes (a
      const int k = lane - 1;     // consumer warp waiting for these two round trips would hold back the whole ring)
      const int x = min(max(xs[k], 0), V - 1);
      sh.px[k] = Load8<T>::one(tgt + (size_t)k * V, x);
      sh.qx[k] = Load8<T>::one(drf + (size_t)k * V, x);
      sh.ua[k] = u_accept[(size_t)b * gamma + k];
    }
  } else {
    for (int row = 0; row < nrows; ++row) consume_row_stats<T>(ring, sh, pp, row, V, scale, cx);
  }
  combine_stats(gamma, kCons, scale, sh, cx);
  const int n = accept_prefix<true>(gamma, scale, sh);
  const float4 v = sh.stat[n];
  const RowStats st = row_stats_of(v.x, v.y, scale), sd = (n < gamma) ? row_stats_of(v.z, v.w, scale) : RowStats{0.f};
  const T* trow = tgt + (size_t)n * V;
  const T* drow = (n < gamma) ? drf + (size_t)n * V : nullptr;
  const float r = u_sample[b];
  const bool vec = true;
  int tok = -1;
  for (int pass = 0; pass < 2 && tok == -1; ++pass) {   // pass 1 only if there is no residual mass: p itself
    const bool use_q = (pass == 0) && n < gamma;
    if (pass == 1 && n == gamma) break;
    if (warp == kCons) {
      if ((tid & 31) == 0) produce_rows<T>(ring, sh, pp, trow, use_q ? drow : (const T*)nullptr, V, cx, kCons);
    } else {
      consume_segment_sums<T>(ring, sh, pp, V, scale, st, sd, use_q, cx, seg_sums);
    }
    __syncthreads();
    tok = draw_finish<T, true>(trow, use_q ? drow : nullptr, V, vec, scale, st, sd, use_q, r, sh, cx, seg_sums);
  }
  write_outputs(tok, n, b, gamma, V, xs, cx, accept_count, out_tokens);
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

template <typename T>
int launch_verify_ring(int cluster_size, size_t seg_bytes, cudaStream_t s, const T* target, const T* draft,
                       float scale, const int32_t* draft_tokens, const float* u_accept, const float* u_sample, int B,
                       int gamma, int V, int32_t* accept_count, int32_t* out_tokens) {
  static bool attr_set[er::kMaxDevices];   // the opt-in to > 48 KB of dynamic shared memory is per device
  const int dev = er::current_device();
  const size_t smem = (size_t)kRingBytes + seg_bytes;
  if (dev < 0 || dev >= er::kMaxDevices || !attr_set[dev]) {
    ER_CUDA_TRY(cudaFuncSetAttribute(spec_verify_ring_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     kRingBytes + (kMaxV / kSeg) * (int)sizeof(float)));
    if (dev >= 0 && dev < er::kMaxDevices) attr_set[dev] = true;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(B * cluster_size));
  cfg.blockDim = dim3(kRingThreads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)cluster_size;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  ER_CUDA_TRY(cudaLaunchKernelEx(&cfg, spec_verify_ring_kernel<T>, target, draft, scale, draft_tokens, u_accept,
                                 u_sample, gamma, V, accept_count, out_tokens));
  return ER_OK;
}

#ifdef ER_DEV
int g_force_cluster = 0;          // development library only (er_dev.h): 0 = automatic
int g_force_register_path = 0;    // 1 = never the ring kernel
#else
constexpr int g_force_cluster = 0;
constexpr int g_force_register_path = 0;
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
  if (cluster >= 16 && cluster <= 17) {   // 16 / 17: shared-memory ring kernel allowed / never used
    g_force_register_path = cluster - 16;
    return ER_OK;
  }
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
  const size_t elem = in_dtype == ER_BF16 ? 2 : 4;
  const bool ring = inputs_are_logits && ((size_t)V * elem) % 16 == 0 && !g_force_register_path;
  int rc;
  if (ring && in_dtype == ER_BF16) {
    rc = launch_verify_ring<__nv_bfloat16>(cluster, smem, s, (const __nv_bfloat16*)target, (const __nv_bfloat16*)draft,
                                           scale, draft_tokens, u_accept, u_sample, B, gamma, V, accept_count,
                                           out_tokens);
  } else if (ring) {
    rc = launch_verify_ring<float>(cluster, smem, s, (const float*)target, (const float*)draft, scale, draft_tokens,
                                   u_accept, u_sample, B, gamma, V, accept_count, out_tokens);
  } else if (in_dtype == ER_F32 && !inputs_are_logits) {
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
