// spec_verify.cu -- er_spec_verify: speculative-decoding verification by rejection sampling
// (sec. 2.2; L445 sec. D.1: accept drafted tokens, resample at the first rejection "from the
// adjusted target distribution", bonus token when everything is accepted; L544: needs the full
// distribution at the rejected position).
//
// One CTA of 1024 threads per sequence.  Rows of the vocabulary are streamed with 128-bit loads in tiles
// of 8192 elements (8 consecutive elements per thread).  The accept scan is lazy: position i's softmax
// normalisers are only computed if positions < i were all accepted, so a sequence rejected at position n
// reads 2 (n + 1) rows instead of 2 gamma + 1.  The residual draw is a two-level inverse CDF: per-warp
// segment sums (256 consecutive tokens) -> fp64 prefix over segments by one thread -> warp scan inside
// the one segment that contains the threshold.
#include "er_common.cuh"

namespace {

constexpr int kThreads = 1024;
constexpr int kWarps = kThreads / 32;
constexpr int kPerThread = 8;
constexpr int kTile = kThreads * kPerThread;  // 8192 tokens
constexpr int kMaxV = 1 << 20;
constexpr float kNegInf = -3.0e38f;

// ---- 8 consecutive elements starting at token v0 (clipped to V), widened to fp32 -------------
template <typename T>
struct Load8;
template <>
struct Load8<float> {
  static __device__ __forceinline__ void run(const float* row, int v0, int V, bool vec, float fill, float (&f)[8]) {
    if (vec && v0 + 8 <= V) {
      const float4 a = *reinterpret_cast<const float4*>(row + v0);
      const float4 b = *reinterpret_cast<const float4*>(row + v0 + 4);
      f[0] = a.x; f[1] = a.y; f[2] = a.z; f[3] = a.w;
      f[4] = b.x; f[5] = b.y; f[6] = b.z; f[7] = b.w;
    } else {
#pragma unroll
      for (int i = 0; i < 8; ++i) f[i] = (v0 + i < V) ? row[v0 + i] : fill;
    }
  }
  static __device__ __forceinline__ float one(const float* row, int v) { return row[v]; }
};
template <>
struct Load8<__nv_bfloat16> {
  static __device__ __forceinline__ void run(const __nv_bfloat16* row, int v0, int V, bool vec, float fill,
                                             float (&f)[8]) {
    if (vec && v0 + 8 <= V) {
      const uint4 a = *reinterpret_cast<const uint4*>(row + v0);
      const uint32_t r[4] = {a.x, a.y, a.z, a.w};
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        f[2 * i] = __uint_as_float(r[i] << 16);
        f[2 * i + 1] = __uint_as_float(r[i] & 0xFFFF0000u);
      }
    } else {
#pragma unroll
      for (int i = 0; i < 8; ++i) f[i] = (v0 + i < V) ? __bfloat162float(row[v0 + i]) : fill;
    }
  }
  static __device__ __forceinline__ float one(const __nv_bfloat16* row, int v) { return __bfloat162float(row[v]); }
};

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
  float red_a[kWarps];
  float red_b[kWarps];
  float bc[4];
  int seg;
  int token;
  int flag;
  double thr_local;
};

// Softmax normalisers of one target row and (optionally) one draft row in a single pass; online max/sum.
template <typename T>
__device__ void row_stats(const T* trow, const T* drow, int V, bool vec, float scale, Shared& sh, RowStats& st,
                          RowStats& sd) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  float mt = kNegInf, st_ = 0.f, md = kNegInf, sd_ = 0.f;
  for (int base = 0; base < V; base += kTile) {
    const int v0 = base + tid * kPerThread;
    if (v0 >= V) break;
    float f[8];
    Load8<T>::run(trow, v0, V, vec, kNegInf, f);
    float cm = f[0];
#pragma unroll
    for (int i = 1; i < 8; ++i) cm = fmaxf(cm, f[i]);
    if (cm > mt) { st_ *= exp2f((mt - cm) * scale); mt = cm; }
#pragma unroll
    for (int i = 0; i < 8; ++i) st_ += exp2f((f[i] - mt) * scale);
    if (drow) {
      Load8<T>::run(drow, v0, V, vec, kNegInf, f);
      cm = f[0];
#pragma unroll
      for (int i = 1; i < 8; ++i) cm = fmaxf(cm, f[i]);
      if (cm > md) { sd_ *= exp2f((md - cm) * scale); md = cm; }
#pragma unroll
      for (int i = 0; i < 8; ++i) sd_ += exp2f((f[i] - md) * scale);
    }
  }
  // block max
  float wm_t = warp_max(mt), wm_d = warp_max(md);
  if (lane == 0) { sh.red_a[warp] = wm_t; sh.red_b[warp] = wm_d; }
  __syncthreads();
  float bm_t = sh.red_a[lane], bm_d = sh.red_b[lane];
  bm_t = warp_max(bm_t); bm_d = warp_max(bm_d);
  __syncthreads();
  // block sum of rescaled partial sums
  st_ = (mt > kNegInf) ? st_ * exp2f((mt - bm_t) * scale) : 0.f;
  sd_ = (md > kNegInf) ? sd_ * exp2f((md - bm_d) * scale) : 0.f;
  float ws_t = warp_sum(st_), ws_d = warp_sum(sd_);
  if (lane == 0) { sh.red_a[warp] = ws_t; sh.red_b[warp] = ws_d; }
  __syncthreads();
  float bs_t = warp_sum(sh.red_a[lane]), bs_d = warp_sum(sh.red_b[lane]);
  __syncthreads();
  st.max = bm_t; st.inv_sum = __fdiv_rn(1.0f, bs_t);
  sd.max = bm_d; sd.inv_sum = drow ? __fdiv_rn(1.0f, bs_d) : 0.f;
}

// The 8 residual weights of one thread chunk.  use_q == false: w = p (bonus token / degenerate residual).
template <typename T, bool kLogits>
__device__ __forceinline__ void weights8(const T* trow, const T* drow, int v0, int V, bool vec, float scale,
                                         const RowStats& st, const RowStats& sd, bool use_q, float (&w)[8]) {
  float p[8];
  Load8<T>::run(trow, v0, V, vec, kLogits ? kNegInf : 0.f, p);
  if (kLogits) {
#pragma unroll
    for (int i = 0; i < 8; ++i) p[i] = exp2f((p[i] - st.max) * scale) * st.inv_sum;
  }
  if (use_q) {
    float q[8];
    Load8<T>::run(drow, v0, V, vec, kLogits ? kNegInf : 0.f, q);
    if (kLogits) {
#pragma unroll
      for (int i = 0; i < 8; ++i) q[i] = exp2f((q[i] - sd.max) * scale) * sd.inv_sum;
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) w[i] = fmaxf(0.f, p[i] - q[i]);
  } else {
#pragma unroll
    for (int i = 0; i < 8; ++i) w[i] = p[i];
  }
}

// Inverse-CDF draw over w in vocab order: token = min{v : C(v) > r R}.  Returns -1 if R == 0.
template <typename T, bool kLogits>
__device__ int draw_token(const T* trow, const T* drow, int V, bool vec, float scale, const RowStats& st,
                          const RowStats& sd, bool use_q, float r, Shared& sh, float* seg_sums) {
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int tiles = (V + kTile - 1) / kTile;
  // level 1: sums of 256-token segments (one warp, one tile each)
  for (int t = 0; t < tiles; ++t) {
    const int v0 = t * kTile + tid * kPerThread;
    float s = 0.f;
    if (v0 < V) {
      float w[8];
      weights8<T, kLogits>(trow, drow, v0, V, vec, scale, st, sd, use_q, w);
      s = ((w[0] + w[1]) + (w[2] + w[3])) + ((w[4] + w[5]) + (w[6] + w[7]));
    }
    s = warp_sum(s);
    if (lane == 0) seg_sums[t * kWarps + warp] = s;
  }
  __syncthreads();
  // level 2: fp64 prefix over segments in vocab order by one thread
  if (tid == 0) {
    const int nseg = tiles * kWarps;
    double R = 0.0;
    for (int i = 0; i < nseg; ++i) R += (double)seg_sums[i];
    int seg = -1;
    double excl = 0.0;
    if (R > 0.0) {
      const double thr = (double)r * R;
      double c = 0.0;
      seg = nseg - 1;
      for (int i = 0; i < nseg; ++i) {
        const double nc = c + (double)seg_sums[i];
        if (nc > thr) { seg = i; break; }
        c = nc;
      }
      // if rounding left no segment (cannot happen for r < 1), fall to the last segment with mass
      while (seg > 0 && !(seg_sums[seg] > 0.f)) --seg;
      excl = 0.0;
      for (int i = 0; i < seg; ++i) excl += (double)seg_sums[i];
      sh.thr_local = thr - excl;
    }
    sh.seg = seg;
    sh.token = -1;
  }
  __syncthreads();
  const int seg = sh.seg;
  if (seg < 0) return -1;
  // level 3: warp scan inside the chosen 256-token segment
  if (warp == 0) {
    const int v0 = (seg / kWarps) * kTile + (seg % kWarps) * 256 + lane * kPerThread;
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
__global__ void __launch_bounds__(kThreads, 1)
spec_verify_kernel(const T* __restrict__ target, const T* __restrict__ draft, float scale,
                   const int32_t* __restrict__ draft_tokens, const float* __restrict__ u_accept,
                   const float* __restrict__ u_sample, int gamma, int V, int32_t* __restrict__ accept_count,
                   int32_t* __restrict__ out_tokens) {
  extern __shared__ float seg_sums[];
  __shared__ Shared sh;
  const int b = blockIdx.x, tid = threadIdx.x;
  const bool vec = ((size_t)V * sizeof(T)) % 16 == 0;
  const T* tgt = target + (size_t)b * (gamma + 1) * V;
  const T* drf = draft + (size_t)b * gamma * V;
  const int32_t* xs = draft_tokens + (size_t)b * gamma;

  RowStats st{0.f, 1.f}, sd{0.f, 1.f};
  int n = 0;
  for (; n < gamma; ++n) {
    const T* trow = tgt + (size_t)n * V;
    const T* drow = drf + (size_t)n * V;
    if (kLogits) row_stats<T>(trow, drow, V, vec, scale, sh, st, sd);
    if (tid == 0) {
      int x = xs[n];
      x = min(max(x, 0), V - 1);
      float p = Load8<T>::one(trow, x), q = Load8<T>::one(drow, x);
      if (kLogits) {
        p = exp2f((p - st.max) * scale) * st.inv_sum;
        q = exp2f((q - sd.max) * scale) * sd.inv_sum;
      }
      const float lhs = __fmul_rn(u_accept[(size_t)b * gamma + n], q);
      sh.flag = (lhs < p) ? 1 : 0;
    }
    __syncthreads();
    const int acc = sh.flag;
    __syncthreads();
    if (!acc) break;
  }
  const T* trow = tgt + (size_t)n * V;
  const T* drow = (n < gamma) ? drf + (size_t)n * V : nullptr;
  if (n == gamma && kLogits) row_stats<T>(trow, nullptr, V, vec, scale, sh, st, sd);
  const float r = u_sample[b];
  int tok = draw_token<T, kLogits>(trow, drow, V, vec, scale, st, sd, n < gamma, r, sh, seg_sums);
  if (tok < 0) tok = draw_token<T, kLogits>(trow, nullptr, V, vec, scale, st, sd, false, r, sh, seg_sums);
  if (tok < 0) tok = V - 1;  // all-zero target row: outside the contract, stay memory-safe
  if (tid == 0) accept_count[b] = n;
  if (tid <= gamma) {
    int32_t o = -1;
    if (tid < n) o = xs[tid];
    else if (tid == n) o = tok;
    out_tokens[(size_t)b * (gamma + 1) + tid] = o;
  }
}

}  // namespace

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
  const size_t smem = (size_t)tiles * kWarps * sizeof(float);
  const float scale = (float)(1.4426950408889634 / (double)temperature);
  cudaStream_t s = (cudaStream_t)stream;
  if (in_dtype == ER_F32 && !inputs_are_logits) {
    spec_verify_kernel<float, false><<<B, kThreads, smem, s>>>((const float*)target, (const float*)draft, scale,
                                                               draft_tokens, u_accept, u_sample, gamma, V,
                                                               accept_count, out_tokens);
  } else if (in_dtype == ER_F32) {
    spec_verify_kernel<float, true><<<B, kThreads, smem, s>>>((const float*)target, (const float*)draft, scale,
                                                              draft_tokens, u_accept, u_sample, gamma, V,
                                                              accept_count, out_tokens);
  } else {
    spec_verify_kernel<__nv_bfloat16, true><<<B, kThreads, smem, s>>>(
        (const __nv_bfloat16*)target, (const __nv_bfloat16*)draft, scale, draft_tokens, u_accept, u_sample, gamma, V,
        accept_count, out_tokens);
  }
  ER_CUDA_TRY(cudaGetLastError());
  return ER_OK;
}
