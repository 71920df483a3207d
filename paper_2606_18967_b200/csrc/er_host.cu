// er_host.cu -- the *_host entry points of include/er.h: the same three operations for callers whose
// per-call operands live in HOST memory (the end-to-end leg of bench.py).  Each call stages its streaming
// operands into a caller-owned device arena with cudaMemcpyAsync, runs the device entry point on the same
// stream, and copies the result back -- all enqueued on `stream`, no synchronisation.  Operands that stay
// resident between calls (the drafter's packed weights and scales) remain device pointers.
#include "er_common.cuh"

namespace {

inline size_t up256(size_t x) { return (x + 255) & ~size_t(255); }

struct Arena {
  uint8_t* base;
  size_t size, used;
  void* take(size_t bytes) {
    void* p = base + used;
    used += up256(bytes);
    return p;
  }
};

}  // namespace

extern "C" {

size_t er_quantize_host_arena_bytes(int64_t N, int64_t K) {
  if (er_packed_bytes(N, K) == 0) return 0;
  return ER_GEMM_COUNTER_BYTES + up256((size_t)N * (size_t)K * 2);
}

size_t er_gemm_host_arena_bytes(int64_t M, int64_t N, int64_t K) {
  const size_t ws = er_gemm_workspace_bytes(M, N, K);
  if (ws == 0) return 0;
  return up256((size_t)M * K * 2) + up256((size_t)M * N * 4) + up256(ws);
}

size_t er_verify_host_arena_bytes(int32_t B, int32_t gamma, int32_t V, int in_dtype) {
  if (B < 0 || gamma < 1 || gamma > 16 || V < 1) return 0;
  const size_t es = (in_dtype == ER_F32) ? 4 : 2;
  return ER_GEMM_COUNTER_BYTES + up256((size_t)B * (gamma + 1) * V * es) + up256((size_t)B * gamma * V * es) +
         3 * up256((size_t)B * gamma * 4) + 2 * up256((size_t)B * 4) + up256((size_t)B * (gamma + 1) * 4);
}

int er_quantize_pack_host(const void* w_host, int64_t N, int64_t K, int group, void* qweight_out, void* scales_out,
                          void* arena, size_t arena_bytes, void* stream) {
  if (!w_host || !arena) return ER_ERR_NULL;
  const size_t need = er_quantize_host_arena_bytes(N, K);
  if (need == 0) return ER_ERR_SHAPE;
  if (arena_bytes < need) return ER_ERR_WORKSPACE;
  if (!er::aligned16(arena)) return ER_ERR_ALIGN;
  if (!qweight_out || !scales_out) return ER_ERR_NULL;
  int st = er::check_arch();
  if (st != ER_OK) return st;
  cudaStream_t s = (cudaStream_t)stream;
  // the first ER_GEMM_COUNTER_BYTES of any arena belong to the GEMM's tile counters: never staged over
  void* wd = reinterpret_cast<uint8_t*>(arena) + ER_GEMM_COUNTER_BYTES;
  ER_CUDA_TRY(cudaMemcpyAsync(wd, w_host, (size_t)N * K * 2, cudaMemcpyHostToDevice, s));
  return er_quantize_pack(wd, N, K, K, group, qweight_out, scales_out, stream);
}

int er_w4a16_gemm_host(const void* x_host, int64_t M, int64_t K, const void* qweight, const void* scales, int64_t N,
                       int group, void* y_host, int y_dtype, void* arena, size_t arena_bytes, void* stream) {
  if (!x_host || !y_host || !arena) return ER_ERR_NULL;
  if (y_dtype != ER_BF16 && y_dtype != ER_F32) return ER_ERR_DTYPE;
  const size_t need = er_gemm_host_arena_bytes(M, N, K);
  if (need == 0) return ER_ERR_SHAPE;
  if (arena_bytes < need) return ER_ERR_WORKSPACE;
  if (!er::aligned16(arena)) return ER_ERR_ALIGN;
  int st = er::check_arch();
  if (st != ER_OK) return st;
  Arena a{reinterpret_cast<uint8_t*>(arena), arena_bytes, 0};
  // counters first: they sit at a fixed place of the arena so that they stay zero from call to call
  const size_t ws_bytes = er_gemm_workspace_bytes(M, N, K);
  void* ws = a.take(ws_bytes);
  void* xd = a.take((size_t)M * K * 2);
  void* yd = a.take((size_t)M * N * 4);
  cudaStream_t s = (cudaStream_t)stream;
  ER_CUDA_TRY(cudaMemcpyAsync(xd, x_host, (size_t)M * K * 2, cudaMemcpyHostToDevice, s));
  st = er_w4a16_gemm(xd, M, K, K, qweight, scales, N, group, yd, N, y_dtype, ws, ws_bytes, stream);
  if (st != ER_OK) return st;
  ER_CUDA_TRY(cudaMemcpyAsync(y_host, yd, (size_t)M * N * (y_dtype == ER_F32 ? 4 : 2), cudaMemcpyDeviceToHost, s));
  return ER_OK;
}

int er_spec_verify_host(const void* target_host, const void* draft_host, int in_dtype, int inputs_are_logits,
                        float temperature, const int32_t* draft_tokens_host, const float* u_accept_host,
                        const float* u_sample_host, int32_t B, int32_t gamma, int32_t V, int32_t* accept_count_host,
                        int32_t* out_tokens_host, void* arena, size_t arena_bytes, void* stream) {
  if (in_dtype != ER_BF16 && in_dtype != ER_F32) return ER_ERR_DTYPE;
  const size_t need = er_verify_host_arena_bytes(B, gamma, V, in_dtype);
  if (need == 0) return ER_ERR_SHAPE;
  if (B == 0) return ER_OK;
  if (!target_host || !draft_host || !draft_tokens_host || !u_accept_host || !u_sample_host || !accept_count_host ||
      !out_tokens_host || !arena)
    return ER_ERR_NULL;
  if (arena_bytes < need) return ER_ERR_WORKSPACE;
  if (!er::aligned16(arena)) return ER_ERR_ALIGN;
  int st = er::check_arch();
  if (st != ER_OK) return st;
  const size_t es = (in_dtype == ER_F32) ? 4 : 2;
  const size_t tb = (size_t)B * (gamma + 1) * V * es, db = (size_t)B * gamma * V * es;
  const size_t gb = (size_t)B * gamma * 4, bb = (size_t)B * 4, ob = (size_t)B * (gamma + 1) * 4;
  Arena a{reinterpret_cast<uint8_t*>(arena), arena_bytes, ER_GEMM_COUNTER_BYTES};
  void* t = a.take(tb);
  void* d = a.take(db);
  int32_t* x = (int32_t*)a.take(gb);
  float* ua = (float*)a.take(gb);
  float* us = (float*)a.take(bb);
  int32_t* ac = (int32_t*)a.take(bb);
  int32_t* ot = (int32_t*)a.take(ob);
  cudaStream_t s = (cudaStream_t)stream;
  ER_CUDA_TRY(cudaMemcpyAsync(t, target_host, tb, cudaMemcpyHostToDevice, s));
  ER_CUDA_TRY(cudaMemcpyAsync(d, draft_host, db, cudaMemcpyHostToDevice, s));
  ER_CUDA_TRY(cudaMemcpyAsync(x, draft_tokens_host, gb, cudaMemcpyHostToDevice, s));
  ER_CUDA_TRY(cudaMemcpyAsync(ua, u_accept_host, gb, cudaMemcpyHostToDevice, s));
  ER_CUDA_TRY(cudaMemcpyAsync(us, u_sample_host, bb, cudaMemcpyHostToDevice, s));
  st = er_spec_verify(t, d, in_dtype, inputs_are_logits, temperature, x, ua, us, B, gamma, V, ac, ot, stream);
  if (st != ER_OK) return st;
  ER_CUDA_TRY(cudaMemcpyAsync(accept_count_host, ac, bb, cudaMemcpyDeviceToHost, s));
  ER_CUDA_TRY(cudaMemcpyAsync(out_tokens_host, ot, ob, cudaMemcpyDeviceToHost, s));
  return ER_OK;
}

}  // extern "C"
