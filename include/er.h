/*
 * er.h -- C ABI of the B200-native hot path of EfficientRollout's self-speculative decoding
 * (arxiv/paper_2606_18967).  Three operations, named by BASELINE.json's north_star:
 *
 *   er_quantize_pack   per-RL-step drafter refresh: bf16 linear weight -> RTN int4 (g128) + bf16 scales
 *                      PAPER.md:L101 (sec. 4.1 "lightweight RTN quantization to the FFN and QKVO projection
 *                      layers"), L150 (Alg. 1 line 3), L429 ("vanilla round-to-nearest (RTN) 4-bit")
 *   er_w4a16_gemm      drafter linear  Y = X . dequant(Wq)^T  at M = 1..256 rows
 *                      PAPER.md:L99-L101 (dense projections ~90 % of tail decode latency, weight loading
 *                      dominates), L175 (W4A16 weight-only kernel), L467 (on-the-fly dequantization)
 *   er_spec_verify     speculative-decoding verification by rejection sampling
 *                      PAPER.md:L54 (sec. 2.2), L445 (sec. D.1: accept / resample at the first rejection from
 *                      the adjusted target distribution / bonus token), L544 (needs the full distribution)
 *
 * Conventions (every entry point):
 *   - Every data pointer is a caller-owned DEVICE pointer unless the comment says "host".  The library
 *     allocates no device memory and keeps no device state.
 *   - All work is enqueued on `stream` (a cudaStream_t passed as void*; NULL = legacy default stream).
 *     No call synchronises.  Outputs are valid once the stream reaches the end of the call.
 *     Calls are CUDA-graph capturable.
 *   - Errors: the return code only (no exceptions, no abort, no printing).  Arguments are validated before
 *     anything is launched; on error nothing is enqueued.  There is NO CPU fallback: on a device that is
 *     not sm_100 the compute calls return ER_ERR_ARCH.
 *   - Determinism: identical inputs give bit-identical outputs (fixed split-K reduction order, no
 *     floating-point atomics).
 *   - Host-side state is limited to per-device caches of idempotent values (SM count, occupancy answers, "shared-memory
 *     opt-in done"); the calls may be made from several host threads and on several devices of one process.
 *
 * Data layouts:
 *   W        bf16 [N][K], row-major, K contiguous, row stride ldw elements (torch nn.Linear.weight)
 *   qweight  N*K/8 uint32 words, "ER_PACK_V2": blocks of 128 rows x 128 k (2048 words = 8 KiB, contiguous),
 *            stored tile-major then group: block (T, g) starts at word (T * K/128 + g) * 2048.  Inside a block
 *            row r keeps its place (16 words) and its four 16-byte chunks are XOR-permuted by (r >> 1) & 3: the
 *            word of k-octet j (0..15) of row r sits at  r*16 + ((j/4) ^ ((r>>1)&3))*4 + j%4.  A word holds the
 *            8 codes of logical k = 8 j + pi[i] in bits [4 i, 4 i + 4), pi = (0,2,4,6,1,3,5,7); stored nibble
 *            u = q + 8, q in [-8, 7]: (word >> 4 t) & 0x000F000F is the pair (k = 8 j + 2 t, 8 j + 2 t + 1).
 *            (One block = one contiguous, bank-conflict-free shared-memory stage of the GEMM.)
 *   scales   bf16 [K/128][N] (group-major, N contiguous); s = bf16_rne(max|w| / 7) per 128 consecutive k
 *   X        bf16 [M][K], row stride ldx elements
 *   Y        bf16 or fp32 [M][N], row stride ldy elements
 */
#ifndef ER_H_
#define ER_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ER_ABI_VERSION 1
#define ER_GROUP 128

typedef enum {
  ER_OK = 0,
  ER_ERR_NULL = 1,      /* a required pointer is NULL */
  ER_ERR_SHAPE = 2,     /* a size is out of the supported range (see each call) */
  ER_ERR_ALIGN = 3,     /* a pointer or leading dimension violates the stated alignment */
  ER_ERR_DTYPE = 4,     /* unsupported dtype / input-form combination */
  ER_ERR_WORKSPACE = 5, /* workspace missing or smaller than er_gemm_workspace_bytes() */
  ER_ERR_ARCH = 6,      /* current device is not compute capability 10.x */
  ER_ERR_CUDA = 7       /* a CUDA runtime/driver call failed; see er_last_cuda_error() */
} er_status;

typedef enum { ER_BF16 = 0, ER_F32 = 1 } er_dtype;

/* Static, never-freed description of a status code. */
const char* er_status_str(int status);
/* Thread-local cudaError_t (as int) behind the last ER_ERR_CUDA returned on this thread; 0 if none. */
int er_last_cuda_error(void);
int er_abi_version(void);

/* Sizes in bytes of the refresh outputs for a [N][K] weight.  0 if the shape is unsupported. */
size_t er_packed_bytes(int64_t N, int64_t K);            /* N*K/2 */
size_t er_scales_bytes(int64_t N, int64_t K, int group); /* (K/group)*N*2 */
/* Workspace er_w4a16_gemm needs for this problem (split-K partials + tile counters).  Never 0 for a
 * valid shape.  The first ER_GEMM_COUNTER_BYTES of the workspace hold tile counters that MUST be zero
 * before the first call that uses the workspace (er_gemm_workspace_init does that); every call leaves
 * them zero again, so one workspace may be reused by any number of calls on one stream.  (SURVEY 8(b) proposed a
 * workspace that "need not be zeroed"; a split-K ticket that recognises stale counters needs an epoch word per call,
 * i.e. library state, or a memset node per call -- one init per workspace was kept instead.) */
size_t er_gemm_workspace_bytes(int64_t M, int64_t N, int64_t K);
#define ER_GEMM_COUNTER_BYTES 16384
int er_gemm_workspace_init(void* workspace, size_t workspace_bytes, void* stream);

/* (2) Drafter refresh: quantize + pack one linear weight.
 *   w_bf16      [N][K] bf16, row stride ldw_elems (>= K); base 16-byte aligned, ldw_elems % 8 == 0
 *   group       must be 128 (ER_GROUP); K % 128 == 0, N % 128 == 0
 *   qweight_out N*K/8 uint32 words, ER_PACK_V2 (er_packed_bytes), 16-byte aligned
 *   scales_out  bf16 [K/128][N]   (er_scales_bytes), 2-byte aligned
 * Per group of 128 consecutive k of a row: amax = max|w|; s = bf16_rne(amax / 7) (IEEE fp32 divide);
 * q = clamp(rint(w / s), -8, 7) (ties to even, divide by the ROUNDED scale); s == 0 -> q = 0, s = +0.
 * NaN/Inf weights are outside the contract (no fault, unspecified codes). */
int er_quantize_pack(const void* w_bf16, int64_t N, int64_t K, int64_t ldw_elems, int group,
                     void* qweight_out, void* scales_out, void* stream);

/* The same for `count` weight matrices in as few launches as possible (the refresh of a decoder layer or of the
 * whole model: every FFN / QKVO weight, every RL step).  `descs` is a HOST array; the pointers
 * inside are DEVICE pointers with the meaning and constraints of er_quantize_pack.  Everything is validated
 * before anything is launched.  Results are identical to `count` separate calls. */
typedef struct {
  const void* w;   /* bf16 [N][K], row stride ldw elements */
  int64_t N, K, ldw;
  void* qweight;   /* out: ER_PACK_V2 */
  void* scales;    /* out: bf16 [K/128][N] */
} er_linear_desc;
int er_quantize_pack_batched(const er_linear_desc* descs, int count, int group, void* stream);

/* (1) Drafter linear:  Y[m][n] = sum_k X[m][k] * q[n][k] * s[k/128][n].
 *   x_bf16   [M][K] bf16, row stride ldx_elems; base 16-byte aligned, ldx_elems % 8 == 0; M >= 1
 *   qweight, scales  as produced by er_quantize_pack (any nibble incl. -8 is legal); N % 128 == 0,
 *            K % 128 == 0, group == 128; qweight 16-byte aligned, scales 16-byte aligned
 *   y        [M][N] of y_dtype (ER_BF16: fp32 accumulator rounded RNE; ER_F32: the accumulator itself),
 *            row stride ldy_elems; rows >= M are never written
 *   workspace  caller-provided, >= er_gemm_workspace_bytes(M,N,K), 16-byte aligned, counters zeroed once
 *            (N/128) * (K/128) * ceil(M / 64) must stay below 2^31 (else ER_ERR_SHAPE)
 * Arithmetic (three kernels, chosen from M and the work plan), the same at every M:
 *   stored nibbles u = q + 8 are widened exactly to bf16 (as 128 + u) and contracted with X on the tensor cores with fp32
 *   accumulation per 128-k group; the 136 * sum_k x[m][k] the offset adds is removed on that fp32 sum (M <= 16: through a
 *   constant operand tile, or with the x sums computed beside the contraction) or on the widened nibbles (M > 16: one
 *   packed fma, exact), so the sum holds sum_k x * q up to fp32 rounding; each group's sum is multiplied by its fp32 scale
 *   and added in fp32: q * s is NEVER rounded.  M > 64 runs in tiles of 128 or chunks of 64 batch rows (chosen per problem).
 *   Split-K partials are reduced in ascending CTA order, or inside a thread-block cluster in rank order; every kernel is
 *   deterministic (identical inputs, identical bits; no floating-point atomics).
 * Launch: one persistent kernel, launched with programmatic stream serialization; it touches no global memory before
 * griddepcontrol.wait, so ordering against earlier work in the stream (a preceding er_quantize_pack included) is the
 * usual one. */
int er_w4a16_gemm(const void* x_bf16, int64_t M, int64_t K, int64_t ldx_elems,
                  const void* qweight, const void* scales, int64_t N, int group,
                  void* y, int64_t ldy_elems, int y_dtype,
                  void* workspace, size_t workspace_bytes, void* stream);

/* Same contract and results up to fp32 summation order, computed by a plain CUDA-core kernel (no TMA, no
 * tensor cores).  Debug / cross-check aid, not a timed path; needs no workspace. */
int er_w4a16_gemm_simt(const void* x_bf16, int64_t M, int64_t K, int64_t ldx_elems,
                       const void* qweight, const void* scales, int64_t N, int group,
                       void* y, int64_t ldy_elems, int y_dtype, void* stream);

/* (1b) bf16 linear  Y[m][n] = sum_k X[m][k] * W[n][k]  with UNQUANTIZED bf16 weights: the drafter's lm_head, which the
 * paper keeps in higher precision (PAPER.md:L455 sec. D.2 "embedding, LM head, norms"; L101 quantizes only the FFN and
 * QKVO projections), and the target model's own linears -- the T_p and T_V(gamma) of the paper's speedup model
 * tau * T_p / (gamma * T_q + T_V) (Eq. 1, L488-L492 Eq. 5).
 *   x_bf16  [M][K] bf16, row stride ldx_elems; w_bf16 [N][K] bf16 (torch nn.Linear.weight), row stride ldw_elems;
 *           both bases 16-byte aligned, ldx_elems % 8 == 0, ldw_elems % 8 == 0; M >= 1, N % 128 == 0, K % 128 == 0
 *   y       [M][N] of y_dtype (ER_F32: the fp32 accumulator; ER_BF16: it rounded RNE), row stride ldy_elems
 *   workspace  >= er_bf16_gemm_workspace_bytes(M,N,K), 16-byte aligned, its first ER_GEMM_COUNTER_BYTES zero before
 *           the first use (er_gemm_workspace_init) and left zero by every call; may be shared with er_w4a16_gemm
 * Arithmetic: bf16 x bf16 products (exact in fp32) accumulated in fp32 on the tensor cores; split-K partials are
 * reduced in ascending CTA order (deterministic). */
size_t er_bf16_gemm_workspace_bytes(int64_t M, int64_t N, int64_t K);
int er_bf16_gemm(const void* x_bf16, int64_t M, int64_t K, int64_t ldx_elems, const void* w_bf16, int64_t N,
                 int64_t ldw_elems, void* y, int64_t ldy_elems, int y_dtype, void* workspace, size_t workspace_bytes,
                 void* stream);

/* (1'') er_w4a16_gemm for callers that may not allocate device memory (code under CUDA-graph capture, serving loops,
 * harnesses that forbid cudaMalloc): same operation, arithmetic and results as er_w4a16_gemm, M <= ER_STATIC_GEMM_MAX_M
 * (the memory-bound regime), but NO workspace argument -- the tile counters and split-K partial tiles live in a static
 * device array inside the library (3.2 MB; every GPU that loads the library holds it until exit).  The call allocates
 * nothing (no cudaMalloc / cudaFree, no allocating library routine) and enqueues one 16 KiB memset of the counters plus
 * the kernel on `stream`.  All calls on a device share that one array: calls that may OVERLAP on the GPU (different
 * streams, or graph branches without a dependency) race on it -- keep them ordered.  Errors as er_w4a16_gemm (on an
 * argument error at most the memset of the library's own counters has been enqueued), plus
 * ER_ERR_SHAPE for M > ER_STATIC_GEMM_MAX_M and ER_ERR_WORKSPACE on a device whose SM count the array is too small for
 * (> 192 SMs). */
#define ER_STATIC_GEMM_MAX_M 16
int er_w4a16_gemm_static(const void* x_bf16, int64_t M, int64_t K, int64_t ldx_elems, const void* qweight,
                         const void* scales, int64_t N, int group, void* y, int64_t ldy_elems, int y_dtype, void* stream);

/* (1') and (2') W8A16 drafter (Table 4 "RTN W8": the more accurate, twice as heavy
 * drafter).  RTN int8, symmetric, group 128 along K, s = bf16_rne(fp32(amax) / 127), q = clamp(rint(fp32(w) / fp32(s)),
 * -127, 127), IEEE division, ties to even; s == 0 -> q = 0 (readings W1-W3).
 *   Storage: TWO NIBBLE PLANES in the W4 layout.  With q + 128 = 16 a + b (a, b in [0, 15]), group g of the matrix becomes
 *   groups 2g (stored nibbles a) and 2g + 1 (stored nibbles b) of an ER_PACK_V2 matrix with 2 K columns:
 *   qweight_out  N * K bytes (N * 2K / 8 words), scales_out  bf16 [2K/128][N] with rows (16 s_g, s_g) -- 1 + 4/128 bytes per
 *   weight.  er_unpack_codes(qweight, N, 2 K) returns the planes as (a - 8, b - 8).
 *   er_w8a16_gemm: Y = X . dequant^T with q * s never rounded: the W4 per-group kernel contracts both planes of a group
 *   against the same 128 columns of X with fp32 accumulation and applies the fp32 scales 16 s and s to the two partial
 *   sums; the offset of the stored nibbles (128 sum_k x) is removed on the fp32 sums or on the widened nibbles.  Every M >= 1.
 *   Workspace: er_w8_gemm_workspace_bytes, counters zeroed once (er_gemm_workspace_init), shared with er_w4a16_gemm
 *   if large enough for both.  Arguments, alignment, errors, determinism as for er_quantize_pack / er_w4a16_gemm. */
int er_quantize_pack8(const void* w_bf16, int64_t N, int64_t K, int64_t ldw_elems, int group, void* qweight_out,
                      void* scales_out, void* stream);
size_t er_w8_gemm_workspace_bytes(int64_t M, int64_t N, int64_t K);
int er_w8a16_gemm(const void* x_bf16, int64_t M, int64_t K, int64_t ldx_elems, const void* qweight, const void* scales,
                  int64_t N, int group, void* y, int64_t ldy_elems, int y_dtype, void* workspace, size_t workspace_bytes,
                  void* stream);

/* (3) Speculative-decoding verification, one result per sequence b < B.
 *   target  [B][gamma+1][V]  (row gamma = bonus position), draft [B][gamma][V]; contiguous, 16-byte aligned
 *   in_dtype / inputs_are_logits: (ER_F32, 0) = fp32 probabilities; (ER_BF16, 1) and (ER_F32, 1) = logits,
 *            softmax(logit / temperature) is computed in fp32 inside the kernel; (ER_BF16, 0) -> ER_ERR_DTYPE
 *   temperature > 0 (used only for logits)
 *   draft_tokens int32 [B][gamma] in [0, V) (out-of-range ids are clamped for reads)
 *   u_accept fp32 [B][gamma] in [0,1);  u_sample fp32 [B] in [0,1)
 *   1 <= gamma <= 16, B >= 0 (B == 0 is a no-op), 1 <= V <= 2^20
 *   accept_count int32 [B] out: n = number of leading i with  fp32(u_i * q_i(x_i)) < p_i(x_i)
 *   out_tokens   int32 [B][gamma+1] out: x_1..x_n, then the token drawn at position n+1 by inverse CDF
 *            (vocab order, token = min{v : C(v) > u_sample * R}) from w = max(0, p_{n+1} - q_{n+1})
 *            (n < gamma; w = p_{n+1} if that residual is identically 0) or w = p_{gamma+1} (n == gamma),
 *            then -1 padding.
 *   Logits may be -inf (masked tokens: probability 0); a row needs at least one finite logit.  Arithmetic for logits:
 *   p(v) = 2^((l_v - m) * log2(e) / temperature) / sum, fp32, with ex2.approx (relative error 2^-22) and m a logit of the
 *   row within 32 * temperature / log2(e) of its maximum (a lazily raised reference: no term exceeds 2^32); the accept
 *   test and the residual use the same (m, sum).  One launch, one thread-block cluster per sequence. */
int er_spec_verify(const void* target, const void* draft, int in_dtype, int inputs_are_logits,
                   float temperature, const int32_t* draft_tokens, const float* u_accept,
                   const float* u_sample, int32_t B, int32_t gamma, int32_t V,
                   int32_t* accept_count, int32_t* out_tokens, void* stream);

/* Parity helper: qweight (ER_PACK_V2) -> int8 codes [N][K] in [-8, 7], row-major (device). Not timed. */
int er_unpack_codes(const void* qweight, int64_t N, int64_t K, int8_t* codes_out, void* stream);

/* ---- HOST-buffer forms of the three calls (the end-to-end path) -------------------------------------
 * Same operations and results as the device forms above.  Pointers named *_host are caller-owned HOST
 * buffers (pinned memory makes the copies asynchronous; pageable memory works, staged by the runtime),
 * dense (leading dimension = row length).  `arena` is a caller-owned DEVICE scratch buffer of at least
 * er_*_host_arena_bytes(...) bytes, 16-byte aligned; each call stages its host operands into it
 * (cudaMemcpyAsync on `stream`), runs the kernels, and copies results back to the host buffers, all on
 * `stream` without synchronising: host outputs are valid once the stream reaches the end of the call, and
 * host inputs must stay untouched until then.  Errors as above, plus ER_ERR_WORKSPACE for a small arena.
 *   er_quantize_pack_host  W comes from the host; qweight_out / scales_out stay DEVICE pointers (they are
 *                          the drafter's resident weights, consumed by er_w4a16_gemm).
 *   er_w4a16_gemm_host     X from the host, Y to the host; qweight / scales are DEVICE pointers.  The first
 *                          ER_GEMM_COUNTER_BYTES of ANY arena are reserved for the GEMM's tile counters (the
 *                          other two calls never stage over them, so one arena serves all three): zero them
 *                          once with er_gemm_workspace_init(arena, ...) before the first call.
 *   er_spec_verify_host    every operand on the host. */
size_t er_quantize_host_arena_bytes(int64_t N, int64_t K);
size_t er_gemm_host_arena_bytes(int64_t M, int64_t N, int64_t K);
size_t er_verify_host_arena_bytes(int32_t B, int32_t gamma, int32_t V, int in_dtype);
int er_quantize_pack_host(const void* w_host, int64_t N, int64_t K, int group, void* qweight_out, void* scales_out,
                          void* arena, size_t arena_bytes, void* stream);
int er_w4a16_gemm_host(const void* x_host, int64_t M, int64_t K, const void* qweight, const void* scales, int64_t N,
                       int group, void* y_host, int y_dtype, void* arena, size_t arena_bytes, void* stream);
int er_spec_verify_host(const void* target_host, const void* draft_host, int in_dtype, int inputs_are_logits,
                        float temperature, const int32_t* draft_tokens_host, const float* u_accept_host,
                        const float* u_sample_host, int32_t B, int32_t gamma, int32_t V, int32_t* accept_count_host,
                        int32_t* out_tokens_host, void* arena, size_t arena_bytes, void* stream);

/* ---- SD toggle, draft length and calibration ---------------------------------------------------
 * Scalar HOST logic of the paper's method around the three kernels: every pointer below is a HOST pointer, nothing
 * touches a device, the calls work without a GPU.  Units are SI (bytes, flop, seconds).
 *   er_roofline_model   PAPER.md:L111 (M_T, M_D, C), L455-L469 (parameter details), L473 Eq. 4 (c_comm; 0 for TP = 1):
 *     static, from the architecture:  W_T, W_D weight bytes of target and W4 drafter; C_dense flop per token; C_attn
 *       flop per token and per token of context; kappa theoretical KV bytes per token of context
 *     calibrated: F_eff (stage 1, flop/s), BW_eff (bytes/s), rho_kappa, eta_D, c_T, c_D, c_V (seconds per sequence)
 *   er_tau_of_alpha       tau = (1 - alpha^(gamma+1)) / (1 - alpha); gamma + 1 at alpha = 1
 *   er_alpha_of_tau       its inverse on [0, 1], clamped: 0 for tau <= 1, 1 for tau >= gamma + 1
 *   er_roofline_times     T_p = max{M_T, C} + c_T B, T_q = max{M_D, C} + c_D B, T_V = max{M_T, (gamma+1) C} + c_V B,
 *                         each + c_comm
 *   er_sd_toggle          pi_SD of Eq. 3: *on = 1 iff tau T_p / (gamma T_q + T_V) >= 1 + eps; the
 *                         predicted speedup goes to *speedup if that is not NULL.  (Stickiness -- "once activated, SD
 *                         remains enabled until the end of the rollout", L122 -- is the caller's one flag.)
 *   er_gamma_next         Alg. 1 lines 11-12: Gamma[0..n) ascending, gamma_t a member; tau_hist the
 *                         block efficiencies recorded so far, oldest first; returns in *gamma_out next_Gamma(gamma_t) if
 *                         the minimum of the last P is >= 1 + gamma_t alpha_up (and gamma_t < gamma_high), prev_Gamma if
 *                         the maximum of the last P is <= 1 + gamma_t alpha_down (and gamma_t > gamma_low), else gamma_t
 *                         (also when fewer than P values are recorded).  Paper's setting: {5,7,9,11}, 0.94, 0.85, P = 2.
 *   er_roofline_calibrate PAPER.md:L478-L484, steps 2-3 (F_eff and the static terms come in through *model): the target
 *                         sweep (B, S, T_p) fits BW_eff, rho_kappa, c_T; then, with those fixed, the drafter sweep
 *                         (B, S, T_q) fits eta_D, c_D and the verification sweep (B, S, gamma, T_V) fits c_V.  Ordinary
 *                         least squares on seconds; a sample counts as memory- or compute-bound by the current estimate
 *                         and classification and fit are iterated to a fixed point, starting from the values in *model
 *                         (readings P1-P2).  Arrays are parallel, n_* entries each; a sweep with n = 0 leaves
 *                         its parameters unchanged.  *model is updated in place.
 *   er_rollout_simulate   measurement driver (reading P5, not part of the paper): a batch of `n` responses of
 *                         lengths[i] tokens decoded in lockstep, B = #{lengths > position}, S = S0 + position; an AR step
 *                         costs T_p and advances 1 token, an SD block costs gamma T_q + T_V and advances tau tokens.
 *                         mode 0: AR only, 1: SD throughout, 2: pi_SD decides, sticky.  Outputs: seconds, steps, and
 *                         the steps decoded autoregressively.
 * Errors: ER_ERR_NULL, ER_ERR_SHAPE (gamma < 1, n < 0, P < 1, gamma_t not in Gamma, Gamma not ascending, a
 * non-positive F_eff / BW_eff, mode outside 0..2). */
typedef struct {
  double W_T, W_D, C_dense, C_attn, kappa;
  double F_eff, BW_eff, rho_kappa, eta_D, c_T, c_D, c_V, c_comm;
} er_roofline_model;
int er_tau_of_alpha(double alpha, int32_t gamma, double* tau_out);
int er_alpha_of_tau(double tau, int32_t gamma, double* alpha_out);
int er_roofline_times(const er_roofline_model* model, double B, double S, int32_t gamma, double* T_p, double* T_q,
                      double* T_V);
int er_sd_toggle(const er_roofline_model* model, double B, double S, double tau, int32_t gamma, double eps, int32_t* on,
                 double* speedup);
int er_gamma_next(const int32_t* Gamma, int32_t n, int32_t gamma_t, const double* tau_hist, int32_t n_hist, int32_t P,
                  double alpha_up, double alpha_down, int32_t* gamma_out);
int er_roofline_calibrate(er_roofline_model* model, const double* tB, const double* tS, const double* tT, int32_t n_target,
                          const double* dB, const double* dS, const double* dT, int32_t n_drafter, const double* vB,
                          const double* vS, const int32_t* vgamma, const double* vT, int32_t n_verify);
int er_rollout_simulate(const er_roofline_model* model, const double* lengths, int32_t n, double S0, int32_t gamma,
                        double tau, double eps, int32_t mode, double* seconds, int64_t* steps, int64_t* ar_steps);

#ifdef __cplusplus
}
#endif
#endif /* ER_H_ */
