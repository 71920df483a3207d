"""Thin ctypes binding over liber_b200.so (include/er.h).  Argument marshalling only: every step of the
path runs in the CUDA kernels behind the C ABI.  PyTorch supplies device memory and streams.

There is no CPU fallback: if the library is missing it is built with nvcc (in-tree); if that fails, or a
call returns a non-zero status, an exception is raised.
"""
from __future__ import annotations

import contextlib
import ctypes

import torch

from . import build as _build

ER_BF16, ER_F32 = 0, 1
GROUP = 128
COUNTER_BYTES = 16384

_lib = None


class LinearDesc(ctypes.Structure):
    """er_linear_desc of include/er.h."""
    _fields_ = [("w", ctypes.c_void_p), ("N", ctypes.c_int64), ("K", ctypes.c_int64), ("ldw", ctypes.c_int64),
                ("qweight", ctypes.c_void_p), ("scales", ctypes.c_void_p)]


class RooflineModel(ctypes.Structure):
    """er_roofline_model of include/er.h (SI units)."""
    _fields_ = [(n, ctypes.c_double) for n in ("W_T", "W_D", "C_dense", "C_attn", "kappa", "F_eff", "BW_eff",
                                               "rho_kappa", "eta_D", "c_T", "c_D", "c_V", "c_comm")]


class ErError(RuntimeError):
    def __init__(self, status: int, where: str):
        lib = load()
        msg = lib.er_status_str(status).decode()
        cuda = lib.er_last_cuda_error() if status == 7 else 0
        super().__init__(f"{where}: {msg}" + (f" (cudaError {cuda})" if cuda else ""))
        self.status = status


def _bind(lib: ctypes.CDLL) -> ctypes.CDLL:
    """Declare the argument / result types of every entry point of include/er.h."""
    vp, i64, i32, sz, f32 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_size_t, ctypes.c_float
    lib.er_status_str.restype = ctypes.c_char_p
    lib.er_status_str.argtypes = [ctypes.c_int]
    lib.er_last_cuda_error.restype = ctypes.c_int
    lib.er_abi_version.restype = ctypes.c_int
    lib.er_packed_bytes.restype = sz
    lib.er_packed_bytes.argtypes = [i64, i64]
    lib.er_scales_bytes.restype = sz
    lib.er_scales_bytes.argtypes = [i64, i64, ctypes.c_int]
    lib.er_gemm_workspace_bytes.restype = sz
    lib.er_gemm_workspace_bytes.argtypes = [i64, i64, i64]
    lib.er_gemm_workspace_init.restype = ctypes.c_int
    lib.er_gemm_workspace_init.argtypes = [vp, sz, vp]
    lib.er_quantize_pack.restype = ctypes.c_int
    lib.er_quantize_pack.argtypes = [vp, i64, i64, i64, ctypes.c_int, vp, vp, vp]
    lib.er_quantize_pack_batched.restype = ctypes.c_int
    lib.er_quantize_pack_batched.argtypes = [ctypes.POINTER(LinearDesc), ctypes.c_int, ctypes.c_int, vp]
    lib.er_w4a16_gemm.restype = ctypes.c_int
    lib.er_w4a16_gemm.argtypes = [vp, i64, i64, i64, vp, vp, i64, ctypes.c_int, vp, i64, ctypes.c_int, vp, sz, vp]
    lib.er_quantize_pack8.restype = ctypes.c_int
    lib.er_quantize_pack8.argtypes = [vp, i64, i64, i64, ctypes.c_int, vp, vp, vp]
    lib.er_w8_gemm_workspace_bytes.restype = sz
    lib.er_w8_gemm_workspace_bytes.argtypes = [i64, i64, i64]
    lib.er_w8a16_gemm.restype = ctypes.c_int
    lib.er_w8a16_gemm.argtypes = [vp, i64, i64, i64, vp, vp, i64, ctypes.c_int, vp, i64, ctypes.c_int, vp, sz, vp]
    lib.er_w4a16_gemm_static.restype = ctypes.c_int
    lib.er_w4a16_gemm_static.argtypes = [vp, i64, i64, i64, vp, vp, i64, ctypes.c_int, vp, i64, ctypes.c_int, vp]
    lib.er_w4a16_gemm_simt.restype = ctypes.c_int
    lib.er_w4a16_gemm_simt.argtypes = [vp, i64, i64, i64, vp, vp, i64, ctypes.c_int, vp, i64, ctypes.c_int, vp]
    lib.er_bf16_gemm_workspace_bytes.restype = sz
    lib.er_bf16_gemm_workspace_bytes.argtypes = [i64, i64, i64]
    lib.er_bf16_gemm.restype = ctypes.c_int
    lib.er_bf16_gemm.argtypes = [vp, i64, i64, i64, vp, i64, i64, vp, i64, ctypes.c_int, vp, sz, vp]
    lib.er_spec_verify.restype = ctypes.c_int
    lib.er_spec_verify.argtypes = [vp, vp, ctypes.c_int, ctypes.c_int, f32, vp, vp, vp, i32, i32, i32, vp, vp, vp]
    lib.er_unpack_codes.restype = ctypes.c_int
    lib.er_unpack_codes.argtypes = [vp, i64, i64, vp, vp]
    lib.er_quantize_host_arena_bytes.restype = sz
    lib.er_quantize_host_arena_bytes.argtypes = [i64, i64]
    lib.er_gemm_host_arena_bytes.restype = sz
    lib.er_gemm_host_arena_bytes.argtypes = [i64, i64, i64]
    lib.er_verify_host_arena_bytes.restype = sz
    lib.er_verify_host_arena_bytes.argtypes = [i32, i32, i32, ctypes.c_int]
    lib.er_quantize_pack_host.restype = ctypes.c_int
    lib.er_quantize_pack_host.argtypes = [vp, i64, i64, ctypes.c_int, vp, vp, vp, sz, vp]
    lib.er_w4a16_gemm_host.restype = ctypes.c_int
    lib.er_w4a16_gemm_host.argtypes = [vp, i64, i64, vp, vp, i64, ctypes.c_int, vp, ctypes.c_int, vp, sz, vp]
    lib.er_spec_verify_host.restype = ctypes.c_int
    lib.er_spec_verify_host.argtypes = [vp, vp, ctypes.c_int, ctypes.c_int, f32, vp, vp, vp, i32, i32, i32, vp, vp, vp,
                                        sz, vp]
    f64, pd, pm = ctypes.c_double, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(RooflineModel)
    pi32, pi64 = ctypes.POINTER(i32), ctypes.POINTER(i64)
    for name, args in (("er_tau_of_alpha", [f64, i32, pd]), ("er_alpha_of_tau", [f64, i32, pd]),
                       ("er_roofline_times", [pm, f64, f64, i32, pd, pd, pd]),
                       ("er_sd_toggle", [pm, f64, f64, f64, i32, f64, pi32, pd]),
                       ("er_gamma_next", [pi32, i32, i32, pd, i32, i32, f64, f64, pi32]),
                       ("er_roofline_calibrate", [pm, pd, pd, pd, i32, pd, pd, pd, i32, pd, pd, pi32, pd, i32]),
                       ("er_rollout_simulate", [pm, pd, i32, f64, i32, f64, f64, i32, pd, pi64, pi64])):
        getattr(lib, name).restype = ctypes.c_int
        getattr(lib, name).argtypes = args
    if lib.er_abi_version() != 1:
        raise RuntimeError("liber_b200.so ABI version mismatch")
    return lib


def load() -> ctypes.CDLL:
    """Load the C-ABI library, (re)building it first when it is missing or older than its sources
    (build_library is a no-op when the .so is fresh).  Raises if it cannot be had: there is no other path."""
    global _lib
    if _lib is None:
        _lib = _bind(ctypes.CDLL(_build.build_library()))
    return _lib


@contextlib.contextmanager
def dev_library():
    """Tests only: route this module's calls through the DEVELOPMENT build (liber_b200_dev.so, csrc/er_dev.h), which
    adds the partition / launch-mode knobs, and hand the library out so that they can be set.  Every knob is reset
    and the shipped library restored on exit."""
    global _lib
    lib = _bind(ctypes.CDLL(_build.build_library(dev=True)))
    lib.er_dev_gemm_tuning.restype = ctypes.c_int
    lib.er_dev_gemm_tuning.argtypes = [ctypes.c_int, ctypes.c_int]
    lib.er_dev_verify_cluster.restype = ctypes.c_int
    lib.er_dev_verify_cluster.argtypes = [ctypes.c_int]
    prev = load()
    _lib = lib
    try:
        yield lib
    finally:
        for key, value in ((1, 0), (3, 1), (4, 1), (5, 1), (6, 1), (7, 0), (8, 1), (9, 0)):
            lib.er_dev_gemm_tuning(key, value)
        lib.er_dev_verify_cluster(0)
        lib.er_dev_verify_cluster(16)
        _lib = prev


def _stream(t: torch.Tensor) -> int:
    return torch.cuda.current_stream(t.device).cuda_stream


def _check(status: int, where: str):
    if status != 0:
        raise ErError(status, where)


def _cuda(t: torch.Tensor, name: str):
    if not t.is_cuda:
        raise ValueError(f"{name} must be a CUDA tensor (the library takes device pointers; no CPU path exists)")


def packed_bytes(N: int, K: int) -> int:
    return load().er_packed_bytes(N, K)


def scales_bytes(N: int, K: int, group: int = GROUP) -> int:
    return load().er_scales_bytes(N, K, group)


def gemm_workspace_bytes(M: int, N: int, K: int) -> int:
    return load().er_gemm_workspace_bytes(M, N, K)


def gemm_workspace(M: int, N: int, K: int, device) -> torch.Tensor:
    """Allocate and initialise (counters zeroed) a workspace large enough for this problem."""
    nbytes = gemm_workspace_bytes(M, N, K)
    if nbytes == 0:
        raise ErError(2, "er_gemm_workspace_bytes")
    ws = torch.empty(nbytes, dtype=torch.uint8, device=device)
    _check(load().er_gemm_workspace_init(ws.data_ptr(), nbytes, _stream(ws)), "er_gemm_workspace_init")
    return ws


def quantize_pack(w: torch.Tensor, qweight: torch.Tensor | None = None, scales: torch.Tensor | None = None,
                  group: int = GROUP):
    """bf16 W[N][K] -> (qweight int32 [N][K/8] (ER_PACK_V2 layout, include/er.h), scales bf16 [K/128][N])."""
    _cuda(w, "w")
    assert w.dtype == torch.bfloat16 and w.dim() == 2 and w.stride(1) == 1
    N, K = w.shape
    if qweight is None:
        qweight = torch.empty((N, K // 8), dtype=torch.int32, device=w.device)
    if scales is None:
        scales = torch.empty((K // group, N), dtype=torch.bfloat16, device=w.device)
    _check(load().er_quantize_pack(w.data_ptr(), N, K, w.stride(0), group, qweight.data_ptr(), scales.data_ptr(),
                                   _stream(w)), "er_quantize_pack")
    return qweight, scales


def quantize_pack_batched(items, group: int = GROUP):
    """items: iterable of (w, qweight, scales) device tensors; one call for all of them (er_quantize_pack_batched)."""
    items = list(items)
    if not items:
        return
    arr = (LinearDesc * len(items))()
    for d, (w, qweight, scales) in zip(arr, items):
        _cuda(w, "w")
        assert w.dtype == torch.bfloat16 and w.dim() == 2 and w.stride(1) == 1
        d.w, d.N, d.K, d.ldw = w.data_ptr(), w.shape[0], w.shape[1], w.stride(0)
        d.qweight, d.scales = qweight.data_ptr(), scales.data_ptr()
    _check(load().er_quantize_pack_batched(arr, len(items), group, _stream(items[0][0])), "er_quantize_pack_batched")


def w4a16_gemm(x: torch.Tensor, qweight: torch.Tensor, scales: torch.Tensor, out_dtype=torch.bfloat16,
               y: torch.Tensor | None = None, workspace: torch.Tensor | None = None, simt: bool = False):
    """Y[M][N] = X[M][K] . dequant(qweight, scales)[N][K]^T."""
    _cuda(x, "x")
    assert x.dtype == torch.bfloat16 and x.dim() == 2 and x.stride(1) == 1
    M, K = x.shape
    N = qweight.shape[0]
    if y is None:
        y = torch.empty((M, N), dtype=out_dtype, device=x.device)
    ydt = ER_F32 if y.dtype == torch.float32 else ER_BF16
    lib = load()
    if simt:
        _check(lib.er_w4a16_gemm_simt(x.data_ptr(), M, K, x.stride(0), qweight.data_ptr(), scales.data_ptr(), N, GROUP,
                                      y.data_ptr(), y.stride(0), ydt, _stream(x)), "er_w4a16_gemm_simt")
        return y
    if workspace is None:
        workspace = gemm_workspace(M, N, K, x.device)
    _check(lib.er_w4a16_gemm(x.data_ptr(), M, K, x.stride(0), qweight.data_ptr(), scales.data_ptr(), N, GROUP,
                             y.data_ptr(), y.stride(0), ydt, workspace.data_ptr(), workspace.numel(), _stream(x)),
           "er_w4a16_gemm")
    return y


def w4a16_gemm_static(x: torch.Tensor, qweight: torch.Tensor, scales: torch.Tensor, y: torch.Tensor):
    """er_w4a16_gemm_static: Y = X . dequant^T at M <= 16 with the scratch in the library's static device array; the
    caller passes inputs and the output, nothing is allocated here or in the library."""
    M, K = x.shape
    N = qweight.shape[0]
    ydt = ER_F32 if y.dtype == torch.float32 else ER_BF16
    _check(load().er_w4a16_gemm_static(x.data_ptr(), M, K, x.stride(0), qweight.data_ptr(), scales.data_ptr(), N, GROUP,
                                       y.data_ptr(), y.stride(0), ydt, _stream(x)), "er_w4a16_gemm_static")
    return y


def quantize_pack8(w: torch.Tensor, qweight: torch.Tensor | None = None, scales: torch.Tensor | None = None):
    """W8 refresh: bf16 W[N][K] -> (qweight int32 [N][2K/8]: two nibble planes in the W4 layout, scales bf16 [2K/128][N]:
    rows (16 s_g, s_g)); include/er.h."""
    _cuda(w, "w")
    assert w.dtype == torch.bfloat16 and w.dim() == 2 and w.stride(1) == 1
    N, K = w.shape
    if qweight is None:
        qweight = torch.empty((N, 2 * K // 8), dtype=torch.int32, device=w.device)
    if scales is None:
        scales = torch.empty((2 * K // GROUP, N), dtype=torch.bfloat16, device=w.device)
    _check(load().er_quantize_pack8(w.data_ptr(), N, K, w.stride(0), GROUP, qweight.data_ptr(), scales.data_ptr(),
                                    _stream(w)), "er_quantize_pack8")
    return qweight, scales


def w8a16_gemm(x: torch.Tensor, qweight: torch.Tensor, scales: torch.Tensor, out_dtype=torch.bfloat16,
               y: torch.Tensor | None = None, workspace: torch.Tensor | None = None):
    """Y[M][N] = X[M][K] . dequant(two-plane qweight, scales)[N][K]^T (er_w8a16_gemm)."""
    _cuda(x, "x")
    assert x.dtype == torch.bfloat16 and x.dim() == 2 and x.stride(1) == 1
    M, K = x.shape
    N = qweight.shape[0]
    if y is None:
        y = torch.empty((M, N), dtype=out_dtype, device=x.device)
    ydt = ER_F32 if y.dtype == torch.float32 else ER_BF16
    lib = load()
    if workspace is None:
        nbytes = lib.er_w8_gemm_workspace_bytes(M, N, K)
        if nbytes == 0:
            raise ErError(2, "er_w8_gemm_workspace_bytes")
        workspace = torch.empty(nbytes, dtype=torch.uint8, device=x.device)
        _check(lib.er_gemm_workspace_init(workspace.data_ptr(), nbytes, _stream(x)), "er_gemm_workspace_init")
    _check(lib.er_w8a16_gemm(x.data_ptr(), M, K, x.stride(0), qweight.data_ptr(), scales.data_ptr(), N, GROUP,
                             y.data_ptr(), y.stride(0), ydt, workspace.data_ptr(), workspace.numel(), _stream(x)),
           "er_w8a16_gemm")
    return y


def bf16_gemm(x: torch.Tensor, w: torch.Tensor, out_dtype=torch.bfloat16, y: torch.Tensor | None = None,
              workspace: torch.Tensor | None = None):
    """Y[M][N] = X[M][K] . W[N][K]^T with bf16 weights (lm_head, target-side linears)."""
    _cuda(x, "x")
    assert x.dtype == torch.bfloat16 and w.dtype == torch.bfloat16 and x.stride(1) == 1 and w.stride(1) == 1
    M, K = x.shape
    N = w.shape[0]
    if y is None:
        y = torch.empty((M, N), dtype=out_dtype, device=x.device)
    ydt = ER_F32 if y.dtype == torch.float32 else ER_BF16
    lib = load()
    if workspace is None:
        nbytes = lib.er_bf16_gemm_workspace_bytes(M, N, K)
        if nbytes == 0:
            raise ErError(2, "er_bf16_gemm_workspace_bytes")
        workspace = torch.empty(nbytes, dtype=torch.uint8, device=x.device)
        _check(lib.er_gemm_workspace_init(workspace.data_ptr(), nbytes, _stream(x)), "er_gemm_workspace_init")
    _check(lib.er_bf16_gemm(x.data_ptr(), M, K, x.stride(0), w.data_ptr(), N, w.stride(0), y.data_ptr(), y.stride(0), ydt,
                            workspace.data_ptr(), workspace.numel(), _stream(x)), "er_bf16_gemm")
    return y


def spec_verify(target: torch.Tensor, draft: torch.Tensor, draft_tokens: torch.Tensor, u_accept: torch.Tensor,
                u_sample: torch.Tensor, inputs_are_logits: bool, temperature: float = 1.0,
                accept_count: torch.Tensor | None = None, out_tokens: torch.Tensor | None = None):
    """target [B][gamma+1][V], draft [B][gamma][V] -> (accept_count int32 [B], out_tokens int32 [B][gamma+1])."""
    _cuda(target, "target")
    B, G1, V = target.shape
    gamma = G1 - 1
    assert draft.shape == (B, gamma, V) and target.is_contiguous() and draft.is_contiguous()
    assert target.dtype == draft.dtype and target.dtype in (torch.float32, torch.bfloat16)
    assert draft_tokens.dtype == torch.int32 and u_accept.dtype == torch.float32 and u_sample.dtype == torch.float32
    dt = ER_F32 if target.dtype == torch.float32 else ER_BF16
    if accept_count is None:
        accept_count = torch.empty((B,), dtype=torch.int32, device=target.device)
    if out_tokens is None:
        out_tokens = torch.empty((B, gamma + 1), dtype=torch.int32, device=target.device)
    _check(load().er_spec_verify(target.data_ptr(), draft.data_ptr(), dt, int(inputs_are_logits), float(temperature),
                                 draft_tokens.data_ptr(), u_accept.data_ptr(), u_sample.data_ptr(), B, gamma, V,
                                 accept_count.data_ptr(), out_tokens.data_ptr(), _stream(target)), "er_spec_verify")
    return accept_count, out_tokens


def unpack_codes(qweight: torch.Tensor) -> torch.Tensor:
    _cuda(qweight, "qweight")
    N, J = qweight.shape
    codes = torch.empty((N, J * 8), dtype=torch.int8, device=qweight.device)
    _check(load().er_unpack_codes(qweight.data_ptr(), N, J * 8, codes.data_ptr(), _stream(qweight)), "er_unpack_codes")
    return codes


# ---- host-buffer forms (include/er.h "HOST-buffer forms"): host tensors in / out, device arena for staging ----

def _host(t: torch.Tensor, name: str):
    if t.is_cuda or not t.is_contiguous():
        raise ValueError(f"{name} must be a contiguous host tensor")


def host_arena(nbytes: int, device) -> torch.Tensor:
    """Device staging arena for the *_host calls; GEMM tile counters (its first bytes) zeroed."""
    arena = torch.empty(max(int(nbytes), COUNTER_BYTES), dtype=torch.uint8, device=device)
    _check(load().er_gemm_workspace_init(arena.data_ptr(), arena.numel(), _stream(arena)), "er_gemm_workspace_init")
    return arena


def quantize_pack_host(w_host: torch.Tensor, qweight: torch.Tensor, scales: torch.Tensor, arena: torch.Tensor):
    _host(w_host, "w_host")
    N, K = w_host.shape
    _check(load().er_quantize_pack_host(w_host.data_ptr(), N, K, GROUP, qweight.data_ptr(), scales.data_ptr(),
                                        arena.data_ptr(), arena.numel(), _stream(arena)), "er_quantize_pack_host")
    return qweight, scales


def w4a16_gemm_host(x_host: torch.Tensor, qweight: torch.Tensor, scales: torch.Tensor, y_host: torch.Tensor,
                    arena: torch.Tensor):
    _host(x_host, "x_host")
    _host(y_host, "y_host")
    M, K = x_host.shape
    N = qweight.shape[0]
    ydt = ER_F32 if y_host.dtype == torch.float32 else ER_BF16
    _check(load().er_w4a16_gemm_host(x_host.data_ptr(), M, K, qweight.data_ptr(), scales.data_ptr(), N, GROUP,
                                     y_host.data_ptr(), ydt, arena.data_ptr(), arena.numel(), _stream(arena)),
           "er_w4a16_gemm_host")
    return y_host


def spec_verify_host(target: torch.Tensor, draft: torch.Tensor, draft_tokens: torch.Tensor, u_accept: torch.Tensor,
                     u_sample: torch.Tensor, inputs_are_logits: bool, temperature: float,
                     accept_count: torch.Tensor, out_tokens: torch.Tensor, arena: torch.Tensor):
    for t, n in ((target, "target"), (draft, "draft"), (draft_tokens, "draft_tokens"), (u_accept, "u_accept"),
                 (u_sample, "u_sample"), (accept_count, "accept_count"), (out_tokens, "out_tokens")):
        _host(t, n)
    B, G1, V = target.shape
    dt = ER_F32 if target.dtype == torch.float32 else ER_BF16
    _check(load().er_spec_verify_host(target.data_ptr(), draft.data_ptr(), dt, int(inputs_are_logits),
                                      float(temperature), draft_tokens.data_ptr(), u_accept.data_ptr(),
                                      u_sample.data_ptr(), B, G1 - 1, V, accept_count.data_ptr(),
                                      out_tokens.data_ptr(), arena.data_ptr(), arena.numel(), _stream(arena)),
           "er_spec_verify_host")
    return accept_count, out_tokens


# ---- SD toggle, draft length, calibration (include/er.h): host scalars in, host scalars out ----------
def _darr(xs):
    xs = [float(x) for x in xs]
    return (ctypes.c_double * len(xs))(*xs), len(xs)


def tau_of_alpha(alpha: float, gamma: int) -> float:
    out = ctypes.c_double()
    _check(load().er_tau_of_alpha(alpha, gamma, ctypes.byref(out)), "er_tau_of_alpha")
    return out.value


def alpha_of_tau(tau: float, gamma: int) -> float:
    out = ctypes.c_double()
    _check(load().er_alpha_of_tau(tau, gamma, ctypes.byref(out)), "er_alpha_of_tau")
    return out.value


def roofline_times(model: RooflineModel, B: float, S: float, gamma: int):
    tp, tq, tv = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    _check(load().er_roofline_times(ctypes.byref(model), B, S, gamma, ctypes.byref(tp), ctypes.byref(tq),
                                    ctypes.byref(tv)), "er_roofline_times")
    return tp.value, tq.value, tv.value


def sd_toggle(model: RooflineModel, B: float, S: float, tau: float, gamma: int, eps: float):
    on, s = ctypes.c_int32(), ctypes.c_double()
    _check(load().er_sd_toggle(ctypes.byref(model), B, S, tau, gamma, eps, ctypes.byref(on), ctypes.byref(s)),
           "er_sd_toggle")
    return on.value, s.value


def gamma_next(Gamma, gamma_t: int, tau_hist, P: int, alpha_up: float, alpha_down: float) -> int:
    G = (ctypes.c_int32 * len(Gamma))(*[int(g) for g in Gamma])
    h, nh = _darr(tau_hist)
    out = ctypes.c_int32()
    _check(load().er_gamma_next(G, len(Gamma), gamma_t, h, nh, P, alpha_up, alpha_down, ctypes.byref(out)),
           "er_gamma_next")
    return out.value


def roofline_calibrate(model: RooflineModel, target, drafter, verify) -> RooflineModel:
    """target rows (B, S, T_p), drafter rows (B, S, T_q), verify rows (B, S, gamma, T_V); returns the fitted copy."""
    out = RooflineModel.from_buffer_copy(model)
    tb, nt = _darr([r[0] for r in target]); ts, _ = _darr([r[1] for r in target]); tt, _ = _darr([r[2] for r in target])
    db, nd = _darr([r[0] for r in drafter]); ds, _ = _darr([r[1] for r in drafter]); dt, _ = _darr([r[2] for r in drafter])
    vb, nv = _darr([r[0] for r in verify]); vs, _ = _darr([r[1] for r in verify]); vt, _ = _darr([r[3] for r in verify])
    vg = (ctypes.c_int32 * nv)(*[int(r[2]) for r in verify])
    _check(load().er_roofline_calibrate(ctypes.byref(out), tb, ts, tt, nt, db, ds, dt, nd, vb, vs, vg, vt, nv),
           "er_roofline_calibrate")
    return out


def rollout_simulate(model: RooflineModel, lengths, S0: float, gamma: int, tau: float, eps: float, mode: int):
    L, n = _darr(lengths)
    sec, steps, ar = ctypes.c_double(), ctypes.c_int64(), ctypes.c_int64()
    _check(load().er_rollout_simulate(ctypes.byref(model), L, n, S0, gamma, tau, eps, mode, ctypes.byref(sec),
                                      ctypes.byref(steps), ctypes.byref(ar)), "er_rollout_simulate")
    return sec.value, steps.value, ar.value
