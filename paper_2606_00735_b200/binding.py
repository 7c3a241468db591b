"""Thin ctypes binding over libvibe.so (include/vibe.h) -- argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels; PyTorch is used here
for device memory and streams only.  Names mirror the C ABI:

    route_topk, permute, grouped_ffn, combine, profile_expert_latency,
    moe_layer_forward, moe_layer_forward_host,
    placement_eval, placement_greedy, placement_token_balanced, placement_contiguous,
    drift_cosine, DriftMonitor, placement_swap_refine

There is NO fallback: if libvibe.so is missing or a call fails, a VibeError is raised.
"""
from __future__ import annotations

import ctypes as C
import dataclasses
import os
from typing import Optional, Sequence

import numpy as np
import torch

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libvibe.so")

VIBE_OK = 0
SCORE_SOFTMAX = 0
SCORE_SIGMOID = 1
WS_PERMUTE, WS_FFN, WS_PROFILE, WS_LAYER, WS_LAYER_HOST, WS_LAYER_FP8, WS_LAYER_MXFP8 = 0, 1, 2, 3, 4, 5, 6
MX_SF_ROWMAJOR, MX_SF_TOKENS, MX_SF_GATE_UP, MX_SF_DOWN = 0, 1, 2, 3
MX_ROLE_DOWN, MX_ROLE_GATE, MX_ROLE_UP = 0, 1, 2
MX_ROW_ALIGN = 64
MODEL_A, MODEL_B = 0, 1

# every symbol include/vibe.h declares (tests check that the .so exports exactly these)
EXPORTED_SYMBOLS = (
    "vibe_route_topk", "vibe_permute", "vibe_permute_static", "vibe_grouped_ffn", "vibe_combine",
    "vibe_profile_expert_latency", "vibe_moe_layer_forward", "vibe_moe_layer_forward_host", "vibe_workspace_bytes", "vibe_rows_cap",
    "vibe_status_string", "vibe_last_error", "vibe_version", "vibe_launch_count",
    "vibe_placement_eval", "vibe_placement_greedy", "vibe_placement_token_balanced", "vibe_placement_contiguous",
    "vibe_grouped_ffn_scatter", "vibe_combine_scattered",
    "vibe_fp8_quantize_rows", "vibe_fp8_pack_weights", "vibe_grouped_ffn_fp8", "vibe_moe_layer_forward_fp8",
    "vibe_profile_expert_latency_fp8", "vibe_moe_layer_forward_host_chunked",
    "vibe_profile_expert_latency_mxfp8", "vibe_l2_flush", "vibe_moe_layer_forward_host_async", "vibe_host_wait", "vibe_mxfp8_sf_bytes", "vibe_mxfp8_quantize_rows", "vibe_mxfp8_pack_weights", "vibe_grouped_ffn_mxfp8",
    "vibe_moe_layer_forward_mxfp8",
    "vibe_drift_cosine", "vibe_drift_monitor_create", "vibe_drift_monitor_destroy",
    "vibe_drift_monitor_set_reference", "vibe_drift_monitor_push", "vibe_drift_monitor_rearranged",
    "vibe_drift_monitor_window_mean", "vibe_placement_swap_refine",
)


class VibeError(RuntimeError):
    pass


class _RouteCfg(C.Structure):
    _fields_ = [("num_experts", C.c_int32), ("top_k", C.c_int32), ("score_fn", C.c_int32),
                ("renormalize", C.c_int32), ("routed_scale", C.c_float), ("n_group", C.c_int32),
                ("topk_group", C.c_int32), ("select_bias", C.c_void_p)]


class _LatencyModel(C.Structure):
    _fields_ = [("n_points", C.c_int32), ("tokens", C.POINTER(C.c_double)),
                ("latency_us", C.POINTER(C.c_double)), ("E_prof", C.c_int32)]


@dataclasses.dataclass
class RouteConfig:
    num_experts: int
    top_k: int
    score_fn: int = SCORE_SOFTMAX
    renormalize: int = 1
    routed_scale: float = 1.0
    n_group: int = 0
    topk_group: int = 0
    select_bias: Optional[torch.Tensor] = None      # device f32 [E]

    def _c(self) -> _RouteCfg:
        b = self.select_bias
        if b is not None:
            _check(b, torch.float32, "select_bias")
        return _RouteCfg(self.num_experts, self.top_k, self.score_fn, self.renormalize, self.routed_scale,
                         self.n_group, self.topk_group, b.data_ptr() if b is not None else None)


@dataclasses.dataclass
class LatencyModel:
    tokens: Sequence[float]
    latency_us: Sequence[float]
    E_prof: int = 1


_lib = None


def load() -> C.CDLL:
    """Load libvibe.so (built in-tree by `python -m paper_2606_00735_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise VibeError(f"{LIB_PATH} not found: build it with `python -m paper_2606_00735_b200.build` "
                        "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, sz = C.c_void_p, C.c_int32, C.c_size_t
    lib.vibe_route_topk.argtypes = [C.POINTER(_RouteCfg), vp, i32, vp, vp, vp, vp]
    lib.vibe_permute.argtypes = [vp, vp, vp, vp, i32, i32, i32, i32, i32, i32, vp, vp, vp, vp, vp, sz, vp]
    lib.vibe_permute_static.argtypes = [vp, vp, vp, vp, i32, i32, i32, i32, i32, i32, vp, vp, vp, vp, vp]
    lib.vibe_permute_static.restype = C.c_int
    lib.vibe_grouped_ffn.argtypes = [vp, vp, i32, i32, i32, i32, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.vibe_combine.argtypes = [vp, vp, vp, i32, i32, i32, vp, vp]
    lib.vibe_grouped_ffn_scatter.argtypes = [vp, vp, i32, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    lib.vibe_combine_scattered.argtypes = [vp, vp, i32, i32, i32, vp, vp]
    lib.vibe_fp8_quantize_rows.argtypes = [vp, i32, i32, vp, vp, vp]
    lib.vibe_fp8_pack_weights.argtypes = [vp, i32, i32, i32, vp, vp, vp]
    lib.vibe_grouped_ffn_fp8.argtypes = [vp, vp, vp, i32, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.vibe_profile_expert_latency.argtypes = [i32, i32, i32, vp, vp, vp, C.POINTER(i32), i32, i32, i32, i32,
                                                C.POINTER(C.c_float), C.POINTER(C.c_float), vp, sz, vp]
    lib.vibe_profile_expert_latency_fp8.argtypes = [i32, i32, i32, vp, vp, vp, vp, vp, vp, vp, C.POINTER(i32), i32, i32, i32,
                                                    i32, C.POINTER(C.c_float), C.POINTER(C.c_float), vp, sz, vp]
    lib.vibe_moe_layer_forward.argtypes = [C.POINTER(_RouteCfg), vp, vp, vp, i32, i32, i32, i32, vp, vp, vp, vp, vp,
                                           vp, vp, vp, sz, vp]
    lib.vibe_moe_layer_forward_host.argtypes = [C.POINTER(_RouteCfg), vp, vp, vp, i32, i32, i32, i32, vp, vp, vp,
                                                vp, vp, vp, sz, vp]
    lib.vibe_moe_layer_forward_host_chunked.argtypes = [C.POINTER(_RouteCfg), vp, vp, vp, i32, i32, i32, i32, vp, vp,
                                                        vp, vp, vp, i32, vp, sz, vp]
    lib.vibe_moe_layer_forward_fp8.argtypes = [C.POINTER(_RouteCfg), vp, vp, vp, i32, i32, i32, i32, vp, vp, vp, vp, vp,
                                               vp, vp, vp, vp, vp, sz, vp]
    lib.vibe_profile_expert_latency_mxfp8.argtypes = [i32, i32, i32, vp, vp, vp, vp, vp, C.POINTER(i32), i32, i32, i32, i32,
                                                      C.POINTER(C.c_float), C.POINTER(C.c_float), vp, sz, vp]
    lib.vibe_profile_expert_latency_mxfp8.restype = C.c_int
    lib.vibe_moe_layer_forward_host_async.argtypes = [C.POINTER(_RouteCfg), vp, vp, vp, i32, i32, i32, i32, vp, vp, vp,
                                                      vp, vp, vp, sz, vp, C.POINTER(i32)]
    lib.vibe_moe_layer_forward_host_async.restype = C.c_int
    lib.vibe_host_wait.argtypes = [i32]
    lib.vibe_host_wait.restype = C.c_int
    lib.vibe_l2_flush.argtypes = [vp, sz, vp]
    lib.vibe_l2_flush.restype = C.c_int
    lib.vibe_mxfp8_sf_bytes.argtypes = [i32] * 4
    lib.vibe_mxfp8_sf_bytes.restype = sz
    lib.vibe_mxfp8_quantize_rows.argtypes = [vp, i32, i32, i32, vp, vp, i32, i32, vp]
    lib.vibe_mxfp8_pack_weights.argtypes = [vp, i32, i32, i32, i32, i32, vp, vp, vp]
    lib.vibe_grouped_ffn_mxfp8.argtypes = [vp, vp, vp, i32, i32, i32, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.vibe_moe_layer_forward_mxfp8.argtypes = [C.POINTER(_RouteCfg), vp, vp, vp, i32, i32, i32, i32, vp, vp, vp, vp, vp,
                                                 vp, vp, vp, sz, vp]
    lib.vibe_workspace_bytes.argtypes = [i32] * 8
    lib.vibe_workspace_bytes.restype = sz
    lib.vibe_rows_cap.argtypes = [i32] * 4
    lib.vibe_rows_cap.restype = C.c_int64
    lib.vibe_status_string.argtypes = [C.c_int]
    lib.vibe_status_string.restype = C.c_char_p
    lib.vibe_last_error.restype = C.c_char_p
    lib.vibe_version.restype = i32
    lib.vibe_launch_count.restype = C.c_int64
    dp = C.POINTER(C.c_double)
    lib.vibe_placement_eval.argtypes = [C.POINTER(i32), dp, i32, i32, dp, C.POINTER(_LatencyModel), i32, dp]
    lib.vibe_placement_eval.restype = C.c_double
    lib.vibe_placement_greedy.argtypes = [dp, i32, i32, dp, C.POINTER(_LatencyModel), i32, C.POINTER(i32)]
    lib.vibe_placement_token_balanced.argtypes = [dp, i32, i32, i32, C.POINTER(i32)]
    lib.vibe_placement_contiguous.argtypes = [i32, i32, C.POINTER(i32)]
    lib.vibe_drift_cosine.argtypes = [dp, dp, i32]
    lib.vibe_drift_cosine.restype = C.c_double
    lib.vibe_drift_monitor_create.argtypes = [i32, i32, i32, i32, C.c_double]
    lib.vibe_drift_monitor_create.restype = vp
    lib.vibe_drift_monitor_destroy.argtypes = [vp]
    lib.vibe_drift_monitor_destroy.restype = None
    lib.vibe_drift_monitor_set_reference.argtypes = [vp, dp]
    lib.vibe_drift_monitor_push.argtypes = [vp, dp, dp, C.POINTER(i32)]
    lib.vibe_drift_monitor_push.restype = i32
    lib.vibe_drift_monitor_rearranged.argtypes = [vp]
    lib.vibe_drift_monitor_window_mean.argtypes = [vp, dp]
    lib.vibe_placement_swap_refine.argtypes = [C.POINTER(i32), dp, i32, i32, dp, C.POINTER(_LatencyModel), i32,
                                               C.c_double, i32, C.POINTER(i32), C.POINTER(i32)]
    for name in ("vibe_route_topk", "vibe_permute", "vibe_grouped_ffn", "vibe_combine", "vibe_grouped_ffn_scatter",
                 "vibe_combine_scattered", "vibe_moe_layer_forward_fp8", "vibe_fp8_quantize_rows", "vibe_fp8_pack_weights", "vibe_grouped_ffn_fp8",
                 "vibe_profile_expert_latency", "vibe_profile_expert_latency_fp8", "vibe_moe_layer_forward", "vibe_moe_layer_forward_host",
                 "vibe_moe_layer_forward_host_chunked", "vibe_placement_greedy", "vibe_placement_token_balanced", "vibe_placement_contiguous",
                 "vibe_drift_monitor_set_reference", "vibe_drift_monitor_rearranged",
                 "vibe_mxfp8_quantize_rows", "vibe_mxfp8_pack_weights", "vibe_grouped_ffn_mxfp8", "vibe_moe_layer_forward_mxfp8",
                 "vibe_drift_monitor_window_mean", "vibe_placement_swap_refine"):
        getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def _ok(status: int, what: str) -> None:
    if status != VIBE_OK:
        lib = load()
        raise VibeError(f"{what}: {lib.vibe_status_string(status).decode()}: {lib.vibe_last_error().decode()}")


def _check(t: torch.Tensor, dtype, name: str) -> None:
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise VibeError(f"{name} must be a CUDA tensor (no CPU fallback)")
    if t.dtype != dtype:
        raise VibeError(f"{name} must be {dtype}, got {t.dtype}")
    if not t.is_contiguous():
        raise VibeError(f"{name} must be contiguous")


def _stream(stream) -> int:
    s = stream if stream is not None else torch.cuda.current_stream()
    return s.cuda_stream


def _scratch(nbytes: int, device, stream) -> torch.Tensor:
    """A temporary workspace / arena the call itself allocates.  It is allocated UNDER the launch stream: the caching
    allocator then ties its reuse to that stream, so returning it to the pool right after the (asynchronous) call is
    safe even when `stream` is not torch's current stream."""
    if stream is None:
        return torch.empty((max(nbytes, 16),), dtype=torch.uint8, device=device)
    with torch.cuda.stream(stream):
        return torch.empty((max(nbytes, 16),), dtype=torch.uint8, device=device)


def l2_flush(scratch: torch.Tensor, stream=None) -> None:
    """evict the L2 before a timed region (scratch: a uint8 CUDA tensor of >= 2 x the L2 size)"""
    _ok(load().vibe_l2_flush(scratch.data_ptr(), scratch.numel(), _stream(stream)), "vibe_l2_flush")


def launch_count() -> int:
    return int(load().vibe_launch_count())


def workspace_bytes(which: int, T: int, k: int, E: int, E_loc: int, d: int, f: int, align: int = 1) -> int:
    return int(load().vibe_workspace_bytes(which, T, k, E, E_loc, d, f, align))


def rows_cap(T: int, k: int, E_loc: int, align: int = 1) -> int:
    return int(load().vibe_rows_cap(T, k, E_loc, align))


# ------------------------------------------------------------------------------------ a1+a2
def route_topk(logits: torch.Tensor, cfg: RouteConfig, out=None, stream=None):
    """-> (topk_ids i32 [T,k], topk_w f32 [T,k], counts i32 [E])"""
    lib = load()
    _check(logits, torch.float32, "logits")
    T, E = logits.shape
    if E != cfg.num_experts:
        raise VibeError("logits.shape[1] != cfg.num_experts")
    dev = logits.device
    if out is None:
        ids = torch.empty((T, cfg.top_k), dtype=torch.int32, device=dev)
        w = torch.empty((T, cfg.top_k), dtype=torch.float32, device=dev)
        counts = torch.empty((E,), dtype=torch.int32, device=dev)
    else:
        ids, w, counts = out
    c = cfg._c()
    _ok(lib.vibe_route_topk(C.byref(c), logits.data_ptr(), T, ids.data_ptr(), w.data_ptr(), counts.data_ptr(),
                            _stream(stream)), "vibe_route_topk")
    return ids, w, counts


# ------------------------------------------------------------------------------------ a3
def permute(X: torch.Tensor, topk_ids: torch.Tensor, counts: Optional[torch.Tensor],
            expert_map: Optional[torch.Tensor], E: int, E_loc: int, align: int = 1, out=None, ws=None, stream=None):
    """-> (Xp bf16 [R_cap,d], offsets i32 [E_loc+1], row_to_assign i32 [R_cap], assign_to_row i32 [T*k])"""
    lib = load()
    _check(X, torch.bfloat16, "X")
    _check(topk_ids, torch.int32, "topk_ids")
    T, d = X.shape
    k = topk_ids.shape[1]
    dev = X.device
    Rcap = max(1, rows_cap(T, k, E_loc, align))
    if out is None:
        Xp = torch.empty((Rcap, d), dtype=torch.bfloat16, device=dev)
        offsets = torch.empty((E_loc + 1,), dtype=torch.int32, device=dev)
        r2a = torch.empty((Rcap,), dtype=torch.int32, device=dev)
        a2r = torch.empty((T * k,), dtype=torch.int32, device=dev)
    else:
        Xp, offsets, r2a, a2r = out
    need = workspace_bytes(WS_PERMUTE, T, k, E, E_loc, d, 0, align)
    if ws is None:
        ws = _scratch(need, dev, stream)
    _ok(lib.vibe_permute(X.data_ptr(), topk_ids.data_ptr(), counts.data_ptr() if counts is not None else None,
                         expert_map.data_ptr() if expert_map is not None else None, T, d, k, E, E_loc, align,
                         Xp.data_ptr(), offsets.data_ptr(), r2a.data_ptr(), a2r.data_ptr(), ws.data_ptr(),
                         ws.numel(), _stream(stream)), "vibe_permute")
    return Xp, offsets, r2a, a2r


PERMUTE_STATIC_BYTES = 304 * 1024


def permute_static(X: torch.Tensor, topk_ids: torch.Tensor, counts: Optional[torch.Tensor],
                   expert_map: Optional[torch.Tensor], E: int, E_loc: int, align: int, out, stream=None):
    """vibe_permute_static: permute() with the scratch in the library's static device array -- the call allocates
    nothing, so every output is the caller's (`out` = (Xp, offsets, row_to_assign, assign_to_row), required)."""
    lib = load()
    _check(X, torch.bfloat16, "X")
    _check(topk_ids, torch.int32, "topk_ids")
    T, d = X.shape
    k = topk_ids.shape[1]
    Xp, offsets, r2a, a2r = out
    _ok(lib.vibe_permute_static(X.data_ptr(), topk_ids.data_ptr(), counts.data_ptr() if counts is not None else None,
                                expert_map.data_ptr() if expert_map is not None else None, T, d, k, E, E_loc, align,
                                Xp.data_ptr(), offsets.data_ptr(), r2a.data_ptr(), a2r.data_ptr(), _stream(stream)),
        "vibe_permute_static")
    return Xp, offsets, r2a, a2r


# ------------------------------------------------------------------------------------ a4
def grouped_ffn(Xp: torch.Tensor, offsets: torch.Tensor, W1: torch.Tensor, W3: torch.Tensor, W2: torch.Tensor,
                H: Optional[torch.Tensor] = None, Y: Optional[torch.Tensor] = None, stream=None, ws="auto"):
    """-> Y bf16 [R_cap,d]  (H bf16 [R_cap,f] scratch is returned too).  ws: split-K workspace (WS_FFN bytes);
    "auto" allocates one for the call, None runs without (no split-K)."""
    lib = load()
    for t, n in ((Xp, "Xp"), (W1, "W1"), (W3, "W3"), (W2, "W2")):
        _check(t, torch.bfloat16, n)
    _check(offsets, torch.int32, "offsets")
    Rcap, d = Xp.shape
    E_loc, d1, f = W1.shape
    if d1 != d or tuple(W3.shape) != (E_loc, d, f) or tuple(W2.shape) != (E_loc, f, d):
        raise VibeError("weight shapes must be W1,W3 [E_loc,d,f], W2 [E_loc,f,d]")
    if offsets.numel() != E_loc + 1:
        raise VibeError("offsets must have E_loc+1 entries")
    if H is None:
        H = torch.empty((Rcap, f), dtype=torch.bfloat16, device=Xp.device)
    if Y is None:
        Y = torch.empty((Rcap, d), dtype=torch.bfloat16, device=Xp.device)
    if isinstance(ws, str):
        ws = _scratch(workspace_bytes(WS_FFN, 1, 1, 1, E_loc, d, f, 1), Xp.device, stream)
    _ok(lib.vibe_grouped_ffn(Xp.data_ptr(), offsets.data_ptr(), E_loc, Rcap, d, f, W1.data_ptr(), W3.data_ptr(),
                             W2.data_ptr(), H.data_ptr(), Y.data_ptr(), ws.data_ptr() if ws is not None else None,
                             ws.numel() if ws is not None else 0, _stream(stream)), "vibe_grouped_ffn")
    return Y, H


def grouped_ffn_scatter(Xp: torch.Tensor, offsets: torch.Tensor, W1: torch.Tensor, W3: torch.Tensor,
                        W2: torch.Tensor, row_to_assign: torch.Tensor, topk_w: torch.Tensor,
                        H: Optional[torch.Tensor] = None, Yw: Optional[torch.Tensor] = None, stream=None, ws="auto"):
    """-> Yw bf16 [T*k, d] in assignment order, gate-weighted (rows of non-resident assignments untouched)"""
    lib = load()
    for t, n in ((Xp, "Xp"), (W1, "W1"), (W3, "W3"), (W2, "W2")):
        _check(t, torch.bfloat16, n)
    _check(offsets, torch.int32, "offsets")
    _check(row_to_assign, torch.int32, "row_to_assign")
    _check(topk_w, torch.float32, "topk_w")
    Rcap, d = Xp.shape
    E_loc, d1, f = W1.shape
    if d1 != d or tuple(W3.shape) != (E_loc, d, f) or tuple(W2.shape) != (E_loc, f, d):
        raise VibeError("weight shapes must be W1,W3 [E_loc,d,f], W2 [E_loc,f,d]")
    if H is None:
        H = torch.empty((Rcap, f), dtype=torch.bfloat16, device=Xp.device)
    if Yw is None:
        Yw = torch.empty((topk_w.numel(), d), dtype=torch.bfloat16, device=Xp.device)
    if isinstance(ws, str):
        ws = _scratch(workspace_bytes(WS_FFN, 1, 1, 1, E_loc, d, f, 1), Xp.device, stream)
    _ok(lib.vibe_grouped_ffn_scatter(Xp.data_ptr(), offsets.data_ptr(), E_loc, Rcap, d, f, W1.data_ptr(),
                                     W3.data_ptr(), W2.data_ptr(), row_to_assign.data_ptr(), topk_w.data_ptr(),
                                     H.data_ptr(), Yw.data_ptr(), ws.data_ptr() if ws is not None else None,
                                     ws.numel() if ws is not None else 0, _stream(stream)),
        "vibe_grouped_ffn_scatter")
    return Yw, H


def combine_scattered(Yw: torch.Tensor, assign_to_row: torch.Tensor, T: int, k: int,
                      out: Optional[torch.Tensor] = None, stream=None):
    lib = load()
    _check(Yw, torch.bfloat16, "Yw")
    _check(assign_to_row, torch.int32, "assign_to_row")
    d = Yw.shape[1]
    if out is None:
        out = torch.empty((T, d), dtype=torch.bfloat16, device=Yw.device)
    _ok(lib.vibe_combine_scattered(Yw.data_ptr(), assign_to_row.data_ptr(), T, k, d, out.data_ptr(),
                                   _stream(stream)), "vibe_combine_scattered")
    return out


# ------------------------------------------------------------------------------------ f2: FP8
def fp8_quantize_rows(X: torch.Tensor, stream=None):
    """bf16 [R,d] -> (Xq uint8 e4m3 codes [R,d], row_scale f32 [R])"""
    lib = load()
    _check(X, torch.bfloat16, "X")
    R, d = X.shape
    Xq = torch.empty((R, d), dtype=torch.uint8, device=X.device)
    rs = torch.empty((R,), dtype=torch.float32, device=X.device)
    _ok(lib.vibe_fp8_quantize_rows(X.data_ptr(), R, d, Xq.data_ptr(), rs.data_ptr(), _stream(stream)),
        "vibe_fp8_quantize_rows")
    return Xq, rs


def fp8_pack_weights(W: torch.Tensor, stream=None):
    """bf16 [E,K,N] -> (Wq uint8 e4m3 codes [E,N,K], scale f32 [E])"""
    lib = load()
    _check(W, torch.bfloat16, "W")
    E, K, N = W.shape
    Wq = torch.empty((E, N, K), dtype=torch.uint8, device=W.device)
    sc = torch.empty((E,), dtype=torch.float32, device=W.device)
    _ok(lib.vibe_fp8_pack_weights(W.data_ptr(), E, K, N, Wq.data_ptr(), sc.data_ptr(), _stream(stream)),
        "vibe_fp8_pack_weights")
    return Wq, sc


def grouped_ffn_fp8(Xq, row_scale, offsets, W1q, s1, W3q, s3, W2q, s2, h_scale, Hq=None, Y=None, stream=None):
    """-> (Y bf16 [R_cap,d], Hq uint8 [R_cap,f])"""
    lib = load()
    for t, n in ((Xq, "Xq"), (W1q, "W1q"), (W3q, "W3q"), (W2q, "W2q")):
        _check(t, torch.uint8, n)
    for t, n in ((row_scale, "row_scale"), (s1, "s1"), (s3, "s3"), (s2, "s2"), (h_scale, "h_scale")):
        _check(t, torch.float32, n)
    _check(offsets, torch.int32, "offsets")
    Rcap, d = Xq.shape
    E_loc, f, d1 = W1q.shape
    if d1 != d or tuple(W3q.shape) != (E_loc, f, d) or tuple(W2q.shape) != (E_loc, d, f):
        raise VibeError("packed weight shapes must be W1q,W3q [E_loc,f,d], W2q [E_loc,d,f]")
    if Hq is None:
        Hq = torch.empty((Rcap, f), dtype=torch.uint8, device=Xq.device)
    if Y is None:
        Y = torch.empty((Rcap, d), dtype=torch.bfloat16, device=Xq.device)
    _ok(lib.vibe_grouped_ffn_fp8(Xq.data_ptr(), row_scale.data_ptr(), offsets.data_ptr(), E_loc, Rcap, d, f,
                                 W1q.data_ptr(), s1.data_ptr(), W3q.data_ptr(), s3.data_ptr(), W2q.data_ptr(),
                                 s2.data_ptr(), h_scale.data_ptr(), Hq.data_ptr(), Y.data_ptr(), _stream(stream)),
        "vibe_grouped_ffn_fp8")
    return Y, Hq


# ------------------------------------------------------------------------------------ a5
# ------------------------------------------------------------------------------------ f2: block-scaled FP8
def mxfp8_sf_bytes(which: int, rows: int, K: int, E_loc: int = 1) -> int:
    return int(load().vibe_mxfp8_sf_bytes(which, rows, K, E_loc))


def mxfp8_sf_offsets(which: int, rows: int, K: int, R_cap: int = 0, role: int = MX_ROLE_DOWN):
    """Byte offsets [rows, K/32] (int64, CPU) of the scale of (row r, 32-block b) inside one expert's part of a
    scale array: the layout formulas of include/vibe.h written out as index arithmetic (no arithmetic of the
    method).  Tests use it to read a device layout back into row-major order."""
    r = torch.arange(rows, dtype=torch.int64)[:, None]
    b = torch.arange(K // 32, dtype=torch.int64)[None, :]
    if which == MX_SF_ROWMAJOR:
        return r * (K // 32) + b
    if which == MX_SF_TOKENS:
        Rb = ((max(R_cap, rows) + 31) // 32 + 3) // 4 * 4
        return (((b // 4) * 32 + r % 32) * Rb + r // 32) * 4 + b % 4
    if which == MX_SF_GATE_UP:
        return ((b // 4) * (rows // 64) + r // 64) * 512 + (r % 32) * 16 + ((r % 64) // 32 + (2 if role == MX_ROLE_UP else 0)) * 4 + b % 4
    if which == MX_SF_DOWN:
        return ((b // 4) * (rows // 128) + r // 128) * 512 + (r % 32) * 16 + ((r % 128) // 32) * 4 + b % 4
    raise VibeError("bad scale-factor layout")


def mxfp8_quantize_rows(X: torch.Tensor, block: int = 32, sf_layout: int = MX_SF_ROWMAJOR, R_cap: int = 0, stream=None):
    """bf16 [R,d] -> (Xq uint8 e4m3 codes [R,d], sf uint8: [R,d/32] row-major, or the flat TOKENS-layout array)"""
    lib = load()
    _check(X, torch.bfloat16, "X")
    R, d = X.shape
    R_cap = max(R_cap, R)
    Xq = torch.empty((R, d), dtype=torch.uint8, device=X.device)
    if sf_layout == MX_SF_ROWMAJOR:
        sf = torch.empty((R, d // 32), dtype=torch.uint8, device=X.device)
    else:
        sf = torch.full((max(16, mxfp8_sf_bytes(MX_SF_TOKENS, R_cap, d)),), 127, dtype=torch.uint8, device=X.device)
    _ok(lib.vibe_mxfp8_quantize_rows(X.data_ptr(), R, d, block, Xq.data_ptr(), sf.data_ptr(), sf_layout, R_cap,
                                     _stream(stream)), "vibe_mxfp8_quantize_rows")
    return Xq, sf


def mxfp8_pack_weights(W: torch.Tensor, role: int, block: int = 32, sf: Optional[torch.Tensor] = None, stream=None):
    """bf16 [E,K,N] -> (Wq uint8 e4m3 codes [E,N,K], sf uint8 flat): role DOWN -> a DOWN scale array; roles GATE / UP
    fill their halves of one GATE_UP array (pass the array returned for W1 as `sf` when packing W3)."""
    lib = load()
    _check(W, torch.bfloat16, "W")
    E, K, N = W.shape
    Wq = torch.empty((E, N, K), dtype=torch.uint8, device=W.device)
    if sf is None:
        which = MX_SF_DOWN if role == MX_ROLE_DOWN else MX_SF_GATE_UP
        sf = torch.full((max(16, mxfp8_sf_bytes(which, N, K, E)),), 127, dtype=torch.uint8, device=W.device)
    _ok(lib.vibe_mxfp8_pack_weights(W.data_ptr(), E, K, N, block, role, Wq.data_ptr(), sf.data_ptr(), _stream(stream)),
        "vibe_mxfp8_pack_weights")
    return Wq, sf


def grouped_ffn_mxfp8(Xq, Xsf, offsets, W1q, W3q, sf13, W2q, sf2, Hq=None, Hsf=None, Y=None, stream=None):
    """-> (Y bf16 [R_cap,d], Hq uint8 [R_cap,f], Hsf uint8 flat (TOKENS layout, K = f)); offsets multiples of 32."""
    lib = load()
    for t, n in ((Xq, "Xq"), (Xsf, "Xsf"), (W1q, "W1q"), (W3q, "W3q"), (W2q, "W2q"), (sf13, "sf13"), (sf2, "sf2")):
        _check(t, torch.uint8, n)
    _check(offsets, torch.int32, "offsets")
    Rcap, d = Xq.shape
    E_loc, f, d1 = W1q.shape
    if d1 != d or tuple(W3q.shape) != (E_loc, f, d) or tuple(W2q.shape) != (E_loc, d, f):
        raise VibeError("packed weight shapes must be W1q,W3q [E_loc,f,d], W2q [E_loc,d,f]")
    if Xsf.numel() < mxfp8_sf_bytes(MX_SF_TOKENS, Rcap, d) or sf13.numel() < mxfp8_sf_bytes(MX_SF_GATE_UP, f, d, E_loc) \
            or sf2.numel() < mxfp8_sf_bytes(MX_SF_DOWN, d, f, E_loc):
        raise VibeError("scale-factor array too small for its layout")
    if Hq is None:
        Hq = torch.empty((Rcap, f), dtype=torch.uint8, device=Xq.device)
    if Hsf is None:
        Hsf = torch.full((max(16, mxfp8_sf_bytes(MX_SF_TOKENS, Rcap, f)),), 127, dtype=torch.uint8, device=Xq.device)
    if Y is None:
        Y = torch.empty((Rcap, d), dtype=torch.bfloat16, device=Xq.device)
    _ok(lib.vibe_grouped_ffn_mxfp8(Xq.data_ptr(), Xsf.data_ptr(), offsets.data_ptr(), E_loc, Rcap, d, f, W1q.data_ptr(),
                                   W3q.data_ptr(), sf13.data_ptr(), W2q.data_ptr(), sf2.data_ptr(), Hq.data_ptr(),
                                   Hsf.data_ptr(), Y.data_ptr(), _stream(stream)), "vibe_grouped_ffn_mxfp8")
    return Y, Hq, Hsf


def moe_layer_forward_mxfp8(cfg: RouteConfig, logits, X, expert_map, W1q, W3q, sf13, W2q, sf2, out=None, counts=None,
                            arena=None, stream=None):
    """The whole layer with the block-scaled FP8 FFN (weights packed by mxfp8_pack_weights)."""
    lib = load()
    _check(logits, torch.float32, "logits")
    _check(X, torch.bfloat16, "X")
    T, d = X.shape
    E_loc, f, _ = W1q.shape
    dev = X.device
    if out is None:
        out = torch.empty((T, d), dtype=torch.bfloat16, device=dev)
    if counts is None:
        counts = torch.empty((cfg.num_experts,), dtype=torch.int32, device=dev)
    need = workspace_bytes(WS_LAYER_MXFP8, T, cfg.top_k, cfg.num_experts, E_loc, d, f, 1)
    if arena is None:
        arena = _scratch(need, dev, stream)
    c = cfg._c()
    _ok(lib.vibe_moe_layer_forward_mxfp8(C.byref(c), logits.data_ptr(), X.data_ptr(),
                                         expert_map.data_ptr() if expert_map is not None else None, T, d, f, E_loc,
                                         W1q.data_ptr(), W3q.data_ptr(), sf13.data_ptr(), W2q.data_ptr(), sf2.data_ptr(),
                                         out.data_ptr(), counts.data_ptr(), arena.data_ptr(), arena.numel(),
                                         _stream(stream)), "vibe_moe_layer_forward_mxfp8")
    return out, counts


def combine(Y: torch.Tensor, assign_to_row: torch.Tensor, topk_w: torch.Tensor, T: int, k: int,
            out: Optional[torch.Tensor] = None, stream=None):
    lib = load()
    _check(Y, torch.bfloat16, "Y")
    _check(assign_to_row, torch.int32, "assign_to_row")
    _check(topk_w, torch.float32, "topk_w")
    d = Y.shape[1]
    if out is None:
        out = torch.empty((T, d), dtype=torch.bfloat16, device=Y.device)
    _ok(lib.vibe_combine(Y.data_ptr(), assign_to_row.data_ptr(), topk_w.data_ptr(), T, k, d, out.data_ptr(),
                         _stream(stream)), "vibe_combine")
    return out


# ------------------------------------------------------------------------------------ a6
DEFAULT_SWEEP = (1, 2, 3, 4, 6, 8, 12, 16, 24, 32, 48, 64, 96, 128, 192, 256, 384, 512, 768, 1024, 1536, 2048,
                 3072, 4096)


def profile_expert_latency(W1: torch.Tensor, W3: torch.Tensor, W2: torch.Tensor,
                           tokens_per_expert: Sequence[int] = DEFAULT_SWEEP, mode: int = 0, warmup: int = 10,
                           iters: int = 100, return_samples: bool = False, ws=None, stream=None):
    """Measured grouped-FFN latency [us] per sweep point (median); mode 0 = per-expert cost with all
    experts loaded uniformly, mode 1 = one loaded expert."""
    lib = load()
    for t, n in ((W1, "W1"), (W3, "W3"), (W2, "W2")):
        _check(t, torch.bfloat16, n)
    E_loc, d, f = W1.shape
    toks = (C.c_int32 * len(tokens_per_expert))(*[int(x) for x in tokens_per_expert])
    npts = len(tokens_per_expert)
    lat = (C.c_float * npts)()
    samples = (C.c_float * (npts * iters))() if return_samples else None
    need = workspace_bytes(WS_PROFILE, max(tokens_per_expert), 1, E_loc, E_loc, d, f, 1)
    if ws is None:
        ws = _scratch(need, W1.device, stream)
    _ok(lib.vibe_profile_expert_latency(E_loc, d, f, W1.data_ptr(), W3.data_ptr(), W2.data_ptr(), toks, npts, mode,
                                        warmup, iters, lat, samples, ws.data_ptr(), ws.numel(), _stream(stream)),
        "vibe_profile_expert_latency")
    lat_np = np.array(lat[:], dtype=np.float64)
    if return_samples:
        return lat_np, np.array(samples[:], dtype=np.float64).reshape(npts, iters)
    return lat_np


def profile_expert_latency_fp8(W1q, s1, W3q, s3, W2q, s2, h_scale, tokens_per_expert: Sequence[int] = DEFAULT_SWEEP,
                               mode: int = 0, warmup: int = 10, iters: int = 100, stream=None):
    """vibe_profile_expert_latency for the FP8 FFN (median latency [us] per sweep point)."""
    lib = load()
    E_loc, f, d = W1q.shape
    toks = (C.c_int32 * len(tokens_per_expert))(*[int(x) for x in tokens_per_expert])
    npts = len(tokens_per_expert)
    lat = (C.c_float * npts)()
    nmax = max(tokens_per_expert)
    need = (workspace_bytes(WS_PROFILE, nmax, 1, E_loc, E_loc, d, f, 1) + 255) // 256 * 256 + \
        (4 * E_loc * max(nmax, 1) + 255) // 256 * 256
    ws = _scratch(need, W1q.device, stream)
    _ok(lib.vibe_profile_expert_latency_fp8(E_loc, d, f, W1q.data_ptr(), s1.data_ptr(), W3q.data_ptr(), s3.data_ptr(),
                                            W2q.data_ptr(), s2.data_ptr(), h_scale.data_ptr(), toks, npts, mode, warmup,
                                            iters, lat, None, ws.data_ptr(), ws.numel(), _stream(stream)),
        "vibe_profile_expert_latency_fp8")
    return np.array(lat[:], dtype=np.float64)


def profile_expert_latency_mxfp8(W1q, W3q, sf13, W2q, sf2, tokens_per_expert: Sequence[int] = DEFAULT_SWEEP, mode: int = 0,
                                 warmup: int = 10, iters: int = 100, stream=None):
    """vibe_profile_expert_latency for the block-scaled FP8 FFN (median latency [us] per sweep point)."""
    lib = load()
    E_loc, f, d = W1q.shape
    toks = (C.c_int32 * len(tokens_per_expert))(*[int(x) for x in tokens_per_expert])
    npts = len(tokens_per_expert)
    lat = (C.c_float * npts)()
    n_pad = max((max(tokens_per_expert) + MX_ROW_ALIGN - 1) // MX_ROW_ALIGN * MX_ROW_ALIGN, MX_ROW_ALIGN)
    r256 = lambda x: (x + 255) // 256 * 256
    need = r256(workspace_bytes(WS_PROFILE, n_pad, 1, E_loc, E_loc, d, f, 1)) + \
        r256(mxfp8_sf_bytes(MX_SF_TOKENS, E_loc * n_pad, d)) + r256(mxfp8_sf_bytes(MX_SF_TOKENS, E_loc * n_pad, f))
    ws = _scratch(need, W1q.device, stream)
    _ok(lib.vibe_profile_expert_latency_mxfp8(E_loc, d, f, W1q.data_ptr(), W3q.data_ptr(), sf13.data_ptr(), W2q.data_ptr(),
                                              sf2.data_ptr(), toks, npts, mode, warmup, iters, lat, None, ws.data_ptr(),
                                              ws.numel(), _stream(stream)), "vibe_profile_expert_latency_mxfp8")
    return np.array(lat[:], dtype=np.float64)


# ------------------------------------------------------------------------------------ layer
def moe_layer_forward(cfg: RouteConfig, logits, X, expert_map, W1, W3, W2, out=None, counts=None, topk_ids=None,
                      topk_w=None, arena=None, stream=None):
    lib = load()
    _check(logits, torch.float32, "logits")
    _check(X, torch.bfloat16, "X")
    T, d = X.shape
    E_loc, _, f = W1.shape
    dev = X.device
    if out is None:
        out = torch.empty((T, d), dtype=torch.bfloat16, device=dev)
    if counts is None:
        counts = torch.empty((cfg.num_experts,), dtype=torch.int32, device=dev)
    need = workspace_bytes(WS_LAYER, T, cfg.top_k, cfg.num_experts, E_loc, d, f, 1)
    if arena is None:
        arena = _scratch(need, dev, stream)
    c = cfg._c()
    _ok(lib.vibe_moe_layer_forward(C.byref(c), logits.data_ptr(), X.data_ptr(),
                                   expert_map.data_ptr() if expert_map is not None else None, T, d, f, E_loc,
                                   W1.data_ptr(), W3.data_ptr(), W2.data_ptr(), out.data_ptr(), counts.data_ptr(),
                                   topk_ids.data_ptr() if topk_ids is not None else None,
                                   topk_w.data_ptr() if topk_w is not None else None, arena.data_ptr(),
                                   arena.numel(), _stream(stream)), "vibe_moe_layer_forward")
    return out, counts


def moe_layer_forward_fp8(cfg: RouteConfig, logits, X, expert_map, W1q, s1, W3q, s3, W2q, s2, h_scale, out=None,
                          counts=None, arena=None, stream=None):
    """The whole layer with the FP8 FFN (weights packed by fp8_pack_weights)."""
    lib = load()
    _check(logits, torch.float32, "logits")
    _check(X, torch.bfloat16, "X")
    T, d = X.shape
    E_loc, f, _ = W1q.shape
    dev = X.device
    if out is None:
        out = torch.empty((T, d), dtype=torch.bfloat16, device=dev)
    if counts is None:
        counts = torch.empty((cfg.num_experts,), dtype=torch.int32, device=dev)
    need = workspace_bytes(WS_LAYER_FP8, T, cfg.top_k, cfg.num_experts, E_loc, d, f, 1)
    if arena is None:
        arena = _scratch(need, dev, stream)
    c = cfg._c()
    _ok(lib.vibe_moe_layer_forward_fp8(C.byref(c), logits.data_ptr(), X.data_ptr(),
                                       expert_map.data_ptr() if expert_map is not None else None, T, d, f, E_loc,
                                       W1q.data_ptr(), s1.data_ptr(), W3q.data_ptr(), s3.data_ptr(), W2q.data_ptr(),
                                       s2.data_ptr(), h_scale.data_ptr(), out.data_ptr(), counts.data_ptr(),
                                       arena.data_ptr(), arena.numel(), _stream(stream)),
        "vibe_moe_layer_forward_fp8")
    return out, counts


def moe_layer_forward_host(cfg: RouteConfig, logits_h: torch.Tensor, X_h: torch.Tensor, expert_map, W1, W3, W2,
                           out_h: torch.Tensor, counts_h: torch.Tensor, arena: torch.Tensor, stream=None,
                           n_chunks: int = 0):
    """End to end from (pinned) HOST tensors; returns when out_h / counts_h are filled.  n_chunks: token chunks of
    the copy/compute pipeline (0 = chosen by the library)."""
    lib = load()
    T, d = X_h.shape
    E_loc, _, f = W1.shape
    assert not logits_h.is_cuda and not X_h.is_cuda and not out_h.is_cuda and not counts_h.is_cuda
    c = cfg._c()
    emap = expert_map.data_ptr() if expert_map is not None else None
    if n_chunks == 0:
        _ok(lib.vibe_moe_layer_forward_host(C.byref(c), logits_h.data_ptr(), X_h.data_ptr(), emap, T, d, f, E_loc,
                                            W1.data_ptr(), W3.data_ptr(), W2.data_ptr(), out_h.data_ptr(),
                                            counts_h.data_ptr(), arena.data_ptr(), arena.numel(), _stream(stream)),
            "vibe_moe_layer_forward_host")
    else:
        _ok(lib.vibe_moe_layer_forward_host_chunked(C.byref(c), logits_h.data_ptr(), X_h.data_ptr(), emap, T, d, f,
                                                    E_loc, W1.data_ptr(), W3.data_ptr(), W2.data_ptr(),
                                                    out_h.data_ptr(), counts_h.data_ptr(), int(n_chunks),
                                                    arena.data_ptr(), arena.numel(), _stream(stream)),
            "vibe_moe_layer_forward_host_chunked")
    return out_h, counts_h


def moe_layer_forward_host_async(cfg: RouteConfig, logits_h: torch.Tensor, X_h: torch.Tensor, expert_map, W1, W3, W2,
                                 out_h: torch.Tensor, counts_h: torch.Tensor, arena: torch.Tensor, stream=None) -> int:
    """Enqueue one step from PINNED host tensors and return its ticket; host_wait(ticket) blocks until out_h / counts_h
    are filled.  The arena, the result buffers and the inputs belong to the call until then (use two sets to overlap
    consecutive steps)."""
    lib = load()
    T, d = X_h.shape
    E_loc, _, f = W1.shape
    assert not logits_h.is_cuda and not X_h.is_cuda and not out_h.is_cuda and not counts_h.is_cuda
    c = cfg._c()
    t = C.c_int32(-1)
    _ok(lib.vibe_moe_layer_forward_host_async(C.byref(c), logits_h.data_ptr(), X_h.data_ptr(),
                                              expert_map.data_ptr() if expert_map is not None else None, T, d, f, E_loc,
                                              W1.data_ptr(), W3.data_ptr(), W2.data_ptr(), out_h.data_ptr(),
                                              counts_h.data_ptr(), arena.data_ptr(), arena.numel(), _stream(stream),
                                              C.byref(t)), "vibe_moe_layer_forward_host_async")
    return int(t.value)


def host_wait(ticket: int) -> None:
    _ok(load().vibe_host_wait(int(ticket)), "vibe_host_wait")


# ------------------------------------------------------------------------------------ placement (host)
def _dp(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.POINTER(C.c_double))


def _model(m: Optional[LatencyModel]):
    if m is None:
        return None, None
    t, tp = _dp(m.tokens)
    l, lp = _dp(m.latency_us)
    return C.byref(_LatencyModel(len(t), tp, lp, int(m.E_prof))), (t, l)


def placement_eval(assign, load_, G: int, scale, model: Optional[LatencyModel], model_kind: int = MODEL_B):
    lib = load()
    a = np.ascontiguousarray(assign, dtype=np.int32)
    ld, ldp = _dp(load_)
    sc, scp = _dp(scale)
    per = np.zeros(G, dtype=np.float64)
    mref, keep = _model(model)
    v = lib.vibe_placement_eval(a.ctypes.data_as(C.POINTER(C.c_int32)), ldp, len(ld), G, scp, mref, model_kind,
                                per.ctypes.data_as(C.POINTER(C.c_double)))
    if v < 0:
        raise VibeError("vibe_placement_eval: " + lib.vibe_last_error().decode())
    return float(v), per


def placement_greedy(load_, G: int, scale, model: Optional[LatencyModel], cap: int = 0):
    lib = load()
    ld, ldp = _dp(load_)
    sc, scp = _dp(scale)
    out = np.empty(len(ld), dtype=np.int32)
    mref, keep = _model(model)
    _ok(lib.vibe_placement_greedy(ldp, len(ld), G, scp, mref, cap, out.ctypes.data_as(C.POINTER(C.c_int32))),
        "vibe_placement_greedy")
    return out


def placement_token_balanced(load_, G: int, cap: int = 0):
    lib = load()
    ld, ldp = _dp(load_)
    out = np.empty(len(ld), dtype=np.int32)
    _ok(lib.vibe_placement_token_balanced(ldp, len(ld), G, cap, out.ctypes.data_as(C.POINTER(C.c_int32))),
        "vibe_placement_token_balanced")
    return out


def placement_contiguous(E: int, G: int):
    lib = load()
    out = np.empty(E, dtype=np.int32)
    _ok(lib.vibe_placement_contiguous(E, G, out.ctypes.data_as(C.POINTER(C.c_int32))), "vibe_placement_contiguous")
    return out


# ------------------------------------------------------------------------------------ f1: recalibration (host)
def drift_cosine(w, w_ref) -> float:
    lib = load()
    a, ap = _dp(w)
    b, bp = _dp(w_ref)
    if len(a) != len(b):
        raise VibeError("drift_cosine: length mismatch")
    v = lib.vibe_drift_cosine(ap, bp, len(a))
    if v < -0.5:
        raise VibeError("vibe_drift_cosine: " + lib.vibe_last_error().decode())
    return float(v)


class DriftMonitor:
    """Handle on a library-owned vibe_drift_monitor (Alg. 1 phase 3)."""

    def __init__(self, L: int, E: int, window: int = 100, H: int = 10, delta: float = 0.05):
        self._lib = load()
        self.L, self.E = L, E
        self._h = self._lib.vibe_drift_monitor_create(L, E, window, H, delta)
        if not self._h:
            raise VibeError("vibe_drift_monitor_create: " + self._lib.vibe_last_error().decode())

    def close(self):
        if self._h:
            self._lib.vibe_drift_monitor_destroy(self._h)
            self._h = None

    __del__ = close

    def set_reference(self, W):
        a, ap = _dp(np.asarray(W, dtype=np.float64).reshape(self.L * self.E))
        _ok(self._lib.vibe_drift_monitor_set_reference(self._h, ap), "vibe_drift_monitor_set_reference")

    def push(self, loads):
        """-> (triggered, d[L] or None when no check ran on this pass)"""
        a, ap = _dp(np.asarray(loads, dtype=np.float64).reshape(self.L * self.E))
        d = np.zeros(self.L, dtype=np.float64)
        chk = C.c_int32(0)
        r = self._lib.vibe_drift_monitor_push(self._h, ap, d.ctypes.data_as(C.POINTER(C.c_double)), C.byref(chk))
        if r < 0:
            raise VibeError("vibe_drift_monitor_push: " + self._lib.vibe_last_error().decode())
        return bool(r), (d if chk.value else None)

    def rearranged(self):
        _ok(self._lib.vibe_drift_monitor_rearranged(self._h), "vibe_drift_monitor_rearranged")

    def window_mean(self):
        W = np.zeros(self.L * self.E, dtype=np.float64)
        _ok(self._lib.vibe_drift_monitor_window_mean(self._h, W.ctypes.data_as(C.POINTER(C.c_double))),
            "vibe_drift_monitor_window_mean")
        return W.reshape(self.L, self.E)


def placement_swap_refine(assign, load_, G: int, scale, model: Optional[LatencyModel], model_kind: int = MODEL_B,
                          eps: float = 0.03, max_swaps: int = 1 << 20):
    """Algorithm 2 on one layer -> (assign', [(e_i, e_j), ...])"""
    lib = load()
    a = np.array(assign, dtype=np.int32)
    ld, ldp = _dp(load_)
    sc, scp = _dp(scale)
    mref, keep = _model(model)
    cap = int(min(max_swaps, 1 << 20))
    n = C.c_int32(0)
    sw = np.zeros(2 * max(cap, 1), dtype=np.int32)
    _ok(lib.vibe_placement_swap_refine(a.ctypes.data_as(C.POINTER(C.c_int32)), ldp, len(ld), G, scp, mref, model_kind,
                                       eps, cap, C.byref(n), sw.ctypes.data_as(C.POINTER(C.c_int32))),
        "vibe_placement_swap_refine")
    return a, [(int(sw[2 * i]), int(sw[2 * i + 1])) for i in range(n.value)]
