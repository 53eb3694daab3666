"""Thin Python binding of the C ABI in include/eldr_moe.h (argument marshalling only).

Same names as the C entry points.  Every step of the path runs in the CUDA library
(csrc/libeldr_moe.so); there is no CPU or PyTorch fallback: if the library is missing or a call
fails, a RuntimeError is raised.  PyTorch is used for device memory and streams only.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np
import torch

from . import build as _build

_lib = None

EXPORTS = [
    "eldr_moe_gate_topk", "eldr_moe_gate_topk_static", "eldr_moe_decode_layer", "eldr_moe_decode_layer_host", "eldr_moe_decode_layer_mxfp4",
    "eldr_signature_accumulate", "eldr_signature_accumulate_layers", "eldr_signature_reset_blocks", "eldr_signature_readout", "eldr_route_decide",
    "eldr_moe_workspace_bytes", "eldr_moe_workspace_bytes_host", "eldr_moe_workspace_layout",
    "eldr_moe_last_launch_count", "eldr_status_string", "eldr_last_cuda_error",
    "eldr_moe_profile_enable", "eldr_moe_profile_read", "eldr_moe_set_option",
    "eldr_fit_idf", "eldr_fit_layer_mask", "eldr_fit_balanced_assign", "eldr_fit_kmeans_balanced",
]
OPT_FFN_PATH, FFN_MMA_SYNC, FFN_TCGEN05, FFN_GEMV = 0, 0, 1, 2
OPT_PDL = 1
OPT_STEP_PATH, STEP_STAGED, STEP_FUSED, STEP_AUTO = 2, 0, 1, 2
OPT_RING_KB = 3
OPT_DP_MIN_ROUNDS = 4
OPT_FFN_PAIR = 5
OPT_SK_SPLIT_PCT = 6
OPT_COOPERATIVE = 7
OPT_HEAD_FIRST = 8
OPT_XS_MIN_NP = 9
OPT_SK_MAX_SPLIT = 10
OPT_GATE_TC = 11
PROFILE_SLOTS = ("gate", "route", "gather", "ffn13", "ffn2", "combine")


class Shape(C.Structure):
    """eldr_moe_shape_t"""
    _fields_ = [(n, C.c_int32) for n in ("hidden", "inter", "n_experts", "top_k", "n_shared",
                                         "renormalize", "n_layers", "kv_block_size")]


class WsLayout(C.Structure):
    """eldr_moe_ws_layout_t"""
    _fields_ = [(n, C.c_size_t) for n in ("z", "cnt", "off", "perm", "pair_pos", "work", "n_work", "sync",
                                          "x_perm", "h", "y", "partial", "total")]


def lib_path() -> str:
    return _build.LIB


def load(build_if_missing: bool = False, path: Optional[str] = None):
    """dlopen the CUDA library.  Raises if it is not built (no fallback).  `path`: another build of the same library
    (the -DELDR_TRACE one of `bench.py --timeline`); must be given on the first load of the process."""
    global _lib
    if _lib is not None:
        return _lib
    path = path or _build.LIB
    if not os.path.exists(path):
        if build_if_missing:
            _build.build()
        else:
            raise RuntimeError("CUDA library %s is not built; run `python -c 'import __graft_entry__ as g; "
                               "g.build()'` (there is no CPU fallback)" % path)
    lib = C.CDLL(path)
    lib.eldr_moe_workspace_bytes.restype = C.c_size_t
    lib.eldr_moe_workspace_bytes_host.restype = C.c_size_t
    lib.eldr_status_string.restype = C.c_char_p
    lib.eldr_last_cuda_error.restype = C.c_char_p
    for n in EXPORTS:
        getattr(lib, n)          # fail loudly if a declared symbol is missing
    _lib = lib
    return lib


def make_shape(s) -> Shape:
    return Shape(s.hidden, s.inter, s.n_experts, s.top_k, s.n_shared, s.renormalize, s.n_layers,
                 s.kv_block_size)


def _check(rc: int, what: str):
    if rc != 0:
        lib = load()
        raise RuntimeError("%s failed: %s (%d) %s" % (what, lib.eldr_status_string(rc).decode(), rc,
                                                       lib.eldr_last_cuda_error().decode()))


def _ptr(t: Optional[torch.Tensor], dtype=None, cuda: bool = True):
    if t is None:
        return C.c_void_p(0)
    assert t.is_contiguous()
    if dtype is not None:
        assert t.dtype == dtype, (t.dtype, dtype)
    assert t.is_cuda == cuda, "tensor on the wrong side of the PCIe bus"
    return C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def bf16_from_bits(bits: np.ndarray, device="cuda") -> torch.Tensor:
    """uint16 bf16 bit patterns (synth.py) -> torch.bfloat16 tensor (same bits)."""
    t = torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16)
    return t.to(device) if device is not None else t


def bits_from_bf16(t: torch.Tensor) -> np.ndarray:
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16)


def eldr_moe_workspace_bytes(shape, max_T: int) -> int:
    s = make_shape(shape)
    return int(load().eldr_moe_workspace_bytes(C.byref(s), C.c_int32(max_T)))


def eldr_moe_workspace_bytes_host(shape, max_T: int) -> int:
    s = make_shape(shape)
    return int(load().eldr_moe_workspace_bytes_host(C.byref(s), C.c_int32(max_T)))


def eldr_moe_workspace_layout(shape, T: int) -> WsLayout:
    s = make_shape(shape)
    L = WsLayout()
    _check(load().eldr_moe_workspace_layout(C.byref(s), C.c_int32(T), C.byref(L)), "eldr_moe_workspace_layout")
    return L


def eldr_moe_last_launch_count() -> int:
    return int(load().eldr_moe_last_launch_count())


def eldr_moe_set_option(key: int, value: int) -> None:
    _check(load().eldr_moe_set_option(C.c_int32(key), C.c_int32(value)), "eldr_moe_set_option")


def eldr_moe_profile_enable(on: bool) -> None:
    _check(load().eldr_moe_profile_enable(C.c_int32(1 if on else 0)), "eldr_moe_profile_enable")


def eldr_moe_profile_read() -> dict:
    """Per-kernel milliseconds of the last eldr_moe_decode_layer call (waits for it)."""
    ms = (C.c_float * len(PROFILE_SLOTS))()
    _check(load().eldr_moe_profile_read(ms), "eldr_moe_profile_read")
    return dict(zip(PROFILE_SLOTS, [float(v) for v in ms]))


def eldr_moe_gate_topk(shape, layer: int, x, gate_w, gate_bias, topk_ids, topk_w, token_req=None,
                       token_block=None, sig_req=None, sig_block=None, workspace=None):
    s = make_shape(shape)
    T = x.shape[0]
    _check(load().eldr_moe_gate_topk(
        C.byref(s), C.c_int32(layer), C.c_int32(T), _ptr(x, torch.bfloat16), _ptr(gate_w, torch.float32),
        _ptr(gate_bias, torch.float32), _ptr(topk_ids, torch.int32), _ptr(topk_w, torch.float32),
        _ptr(token_req, torch.int32), _ptr(token_block, torch.int32), _ptr(sig_req, torch.int32),
        _ptr(sig_block, torch.int8), _ptr(workspace), C.c_size_t(workspace.numel() * workspace.element_size()),
        _stream()), "eldr_moe_gate_topk")


STATIC_SCRATCH_BYTES = 1 << 20


def eldr_moe_gate_topk_static(shape, layer: int, x, gate_w, gate_bias, topk_ids, topk_w, token_req=None,
                              token_block=None, sig_req=None, sig_block=None):
    """eldr_moe_gate_topk without a workspace: the logits scratch is a static array inside the library (no allocation)."""
    s = make_shape(shape)
    T = x.shape[0]
    _check(load().eldr_moe_gate_topk_static(
        C.byref(s), C.c_int32(layer), C.c_int32(T), _ptr(x, torch.bfloat16), _ptr(gate_w, torch.float32),
        _ptr(gate_bias, torch.float32), _ptr(topk_ids, torch.int32), _ptr(topk_w, torch.float32),
        _ptr(token_req, torch.int32), _ptr(token_block, torch.int32), _ptr(sig_req, torch.int32),
        _ptr(sig_block, torch.int8), _stream()), "eldr_moe_gate_topk_static")


def eldr_moe_decode_layer(shape, layer: int, x, gate_w, gate_bias, w13, w2, shared_w13, shared_w2, out,
                          topk_ids, topk_w, force_routing: int, active_experts, n_active,
                          token_req=None, token_block=None, sig_req=None, sig_block=None, workspace=None):
    s = make_shape(shape)
    T = x.shape[0]
    _check(load().eldr_moe_decode_layer(
        C.byref(s), C.c_int32(layer), C.c_int32(T), _ptr(x, torch.bfloat16), _ptr(gate_w, torch.float32),
        _ptr(gate_bias, torch.float32), _ptr(w13, torch.bfloat16), _ptr(w2, torch.bfloat16),
        _ptr(shared_w13, torch.bfloat16), _ptr(shared_w2, torch.bfloat16), _ptr(out, torch.bfloat16),
        _ptr(topk_ids, torch.int32), _ptr(topk_w, torch.float32), C.c_int32(force_routing),
        _ptr(active_experts, torch.int32), _ptr(n_active, torch.int32),
        _ptr(token_req, torch.int32), _ptr(token_block, torch.int32), _ptr(sig_req, torch.int32),
        _ptr(sig_block, torch.int8), _ptr(workspace), C.c_size_t(workspace.numel() * workspace.element_size()),
        _stream()), "eldr_moe_decode_layer")


def eldr_moe_decode_layer_mxfp4(shape, layer: int, x, gate_w, gate_bias, w13_codes, w13_scales, w2_codes, w2_scales, out,
                                topk_ids, topk_w, force_routing: int, active_experts, n_active,
                                token_req=None, token_block=None, sig_req=None, sig_block=None, workspace=None):
    s = make_shape(shape)
    T = x.shape[0]
    _check(load().eldr_moe_decode_layer_mxfp4(
        C.byref(s), C.c_int32(layer), C.c_int32(T), _ptr(x, torch.bfloat16), _ptr(gate_w, torch.float32),
        _ptr(gate_bias, torch.float32), _ptr(w13_codes, torch.uint8), _ptr(w13_scales, torch.uint8),
        _ptr(w2_codes, torch.uint8), _ptr(w2_scales, torch.uint8), _ptr(out, torch.bfloat16),
        _ptr(topk_ids, torch.int32), _ptr(topk_w, torch.float32), C.c_int32(force_routing),
        _ptr(active_experts, torch.int32), _ptr(n_active, torch.int32),
        _ptr(token_req, torch.int32), _ptr(token_block, torch.int32), _ptr(sig_req, torch.int32),
        _ptr(sig_block, torch.int8), _ptr(workspace), C.c_size_t(workspace.numel() * workspace.element_size()),
        _stream()), "eldr_moe_decode_layer_mxfp4")


def eldr_moe_decode_layer_host(shape, layer: int, h_x, gate_w, gate_bias, w13, w2, shared_w13, shared_w2,
                               h_out, h_topk_ids, h_topk_w, h_n_active, h_token_req=None, h_token_block=None,
                               sig_req=None, sig_block=None, workspace=None):
    """h_* are HOST (pinned) tensors; everything else lives on the device.  Synchronous."""
    s = make_shape(shape)
    T = h_x.shape[0]
    _check(load().eldr_moe_decode_layer_host(
        C.byref(s), C.c_int32(layer), C.c_int32(T), _ptr(h_x, torch.bfloat16, cuda=False),
        _ptr(gate_w, torch.float32), _ptr(gate_bias, torch.float32), _ptr(w13, torch.bfloat16),
        _ptr(w2, torch.bfloat16), _ptr(shared_w13, torch.bfloat16), _ptr(shared_w2, torch.bfloat16),
        _ptr(h_out, torch.bfloat16, cuda=False), _ptr(h_topk_ids, torch.int32, cuda=False),
        _ptr(h_topk_w, torch.float32, cuda=False), _ptr(h_n_active, torch.int32, cuda=False),
        _ptr(h_token_req, torch.int32, cuda=False), _ptr(h_token_block, torch.int32, cuda=False),
        _ptr(sig_req, torch.int32), _ptr(sig_block, torch.int8), _ptr(workspace),
        C.c_size_t(workspace.numel() * workspace.element_size()), _stream()), "eldr_moe_decode_layer_host")


def eldr_signature_accumulate(shape, layer: int, topk_ids, token_req, token_block, sig_req, sig_block):
    s = make_shape(shape)
    T = topk_ids.shape[0]
    _check(load().eldr_signature_accumulate(
        C.byref(s), C.c_int32(layer), C.c_int32(T), _ptr(topk_ids, torch.int32), _ptr(token_req, torch.int32),
        _ptr(token_block, torch.int32), _ptr(sig_req, torch.int32), _ptr(sig_block, torch.int8), _stream()),
        "eldr_signature_accumulate")


def eldr_signature_accumulate_layers(shape, topk_ids, token_req, token_block, sig_req, sig_block, layer0: int = 0):
    """topk_ids [n_layers, T, k]: all layers of a prefill-shaped capture in one launch."""
    s = make_shape(shape)
    n_layers, T = topk_ids.shape[0], topk_ids.shape[1]
    _check(load().eldr_signature_accumulate_layers(
        C.byref(s), C.c_int32(layer0), C.c_int32(n_layers), C.c_int32(T), _ptr(topk_ids, torch.int32),
        _ptr(token_req, torch.int32), _ptr(token_block, torch.int32), _ptr(sig_req, torch.int32),
        _ptr(sig_block, torch.int8), _stream()), "eldr_signature_accumulate_layers")


def eldr_signature_reset_blocks(shape, block_ids, sig_block):
    s = make_shape(shape)
    _check(load().eldr_signature_reset_blocks(C.byref(s), _ptr(block_ids, torch.int32),
                                              C.c_int32(block_ids.numel()), _ptr(sig_block, torch.int8),
                                              _stream()), "eldr_signature_reset_blocks")


def eldr_signature_readout(shape, block_ids, req_off, sig_block, sig_out):
    s = make_shape(shape)
    _check(load().eldr_signature_readout(C.byref(s), _ptr(block_ids, torch.int32), _ptr(req_off, torch.int32),
                                         C.c_int32(req_off.numel() - 1), _ptr(sig_block, torch.int8),
                                         _ptr(sig_out, torch.int32), _stream()), "eldr_signature_readout")


def eldr_route_decide(shape, sig_req, idf, layer_mask, centroids, loads, tau: float, worker, sims):
    s = make_shape(shape)
    R, K = sig_req.shape[0], centroids.shape[0]
    _check(load().eldr_route_decide(C.byref(s), C.c_int32(R), C.c_int32(K), _ptr(sig_req, torch.int32),
                                    _ptr(idf, torch.float32), _ptr(layer_mask, torch.uint8),
                                    _ptr(centroids, torch.float32), _ptr(loads, torch.int32), C.c_float(tau),
                                    _ptr(worker, torch.int32), _ptr(sims, torch.float32), _stream()),
           "eldr_route_decide")


class DecodeLayer:
    """Convenience holder of one layer's device tensors + workspace (plumbing; no arithmetic)."""

    def __init__(self, shape, lw, max_T: int, device="cuda"):
        self.shape = shape
        self.gate_w = torch.from_numpy(lw.gate_w).to(device)
        self.w13 = bf16_from_bits(lw.w13, device)
        self.w2 = bf16_from_bits(lw.w2, device)
        self.shared_w13 = bf16_from_bits(lw.shared_w13, device) if lw.shared_w13 is not None else None
        self.shared_w2 = bf16_from_bits(lw.shared_w2, device) if lw.shared_w2 is not None else None
        self.max_T = max_T
        self.workspace = torch.zeros(eldr_moe_workspace_bytes_host(shape, max_T), dtype=torch.uint8, device=device)   # zeroed once (include/eldr_moe.h: recommended)
        E, k, H = shape.n_experts, shape.top_k, shape.hidden
        self.out = torch.empty((max_T, H), dtype=torch.bfloat16, device=device)
        self.ids = torch.empty((max_T, k), dtype=torch.int32, device=device)
        self.w = torch.empty((max_T, k), dtype=torch.float32, device=device)
        self.active = torch.empty((E,), dtype=torch.int32, device=device)
        self.n_active = torch.zeros((1,), dtype=torch.int32, device=device)

    def run(self, x, gate_bias=None, layer=0, force_routing=0, token_req=None, token_block=None,
            sig_req=None, sig_block=None):
        T = x.shape[0]
        eldr_moe_decode_layer(self.shape, layer, x, self.gate_w, gate_bias, self.w13, self.w2,
                              self.shared_w13, self.shared_w2, self.out[:T], self.ids[:T], self.w[:T],
                              force_routing, self.active, self.n_active, token_req, token_block,
                              sig_req, sig_block, self.workspace)
        return self.out[:T]

    def ws_view(self, name: str, T: int):
        """Typed view of one workspace intermediate (for per-kernel parity tests)."""
        L = eldr_moe_workspace_layout(self.shape, T)
        s = self.shape
        k, E, H, I, ns = s.top_k, s.n_experts, s.hidden, s.inter, s.n_shared
        spec = {"z": (torch.float32, (T, E)), "cnt": (torch.int32, (E,)), "off": (torch.int32, (E + 1,)),
                "perm": (torch.int32, (T * k,)), "pair_pos": (torch.int32, (T * k,)),
                "work": (torch.int32, (E + ns, 4)), "n_work": (torch.int32, (1,)),
                "x_perm": (torch.bfloat16, (T * k + T, H)), "h": (torch.bfloat16, (T * (k + ns), I)),
                "y": (torch.float32, (T * (k + ns), H))}[name]
        off = getattr(L, name)
        n = int(np.prod(spec[1])) * torch.empty((), dtype=spec[0]).element_size()
        return self.workspace[off: off + n].view(spec[0]).view(spec[1])


# ---- offline fit (host functions of the library: numpy arrays in, numpy arrays out; marshalling only) ----------------
def _np(a, dtype):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a, a.ctypes.data_as(C.c_void_p)


def eldr_fit_idf(counts: np.ndarray) -> np.ndarray:
    counts, pc = _np(counts, np.int32)
    N, L, E = counts.shape
    idf = np.empty((L, E), np.float64)
    _check(load().eldr_fit_idf(pc, C.c_int32(N), C.c_int32(L), C.c_int32(E), idf.ctypes.data_as(C.c_void_p)), "eldr_fit_idf")
    return idf


def eldr_fit_layer_mask(counts, idf, decode_p, pairs):
    counts, pc = _np(counts, np.int32)
    idf, pi = _np(idf, np.float64)
    decode_p, pd = _np(decode_p, np.float64)
    pairs, pp = _np(pairs, np.int32)
    N, L, E = counts.shape
    order, cum = np.empty(L, np.int32), np.empty(L, np.float64)
    n_star, mask = np.zeros(1, np.int32), np.empty(L, np.uint8)
    _check(load().eldr_fit_layer_mask(pc, pi, pd, C.c_int32(N), C.c_int32(L), C.c_int32(E), pp, C.c_int32(len(pairs)),
                                      order.ctypes.data_as(C.c_void_p), cum.ctypes.data_as(C.c_void_p),
                                      n_star.ctypes.data_as(C.c_void_p), mask.ctypes.data_as(C.c_void_p)), "eldr_fit_layer_mask")
    return order, cum, int(n_star[0]), mask


def eldr_fit_balanced_assign(cost, cap: int):
    cost, pc = _np(cost, np.float64)
    N, K = cost.shape
    assign, total = np.empty(N, np.int32), np.zeros(1, np.float64)
    _check(load().eldr_fit_balanced_assign(pc, C.c_int32(N), C.c_int32(K), C.c_int32(cap), assign.ctypes.data_as(C.c_void_p),
                                           total.ctypes.data_as(C.c_void_p)), "eldr_fit_balanced_assign")
    return assign, float(total[0])


def eldr_fit_kmeans_balanced(sig, K: int, init_idx, max_iter: int = 50):
    sig, ps = _np(sig, np.float64)
    init_idx, pi = _np(init_idx, np.int32)
    N, d = sig.shape
    cent, assign = np.empty((K, d), np.float64), np.empty(N, np.int32)
    steps, total = np.zeros(1, np.int32), np.zeros(1, np.float64)
    _check(load().eldr_fit_kmeans_balanced(ps, C.c_int32(N), C.c_int32(d), C.c_int32(K), pi, C.c_int32(max_iter),
                                           cent.ctypes.data_as(C.c_void_p), assign.ctypes.data_as(C.c_void_p),
                                           steps.ctypes.data_as(C.c_void_p), total.ctypes.data_as(C.c_void_p)), "eldr_fit_kmeans_balanced")
    return cent, assign, int(steps[0]), float(total[0])


class MxDecodeLayer:
    """Holder of one MXFP4 layer's device tensors + workspace (plumbing; no arithmetic).  `w13` / `w2` are
    (codes uint8 [E,rows,K/2], scales uint8 [E,rows,K/32]) numpy pairs."""

    def __init__(self, shape, gate_w, w13, w2, max_T: int, device="cuda"):
        self.shape = shape
        self.gate_w = torch.from_numpy(gate_w).to(device)
        self.w13_codes, self.w13_scales = (torch.from_numpy(np.ascontiguousarray(a)).to(device) for a in w13)
        self.w2_codes, self.w2_scales = (torch.from_numpy(np.ascontiguousarray(a)).to(device) for a in w2)
        self.max_T = max_T
        self.workspace = torch.zeros(eldr_moe_workspace_bytes(shape, max_T), dtype=torch.uint8, device=device)
        E, k, H = shape.n_experts, shape.top_k, shape.hidden
        self.out = torch.empty((max_T, H), dtype=torch.bfloat16, device=device)
        self.ids = torch.empty((max_T, k), dtype=torch.int32, device=device)
        self.w = torch.empty((max_T, k), dtype=torch.float32, device=device)
        self.active = torch.empty((E,), dtype=torch.int32, device=device)
        self.n_active = torch.zeros((1,), dtype=torch.int32, device=device)

    def run(self, x, gate_bias=None, layer=0, force_routing=0, token_req=None, token_block=None,
            sig_req=None, sig_block=None):
        T = x.shape[0]
        eldr_moe_decode_layer_mxfp4(self.shape, layer, x, self.gate_w, gate_bias, self.w13_codes, self.w13_scales,
                                    self.w2_codes, self.w2_scales, self.out[:T], self.ids[:T], self.w[:T],
                                    force_routing, self.active, self.n_active, token_req, token_block,
                                    sig_req, sig_block, self.workspace)
        return self.out[:T]

    ws_view = DecodeLayer.ws_view
