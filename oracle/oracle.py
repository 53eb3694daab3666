"""ctypes wrapper of the fp64 CPU oracle (oracle/eldr_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It imports nothing from the CUDA package.
All arithmetic lives in the C file; this module only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "eldr_oracle.c")
_LIB = os.path.join(_HERE, "libeldr_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (fp64, -O2, OpenMP over tokens).  No -ffast-math."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c11",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


class OracleShape(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("hidden", "inter", "n_experts", "top_k", "n_shared",
                                         "renormalize", "n_layers", "kv_block_size")]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_num_threads.restype = C.c_int
    return _lib


def _shape(s) -> OracleShape:
    return OracleShape(s.hidden, s.inter, s.n_experts, s.top_k, s.n_shared, s.renormalize,
                       s.n_layers, s.kv_block_size)


def _p(a: Optional[np.ndarray], dtype=None):
    if a is None:
        return None
    if dtype is not None:
        assert a.dtype == dtype, (a.dtype, dtype)
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.c_void_p)


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_threads(n: int) -> None:
    lib().oracle_set_threads(C.c_int(n))


def gate_topk(shape, x_bf16, gate_w, gate_bias=None):
    """-> dict(z[T,E] f64, ids[T,k] i32, w[T,k] f64, margin[T] f64)."""
    T = x_bf16.shape[0]
    E, k = shape.n_experts, shape.top_k
    z = np.empty((T, E), np.float64)
    ids = np.empty((T, k), np.int32)
    w = np.empty((T, k), np.float64)
    margin = np.empty((T,), np.float64)
    s = _shape(shape)
    rc = lib().oracle_gate_topk(C.byref(s), C.c_int32(T), _p(x_bf16, np.uint16),
                                _p(gate_w, np.float32), _p(gate_bias, np.float32),
                                _p(z), _p(ids), _p(w), _p(margin))
    assert rc == 0, rc
    return dict(z=z, ids=ids, w=w, margin=margin)


def expert_ffn(shape, x_row, w13_e, w2_e):
    h = np.empty((shape.inter,), np.float64)
    y = np.empty((shape.hidden,), np.float64)
    s = _shape(shape)
    lib().oracle_expert_ffn(C.byref(s), _p(x_row, np.uint16), _p(w13_e, np.uint16),
                            _p(w2_e, np.uint16), _p(h), _p(y))
    return h, y


def moe_decode_layer(shape, x_bf16, gate_w, gate_bias, w13, w2, shared_w13=None, shared_w2=None,
                     force_ids=None, force_w=None, dump_pairs: bool = False):
    """-> dict(out[T,H], ids, w, margin, cnt[E], active[E], n_active, bytes_loaded, h_pairs?, y_pairs?)."""
    T = x_bf16.shape[0]
    H, I, E, k = shape.hidden, shape.inter, shape.n_experts, shape.top_k
    out = np.empty((T, H), np.float64)
    ids = np.empty((T, k), np.int32)
    w = np.empty((T, k), np.float64)
    margin = np.empty((T,), np.float64)
    cnt = np.empty((E,), np.int32)
    active = np.empty((E,), np.int32)
    n_active = C.c_int32(0)
    nbytes = C.c_int64(0)
    h_pairs = np.empty((T * k, I), np.float64) if dump_pairs else None
    y_pairs = np.empty((T * k, H), np.float64) if dump_pairs else None
    if force_ids is not None:
        force_ids = np.ascontiguousarray(force_ids, np.int32)
        force_w = np.ascontiguousarray(force_w, np.float64)
    s = _shape(shape)
    rc = lib().oracle_moe_decode_layer(
        C.byref(s), C.c_int32(T), _p(x_bf16, np.uint16), _p(gate_w, np.float32),
        _p(gate_bias, np.float32), _p(w13, np.uint16), _p(w2, np.uint16),
        _p(shared_w13, np.uint16), _p(shared_w2, np.uint16), _p(force_ids), _p(force_w),
        _p(out), _p(ids), _p(w), _p(margin), _p(h_pairs), _p(y_pairs), _p(cnt), _p(active),
        C.byref(n_active), C.byref(nbytes))
    assert rc == 0, rc
    r = dict(out=out, ids=ids, w=w, margin=margin, cnt=cnt, active=active,
             n_active=int(n_active.value), bytes_loaded=int(nbytes.value))
    if dump_pairs:
        r["h_pairs"] = h_pairs
        r["y_pairs"] = y_pairs
    return r


def permutation(shape, ids):
    T = ids.shape[0]
    E, k = shape.n_experts, shape.top_k
    cnt = np.empty((E,), np.int32)
    off = np.empty((E + 1,), np.int32)
    perm = np.empty((T * k,), np.int32)
    active = np.empty((E,), np.int32)
    n_active = C.c_int32(0)
    s = _shape(shape)
    rc = lib().oracle_permutation(C.byref(s), C.c_int32(T), _p(np.ascontiguousarray(ids), np.int32),
                                  _p(cnt), _p(off), _p(perm), _p(active), C.byref(n_active))
    assert rc == 0, rc
    return dict(cnt=cnt, off=off, perm=perm, active=active, n_active=int(n_active.value))


def signature_accumulate(shape, layer, ids, token_req, token_block, sig_req, sig_block):
    """In-place on sig_req [R,L,E] int32 and sig_block [NB,L,E] int8 (either may be None)."""
    T = ids.shape[0]
    s = _shape(shape)
    rc = lib().oracle_signature_accumulate(
        C.byref(s), C.c_int32(layer), C.c_int32(T), _p(np.ascontiguousarray(ids), np.int32),
        _p(token_req, np.int32), _p(token_block, np.int32), _p(sig_req, np.int32),
        _p(sig_block, np.int8))
    assert rc == 0, rc


def signature_reset_blocks(shape, block_ids, sig_block):
    s = _shape(shape)
    block_ids = np.ascontiguousarray(block_ids, np.int32)
    lib().oracle_signature_reset_blocks(C.byref(s), _p(block_ids), C.c_int32(len(block_ids)),
                                        _p(sig_block, np.int8))


def signature_readout(shape, block_ids, sig_block):
    s = _shape(shape)
    block_ids = np.ascontiguousarray(block_ids, np.int32)
    out = np.empty((shape.n_layers, shape.n_experts), np.int32)
    lib().oracle_signature_readout(C.byref(s), _p(block_ids), C.c_int32(len(block_ids)),
                                   _p(sig_block, np.int8), _p(out))
    return out


# ---------------------------------------------------------------- routing decision
def idf_table(df: np.ndarray, n_calib: int) -> np.ndarray:
    """w(l,e) = log((|C|+1)/(df(l,e)+1)).  df int32 [L,E] -> float64 [L,E]."""
    df = np.ascontiguousarray(df, dtype=np.int32)
    w = np.empty(df.shape, dtype=np.float64)
    lib().oracle_idf_table(C.c_int32(df.size), _p(df), C.c_int32(n_calib), _p(w))
    return w


def route_decide(counts: np.ndarray, idf: np.ndarray, layer_mask: np.ndarray, centroids: np.ndarray,
                 loads: np.ndarray, tau: float):
    """Locality-band routing of R requests in index order.  counts int32 [R,L,E];
    idf float64 [L,E]; layer_mask uint8 [L]; centroids float64 [K,L,E]; loads int64 [K] (updated IN PLACE).
    Returns dict(worker [R] int32, sims [R,K] float64, band_gap [R] float64 = distance of the nearest similarity
    to the band edge s* - tau, for near-tie reporting)."""
    R, L, E = counts.shape
    K = centroids.shape[0]
    assert counts.dtype == np.int32 and idf.dtype == np.float64 and centroids.dtype == np.float64
    assert layer_mask.dtype == np.uint8 and loads.dtype == np.int64
    worker = np.empty((R,), np.int32)
    sims = np.empty((R, K), np.float64)
    gap = np.empty((R,), np.float64)
    rc = lib().oracle_route_decide(C.c_int32(R), C.c_int32(L), C.c_int32(E), C.c_int32(K), _p(counts), _p(idf),
                                   _p(layer_mask), _p(centroids), _p(loads), C.c_double(tau), _p(worker),
                                   _p(sims), _p(gap))
    assert rc == 0, rc
    return dict(worker=worker, sims=sims, band_gap=gap)
