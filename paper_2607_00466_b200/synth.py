"""Seeded synthetic inputs for the ELDR decode-MoE hot path.

This module serves BOTH the CUDA path and the CPU oracle with the same bits.  It holds none of
the method's arithmetic (no gate, no softmax, no top-k, no FFN, no histogram): only random
draws, bf16 rounding of the drawn values, and index bookkeeping.  It imports neither the CUDA
binding nor ``oracle/``.

Recipes follow BASELINE.json ``configs`` (the stand-ins for the paper's models and prompts, which
are not available offline) and SURVEY.md section 8(d); DESIGN.md restates them.

bf16 tensors are carried as ``numpy.uint16`` bit patterns (numpy has no bfloat16); the rounding is
round-to-nearest-even on the fp32 bit pattern and happens exactly once, here.
"""
from __future__ import annotations

import dataclasses
import zlib
from typing import Dict, Optional

import numpy as np


# ----------------------------------------------------------------------------------------------
# bf16 <-> fp32 bit helpers (input preparation only)
# ----------------------------------------------------------------------------------------------
def f32_to_bf16_bits(a: np.ndarray) -> np.ndarray:
    """Round fp32 -> bf16 (RNE), returned as uint16 bit patterns.  Inputs must be finite."""
    a = np.ascontiguousarray(a, dtype=np.float32)
    u = a.view(np.uint32)
    bias = ((u >> np.uint32(16)) & np.uint32(1)) + np.uint32(0x7FFF)
    return ((u + bias) >> np.uint32(16)).astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    b = np.ascontiguousarray(b, dtype=np.uint16)
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32)


def sub_seed(seed: int, *names) -> int:
    """Stable 63-bit sub-seed = f(seed, tensor name, layer, ...)."""
    s = ("%d|" % seed) + "|".join(str(n) for n in names)
    return (zlib.crc32(s.encode()) | (zlib.adler32(s.encode()) << 32)) & 0x7FFFFFFFFFFFFFFF


def _normal_bf16(rng: np.random.Generator, shape, std: float, chunk: int = 1 << 24) -> np.ndarray:
    """N(0, std) rounded to bf16 bits; generated in chunks to bound host memory."""
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.uint16)
    for s in range(0, n, chunk):
        e = min(n, s + chunk)
        v = rng.standard_normal(e - s, dtype=np.float32)
        v *= np.float32(std)
        out[s:e] = f32_to_bf16_bits(v)
    return out.reshape(shape)


# ----------------------------------------------------------------------------------------------
# Shapes (BASELINE.json configs; names follow the paper: E experts, top-k, L MoE layers)
# ----------------------------------------------------------------------------------------------
@dataclasses.dataclass(frozen=True)
class MoEShape:
    hidden: int          # H
    inter: int           # I  (SwiGLU intermediate)
    n_experts: int       # E  routed experts
    top_k: int           # k
    n_shared: int = 0    # always-on shared experts
    renormalize: int = 1
    n_layers: int = 1    # L
    kv_block_size: int = 16

    @property
    def expert_bytes(self) -> int:
        """bf16 bytes of one expert's w1,w3,w2: 3*H*I*2 (north_star roofline numerator)."""
        return 3 * self.hidden * self.inter * 2


SHAPE_C1 = MoEShape(hidden=256, inter=128, n_experts=16, top_k=2, n_layers=1, kv_block_size=2)
SHAPE_QWEN = MoEShape(hidden=2048, inter=768, n_experts=128, top_k=8, n_layers=1)
SHAPE_QWEN48 = dataclasses.replace(SHAPE_QWEN, n_layers=48)
SHAPE_C5 = MoEShape(hidden=2048, inter=1408, n_experts=64, top_k=6, n_shared=2, n_layers=27)


@dataclasses.dataclass
class LayerWeights:
    gate_w: np.ndarray                 # [E,H] fp32
    w13: np.ndarray                    # [E,2I,H] bf16 bits; rows 0..I-1 = w1 (SiLU branch), I..2I-1 = w3
    w2: np.ndarray                     # [E,H,I] bf16 bits
    shared_w13: Optional[np.ndarray]   # [n_shared,2I,H] bf16 bits or None
    shared_w2: Optional[np.ndarray]    # [n_shared,H,I] bf16 bits or None


def make_gate_w(shape: "MoEShape", seed: int, layer: int = 0, gate_std: float = 0.05) -> np.ndarray:
    """fp32 gate rows ~N(0,0.05), [E,H]."""
    g = np.random.default_rng(sub_seed(seed, "gate_w", layer))
    return (g.standard_normal((shape.n_experts, shape.hidden), dtype=np.float32)
            * np.float32(gate_std)).astype(np.float32)


def make_layer_weights(shape: MoEShape, seed: int, layer: int = 0,
                       w_std: float = 0.02, gate_std: float = 0.05) -> LayerWeights:
    """bf16 expert weights ~N(0,0.02), fp32 gate ~N(0,0.05) (BASELINE.json configs 1-2)."""
    H, I, E = shape.hidden, shape.inter, shape.n_experts
    gate_w = make_gate_w(shape, seed, layer, gate_std)
    w13 = _normal_bf16(np.random.default_rng(sub_seed(seed, "w13", layer)), (E, 2 * I, H), w_std)
    w2 = _normal_bf16(np.random.default_rng(sub_seed(seed, "w2", layer)), (E, H, I), w_std)
    s13 = s2 = None
    if shape.n_shared:
        s13 = _normal_bf16(np.random.default_rng(sub_seed(seed, "sw13", layer)),
                           (shape.n_shared, 2 * I, H), w_std)
        s2 = _normal_bf16(np.random.default_rng(sub_seed(seed, "sw2", layer)),
                          (shape.n_shared, H, I), w_std)
    return LayerWeights(gate_w, w13, w2, s13, s2)


def make_mxfp4_tensor(rows: int, K: int, seed: int, tag="mx", scale_lo: int = 118, scale_hi: int = 122):
    """Seeded MXFP4-shaped raw bytes for SURVEY.md 8(f) row 3 (GPT-OSS-style experts): packed 4-bit codes
    [rows, K/2] uint8 (uniform over the 16 codes) and one scale byte per 32 elements [rows, K/32] uint8, uniform in
    scale_lo..scale_hi (2^-9..2^-5, so the decoded magnitudes are those of ~N(0,0.02) weights).  The generator draws
    BYTES only -- what they mean is defined by the oracle (oracle/mxfp4.py) and, later, by the kernels."""
    if K % 32:
        raise ValueError("K must be a multiple of 32")
    rng = np.random.default_rng(sub_seed(seed, tag, rows, K))
    packed = rng.integers(0, 256, size=(rows, K // 2), dtype=np.uint8)
    scales = rng.integers(scale_lo, scale_hi + 1, size=(rows, K // 32), dtype=np.uint8)
    return packed, scales


def make_hidden(T: int, H: int, seed: int, tag="x") -> np.ndarray:
    """Decode-token hiddens ~N(0,1) rounded to bf16 bits, [T,H]."""
    return _normal_bf16(np.random.default_rng(sub_seed(seed, tag, T)), (T, H), 1.0)


def union_bias(E: int, u: int, seed: int, boost: float = 40.0) -> np.ndarray:
    """Config 2/3: gate_bias = +boost on a seeded subset S_u of size u, 0 elsewhere.

    The gate logits have std ~ 0.05*sqrt(2048) ~ 2.3, so +40 confines every token's top-k to S_u;
    the common shift cancels in the renormalised weights.
    """
    perm = np.random.default_rng(sub_seed(seed, "subset", u)).permutation(E)
    b = np.zeros(E, dtype=np.float32)
    b[perm[:u]] = np.float32(boost)
    return b


# Decode-shaped request/block maps: one token per request, each in its own KV block.
def decode_maps(T: int, block_base: int = 0):
    token_req = np.arange(T, dtype=np.int32)
    token_block = (np.arange(T, dtype=np.int32) + block_base).astype(np.int32)
    return token_req, token_block


def c1_maps():
    """Config 1: 2 requests x 4 tokens, kv_block_size=2 so each request spans 2 blocks."""
    token_req = np.array([0, 0, 0, 0, 1, 1, 1, 1], dtype=np.int32)
    token_block = np.array([0, 0, 1, 1, 2, 2, 3, 3], dtype=np.int32)
    return token_req, token_block


# ----------------------------------------------------------------------------------------------
# Config 4: clustered hiddens + cluster-aligned gate rows
# ----------------------------------------------------------------------------------------------
def c4_centroids(H: int, seed: int, n_clusters: int = 8) -> np.ndarray:
    return np.random.default_rng(sub_seed(seed, "centroids")).standard_normal((n_clusters, H)).astype(np.float32)


def c4_hidden(T: int, centroids: np.ndarray, cluster_of_token: np.ndarray, seed: int,
              sigma: float = 0.3) -> np.ndarray:
    """x_t = mu_{c(t)} + sigma*N(0,1), rounded to bf16 bits."""
    rng = np.random.default_rng(sub_seed(seed, "c4x", T))
    x = centroids[cluster_of_token] + np.float32(sigma) * rng.standard_normal(
        (T, centroids.shape[1]), dtype=np.float32)
    return f32_to_bf16_bits(x)


def c4_gate(shape: MoEShape, centroids: np.ndarray, seed: int, layer: int, alpha: float = 0.2,
            gate_std: float = 0.05) -> np.ndarray:
    """Wg[e] = N(0,0.05) + alpha * mu_{home(e)}/||mu||, home = seeded expert->cluster map."""
    E, H = shape.n_experts, shape.hidden
    rng = np.random.default_rng(sub_seed(seed, "c4gate", layer))
    gw = rng.standard_normal((E, H), dtype=np.float32) * np.float32(gate_std)
    nC = centroids.shape[0]
    home = rng.permutation(E) % nC
    unit = centroids / np.linalg.norm(centroids, axis=1, keepdims=True)
    return (gw + np.float32(alpha) * unit[home]).astype(np.float32)


def c4_cluster_assignment(T: int, mode: str, step: int, seed: int, n_clusters: int = 8) -> np.ndarray:
    if mode == "single":
        return np.full(T, step % n_clusters, dtype=np.int64)
    rng = np.random.default_rng(sub_seed(seed, "c4mix", step))
    return rng.integers(0, n_clusters, size=T)


# ----------------------------------------------------------------------------------------------
# Config 5: prefill-shaped signature workload (32 requests, block 16, prompts 512..4096)
# ----------------------------------------------------------------------------------------------
@dataclasses.dataclass
class SignatureWorkload:
    topk_ids: np.ndarray      # [T,k] int32, k distinct experts per token
    token_req: np.ndarray     # [T] int32 (request that FIRST prefilled the token; -1 = padding)
    token_block: np.ndarray   # [T] int32 KV block id (non-contiguous, seeded permutation)
    n_requests: int
    n_blocks: int
    req_blocks: Dict[int, np.ndarray]   # request -> its block set B(r) (shared prefix blocks included)
    req_len: np.ndarray                  # [R] prompt lengths
    cold_ids: Dict[int, np.ndarray]      # request -> [len_r,k] ids a cold prefill of r would produce


def zipf_topk_ids(rng: np.random.Generator, n_tokens: int, E: int, k: int, a: float = 1.1) -> np.ndarray:
    """k distinct experts per token from a skewed (Zipf-like) popularity, via Gumbel top-k."""
    p = 1.0 / np.arange(1, E + 1, dtype=np.float64) ** a
    p = p[rng.permutation(E)]
    logp = np.log(p / p.sum())
    ids = np.empty((n_tokens, k), dtype=np.int32)
    chunk = 1 << 15
    for s in range(0, n_tokens, chunk):
        e = min(n_tokens, s + chunk)
        gum = rng.gumbel(size=(e - s, E)) + logp
        ids[s:e] = np.argpartition(-gum, k - 1, axis=1)[:, :k].astype(np.int32)
    return ids


def make_signature_workload(E: int, k: int, seed: int, n_requests: int = 32, block: int = 16,
                            min_len: int = 512, max_len: int = 4096,
                            share_prefix: bool = True) -> SignatureWorkload:
    """Requests 2i and 2i+1 share a leading block-aligned prefix.  Shared blocks are accumulated
    once, by the first request (cached blocks contribute rows from the earlier request
    that first prefilled them)."""
    rng = np.random.default_rng(sub_seed(seed, "sigwl", E, k))
    lens = rng.integers(min_len, max_len + 1, size=n_requests)
    nblk = (lens + block - 1) // block
    cold_ids: Dict[int, np.ndarray] = {}
    shared_blocks = np.zeros(n_requests, dtype=np.int64)
    for r in range(n_requests):
        ids = zipf_topk_ids(rng, int(lens[r]), E, k)
        if share_prefix and r % 2 == 1:
            max_sh = int(min(lens[r - 1], lens[r]) // block)
            sh = int(rng.integers(1, max(2, max_sh)))
            sh = min(sh, max_sh)
            shared_blocks[r] = sh
            ids[: sh * block] = cold_ids[r - 1][: sh * block]
        cold_ids[r] = ids
    total_blocks = int(sum(int(nblk[r] - shared_blocks[r]) for r in range(n_requests)))
    pool = rng.permutation(total_blocks + 64).astype(np.int32)   # non-contiguous ids, some never used
    nxt = 0
    req_blocks: Dict[int, np.ndarray] = {}
    tok_ids, tok_req, tok_blk = [], [], []
    for r in range(n_requests):
        sh = int(shared_blocks[r])
        own = int(nblk[r]) - sh
        mine = pool[nxt: nxt + own]
        nxt += own
        blocks = np.concatenate([req_blocks[r - 1][:sh], mine]) if sh else mine
        req_blocks[r] = blocks.astype(np.int32)
        start = sh * block
        n_new = int(lens[r]) - start
        tok_ids.append(cold_ids[r][start:])
        tok_req.append(np.full(n_new, r, dtype=np.int32))
        tok_blk.append(blocks[(np.arange(start, int(lens[r])) // block)].astype(np.int32))
    return SignatureWorkload(
        topk_ids=np.ascontiguousarray(np.concatenate(tok_ids), dtype=np.int32),
        token_req=np.concatenate(tok_req), token_block=np.concatenate(tok_blk),
        n_requests=n_requests, n_blocks=int(pool.max()) + 1, req_blocks=req_blocks,
        req_len=lens.astype(np.int64), cold_ids=cold_ids)


# ----------------------------------------------------------------------------------------------
# Hand-worked 4-expert example (all values small integers, exact in bf16).
# Embedded in H=8 / I=8 by zero padding so it also satisfies the library's 16-byte-vector shapes.
# ----------------------------------------------------------------------------------------------
def hand_example(pad_h: int = 2, pad_i: int = 1):
    H0, I0, E, k = 2, 1, 4, 2
    H, I = max(pad_h, H0), max(pad_i, I0)
    gate = np.zeros((E, H), np.float32)
    gate[:, :2] = np.array([[1, 0], [0, 1], [1, 1], [-1, 0]], np.float32)
    w1 = np.array([[1, 1], [-1, 0], [1, 0], [0, 1]], np.float32)
    w3 = np.array([[0, 1], [1, 0], [0, 1], [1, 1]], np.float32)
    w2t = np.array([[1, 1], [2, 0], [1, -1], [0, 1]], np.float32)   # W2_e^T : [H0] column of the [H,1] matrix
    w13 = np.zeros((E, 2 * I, H), np.float32)
    w2 = np.zeros((E, H, I), np.float32)
    w13[:, 0, :2] = w1
    w13[:, I, :2] = w3
    w2[:, :2, 0] = w2t
    x = np.zeros((2, H), np.float32)
    x[:, :2] = np.array([[1, 2], [2, -1]], np.float32)
    shape = MoEShape(hidden=H, inter=I, n_experts=E, top_k=k, n_layers=1, kv_block_size=16)
    lw = LayerWeights(gate, f32_to_bf16_bits(w13), f32_to_bf16_bits(w2), None, None)
    token_req = np.array([0, 1], np.int32)
    token_block = np.array([0, 1], np.int32)
    return shape, lw, f32_to_bf16_bits(x), token_req, token_block


# ----------------------------------------------------------------------------------------------
# Config 2/3 cases: (T, u) -> hiddens + gate bias.  The realised union can fall short of u by chance,
# so seeds are rejection-sampled ONCE by oracle/find_union_seeds.py (which calls only the oracle) and
# stored in union_seeds.json beside this file; this module only looks the accepted seed up.
# ----------------------------------------------------------------------------------------------
WEIGHT_SEED = 0


def union_case(shape: MoEShape, T: int, u: int, try_seed: int):
    """x [T,H] bf16 bits and gate_bias [E] for one (T,u) case at one try seed."""
    x = make_hidden(T, shape.hidden, try_seed, tag="xu%d" % u)
    bias = union_bias(shape.n_experts, u, try_seed)
    return x, bias


def accepted_union_seed(T: int, u: int) -> int:
    import json
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "union_seeds.json")
    with open(path) as f:
        table = json.load(f)
    return int(table["T%d_u%d" % (T, u)]["seed"])


# ------------------------------------------------------------------ routing-decision inputs
@dataclasses.dataclass
class RouteWorkload:
    counts: np.ndarray       # [R,L,E] int32 per-request expert counts (what eldr_signature_readout returns)
    df: np.ndarray           # [L,E] int32 document frequencies of a calibration corpus of n_calib requests
    n_calib: int
    layer_mask: np.ndarray   # [L] uint8, the kept layers S
    centroids: np.ndarray    # [K,L,E] float32, non-negative, NOT normalised
    loads: np.ndarray        # [K] int32 in-flight decode requests per worker
    domain: np.ndarray       # [R] which prototype the request was drawn around


def make_route_workload(R: int, L: int, E: int, K: int, k: int, seed: int, prompt_len=(512, 4096),
                        keep_layers: Optional[int] = None) -> RouteWorkload:
    """Stand-in for calibration artefacts and prefill signatures (the paper's corpora are not available offline):
    K non-negative prototypes over (layer, expert) with a few dominant "specialist" experts per layer and a few
    "generalist" experts shared by all; each request draws its prompt length and, per layer, multinomial counts of
    len*k picks around its domain's prototype; df is a seeded table that is large on the generalists."""
    g = np.random.default_rng(sub_seed(seed, "route", R, L, E, K))
    proto = g.random((K, L, E)) ** 4                       # skewed: a few specialists per (prototype, layer)
    generalists = g.permutation(E)[: max(1, E // 16)]
    proto[:, :, generalists] += 2.0
    centroids = (proto + 0.05 * g.random((K, L, E))).astype(np.float32)
    domain = g.integers(0, K, size=R)
    lens = g.integers(prompt_len[0], prompt_len[1] + 1, size=R)
    counts = np.empty((R, L, E), np.int32)
    for r in range(R):
        p = proto[domain[r]] + 0.02
        p = p / p.sum(axis=1, keepdims=True)
        for l in range(L):
            counts[r, l] = g.multinomial(int(lens[r]) * k, p[l]).astype(np.int32)
    n_calib = 1000
    df = g.integers(1, n_calib // 4, size=(L, E)).astype(np.int32)
    df[:, generalists] = n_calib - g.integers(0, 5, size=(L, generalists.size)).astype(np.int32)
    mask = np.zeros(L, np.uint8)
    keep = keep_layers if keep_layers is not None else max(1, (2 * L) // 3)
    mask[g.permutation(L)[:keep]] = 1
    loads = g.integers(0, 6, size=K).astype(np.int32)
    return RouteWorkload(counts, df, n_calib, mask, centroids, loads, domain)
