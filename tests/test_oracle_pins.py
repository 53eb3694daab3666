"""Pins of the fp64 CPU oracle against things OTHER than itself (CPU only, no GPU).

Each test is chosen so that a plausible mistake in oracle/eldr_oracle.c (dropped term, wrong sign
or index, transposed operand, wrong tie-break) fails at least one of them:
  * library routines (numpy fp64 matmul, scipy softmax / expit) on special cases,
  * closed forms (renormalised weights = softmax over the selected logits),
  * brute force over all C(E,k) subsets on tiny gates,
  * a second, differently organised formulation of the whole layer,
  * the hand-worked 4-expert example (tests/golden/hand_example.txt),
  * the integer invariants of the signature path.
"""
import dataclasses
import itertools
import os

import numpy as np
import pytest
from scipy.special import expit, softmax

from paper_2607_00466_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _f64(bits):
    return synth.bf16_bits_to_f32(bits).astype(np.float64)


def _tiny(seed, H=8, I=4, E=6, k=2, T=5, n_shared=0, renorm=1):
    shape = synth.MoEShape(hidden=H, inter=I, n_experts=E, top_k=k, n_shared=n_shared,
                           renormalize=renorm, n_layers=1, kv_block_size=16)
    lw = synth.make_layer_weights(shape, seed, w_std=0.5, gate_std=0.7)
    x = synth.make_hidden(T, H, seed)
    return shape, lw, x


# ------------------------------------------------------------------------------------------ gate
def test_gate_logits_match_numpy_matmul(oracle):
    shape = synth.SHAPE_C1
    lw = synth.make_layer_weights(shape, 0)
    x = synth.make_hidden(8, shape.hidden, 0)
    bias = np.linspace(-1, 1, shape.n_experts).astype(np.float32)
    r = oracle.gate_topk(shape, x, lw.gate_w, bias)
    z_ref = _f64(x) @ lw.gate_w.astype(np.float64).T + bias.astype(np.float64)
    assert np.abs(r["z"] - z_ref).max() <= 1e-12


def test_topk_is_argsort_and_weights_closed_form(oracle):
    shape = synth.SHAPE_C1
    lw = synth.make_layer_weights(shape, 1)
    x = synth.make_hidden(32, shape.hidden, 1)
    r = oracle.gate_topk(shape, x, lw.gate_w, None)
    z = _f64(x) @ lw.gate_w.astype(np.float64).T
    order = np.argsort(-z, axis=1, kind="stable")[:, : shape.top_k]
    assert np.array_equal(r["ids"], order.astype(np.int32))
    # closed form: the full-E softmax denominator cancels -> softmax over the k selected logits
    zsel = np.take_along_axis(z, order, axis=1)
    assert np.abs(r["w"] - softmax(zsel, axis=1)).max() <= 1e-12
    assert np.abs(r["w"].sum(axis=1) - 1.0).max() <= 1e-12
    # margin = z_(k) - z_(k+1)
    zs = -np.sort(-z, axis=1)
    assert np.abs(r["margin"] - (zs[:, shape.top_k - 1] - zs[:, shape.top_k])).max() <= 1e-12


def test_no_renormalise_gives_full_softmax(oracle):
    shape, lw, x = _tiny(3, E=7, k=3, renorm=0)
    r = oracle.gate_topk(shape, x, lw.gate_w, None)
    p = softmax(_f64(x) @ lw.gate_w.astype(np.float64).T, axis=1)
    assert np.abs(r["w"] - np.take_along_axis(p, r["ids"].astype(np.int64), axis=1)).max() <= 1e-12


@pytest.mark.parametrize("E,k", [(4, 1), (5, 2), (6, 3), (8, 4), (8, 7)])
def test_topk_brute_force_subsets(oracle, E, k):
    shape, lw, x = _tiny(10 + E + k, E=E, k=k, T=9)
    r = oracle.gate_topk(shape, x, lw.gate_w, None)
    z = _f64(x) @ lw.gate_w.astype(np.float64).T
    for t in range(x.shape[0]):
        best = max(itertools.combinations(range(E), k), key=lambda S: sum(z[t, list(S)]))
        assert set(best) == set(r["ids"][t].tolist())
        assert len(set(r["ids"][t].tolist())) == k          # distinct experts per token


def test_gate_shift_invariance_and_expert_permutation(oracle):
    shape, lw, x = _tiny(5, E=6, k=3, T=7)
    r0 = oracle.gate_topk(shape, x, lw.gate_w, None)
    r1 = oracle.gate_topk(shape, x, lw.gate_w, np.full(6, 3.25, np.float32))
    assert np.array_equal(r0["ids"], r1["ids"])
    assert np.abs(r0["w"] - r1["w"]).max() <= 1e-12
    perm = np.array([3, 0, 5, 1, 4, 2])
    r2 = oracle.gate_topk(shape, x, np.ascontiguousarray(lw.gate_w[perm]), None)
    assert np.array_equal(perm[r2["ids"]], r0["ids"])
    assert np.abs(r2["w"] - r0["w"]).max() <= 1e-12


def test_tie_break_prefers_lower_id(oracle):
    shape = synth.MoEShape(hidden=8, inter=8, n_experts=5, top_k=2)
    gate = np.zeros((5, 8), np.float32)
    gate[:, 0] = [1.0, 2.0, 2.0, 2.0, 0.5]      # experts 1,2,3 tie
    x = synth.f32_to_bf16_bits(np.eye(1, 8, dtype=np.float32))
    r = oracle.gate_topk(shape, x, gate, None)
    assert r["ids"].tolist() == [[1, 2]]
    assert r["margin"][0] == 0.0
    assert np.allclose(r["w"], [[0.5, 0.5]])


# ------------------------------------------------------------------------------------------- FFN
def test_silu_pin_scalar_expert(oracle):
    shape = synth.MoEShape(hidden=1, inter=1, n_experts=1, top_k=1)
    for a in (-3.0, -0.5, 0.0, 0.75, 2.0):
        w13 = synth.f32_to_bf16_bits(np.array([[[a]], [[1.0]]], np.float32).reshape(2, 1))
        w2 = synth.f32_to_bf16_bits(np.array([[1.0]], np.float32))
        x = synth.f32_to_bf16_bits(np.array([1.0], np.float32))
        h, y = oracle.expert_ffn(shape, x, w13, w2)
        assert abs(h[0] - a * expit(a)) <= 1e-15 and abs(y[0] - h[0]) == 0.0


def _dense_ffn_numpy(x, w13_e, w2_e, I):
    g = x @ w13_e[:I].T
    u = x @ w13_e[I:].T
    return (g * expit(g) * u) @ w2_e.T


def test_identical_experts_reduce_to_dense_ffn(oracle):
    shape, lw, x = _tiny(7, H=16, I=12, E=6, k=3, T=6)
    w13 = np.ascontiguousarray(np.broadcast_to(lw.w13[0], lw.w13.shape))
    w2 = np.ascontiguousarray(np.broadcast_to(lw.w2[0], lw.w2.shape))
    r = oracle.moe_decode_layer(shape, x, lw.gate_w, None, w13, w2)
    ref = _dense_ffn_numpy(_f64(x), _f64(w13[0]), _f64(w2[0]), shape.inter)
    assert np.abs(r["out"] - ref).max() <= 1e-12 * max(1.0, np.abs(ref).max())


def test_k1_is_argmax_expert_and_kE_is_full_softmax_mixture(oracle):
    shape, lw, x = _tiny(8, H=16, I=12, E=5, k=1, T=6)
    r = oracle.moe_decode_layer(shape, x, lw.gate_w, None, lw.w13, lw.w2)
    z = _f64(x) @ lw.gate_w.astype(np.float64).T
    for t in range(6):
        e = int(np.argmax(z[t]))
        ref = _dense_ffn_numpy(_f64(x[t:t + 1]), _f64(lw.w13[e]), _f64(lw.w2[e]), shape.inter)[0]
        assert r["ids"][t, 0] == e and r["w"][t, 0] == 1.0
        assert np.abs(r["out"][t] - ref).max() <= 1e-12 * max(1.0, np.abs(ref).max())
    shapeE = dataclasses.replace(shape, top_k=5)
    rE = oracle.moe_decode_layer(shapeE, x, lw.gate_w, None, lw.w13, lw.w2)
    p = softmax(z, axis=1)
    ref = sum(p[:, e:e + 1] * _dense_ffn_numpy(_f64(x), _f64(lw.w13[e]), _f64(lw.w2[e]), shape.inter)
              for e in range(5))
    assert rE["n_active"] == 5
    assert np.abs(rE["out"] - ref).max() <= 1e-12 * max(1.0, np.abs(ref).max())


def test_zero_branch_gives_zero_and_w2_scaling_is_linear(oracle):
    shape, lw, x = _tiny(9, H=16, I=12, E=6, k=2, T=4)
    I = shape.inter
    w13 = lw.w13.copy()
    w13[:, I:, :] = 0                      # W3 = 0  -> u = 0 -> out = 0
    assert np.all(oracle.moe_decode_layer(shape, x, lw.gate_w, None, w13, lw.w2)["out"] == 0.0)
    w13 = lw.w13.copy()
    w13[:, :I, :] = 0                      # W1 = 0 -> silu(0) = 0 -> out = 0
    assert np.all(oracle.moe_decode_layer(shape, x, lw.gate_w, None, w13, lw.w2)["out"] == 0.0)
    base = oracle.moe_decode_layer(shape, x, lw.gate_w, None, lw.w13, lw.w2)["out"]
    w2x2 = synth.f32_to_bf16_bits(synth.bf16_bits_to_f32(lw.w2) * np.float32(2.0))   # exact in bf16
    dbl = oracle.moe_decode_layer(shape, x, lw.gate_w, None, lw.w13, w2x2)["out"]
    assert np.array_equal(dbl, 2.0 * base)


@pytest.mark.parametrize("n_shared", [0, 2])
def test_layer_matches_second_formulation_all_experts_masked(oracle, n_shared):
    """Dense 'compute every expert, mask by routing weight' with numpy einsum -- organised
    differently from the oracle's per-token loop, and with non-square W2 so a transposed operand fails."""
    shape, lw, x = _tiny(11, H=24, I=10, E=6, k=3, T=7, n_shared=n_shared)
    bias = np.array([0.3, -0.2, 0, 0.1, 0, -0.4], np.float32)
    r = oracle.moe_decode_layer(shape, x, lw.gate_w, bias, lw.w13, lw.w2, lw.shared_w13, lw.shared_w2,
                                dump_pairs=True)
    X = _f64(x)
    z = X @ lw.gate_w.astype(np.float64).T + bias
    p = softmax(z, axis=1)
    order = np.argsort(-z, axis=1, kind="stable")[:, : shape.top_k]
    mask = np.zeros_like(p)
    np.put_along_axis(mask, order, 1.0, axis=1)
    wfull = p * mask
    wfull /= wfull.sum(axis=1, keepdims=True)
    W13, W2 = _f64(lw.w13), _f64(lw.w2)
    I = shape.inter
    G = np.einsum("th,eih->tei", X, W13[:, :I])
    U = np.einsum("th,eih->tei", X, W13[:, I:])
    Hh = G * expit(G) * U
    Y = np.einsum("tei,ehi->teh", Hh, W2)
    ref = np.einsum("te,teh->th", wfull, Y)
    for s in range(n_shared):
        ref = ref + _dense_ffn_numpy(X, _f64(lw.shared_w13[s]), _f64(lw.shared_w2[s]), I)
    assert np.abs(r["out"] - ref).max() <= 1e-11 * max(1.0, np.abs(ref).max())
    # per-pair dumps are indexed by (token, slot)
    for t in range(7):
        for j in range(shape.top_k):
            e = r["ids"][t, j]
            assert np.abs(r["h_pairs"][t * shape.top_k + j] - Hh[t, e]).max() <= 1e-11
            assert np.abs(r["y_pairs"][t * shape.top_k + j] - Y[t, e]).max() <= 1e-11
    # union / bytes invariant (north_star): bytes = (|U| + n_shared) * 3*H*I*2
    U_set = sorted(set(order.ravel().tolist()))
    assert r["active"][: r["n_active"]].tolist() == U_set
    assert r["bytes_loaded"] == (len(U_set) + n_shared) * shape.expert_bytes
    assert np.array_equal(r["cnt"], np.bincount(order.ravel(), minlength=shape.n_experts))


def test_force_routing_uses_given_ids_and_weights(oracle):
    shape, lw, x = _tiny(12, H=16, I=8, E=6, k=2, T=3)
    ids = np.array([[5, 0], [1, 2], [3, 3 - 3]], np.int32)
    w = np.array([[0.25, 0.75], [1.0, 0.0], [0.5, 0.5]], np.float64)
    r = oracle.moe_decode_layer(shape, x, lw.gate_w, None, lw.w13, lw.w2, force_ids=ids, force_w=w)
    X = _f64(x)
    for t in range(3):
        ref = sum(w[t, j] * _dense_ffn_numpy(X[t:t + 1], _f64(lw.w13[ids[t, j]]), _f64(lw.w2[ids[t, j]]),
                                             shape.inter)[0] for j in range(2))
        assert np.abs(r["out"][t] - ref).max() <= 1e-12 * max(1.0, np.abs(ref).max())
    assert r["n_active"] == 5 and r["active"][:5].tolist() == [0, 1, 2, 3, 5]


# ------------------------------------------------------------------------------ hand-worked example
def _golden():
    vals = {}
    with open(os.path.join(GOLDEN, "hand_example.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, *v = line.split()
            vals[k] = np.array([float(t) for t in v])
    return vals


@pytest.mark.parametrize("pad", [(2, 1), (8, 8)])
def test_hand_worked_example(oracle, pad):
    g = _golden()
    shape, lw, x, token_req, token_block = synth.hand_example(*pad)
    r = oracle.moe_decode_layer(shape, x, lw.gate_w, None, lw.w13, lw.w2, dump_pairs=True)
    gr = oracle.gate_topk(shape, x, lw.gate_w, None)
    tol = 2e-7
    for t in range(2):
        assert np.abs(gr["z"][t] - g["z%d" % t]).max() == 0.0
        assert np.abs(softmax(gr["z"][t]) - g["p%d" % t]).max() <= tol
        assert r["ids"][t].tolist() == g["ids%d" % t].astype(int).tolist()
        assert np.abs(r["w"][t] - g["w%d" % t]).max() <= tol
        assert np.abs(r["h_pairs"][2 * t: 2 * t + 2, 0] - g["h%d" % t]).max() <= tol
        for j in range(2):
            assert np.abs(r["y_pairs"][2 * t + j, :2] - g["y%d%d" % (t, j)]).max() <= tol
        assert np.abs(r["out"][t, :2] - g["out%d" % t]).max() <= tol
        assert np.all(r["out"][t, 2:] == 0.0)
    assert r["n_active"] == int(g["n_active"][0])
    assert r["active"][: r["n_active"]].tolist() == g["active"].astype(int).tolist()
    if pad == (2, 1):
        assert r["bytes_loaded"] == int(g["bytes"][0])
    sig_req = np.zeros((2, 1, 4), np.int32)
    sig_block = np.zeros((2, 1, 4), np.int8)
    oracle.signature_accumulate(shape, 0, r["ids"], token_req, token_block, sig_req, sig_block)
    assert sig_req[0, 0].tolist() == g["sig_req0"].astype(int).tolist()
    assert sig_req[1, 0].tolist() == g["sig_req1"].astype(int).tolist()
    assert np.array_equal(sig_block.astype(np.int32), sig_req)
    assert int(sig_req.sum()) == int(g["sig_total"][0])


# ------------------------------------------------------------------------------------ permutation
def test_permutation_against_numpy(oracle):
    shape = synth.MoEShape(hidden=8, inter=8, n_experts=12, top_k=3)
    rng = np.random.default_rng(4)
    ids = np.stack([rng.permutation(12)[:3] for _ in range(37)]).astype(np.int32)
    p = oracle.permutation(shape, ids)
    flat = ids.ravel()
    assert np.array_equal(p["cnt"], np.bincount(flat, minlength=12))
    assert np.array_equal(p["off"], np.concatenate([[0], np.cumsum(np.bincount(flat, minlength=12))]))
    assert np.array_equal(p["perm"], np.argsort(flat, kind="stable").astype(np.int32))
    act = np.nonzero(np.bincount(flat, minlength=12))[0]
    assert p["n_active"] == len(act) and np.array_equal(p["active"][: len(act)], act)
    assert np.all(p["active"][len(act):] == -1)


# ------------------------------------------------------------------------------------- signatures
def test_c1_signature_counts(oracle):
    """BASELINE.json config 1: 2 requests x 4 tokens; each request row sums to 4*1*2 = 8."""
    shape = synth.SHAPE_C1
    lw = synth.make_layer_weights(shape, 0)
    x = synth.make_hidden(8, shape.hidden, 0)
    token_req, token_block = synth.c1_maps()
    ids = oracle.gate_topk(shape, x, lw.gate_w, None)["ids"]
    sig_req = np.zeros((2, 1, shape.n_experts), np.int32)
    sig_block = np.zeros((4, 1, shape.n_experts), np.int8)
    oracle.signature_accumulate(shape, 0, ids, token_req, token_block, sig_req, sig_block)
    assert sig_req.sum(axis=(1, 2)).tolist() == [8, 8]
    assert int(sig_req.sum()) == 8 * 1 * 2                       # tokens x layers x k
    for r, blocks in ((0, [0, 1]), (1, [2, 3])):                 # s_r = sum_b sig[b]
        assert np.array_equal(oracle.signature_readout(shape, blocks, sig_block), sig_req[r])
    assert sig_block.max() <= shape.kv_block_size
    # bincount is the library definition of "count how many tokens are routed to each expert" (:198)
    for r in range(2):
        assert np.array_equal(sig_req[r, 0], np.bincount(ids[token_req == r].ravel(), minlength=16))


def test_signature_prefix_sharing_equals_cold_prefill_and_reset(oracle):
    E, k, L = 16, 3, 4
    shape = synth.MoEShape(hidden=8, inter=8, n_experts=E, top_k=k, n_layers=L, kv_block_size=16)
    wl = synth.make_signature_workload(E, k, seed=3, n_requests=6, min_len=40, max_len=200)
    sig_req = np.zeros((wl.n_requests, L, E), np.int32)
    sig_block = np.zeros((wl.n_blocks, L, E), np.int8)
    for layer in range(L):
        ids_l = (wl.topk_ids + layer) % E        # a different (still distinct-per-token) pick per layer
        oracle.signature_accumulate(shape, layer, np.ascontiguousarray(ids_l), wl.token_req,
                                    wl.token_block, sig_req, sig_block)
    n_tok = wl.topk_ids.shape[0]
    assert int(sig_block.astype(np.int64).sum()) == n_tok * L * k       # tokens x layers x k
    assert int(sig_req.sum()) == n_tok * L * k
    for r in range(wl.n_requests):
        read = oracle.signature_readout(shape, wl.req_blocks[r], sig_block)
        cold = np.stack([np.bincount(((wl.cold_ids[r] + layer) % E).ravel(), minlength=E)
                         for layer in range(L)])
        assert np.array_equal(read, cold)        # "the sum matches a cold prefill of the same prompt"
        assert np.all(read.sum(axis=1) == wl.req_len[r] * k)
    assert sig_block.max() <= 16 and sig_block.min() >= 0
    # negative maps => token not recorded
    before = sig_req.copy()
    oracle.signature_accumulate(shape, 0, wl.topk_ids[:5], np.full(5, -1, np.int32),
                                np.full(5, -1, np.int32), sig_req, sig_block)
    assert np.array_equal(before, sig_req)
    # reused block resets its signature
    b = wl.req_blocks[0][:2]
    oracle.signature_reset_blocks(shape, b, sig_block)
    assert not sig_block[b].any()
    other = wl.req_blocks[2]
    assert sig_block[other].any()


def test_int8_block_cells_saturate_at_127(oracle):
    """DESIGN.md 2 reading "int8 cells saturate": 130 tokens written into ONE block row (outside PAPER.md:255's
    contract of <= block-size tokens per block) leave the cell at 127, its neighbours untouched, and the int32
    request row at the true count -- pinned against numpy's clip."""
    shape = synth.MoEShape(hidden=8, inter=8, n_experts=8, top_k=2, n_layers=1, kv_block_size=16)
    T = 130
    ids = np.tile(np.array([[3, 5]], np.int32), (T, 1))
    req = np.zeros(T, np.int32)
    blk = np.zeros(T, np.int32)
    sig_req = np.zeros((1, 1, 8), np.int32)
    sig_blk = np.zeros((1, 1, 8), np.int8)
    oracle.signature_accumulate(shape, 0, ids, req, blk, sig_req, sig_blk)
    want = np.clip(np.bincount(ids.ravel(), minlength=8), 0, 127)
    assert sig_blk[0, 0].tolist() == want.tolist() == [0, 0, 0, 127, 0, 127, 0, 0]
    assert sig_req[0, 0].tolist() == [0, 0, 0, 130, 0, 130, 0, 0]
