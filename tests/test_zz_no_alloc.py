"""eldr_moe_gate_topk_static (include/eldr_moe.h): the gate + top-k (+ signature) entry point that allocates nothing -- its
logits scratch is a file-scope static __device__ array inside the library (ELDR_STATIC_SCRATCH_BYTES).  Checked against
the existing eldr_moe_gate_topk (caller's workspace) on the same inputs, on two calls in a row: the second call is
smaller than the first, so the shared array still holds the first call's logits past the second call's T * E.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import dataclasses

import numpy as np
import pytest

from paper_2607_00466_b200 import synth

pytestmark = pytest.mark.gpu

W_ABS = 1e-5          # the weight / logit gate of tests/parity_utils.py (same kernels on both sides: bit equality expected)


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests must run on the B200 box")
    from paper_2607_00466_b200 import api
    api.load()           # raises if the CUDA library is missing: no fallback
    return api


def _both(gpu, shape, T, seed, layer, n_req, n_blk):
    import torch
    k, E, L = shape.top_k, shape.n_experts, shape.n_layers
    gate_w = torch.from_numpy(synth.make_gate_w(shape, seed)).cuda()
    bias = torch.from_numpy((np.random.default_rng(seed).standard_normal(E) * 0.1).astype(np.float32)).cuda()
    x = gpu.bf16_from_bits(synth.make_hidden(T, shape.hidden, seed))
    token_req = torch.from_numpy((np.arange(T) % n_req).astype(np.int32)).cuda()
    token_block = torch.from_numpy((np.arange(T) % n_blk).astype(np.int32)).cuda()
    res = []
    for static in (False, True):
        ids = torch.full((T, k), -7, dtype=torch.int32, device="cuda")
        w = torch.full((T, k), -7.0, dtype=torch.float32, device="cuda")
        sig_req = torch.zeros((n_req, L, E), dtype=torch.int32, device="cuda")
        sig_blk = torch.zeros((n_blk, L, E), dtype=torch.int8, device="cuda")
        if static:
            gpu.eldr_moe_gate_topk_static(shape, layer, x, gate_w, bias, ids, w, token_req, token_block, sig_req, sig_blk)
        else:
            ws = torch.empty(gpu.eldr_moe_workspace_bytes(shape, T), dtype=torch.uint8, device="cuda")
            gpu.eldr_moe_gate_topk(shape, layer, x, gate_w, bias, ids, w, token_req, token_block, sig_req, sig_blk, ws)
        torch.cuda.synchronize()
        res.append((ids.cpu().numpy(), w.cpu().numpy(), sig_req.cpu().numpy(), sig_blk.cpu().numpy()))
    return res


def test_static_scratch_gate_topk_matches_the_workspace_path_on_two_calls_in_a_row(gpu):
    shape = dataclasses.replace(synth.SHAPE_QWEN, n_layers=2)
    # first call: T * E * 4 = 983040 bytes (almost the whole array), ragged tail; second: 37 tokens, other inputs
    for T, seed, layer in ((1920 - 3, 21, 1), (37, 22, 0)):
        (ids_a, w_a, sr_a, sb_a), (ids_b, w_b, sr_b, sb_b) = _both(gpu, shape, T, seed, layer, n_req=5, n_blk=64)
        assert ids_a.min() >= 0 and ids_a.max() < shape.n_experts
        assert np.array_equal(ids_a, ids_b)                                  # integer work: bit-exact
        assert np.abs(w_a.astype(np.float64) - w_b.astype(np.float64)).max() <= W_ABS
        assert np.allclose(w_b.sum(axis=1), 1.0, atol=1e-5)
        assert np.array_equal(sr_a, sr_b) and np.array_equal(sb_a, sb_b)
        assert int(sr_b.sum()) == T * shape.top_k and int(sr_b[:, 1 - layer].sum()) == 0


def test_static_scratch_limit_is_enforced(gpu):
    import torch
    shape = synth.SHAPE_QWEN
    T = gpu.STATIC_SCRATCH_BYTES // (4 * shape.n_experts) + 1                  # one token too many
    x = torch.zeros((T, shape.hidden), dtype=torch.bfloat16, device="cuda")
    gate_w = torch.zeros((shape.n_experts, shape.hidden), dtype=torch.float32, device="cuda")
    ids = torch.full((T, shape.top_k), -7, dtype=torch.int32, device="cuda")
    w = torch.zeros((T, shape.top_k), dtype=torch.float32, device="cuda")
    with pytest.raises(RuntimeError, match="workspace too small.*static scratch"):
        gpu.eldr_moe_gate_topk_static(shape, 0, x, gate_w, None, ids, w)
    torch.cuda.synchronize()
    assert int(ids.max().item()) == -7                                       # nothing was launched
    # exactly at the limit it runs
    gpu.eldr_moe_gate_topk_static(shape, 0, x[: T - 1], gate_w, None, ids[: T - 1], w[: T - 1])
    torch.cuda.synchronize()
    assert int(ids[: T - 1].min().item()) >= 0
