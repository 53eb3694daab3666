"""Seeded random-shape sweep of eldr_moe_decode_layer against the oracle: shapes, paths, token maps and forced routing
drawn from a fixed generator (the same cases on every run).  A longer run of this generator (thousands of cases, other
seeds) found four defects the hand-written cases had missed -- a TMA-descriptor cache key without I, epochs that a
recycled workspace could replay, a packed int8 saturating add that could wrap, a partial GEMV tile -- each of which now
has a regression test of its own in test_gpu_parity.py; this file keeps a short version of the sweep in the suite.

Collected after the hand-written GPU tests (the suite runs with pytest -x)."""
import numpy as np
import pytest

from paper_2607_00466_b200 import synth
from test_gpu_parity import run_case

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests must run on the B200 box")
    from paper_2607_00466_b200 import api
    api.load()
    return api


def _paths(gpu):
    return [("fused", []), ("staged", [(gpu.OPT_STEP_PATH, gpu.STEP_STAGED)]),
            ("staged-mma_sync", [(gpu.OPT_STEP_PATH, gpu.STEP_STAGED), (gpu.OPT_FFN_PATH, gpu.FFN_MMA_SYNC)]),
            ("staged-gemv", [(gpu.OPT_STEP_PATH, gpu.STEP_STAGED), (gpu.OPT_FFN_PATH, gpu.FFN_GEMV)]),
            ("fused-streamk", [(gpu.OPT_DP_MIN_ROUNDS, 1 << 20)]), ("fused-split3", [(gpu.OPT_SK_MAX_SPLIT, 3)]),
            ("fused-headfirst", [(gpu.OPT_HEAD_FIRST, 1), (gpu.OPT_DP_MIN_ROUNDS, 1 << 20)])]


def _reset(gpu):
    gpu.eldr_moe_set_option(gpu.OPT_STEP_PATH, gpu.STEP_AUTO)
    gpu.eldr_moe_set_option(gpu.OPT_FFN_PATH, gpu.FFN_TCGEN05)
    gpu.eldr_moe_set_option(gpu.OPT_DP_MIN_ROUNDS, 1)
    gpu.eldr_moe_set_option(gpu.OPT_SK_MAX_SPLIT, 1)
    gpu.eldr_moe_set_option(gpu.OPT_HEAD_FIRST, 0)


@pytest.mark.parametrize("block", range(4))
def test_random_shapes_paths_maps_and_forced_routing(gpu, oracle, block):
    rng = np.random.default_rng(20260 + block)
    paths = _paths(gpu)
    done = 0
    while done < 14:
        H = int(rng.choice([64, 72, 128, 200, 256, 320, 512]))
        I = int(rng.choice([64, 40, 128, 192, 256, 448]))
        E = int(rng.integers(1, 160))
        k = int(rng.integers(1, min(E, 16) + 1))
        ns = int(rng.choice([0, 0, 0, 1, 2, 3]))
        T = int(rng.choice([9, 16, 31, 64, 96, 128, 130, 255, 256, 257, 400]))     # (T <= 8: the mean gate is a tiny-sample statistic)
        if T * k * max(H, I) > 12_000_000:
            continue
        shape = synth.MoEShape(hidden=H, inter=I, n_experts=E, top_k=k, n_shared=ns, n_layers=2, kv_block_size=16)
        seed = int(rng.integers(1, 1 << 20))
        lw = synth.make_layer_weights(shape, seed, w_std=0.05, gate_std=0.1)
        x = synth.make_hidden(T, H, seed + 1)
        name, opts = paths[int(rng.integers(0, len(paths)))]
        bias = synth.union_bias(E, max(int(rng.integers(1, 5)), k), seed, boost=30.0) if (rng.random() < 0.4 and E > k) else None
        n_req = int(rng.integers(1, T + 1))
        n_blk = T // 100 + 1 + int(rng.integers(0, T))
        token_req = rng.integers(-1, n_req, size=T).astype(np.int32)
        token_block = (np.arange(T) % n_blk).astype(np.int32)                      # at most 100 tokens per block (int8 cells)
        token_block[rng.random(T) < 0.05] = -1
        force = None
        if rng.random() < 0.25:
            fi = np.stack([rng.choice(E, size=k, replace=False) for _ in range(T)]).astype(np.int32)
            fw = rng.random((T, k)).astype(np.float32)
            force = (fi, fw / fw.sum(1, keepdims=True))
            bias = None
        for key, value in opts:
            gpu.eldr_moe_set_option(key, value)
        try:
            run_case(gpu, oracle, shape, lw, x, bias, token_req, token_block, n_req=n_req, n_blk=n_blk,
                     layer=int(rng.integers(0, 2)), check_pairs=False, force=force)
        except AssertionError as e:
            raise AssertionError("%s H=%d I=%d E=%d k=%d ns=%d T=%d bias=%s force=%s seed=%d: %s" %
                                 (name, H, I, E, k, ns, T, bias is not None, force is not None, seed, e))
        finally:
            _reset(gpu)
        done += 1
