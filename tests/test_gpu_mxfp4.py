"""GPU parity of the MXFP4 expert path: eldr_moe_decode_layer_mxfp4 through the C
ABI against the fp64 oracle.  An MXFP4 layer is by definition the plain layer on the decoded weights (oracle/mxfp4.py,
pinned by tests/test_mxfp4_pins.py), so the expected values come from oracle.moe_decode_layer on mxfp4_to_bf16_bits of
the same seeded bytes; gates as in test_gpu_parity.py (ids exact on clean tokens, h / y / out within 2e-2 / 2e-3)."""
import numpy as np
import pytest

from paper_2607_00466_b200 import synth

from parity_utils import check_gate, check_numeric, check_permutation

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests must run on the B200 box")
    from paper_2607_00466_b200 import api
    api.load()
    return api


def make_layer(shape, seed, scale_lo=118, scale_hi=122):
    E, H, I = shape.n_experts, shape.hidden, shape.inter
    c13, s13 = synth.make_mxfp4_tensor(E * 2 * I, H, seed, "w13", scale_lo, scale_hi)
    c2, s2 = synth.make_mxfp4_tensor(E * H, I, seed, "w2", scale_lo, scale_hi)
    gate_w = synth.make_gate_w(shape, seed)
    return gate_w, (c13.reshape(E, 2 * I, H // 2), s13.reshape(E, 2 * I, H // 32)), (c2.reshape(E, H, I // 2), s2.reshape(E, H, I // 32))


def run_mx(gpu, oracle, shape, T, seed, force=False, scale_lo=118, scale_hi=122, check_pairs=True):
    import torch
    from oracle import mxfp4
    k, E = shape.top_k, shape.n_experts
    gate_w, w13, w2 = make_layer(shape, seed, scale_lo, scale_hi)
    x_bits = synth.make_hidden(T, shape.hidden, seed + 1)
    dl = gpu.MxDecodeLayer(shape, gate_w, w13, w2, max_T=T)
    token_req = (np.arange(T) % 3).astype(np.int32)
    token_block = (np.arange(T) // 16).astype(np.int32)
    sig_req = torch.zeros((3, shape.n_layers, E), dtype=torch.int32, device="cuda")
    sig_blk = torch.zeros((T // 16 + 1, shape.n_layers, E), dtype=torch.int8, device="cuda")
    force_ids = force_w = None
    if force:
        rng = np.random.default_rng(seed)
        force_ids = np.stack([rng.choice(E, size=k, replace=False) for _ in range(T)]).astype(np.int32)
        force_w = rng.random((T, k)).astype(np.float32)
        force_w /= force_w.sum(1, keepdims=True)
        dl.ids[:T].copy_(torch.from_numpy(force_ids))
        dl.w[:T].copy_(torch.from_numpy(force_w))
    out = dl.run(gpu.bf16_from_bits(x_bits), None, 0, 1 if force else 0, torch.from_numpy(token_req).cuda(),
                 torch.from_numpy(token_block).cuda(), sig_req, sig_blk)
    torch.cuda.synchronize()
    assert gpu.eldr_moe_last_launch_count() == 5
    # the oracle's definition: the plain layer on the decoded weights (exact bf16 numbers)
    w13_bits = mxfp4.mxfp4_to_bf16_bits(*w13)
    w2_bits = mxfp4.mxfp4_to_bf16_bits(*w2)
    ora = oracle.moe_decode_layer(shape, x_bits, gate_w, None, w13_bits, w2_bits,
                                  force_ids=force_ids, force_w=None if force_w is None else force_w.astype(np.float64),
                                  dump_pairs=check_pairs)
    ids_gpu, w_gpu = dl.ids[:T].cpu().numpy(), dl.w[:T].cpu().numpy()
    if force:
        clean = np.ones(T, bool)
        assert np.array_equal(ids_gpu, force_ids)
    else:
        ora["z"] = oracle.gate_topk(shape, x_bits, gate_w, None)["z"]
        clean = check_gate(shape, ora, ids_gpu, w_gpu, dl.ws_view("z", T).cpu().numpy())
    op = oracle.permutation(shape, ids_gpu)
    pair_pos = dl.ws_view("pair_pos", T).cpu().numpy()
    check_permutation(shape, ids_gpu, dl.ws_view("cnt", T).cpu().numpy(), dl.ws_view("off", T).cpu().numpy(),
                      dl.ws_view("perm", T).cpu().numpy(), pair_pos, dl.active.cpu().numpy(), int(dl.n_active.item()), op)
    if check_pairs:
        h_gpu = dl.ws_view("h", T).float().cpu().numpy()
        # the MXFP4 step keeps h in the K-slot order of its decoder (e0 e4 e1 e5 e2 e6 e3 e7 per group of eight)
        h_gpu = h_gpu.reshape(h_gpu.shape[0], -1, 8)[:, :, [0, 2, 4, 6, 1, 3, 5, 7]].reshape(h_gpu.shape)
        y_gpu = dl.ws_view("y", T).cpu().numpy()
        rows_g, rows_o = [], []
        for t in np.nonzero(clean)[0]:
            omap = {int(e): j for j, e in enumerate(ora["ids"][t])}
            for j in range(k):
                rows_g.append(pair_pos[t * k + j])
                rows_o.append(t * k + omap[int(ids_gpu[t, j])])
        check_numeric(h_gpu[rows_g], ora["h_pairs"][rows_o], "h")
        check_numeric(y_gpu[rows_g], ora["y_pairs"][rows_o], "y")
    mx, mn = check_numeric(out.float().cpu().numpy()[clean], ora["out"][clean], "out")
    if clean.all():
        o_req = np.zeros(tuple(sig_req.shape), np.int32)
        o_blk = np.zeros(tuple(sig_blk.shape), np.int8)
        oracle.signature_accumulate(shape, 0, ora["ids"], token_req, token_block, o_req, o_blk)
        assert np.array_equal(sig_req.cpu().numpy(), o_req) and np.array_equal(sig_blk.cpu().numpy(), o_blk)
    return dl, out, mx, mn


@pytest.mark.parametrize("H,I,E,k,T", [(128, 64, 8, 2, 37),        # one row tile per matrix, ragged T
                                        (320, 192, 6, 3, 70),       # 5 / 3 k-chunks, 128-token passes (T > 64)
                                        (256, 128, 16, 4, 300),     # several passes per expert (75 tokens each, T > 256)
                                        (192, 320, 5, 5, 3)])       # H not a multiple of 128: partial last w2 row tile
def test_mxfp4_layer_ragged(gpu, oracle, H, I, E, k, T):
    shape = synth.MoEShape(hidden=H, inter=I, n_experts=E, top_k=k, n_layers=1, kv_block_size=16)
    run_mx(gpu, oracle, shape, T, seed=40 + H)


def test_mxfp4_scale_range_and_signs(gpu, oracle):
    """Scale bytes over a wide range (2^-40 .. 2^-20 here: every decoded value still an exact bf16 number, the outputs
    tiny but normal) -- a decoder that mishandled the exponent add, a sign nibble or the zero code fails this."""
    shape = synth.MoEShape(hidden=128, inter=128, n_experts=4, top_k=2, n_layers=1)
    run_mx(gpu, oracle, shape, 24, seed=77, scale_lo=87, scale_hi=107)


def test_mxfp4_scales_around_and_above_one(gpu, oracle):
    """Scale bytes 125..131 (2^-2 .. 2^4): the decoder folds its 2^126 into the block-scale multiplier while 2^(b-1) is a
    finite bf16 (b <= 128) and multiplies twice above that -- both sides of the switch, mixed inside one row."""
    shape = synth.MoEShape(hidden=128, inter=128, n_experts=4, top_k=2, n_layers=1)
    run_mx(gpu, oracle, shape, 24, seed=78, scale_lo=125, scale_hi=131)


def test_mxfp4_gpt_oss_shaped_layer(gpu, oracle):
    """GPT-OSS-120B-shaped experts (top-4, mxfp4; hidden = intermediate = 2880) with 16 of the 128 experts
    (the oracle's decoded copy of all 128 would take 6 GB): 45 k-chunks, 45 w1/w3 row tiles, 22.5 w2 row tiles."""
    shape = synth.MoEShape(hidden=2880, inter=2880, n_experts=16, top_k=4, n_layers=1)
    run_mx(gpu, oracle, shape, 64, seed=99, check_pairs=False)


def test_mxfp4_forced_routing_and_determinism(gpu, oracle):
    import torch
    shape = synth.MoEShape(hidden=256, inter=192, n_experts=12, top_k=3, n_layers=1)
    dl, out, _, _ = run_mx(gpu, oracle, shape, 50, seed=5, force=True)
    first = out.clone()
    x = gpu.bf16_from_bits(synth.make_hidden(50, shape.hidden, 6))
    for _ in range(3):
        again = dl.run(x, None, 0, 1)
        torch.cuda.synchronize()
        assert torch.equal(again.view(torch.int16), first.view(torch.int16))


def test_mxfp4_rejects_unsupported_shapes(gpu):
    import torch
    shape = synth.MoEShape(hidden=96, inter=64, n_experts=4, top_k=2, n_layers=1)      # H % 64 != 0
    gate_w = synth.make_gate_w(shape, 1)
    w13 = (np.zeros((4, 128, 48), np.uint8), np.full((4, 128, 3), 120, np.uint8))
    w2 = (np.zeros((4, 96, 32), np.uint8), np.full((4, 96, 2), 120, np.uint8))
    dl = gpu.MxDecodeLayer(shape, gate_w, w13, w2, max_T=8)
    with pytest.raises(RuntimeError, match="unsupported"):
        dl.run(torch.zeros((8, 96), dtype=torch.bfloat16, device="cuda"))
