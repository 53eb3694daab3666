"""Pins of the MXFP4 oracle (oracle/mxfp4.py): the hand-typed format table in
tests/golden/mxfp4_e2m1.txt, the sign/exponent/mantissa formula evaluated independently, block structure, nibble
order, exact bf16 representability, and the layer oracle on decoded weights in two special cases."""
import os

import numpy as np
import pytest

from oracle import mxfp4
from paper_2607_00466_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "mxfp4_e2m1.txt")


def _golden():
    codes, scales = {}, {}
    for line in open(GOLDEN):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        f = line.split()
        if f[0] == "scale":
            scales[int(f[1])] = float(f[2])
        else:
            codes[int(f[0], 2)] = float(f[1])
    return codes, scales


def test_element_and_scale_tables_match_the_hand_typed_format_table():
    codes, scales = _golden()
    assert sorted(codes) == list(range(16))
    got = mxfp4.e2m1_value(np.arange(16, dtype=np.uint8))
    for c, v in codes.items():
        assert got[c] == v and np.signbit(got[c]) == np.signbit(v)
    for b, v in scales.items():
        assert mxfp4.e8m0_value(np.array([b], dtype=np.uint8))[0] == v
    assert np.isnan(mxfp4.e8m0_value(np.array([255], dtype=np.uint8))[0])


def test_element_values_follow_the_sign_exponent_mantissa_formula():
    """Independent of the oracle's table: (-1)^s * (e ? 2^(e-1) * (1 + m/2) : m/2), bias 1, no Inf/NaN."""
    for code in range(16):
        s, e, m = code >> 3, (code >> 1) & 3, code & 1
        want = (-1.0) ** s * ((2.0 ** (e - 1)) * (1 + m / 2) if e else m / 2)
        assert mxfp4.e2m1_value(np.array([code], dtype=np.uint8))[0] == want


def test_nibble_order_and_block_structure():
    packed = np.zeros((1, 32), dtype=np.uint8)            # K = 64: two blocks
    packed[0, 0] = 0x21                                   # element 0 = code 1 (0.5), element 1 = code 2 (1.0)
    packed[0, 16] = 0xF7                                  # element 32 = code 7 (6.0), element 33 = code 15 (-6.0)
    scales = np.array([[127, 128]], dtype=np.uint8)       # block 0 x1, block 1 x2
    v = mxfp4.mxfp4_decode(packed, scales)
    assert v.shape == (1, 64)
    assert list(v[0, :3]) == [0.5, 1.0, 0.0] and list(v[0, 32:35]) == [12.0, -12.0, 0.0]
    # raising one block's scale byte by one doubles exactly that block
    p, s = synth.make_mxfp4_tensor(5, 128, 3)
    base = mxfp4.mxfp4_decode(p, s)
    s2 = s.copy()
    s2[:, 2] += 1
    bumped = mxfp4.mxfp4_decode(p, s2)
    assert np.array_equal(bumped[:, 64:96], 2.0 * base[:, 64:96])
    assert np.array_equal(np.delete(bumped, np.s_[64:96], axis=1), np.delete(base, np.s_[64:96], axis=1))
    with pytest.raises(ValueError):
        mxfp4.mxfp4_decode(p[:, :-1], s)


def test_decoded_weights_are_exact_bf16_numbers():
    p, s = synth.make_mxfp4_tensor(64, 256, 7, scale_lo=3, scale_hi=250)
    bits = mxfp4.mxfp4_to_bf16_bits(p, s)
    assert np.array_equal(synth.bf16_bits_to_f32(bits).astype(np.float64), mxfp4.mxfp4_decode(p, s))
    with pytest.raises(ValueError):                       # 6 * 2^127 is not finite in bf16
        mxfp4.mxfp4_to_bf16_bits(np.full((1, 16), 0x77, np.uint8), np.array([[254]], np.uint8))
    with pytest.raises(ValueError):
        mxfp4.mxfp4_to_bf16_bits(p[:1], np.full((1, 8), 255, np.uint8))


def test_layer_on_decoded_weights_special_cases():
    """An MXFP4 layer is the plain layer on the decoded weights.  Two cases with a closed form: all codes zero -> the
    output is exactly zero; every expert the same tensor with k = 1 -> the output is that expert's dense SwiGLU FFN,
    computed here with numpy matmuls on the decoded fp64 values."""
    from oracle import oracle
    shape = synth.MoEShape(hidden=64, inter=32, n_experts=4, top_k=1, n_layers=1)
    H, I, E = shape.hidden, shape.inter, shape.n_experts
    gate_w = synth.make_gate_w(shape, 11)
    x = synth.make_hidden(6, H, 12)
    p13, s13 = synth.make_mxfp4_tensor(2 * I, H, 13)
    p2, s2 = synth.make_mxfp4_tensor(H, I, 14)
    w13 = np.broadcast_to(mxfp4.mxfp4_to_bf16_bits(p13, s13), (E, 2 * I, H)).copy()
    w2 = np.broadcast_to(mxfp4.mxfp4_to_bf16_bits(p2, s2), (E, H, I)).copy()
    out = oracle.moe_decode_layer(shape, x, gate_w, None, w13, w2)["out"]
    xd = synth.bf16_bits_to_f32(x).astype(np.float64)
    W13, W2 = mxfp4.mxfp4_decode(p13, s13), mxfp4.mxfp4_decode(p2, s2)
    g, u = xd @ W13[:I].T, xd @ W13[I:].T
    want = (g / (1.0 + np.exp(-g)) * u) @ W2.T
    assert np.allclose(out, want, rtol=1e-12, atol=1e-15)
    zero13 = mxfp4.mxfp4_to_bf16_bits(np.zeros_like(p13), s13)
    out0 = oracle.moe_decode_layer(shape, x, gate_w, None, np.broadcast_to(zero13, (E, 2 * I, H)).copy(), w2)["out"]
    assert not np.any(out0)
