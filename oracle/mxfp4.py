"""TEST INFRASTRUCTURE ONLY -- fp64 oracle for MXFP4 expert weights ("GPT-OSS-120B
(128 experts, top-4, mxfp4)").  No CUDA kernel consumes this format yet; the oracle and its pins are committed first.

The paper only names the format.  Its definition is the OCP Microscaling (MX) v1.0 element / scale encoding, restated
here (readings, also listed in DESIGN.md section 2):
  * element: FP4 E2M1 -- 1 sign bit, 2 exponent bits (bias 1), 1 mantissa bit, no Inf / NaN:
        code = s e1 e0 m ;  value = (-1)^s * (e == 0 ? m * 0.5 : 2^(e-1) * (1 + m/2))
    i.e. magnitudes 0, 0.5, 1, 1.5, 2, 3, 4, 6 for codes 0..7;
  * scale: E8M0 -- one unsigned byte per block, value 2^(byte - 127); byte 255 is NaN;
  * block: 32 consecutive elements along the contraction (K, innermost) axis share one scale;
  * packing [reading: the paper is silent; this is the layout of the public GPT-OSS checkpoints]: two codes per byte,
    element 2i in the LOW nibble, element 2i+1 in the HIGH nibble.
An MoE layer with MXFP4 experts is then, by definition, the plain layer (oracle.moe_decode_layer) on the decoded
weights: every decoded value with scale byte in 3..250 is exactly a bf16 number (mxfp4_to_bf16_bits checks that), so
the existing fp64 layer oracle applies unchanged -- nothing is approximated.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module.
"""
import numpy as np

BLOCK = 32
# magnitudes of the eight E2M1 codes (sign bit clear), from the formula above written out
_E2M1 = np.array([0.0, 0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 6.0], dtype=np.float64)


def e2m1_value(code: np.ndarray) -> np.ndarray:
    """fp64 value of 4-bit codes (uint8 array, values 0..15)."""
    code = np.asarray(code, dtype=np.uint8)
    mag = _E2M1[code & 7]
    return np.where(code & 8, -mag, mag)


def e8m0_value(byte: np.ndarray) -> np.ndarray:
    """fp64 value of scale bytes: 2^(byte - 127); 255 -> NaN."""
    b = np.asarray(byte, dtype=np.uint8).astype(np.int64)
    out = np.ldexp(1.0, b - 127)
    return np.where(b == 255, np.nan, out)


def unpack_codes(packed: np.ndarray) -> np.ndarray:
    """[..., K/2] bytes -> [..., K] codes; element 2i = low nibble of byte i, element 2i+1 = high nibble."""
    packed = np.asarray(packed, dtype=np.uint8)
    out = np.empty(packed.shape[:-1] + (packed.shape[-1] * 2,), dtype=np.uint8)
    out[..., 0::2] = packed & 0x0F
    out[..., 1::2] = packed >> 4
    return out


def mxfp4_decode(packed: np.ndarray, scales: np.ndarray) -> np.ndarray:
    """packed [..., K/2] uint8, scales [..., K/32] uint8 -> fp64 [..., K]: value = e2m1(code) * 2^(scale - 127)."""
    codes = unpack_codes(packed)
    K = codes.shape[-1]
    if K % BLOCK or scales.shape[-1] * BLOCK != K or scales.shape[:-1] != codes.shape[:-1]:
        raise ValueError("K must be a multiple of 32 with one scale byte per block")
    return e2m1_value(codes) * np.repeat(e8m0_value(scales), BLOCK, axis=-1)


def mxfp4_to_bf16_bits(packed: np.ndarray, scales: np.ndarray) -> np.ndarray:
    """Decoded weights as bf16 bit patterns (uint16); raises unless every value is exactly representable."""
    v = mxfp4_decode(packed, scales)
    if not np.all(np.isfinite(v)):
        raise ValueError("NaN scale (byte 255) in the tensor")
    with np.errstate(over="ignore"):
        f32 = v.astype(np.float32)
    bits = f32.view(np.uint32)
    if np.any(f32.astype(np.float64) != v) or np.any(bits & 0xFFFF):
        raise ValueError("a decoded value is not a bf16 number (scale byte outside 3..250?)")
    return (bits >> 16).astype(np.uint16)
