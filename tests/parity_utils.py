"""Shared comparison rules for the GPU parity tests.

Gate A (exact):   on tokens whose oracle margin z_(k)-z_(k+1) > 1e-5, ids are set-equal per token and
                  signature cells are bit-exact.  Near-tie tokens are excluded and counted.
Gate B (numeric): out max floored-relative error <= 2e-2 and mean <= 2e-3 (north_star tolerances):
                  rel_i = |gpu_i - ref_i| / max(|ref_i|, rms(ref_token)).
Gate C:           invariants of the GPU outputs themselves.
"""
import numpy as np

NEAR_TIE = 1e-5
Z_ABS = 1e-5
MAX_REL = 2e-2
MEAN_REL = 2e-3


def floored_rel(gpu: np.ndarray, ref: np.ndarray) -> np.ndarray:
    """Per-element |gpu-ref| / max(|ref|, rms(ref row)); rows are tokens (or pairs)."""
    gpu = np.asarray(gpu, np.float64)
    ref = np.asarray(ref, np.float64)
    rms = np.sqrt((ref * ref).mean(axis=-1, keepdims=True))
    floor = np.maximum(np.abs(ref), np.maximum(rms, 1e-300))
    return np.abs(gpu - ref) / floor


def check_numeric(gpu, ref, what="out", max_rel=MAX_REL, mean_rel=MEAN_REL):
    if np.asarray(ref).size == 0:
        return 0.0, 0.0
    rel = floored_rel(gpu, ref)
    mx, mn = float(rel.max()), float(rel.mean())
    assert np.isfinite(np.asarray(gpu, np.float64)).all(), "%s: non-finite GPU values" % what
    assert mx <= max_rel, "%s: max floored-rel error %.3e > %.1e" % (what, mx, max_rel)
    assert mn <= mean_rel, "%s: mean floored-rel error %.3e > %.1e" % (what, mn, mean_rel)
    return mx, mn


def clean_tokens(margin: np.ndarray) -> np.ndarray:
    return np.asarray(margin) > NEAR_TIE


def check_gate(shape, ora, ids_gpu, w_gpu, z_gpu=None):
    """Gate A on ids (+ weights matched by id, abs 1e-5) for clean tokens; returns the clean mask."""
    clean = clean_tokens(ora["margin"])
    k, E = shape.top_k, shape.n_experts
    ids_gpu = np.asarray(ids_gpu)
    w_gpu = np.asarray(w_gpu, np.float64)
    assert ids_gpu.min() >= 0 and ids_gpu.max() < E
    for t in range(ids_gpu.shape[0]):
        assert len(set(ids_gpu[t].tolist())) == k, "token %d: ids not distinct" % t
    assert np.abs(w_gpu.sum(axis=1) - 1.0).max() <= 1e-5 if shape.renormalize else True
    for t in np.nonzero(clean)[0]:
        assert set(ids_gpu[t].tolist()) == set(ora["ids"][t].tolist()), "token %d: top-k set differs" % t
        wmap = dict(zip(ora["ids"][t].tolist(), ora["w"][t].tolist()))
        for j in range(k):
            assert abs(w_gpu[t, j] - wmap[int(ids_gpu[t, j])]) <= 1e-5, "token %d slot %d weight" % (t, j)
    if z_gpu is not None:
        # "z: abs err <= 1e-5", absolute, on logits including the bias (no scaling with |z|)
        zerr = np.abs(np.asarray(z_gpu, np.float64) - ora["z"])
        assert zerr.max() <= Z_ABS, "gate logits abs err %.3e > %.1e" % (zerr.max(), Z_ABS)
    return clean


def check_permutation(shape, ids_gpu, cnt, off, perm, pair_pos, active, n_active, oracle_perm):
    """Kernel P outputs: cnt/off/active exact vs the oracle run on the GPU's own ids; perm compared per
    expert segment as a multiset (order inside a segment is not unique)."""
    E, k = shape.n_experts, shape.top_k
    assert np.array_equal(cnt, oracle_perm["cnt"])
    assert np.array_equal(off, oracle_perm["off"])
    assert int(n_active) == oracle_perm["n_active"]
    assert np.array_equal(active, oracle_perm["active"])
    assert int(cnt.sum()) == ids_gpu.size
    flat = np.asarray(ids_gpu).ravel()
    for e in range(E):
        seg = perm[off[e]: off[e + 1]]
        ref = oracle_perm["perm"][off[e]: off[e + 1]]
        assert sorted(seg.tolist()) == sorted(ref.tolist())
        assert np.all(flat[seg] == e)
    assert np.array_equal(perm[pair_pos], np.arange(flat.size))
