"""Pins of the offline-fit oracle (oracle/fit.py): library routines
(scipy.stats.spearmanr / rankdata), brute force over all assignments on tiny cases, closed forms and invariants -- chosen
so that a dropped term, a wrong sign or a transposed operand in the oracle fails one of them."""
import itertools

import numpy as np
import pytest
from scipy import stats

from oracle import fit


def _calib(n, L, E, seed, n_domains=3):
    """Seeded calibration stand-in: domains with specialist experts on SOME layers only (the others carry noise), a few
    generalist experts everywhere; decode patterns follow the same domain prototypes."""
    g = np.random.default_rng(seed)
    informative = g.permutation(L)[: max(1, L // 2)]
    proto = np.full((n_domains, L, E), 0.05)
    for d in range(n_domains):
        for l in informative:
            proto[d, l, g.permutation(E)[:2]] += 3.0
    proto[:, :, 0] += 2.0                                    # a generalist
    dom = g.integers(0, n_domains, size=n)
    counts = np.empty((n, L, E), np.int32)
    dec = np.empty((n, L, E))
    for r in range(n):
        p = proto[dom[r]] / proto[dom[r]].sum(axis=1, keepdims=True)
        for l in range(L):
            counts[r, l] = g.multinomial(12, p[l] if l in informative else np.full(E, 1.0 / E))      # few tokens: rare experts have df < N
            dec[r, l] = np.clip(p[l] * 4 + 0.05 * g.random(E), 0, 1)
    return counts, dec, dom


def test_idf_closed_form_and_numpy():
    counts = np.zeros((3, 2, 4), np.int32)
    counts[0, 0, 1] = 5
    counts[1, 0, 1] = 1
    counts[2, 1, 3] = 2
    w = fit.idf_table(counts)
    assert w[0, 1] == np.log(4 / 3) and w[1, 3] == np.log(4 / 2) and w[0, 0] == np.log(4 / 1)
    c, _, _ = _calib(40, 3, 6, 1)
    assert np.allclose(fit.idf_table(c), np.log(41.0 / ((c > 0).sum(0) + 1.0)), rtol=0, atol=0)


def test_ranks_and_spearman_against_scipy():
    g = np.random.default_rng(2)
    for n in (2, 7, 50):
        a, b = g.integers(0, 6, n).astype(float), g.standard_normal(n)          # ties in a
        assert np.array_equal(fit.average_ranks(a), stats.rankdata(a, method="average"))
        if n > 2:
            assert abs(fit.spearman(a, b) - stats.spearmanr(a, b)[0]) < 1e-12
    assert fit.spearman(np.arange(5.0), np.arange(5.0) ** 3) == pytest.approx(1.0)
    assert fit.spearman(np.arange(5.0), -np.arange(5.0)) == pytest.approx(-1.0)
    assert fit.spearman(np.ones(4), np.arange(4.0)) == 0.0                         # reading: constant -> 0


def test_cos_dist_pairs_closed_forms():
    x = np.array([[1.0, 0.0], [0.0, 2.0], [3.0, 0.0], [-1.0, 0.0], [0.0, 0.0], [1.0, 1.0]])
    pairs = np.array([[0, 1], [0, 2], [0, 3], [0, 4], [0, 5]])
    assert np.allclose(fit.cos_dist_pairs(x, pairs), [1.0, 0.0, 2.0, 1.0, 1.0 - 1.0 / np.sqrt(2.0)])


def test_signature_quality_matches_an_independent_formulation():
    counts, dec, _ = _calib(30, 4, 5, 3)
    idf = fit.idf_table(counts)
    g = np.random.default_rng(4)
    pairs = g.integers(0, 30, size=(60, 2))
    layers = [2, 0]
    x = np.stack([np.concatenate([counts[r, l] * idf[l] for l in layers]) for r in range(30)])
    xs = x / np.linalg.norm(x, axis=1, keepdims=True)
    p = dec.reshape(30, -1)
    ps = p / np.linalg.norm(p, axis=1, keepdims=True)
    ds = [1.0 - xs[i] @ xs[j] for i, j in pairs]
    dp = [1.0 - ps[i] @ ps[j] for i, j in pairs]
    assert abs(fit.signature_quality(counts, idf, layers, dec, pairs) - stats.spearmanr(ds, dp)[0]) < 1e-12


def test_greedy_layer_mask_is_the_greedy_order_by_brute_force():
    counts, dec, _ = _calib(24, 4, 5, 5)
    idf = fit.idf_table(counts)
    pairs = np.array(list(itertools.combinations(range(24), 2)))[::3]
    order, cum, n_star, mask = fit.greedy_layer_mask(counts, idf, dec, pairs)
    assert sorted(order.tolist()) == [0, 1, 2, 3]
    chosen = []
    for step in range(4):                                   # replay: every step's pick maximises rho over the remaining layers
        cands = {l: fit.signature_quality(counts, idf, chosen + [l], dec, pairs) for l in range(4) if l not in chosen}
        best = max(cands.values())
        assert cands[int(order[step])] == best and cum[step] == best
        chosen.append(int(order[step]))
    assert n_star == int(np.argmax(cum)) + 1 and mask.sum() == n_star and set(np.nonzero(mask)[0]) == set(order[:n_star].tolist())
    # an uninformative (uniform-noise) layer must not be picked first
    counts2, dec2, _ = _calib(40, 6, 8, 6)
    o2, c2, n2, m2 = fit.greedy_layer_mask(counts2, fit.idf_table(counts2), dec2, np.array(list(itertools.combinations(range(40), 2)))[::7])
    assert c2[n2 - 1] >= c2[-1]                              # the kept prefix is at least as good as all layers (Fig. 8)


def test_signatures_are_unit_rows_on_the_kept_layers():
    counts, _, _ = _calib(10, 3, 4, 7)
    idf = fit.idf_table(counts)
    s = fit.signatures(counts, idf, np.array([1, 0, 1], np.uint8))
    assert s.shape == (10, 8) and np.allclose(np.linalg.norm(s, axis=1), 1.0)
    assert np.allclose(s[3] * np.linalg.norm(np.concatenate([counts[3, 0] * idf[0], counts[3, 2] * idf[2]])),
                       np.concatenate([counts[3, 0] * idf[0], counts[3, 2] * idf[2]]))


def test_balanced_assign_is_optimal_and_balanced_by_brute_force():
    g = np.random.default_rng(8)
    for n, k in ((4, 2), (5, 2), (6, 3), (7, 3)):
        cap = -(-n // k)
        cost = g.random((n, k))
        assign, total = fit.balanced_assign(cost, cap)
        assert np.bincount(assign, minlength=k).max() <= cap
        best = min(sum(cost[i, a[i]] for i in range(n)) for a in itertools.product(range(k), repeat=n)
                   if np.bincount(a, minlength=k).max() <= cap)
        assert abs(total - best) < 1e-12 and abs(cost[np.arange(n), assign].sum() - best) < 1e-12
    # with room for everyone (cap = N) the constraint is inactive: nearest centroid
    cost = g.random((9, 3))
    assign, _ = fit.balanced_assign(cost, 9)
    assert np.array_equal(assign, cost.argmin(axis=1))


def test_kmeans_balanced_invariants_and_well_separated_clusters():
    g = np.random.default_rng(9)
    K, per, d = 3, 7, 12
    base = np.eye(d)[:K] * 5.0
    pts = np.concatenate([base[k] + 0.1 * g.random((per, d)) for k in range(K)])
    pts /= np.linalg.norm(pts, axis=1, keepdims=True)
    perm = g.permutation(K * per)
    pts, truth = pts[perm], np.repeat(np.arange(K), per)[perm]
    init = [int(np.nonzero(truth == k)[0][0]) for k in range(K)]
    cent, assign, steps, total = fit.kmeans_balanced(pts, K, init)
    assert np.array_equal(assign, truth) and steps >= 2
    assert np.allclose(np.linalg.norm(cent, axis=1), 1.0)
    for k in range(K):                                       # centroid = renormalised mean of its members
        m = pts[assign == k].sum(0)
        assert np.allclose(cent[k], m / np.linalg.norm(m))
    assert abs(total - (1.0 - (pts * cent[assign]).sum(1)).sum()) < 1e-12
    # skewed data: 15 points near one direction, 3 + 3 near two others; K = 3 -> every cluster holds exactly 7
    skew = np.concatenate([base[0] + 0.3 * g.random((15, d)), base[1] + 0.3 * g.random((3, d)), base[2] + 0.3 * g.random((3, d))])
    skew /= np.linalg.norm(skew, axis=1, keepdims=True)
    _, a2, _, _ = fit.kmeans_balanced(skew, 3, [0, 15, 18])
    assert np.bincount(a2, minlength=3).tolist() == [7, 7, 7]
