"""Parity of the library's offline fit (host functions of libeldr_moe.so: eldr_fit_*) against the
fp64 oracle oracle/fit.py, through the C ABI.  No GPU needed -- the paper fits on the CPU -- so these
run in the CPU suite.  Integer results (layer order, N*, mask, assignments, step counts) are compared exactly on
generic real-valued data (where the optimum is unique); floating-point results to 1e-9."""
import itertools

import numpy as np
import pytest
from scipy.optimize import linear_sum_assignment

from oracle import fit
from test_fit_pins import _calib


@pytest.fixture(scope="module")
def lib():
    from paper_2607_00466_b200 import api
    api.load(build_if_missing=True)
    return api


def test_idf_matches_oracle(lib):
    counts, _, _ = _calib(200, 6, 16, 11)
    assert np.array_equal(lib.eldr_fit_idf(counts), fit.idf_table(counts))


@pytest.mark.parametrize("n,L,E,seed", [(40, 5, 24, 5), (60, 8, 32, 21), (120, 12, 16, 22)])
def test_layer_mask_matches_oracle(lib, n, L, E, seed):
    """Distinct pairs of distinct requests with generic count vectors: exactly tied pair distances (two requests with the
    same counts, a pair listed twice) would make the ranks depend on the last bit of the distance, i.e. on the summation
    order, which the oracle (one flat dot product) and the library (per-layer partial sums) do not share."""
    counts, dec, _ = _calib(n, L, E, seed)
    idf = fit.idf_table(counts)
    g = np.random.default_rng(seed)
    allp = np.array(list(itertools.combinations(range(n), 2)), np.int32)
    pairs = allp[g.permutation(len(allp))[:400]]
    assert len({counts[r].tobytes() for r in range(n)}) == n
    o_order, o_cum, o_ns, o_mask = fit.greedy_layer_mask(counts, idf, dec, pairs)
    order, cum, ns, mask = lib.eldr_fit_layer_mask(counts, idf, dec, pairs)
    assert np.array_equal(order, o_order) and ns == o_ns and np.array_equal(mask, o_mask)
    assert np.abs(cum - o_cum).max() <= 1e-9


@pytest.mark.parametrize("n,k,seed", [(5, 2, 1), (7, 3, 2), (40, 4, 3), (203, 8, 4), (500, 16, 5), (64, 64, 6)])
def test_balanced_assign_matches_the_hungarian_algorithm(lib, n, k, seed):
    g = np.random.default_rng(seed)
    cap = -(-n // k)
    cost = g.random((n, k))
    assign, total = lib.eldr_fit_balanced_assign(cost, cap)
    o_assign, o_total = fit.balanced_assign(cost, cap)
    assert np.bincount(assign, minlength=k).max() <= cap and assign.min() >= 0
    assert abs(total - o_total) <= 1e-9 and np.array_equal(assign, o_assign)
    if n <= 7:                                              # and against brute force over all assignments
        best = min(sum(cost[i, a[i]] for i in range(n)) for a in itertools.product(range(k), repeat=n)
                   if np.bincount(a, minlength=k).max() <= cap)
        assert abs(total - best) <= 1e-12


def test_balanced_assign_degenerate_costs_keep_the_bound_and_the_optimum(lib):
    """Many exact ties (integer costs): several optimal assignments exist; the total and the bound are what is unique."""
    g = np.random.default_rng(9)
    cost = g.integers(0, 3, size=(90, 6)).astype(np.float64)
    assign, total = lib.eldr_fit_balanced_assign(cost, 15)
    rows, cols = linear_sum_assignment(np.repeat(cost, 15, axis=1))
    assert total == cost[rows, cols // 15].sum() and np.bincount(assign, minlength=6).max() <= 15
    with pytest.raises(RuntimeError):
        lib.eldr_fit_balanced_assign(cost, 14)               # K * cap < N


@pytest.mark.parametrize("n,d,K,seed", [(21, 12, 3, 9), (160, 40, 8, 10), (301, 64, 7, 11)])
def test_kmeans_balanced_matches_oracle(lib, n, d, K, seed):
    g = np.random.default_rng(seed)
    centres = g.random((K, d)) ** 6
    pts = centres[g.integers(0, max(1, K // 2), size=n)] + 0.15 * g.random((n, d))       # skewed: half of the centres are empty
    pts /= np.linalg.norm(pts, axis=1, keepdims=True)
    init = g.permutation(n)[:K].astype(np.int32)
    o_cent, o_assign, o_steps, o_total = fit.kmeans_balanced(pts, K, init, max_iter=30)
    cent, assign, steps, total = lib.eldr_fit_kmeans_balanced(pts, K, init, max_iter=30)
    assert steps == o_steps and np.array_equal(assign, o_assign)
    assert np.abs(cent - o_cent).max() <= 1e-9 and abs(total - o_total) <= 1e-9
    assert np.bincount(assign, minlength=K).max() <= -(-n // K)                            # at most ceil(N/K) points
    assert np.allclose(np.linalg.norm(cent, axis=1), 1.0)


def test_fit_to_route_chain_on_a_qwen_shaped_signature_space(lib):
    """The whole offline stage at the paper's scale ("under 10 s on CPU"): 1000 calibration requests, 48 layers
    x 128 experts -> IDF, greedy mask, Eq. 2 signatures, K = 8 balanced centroids; every cluster holds exactly 125."""
    import time
    counts, dec, dom = _calib(1000, 48, 128, 33, n_domains=8)
    g = np.random.default_rng(33)
    pairs = g.integers(0, 1000, size=(2000, 2)).astype(np.int32)
    t0 = time.perf_counter()
    idf = lib.eldr_fit_idf(counts)
    order, cum, ns, mask = lib.eldr_fit_layer_mask(counts, idf, dec, pairs)
    sig = fit.signatures(counts, idf, mask)                                                # Eq. 2 (input preparation for the clustering)
    cent, assign, steps, total = lib.eldr_fit_kmeans_balanced(sig, 8, g.permutation(1000)[:8].astype(np.int32), 50)
    dt = time.perf_counter() - t0
    assert np.bincount(assign, minlength=8).tolist() == [125] * 8
    assert 1 <= ns <= 48 and cum[ns - 1] == cum.max() and cum[ns - 1] > 0.5
    assert dt < 60.0, "offline fit took %.1f s" % dt
