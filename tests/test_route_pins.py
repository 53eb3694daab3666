"""Pins of the routing-decision oracle (PAPER.md:196-203 signature steps 2-4, PAPER.md:239
locality-band routing) against what the paper and the mathematics fix -- none of them re-types the oracle's loop."""
import os

import numpy as np
import pytest

from oracle import oracle
from paper_2607_00466_b200 import synth

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "route_example.txt")


def _wl(R=24, L=6, E=16, K=5, k=2, seed=7, **kw):
    w = synth.make_route_workload(R, L, E, K, k, seed, prompt_len=(64, 256), **kw)
    idf = oracle.idf_table(w.df, w.n_calib)
    return w, idf


def _numpy_cosine(w, idf):
    """Independent route to the similarities: numpy normalise + matmul on the masked, reweighted vectors."""
    m = w.layer_mask.astype(bool)
    x = (w.counts.astype(np.float64) * idf[None])[:, m, :].reshape(w.counts.shape[0], -1)
    c = w.centroids.astype(np.float64)[:, m, :].reshape(w.centroids.shape[0], -1)
    x = x / np.linalg.norm(x, axis=1, keepdims=True)
    c = c / np.linalg.norm(c, axis=1, keepdims=True)
    return x @ c.T


def test_hand_worked_example_and_idf_closed_form():
    rows = [l.split() for l in open(GOLD) if l.strip() and not l.startswith("#")]
    counts = np.array([[[3, 4]]], np.int32)
    idf = np.ones((1, 2))
    mask = np.ones(1, np.uint8)
    cen = np.array([[[1.0, 0.0]], [[0.0, 1.0]]])
    n_cases = 0
    for r in rows:
        if r[0] == "IDF":
            got = oracle.idf_table(np.array([[int(r[2])]], np.int32), int(r[1]))
            assert got[0, 0] == pytest.approx(float(r[3]), abs=1e-15)
            continue
        tau, l0, l1, s0, s1, wk, n0, n1 = float(r[1]), int(r[2]), int(r[3]), float(r[4]), float(r[5]), int(r[6]), int(r[7]), int(r[8])
        loads = np.array([l0, l1], np.int64)
        o = oracle.route_decide(counts, idf, mask, cen, loads, tau)
        assert o["sims"][0] == pytest.approx([s0, s1], abs=1e-15)
        assert int(o["worker"][0]) == wk and loads.tolist() == [n0, n1]
        n_cases += 1
    assert n_cases == 3


def test_similarities_match_numpy_and_tau0_is_top1():
    w, idf = _wl()
    ref = _numpy_cosine(w, idf)
    loads = w.loads.astype(np.int64)
    o = oracle.route_decide(w.counts, idf, w.layer_mask, w.centroids.astype(np.float64), loads, 0.0)
    assert np.abs(o["sims"] - ref).max() <= 1e-12
    assert np.array_equal(o["worker"], ref.argmax(1))                # tau = 0: pure top-1 routing
    assert loads.sum() == w.loads.sum() + w.counts.shape[0]           # every request dispatched exactly once


def test_tau1_is_join_shortest_queue():
    """Non-negative signatures and centroids have similarities in [0,1], so tau = 1 puts every worker in the band:
    pure shortest-queue routing.  From equal loads, m*K requests leave every worker with m more."""
    w, idf = _wl(R=20, K=5)
    loads = np.full(5, 3, np.int64)
    o = oracle.route_decide(w.counts, idf, w.layer_mask, w.centroids.astype(np.float64), loads, 1.0)
    assert loads.tolist() == [7] * 5
    # and each single decision went to a worker that was least loaded at that moment
    cur = np.full(5, 3, np.int64)
    for r in range(20):
        assert cur[o["worker"][r]] == cur.min()
        cur[o["worker"][r]] += 1


def test_band_rule_by_brute_force():
    """Replay the decisions from the similarities alone: the pick is in the band, no band member has a smaller
    load, and among equal loads none has a larger similarity."""
    w, idf = _wl(R=40, K=6, seed=11)
    loads0 = w.loads.astype(np.int64)
    loads = loads0.copy()
    tau = 0.25                      # wide enough that many bands hold several workers on this workload
    o = oracle.route_decide(w.counts, idf, w.layer_mask, w.centroids.astype(np.float64), loads, tau)
    cur = loads0.copy()
    sizes = []
    for r in range(40):
        s = o["sims"][r]
        band = np.nonzero(s >= s.max() - tau)[0]
        p = int(o["worker"][r])
        assert p in band
        assert cur[p] == cur[band].min()
        ties = band[cur[band] == cur[p]]
        assert s[p] == s[ties].max()
        cur[p] += 1
        sizes.append(len(band))
    assert np.array_equal(cur, loads) and max(sizes) > 1 and min(sizes) >= 1


def test_scale_invariance_masked_layers_and_unnormalised_centroids():
    w, idf = _wl(seed=3)
    cen = w.centroids.astype(np.float64)
    base = oracle.route_decide(w.counts, idf, w.layer_mask, cen, w.loads.astype(np.int64), 0.1)
    # Eq. 2: the token count of the request does not matter
    o = oracle.route_decide(w.counts * 3, idf, w.layer_mask, cen, w.loads.astype(np.int64), 0.1)
    assert np.abs(o["sims"] - base["sims"]).max() <= 1e-12 and np.array_equal(o["worker"], base["worker"])
    # layers outside S do not matter, neither in the counts nor in the centroids
    c2, cen2 = w.counts.copy(), cen.copy()
    off = np.nonzero(w.layer_mask == 0)[0]
    assert off.size > 0
    c2[:, off, :] = 12345
    cen2[:, off, :] = 77.0
    o = oracle.route_decide(c2, idf, w.layer_mask, cen2, w.loads.astype(np.int64), 0.1)
    assert np.array_equal(o["sims"], base["sims"]) and np.array_equal(o["worker"], base["worker"])
    # cosine: scaling a centroid changes nothing
    cen3 = cen * np.arange(1, cen.shape[0] + 1)[:, None, None]
    o = oracle.route_decide(w.counts, idf, w.layer_mask, cen3, w.loads.astype(np.int64), 0.1)
    assert np.abs(o["sims"] - base["sims"]).max() <= 1e-12 and np.array_equal(o["worker"], base["worker"])


def test_idf_downweights_generalists_and_empty_request():
    w, idf = _wl(seed=5)
    ref = np.log((w.n_calib + 1.0) / (w.df.astype(np.float64) + 1.0))      # PAPER.md:199, via numpy
    assert np.abs(idf - ref).max() <= 1e-15 and idf.min() >= 0.0
    gen = np.nonzero(w.df[0] > w.n_calib // 2)[0]
    assert gen.size > 0 and idf[:, gen].max() < idf[:, np.setdiff1d(np.arange(w.df.shape[1]), gen)].min()
    # a request with no counts has similarity 0 to everything: the band is everybody, it joins the shortest queue
    c = w.counts.copy()
    c[0] = 0
    loads = w.loads.astype(np.int64)
    want = int(np.argmin(loads))
    o = oracle.route_decide(c[:1], idf, w.layer_mask, w.centroids.astype(np.float64), loads, 0.1)
    assert np.all(o["sims"][0] == 0.0) and w.loads[int(o["worker"][0])] == w.loads.min() and int(o["worker"][0]) == want
