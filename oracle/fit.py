"""TEST INFRASTRUCTURE ONLY -- fp64 oracle of ELDR's OFFLINE FIT: the IDF table, the greedy layer
mask and the Hungarian-balanced K-means over calibration signatures.  Plain numpy / scipy, step by step in the paper's
order and notation; no blocking, no shortcuts.  Only tests/ and bench.py's cpu_baseline leg may import this module.

PAPER.md:199 (section 4.2.2 step 2)  w(l,e) = log((|C|+1) / (df(l,e)+1)), df = calibration requests in which expert e
                                      fires at least once at layer l;  c~_r(l,e) = c_r(l,e) * w(l,e).
PAPER.md:200 (step 3)                 "greedy layer selection on rho: starting from an empty mask, the layer whose
                                      inclusion most increases cumulative rho is appended at each step, producing an
                                      ordering of all L layers.  We keep the first N* layers in this ordering, where N* is
                                      the size at which cumulative rho peaks".
PAPER.md:183 (Eq. 1)                  rho = Spearman(cos-dist(s_i, s_j), cos-dist(p_i, p_j)) over random calibration pairs,
                                      p_i = the request's decode-time activation probabilities, flattened over (l,e).
PAPER.md:203 (Eq. 2)                  s_r = x_r / ||x_r||_2,  x_r = [c~_r(l)]_{l in S}.
PAPER.md:227 (section 4.3.1)          "Hungarian-balanced K-means, which replaces nearest-neighbor assignment with a
                                      globally optimal assignment: each centroid takes at most ceil(N/K) points, and the
                                      assignment minimizing total cosine distance is found by the Hungarian algorithm";
                                      "K unit centroids".

Readings where the paper is silent (also DESIGN.md 9d):
  * the "random calibration pairs" and the K initial centroids are INPUTS (pairs [P,2]; init_idx [K] = calibration
    requests whose signatures seed the centroids) -- the method's random draws are passed in;
  * Spearman with average ranks for ties; a constant vector has correlation 0;
  * cos-dist = 1 - cosine; a zero vector has cosine 0 with everything (distance 1);
  * greedy ties -> the lowest layer index; N* = the FIRST size at which cumulative rho attains its maximum;
  * K-means update: centroid = mean of the assigned unit signatures, renormalised to unit length ("unit centroids");
    a centroid left without points, or with a zero mean, keeps its previous value; the iteration stops when the
    assignment repeats or after max_iter assignment steps;
  * among equally cheap optimal assignments any one is acceptable (tests compare total cost and the balance bound,
    and the assignment itself only on generic real-valued data, where it is unique).
"""
import numpy as np
from scipy.optimize import linear_sum_assignment


def idf_table(counts: np.ndarray) -> np.ndarray:
    """counts [N,L,E] -> w [L,E] fp64."""
    counts = np.asarray(counts)
    n = counts.shape[0]
    df = (counts > 0).sum(axis=0)
    return np.log((n + 1.0) / (df + 1.0))


def average_ranks(v: np.ndarray) -> np.ndarray:
    """1-based ranks, ties share the mean of the positions they occupy."""
    v = np.asarray(v, np.float64)
    order = np.argsort(v, kind="stable")
    ranks = np.empty(len(v), np.float64)
    i = 0
    while i < len(v):
        j = i
        while j + 1 < len(v) and v[order[j + 1]] == v[order[i]]:
            j += 1
        ranks[order[i:j + 1]] = 0.5 * (i + j) + 1.0
        i = j + 1
    return ranks


def spearman(a: np.ndarray, b: np.ndarray) -> float:
    ra, rb = average_ranks(a), average_ranks(b)
    ra -= ra.mean()
    rb -= rb.mean()
    den = np.sqrt((ra * ra).sum() * (rb * rb).sum())
    return float((ra * rb).sum() / den) if den > 0 else 0.0


def cos_dist_pairs(x: np.ndarray, pairs: np.ndarray) -> np.ndarray:
    """x [N,d], pairs [P,2] -> 1 - cosine(x_i, x_j); a zero vector has cosine 0."""
    x = np.asarray(x, np.float64)
    out = np.empty(len(pairs), np.float64)
    for p, (i, j) in enumerate(pairs):
        ni, nj = np.sqrt((x[i] * x[i]).sum()), np.sqrt((x[j] * x[j]).sum())
        out[p] = 1.0 - ((x[i] * x[j]).sum() / (ni * nj) if ni > 0 and nj > 0 else 0.0)
    return out


def signature_quality(counts, idf, layers, decode_p, pairs) -> float:
    """rho (Eq. 1) of the signature built on the layer subset `layers`."""
    n = counts.shape[0]
    x = (np.asarray(counts, np.float64) * idf[None])[:, list(layers), :].reshape(n, -1)
    ds = cos_dist_pairs(x, pairs)
    dp = cos_dist_pairs(np.asarray(decode_p, np.float64).reshape(n, -1), pairs)
    return spearman(ds, dp)


def greedy_layer_mask(counts, idf, decode_p, pairs):
    """-> order [L], cum_rho [L], n_star, mask [L] uint8."""
    L = counts.shape[1]
    order, cum = [], []
    for _ in range(L):
        best, best_rho = -1, -np.inf
        for l in range(L):
            if l in order:
                continue
            r = signature_quality(counts, idf, order + [l], decode_p, pairs)
            if r > best_rho:
                best, best_rho = l, r
        order.append(best)
        cum.append(best_rho)
    cum = np.array(cum)
    n_star = int(np.argmax(cum)) + 1
    mask = np.zeros(L, np.uint8)
    mask[order[:n_star]] = 1
    return np.array(order, np.int32), cum, n_star, mask


def signatures(counts, idf, mask) -> np.ndarray:
    """s_r = x_r / ||x_r||_2 on the kept layers (Eq. 2); [N, n_kept*E] fp64; a zero x_r stays zero."""
    n = counts.shape[0]
    x = (np.asarray(counts, np.float64) * idf[None])[:, np.nonzero(mask)[0], :].reshape(n, -1)
    nrm = np.sqrt((x * x).sum(axis=1, keepdims=True))
    return np.divide(x, nrm, out=np.zeros_like(x), where=nrm > 0)


def balanced_assign(cost: np.ndarray, cap: int):
    """cost [N,K], each centroid at most `cap` points: every centroid is expanded into `cap` identical slots and the
    Hungarian algorithm (scipy's linear_sum_assignment) solves the N x (K*cap) assignment.  -> assign [N], total cost."""
    cost = np.asarray(cost, np.float64)
    n, k = cost.shape
    assert k * cap >= n
    rows, cols = linear_sum_assignment(np.repeat(cost, cap, axis=1))
    assign = np.empty(n, np.int32)
    assign[rows] = (cols // cap).astype(np.int32)
    return assign, float(cost[np.arange(n), assign].sum())


def kmeans_balanced(sig: np.ndarray, K: int, init_idx, max_iter: int = 50):
    """Hungarian-balanced spherical K-means.  sig [N,d] unit rows -> centroids [K,d], assign [N],
    assignment steps run, total cosine distance of the final assignment to the centroids it was computed against."""
    sig = np.asarray(sig, np.float64)
    n = sig.shape[0]
    cap = -(-n // K)
    cent = sig[np.asarray(init_idx)].copy()
    assign, total, steps = None, 0.0, 0
    for _ in range(max_iter):
        cost = 1.0 - sig @ cent.T
        new_assign, total = balanced_assign(cost, cap)
        steps += 1
        if assign is not None and np.array_equal(new_assign, assign):
            break
        assign = new_assign
        for k in range(K):
            members = sig[assign == k]
            if len(members):
                mean = members.sum(axis=0)
                nrm = np.sqrt((mean * mean).sum())
                if nrm > 0:
                    cent[k] = mean / nrm
    return cent, assign, steps, total
