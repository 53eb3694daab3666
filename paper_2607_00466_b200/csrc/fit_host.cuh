// ELDR's offline fit -- HOST code: the paper runs it on the CPU before serving ("the balanced
// K-means clustering over the captured signatures completes in under 10 s on CPU") and it is not on the
// decode hot path.  fp64 throughout.
//   IDF table            PAPER.md:199  w(l,e) = log((|C|+1) / (df(l,e)+1))
//   greedy layer mask    PAPER.md:200  append the layer that most increases cumulative rho (Eq. 1, PAPER.md:183:
//                                      Spearman correlation of signature pair distances with decode-pattern pair
//                                      distances), keep the prefix at which cumulative rho peaks
//   balanced K-means     PAPER.md:227  "each centroid takes at most ceil(N/K) points, and the assignment minimizing total
//                                      cosine distance is found by the Hungarian algorithm"; K unit centroids
// Readings where the paper is silent are those of oracle/fit.py.
//
// How it differs from a textbook transcription:
//   * rho of a candidate mask costs O(P), not O(P * |S| * E): per-layer pair dot products D_l(i,j) and per-layer squared
//     norms n_l(i) are computed once; for a mask S, cos(s_i, s_j) = sum_{l in S} D_l(i,j) / sqrt(sum n_l(i) * sum n_l(j)).
//     The greedy search keeps the running sums of the chosen prefix and adds one layer's terms per candidate.
//   * the balanced assignment is solved on the COMPACT graph (N points, K centroids with capacity), not on the
//     N x (K * ceil(N/K)) matrix of duplicated slots: successive shortest augmenting paths where a path moves one point out
//     of each full centroid it crosses.  Each augmentation costs O(N*K + K^3) (edge weights between centroids = the
//     cheapest point to move; Bellman-Ford over K nodes), O(N^2 K) in all instead of O(N^3) -- milliseconds at N = 1000.
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <limits>
#include <numeric>
#include <vector>

namespace eldr_fit {

// 1-based average ranks (ties share the mean of the positions they occupy), centred on their mean
inline void centred_ranks(const std::vector<double>& v, std::vector<double>& r, std::vector<int>& idx) {
  const int n = (int)v.size();
  idx.resize(n);
  std::iota(idx.begin(), idx.end(), 0);
  std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) { return v[a] < v[b]; });
  r.assign(n, 0.0);
  for (int i = 0; i < n;) {
    int j = i;
    while (j + 1 < n && v[idx[j + 1]] == v[idx[i]]) ++j;
    const double rk = 0.5 * (i + j) + 1.0;
    for (int q = i; q <= j; ++q) r[idx[q]] = rk;
    i = j + 1;
  }
  double mean = 0.0;
  for (double x : r) mean += x;
  mean /= n > 0 ? n : 1;
  for (double& x : r) x -= mean;
}

inline double corr_centred(const std::vector<double>& a, const std::vector<double>& b) {
  double ab = 0.0, aa = 0.0, bb = 0.0;
  for (size_t i = 0; i < a.size(); ++i) { ab += a[i] * b[i]; aa += a[i] * a[i]; bb += b[i] * b[i]; }
  const double den = std::sqrt(aa * bb);
  return den > 0.0 ? ab / den : 0.0;
}

inline void idf_table(const int32_t* counts, int N, int L, int E, double* idf) {
  for (int c = 0; c < L * E; ++c) {
    int df = 0;
    for (int r = 0; r < N; ++r) df += counts[(size_t)r * L * E + c] > 0;
    idf[c] = std::log((N + 1.0) / (df + 1.0));
  }
}

// Balanced assignment on the compact graph.  cost [N,K] row-major.  Returns the total cost; assign[i] in [0,K).
inline double balanced_assign(const double* cost, int N, int K, int cap, int32_t* assign) {
  const double INF = std::numeric_limits<double>::infinity();
  std::vector<std::vector<int>> members(K);
  std::vector<double> dist(K), W((size_t)K * K);
  std::vector<int> J((size_t)K * K), par_c(K), par_pt(K);
  for (int i = 0; i < N; ++i) assign[i] = -1;
  for (int i = 0; i < N; ++i) {
    // cheapest point to move from centroid a to centroid b, for every ordered pair
    for (int a = 0; a < K; ++a) {
      for (int b = 0; b < K; ++b) { W[(size_t)a * K + b] = INF; J[(size_t)a * K + b] = -1; }
      for (int j : members[a]) {
        const double* cj = cost + (size_t)j * K;
        for (int b = 0; b < K; ++b) {
          const double w = cj[b] - cj[a];
          if (b != a && w < W[(size_t)a * K + b]) { W[(size_t)a * K + b] = w; J[(size_t)a * K + b] = j; }
        }
      }
    }
    for (int b = 0; b < K; ++b) { dist[b] = cost[(size_t)i * K + b]; par_c[b] = -1; par_pt[b] = i; }
    for (int round = 0; round < K; ++round) {            // Bellman-Ford: the residual graph has no negative cycle
      bool changed = false;
      for (int a = 0; a < K; ++a) {
        if (members[a].empty()) continue;
        for (int b = 0; b < K; ++b) {
          const double w = W[(size_t)a * K + b];
          if (b != a && w < INF && dist[a] + w < dist[b]) {
            dist[b] = dist[a] + w; par_c[b] = a; par_pt[b] = J[(size_t)a * K + b];
            changed = true;
          }
        }
      }
      if (!changed) break;
    }
    int t = -1;
    for (int b = 0; b < K; ++b)
      if ((int)members[b].size() < cap && (t < 0 || dist[b] < dist[t])) t = b;
    // augment: walk the path back from the centroid with a free slot, moving one point per edge
    int b = t;
    for (int guard = 0; par_c[b] >= 0 && guard <= K; ++guard) {
      const int a = par_c[b], j = par_pt[b];
      auto& ma = members[a];
      ma.erase(std::find(ma.begin(), ma.end(), j));
      members[b].push_back(j);
      assign[j] = b;
      b = a;
    }
    members[b].push_back(i);
    assign[i] = b;
  }
  double total = 0.0;
  for (int i = 0; i < N; ++i) total += cost[(size_t)i * K + assign[i]];
  return total;
}

// Hungarian-balanced spherical K-means.  sig [N,d] unit rows; centroids seeded from sig[init_idx[k]].
inline void kmeans_balanced(const double* sig, int N, int d, int K, const int32_t* init_idx, int max_iter,
                            double* cent, int32_t* assign, int32_t* steps, double* total) {
  const int cap = (N + K - 1) / K;
  for (int k = 0; k < K; ++k) std::copy(sig + (size_t)init_idx[k] * d, sig + (size_t)init_idx[k] * d + d, cent + (size_t)k * d);
  std::vector<double> cost((size_t)N * K), mean(d);
  std::vector<int32_t> prev(N, -1), cur(N);
  *steps = 0;
  *total = 0.0;
  for (int it = 0; it < max_iter; ++it) {
    for (int i = 0; i < N; ++i)
      for (int k = 0; k < K; ++k) {
        const double* a = sig + (size_t)i * d;
        const double* c = cent + (size_t)k * d;
        double dot = 0.0;
        for (int q = 0; q < d; ++q) dot += a[q] * c[q];
        cost[(size_t)i * K + k] = 1.0 - dot;
      }
    *total = balanced_assign(cost.data(), N, K, cap, cur.data());
    ++*steps;
    const bool same = it > 0 && cur == prev;
    if (!same) prev = cur;
    if (same) break;
    for (int k = 0; k < K; ++k) {
      std::fill(mean.begin(), mean.end(), 0.0);
      int cnt = 0;
      for (int i = 0; i < N; ++i)
        if (cur[i] == k) {
          const double* a = sig + (size_t)i * d;
          for (int q = 0; q < d; ++q) mean[q] += a[q];
          ++cnt;
        }
      double nrm = 0.0;
      for (int q = 0; q < d; ++q) nrm += mean[q] * mean[q];
      nrm = std::sqrt(nrm);
      if (cnt > 0 && nrm > 0.0)
        for (int q = 0; q < d; ++q) cent[(size_t)k * d + q] = mean[q] / nrm;
    }
  }
  std::copy(prev.begin(), prev.end(), assign);
}

// Greedy layer selection on rho (Eq. 1).  counts [N,L,E] int32, idf [L,E], decode_p [N,L,E], pairs [P,2].
inline void greedy_layer_mask(const int32_t* counts, const double* idf, const double* decode_p, int N, int L, int E,
                              const int32_t* pairs, int P, int32_t* order, double* cum_rho, int32_t* n_star, uint8_t* mask) {
  const size_t LE = (size_t)L * E;
  // decode-pattern pair distances (all layers) and their centred ranks: fixed for the whole search
  std::vector<double> dp(P), rp, tmp;
  std::vector<int> idx;
  {
    std::vector<double> pn(N);
    for (int r = 0; r < N; ++r) {
      double s = 0.0;
      for (size_t c = 0; c < LE; ++c) s += decode_p[r * LE + c] * decode_p[r * LE + c];
      pn[r] = std::sqrt(s);
    }
    for (int p = 0; p < P; ++p) {
      const int i = pairs[2 * p], j = pairs[2 * p + 1];
      double dot = 0.0;
      for (size_t c = 0; c < LE; ++c) dot += decode_p[i * LE + c] * decode_p[j * LE + c];
      dp[p] = 1.0 - ((pn[i] > 0 && pn[j] > 0) ? dot / (pn[i] * pn[j]) : 0.0);
    }
    centred_ranks(dp, rp, idx);
  }
  // per-layer pieces of the reweighted counts: squared norms n_l(i) and pair dot products D_l(i,j)
  std::vector<double> nl((size_t)L * N), Dl((size_t)L * P), x((size_t)N * E);
  for (int l = 0; l < L; ++l) {
    for (int r = 0; r < N; ++r) {
      double s = 0.0;
      for (int e = 0; e < E; ++e) {
        const double v = (double)counts[r * LE + (size_t)l * E + e] * idf[(size_t)l * E + e];
        x[(size_t)r * E + e] = v;
        s += v * v;
      }
      nl[(size_t)l * N + r] = s;
    }
    for (int p = 0; p < P; ++p) {
      const double* a = &x[(size_t)pairs[2 * p] * E];
      const double* b = &x[(size_t)pairs[2 * p + 1] * E];
      double dot = 0.0;
      for (int e = 0; e < E; ++e) dot += a[e] * b[e];
      Dl[(size_t)l * P + p] = dot;
    }
  }
  std::vector<double> accD(P, 0.0), accN(N, 0.0), ds(P), rs;
  std::vector<char> used(L, 0);
  auto rho_with = [&](int l) {
    for (int p = 0; p < P; ++p) {
      const int i = pairs[2 * p], j = pairs[2 * p + 1];
      const double ni = accN[i] + nl[(size_t)l * N + i], nj = accN[j] + nl[(size_t)l * N + j];
      const double dot = accD[p] + Dl[(size_t)l * P + p];
      ds[p] = 1.0 - ((ni > 0 && nj > 0) ? dot / (std::sqrt(ni) * std::sqrt(nj)) : 0.0);
    }
    centred_ranks(ds, rs, idx);
    return corr_centred(rs, rp);
  };
  for (int step = 0; step < L; ++step) {
    int best = -1;
    double best_rho = -std::numeric_limits<double>::infinity();
    for (int l = 0; l < L; ++l) {
      if (used[l]) continue;
      const double r = rho_with(l);
      if (r > best_rho) { best = l; best_rho = r; }
    }
    used[best] = 1;
    order[step] = best;
    cum_rho[step] = best_rho;
    for (int p = 0; p < P; ++p) accD[p] += Dl[(size_t)best * P + p];
    for (int r = 0; r < N; ++r) accN[r] += nl[(size_t)best * N + r];
  }
  int ns = 0;
  for (int s = 1; s < L; ++s)
    if (cum_rho[s] > cum_rho[ns]) ns = s;
  *n_star = ns + 1;
  for (int l = 0; l < L; ++l) mask[l] = 0;
  for (int s = 0; s <= ns; ++s) mask[order[s]] = 1;
}

}  // namespace eldr_fit
