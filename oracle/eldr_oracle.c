/*
 * eldr_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of what the ELDR decode-MoE hot path computes, written from the
 * paper (/root/reference/PAPER.md, cited per function as PAPER.md:<line>) and, where the paper is
 * silent, from the readings listed in DESIGN.md ("Readings of the paper").  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 * It shares no code, header, table or helper with the CUDA path (paper_2607_00466_b200/csrc).
 *
 * The GPU path computes exactly the standard definition ("expert selections -- and
 * hence outputs -- are identical to standard top-k gating"), so the oracle is that definition
 * written densely: no blocking, no fusion, no reordering.  Inputs are the same bits the GPU gets
 * (bf16 as uint16 patterns, fp32 gate), widened exactly to double.
 *
 * Pins (tests/test_oracle_pins.py): gate logits vs numpy fp64 matmul; renormalised weights vs the
 * closed form softmax over the k selected logits; brute-force subset maximisation for E<=8;
 * shift invariance; identical-experts => dense SwiGLU FFN (numpy); k=1; k=E; W3=0 => 0; W2 doubling;
 * a second, differently organised formulation ("all experts, masked"); the hand-worked 4-expert
 * example in tests/golden/hand_example.txt; signature sum / block-sum / prefix-sharing invariants.
 * The paper prints no numeric worked example for this path; beyond the pins above: parity unpinned.
 *
 * OpenMP (over tokens) is a compile-time option used only to report the multi-core CPU baseline;
 * results do not depend on the thread count (each token is computed by one thread, serially).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
  int32_t hidden;        /* H */
  int32_t inter;         /* I */
  int32_t n_experts;     /* E routed experts */
  int32_t top_k;         /* k */
  int32_t n_shared;      /* always-on shared experts */
  int32_t renormalize;   /* 1: w /= sum over the top-k */
  int32_t n_layers;      /* L */
  int32_t kv_block_size; /* tokens per KV block */
} oracle_shape_t;

static double bf16_to_double(uint16_t b) {
  uint32_t u = ((uint32_t)b) << 16;
  float f;
  memcpy(&f, &u, 4);
  return (double)f;
}

int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void oracle_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

/* ------------------------------------------------------------------------------------------------
 * Gate for one token.  PAPER.md:89 "The gate scores experts using the token's hidden representation
 * and dispatches the token to the top-scoring experts"; "standard top-k gating".
 * Reading (R1): z = x.Wg^T (+bias); p = softmax over ALL E routed experts; the k largest
 * z, ties to the lower expert id, listed z-descending; w_j = p_j / sum_{i in topk} p_i if renormalize.
 * Experts are distinct per token ("indicator that an expert appears in the top-k").
 * margin = z_(k) - z_(k+1) (near-tie classifier, north_star: "near-ties within 1e-5").
 * ---------------------------------------------------------------------------------------------- */
static void gate_one_token(const oracle_shape_t *s, const uint16_t *x, const float *gate_w,
                           const float *gate_bias, double *z, int32_t *ids, double *w,
                           double *margin) {
  const int H = s->hidden, E = s->n_experts, k = s->top_k;
  for (int e = 0; e < E; ++e) {
    double acc = 0.0;
    for (int h = 0; h < H; ++h) acc += bf16_to_double(x[h]) * (double)gate_w[(size_t)e * H + h];
    if (gate_bias) acc += (double)gate_bias[e];
    z[e] = acc;
  }
  /* softmax over all E, max-subtracted */
  double zmax = z[0];
  for (int e = 1; e < E; ++e)
    if (z[e] > zmax) zmax = z[e];
  double *p = (double *)malloc(sizeof(double) * (size_t)E);
  double denom = 0.0;
  for (int e = 0; e < E; ++e) {
    p[e] = exp(z[e] - zmax);
    denom += p[e];
  }
  for (int e = 0; e < E; ++e) p[e] /= denom;
  /* top-k by selection: largest z first, ties -> lower id */
  char *taken = (char *)calloc((size_t)E, 1);
  for (int j = 0; j < k; ++j) {
    int best = -1;
    for (int e = 0; e < E; ++e) {
      if (taken[e]) continue;
      if (best < 0 || z[e] > z[best]) best = e; /* strict > keeps the lower id on ties */
    }
    taken[best] = 1;
    ids[j] = best;
  }
  if (margin) {
    if (k < E) {
      int nxt = -1;
      for (int e = 0; e < E; ++e) {
        if (taken[e]) continue;
        if (nxt < 0 || z[e] > z[nxt]) nxt = e;
      }
      *margin = z[ids[k - 1]] - z[nxt];
    } else {
      *margin = INFINITY;
    }
  }
  double sel = 0.0;
  for (int j = 0; j < k; ++j) sel += p[ids[j]];
  for (int j = 0; j < k; ++j) w[j] = s->renormalize ? p[ids[j]] / sel : p[ids[j]];
  free(taken);
  free(p);
}

int oracle_gate_topk(const oracle_shape_t *s, int32_t T, const uint16_t *x, const float *gate_w,
                     const float *gate_bias, double *z_out /*[T,E] or NULL*/,
                     int32_t *ids /*[T,k]*/, double *w /*[T,k]*/, double *margin /*[T] or NULL*/) {
  if (!s || s->top_k < 1 || s->top_k > s->n_experts) return -1;
  const int H = s->hidden, E = s->n_experts, k = s->top_k;
#pragma omp parallel for schedule(dynamic, 1)
  for (int t = 0; t < T; ++t) {
    double *z = (double *)malloc(sizeof(double) * (size_t)E);
    gate_one_token(s, x + (size_t)t * H, gate_w, gate_bias, z, ids + (size_t)t * k,
                   w + (size_t)t * k, margin ? margin + t : NULL);
    if (z_out) memcpy(z_out + (size_t)t * E, z, sizeof(double) * (size_t)E);
    free(z);
  }
  return 0;
}

/* ------------------------------------------------------------------------------------------------
 * One expert applied to one token.  PAPER.md:57 "an MoE layer replaces the FFN with multiple expert
 * FFNs"; the FFN form is not in the paper -- reading R5 (BASELINE.json north_star: "grouped SwiGLU
 * expert FFN (w1/w3 then w2)"): g = W1 x, u = W3 x, h = silu(g)*u with silu(v) = v/(1+e^-v), y = W2 h.
 * w13 is [2I,H] with rows 0..I-1 = W1 (SiLU branch) and I..2I-1 = W3; w2 is [H,I].  No biases.
 * ---------------------------------------------------------------------------------------------- */
static void expert_ffn(int H, int I, const uint16_t *x, const uint16_t *w13, const uint16_t *w2,
                       double *h /*[I]*/, double *y /*[H]*/) {
  for (int i = 0; i < I; ++i) {
    double g = 0.0, u = 0.0;
    const uint16_t *r1 = w13 + (size_t)i * H;
    const uint16_t *r3 = w13 + (size_t)(I + i) * H;
    for (int c = 0; c < H; ++c) {
      double xv = bf16_to_double(x[c]);
      g += bf16_to_double(r1[c]) * xv;
      u += bf16_to_double(r3[c]) * xv;
    }
    h[i] = g / (1.0 + exp(-g)) * u;
  }
  for (int r = 0; r < H; ++r) {
    double acc = 0.0;
    const uint16_t *row = w2 + (size_t)r * I;
    for (int i = 0; i < I; ++i) acc += bf16_to_double(row[i]) * h[i];
    y[r] = acc;
  }
}

int oracle_expert_ffn(const oracle_shape_t *s, const uint16_t *x_row, const uint16_t *w13_e,
                      const uint16_t *w2_e, double *h, double *y) {
  expert_ffn(s->hidden, s->inter, x_row, w13_e, w2_e, h, y);
  return 0;
}

/* ------------------------------------------------------------------------------------------------
 * The whole layer step.  PAPER.md:79 "the gate partitions the batch among
 * experts ... each step fetches the weights of every expert the batch activates" -- U = set of
 * experts some token chose; bytes_loaded = (|U| + n_shared) * 3*H*I*2 (north_star invariant).
 * out[t] = sum_j w[t,j] * FFN_{e_j}(x_t) + sum_s FFN_shared_s(x_t)   (shared: weight 1, reading R11).
 * If force_ids/force_w are given they replace the gate (the Fig. 2 sweep moves experts and batch
 * independently); ids/w outputs then echo them.
 * Optional per-pair dumps h_pairs [T*k,I], y_pairs [T*k,H] are indexed by (token, slot).
 * ---------------------------------------------------------------------------------------------- */
int oracle_moe_decode_layer(const oracle_shape_t *s, int32_t T, const uint16_t *x,
                            const float *gate_w, const float *gate_bias, const uint16_t *w13,
                            const uint16_t *w2, const uint16_t *shared_w13,
                            const uint16_t *shared_w2, const int32_t *force_ids,
                            const double *force_w, double *out /*[T,H]*/, int32_t *ids /*[T,k]*/,
                            double *w /*[T,k]*/, double *margin /*[T] or NULL*/,
                            double *h_pairs /*or NULL*/, double *y_pairs /*or NULL*/,
                            int32_t *cnt /*[E]*/, int32_t *active /*[E]*/, int32_t *n_active,
                            int64_t *bytes_loaded) {
  if (!s || s->top_k < 1 || s->top_k > s->n_experts) return -1;
  const int H = s->hidden, I = s->inter, E = s->n_experts, k = s->top_k;
  const size_t e13 = (size_t)2 * I * H, e2 = (size_t)H * I;
  if (force_ids) {
    for (size_t i = 0; i < (size_t)T * k; ++i) {
      ids[i] = force_ids[i];
      w[i] = force_w[i];
    }
    if (margin)
      for (int t = 0; t < T; ++t) margin[t] = INFINITY;
  } else {
    oracle_gate_topk(s, T, x, gate_w, gate_bias, NULL, ids, w, margin);
  }
#pragma omp parallel for schedule(dynamic, 1)
  for (int t = 0; t < T; ++t) {
    double *h = (double *)malloc(sizeof(double) * (size_t)I);
    double *y = (double *)malloc(sizeof(double) * (size_t)H);
    double *o = out + (size_t)t * H;
    for (int c = 0; c < H; ++c) o[c] = 0.0;
    for (int j = 0; j < k; ++j) {
      int e = ids[(size_t)t * k + j];
      expert_ffn(H, I, x + (size_t)t * H, w13 + e13 * e, w2 + e2 * e, h, y);
      double wj = w[(size_t)t * k + j];
      for (int c = 0; c < H; ++c) o[c] += wj * y[c];
      if (h_pairs) memcpy(h_pairs + ((size_t)t * k + j) * I, h, sizeof(double) * (size_t)I);
      if (y_pairs) memcpy(y_pairs + ((size_t)t * k + j) * H, y, sizeof(double) * (size_t)H);
    }
    for (int sh = 0; sh < s->n_shared; ++sh) {
      expert_ffn(H, I, x + (size_t)t * H, shared_w13 + e13 * sh, shared_w2 + e2 * sh, h, y);
      for (int c = 0; c < H; ++c) o[c] += y[c];
    }
    free(h);
    free(y);
  }
  for (int e = 0; e < E; ++e) cnt[e] = 0;
  for (size_t i = 0; i < (size_t)T * k; ++i) cnt[ids[i]] += 1;
  int na = 0;
  for (int e = 0; e < E; ++e)
    if (cnt[e] > 0) active[na++] = e;
  for (int e = na; e < E; ++e) active[e] = -1;
  *n_active = na;
  if (bytes_loaded) *bytes_loaded = (int64_t)(na + s->n_shared) * 3 * (int64_t)H * I * 2;
  return 0;
}

/* ------------------------------------------------------------------------------------------------
 * Token -> expert permutation with union compaction.  PAPER.md:79 "the gate partitions the batch
 * among experts".  cnt[e] = pairs routed to e; off = exclusive scan; perm lists pair indices
 * (t*k + slot) grouped by expert, canonical order ascending (token, slot) inside a group (the
 * order inside a group is not unique -- tests compare groups as multisets); active = ascending
 * ids of experts with cnt>0.
 * ---------------------------------------------------------------------------------------------- */
int oracle_permutation(const oracle_shape_t *s, int32_t T, const int32_t *ids, int32_t *cnt,
                       int32_t *off /*[E+1]*/, int32_t *perm /*[T*k]*/, int32_t *active,
                       int32_t *n_active) {
  const int E = s->n_experts, k = s->top_k;
  for (int e = 0; e < E; ++e) cnt[e] = 0;
  for (size_t i = 0; i < (size_t)T * k; ++i) {
    if (ids[i] < 0 || ids[i] >= E) return -1;
    cnt[ids[i]] += 1;
  }
  off[0] = 0;
  for (int e = 0; e < E; ++e) off[e + 1] = off[e] + cnt[e];
  int32_t *cur = (int32_t *)malloc(sizeof(int32_t) * (size_t)E);
  for (int e = 0; e < E; ++e) cur[e] = off[e];
  for (size_t i = 0; i < (size_t)T * k; ++i) perm[cur[ids[i]]++] = (int32_t)i;
  free(cur);
  int na = 0;
  for (int e = 0; e < E; ++e)
    if (cnt[e] > 0) active[na++] = e;
  for (int e = na; e < E; ++e) active[e] = -1;
  *n_active = na;
  return 0;
}

/* ------------------------------------------------------------------------------------------------
 * Signature accumulation.  PAPER.md:198 "Count. At each layer l, count how many prefill tokens are
 * routed to each expert, giving c_r(l) in N^E"; "As prefill writes a token's K/V into a
 * block, the top-k experts selected for that token at each MoE layer are written to the matching
 * signature row"; "one int8 per (block, MoE layer, expert)".
 * sig_req [R,L,E] int32, sig_block [NB,L,E] int8.  token_req/token_block < 0 => token not recorded
 * (padding; reading R9).  Either table or map may be NULL.  Serial loop in token order.
 * An int8 cell holds at most 127: under PAPER.md:255's layout a cell counts the tokens of ONE KV block that picked
 * the expert (<= block size <= 127), so the bound is never reached by a conforming caller; past it the cell stays at
 * 127 (reading "int8 cells saturate") instead of wrapping to -128.
 * ---------------------------------------------------------------------------------------------- */
int oracle_signature_accumulate(const oracle_shape_t *s, int32_t layer, int32_t T,
                                const int32_t *ids, const int32_t *token_req,
                                const int32_t *token_block, int32_t *sig_req, int8_t *sig_block) {
  const int E = s->n_experts, k = s->top_k, L = s->n_layers;
  if (layer < 0 || layer >= L) return -1;
  for (int t = 0; t < T; ++t) {
    for (int j = 0; j < k; ++j) {
      int e = ids[(size_t)t * k + j];
      if (e < 0 || e >= E) return -1;
      if (sig_req && token_req && token_req[t] >= 0)
        sig_req[((size_t)token_req[t] * L + layer) * E + e] += 1;
      if (sig_block && token_block && token_block[t] >= 0) {
        int8_t *cell = &sig_block[((size_t)token_block[t] * L + layer) * E + e];
        if (*cell < 127) *cell += 1;
      }
    }
  }
  return 0;
}

/* PAPER.md:253 "a reused block resets its signature": zero all L*E cells of the listed rows. */
int oracle_signature_reset_blocks(const oracle_shape_t *s, const int32_t *block_ids, int32_t n,
                                  int8_t *sig_block) {
  const size_t row = (size_t)s->n_layers * s->n_experts;
  for (int i = 0; i < n; ++i)
    if (block_ids[i] >= 0) memset(sig_block + row * (size_t)block_ids[i], 0, row);
  return 0;
}

/* PAPER.md:253 "s_r = sum_{b in B(r)} sig[b]"; "retrieving a request's signature sums
 * its blocks' rows into its [L, E] signature". */
int oracle_signature_readout(const oracle_shape_t *s, const int32_t *block_ids, int32_t n,
                             const int8_t *sig_block, int32_t *sig_out /*[L,E]*/) {
  const size_t row = (size_t)s->n_layers * s->n_experts;
  for (size_t c = 0; c < row; ++c) sig_out[c] = 0;
  for (int i = 0; i < n; ++i) {
    if (block_ids[i] < 0) continue;
    const int8_t *r = sig_block + row * (size_t)block_ids[i];
    for (size_t c = 0; c < row; ++c) sig_out[c] += (int32_t)r[c];
  }
  return 0;
}

/* ------------------------------------------------------------------------------------------------
 * signature -> routing decision ("Four steps build s_r",
 * PAPER.md:239 "locality-band routing").  Followed step by step in the paper's order and notation:
 *
 *   2. downweight: c~_r(l,e) = c_r(l,e) * w(l,e), w(l,e) = log((|C|+1)/(df(l,e)+1))
 *   3. select layers: x_r = [c~_r(l)]_{l in S}
 *   4. normalise: s_r = x_r / ||x_r||_2                                                    (Eq. 2)
 *   routing: s_k = cosine(s_r, centroid_k); s* = max_k s_k; among workers with s_k >= s* - tau pick
 *            the one with the smallest load (in-flight decode requests), then load += 1
 *
 * Readings where the paper is silent: requests of one call are routed in index order and
 * each sees the loads left by the previous ones ("updated as requests are dispatched"); equal loads in
 * the band -> the larger similarity, then the lower worker index; an all-zero x_r (or centroid) has
 * similarity 0 to everything; centroids need not arrive normalised (cosine divides by both norms) and
 * their entries on layers outside S are ignored.
 * Pins (tests/test_route_pins.py): tau = 0 => argmax cosine (numpy); tau = 1 on non-negative vectors =>
 * join-shortest-queue; scale invariance of Eq. 2; masked layers do not matter; IDF closed form; the
 * hand-worked 2-expert example in tests/golden/route_example.txt.
 */
void oracle_idf_table(int32_t n, const int32_t *df, int32_t n_calib, double *w) {
  for (int32_t i = 0; i < n; ++i) w[i] = log(((double)n_calib + 1.0) / ((double)df[i] + 1.0));
}

int oracle_route_decide(int32_t R, int32_t L, int32_t E, int32_t K, const int32_t *counts /*[R,L,E]*/,
                        const double *idf /*[L,E]*/, const uint8_t *layer_mask /*[L]*/,
                        const double *centroids /*[K,L,E]*/, int64_t *loads /*[K] in/out*/, double tau,
                        int32_t *worker /*[R]*/, double *sims /*[R,K]*/, double *band_gap /*[R] or NULL*/) {
  if (R < 0 || L <= 0 || E <= 0 || K <= 0) return -1;
  const size_t D = (size_t)L * E;
  double *x = (double *)malloc(D * sizeof(double));
  if (!x) return -2;
  for (int32_t r = 0; r < R; ++r) {
    double xn = 0.0;
    for (int32_t l = 0; l < L; ++l)
      for (int32_t e = 0; e < E; ++e) {
        const size_t i = (size_t)l * E + e;
        x[i] = layer_mask[l] ? (double)counts[(size_t)r * D + i] * idf[i] : 0.0;
        xn += x[i] * x[i];
      }
    xn = sqrt(xn);
    double best = -2.0;
    for (int32_t k = 0; k < K; ++k) {
      double dot = 0.0, cn = 0.0;
      for (int32_t l = 0; l < L; ++l) {
        if (!layer_mask[l]) continue;
        for (int32_t e = 0; e < E; ++e) {
          const size_t i = (size_t)l * E + e;
          const double c = centroids[(size_t)k * D + i];
          dot += (x[i] / (xn > 0.0 ? xn : 1.0)) * c;          /* s_r . centroid_k with s_r = x_r/||x_r|| (Eq. 2) */
          cn += c * c;
        }
      }
      cn = sqrt(cn);
      const double s = (xn > 0.0 && cn > 0.0) ? dot / cn : 0.0;
      sims[(size_t)r * K + k] = s;
      if (s > best) best = s;
    }
    int32_t pick = -1;
    double gap = 1e300;                                        /* distance of the nearest similarity to the band edge */
    for (int32_t k = 0; k < K; ++k) {
      const double s = sims[(size_t)r * K + k];
      const double d = fabs(s - (best - tau));
      if (d < gap) gap = d;
      if (s >= best - tau) {
        if (pick < 0 || loads[k] < loads[pick] ||
            (loads[k] == loads[pick] && s > sims[(size_t)r * K + pick]))
          pick = k;
      }
    }
    worker[r] = pick;
    loads[pick] += 1;
    if (band_gap) band_gap[r] = gap;
  }
  free(x);
  return 0;
}
