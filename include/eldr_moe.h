/*
 * eldr_moe.h -- C ABI of the B200 (sm_100a) batched-decode MoE layer with fused ELDR expert-signature
 * accumulation.  Source of the method: "ELDR: Expert-Locality-Aware Decode Routing for PD-Disaggregated
 * MoE Serving" (arxiv/paper_2607_00466), cited below as PAPER.md:<line> (section).
 *
 * What the path computes (section 3.1: "the gate partitions the batch among experts ... each
 * step fetches the weights of every expert the batch activates"; "standard top-k gating"):
 *
 *   z[t,e]   = sum_h x[t,h] * gate_w[e,h] (+ gate_bias[e])                       gate GEMV, fp32
 *   p[t,:]   = softmax_E(z[t,:]);  ids[t,:] = the k experts with the largest z (ties -> lower id),
 *              z-descending;  w[t,j] = p[t,ids_j] / sum_i p[t,ids_i]  if renormalize, else p[t,ids_j]
 *   U        = { e : some token chose e }   (the active-expert union, ascending id)
 *   out[t,:] = sum_j w[t,j] * W2_e ( silu(W1_e x_t) * (W3_e x_t) ),  e = ids[t,j]   (SwiGLU, no bias)
 *              + sum_s FFN_shared_s(x_t)                               (always-on shared experts, weight 1)
 *   only experts in U (and the shared experts) are read from HBM, each exactly once per call.
 *
 * Signature (section 4.2.2 step 1 "Count"; section 4.4):
 *   for every recorded token t and each of its k ids e:
 *     sig_req  [token_req[t],   layer, e] += 1      int32 [R , L, E]   per-request counts c_r(l,e)
 *     sig_block[token_block[t], layer, e] += 1      int8  [NB, L, E]   "one int8 per (block, MoE layer, expert)"
 *   so that  s_r = sum_{b in B(r)} sig_block[b].
 *
 * Conventions for every entry point
 *   - Pointers are DEVICE pointers unless the name starts with h_ (host).  The caller owns every buffer;
 *     the library never allocates, frees or retains device memory (it caches only TMA descriptors, by value).
 *   - All work is enqueued on `stream`; no host synchronisation, no hidden streams
 *     (except eldr_moe_decode_layer_host, which is synchronous by contract).
 *   - Layouts are row-major, dense.  bf16 tensors are passed as uint16_t bit patterns (eldr_bf16).
 *     Device pointers must be 16-byte aligned.
 *   - Return value: ELDR_OK (0) or a negative eldr_status_t.  No exceptions cross the ABI.
 *     T == 0 is a no-op returning ELDR_OK.  NaN/Inf inputs are outside the contract (ids stay in [0,E)).
 *   - token_req[t] < 0 / token_block[t] < 0 mean "do not record this token" (padding).
 *   - Shared experts are not gate selections: they are never counted in signatures nor in n_active.
 */
#ifndef ELDR_MOE_H_
#define ELDR_MOE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef uint16_t eldr_bf16;          /* bfloat16 bit pattern */
typedef void*    eldr_stream_t;      /* cudaStream_t */

typedef enum {
  ELDR_OK                   =  0,
  ELDR_ERR_INVALID_ARG      = -1,    /* null pointer, bad shape field, misaligned pointer, k > E, block size > 127 */
  ELDR_ERR_UNSUPPORTED      = -2,    /* shape outside what the kernels support (see each function) */
  ELDR_ERR_WORKSPACE_SMALL  = -3,
  ELDR_ERR_CUDA             = -4     /* a CUDA runtime / driver call or a launch failed */
} eldr_status_t;

typedef struct {                     /* passed by const pointer, HOST memory */
  int32_t hidden;                    /* H, multiple of 8 (16-byte bf16 vectors)                      */
  int32_t inter;                     /* I, multiple of 8                                              */
  int32_t n_experts;                 /* E routed experts, 1..256                                      */
  int32_t top_k;                     /* k, 1..min(E,16)                                               */
  int32_t n_shared;                  /* always-on shared experts, 0..8                                */
  int32_t renormalize;               /* 1: w /= sum over the top-k (all BASELINE configs); 0: w = p   */
  int32_t n_layers;                  /* L, row stride of the signature tensors                        */
  int32_t kv_block_size;             /* tokens per KV block, 1..127 (int8 cells)        */
} eldr_moe_shape_t;

/* Byte offsets of the intermediates eldr_moe_decode_layer leaves in `workspace` (for per-kernel parity
 * tests and profiling; the contents are valid until the next call that uses the workspace). */
typedef struct {
  size_t z;          /* float   [T,E]            gate logits incl. bias                                 */
  size_t cnt;        /* int32   [E]              pairs routed to each expert                             */
  size_t off;        /* int32   [E+1]            exclusive scan of cnt                                   */
  size_t perm;       /* int32   [T*k]            pair index (t*k+slot) at each sorted position           */
  size_t pair_pos;   /* int32   [T*k]            inverse of perm                                         */
  size_t work;       /* int32x4 [E+n_shared]     {expert, x_row0, out_row0, m} per streamed expert: routed experts in id order; the shared ones (ids E..) before them (one-launch step) or after them (staged step) */
  size_t n_work;     /* int32   [1]              n_active + n_shared                                     */
  size_t sync;       /* uint32  [...]            epoch flags + generation words (internal); offset 0                       */
  size_t x_perm;     /* bf16    [T*k + T, H]     x gathered in sorted order, then a plain copy of x      */
  size_t h;          /* bf16    [T*(k+ns), I]    silu(W1 x)*(W3 x) per sorted pair, then shared experts  */
  size_t y;          /* float   [T*(k+ns), H]    W2 h per sorted pair, then shared experts               */
  size_t partial;    /* float   [4][256][128][128] parked fp32 accumulators of tiles split between SMs (internal; 64 MiB for T <= 256, unused above) */
  size_t total;      /* bytes needed                                                                    */
} eldr_moe_ws_layout_t;

/* Gate + softmax top-k + renormalise (+ fused signature accumulation) for T tokens of one layer.
 * Operation: z, ids, w as defined above ("The gate scores experts using the token's hidden
 * representation and dispatches the token to the top-scoring experts").  Any T >= 0.
 *   x [T,H] bf16 in; gate_w [E,H] fp32 in; gate_bias [E] fp32 in or NULL;
 *   topk_ids [T,k] int32 out; topk_w [T,k] fp32 out;
 *   token_req/token_block [T] int32 in or NULL; sig_req [R,L,E] int32 in/out or NULL;
 *   sig_block [NB,L,E] int8 in/out or NULL (accumulated in place; caller zeroes / resets);
 *   workspace: at least eldr_moe_workspace_bytes(shape, T) bytes (holds z). */
int32_t eldr_moe_gate_topk(const eldr_moe_shape_t* shape, int32_t layer, int32_t T,
                           const eldr_bf16* x, const float* gate_w, const float* gate_bias,
                           int32_t* topk_ids, float* topk_w,
                           const int32_t* token_req, const int32_t* token_block,
                           int32_t* sig_req, int8_t* sig_block,
                           void* workspace, size_t workspace_bytes, eldr_stream_t stream);

/* eldr_moe_gate_topk for callers that may not allocate (CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): same operation, same outputs, NO workspace argument and no allocation of any kind inside the call (no
 * cudaMalloc / cudaFree, no allocating library routine).  The logits z [T,E] fp32 live in a file-scope
 * `static __device__` array of ELDR_STATIC_SCRATCH_BYTES bytes inside the library; every GPU that loads the library
 * holds that array until the process exits.
 *   Limit: T * n_experts * 4 <= ELDR_STATIC_SCRATCH_BYTES (1 MiB: T <= 2048 at E = 128); beyond it the call returns
 *   ELDR_ERR_WORKSPACE_SMALL (eldr_last_cuda_error() says by how much) and launches nothing.
 *   All calls on a device share the one array and it keeps the last call's logits; the call overwrites every element
 *   it later reads, so nothing needs clearing -- but two calls that OVERLAP on the GPU (different streams, or graphs
 *   replayed concurrently) race on it: serialise them.  Other arguments exactly as eldr_moe_gate_topk. */
#define ELDR_STATIC_SCRATCH_BYTES (1u << 20)
int32_t eldr_moe_gate_topk_static(const eldr_moe_shape_t* shape, int32_t layer, int32_t T,
                                  const eldr_bf16* x, const float* gate_w, const float* gate_bias,
                                  int32_t* topk_ids, float* topk_w,
                                  const int32_t* token_req, const int32_t* token_block,
                                  int32_t* sig_req, int8_t* sig_block, eldr_stream_t stream);

/* One decode step of one MoE layer: gate -> top-k (+signature) -> token->expert permutation with union
 * compaction -> grouped SwiGLU FFN streaming each ACTIVE expert's weights once -> weighted combine.
 *   w13 [E,2I,H] bf16: rows 0..I-1 = w1 (SiLU branch), rows I..2I-1 = w3;  w2 [E,H,I] bf16;
 *   shared_w13 [n_shared,2I,H], shared_w2 [n_shared,H,I] (NULL iff n_shared == 0);
 *   out [T,H] bf16 (rounded once, RNE, from the fp32 combine);
 *   topk_ids/topk_w: outputs, or INPUTS if force_routing != 0 (ids must be distinct per token, in [0,E));
 *   active_experts [E] int32 out: first n_active entries = U ascending, rest -1;  n_active [1] int32 out.
 *   T in 0..16384 (larger T -> ELDR_ERR_UNSUPPORTED).  T <= 256 with H, I multiples of 64: the whole step is one
 *   persistent launch; T <= 1024: one launch per stage; T > 1024 (prefill-shaped, "prefill forward ...
 *   captures signature"): gate GEMM, top-k + signature, a chunked counting sort, gather, the grouped FFN with 256
 *   tokens per tcgen05 accumulator pass, combine -- same arithmetic, compute-bound instead of HBM-bound.
 * Fast path (TMA + mma) needs H % 64 == 0 and I % 64 == 0; other shapes run a plain CUDA-core path. */
int32_t eldr_moe_decode_layer(const eldr_moe_shape_t* shape, int32_t layer, int32_t T,
                              const eldr_bf16* x, const float* gate_w, const float* gate_bias,
                              const eldr_bf16* w13, const eldr_bf16* w2,
                              const eldr_bf16* shared_w13, const eldr_bf16* shared_w2,
                              eldr_bf16* out,
                              int32_t* topk_ids, float* topk_w, int32_t force_routing,
                              int32_t* active_experts, int32_t* n_active,
                              const int32_t* token_req, const int32_t* token_block,
                              int32_t* sig_req, int8_t* sig_block,
                              void* workspace, size_t workspace_bytes, eldr_stream_t stream);

/* The same step with MXFP4 expert weights (section 6 Testbed: "GPT-OSS-120B (128
 * experts, top-4, mxfp4)").  The paper only names the format; readings (oracle/mxfp4.py): OCP MX v1.0 --
 * element = FP4 E2M1 code (sign, 2 exponent bits bias 1, 1 mantissa bit: magnitudes 0, .5, 1, 1.5, 2, 3, 4, 6), two
 * codes per byte with element 2i in the LOW nibble; one E8M0 scale byte per 32 consecutive elements of the
 * contraction (innermost) axis, value = e2m1(code) * 2^(scale - 127).  Scale bytes must lie in 3..250 (every decoded
 * value is then exactly a bf16 number; 255 = NaN is outside the contract).
 *   w13_codes [E,2I,H/2] uint8, w13_scales [E,2I,H/32] uint8 (rows 0..I-1 = w1, I..2I-1 = w3);
 *   w2_codes  [E,H,I/2]  uint8, w2_scales  [E,H,I/32]  uint8.  All device pointers, 16-byte aligned.
 * Operation: eldr_moe_decode_layer on the DECODED weights -- activations stay bf16 and are not quantised, products
 * accumulate in fp32 -- so the same oracle and tolerances apply.  Only the packed bytes are read from HBM
 * ((|U|)*3*H*I*(1/2 + 1/32) bytes per step); they are decoded to bf16 in shared memory on the way to the tensor cores.
 * Every other argument as eldr_moe_decode_layer.  Restrictions: T <= 1024, n_shared == 0, H % 64 == 0, I % 64 == 0
 * (else ELDR_ERR_UNSUPPORTED).  Five launches (gate+top-k+signature+routing, gather, w1/w3, w2, combine). */
int32_t eldr_moe_decode_layer_mxfp4(const eldr_moe_shape_t* shape, int32_t layer, int32_t T,
                                    const eldr_bf16* x, const float* gate_w, const float* gate_bias,
                                    const uint8_t* w13_codes, const uint8_t* w13_scales,
                                    const uint8_t* w2_codes, const uint8_t* w2_scales,
                                    eldr_bf16* out,
                                    int32_t* topk_ids, float* topk_w, int32_t force_routing,
                                    int32_t* active_experts, int32_t* n_active,
                                    const int32_t* token_req, const int32_t* token_block,
                                    int32_t* sig_req, int8_t* sig_block,
                                    void* workspace, size_t workspace_bytes, eldr_stream_t stream);

/* Same step with the per-step inputs and results in HOST memory (pinned for async copies): copies h_x and
 * the token maps to the device, runs eldr_moe_decode_layer, copies out / ids / weights / n_active back and
 * synchronises `stream` before returning.  Weights, gate, signature tables and workspace stay on the device.
 * `workspace` must hold eldr_moe_workspace_bytes_host(shape, T) bytes (layer workspace + staging). */
int32_t eldr_moe_decode_layer_host(const eldr_moe_shape_t* shape, int32_t layer, int32_t T,
                                   const eldr_bf16* h_x, const float* gate_w, const float* gate_bias,
                                   const eldr_bf16* w13, const eldr_bf16* w2,
                                   const eldr_bf16* shared_w13, const eldr_bf16* shared_w2,
                                   eldr_bf16* h_out, int32_t* h_topk_ids, float* h_topk_w,
                                   int32_t* h_n_active,
                                   const int32_t* h_token_req, const int32_t* h_token_block,
                                   int32_t* sig_req, int8_t* sig_block,
                                   void* workspace, size_t workspace_bytes, eldr_stream_t stream);

/* Signature accumulation alone, from already-computed top-k ids (prefill-shaped calls: "Each
 * forward accumulates the new tokens' expert picks into the matching rows in a single GPU pass").
 * Exact integer adds; the result does not depend on the order of tokens.  Any T >= 0. */
int32_t eldr_signature_accumulate(const eldr_moe_shape_t* shape, int32_t layer, int32_t T,
                                  const int32_t* topk_ids, const int32_t* token_req,
                                  const int32_t* token_block, int32_t* sig_req, int8_t* sig_block,
                                  eldr_stream_t stream);

/* The same for n_layers consecutive layers in ONE launch (prefill-shaped capture: a prefill forward yields the picks of
 * every layer; "in a single GPU pass", Table 1's scatter at PAPER.md:308 is the context figure).
 *   topk_ids [n_layers, T, k] int32 (layer-major); rows layer0 .. layer0+n_layers-1 of the signature tensors are updated.
 * Increments of a 256-token chunk are combined in shared memory before they reach the tables; results are identical
 * to n_layers calls of eldr_signature_accumulate (integer adds commute; int8 cells saturate at 127). */
int32_t eldr_signature_accumulate_layers(const eldr_moe_shape_t* shape, int32_t layer0, int32_t n_layers, int32_t T,
                                         const int32_t* topk_ids, const int32_t* token_req,
                                         const int32_t* token_block, int32_t* sig_req, int8_t* sig_block,
                                         eldr_stream_t stream);

/* PAPER.md:253 "a reused block resets its signature": zero the L*E cells of each listed row (ids < 0 skipped). */
int32_t eldr_signature_reset_blocks(const eldr_moe_shape_t* shape, const int32_t* block_ids, int32_t n,
                                    int8_t* sig_block, eldr_stream_t stream);

/* PAPER.md:253 "s_r = sum_{b in B(r)} sig[b]", "retrieving a request's signature sums its
 * blocks' rows into its [L,E] signature": for request i, sums rows block_ids[req_off[i] .. req_off[i+1])
 * of sig_block into sig_out[i] ([n_req,L,E] int32, overwritten). */
int32_t eldr_signature_readout(const eldr_moe_shape_t* shape, const int32_t* block_ids,
                               const int32_t* req_off, int32_t n_req, const int8_t* sig_block,
                               int32_t* sig_out, eldr_stream_t stream);

/* Signature -> routing decision for R requests.  PAPER.md:196-203: reweight the counts by
 * the IDF table (step 2), keep the layers of the mask S (step 3), normalise (Eq. 2); PAPER.md:239 locality-band
 * routing: s_k = cosine(s_r, centroid_k), s* = max_k s_k, among workers with s_k >= s* - tau pick the one with the
 * smallest load, then loads[pick] += 1.  Requests are routed in index order, each seeing the loads left by the
 * previous ones; equal loads in the band -> larger similarity, then lower index; an all-zero signature (or
 * centroid) has similarity 0 (readings).
 *   sig_req [R,L,E] int32 in (what eldr_signature_readout wrote; L = shape->n_layers, E = shape->n_experts);
 *   idf [L,E] fp32 in (w(l,e) = log((|C|+1)/(df(l,e)+1)), fit offline); layer_mask [L] uint8 in (1 = kept);
 *   centroids [K,L,E] fp32 in (need not be normalised; entries on dropped layers ignored), 1 <= K <= 1024;
 *   loads [K] int32 in/out (in-flight decode requests per worker); tau >= 0;
 *   worker [R] int32 out; sims [R,K] fp32 out (the cosine similarities; required).
 * All pointers are device pointers; two small launches on `stream`; no host sync; R == 0 is a no-op. */
int32_t eldr_route_decide(const eldr_moe_shape_t* shape, int32_t R, int32_t K, const int32_t* sig_req,
                          const float* idf, const uint8_t* layer_mask, const float* centroids, int32_t* loads,
                          float tau, int32_t* worker, float* sims, eldr_stream_t stream);

/* ---- Offline fit.  HOST functions: every pointer is host memory, fp64, synchronous, no CUDA
 * call -- the paper fits on the CPU before serving ("under 10 s on CPU").  Readings where the paper is
 * silent: DESIGN.md 9d (the random calibration pairs and the initial centroids are inputs; average ranks for ties;
 * cos-dist of a zero vector = 1; greedy ties -> lowest layer; N* = first maximum; centroid = renormalised mean, an
 * empty centroid keeps its value).
 *
 * eldr_fit_idf: h_idf[l,e] = log((N+1) / (df(l,e)+1)), df = requests with h_counts[r,l,e] > 0.
 *   h_counts [N,L,E] int32 in (per-request prefill counts c_r(l,e));  h_idf [L,E] double out.
 * eldr_fit_layer_mask (Eq. 1 at :183): greedy layer selection on rho = Spearman(cos-dist of the signatures
 *   restricted to the mask, cos-dist of the decode patterns) over the given request pairs.
 *   h_decode_p [N,L,E] double in (decode-time activation probabilities p_i(l,e)); h_pairs [P,2] int32 in;
 *   h_order [L] int32 out (layers in the order they were appended); h_cum_rho [L] double out (rho of each prefix);
 *   h_n_star [1] out (prefix length at which rho peaks); h_mask [L] uint8 out (1 = kept: the first N* of the order).
 * eldr_fit_balanced_assign: the assignment of N points to K centroids minimising the total cost with at
 *   most `cap` points per centroid (K*cap >= N).  h_cost [N,K] double in; h_assign [N] int32 out; h_total [1] out or NULL.
 * eldr_fit_kmeans_balanced: Hungarian-balanced spherical K-means, cap = ceil(N/K), cost = 1 - cosine.
 *   h_sig [N,d] double in (unit rows: Eq. 2 signatures); h_init_idx [K] int32 in (requests whose signatures seed the
 *   centroids); at most max_iter assignment steps, stops when the assignment repeats;
 *   h_centroids [K,d] double out (unit rows); h_assign [N] int32 out; h_steps [1], h_total [1] out (assignment steps
 *   run; total cosine distance of the final assignment to the centroids it was computed against).
 * Errors: ELDR_ERR_INVALID_ARG for null pointers, non-positive sizes, K*cap < N, indices out of range. */
int32_t eldr_fit_idf(const int32_t* h_counts, int32_t N, int32_t L, int32_t E, double* h_idf);
int32_t eldr_fit_layer_mask(const int32_t* h_counts, const double* h_idf, const double* h_decode_p,
                            int32_t N, int32_t L, int32_t E, const int32_t* h_pairs, int32_t P,
                            int32_t* h_order, double* h_cum_rho, int32_t* h_n_star, uint8_t* h_mask);
int32_t eldr_fit_balanced_assign(const double* h_cost, int32_t N, int32_t K, int32_t cap,
                                 int32_t* h_assign, double* h_total);
int32_t eldr_fit_kmeans_balanced(const double* h_sig, int32_t N, int32_t d, int32_t K,
                                 const int32_t* h_init_idx, int32_t max_iter,
                                 double* h_centroids, int32_t* h_assign, int32_t* h_steps, double* h_total);

/* Workspace: device memory owned by the caller, 16-byte aligned, at least the number of bytes returned here; one
 * workspace serves one call at a time (calls that overlap on the GPU need their own).  It carries state between calls:
 * its first word is the generation of the epoch flags the kernels of a step wait on.  RECOMMENDED: zero the workspace
 * once after allocating it (cudaMemsetAsync).  It is not required: the epoch of a step is a full-period 32-bit sequence
 * state XOR a salt derived from the workspace address, so the stale bytes of a recycled allocation pass for a raised flag
 * only with probability ~ (distinct stale words) / 2^32 on the first step.  Do not copy a live workspace to another
 * address and continue there. */
size_t  eldr_moe_workspace_bytes(const eldr_moe_shape_t* shape, int32_t max_T);
size_t  eldr_moe_workspace_bytes_host(const eldr_moe_shape_t* shape, int32_t max_T);
int32_t eldr_moe_workspace_layout(const eldr_moe_shape_t* shape, int32_t T, eldr_moe_ws_layout_t* layout);

/* Process-wide tuning knobs (defaults are the fast settings; used by tests and profiles to compare paths).
 *   ELDR_OPT_FFN_PATH: ELDR_FFN_TCGEN05 (default; tcgen05.mma + TMEM), ELDR_FFN_MMA_SYNC (legacy mma.sync) or ELDR_FFN_GEMV
 *   (CUDA-core GEMV, 8 tokens per pass: the comparison path for tiny tokens-per-expert counts; staged launches). */
#define ELDR_OPT_FFN_PATH 0
#define ELDR_OPT_PDL      1   /* 1 (default): programmatic dependent launch between the step's kernels; 0: plain */
#define ELDR_OPT_STEP_PATH 2  /* ELDR_STEP_FUSED: the whole step in ONE persistent launch (T <= 256, H,I % 64 == 0);
                                 ELDR_STEP_STAGED: one launch per stage (gate+route, gather, w1/w3, w2, combine), also
                                 the path for shapes the fused kernel does not take; ELDR_STEP_AUTO (default): fused
                                 whenever the shape allows it */
#define ELDR_OPT_RING_KB  3   /* fused step: cap on the shared-memory stage ring in KiB per SM (bytes in flight);
                                 32..208; default 208 (all of it) */
#define ELDR_OPT_DP_MIN_ROUNDS 4 /* fused step: a phase (w1/w3 or w2, decided for each) whose tile count is at least this many
                                 rounds of the grid runs whole tiles (first tile = the CTA's index, then drawn from a counter),
                                 its remainder per ELDR_OPT_SK_MAX_SPLIT; below it the whole phase is one stream-K cut.
                                 1..2^20; default 1 (round 2 started at 4: |U| = 32 74.5 -> 70.1 us, T = 256 98.8 -> 91.2) */
#define ELDR_OPT_SK_SPLIT_PCT 6 /* fused step, small unions (w1/w3 phase shorter than ELDR_OPT_DP_MIN_ROUNDS rounds of tiles): the
                                 active experts are cut into two groups and the step runs w1/w3(g0) w1/w3(g1) w2(g0) w2(g1);
                                 value = percentage of the experts in g0 (0 or 100: one group).  0..100; default 0: measured on
                                 B200 the two-group order is SLOWER (|U| = 16: 76 vs 60 us) -- each group's share per SM is
                                 shorter than one weight tile, so every tile is cut three ways and the fix-ups have no slack */
#define ELDR_OPT_COOPERATIVE 7 /* fused step: 1 (default) = cooperative launch: the persistent grid, whose CTAs wait on one another,
                                 starts only when ALL of its CTAs can be resident (safe next to kernels of other streams, MPS or
                                 green-context SM partitions; a grid that cannot fit returns to the staged path).  Measured on
                                 B200 the driver does not overlap a cooperative launch with its predecessor (PDL has no effect):
                                 +2.5 us per step.  0 = plain launch + PDL, for a GPU the process has to itself */
#define ELDR_OPT_HEAD_FIRST 8 /* fused step, static (stream-K) ranges: 0 (default) = ascending order, a split tile is finished by the
                                 owner of its first stage; 1 = a CTA first computes and parks the head of the tile its range
                                 ends in, then finishes the tile its range starts in with the previous CTA's parked head, then
                                 streams its whole tiles (every range ends without a fix-up).  Measured on B200: 1 is SLOWER
                                 (|U| = 16: 66.6 vs 61.2 us, 32: 82.2 vs 76.4) -- the early fix-up waits for a partner whose
                                 head piece is longer than ours while the ring is still filling */
#define ELDR_OPT_SK_MAX_SPLIT 10 /* fused step, large unions: the stream-K remainder of a phase (the tiles past the last whole round)
                                 is cut over at most this many CTAs per tile; the other CTAs go straight on to the next part.
                                 0 = over the whole grid (round 1).  0..64; default 1 = whole tiles (|U| = 128: 205.8 us at 0,
                                 203.9 at 2, 197.3 at 1; config-5 shape 221.9 / 215.5 / 216.5) */
#define ELDR_OPT_GATE_TC 11    /* prefill-shaped gate (T >= 2048, hidden % 64 == 0): 1 (default) = on the tensor cores with every fp32
                                 gate weight as the exact sum of three bf16 terms and 256-wide K slices summed in fp32 (same
                                 1e-5 logit gate as the CUDA-core kernels); 0 = the register-tiled fp32 CUDA-core GEMM */
#define ELDR_OPT_XS_MIN_NP 9  /* fused step: when some expert receives at least this many tokens (padded to 16) the w1/w3 phase reads
                                 its activations from an expert-sorted copy of x written inside the step (16 rows per TMA
                                 instruction) instead of gathering token rows from x (4 rows per instruction) for every stage;
                                 16..144, 144 = never (one accumulator pass holds at most 128 columns).  Default 48 */
#define ELDR_OPT_FFN_PAIR 5   /* prefill-shaped calls (T > 1024, I % 128 == 0, H % 256 == 0): the expert FFN as tcgen05
                                 cta_group::2 tiles (M = 256 over an SM pair, ffn_umma2.cuh).  1 (default): when the call
                                 has >= 256 tokens per expert on average (T*k >= 256*E); 2: always; 0: never (one CTA
                                 per 128-row tile) */
#define ELDR_STEP_STAGED  0
#define ELDR_STEP_FUSED   1
#define ELDR_STEP_AUTO    2
#define ELDR_FFN_MMA_SYNC 0
#define ELDR_FFN_TCGEN05  1
#define ELDR_FFN_GEMV     2
int32_t eldr_moe_set_option(int32_t key, int32_t value);

/* Per-kernel device timing of eldr_moe_decode_layer (measurement aid, off by default, per host thread).
 * When enabled, the call records a CUDA event on `stream` before each of its kernels and after the last.
 * eldr_moe_profile_read waits for the last call's events and writes the ELDR_PROFILE_SLOTS durations in
 * milliseconds to HOST memory: [0] gate GEMV + top-k/signature + permutation (one launch), [1] permutation alone (force_routing), [2] gather,
 * [3] FFN w1/w3, [4] FFN w2, [5] combine (0 for a kernel that did not run). */
#define ELDR_PROFILE_SLOTS 6
int32_t eldr_moe_profile_enable(int32_t on);
int32_t eldr_moe_profile_read(float* h_ms);

/* Number of kernels the last eldr_moe_decode_layer call on this thread enqueued (bench accounting). */
int32_t eldr_moe_last_launch_count(void);

const char* eldr_status_string(int32_t status);
/* Text of the last CUDA error seen by this thread inside the library ("" if none). */
const char* eldr_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* ELDR_MOE_H_ */
