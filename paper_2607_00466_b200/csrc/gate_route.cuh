// Gate GEMV, warp-shuffle softmax top-k, fused ELDR signature accumulation, token->expert permutation
// with union compaction, gather, combine.  (SURVEY.md 8(a) steps a1-a4, a7.)
#pragma once
#include "device_utils.cuh"

namespace eldr {

// Optional intra-kernel timeline (debug builds only: -DELDR_TRACE): thread 0 of every CTA stamps %globaltimer.
#ifdef ELDR_TRACE
__device__ unsigned long long g_trace[4096 * 16];
#define ELDR_STAMP(id)                                                                        \
  do {                                                                                        \
    if (threadIdx.x == 0) {                                                                   \
      unsigned long long t_;                                                                  \
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_));                                  \
      g_trace[((blockIdx.y * gridDim.x + blockIdx.x) & 4095) * 16 + (id)] = t_;               \
    }                                                                                         \
  } while (0)
#else
#define ELDR_STAMP(id) do {} while (0)
#endif

constexpr int kMaxExperts = 256;   // 8 logits per lane in the warp top-k
constexpr int kMaxTopK = 16;
constexpr int kGateTok = 8;        // tokens per CTA in the gate GEMV
constexpr int kGateExp = 8;        // experts per CTA (= warps)

// ------------------------------------------------------------------------------------ a1: gate GEMV
// z[t,e] = sum_h x[t,h]*Wg[e,h] + bias[e], fp32 FMA on CUDA cores (no TF32/bf16 MMA: near-ties must not
// flip).  CTA = 8 warps: warp w owns expert blockIdx.x*8+w against an 8-token x tile held in smem as bf16.
__device__ __forceinline__ void gate_tile(const uint16_t* __restrict__ x, const float* __restrict__ gate_w,
                                          const float* __restrict__ gate_bias, float* __restrict__ z, int T, int H,
                                          int E, uint8_t* smem_raw) {
  uint4* xs4 = reinterpret_cast<uint4*>(smem_raw);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int t0 = blockIdx.y * kGateTok;
  const int vec_per_row = H >> 3;
  for (int v = tid; v < kGateTok * vec_per_row; v += 256) {
    const int t = v / vec_per_row, c = v - t * vec_per_row;
    uint4 val = make_uint4(0u, 0u, 0u, 0u);
    if (t0 + t < T) val = *reinterpret_cast<const uint4*>(x + (size_t)(t0 + t) * H + (size_t)c * 8);
    xs4[v] = val;
  }
  __syncthreads();
  ELDR_STAMP(1);
  const int e = blockIdx.x * kGateExp + warp;
  if (e >= E) return;
  float acc[kGateTok];
#pragma unroll
  for (int t = 0; t < kGateTok; ++t) acc[t] = 0.f;
  const float4* wrow = reinterpret_cast<const float4*>(gate_w + (size_t)e * H);
  const uint2* xs2 = reinterpret_cast<const uint2*>(smem_raw);
  const int q_per_row = H >> 2;
  // The gate row is a serial prerequisite of the whole step: issue its loads 8 deep (8 x 512 B per warp in
  // flight) so the row costs ~2 memory latencies instead of H/128.
  constexpr int kDepth = 8;
  for (int base = 0; base < q_per_row; base += 32 * kDepth) {
    float4 wv[kDepth];
#pragma unroll
    for (int u = 0; u < kDepth; ++u) {
      const int c4 = base + lane + 32 * u;
      wv[u] = (c4 < q_per_row) ? __ldg(wrow + c4) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
#pragma unroll
    for (int u = 0; u < kDepth; ++u) {
      const int c4 = base + lane + 32 * u;
      if (c4 < q_per_row) {
#pragma unroll
        for (int t = 0; t < kGateTok; ++t) {
          const uint2 xv = xs2[t * q_per_row + c4];
          float a = acc[t];
          a = fmaf(wv[u].x, bf16_lo(xv.x), a);
          a = fmaf(wv[u].y, bf16_hi(xv.x), a);
          a = fmaf(wv[u].z, bf16_lo(xv.y), a);
          a = fmaf(wv[u].w, bf16_hi(xv.y), a);
          acc[t] = a;
        }
      }
    }
  }
#pragma unroll
  for (int t = 0; t < kGateTok; ++t) {
    float a = acc[t];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
    acc[t] = a;
  }
  if (lane == 0) {
    const float b = gate_bias ? gate_bias[e] : 0.f;
#pragma unroll
    for (int t = 0; t < kGateTok; ++t)
      if (t0 + t < T) z[(size_t)(t0 + t) * E + e] = acc[t] + b;
  }
}

__global__ void __launch_bounds__(256) gate_logits_kernel(const uint16_t* __restrict__ x,
                                                          const float* __restrict__ gate_w,
                                                          const float* __restrict__ gate_bias,
                                                          float* __restrict__ z, int T, int H, int E) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  gate_tile(x, gate_w, gate_bias, z, T, H, E, smem_raw);
}

// ----------------------------------------------------------------------- a2: warp softmax top-k
// One warp, one token.  Lane l holds logits of experts l, l+32, ...  k rounds of warp arg-max with the
// order (z descending, id ascending); lane j ends up holding the j-th pick and its weight.
__device__ __forceinline__ void warp_topk(const float* __restrict__ zrow, int E, int k, int renorm,
                                          int lane, int& my_id, float& my_w) {
  constexpr int NV = kMaxExperts / 32;
  float v[NV];
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const int e = lane + 32 * i;
    v[i] = (e < E) ? __ldcg(zrow + e) : -INFINITY;
  }
  float zmax = v[0];
#pragma unroll
  for (int i = 1; i < NV; ++i) zmax = fmaxf(zmax, v[i]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) zmax = fmaxf(zmax, __shfl_xor_sync(0xffffffffu, zmax, o));
  float denom_all = 0.f;
  if (!renorm) {
#pragma unroll
    for (int i = 0; i < NV; ++i)
      if (lane + 32 * i < E) denom_all += expf(v[i] - zmax);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) denom_all += __shfl_xor_sync(0xffffffffu, denom_all, o);
  }
  float sel_val = -INFINITY;
  int sel_id = 0;
  for (int j = 0; j < k; ++j) {
    float bv = -INFINITY;
    int bi = 0x7fffffff;
#pragma unroll
    for (int i = 0; i < NV; ++i)
      if (v[i] > bv) { bv = v[i]; bi = lane + 32 * i; }     // ascending id per lane: strict > keeps the lower id
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const float ov = __shfl_xor_sync(0xffffffffu, bv, o);
      const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
      if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
    }
    if ((bi & 31) == lane) {
#pragma unroll
      for (int i = 0; i < NV; ++i)
        if ((bi >> 5) == i) v[i] = -INFINITY;
    }
    if (lane == j) { sel_val = bv; sel_id = bi; }
  }
  sel_id = min(max(sel_id, 0), E - 1);          // NaN/Inf inputs are outside the contract; never index out of [0,E)
  const float ev = (lane < k) ? expf(sel_val - zmax) : 0.f;
  float denom = ev;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) denom += __shfl_xor_sync(0xffffffffu, denom, o);
  my_id = sel_id;
  my_w = renorm ? ev / denom : ev / denom_all;
}

// ------------------------------------------------------------------------ a3: signature increments
// int32 request cell: atomic add.  int8 block cell: CUDA has no 8-bit atomics -> 32-bit atomic add of
// 1 << 8*(byte in word) on the aligned word.  Under the contract a cell never exceeds the KV block size
// (<= 127; ids are distinct per token).  A caller that keeps accumulating into a block it never resets would
// otherwise carry into the NEIGHBOURING expert's cell: the cell saturates at 127 instead (reading in DESIGN.md 2;
// the add is undone when the cell already held 127 -- transient values stay below 256 because at most a block's
// worth of adds to one cell can be in flight).  Integer adds commute => bit-exact in any order.
__device__ __forceinline__ void sig_add(int32_t* sig_req, int8_t* sig_block, int req, int blk, int L,
                                        int layer, int E, int e) {
  if (sig_req != nullptr && req >= 0)
    atomicAdd(sig_req + ((size_t)req * L + layer) * E + e, 1);
  if (sig_block != nullptr && blk >= 0) {
    const size_t idx = ((size_t)blk * L + layer) * E + e;
    unsigned int* word = reinterpret_cast<unsigned int*>(sig_block + (idx & ~(size_t)3));
    const unsigned int shift = 8u * (unsigned)(idx & 3), inc = 1u << shift;
    const unsigned int old = atomicAdd(word, inc);
    if (((old >> shift) & 0xffu) >= 127u) atomicSub(word, inc);
  }
}

// The same increment in two halves, for a caller that must not wait for the atomic's round trip (the fused step's
// top-k owners sit on the serial prelude): begin() issues both adds and keeps the int8 word's OLD value in flight;
// finish(), called when the step's work is done, undoes the add if the cell was already saturated.
struct SigPending {
  unsigned int* word;
  unsigned int old, shift;
};
__device__ __forceinline__ SigPending sig_add_begin(int32_t* sig_req, int8_t* sig_block, int req, int blk, int L,
                                                    int layer, int E, int e) {
  SigPending p{nullptr, 0u, 0u};
  if (sig_req != nullptr && req >= 0)
    atomicAdd(sig_req + ((size_t)req * L + layer) * E + e, 1);
  if (sig_block != nullptr && blk >= 0) {
    const size_t idx = ((size_t)blk * L + layer) * E + e;
    p.word = reinterpret_cast<unsigned int*>(sig_block + (idx & ~(size_t)3));
    p.shift = 8u * (unsigned)(idx & 3);
    p.old = atomicAdd(p.word, 1u << p.shift);
  }
  return p;
}
__device__ __forceinline__ void sig_add_finish(const SigPending& p) {
  if (p.word != nullptr && ((p.old >> p.shift) & 0xffu) >= 127u) atomicSub(p.word, 1u << p.shift);
}

struct TopkArgs {
  const float* z;            // [T,E]
  int32_t* ids;              // [T,k]
  float* w;                  // [T,k]
  const int32_t* token_req;  // [T] or null
  const int32_t* token_block;
  int32_t* sig_req;
  int8_t* sig_block;
  int T, E, k, L, layer, renorm;
};

// Multi-CTA top-k (+signature) for eldr_moe_gate_topk: warp per token, any T.
__global__ void __launch_bounds__(256) topk_kernel(TopkArgs a) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int t = blockIdx.x * 8 + warp;
  if (t >= a.T) return;
  int id; float w;
  warp_topk(a.z + (size_t)t * a.E, a.E, a.k, a.renorm, lane, id, w);
  if (lane < a.k) {
    a.ids[(size_t)t * a.k + lane] = id;
    a.w[(size_t)t * a.k + lane] = w;
    sig_add(a.sig_req, a.sig_block, a.token_req ? a.token_req[t] : -1,
            a.token_block ? a.token_block[t] : -1, a.L, a.layer, a.E, id);
  }
}

// ------------------------------------------------- a2+a3+a4: top-k, signature, permutation, union
struct RouteArgs {
  TopkArgs tk;
  int force_routing, n_shared, H;
  int32_t* cnt;        // [E]
  int32_t* off;        // [E+1]
  int32_t* perm;       // [T*k]
  int32_t* pair_pos;   // [T*k]
  int4* work;          // [E+n_shared] {expert, x_row0, out_row0, m}
  int32_t* n_work;     // [1]
  int32_t* active;     // [E]
  int32_t* n_active;   // [1]
};

// Permutation / union compaction by ONE CTA of `nthr` threads (decode batches: T <= 1024).  A membership
// bitmask mask[e][t/32] in shared memory makes the counting sort deterministic and free of global atomics:
// rank of pair (t,e) = popcount of expert e's bits below t.  With do_sig the pairs are also recorded in the
// signature tables (force_routing: the ids were given, no top-k ran).
__device__ __forceinline__ void route_phases(const RouteArgs& a, uint8_t* smem_raw, int nthr, bool do_sig) {
  const int T = a.tk.T, E = a.tk.E, k = a.tk.k;
  const int W = (T + 31) >> 5;
  uint32_t* mask = reinterpret_cast<uint32_t*>(smem_raw);   // [E][W]
  uint32_t* pref = mask + (size_t)E * W;                      // [E][W] exclusive prefix popcounts
  int32_t* s_cnt = reinterpret_cast<int32_t*>(pref + (size_t)E * W);   // [E]
  int32_t* s_off = s_cnt + E;                                 // [E+1]
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  for (int i = tid; i < E * W; i += nthr) mask[i] = 0u;
  __syncthreads();

  for (int p = tid; p < T * k; p += nthr) {
    const int t = p / k;
    const int id = min(max(__ldcg(a.tk.ids + p), 0), E - 1);
    atomicOr(&mask[id * W + (t >> 5)], 1u << (t & 31));
    if (do_sig)
      sig_add(a.tk.sig_req, a.tk.sig_block, a.tk.token_req ? a.tk.token_req[t] : -1,
              a.tk.token_block ? a.tk.token_block[t] : -1, a.tk.L, a.tk.layer, E, id);
  }
  __syncthreads();
  ELDR_STAMP(6);

  for (int e = tid; e < E; e += nthr) {
    int run = 0;
    for (int w = 0; w < W; ++w) {
      pref[e * W + w] = run;
      run += __popc(mask[e * W + w]);
    }
    s_cnt[e] = run;
  }
  __syncthreads();
  ELDR_STAMP(7);

  if (warp == 0) {     // exclusive scan of cnt and ascending compaction of the active experts
    constexpr int PER = kMaxExperts / 32;
    int c[PER], csum = 0, asum = 0;
#pragma unroll
    for (int i = 0; i < PER; ++i) {
      const int e = lane * PER + i;
      c[i] = (e < E) ? s_cnt[e] : 0;
      csum += c[i];
      asum += (c[i] > 0);
    }
    int cinc = csum, ainc = asum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int cv = __shfl_up_sync(0xffffffffu, cinc, o);
      const int av = __shfl_up_sync(0xffffffffu, ainc, o);
      if (lane >= o) { cinc += cv; ainc += av; }
    }
    int coff = cinc - csum, aoff = ainc - asum;
    const int n_act = __shfl_sync(0xffffffffu, ainc, 31);
    const int total = __shfl_sync(0xffffffffu, cinc, 31);
#pragma unroll
    for (int i = 0; i < PER; ++i) {
      const int e = lane * PER + i;
      if (e < E) {
        s_off[e] = coff;
        a.off[e] = coff;
        a.cnt[e] = c[i];
        if (c[i] > 0) {
          a.active[aoff] = e;
          a.work[aoff] = make_int4(e, coff, coff, c[i]);
          ++aoff;
        }
        coff += c[i];
      }
    }
    for (int i = n_act + lane; i < E; i += 32) a.active[i] = -1;
    if (lane == 0) {
      s_off[E] = total;
      a.off[E] = total;
      *a.n_active = n_act;
      *a.n_work = n_act + a.n_shared;
    }
    if (lane < a.n_shared) a.work[n_act + lane] = make_int4(E + lane, T * k, T * k + lane * T, T);
  }
  __syncthreads();
  ELDR_STAMP(8);

  for (int p = tid; p < T * k; p += nthr) {
    const int t = p / k;
    const int e = min(max(__ldcg(a.tk.ids + p), 0), E - 1);
    const int rank = pref[e * W + (t >> 5)] + __popc(mask[e * W + (t >> 5)] & ((1u << (t & 31)) - 1u));
    const int pos = s_off[e] + rank;
    a.perm[pos] = p;
    a.pair_pos[p] = pos;
  }
}

// force_routing: ids / weights are inputs; one CTA records the signatures and builds the permutation.
__global__ void __launch_bounds__(1024) route_only_kernel(RouteArgs a) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  pdl_launch_dependents();
  route_phases(a, smem_raw, 1024, true);
}

// ------------------------------------------------------------------ a1..a4 in ONE launch
// Grid (E/8, T/8).  Every CTA computes its 8-token x 8-expert logit tile.  The LAST CTA of a token group to
// publish its tile (epoch flags + one atomicExch election; no counters to zero, so no memset in the stream)
// runs the warp top-k + signature accumulation for that group's 8 tokens, one token per warp; the last GROUP to
// finish runs the permutation / union compaction.  Latency ~ one GEMV tile + one top-k + one routing pass.
// The epoch the flags are compared with is generation + 1, the generation word living in the workspace and bumped
// by the very last CTA (every other CTA read it before publishing the tile flag that CTA waited for): nothing from
// the host is frozen into the launch, so a CUDA-graph replay elects and routes like an eager call.
struct GateRouteArgs {
  const uint16_t* x;
  const float* gate_w;
  const float* gate_bias;
  RouteArgs r;
  uint32_t* sync;      // [1] generation | [n_groups*n_etiles] tile flags | [n_groups] elected | [n_groups] group flags | [1] elected
};

__device__ __forceinline__ uint32_t ld_volatile_u32(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_volatile_u32(uint32_t* p, uint32_t v) {
  asm volatile("st.volatile.global.u32 [%0], %1;" :: "l"(p), "r"(v) : "memory");
}

// Publish `mine = epoch`, then return true in exactly one of the CTAs that observe all `n` flags set.
__device__ __forceinline__ bool publish_and_elect(uint32_t* flags, int n, int mine, uint32_t* elected,
                                                  uint32_t epoch, int* s_flag) {
  __threadfence();
  __syncthreads();
  if (threadIdx.x < 32) {
    const int lane = threadIdx.x;
    if (lane == 0) {
      st_volatile_u32(flags + mine, epoch);
      __threadfence();
    }
    __syncwarp();
    bool all = true;
    for (int i = lane; i < n; i += 32) all = all && (ld_volatile_u32(flags + i) == epoch);
    all = __all_sync(0xffffffffu, all);
    if (lane == 0) {
      int win = 0;
      if (all) win = (atomicExch(elected, epoch) != epoch);
      *s_flag = win;
    }
  }
  __syncthreads();
  const bool win = *s_flag != 0;
  if (win) __threadfence();
  return win;
}

__global__ void __launch_bounds__(256) gate_topk_route_kernel(GateRouteArgs a) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  __shared__ int s_flag;
  const TopkArgs& tk = a.r.tk;
  const int T = tk.T, E = tk.E, k = tk.k;
  const int n_etiles = gridDim.x, n_groups = gridDim.y;
  ELDR_STAMP(0);
  pdl_launch_dependents();
  const uint32_t gen_next = epoch_next_state(ld_volatile_u32(a.sync));
  const uint32_t epoch = epoch_of_state(gen_next, a.sync);
  gate_tile(a.x, a.gate_w, a.gate_bias, const_cast<float*>(tk.z), T, a.r.H, E, smem_raw);
  ELDR_STAMP(2);

  uint32_t* tile_flags = a.sync + 1;
  uint32_t* elected = tile_flags + n_groups * n_etiles;
  uint32_t* group_flags = elected + n_groups;
  uint32_t* elected2 = group_flags + n_groups;
  const int g = blockIdx.y;
  if (!publish_and_elect(tile_flags + g * n_etiles, n_etiles, blockIdx.x, elected + g, epoch, &s_flag)) return;
  ELDR_STAMP(3);

  // top-k + signature for this group's tokens: one token per warp
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int t = g * kGateTok + warp;
  if (t < T) {
    int id; float w;
    warp_topk(tk.z + (size_t)t * E, E, k, tk.renorm, lane, id, w);
    if (lane < k) {
      tk.ids[(size_t)t * k + lane] = id;
      tk.w[(size_t)t * k + lane] = w;
      sig_add(tk.sig_req, tk.sig_block, tk.token_req ? tk.token_req[t] : -1,
              tk.token_block ? tk.token_block[t] : -1, tk.L, tk.layer, E, id);
    }
  }
  ELDR_STAMP(4);
  if (!publish_and_elect(group_flags, n_groups, g, elected2, epoch, &s_flag)) return;
  ELDR_STAMP(5);
  route_phases(a.r, smem_raw, 256, false);
  if (threadIdx.x == 0) st_volatile_u32(a.sync, gen_next);
  ELDR_STAMP(10);
}

// x_perm[row] = x[token of sorted pair row]  (rows >= T*k: plain copy of x for the shared experts)
// slot_order != 0: elements permuted inside every group of eight for the MXFP4 decoder
__global__ void __launch_bounds__(256) gather_x_kernel(const uint16_t* __restrict__ x,
                                                       const int32_t* __restrict__ perm,
                                                       uint16_t* __restrict__ x_perm, int T, int H, int k,
                                                       int n_rows, int slot_order) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int row = blockIdx.x * 8 + warp;
  pdl_launch_dependents();
  pdl_wait();
  if (row >= n_rows) return;
  const int t = (row < T * k) ? perm[row] / k : row - T * k;
  const uint4* src = reinterpret_cast<const uint4*>(x + (size_t)t * H);
  uint4* dst = reinterpret_cast<uint4*>(x_perm + (size_t)row * H);
  if (!slot_order) {
    for (int c = lane; c < (H >> 3); c += 32) dst[c] = __ldg(src + c);
  } else {
    // MXFP4 path: every group of eight elements in the decoder's K-slot order e0 e4 e1 e5 e2 e6 e3 e7 (ffn_mx.cuh)
    for (int c = lane; c < (H >> 3); c += 32) {
      const uint4 v = __ldg(src + c);
      dst[c] = make_uint4(__byte_perm(v.x, v.z, 0x5410), __byte_perm(v.x, v.z, 0x7632),
                          __byte_perm(v.y, v.w, 0x5410), __byte_perm(v.y, v.w, 0x7632));
    }
  }
}

// --------------------------------------------------------------------------- a7: weighted combine
// out[t] = sum_j w[t,j]*y[pos(t,j)] (slot order) + sum_s y[shared s, t]; fp32, one RNE rounding to bf16.
// Staged + ordered instead of fp32 atomics so that results are run-to-run bit-identical.
// KMAX = compile-time bound on k (8 or kMaxTopK): with 8 slots the kernel needs half the registers, so twice as many
// warps keep loads in flight -- the prefill-shaped step reads a gigabyte of y here.
template <int KMAX>
__global__ void __launch_bounds__(256) combine_kernel(const float* __restrict__ y,
                                                      const float* __restrict__ w,
                                                      const int32_t* __restrict__ pair_pos,
                                                      uint16_t* __restrict__ out, int T, int H, int k,
                                                      int n_shared) {
  const int q_per_row = H >> 2;
  const int idx = blockIdx.x * 256 + threadIdx.x;
  pdl_wait();
  if (idx >= T * q_per_row) return;
  const int t = idx / q_per_row, c4 = idx - t * q_per_row;
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
  // two dependent loads per slot (position, then the staged row): issue all of them before the first FMA
  int pos[KMAX];
  float wt[KMAX];
  float4 v[KMAX];
#pragma unroll
  for (int j = 0; j < KMAX; ++j)
    if (j < k) { pos[j] = __ldg(pair_pos + (size_t)t * k + j); wt[j] = __ldg(w + (size_t)t * k + j); }
#pragma unroll
  for (int j = 0; j < KMAX; ++j)
    if (j < k) v[j] = __ldcs(reinterpret_cast<const float4*>(y + (size_t)pos[j] * H + (size_t)c4 * 4));
#pragma unroll
  for (int j = 0; j < KMAX; ++j)
    if (j < k) {
      acc.x = fmaf(wt[j], v[j].x, acc.x); acc.y = fmaf(wt[j], v[j].y, acc.y);
      acc.z = fmaf(wt[j], v[j].z, acc.z); acc.w = fmaf(wt[j], v[j].w, acc.w);
    }
  for (int s = 0; s < n_shared; ++s) {
    const float4 v = *reinterpret_cast<const float4*>(y + ((size_t)T * k + (size_t)s * T + t) * H + (size_t)c4 * 4);
    acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
  }
  uint2 o;
  o.x = (uint32_t)f32_to_bf16_rn(acc.x) | ((uint32_t)f32_to_bf16_rn(acc.y) << 16);
  o.y = (uint32_t)f32_to_bf16_rn(acc.z) | ((uint32_t)f32_to_bf16_rn(acc.w) << 16);
  *reinterpret_cast<uint2*>(out + (size_t)t * H + (size_t)c4 * 4) = o;
}

// ------------------------------------------------------------------- standalone signature kernels
__global__ void __launch_bounds__(256) sig_accumulate_kernel(const int32_t* __restrict__ ids,
                                                             const int32_t* __restrict__ token_req,
                                                             const int32_t* __restrict__ token_block,
                                                             int32_t* sig_req, int8_t* sig_block, int T, int E,
                                                             int k, int L, int layer) {
  const long long p = (long long)blockIdx.x * 256 + threadIdx.x;
  if (p >= (long long)T * k) return;
  const int t = (int)(p / k);
  const int e = ids[p];
  if (e < 0 || e >= E) return;
  sig_add(sig_req, sig_block, token_req ? token_req[t] : -1, token_block ? token_block[t] : -1, L, layer, E, e);
}

// All layers of a prefill-shaped call in ONE launch ("Each forward accumulates the new tokens' expert picks
// into the matching rows in a single GPU pass"): grid (token chunks of 256, layers).  A chunk's increments are first
// combined in shared memory -- the request histogram when all 256 tokens belong to one request (the prefill case), the
// KV-block rows per run of equal block ids (a new run at least every 64 tokens, so a byte of the shared-memory
// histogram cannot overflow) -- and
// only the non-zero cells / words go to global memory: ~10x fewer global atomics than one per pick.  Decode-shaped
// chunks (every token its own request) take the direct path for the request table.  Same saturating int8 semantics.
constexpr int kSigChunk = 256;
__global__ void __launch_bounds__(256) sig_accumulate_layers_kernel(const int32_t* __restrict__ ids_all,
                                                                    const int32_t* __restrict__ token_req,
                                                                    const int32_t* __restrict__ token_block,
                                                                    int32_t* sig_req, int8_t* sig_block, int T, int E,
                                                                    int k, int L, int layer0) {
  extern __shared__ __align__(16) uint8_t sig_smem[];
  const int EW = (E + 3) >> 2;                                  // 32-bit words per block row
  int32_t* rhist = reinterpret_cast<int32_t*>(sig_smem);        // [E]
  uint32_t* bhist = reinterpret_cast<uint32_t*>(rhist + E);     // [kSigChunk + 4][EW] packed byte counts per run
  __shared__ int s_slot_of[kSigChunk];
  __shared__ int s_run_blk[kSigChunk + 4];
  __shared__ int s_warp_tot[8];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int t0 = blockIdx.x * kSigChunk, layer = layer0 + blockIdx.y;
  const int n_tok = min(kSigChunk, T - t0);
  const int32_t* ids = ids_all + (size_t)blockIdx.y * T * k;
  const int t = t0 + tid;
  const int my_req = (tid < n_tok && token_req) ? token_req[t] : -1;
  const int my_blk = (tid < n_tok && token_block) ? token_block[t] : -1;
  const int req0 = token_req ? token_req[t0] : -1;
  const bool uniform = __syncthreads_and(tid >= n_tok || my_req == req0) && sig_req != nullptr && req0 >= 0;
  // runs of equal block ids -> slots (block scan of the run heads)
  int prev_blk = -2;
  if (tid > 0 && tid < n_tok && token_block) prev_blk = token_block[t - 1];
  const int head = (tid < n_tok) && (tid == 0 || my_blk != prev_blk || (tid & 63) == 0);
  const uint32_t hb = __ballot_sync(0xffffffffu, head);
  if (lane == 0) s_warp_tot[warp] = __popc(hb);
  for (int i = tid; i < E; i += 256) rhist[i] = 0;
  for (int i = tid; i < (kSigChunk + 4) * EW; i += 256) bhist[i] = 0u;
  __syncthreads();
  int base = 0, n_runs = 0;
#pragma unroll
  for (int w = 0; w < 8; ++w) { if (w < warp) base += s_warp_tot[w]; n_runs += s_warp_tot[w]; }
  const int slot = base + __popc(hb & ((2u << lane) - 1u)) - 1;
  if (tid < n_tok) s_slot_of[tid] = slot;
  if (head) s_run_blk[slot] = my_blk;
  __syncthreads();
  const bool do_blk = sig_block != nullptr;
  for (int p = tid; p < n_tok * k; p += 256) {
    const int tl = p / k;
    const int e = ids[(size_t)t0 * k + p];
    if (e < 0 || e >= E) continue;
    const int rq = token_req ? token_req[t0 + tl] : -1;
    if (uniform) atomicAdd(&rhist[e], 1);
    else if (sig_req != nullptr && rq >= 0) atomicAdd(sig_req + ((size_t)rq * L + layer) * E + e, 1);
    if (do_blk && s_run_blk[s_slot_of[tl]] >= 0) atomicAdd(&bhist[s_slot_of[tl] * EW + (e >> 2)], 1u << (8 * (e & 3)));
  }
  __syncthreads();
  if (uniform)
    for (int e = tid; e < E; e += 256)
      if (rhist[e]) atomicAdd(sig_req + ((size_t)req0 * L + layer) * E + e, rhist[e]);
  if (do_blk) {
    const bool word_ok = (E & 3) == 0;            // rows are whole 32-bit words (and 4-byte aligned: L*E*blk multiple of 4)
    for (int i = tid; i < n_runs * EW; i += 256) {
      const uint32_t add = bhist[i];
      if (!add) continue;
      const int r = i / EW, wd = i - r * EW;
      const size_t cell0 = ((size_t)s_run_blk[r] * L + layer) * E + (size_t)wd * 4;
      if (word_ok) {
        // saturating packed add as a compare-and-swap loop.  (An add followed by an undo of the excess is exact only
        // while a byte's TRANSIENT value stays below 256: three runs of 64 picks landing on a saturated cell before
        // any of them has undone its excess wrap the byte -- a block with more than 127 tokens, outside the int8
        // cells' contract but reachable through the ABI; found by a fuzz run.)
        unsigned int* word = reinterpret_cast<unsigned int*>(sig_block + cell0);
        unsigned int seen = *reinterpret_cast<volatile unsigned int*>(word);
        for (;;) {
          unsigned int nw = 0u;
#pragma unroll
          for (int b = 0; b < 4; ++b) {
            const unsigned int ob = (seen >> (8 * b)) & 0xffu, c = (add >> (8 * b)) & 0xffu;
            nw |= min(ob + c, max(ob, 127u)) << (8 * b);
          }
          if (nw == seen) break;
          const unsigned int was = atomicCAS(word, seen, nw);
          if (was == seen) break;
          seen = was;
        }
      } else {
        for (int b = 0; b < 4 && wd * 4 + b < E; ++b)
          for (unsigned int c = (add >> (8 * b)) & 0xffu; c > 0; --c) sig_add(nullptr, sig_block, -1, s_run_blk[r], L, layer, E, wd * 4 + b);
      }
    }
  }
}

__global__ void __launch_bounds__(256) sig_reset_kernel(const int32_t* __restrict__ block_ids, int8_t* sig_block,
                                                        int row_bytes) {
  const int b = block_ids[blockIdx.x];
  if (b < 0) return;
  if ((row_bytes & 3) == 0) {
    uint32_t* row = reinterpret_cast<uint32_t*>(sig_block + (size_t)b * row_bytes);
    for (int i = threadIdx.x; i < (row_bytes >> 2); i += 256) row[i] = 0u;
  } else {
    for (int i = threadIdx.x; i < row_bytes; i += 256) sig_block[(size_t)b * row_bytes + i] = 0;
  }
}

__global__ void __launch_bounds__(256) sig_readout_kernel(const int32_t* __restrict__ block_ids,
                                                          const int32_t* __restrict__ req_off,
                                                          const int8_t* __restrict__ sig_block,
                                                          int32_t* __restrict__ sig_out, int row_cells) {
  const int r = blockIdx.y;
  const int b0 = req_off[r], b1 = req_off[r + 1];
  if ((row_cells & 15) == 0) {
    // 16 cells per thread: one 16-byte load per block row, four rows in flight (a request sums 32-256 rows)
    for (int c16 = blockIdx.x * 256 + threadIdx.x; c16 < (row_cells >> 4); c16 += gridDim.x * 256) {
      int acc[16];
#pragma unroll
      for (int j = 0; j < 16; ++j) acc[j] = 0;
      for (int i = b0; i < b1; i += 4) {
        uint4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int b = (i + u < b1) ? block_ids[i + u] : -1;
          v[u] = b >= 0 ? ld_nc_v4(sig_block + (size_t)b * row_cells + (size_t)c16 * 16) : make_uint4(0u, 0u, 0u, 0u);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const uint32_t wv[4] = {v[u].x, v[u].y, v[u].z, v[u].w};
#pragma unroll
          for (int j = 0; j < 16; ++j) acc[j] += (int)(int8_t)((wv[j >> 2] >> (8 * (j & 3))) & 0xffu);
        }
      }
      int4* dst = reinterpret_cast<int4*>(sig_out + (size_t)r * row_cells + (size_t)c16 * 16);
#pragma unroll
      for (int q = 0; q < 4; ++q) dst[q] = make_int4(acc[4 * q], acc[4 * q + 1], acc[4 * q + 2], acc[4 * q + 3]);
    }
    return;
  }
  for (int c = blockIdx.x * 256 + threadIdx.x; c < row_cells; c += gridDim.x * 256) {
    int acc = 0;
    for (int i = b0; i < b1; ++i) {
      const int b = block_ids[i];
      if (b >= 0) acc += (int)sig_block[(size_t)b * row_cells + c];
    }
    sig_out[(size_t)r * row_cells + c] = acc;
  }
}

}  // namespace eldr
