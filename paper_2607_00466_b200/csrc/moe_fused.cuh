// The whole decode step of one MoE layer in ONE persistent launch (PAPER.md:79
// "the gate partitions the batch among experts ... each step fetches the weights of every expert the batch
// activates"; PAPER.md:198/:253 signature counts).  One CTA per SM, 8 warps.
//
//   G  gate GEMV: 8-token x 8-expert logit tiles spread over the grid (fp32 FMA, gate rows prefetched 16 deep
//      while the x tile lands in shared memory); each tile publishes an epoch flag.
//   K  top-k: the CTA that owns token group g polls the group's tile flags, runs a redux-based warp top-k
//      (+ fused signature increments), publishes the group flag.
//   R  routing, redundantly in EVERY CTA from the 4*T*k bytes of ids: membership bitmasks -> counts ->
//      offsets -> union-compacted work list -> token<->position maps, all in shared memory (no second
//      election, no route/gather kernels, no work-list round trip through HBM).  CTA 0 also writes the
//      routing outputs of the C ABI (active list, n_active, cnt/off/perm/pair_pos).
//   F  expert FFN on tcgen05 + TMEM, swap-AB (weights = M operand, the expert's tokens = N operand).  Work
//      units = [w1/w3 tiles of all active experts, expert-major] ++ [w2 tiles, expert-major], claimed from a
//      global counter (first unit static) by the weights-producer lane and broadcast to the other roles through
//      a 4-slot shared-memory ring.  Weights: TMA (SWIZZLE_128B, evict_first), 16 KiB per stage.  Activations:
//      a producer warp gathers the expert's token rows with cp.async straight from x (w1/w3) or h (w2) into the
//      swizzled K-major B tile -- the permutation is never materialised in HBM.  A w2 unit of expert e waits on
//      the epoch flags of e's w1/w3 tiles (release/acquire through L2); the queue order makes this
//      deadlock-free: a unit only ever waits on units claimed before it.
//   C  ordered combine: after a flag barrier over the grid, out[t] = sum_j w[t,j]*y[pos(t,j)] (+ shared) in
//      slot order, one RNE rounding to bf16: run-to-run bit-identical.
//
// No counter needs zeroing by the host: flags compare against epoch = gen+1, gen lives in the workspace and is
// bumped by CTA 0 after the last barrier (so the launch is CUDA-graph capturable and robust to a workspace of
// arbitrary initial contents up to a 2^-32 flag collision).
#pragma once
#include "device_utils.cuh"
#include "ffn_umma.cuh"
#include "gate_route.cuh"

namespace eldr {

constexpr int kFusedThreads = 256;
constexpr int kFusedMaxT = 256;
constexpr int kSchedSlots = 4;
constexpr int kXLag = 4;                  // cp.async groups kept in flight by the activations producer

// sync region (uint32 words) at the START of the layer workspace
constexpr int kSyncGen = 0;
constexpr int kSyncCounter = 1;
constexpr int kSyncSchedReady = 2;
constexpr int kSyncDone = 32;             // [256]  per-CTA "all my units are finished"
constexpr int kSyncGroup = kSyncDone + 256;     // [32]   per token group "ids/weights written"
constexpr int kSyncTile = kSyncGroup + 32;      // [32 groups][32 expert tiles] gate logits written
constexpr int kSyncHReady = kSyncTile + 1024;   // [(E+ns) work slots][tilesA] h tile written

struct FusedArgs {
  const uint16_t* x;
  const float* gate_w;
  const float* gate_bias;
  TopkArgs tk;                 // z, ids, w, token maps, signature tables, T, E, k, L, layer, renorm
  int force_routing, n_shared, H, I;
  int32_t* cnt;                // routing outputs written by CTA 0
  int32_t* off;
  int32_t* perm;
  int32_t* pair_pos;
  int4* work;
  int32_t* n_work;
  int32_t* active;
  int32_t* n_active;
  uint32_t* sync;
  uint16_t* hbuf;              // [T*(k+ns), I] bf16
  float* ybuf;                 // [T*(k+ns), H] fp32
  uint16_t* out;               // [T,H] bf16
  int np, stages;              // token rows per pass (64|128), smem ring depth
};

__device__ __forceinline__ void flag_release(uint32_t* p, uint32_t v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" :: "l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t flag_acquire(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
// One warp waits until flags[0..n) all equal epoch (lanes stride over the flags).  Traps instead of hanging.
__device__ __forceinline__ void warp_wait_flags(const uint32_t* flags, int n, uint32_t epoch, int lane) {
  for (int i = lane; i < n; i += 32) {
    uint32_t spins = 0;
    while (flag_acquire(flags + i) != epoch) {
      if (++spins > (1u << 24)) __trap();
    }
  }
  __syncwarp();
}

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" :: "n"(N) : "memory"); }
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ------------------------------------------------------------------------------------ G: one logit tile
// 8 tokens (group g) x 8 experts (tile et), warp w owns expert et*8+w.  The first 16 float4 of the gate row
// are requested BEFORE the x tile is staged, so the two DRAM/L2 latencies overlap.
__device__ __forceinline__ void fused_gate_tile(const FusedArgs& a, int et, int g, uint8_t* smem_raw) {
  const int T = a.tk.T, H = a.H, E = a.tk.E;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int t0 = g * kGateTok;
  const int e = et * kGateExp + warp;
  const int q_per_row = H >> 2;
  constexpr int kDepth = 16;
  const float4* wrow = reinterpret_cast<const float4*>(a.gate_w + (size_t)(e < E ? e : 0) * H);
  float4 wv[kDepth];
#pragma unroll
  for (int u = 0; u < kDepth; ++u) {
    const int c4 = lane + 32 * u;
    wv[u] = (e < E && c4 < q_per_row) ? __ldg(wrow + c4) : make_float4(0.f, 0.f, 0.f, 0.f);
  }
  uint4* xs4 = reinterpret_cast<uint4*>(smem_raw);
  const int vec_per_row = H >> 3;
  __syncthreads();                       // the previous tile's readers are done with the x tile
  for (int v = tid; v < kGateTok * vec_per_row; v += kFusedThreads) {
    const int t = v / vec_per_row, c = v - t * vec_per_row;
    uint4 val = make_uint4(0u, 0u, 0u, 0u);
    if (t0 + t < T) val = __ldcg(reinterpret_cast<const uint4*>(a.x + (size_t)(t0 + t) * H + (size_t)c * 8));
    xs4[v] = val;
  }
  __syncthreads();
  float acc[kGateTok];
#pragma unroll
  for (int t = 0; t < kGateTok; ++t) acc[t] = 0.f;
  const uint2* xs2 = reinterpret_cast<const uint2*>(smem_raw);
  for (int base = 0; base < q_per_row; base += 32 * kDepth) {
    if (base > 0) {
#pragma unroll
      for (int u = 0; u < kDepth; ++u) {
        const int c4 = base + lane + 32 * u;
        wv[u] = (e < E && c4 < q_per_row) ? __ldg(wrow + c4) : make_float4(0.f, 0.f, 0.f, 0.f);
      }
    }
#pragma unroll
    for (int u = 0; u < kDepth; ++u) {
      const int c4 = base + lane + 32 * u;
      if (c4 < q_per_row) {
#pragma unroll
        for (int t = 0; t < kGateTok; ++t) {
          const uint2 xv = xs2[t * q_per_row + c4];
          float s = acc[t];
          s = fmaf(wv[u].x, bf16_lo(xv.x), s);
          s = fmaf(wv[u].y, bf16_hi(xv.x), s);
          s = fmaf(wv[u].z, bf16_lo(xv.y), s);
          s = fmaf(wv[u].w, bf16_hi(xv.y), s);
          acc[t] = s;
        }
      }
    }
  }
#pragma unroll
  for (int t = 0; t < kGateTok; ++t) {
    float s = acc[t];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    acc[t] = s;
  }
  if (lane == 0 && e < E) {
    const float b = a.gate_bias ? a.gate_bias[e] : 0.f;
    float* z = const_cast<float*>(a.tk.z);
#pragma unroll
    for (int t = 0; t < kGateTok; ++t)
      if (t0 + t < T) z[(size_t)(t0 + t) * E + e] = acc[t] + b;
  }
}

// ------------------------------------------------------------------------------- K: redux-based warp top-k
// Same order as warp_topk (z descending, lower id on ties), but each of the k rounds is two warp reductions
// (redux.sync max on an order-preserving uint key, redux.sync min on the candidate id) instead of ten shuffles.
__device__ __forceinline__ uint32_t f32_order_key(float f) {
  const uint32_t b = __float_as_uint(f + 0.0f);       // -0 -> +0 so that equal values have equal keys
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float f32_from_order_key(uint32_t k) {
  return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}
__device__ __forceinline__ void warp_topk_redux(const float* __restrict__ zrow, int E, int k, int renorm, int lane,
                                                int& my_id, float& my_w) {
  constexpr int NV = kMaxExperts / 32;
  uint32_t key[NV];
#pragma unroll
  for (int i = 0; i < NV; ++i) {
    const int e = lane + 32 * i;
    key[i] = (e < E) ? f32_order_key(__ldcg(zrow + e)) : 0u;      // 0 = "absent": below every finite key
  }
  float denom_all = 0.f;
  uint32_t kmax_all = 0u;
  if (!renorm) {
    uint32_t m = key[0];
#pragma unroll
    for (int i = 1; i < NV; ++i) m = max(m, key[i]);
    kmax_all = __reduce_max_sync(0xffffffffu, m);
    const float zmax = f32_from_order_key(kmax_all);
#pragma unroll
    for (int i = 0; i < NV; ++i)
      if (lane + 32 * i < E) denom_all += expf(f32_from_order_key(key[i]) - zmax);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) denom_all += __shfl_xor_sync(0xffffffffu, denom_all, o);
  }
  uint32_t sel_key = 0u, first_key = 0u;
  int sel_id = 0;
  for (int j = 0; j < k; ++j) {
    uint32_t m = key[0];
#pragma unroll
    for (int i = 1; i < NV; ++i) m = max(m, key[i]);
    const uint32_t wm = __reduce_max_sync(0xffffffffu, m);
    int cand = 0x7fffffff;
#pragma unroll
    for (int i = NV - 1; i >= 0; --i)
      if (key[i] == wm) cand = lane + 32 * i;                    // ends on the lowest matching id of this lane
    const int wid = (int)__reduce_min_sync(0xffffffffu, (unsigned)cand);
    if ((wid & 31) == lane) {
#pragma unroll
      for (int i = 0; i < NV; ++i)
        if ((wid >> 5) == i) key[i] = 0u;
    }
    if (j == 0) first_key = wm;
    if (lane == j) { sel_key = wm; sel_id = wid; }
  }
  sel_id = min(max(sel_id, 0), E - 1);          // NaN/Inf inputs are outside the contract; never index out of [0,E)
  const float zmax = f32_from_order_key(first_key);
  const float ev = (lane < k) ? expf(f32_from_order_key(sel_key) - zmax) : 0.f;
  float denom = ev;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) denom += __shfl_xor_sync(0xffffffffu, denom, o);
  my_id = sel_id;
  my_w = renorm ? ev / denom : ev / denom_all;
}

// ------------------------------------------------------------------------------------ shared-memory plan
struct FusedSmem {
  uint32_t stage_base;     // S stages of [16 KiB weights | np*128 B activations], 1024-aligned
  uint32_t bar_base;       // full[S], empty[S], tfull[2], tempty[2], sfull[4], sempty[4]
  uint32_t tmem_slot;
  int4* ring;              // [kSchedSlots] {unit or -1,..}
  int4* work;              // [E+ns] {expert, x_row0, out_row0, m}
  int32_t* n_work;         // [1]
  uint16_t* tok_of_pos;    // [T*k (+T)]
  uint16_t* pos_of_pair;   // [T*k]
};

__host__ __device__ inline size_t fused_smem_bytes(int S, int np, int E, int ns, int T, int k) {
  size_t o = (size_t)S * (kUmmaWBytes + (size_t)np * 128);
  o += (2 * (size_t)S + 12) * 8 + 16;                    // barriers + tmem slot
  o += kSchedSlots * 16;
  o += (size_t)(E + ns) * 16 + 16;
  o += (((size_t)T * k + T) * 2 + 15) / 16 * 16;
  o += ((size_t)T * k * 2 + 15) / 16 * 16;
  return o + 1024;                                       // alignment slack
}

// ---------------------------------------------------------------------------------------- R: local routing
// Scratch (mask, pref, s_cnt, s_off) lives in the (not yet used) stage area.
__device__ __forceinline__ void fused_route(const FusedArgs& a, const FusedSmem& sm, uint8_t* scratch, bool is_cta0) {
  const int T = a.tk.T, E = a.tk.E, k = a.tk.k, ns = a.n_shared;
  const int W = (T + 31) >> 5;
  uint32_t* mask = reinterpret_cast<uint32_t*>(scratch);     // [E][W]
  uint32_t* pref = mask + (size_t)E * W;                      // [E][W]
  int32_t* s_cnt = reinterpret_cast<int32_t*>(pref + (size_t)E * W);
  int32_t* s_off = s_cnt + E;                                 // [E+1]
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const bool do_sig = is_cta0 && a.force_routing;

  for (int i = tid; i < E * W; i += kFusedThreads) mask[i] = 0u;
  __syncthreads();
  for (int p = tid; p < T * k; p += kFusedThreads) {
    const int t = p / k;
    const int id = min(max(__ldcg(a.tk.ids + p), 0), E - 1);
    atomicOr(&mask[id * W + (t >> 5)], 1u << (t & 31));
    if (do_sig)
      sig_add(a.tk.sig_req, a.tk.sig_block, a.tk.token_req ? a.tk.token_req[t] : -1,
              a.tk.token_block ? a.tk.token_block[t] : -1, a.tk.L, a.tk.layer, E, id);
  }
  __syncthreads();
  for (int e = tid; e < E; e += kFusedThreads) {
    int run = 0;
    for (int w = 0; w < W; ++w) {
      pref[e * W + w] = run;
      run += __popc(mask[e * W + w]);
    }
    s_cnt[e] = run;
  }
  __syncthreads();
  if (warp == 0) {
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
        if (is_cta0) { a.off[e] = coff; a.cnt[e] = c[i]; }
        if (c[i] > 0) {
          const int4 wk = make_int4(e, coff, coff, c[i]);
          sm.work[aoff] = wk;
          if (is_cta0) { a.active[aoff] = e; a.work[aoff] = wk; }
          ++aoff;
        }
        coff += c[i];
      }
    }
    if (is_cta0)
      for (int i = n_act + lane; i < E; i += 32) a.active[i] = -1;
    if (lane == 0) {
      s_off[E] = total;
      *sm.n_work = n_act + ns;
      if (is_cta0) { a.off[E] = total; *a.n_active = n_act; *a.n_work = n_act + ns; }
    }
    if (lane < ns) {
      const int4 wk = make_int4(E + lane, T * k, T * k + lane * T, T);
      sm.work[n_act + lane] = wk;
      if (is_cta0) a.work[n_act + lane] = wk;
    }
  }
  __syncthreads();
  for (int p = tid; p < T * k; p += kFusedThreads) {
    const int t = p / k;
    const int e = min(max(__ldcg(a.tk.ids + p), 0), E - 1);
    const int rank = pref[e * W + (t >> 5)] + __popc(mask[e * W + (t >> 5)] & ((1u << (t & 31)) - 1u));
    const int pos = s_off[e] + rank;
    sm.tok_of_pos[pos] = (uint16_t)t;
    sm.pos_of_pair[p] = (uint16_t)pos;
    if (is_cta0) { a.perm[pos] = p; a.pair_pos[p] = pos; }
  }
  if (ns)
    for (int t = tid; t < T; t += kFusedThreads) sm.tok_of_pos[T * k + t] = (uint16_t)t;
  __syncthreads();
}

// ------------------------------------------------------------------------------------------- the kernel
struct UnitInfo { int mode, ent, rt; };

__global__ void __launch_bounds__(kFusedThreads, 1)
moe_fused_kernel(const __grid_constant__ CUtensorMap tm_w13, const __grid_constant__ CUtensorMap tm_sw13,
                 const __grid_constant__ CUtensorMap tm_w2, const __grid_constant__ CUtensorMap tm_sw2,
                 const FusedArgs a) {
  extern __shared__ uint8_t smem_dyn[];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int G = gridDim.x, cta = blockIdx.x;
  const int T = a.tk.T, E = a.tk.E, k = a.tk.k, H = a.H, I = a.I, ns = a.n_shared;
  const int NP = a.np, S = a.stages;
  const uint32_t stage_bytes = kUmmaWBytes + NP * 128;

  FusedSmem sm;
  {
    const uint32_t base = (smem_u32(smem_dyn) + 1023u) & ~1023u;
    uint8_t* gen = smem_dyn + (base - smem_u32(smem_dyn));
    sm.stage_base = base;
    size_t o = (size_t)S * stage_bytes;
    sm.bar_base = base + (uint32_t)o;
    o += (2 * (size_t)S + 12) * 8;
    sm.tmem_slot = base + (uint32_t)o;
    o += 16;
    sm.ring = reinterpret_cast<int4*>(gen + o);
    o += kSchedSlots * 16;
    sm.work = reinterpret_cast<int4*>(gen + o);
    o += (size_t)(E + ns) * 16;
    sm.n_work = reinterpret_cast<int32_t*>(gen + o);
    o += 16;
    sm.tok_of_pos = reinterpret_cast<uint16_t*>(gen + o);
    o += (((size_t)T * k + T) * 2 + 15) / 16 * 16;
    sm.pos_of_pair = reinterpret_cast<uint16_t*>(gen + o);
  }
  uint8_t* scratch = smem_dyn + (sm.stage_base - smem_u32(smem_dyn));     // stage area, generic pointer
  auto full_bar = [&](int s) { return sm.bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return sm.bar_base + 8u * (S + s); };
  auto tfull_bar = [&](int b) { return sm.bar_base + 8u * (2 * S + b); };
  auto tempty_bar = [&](int b) { return sm.bar_base + 8u * (2 * S + 2 + b); };
  auto sfull_bar = [&](int b) { return sm.bar_base + 8u * (2 * S + 4 + b); };
  auto sempty_bar = [&](int b) { return sm.bar_base + 8u * (2 * S + 8 + b); };

  // ------------------------------------------------------------- prologue (overlaps the previous kernel's tail)
  if (tid == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(full_bar(s), 2); mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(tfull_bar(b), 1); mbar_init(tempty_bar(b), 4); }
    for (int b = 0; b < kSchedSlots; ++b) { mbar_init(sfull_bar(b), 1); mbar_init(sempty_bar(b), 6); }
    mbar_fence_init();
    tma_prefetch_desc(&tm_w13);
    tma_prefetch_desc(&tm_w2);
  }
  const uint32_t tmem_cols = 2 * NP;
  if (warp == 6) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(sm.tmem_slot), "r"(tmem_cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(sm.tmem_slot));
  pdl_launch_dependents();
  pdl_wait();

  const uint32_t epoch = __ldcg(a.sync + kSyncGen) + 1u;
  if (cta == 0 && tid == 0) {
    // dynamic unit counter: unit `cta` is everyone's first (static), the counter hands out the rest
    a.sync[kSyncCounter] = (uint32_t)G;
    __threadfence();
    flag_release(a.sync + kSyncSchedReady, epoch);
  }

  // ------------------------------------------------------------------------------ G + K: gate and top-k
  if (!a.force_routing) {
    const int n_et = (E + kGateExp - 1) / kGateExp, n_gr = (T + kGateTok - 1) / kGateTok;
    const int n_tiles = n_et * n_gr;
    for (int tile = cta; tile < n_tiles; tile += G) {
      const int g = tile / n_et, et = tile - g * n_et;
      fused_gate_tile(a, et, g, scratch);
      __threadfence();
      __syncthreads();
      if (tid == 0) flag_release(a.sync + kSyncTile + g * 32 + et, epoch);
    }
    for (int g = ((cta - n_tiles % G) + G) % G; g < n_gr; g += G) {       // owner(g) = (n_tiles + g) % G
      if (warp == 0) warp_wait_flags(a.sync + kSyncTile + g * 32, n_et, epoch, lane);
      __syncthreads();
      const int t = g * kGateTok + warp;
      if (t < T) {
        int id; float w;
        warp_topk_redux(a.tk.z + (size_t)t * E, E, k, a.tk.renorm, lane, id, w);
        if (lane < k) {
          a.tk.ids[(size_t)t * k + lane] = id;
          a.tk.w[(size_t)t * k + lane] = w;
          sig_add(a.tk.sig_req, a.tk.sig_block, a.tk.token_req ? a.tk.token_req[t] : -1,
                  a.tk.token_block ? a.tk.token_block[t] : -1, a.tk.L, a.tk.layer, E, id);
        }
      }
      __threadfence();
      __syncthreads();
      if (tid == 0) flag_release(a.sync + kSyncGroup + g, epoch);
    }
    if (warp == 0) warp_wait_flags(a.sync + kSyncGroup, n_gr, epoch, lane);
    __syncthreads();
  }

  // ------------------------------------------------------------------------------------------ R: routing
  fused_route(a, sm, scratch, cta == 0);

  // ------------------------------------------------------------------------------------------ F: expert FFN
  const int n_work = *sm.n_work;
  const int tilesA = I / 64, tilesB = (H + 127) / 128;
  const int nA = n_work * tilesA, total_units = nA + n_work * tilesB;
  const int kitA = H / 64, kitB = I / 64;
  uint32_t* hready = a.sync + kSyncHReady;
  auto decode = [&](int u) {
    UnitInfo r;
    if (u < nA) { r.mode = 0; r.ent = u / tilesA; r.rt = u - r.ent * tilesA; }
    else { const int v = u - nA; r.mode = 1; r.ent = v / tilesB; r.rt = v - r.ent * tilesB; }
    return r;
  };
  // consumer side of the unit ring: lane 0 reads, frees the slot, broadcasts
  auto next_unit = [&](uint32_t n) {
    int u = 0;
    if (lane == 0) {
      const int slot = n & (kSchedSlots - 1);
      mbar_wait(sfull_bar(slot), (n / kSchedSlots) & 1);
      u = sm.ring[slot].x;
      mbar_arrive(sempty_bar(slot));
    }
    return __shfl_sync(0xffffffffu, u, 0);
  };

  if (warp == 4) {
    // ================================================================ scheduler + weights producer (one lane)
    if (lane == 0) {
      const uint64_t pol = l2_policy_evict_first();
      { uint32_t spins = 0; while (flag_acquire(a.sync + kSyncSchedReady) != epoch) if (++spins > (1u << 24)) __trap(); }
      uint32_t it = 0, n = 0;
      int u = cta;
      while (true) {
        const int slot = n & (kSchedSlots - 1);
        mbar_wait(sempty_bar(slot), ((n / kSchedSlots) & 1) ^ 1);
        sm.ring[slot] = make_int4(u < total_units ? u : -1, 0, 0, 0);
        mbar_arrive(sfull_bar(slot));
        ++n;
        if (u >= total_units) break;
        const UnitInfo ui = decode(u);
        const int4 wk = sm.work[ui.ent];
        const bool shared = wk.x >= E;
        const int we = shared ? wk.x - E : wk.x;
        const int k_iters = ui.mode == 0 ? kitA : kitB;
        const CUtensorMap* tmw = ui.mode == 0 ? (shared ? &tm_sw13 : &tm_w13) : (shared ? &tm_sw2 : &tm_w2);
        const int claim_at = k_iters > 6 ? k_iters - 6 : 0;
        int next = -1;
        for (int n0 = 0; n0 < wk.w; n0 += NP) {
          const bool last_pass = n0 + NP >= wk.w;
          for (int kc = 0; kc < k_iters; ++kc, ++it) {
            if (last_pass && kc == claim_at) next = (int)atomicAdd(a.sync + kSyncCounter, 1u);
            const int s = it % S;
            mbar_wait(empty_bar(s), ((it / S) & 1) ^ 1);
            mbar_arrive_expect_tx(full_bar(s), kUmmaWBytes);
            const uint32_t dst = sm.stage_base + s * stage_bytes;
            if (ui.mode == 0) tma_load_5d(dst, tmw, kc * 64, 0, 0, ui.rt * 4, we, full_bar(s), pol);
            else tma_load_2d(dst, tmw, kc * 64, we * H + ui.rt * 128, full_bar(s), pol);
          }
        }
        u = next;
      }
    }
    __syncwarp();
  } else if (warp == 5) {
    // ================================================================ activations producer (cp.async gather)
    uint32_t it = 0, pend = 0;
    auto drain = [&]() {
      cp_async_wait<0>();
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0)
        for (uint32_t j = 0; j < pend; ++j) mbar_arrive(full_bar((it - pend + j) % S));
      pend = 0;
    };
    for (uint32_t n = 0;; ++n) {
      const int u = next_unit(n);
      if (u < 0) break;
      const UnitInfo ui = decode(u);
      const int4 wk = sm.work[ui.ent];
      const int k_iters = ui.mode == 0 ? kitA : kitB;
      if (ui.mode == 1) {
        // every h tile of this expert must have landed; first hand over everything already in flight, or a
        // unit of THIS CTA that the flags depend on could starve
        drain();
        warp_wait_flags(hready + (size_t)ui.ent * tilesA, tilesA, epoch, lane);
      }
      const size_t row_bytes = (size_t)(ui.mode == 0 ? H : I) * 2;
      const uint8_t* src_base = reinterpret_cast<const uint8_t*>(ui.mode == 0 ? a.x : a.hbuf);
      for (int n0 = 0; n0 < wk.w; n0 += NP) {
        const int n_here = min(NP, wk.w - n0);
        const int n_pad = (n_here + 15) & ~15;
        for (int kc = 0; kc < k_iters; ++kc) {
          const int s = it % S;
          if (lane == 0) mbar_wait(empty_bar(s), ((it / S) & 1) ^ 1);
          __syncwarp();
          const uint32_t dst = sm.stage_base + s * stage_bytes + kUmmaWBytes;
          for (int q = lane; q < n_pad * 8; q += 32) {
            const int r = q >> 3, c = q & 7;
            const int rr = min(r, n_here - 1);                     // padding rows: any valid row (result ignored)
            const size_t grow = ui.mode == 0 ? (size_t)sm.tok_of_pos[wk.y + n0 + rr] : (size_t)(wk.z + n0 + rr);
            cp_async16(dst + r * 128 + ((c ^ (r & 7)) << 4), src_base + grow * row_bytes + (size_t)kc * 128 + c * 16);
          }
          cp_async_commit();
          ++it;
          ++pend;
          if (pend > kXLag) {
            cp_async_wait<kXLag>();
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(full_bar((it - pend) % S));
            --pend;
          }
        }
      }
    }
    drain();
  } else if (warp == 6) {
    // ================================================================ MMA issuer
    uint32_t it = 0, pass = 0;
    for (uint32_t n = 0;; ++n) {
      const int u = next_unit(n);
      if (u < 0) break;
      const UnitInfo ui = decode(u);
      const int4 wk = sm.work[ui.ent];
      const int k_iters = ui.mode == 0 ? kitA : kitB;
      for (int n0 = 0; n0 < wk.w; n0 += NP, ++pass) {
        const int n_pad = (min(NP, wk.w - n0) + 15) & ~15;
        const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n_pad >> 3) << 17) | (8u << 24);
        const int buf = pass & 1;
        mbar_wait(tempty_bar(buf), ((pass >> 1) & 1) ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + buf * NP;
        for (int kc = 0; kc < k_iters; ++kc, ++it) {
          const int s = it % S;
          mbar_wait(full_bar(s), (it / S) & 1);
          tc_fence_after();
          if (lane == 0) {
            const uint32_t sa = sm.stage_base + s * stage_bytes;
            const uint64_t da = umma_desc_sw128(sa), db = umma_desc_sw128(sa + kUmmaWBytes);
#pragma unroll
            for (int kk = 0; kk < 4; ++kk)
              umma_bf16(d_tmem, da + 2 * kk, db + 2 * kk, idesc, (kc | kk) ? 1u : 0u);
            umma_commit(empty_bar(s));
            if (kc == k_iters - 1) umma_commit(tfull_bar(buf));
          }
          __syncwarp();
        }
      }
    }
  } else if (warp < 4) {
    // ================================================================ epilogue (TMEM lane quarter = warp)
    const int qtr = warp;
    uint32_t pass = 0;
    for (uint32_t n = 0;; ++n) {
      const int u = next_unit(n);
      if (u < 0) break;
      const UnitInfo ui = decode(u);
      const int4 wk = sm.work[ui.ent];
      for (int n0 = 0; n0 < wk.w; n0 += NP, ++pass) {
        const int n_here = min(NP, wk.w - n0);
        const int buf = pass & 1;
        mbar_wait(tfull_bar(buf), (pass >> 1) & 1);
        tc_fence_after();
        const uint32_t t_addr = tmem_base + buf * NP + ((uint32_t)(qtr * 32) << 16);
        for (int c0 = 0; c0 < n_here; c0 += 16) {
          float v[16];
          tmem_ld16(t_addr + c0, v);
          if (ui.mode == 0) {
            // lanes 0-15: g for i = rt*64 + 16*qtr + lane; lanes 16-31: u for the same i
            const bool lo = lane < 16;
            const int i = ui.rt * 64 + 16 * qtr + (lane & 15);
#pragma unroll
            for (int kk = 0; kk < 8; ++kk) {
              const float send = lo ? v[8 + kk] : v[kk];
              const float recv = __shfl_xor_sync(0xffffffffu, send, 16);
              const float gv = lo ? v[kk] : recv;
              const float uv = lo ? recv : v[8 + kk];
              const int tok = n0 + c0 + (lo ? kk : 8 + kk);
              if (tok < wk.w) a.hbuf[(size_t)(wk.z + tok) * I + i] = f32_to_bf16_rn(silu_f(gv) * uv);
            }
          } else {
            const int r = ui.rt * 128 + 32 * qtr + lane;
            if (r < H) {
#pragma unroll
              for (int kk = 0; kk < 16; ++kk) {
                const int tok = n0 + c0 + kk;
                if (tok < wk.w) a.ybuf[(size_t)(wk.z + tok) * H + r] = v[kk];
              }
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(tempty_bar(buf));
      }
      if (ui.mode == 0) {
        // publish "h tile (ent, rt) written": every writer fences, the four epilogue warps meet, one releases
        __threadfence();
        asm volatile("bar.sync 1, 128;" ::: "memory");
        if (tid == 0) flag_release(hready + (size_t)ui.ent * tilesA + ui.rt, epoch);
      }
    }
  }

  // ------------------------------------------------------------------------------ grid barrier, then C: combine
  __threadfence();
  __syncthreads();
  if (tid == 0) flag_release(a.sync + kSyncDone + cta, epoch);
  if (warp == 0) warp_wait_flags(a.sync + kSyncDone, G, epoch, lane);
  __syncthreads();
  {
    const int q_per_row = H >> 2;
    for (int idx = cta * kFusedThreads + tid; idx < T * q_per_row; idx += G * kFusedThreads) {
      const int t = idx / q_per_row, c4 = idx - t * q_per_row;
      int pos[kMaxTopK];
      float wt[kMaxTopK];
      float4 v[kMaxTopK];
#pragma unroll
      for (int j = 0; j < kMaxTopK; ++j)
        if (j < k) { pos[j] = sm.pos_of_pair[t * k + j]; wt[j] = __ldcg(a.tk.w + t * k + j); }
#pragma unroll
      for (int j = 0; j < kMaxTopK; ++j)
        if (j < k) v[j] = __ldcg(reinterpret_cast<const float4*>(a.ybuf + (size_t)pos[j] * H + (size_t)c4 * 4));
      float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
      for (int j = 0; j < kMaxTopK; ++j)
        if (j < k) {
          acc.x = fmaf(wt[j], v[j].x, acc.x); acc.y = fmaf(wt[j], v[j].y, acc.y);
          acc.z = fmaf(wt[j], v[j].z, acc.z); acc.w = fmaf(wt[j], v[j].w, acc.w);
        }
      for (int s = 0; s < ns; ++s) {
        const float4 sv = __ldcg(reinterpret_cast<const float4*>(a.ybuf + ((size_t)T * k + (size_t)s * T + t) * H + (size_t)c4 * 4));
        acc.x += sv.x; acc.y += sv.y; acc.z += sv.z; acc.w += sv.w;
      }
      uint2 o;
      o.x = (uint32_t)f32_to_bf16_rn(acc.x) | ((uint32_t)f32_to_bf16_rn(acc.y) << 16);
      o.y = (uint32_t)f32_to_bf16_rn(acc.z) | ((uint32_t)f32_to_bf16_rn(acc.w) << 16);
      *reinterpret_cast<uint2*>(a.out + (size_t)t * H + (size_t)c4 * 4) = o;
    }
  }
  if (cta == 0 && tid == 0) a.sync[kSyncGen] = epoch;      // every CTA read gen before its done flag

  tc_fence_before();
  __syncthreads();
  if (warp == 6) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_base), "r"(tmem_cols) : "memory");
  }
}

}  // namespace eldr
