// a4 (permutation / union compaction) for PREFILL-shaped calls of eldr_moe_decode_layer (T in the thousands:
// SURVEY.md 8(f) row 2; PAPER.md:168, :261 -- where the paper captures its signatures).  The decode-shaped
// route_phases keeps one membership bitmask [E][T/32] in ONE CTA's shared memory (T <= 1024); here the tokens are
// cut into chunks of 1024 and the same deterministic counting sort runs in two launches:
//   route_count_kernel    chunk b: bitmask of its 1024 tokens -> cnt_blk[b][e] (+ the signature increments when the
//                         ids were given, force_routing)
//   route_scatter_kernel  chunk b: rebuilds its bitmask, sums cnt_blk over the chunks (expert totals) and over the
//                         chunks before b (its base inside each expert's segment), scans the totals, and writes
//                         perm / pair_pos:  pos = off[e] + before_b[e] + rank of the token inside the chunk.
//                         Chunk 0 also writes the ABI's routing outputs (cnt, off, active, n_active, work list).
// No global atomics, so perm is the canonical order (ascending token inside each expert's segment) on every run.
#pragma once
#include "gate_route.cuh"

namespace eldr {

constexpr int kRouteChunk = 1024;   // tokens per routing CTA (32 mask words per expert)
constexpr int kRouteBigThreads = 1024;

struct RouteBigArgs {
  RouteArgs r;
  int32_t* cnt_blk;    // [n_chunks][E]
  int do_sig;
};

__host__ __device__ inline size_t route_big_smem_bytes(int E) {
  return (size_t)E * 32 * 8 + (size_t)(3 * E + 1) * 4;      // mask, pref | total, before, off
}

__device__ __forceinline__ void route_big_masks(const RouteBigArgs& a, uint32_t* mask, int t0, int Tc, bool sig) {
  const int E = a.r.tk.E, k = a.r.tk.k;
  for (int i = threadIdx.x; i < E * 32; i += kRouteBigThreads) mask[i] = 0u;
  __syncthreads();
  for (int p = threadIdx.x; p < Tc * k; p += kRouteBigThreads) {
    const int tl = p / k;
    const int id = min(max(__ldcg(a.r.tk.ids + (size_t)t0 * k + p), 0), E - 1);
    atomicOr(&mask[id * 32 + (tl >> 5)], 1u << (tl & 31));
    if (sig) {
      const int t = t0 + tl;
      sig_add(a.r.tk.sig_req, a.r.tk.sig_block, a.r.tk.token_req ? a.r.tk.token_req[t] : -1,
              a.r.tk.token_block ? a.r.tk.token_block[t] : -1, a.r.tk.L, a.r.tk.layer, E, id);
    }
  }
  __syncthreads();
}

__global__ void __launch_bounds__(kRouteBigThreads) route_count_kernel(RouteBigArgs a) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  uint32_t* mask = reinterpret_cast<uint32_t*>(smem_raw);
  const int E = a.r.tk.E, T = a.r.tk.T;
  const int t0 = blockIdx.x * kRouteChunk, Tc = min(kRouteChunk, T - t0);
  route_big_masks(a, mask, t0, Tc, a.do_sig != 0);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int e = warp; e < E; e += kRouteBigThreads / 32) {
    const int c = __reduce_add_sync(0xffffffffu, __popc(mask[e * 32 + lane]));
    if (lane == 0) a.cnt_blk[(size_t)blockIdx.x * E + e] = c;
  }
}

__global__ void __launch_bounds__(kRouteBigThreads) route_scatter_kernel(RouteBigArgs a) {
  extern __shared__ __align__(16) uint8_t smem_raw[];
  const int E = a.r.tk.E, T = a.r.tk.T, k = a.r.tk.k;
  uint32_t* mask = reinterpret_cast<uint32_t*>(smem_raw);          // [E][32]
  uint32_t* pref = mask + (size_t)E * 32;                           // [E][32] exclusive prefix popcounts in the chunk
  int32_t* s_total = reinterpret_cast<int32_t*>(pref + (size_t)E * 32);   // [E] tokens of the expert, all chunks
  int32_t* s_before = s_total + E;                                  // [E] ... in the chunks before this one
  int32_t* s_off = s_before + E;                                    // [E+1] exclusive scan of s_total
  const int b = blockIdx.x, n_chunks = gridDim.x;
  const int t0 = b * kRouteChunk, Tc = min(kRouteChunk, T - t0);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const bool first = b == 0;
  route_big_masks(a, mask, t0, Tc, false);
  for (int e = warp; e < E; e += kRouteBigThreads / 32) {
    const int c = __popc(mask[e * 32 + lane]);
    int inc = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int v = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += v;
    }
    pref[e * 32 + lane] = inc - c;
    int tot = 0, bef = 0;
    for (int j = lane; j < n_chunks; j += 32) {
      const int v = __ldcg(a.cnt_blk + (size_t)j * E + e);
      tot += v;
      if (j < b) bef += v;
    }
    tot = __reduce_add_sync(0xffffffffu, tot);
    bef = __reduce_add_sync(0xffffffffu, bef);
    if (lane == 0) { s_total[e] = tot; s_before[e] = bef; }
  }
  __syncthreads();
  if (warp == 0) {     // exclusive scan of the expert totals; chunk 0 publishes the union-compacted work list
    constexpr int PER = kMaxExperts / 32;
    int c[PER], csum = 0, asum = 0;
#pragma unroll
    for (int i = 0; i < PER; ++i) {
      const int e = lane * PER + i;
      c[i] = (e < E) ? s_total[e] : 0;
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
        if (first) {
          a.r.off[e] = coff;
          a.r.cnt[e] = c[i];
          if (c[i] > 0) {
            a.r.active[aoff] = e;
            a.r.work[aoff] = make_int4(e, coff, coff, c[i]);
            ++aoff;
          }
        }
        coff += c[i];
      }
    }
    if (first) {
      for (int i = n_act + lane; i < E; i += 32) a.r.active[i] = -1;
      if (lane == 0) {
        a.r.off[E] = total;
        *a.r.n_active = n_act;
        *a.r.n_work = n_act + a.r.n_shared;
      }
      if (lane < a.r.n_shared) a.r.work[n_act + lane] = make_int4(E + lane, T * k, T * k + lane * T, T);
    }
  }
  __syncthreads();
  for (int p = tid; p < Tc * k; p += kRouteBigThreads) {
    const int tl = p / k;
    const size_t pg = (size_t)t0 * k + p;
    const int e = min(max(__ldcg(a.r.tk.ids + pg), 0), E - 1);
    const int rank = pref[e * 32 + (tl >> 5)] + __popc(mask[e * 32 + (tl >> 5)] & ((1u << (tl & 31)) - 1u));
    const int pos = s_off[e] + s_before[e] + rank;
    a.r.perm[pos] = (int32_t)pg;
    a.r.pair_pos[pg] = pos;
  }
}

}  // namespace eldr
