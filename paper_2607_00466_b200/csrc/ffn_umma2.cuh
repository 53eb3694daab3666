// Grouped SwiGLU expert FFN for PREFILL-shaped calls on an SM pair (tcgen05 cta_group::2), swap-AB:
// M = 256 weight rows (two adjacent 128-row tiles, one per CTA of a 2-CTA cluster), N <= 256 tokens of the expert,
// each CTA holding HALF of the token operand.  (steps a5/a6; "prefill forward".)
//
// Why a second kernel: with hundreds of tokens per expert the single-CTA tile of ffn_umma.cuh (M=128 x N=256) moves
// 48 KiB of operands per 540 MMA cycles through every SM (profiles/r1_prefill.md: tensor pipe 34-42 % active, HBM
// 40-50 %).  The pair tile moves 32 KiB per CTA for the same MMA time (16 KiB weights + 128 tokens x 128 B), so six
// stages fit where four did, and the B operand is read from shared memory once per SM pair instead of once per SM.
//
// Work unit = (expert, pair tile, 256-token pass), passes of one weight tile adjacent in the unit order: the pairs that
// run concurrently share their weight tile (the passes of a tile) and their tokens (the tiles of an expert), so the
// live working set is a few tens of MB and every operand byte crosses HBM once.  (With the pass loop INSIDE a tile,
// 74 pairs x 1 MB of weights + the token stream overflowed L2 and each pass re-read its weights from DRAM: ncu
// measured 3.26 GB of DRAM reads for 1.34 GB of operands at T = 16384.)  The unit list also evens out the tail.
//
// Roles per CTA (7 warps, as in ffn_umma.cuh): warp 0 weights producer, warp 1 activations producer, warp 2 MMA issuer
// (LEADER CTA only; the peer's warp 2 only takes part in the TMEM allocation), warps 3..6 epilogue of the CTA's own
// 128 accumulator lanes (its weight tile, all tokens of the pass).
// Barriers: full[s] lives in the leader (both CTAs' TMA loads complete_tx on it, cta_group::2 form); empty[s] and
// tmem_full[b] exist in both CTAs and are signalled by multicast tcgen05.commit; tmem_empty[b] lives in the leader
// and counts the 8 epilogue warps of the pair (remote arrive from the peer).
#pragma once
#include "ffn_umma.cuh"

namespace eldr {

constexpr int kPairNP = 256;                              // tokens per accumulator pass
constexpr int kPairStageBytes = kUmmaWBytes + (kPairNP / 2) * 128;   // 32 KiB per CTA
constexpr uint32_t kPeerBitMask = 0xFEFFFFFFu;            // shared::cluster address of the same offset in CTA rank 0

__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t mapa_rank(uint32_t addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" :: "r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity) {
  uint32_t ok = 0;
  for (uint32_t spins = 0; ; ++spins) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    if (ok) break;
    if (spins > (1u << 24)) __trap();
  }
}
// TMA loads of a CTA pair: data lands in the issuing CTA's shared memory, the bytes are counted on the LEADER's barrier
__device__ __forceinline__ void tma2_load_2d(uint32_t dst, const CUtensorMap* m, int c0, int c1, uint32_t leader_bar,
                                             uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%2, %3}], [%4], %5;"
      :: "r"(dst), "l"(reinterpret_cast<uint64_t>(m)), "r"(c0), "r"(c1), "r"(leader_bar), "l"(policy)
      : "memory");
}
__device__ __forceinline__ void tma2_load_5d(uint32_t dst, const CUtensorMap* m, int c0, int c1, int c2, int c3, int c4,
                                             uint32_t leader_bar, uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.5d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%2, %3, %4, %5, %6}], [%7], %8;"
      :: "r"(dst), "l"(reinterpret_cast<uint64_t>(m)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "r"(leader_bar),
         "l"(policy)
      : "memory");
}
__device__ __forceinline__ void umma2_bf16(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc,
                                           uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      :: "r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate) : "memory");
}
// arrives (once the pair's earlier MMAs have completed) on the barrier at this offset in BOTH CTAs
__device__ __forceinline__ void umma2_commit_both(uint32_t bar) {
  asm volatile(
      "tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
      :: "r"(bar), "h"((uint16_t)3) : "memory");
}

// SiLU with the fast exponential and division (2 ulp each; h is rounded to bf16, 2^-9, right after)
__device__ __forceinline__ float silu_fast(float v) { return __fdividef(v, 1.0f + __expf(-v)); }

template <int MODE>
__global__ void __launch_bounds__(kUmmaThreads, 1)
ffn_umma2_kernel(const __grid_constant__ CUtensorMap tm_w, const __grid_constant__ CUtensorMap tm_ws,
                 const __grid_constant__ CUtensorMap tm_x16, const __grid_constant__ CUtensorMap tm_x64,
                 const FfnArgs a, const int S, const int max_work) {
  extern __shared__ uint8_t smem_dyn[];
  const uint32_t smem_base = (smem_u32(smem_dyn) + 1023u) & ~1023u;
  constexpr int NP = kPairNP;
  const uint32_t bar_base = smem_base + S * kPairStageBytes;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (S + s); };
  auto tfull_bar = [&](int b) { return bar_base + 8u * (2 * S + b); };
  auto tempty_bar = [&](int b) { return bar_base + 8u * (2 * S + 2 + b); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * S + 4);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  if (threadIdx.x == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(full_bar(s), 2); mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(tfull_bar(b), 1); mbar_init(tempty_bar(b), 8); }
    mbar_fence_init();
  }
  constexpr uint32_t tmem_cols = 2 * NP;     // two accumulator buffers of 256 fp32 columns
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(tmem_slot), "r"(tmem_cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();          // both CTAs' barriers initialised before any remote complete_tx / arrive
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));
  pdl_launch_dependents();
  pdl_wait();

  const int n_work = *a.n_work;
  const int tpe2 = a.tiles_per_expert >> 1;
  const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
  const int k_iters = a.K / 64;
  // unit prefix over the work list: entry e owns units [upref[e], upref[e+1]) = tpe2 tiles x passes(e), pass fastest
  int* ucnt = reinterpret_cast<int*>(smem_dyn + ((bar_base + 8u * (2 * S + 5) + 15u) & ~15u) - smem_u32(smem_dyn));
  int* upref = ucnt + max_work;
  for (int e = threadIdx.x; e < n_work; e += blockDim.x) ucnt[e] = tpe2 * ((a.work[e].w + NP - 1) / NP);
  __syncthreads();
  for (int e = threadIdx.x; e <= n_work; e += blockDim.x) {
    int acc = 0;
    for (int j = 0; j < e; ++j) acc += ucnt[j];
    upref[e] = acc;
  }
  __syncthreads();
  const int total = upref[n_work];
  // unit u -> (work entry, tile of this CTA, first token of the pass); `ent` only moves forward
  struct Unit { int4 wk; int rt, n0; };
  int ent = 0;
  auto unit_at = [&](int u) {
    while (u >= upref[ent + 1]) ++ent;
    Unit r;
    r.wk = a.work[ent];
    const int local = u - upref[ent], passes = (r.wk.w + NP - 1) / NP;
    const int t2 = local / passes;
    r.rt = t2 * 2 + (int)rank;
    r.n0 = (local - t2 * passes) * NP;
    return r;
  };

  if (warp == 0) {
    // ================================================================ weights producer (own 128-row tile)
    if (lane == 0) {
      tma_prefetch_desc(&tm_w);
      const uint64_t pol = l2_policy_evict_last();     // the tile's other passes run on neighbouring pairs right now
      uint32_t it = 0;
      for (int u = pair; u < total; u += n_pairs) {
        const Unit un = unit_at(u);
        const bool shared = un.wk.x >= a.E;
        const CUtensorMap* tmw = shared ? &tm_ws : &tm_w;
        const int we = shared ? un.wk.x - a.E : un.wk.x;
        for (int kc = 0; kc < k_iters; ++kc, ++it) {
          const int s = it % S;
          mbar_wait(empty_bar(s), ((it / S) & 1) ^ 1);
          if (rank == 0) mbar_arrive_expect_tx(full_bar(s), 2 * kUmmaWBytes);
          const uint32_t dst = smem_base + s * kPairStageBytes;
          const uint32_t lbar = full_bar(s) & kPeerBitMask;
          if (MODE == 0) tma2_load_5d(dst, tmw, kc * 64, 0, 0, un.rt * 4, we, lbar, pol);
          else tma2_load_2d(dst, tmw, kc * 64, we * a.rows_per_expert + un.rt * 128, lbar, pol);
        }
      }
    }
  } else if (warp == 1) {
    // ================================================================ activations producer (own half of the tokens)
    if (lane == 0) {
      tma_prefetch_desc(&tm_x16);
      const uint64_t pol = l2_policy_evict_last();
      uint32_t it = 0;
      for (int u = pair; u < total; u += n_pairs) {
        const Unit un = unit_at(u);
        const int xrow0 = (MODE == 0) ? un.wk.y : un.wk.z;
        const int n_half = ((min(NP, un.wk.w - un.n0) + 31) & ~31) >> 1;
        const bool big = (n_half & 63) == 0;
        const int n_box = big ? n_half / 64 : n_half / 16;
        const uint32_t box_bytes = big ? 64 * 128 : 16 * 128;
        const CUtensorMap* tmx = big ? &tm_x64 : &tm_x16;
        const int row0 = xrow0 + un.n0 + (int)rank * n_half;
        for (int kc = 0; kc < k_iters; ++kc, ++it) {
          const int s = it % S;
          mbar_wait(empty_bar(s), ((it / S) & 1) ^ 1);
          if (rank == 0) mbar_arrive_expect_tx(full_bar(s), 2 * n_half * 128);
          const uint32_t dst = smem_base + s * kPairStageBytes + kUmmaWBytes;
          const uint32_t lbar = full_bar(s) & kPeerBitMask;
          for (int b = 0; b < n_box; ++b)
            tma2_load_2d(dst + b * box_bytes, tmx, kc * 64, row0 + b * (big ? 64 : 16), lbar, pol);
        }
      }
    }
  } else if (warp == 2) {
    // ================================================================ MMA issuer (leader CTA only)
    if (rank == 0) {
      uint32_t it = 0, unit = 0;
      for (int u = pair; u < total; u += n_pairs, ++unit) {
        const Unit un = unit_at(u);
        const int n_pad = (min(NP, un.wk.w - un.n0) + 31) & ~31;
        // D fp32, A/B bf16 K-major, N = n_pad, M = 256 over the pair
        const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n_pad >> 3) << 17) | (16u << 24);
        const int buf = unit & 1;
        mbar_wait_cluster(tempty_bar(buf), ((unit >> 1) & 1) ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + buf * NP;
        for (int kc = 0; kc < k_iters; ++kc, ++it) {
          const int s = it % S;
          mbar_wait_cluster(full_bar(s), (it / S) & 1);
          tc_fence_after();
          if (lane == 0) {
            const uint32_t sa = smem_base + s * kPairStageBytes;
            const uint64_t da = umma_desc_sw128(sa), db = umma_desc_sw128(sa + kUmmaWBytes);
#pragma unroll
            for (int k = 0; k < 4; ++k)
              umma2_bf16(d_tmem, da + 2 * k, db + 2 * k, idesc, (kc | k) ? 1u : 0u);
            umma2_commit_both(empty_bar(s));
            if (kc == k_iters - 1) umma2_commit_both(tfull_bar(buf));
          }
          __syncwarp();
        }
      }
    }
  } else {
    // ================================================================ epilogue (own 128 lanes: own weight tile, all tokens)
    const int qtr = warp & 3;
    const uint32_t leader_tempty0 = mapa_rank(tempty_bar(0), 0), leader_tempty1 = mapa_rank(tempty_bar(1), 0);
    uint32_t unit = 0;
    for (int u = pair; u < total; u += n_pairs, ++unit) {
      const Unit un = unit_at(u);
      const int4 wk = un.wk;
      const int rt = un.rt, n0 = un.n0;
      const int n_here = min(NP, wk.w - n0);
      const int buf = unit & 1;
      mbar_wait(tfull_bar(buf), (unit >> 1) & 1);
      tc_fence_after();
      const uint32_t t_addr = tmem_base + buf * NP + ((uint32_t)(qtr * 32) << 16);
      for (int c0 = 0; c0 < n_here; c0 += 16) {
        float v[16];
        tmem_ld16(t_addr + c0, v);
        if (MODE == 0) {
          const bool lo = lane < 16;
          const int i = rt * 64 + 16 * qtr + (lane & 15);
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            const float send = lo ? v[8 + k] : v[k];
            const float recv = __shfl_xor_sync(0xffffffffu, send, 16);
            const float gv = lo ? v[k] : recv;
            const float uv = lo ? recv : v[8 + k];
            const int tok = n0 + c0 + (lo ? k : 8 + k);
            if (tok < wk.w) a.h_out[(size_t)(wk.z + tok) * a.I + i] = f32_to_bf16_rn(silu_fast(gv) * uv);
          }
        } else {
          const int r = rt * 128 + 32 * qtr + lane;
#pragma unroll
          for (int k = 0; k < 16; ++k) {
            const int tok = n0 + c0 + k;
            if (tok < wk.w) a.y_out[(size_t)(wk.z + tok) * a.H + r] = v[k];
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_cluster(buf ? leader_tempty1 : leader_tempty0);
    }
  }

  // the peer's shared memory and barriers are targets of the leader's MMAs / commits until the last one has landed
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  if (warp == 2) {
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" :: "r"(tmem_base), "r"(tmem_cols) : "memory");
  }
}

}  // namespace eldr
