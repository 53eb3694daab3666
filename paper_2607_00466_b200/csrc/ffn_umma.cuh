// Grouped SwiGLU expert FFN on the 5th-generation tensor cores (tcgen05 + TMEM), swap-AB:
// the streamed weight tile is the M=128 operand, the expert's gathered tokens are the N operand.
// ("each step fetches the weights of every expert the batch
// activates" -- the kernel's job is to keep HBM busy; the tensor core makes the math free for any m.)
//
// One persistent CTA per SM, 6 warps:
//   warp 0  TMA producer, weights: ONE cp.async.bulk.tensor per stage -> 128 rows x 64 cols bf16 (16 KiB),
//           SWIZZLE_128B, L2 evict_first (each active expert is read exactly once)
//   warp 1  TMA producer, activations: the matching 64-column slice of the expert's token rows (L2-resident)
//   warp 2  MMA issuer (one elected lane): 4 x tcgen05.mma.cta_group::1.kind::f16 (M=128, N=n_pad, K=16) per
//           stage, accumulating in TMEM; tcgen05.commit frees the smem stage / publishes the accumulator.
//           Also owns the TMEM allocation.
//   warps 3..6 -> here warps 2..5 are arranged so that (warp & 3) covers the four TMEM lane quarters.
//
// MODE 0 (w1/w3): the 5-D tensor map orders the 128 rows of a stage as 4 groups of [16 rows of W1 | the same
//   16 rows of W3]; a warp's TMEM lane quarter therefore holds g on lanes 0-15 and u on lanes 16-31 for the same
//   16 intermediate indices, and silu(g)*u needs only a shfl_xor(16) exchange.  Writes h (bf16).
// MODE 1 (w2): 128 rows of W2 per tile; lane = output row; writes y (fp32) for the ordered combine.
#pragma once
#include "device_utils.cuh"
#include "ffn_stream.cuh"   // FfnArgs

namespace eldr {

constexpr int kUmmaWBytes = 128 * 128;        // 16 KiB weight tile per stage
constexpr int kUmmaThreads = 7 * 32;          // warps: 0 W-producer, 1 X-producer, 2 MMA, 3..6 epilogue

struct UmmaCfg {
  int np;          // max token rows per pass (64 or 128); B stage bytes = np*128; TMEM cols = 2*np
  int stages;
};

__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// K-major, SWIZZLE_128B operand tile: rows of 128 bytes, 8-row atoms of 1024 bytes (SBO), LBO unused.
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t smem_addr) {
  return (uint64_t)((smem_addr & 0x3FFFFu) >> 4) | ((uint64_t)(1024u >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// D[tmem] (+)= A[smem] * B[smem]^T, bf16 x bf16 -> fp32
__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc,
                                          uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      :: "r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(bar) : "memory");
}
// Issue-side helpers for a CONVERGED warp: operands made provably warp-uniform (redux result lives in a uniform
// register) and the instruction predicated on the elected lane INSIDE the asm, so the compiler emits the
// uniform-datapath instruction directly instead of an ELECT / R2UR.BROADCAST / BRA.U.ANY waterfall per MMA.
__device__ __forceinline__ uint32_t warp_uniform(uint32_t v) { return __reduce_max_sync(0xffffffffu, v); }
__device__ __forceinline__ uint32_t elect_one() {
  uint32_t pred;
  asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
  return pred;
}
__device__ __forceinline__ void umma_bf16_if(uint32_t leader, uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b,
                                             uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p, q;\n\tsetp.ne.b32 p, %4, 0;\n\tsetp.ne.b32 q, %5, 0;\n\t"
      "@q tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      :: "r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate), "r"(leader) : "memory");
}
// same, A operand (M = 128 rows x 16 bf16 = 8 columns) read from tensor memory
__device__ __forceinline__ void umma_bf16_ts_if(uint32_t leader, uint32_t tmem_d, uint32_t tmem_a, uint64_t desc_b,
                                                uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p, q;\n\tsetp.ne.b32 p, %4, 0;\n\tsetp.ne.b32 q, %5, 0;\n\t"
      "@q tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
      :: "r"(tmem_d), "r"(tmem_a), "l"(desc_b), "r"(idesc), "r"(accumulate), "r"(leader) : "memory");
}
// 16 consecutive 32-bit columns of this thread's TMEM lane <- four uint4
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint4& a, const uint4& b, const uint4& c, const uint4& d) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
      :: "r"(taddr), "r"(a.x), "r"(a.y), "r"(a.z), "r"(a.w), "r"(b.x), "r"(b.y), "r"(b.z), "r"(b.w),
         "r"(c.x), "r"(c.y), "r"(c.z), "r"(c.w), "r"(d.x), "r"(d.y), "r"(d.z), "r"(d.w) : "memory");
}
__device__ __forceinline__ void umma_commit_if(uint32_t leader, uint32_t bar) {
  asm volatile(
      "{\n\t.reg .pred q;\n\tsetp.ne.b32 q, %1, 0;\n\t"
      "@q tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n\t}"
      :: "r"(bar), "r"(leader) : "memory");
}
// 16 consecutive fp32 columns of this thread's TMEM lane
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16]) {
  uint32_t r[16];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
        "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}

__device__ __forceinline__ void tma_load_5d(uint32_t dst, const CUtensorMap* m, int c0, int c1, int c2, int c3,
                                            int c4, uint32_t bar, uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%2, %3, %4, %5, %6}], [%7], %8;"
      :: "r"(dst), "l"(reinterpret_cast<uint64_t>(m)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4), "r"(bar),
         "l"(policy)
      : "memory");
}

template <int MODE>
__global__ void __launch_bounds__(kUmmaThreads, 1)
ffn_umma_kernel(const __grid_constant__ CUtensorMap tm_w, const __grid_constant__ CUtensorMap tm_ws,
                const __grid_constant__ CUtensorMap tm_x16, const __grid_constant__ CUtensorMap tm_x64,
                const FfnArgs a, const UmmaCfg cfg) {
  extern __shared__ uint8_t smem_dyn[];
  const uint32_t smem_base = (smem_u32(smem_dyn) + 1023u) & ~1023u;
  const int NP = cfg.np, S = cfg.stages;
  const uint32_t stage_bytes = kUmmaWBytes + NP * 128;
  const uint32_t bar_base = smem_base + S * stage_bytes;
  // barriers: full[S], empty[S], tmem_full[2], tmem_empty[2]; then the TMEM base address slot
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (S + s); };
  auto tfull_bar = [&](int b) { return bar_base + 8u * (2 * S + b); };
  auto tempty_bar = [&](int b) { return bar_base + 8u * (2 * S + 2 + b); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * S + 4);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(full_bar(s), 2); mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(tfull_bar(b), 1); mbar_init(tempty_bar(b), 4); }
    mbar_fence_init();
  }
  const uint32_t tmem_cols = 2 * NP;     // 128 or 256: power of two >= 32
  if (warp == 2) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(tmem_slot), "r"(tmem_cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));
  // everything above overlapped the previous kernel's tail; the work list / activations are its outputs
  pdl_launch_dependents();
  pdl_wait();

  const int n_work = *a.n_work;
  const int total_tiles = n_work * a.tiles_per_expert;
  const int k_iters = a.K / 64;

  if (warp == 0) {
    // ================================================================ weights producer
    if (lane == 0) {
      tma_prefetch_desc(&tm_w);
      const uint64_t pol_once = l2_policy_evict_first(), pol_again = l2_policy_evict_last();
      uint32_t it = 0;
      for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
        const int ent = tile / a.tiles_per_expert, rt = tile - ent * a.tiles_per_expert;
        const int4 wk = a.work[ent];
        const bool shared = wk.x >= a.E;
        const CUtensorMap* tmw = shared ? &tm_ws : &tm_w;
        const int we = shared ? wk.x - a.E : wk.x;
        // (Pulling this CTA's NEXT weight tile into L2 with cp.async.bulk.prefetch.tensor while the current one is
        // multiplied was measured for the prefill-shaped calls, as a burst and one box per stage: 10-25 % slower both
        // ways -- the prefetches hold TMA request slots for a DRAM latency each and the demand loads queue behind them.)
        for (int n0 = 0; n0 < wk.w; n0 += NP) {
          // the tile is streamed once per accumulator pass: keep it in L2 until the last pass has read it
          const uint64_t pol = (n0 + NP < wk.w) ? pol_again : pol_once;
          for (int kc = 0; kc < k_iters; ++kc, ++it) {
            const int s = it % S;
            mbar_wait(empty_bar(s), ((it / S) & 1) ^ 1);
            mbar_arrive_expect_tx(full_bar(s), kUmmaWBytes);
            const uint32_t dst = smem_base + s * stage_bytes;
            if (MODE == 0) tma_load_5d(dst, tmw, kc * 64, 0, 0, rt * 4, we, full_bar(s), pol);
            else tma_load_2d(dst, tmw, kc * 64, we * a.rows_per_expert + rt * 128, full_bar(s), pol);
          }
        }
      }
    }
  } else if (warp == 1) {
    // ================================================================ activations producer
    if (lane == 0) {
      tma_prefetch_desc(&tm_x16);
      const uint64_t pol = l2_policy_evict_last();
      uint32_t it = 0;
      for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
        const int ent = tile / a.tiles_per_expert;
        const int4 wk = a.work[ent];
        const int xrow0 = (MODE == 0) ? wk.y : wk.z;
        for (int n0 = 0; n0 < wk.w; n0 += NP) {
          const int n_pad = (min(NP, wk.w - n0) + 15) & ~15;
          const bool big = n_pad > 48;
          const int n_box = big ? (n_pad + 63) / 64 : n_pad / 16;
          const uint32_t box_bytes = big ? 64 * 128 : 16 * 128;
          const CUtensorMap* tmx = big ? &tm_x64 : &tm_x16;
          for (int kc = 0; kc < k_iters; ++kc, ++it) {
            const int s = it % S;
            mbar_wait(empty_bar(s), ((it / S) & 1) ^ 1);
            mbar_arrive_expect_tx(full_bar(s), n_box * box_bytes);
            const uint32_t dst = smem_base + s * stage_bytes + kUmmaWBytes;
            for (int b = 0; b < n_box; ++b)
              tma_load_2d(dst + b * box_bytes, tmx, kc * 64, xrow0 + n0 + b * (big ? 64 : 16), full_bar(s), pol);
          }
        }
      }
    }
  } else if (warp == 2) {
    // ================================================================ MMA issuer
    uint32_t it = 0, unit = 0;
    for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
      const int ent = tile / a.tiles_per_expert;
      const int4 wk = a.work[ent];
      for (int n0 = 0; n0 < wk.w; n0 += NP, ++unit) {
        const int n_pad = (min(NP, wk.w - n0) + 15) & ~15;
        const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n_pad >> 3) << 17) | (8u << 24);
        const int buf = unit & 1;
        mbar_wait(tempty_bar(buf), ((unit >> 1) & 1) ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + buf * NP;
        for (int kc = 0; kc < k_iters; ++kc, ++it) {
          const int s = it % S;
          mbar_wait(full_bar(s), (it / S) & 1);
          tc_fence_after();
          if (lane == 0) {
            const uint32_t sa = smem_base + s * stage_bytes;
            const uint64_t da = umma_desc_sw128(sa), db = umma_desc_sw128(sa + kUmmaWBytes);
#pragma unroll
            for (int k = 0; k < 4; ++k)      // K = 16 bf16 = 32 bytes per MMA: advance the start address by 2 (x16 B)
              umma_bf16(d_tmem, da + 2 * k, db + 2 * k, idesc, (kc | k) ? 1u : 0u);
            umma_commit(empty_bar(s));                       // stage free once these MMAs have read it
            if (kc == k_iters - 1) umma_commit(tfull_bar(buf));   // accumulator complete
          }
          __syncwarp();
        }
      }
    }
  } else {
    // ================================================================ epilogue (4 warps, one TMEM lane quarter each)
    const int qtr = warp & 3;
    uint32_t unit = 0;
    for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
      const int ent = tile / a.tiles_per_expert, rt = tile - ent * a.tiles_per_expert;
      const int4 wk = a.work[ent];
      for (int n0 = 0; n0 < wk.w; n0 += NP, ++unit) {
        const int n_here = min(NP, wk.w - n0);
        const int buf = unit & 1;
        mbar_wait(tfull_bar(buf), (unit >> 1) & 1);
        tc_fence_after();
        const uint32_t t_addr = tmem_base + buf * NP + ((uint32_t)(qtr * 32) << 16);
        for (int c0 = 0; c0 < n_here; c0 += 16) {
          float v[16];
          tmem_ld16(t_addr + c0, v);
          if (MODE == 0) {
            // lanes 0-15: g for i = rt*64 + 16*qtr + lane; lanes 16-31: u for the same i.
            // lanes < 16 finish columns 0-7 of the chunk, lanes >= 16 columns 8-15.
            const bool lo = lane < 16;
            const int i = rt * 64 + 16 * qtr + (lane & 15);
#pragma unroll
            for (int k = 0; k < 8; ++k) {
              const float send = lo ? v[8 + k] : v[k];
              const float recv = __shfl_xor_sync(0xffffffffu, send, 16);
              const float gv = lo ? v[k] : recv;
              const float uv = lo ? recv : v[8 + k];
              const int tok = n0 + c0 + (lo ? k : 8 + k);
              if (tok < wk.w) a.h_out[(size_t)(wk.z + tok) * a.I + i] = f32_to_bf16_rn(silu_f(gv) * uv);
            }
          } else {
            const int r = rt * 128 + 32 * qtr + lane;
            if (r < a.H) {
#pragma unroll
              for (int k = 0; k < 16; ++k) {
                const int tok = n0 + c0 + k;
                if (tok < wk.w) a.y_out[(size_t)(wk.z + tok) * a.H + r] = v[k];
              }
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(tempty_bar(buf));
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_base), "r"(tmem_cols) : "memory");
  }
}

}  // namespace eldr
