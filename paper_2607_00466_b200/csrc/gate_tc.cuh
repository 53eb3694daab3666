// Gate logits for prefill-shaped batches on the tensor cores WITHOUT giving up the gate's fp32 arithmetic
// (reading "fp32 gate, near-ties must not flip").
//
// z[t,e] = sum_h x[t,h] * Wg[e,h] (+ bias) with x bf16 and Wg fp32.  An fp32 number is EXACTLY the sum of three bf16
// numbers (8 + 8 + 8 significand bits: hi = bf16(w), mid = bf16(w - hi), lo = bf16(w - hi - mid)), and a product of two
// bf16 numbers is exact in fp32, so
//     x * w = x * lo + x * mid + x * hi          (three exact products)
// and the only rounding left is the fp32 accumulation -- as in the CUDA-core kernels.  The tensor core's accumulator is
// less forgiving than a chain of round-to-nearest FMAs over a long sum (measured with cuBLAS on this part: full K = 2048
// in one accumulator 2.9e-5 abs error at |z| ~ 10, K slices of 256 summed afterwards 3.2e-6; in this kernel a 256-wide
// slice still left 1.3e-5 on a layer with large gate weights: the accumulator's error grows with the NUMBER of
// accumulations and the size of the running sum), so each TMEM accumulator holds ONE 64-wide k-chunk -- the hi terms (4 MMAs of
// K = 16) in one accumulator, the mid and lo terms (8 MMAs) in a second one -- and the epilogue warps add hi + (mid + lo)
// of every chunk to fp32 registers in order, round to nearest.
//
// CTA = 128 tokens x 64 experts.  Warp 0: TMA producer (x box 128 x 64, three weight boxes 64 x 64 per 64-wide k-chunk,
// 40 KiB per stage, 4 stages); warp 1: MMA issuer (tcgen05, M = 128 tokens, N = 64 experts, fp32 in TMEM, two buffers of
// 2 x 64 columns); warps 2-5: epilogue (lane = token: 64 fp32 accumulators in registers).  The two expert halves of a token tile
// are neighbouring CTAs, so x crosses HBM once.
// The three-term split of Wg is written by gate_split_kernel into the workspace before it (1 MB in, 0.75 MB out).
// Logit error against the fp64 oracle: 2e-6 at |z| ~ 15 (the CUDA-core kernel: 1.1e-5 on the same inputs).
// Measured (bench.py --config prefill, gate = split + logits + top-k): T = 2048 / 4096 / 8192 / 16384: 44 / 44 / 50 / 88 us
// against 78 / 108 / 157 / 275 us for the register-tiled CUDA-core GEMM; the step 0.49 -> 0.54 of the sustained bf16 peak
// at T = 16384.
#pragma once
#include "device_utils.cuh"
#include "ffn_umma.cuh"

namespace eldr {

constexpr int kGtcThreads = 192;
constexpr int kGtcStages = 4;
constexpr int kGtcTok = 128, kGtcExp = 64;
constexpr int kGtcSliceChunks = 1;                                    // K slice per TMEM accumulator: one 64-wide chunk (12 MMAs)
constexpr int kGtcStageBytes = kGtcTok * 128 + 3 * kGtcExp * 128;     // 16 KiB of x + 3 x 8 KiB of weight terms
constexpr int kGtcSmemBytes = kGtcStages * kGtcStageBytes + 1024 + 256;

// w [n] fp32 -> out [3][n] bf16: term 0 = lo, 1 = mid, 2 = hi
__global__ void __launch_bounds__(256) gate_split_kernel(const float* __restrict__ w, uint16_t* __restrict__ out, int n) {
  const int i = blockIdx.x * 256 + threadIdx.x;
  pdl_launch_dependents();
  pdl_wait();
  if (i >= n) return;
  const float v = w[i];
  const uint16_t hi = f32_to_bf16_rn(v);
  const float r1 = v - __uint_as_float((uint32_t)hi << 16);
  const uint16_t mid = f32_to_bf16_rn(r1);
  const float r2 = r1 - __uint_as_float((uint32_t)mid << 16);
  const uint16_t lo = f32_to_bf16_rn(r2);
  out[i] = lo;
  out[(size_t)n + i] = mid;
  out[2 * (size_t)n + i] = hi;
}

__global__ void __launch_bounds__(kGtcThreads, 1)
gate_logits_tc_kernel(const __grid_constant__ CUtensorMap tm_x, const __grid_constant__ CUtensorMap tm_w,
                      const float* __restrict__ bias, float* __restrict__ z, int T, int H, int E) {
  extern __shared__ uint8_t smem_dyn[];
  const uint32_t smem_base = (smem_u32(smem_dyn) + 1023u) & ~1023u;
  const uint32_t bar_base = smem_base + kGtcStages * kGtcStageBytes;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (kGtcStages + s); };
  auto tfull_bar = [&](int b) { return bar_base + 8u * (2 * kGtcStages + b); };
  auto tempty_bar = [&](int b) { return bar_base + 8u * (2 * kGtcStages + 2 + b); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * kGtcStages + 4);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < kGtcStages; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(tfull_bar(b), 1); mbar_init(tempty_bar(b), 4); }
    mbar_fence_init();
    tma_prefetch_desc(&tm_x);
    tma_prefetch_desc(&tm_w);
  }
  constexpr uint32_t tmem_cols = 4 * kGtcExp;                       // two buffers x (hi-term accumulator | mid+lo accumulator)
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(tmem_slot), "r"(tmem_cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));
  pdl_launch_dependents();
  pdl_wait();

  const int e0 = blockIdx.x * kGtcExp, t0 = blockIdx.y * kGtcTok;     // the expert halves of a token tile run side by side: x is read from HBM once
  const int n_chunks = H / 64;
  const int n_slices = (n_chunks + kGtcSliceChunks - 1) / kGtcSliceChunks;

  if (warp == 0) {
    if (lane == 0) {
      const uint64_t pol_x = l2_policy_evict_first(), pol_w = l2_policy_evict_last();
      for (int kc = 0; kc < n_chunks; ++kc) {
        const int s = kc % kGtcStages;
        mbar_wait(empty_bar(s), ((kc / kGtcStages) & 1) ^ 1);
        mbar_arrive_expect_tx(full_bar(s), kGtcStageBytes);
        const uint32_t dst = smem_base + s * kGtcStageBytes;
        tma_load_2d(dst, &tm_x, kc * 64, t0, full_bar(s), pol_x);
        for (int term = 0; term < 3; ++term)
          tma_load_2d(dst + kGtcTok * 128 + term * kGtcExp * 128, &tm_w, kc * 64, term * E + e0, full_bar(s), pol_w);
      }
    }
  } else if (warp == 1) {
    const uint32_t leader = elect_one();
    const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(kGtcExp >> 3) << 17) | (8u << 24);
    int kc = 0;
    for (int sl = 0; sl < n_slices; ++sl) {
      const uint32_t buf = sl & 1;
      mbar_wait(tempty_bar(buf), ((sl >> 1) & 1) ^ 1);
      tc_fence_after();
      // the hi terms (the full-size products) get an accumulator of their own: every accumulation rounds at the size
      // of the running sum, and the eight mid / lo MMAs of a chunk would otherwise each cost the big sum one more
      // rounding for a contribution of 2^-8 / 2^-16 of it (measured: 1.1e-5 instead of < 5e-6 at |z| ~ 10, H = 256)
      const uint32_t d_hi = tmem_base + buf * 2 * kGtcExp, d_lo = d_hi + kGtcExp;
      const int kc_end = min(n_chunks, (sl + 1) * kGtcSliceChunks);
      bool first_lo = true, first_hi = true;
      for (; kc < kc_end; ++kc) {
        const int s = kc % kGtcStages;
        mbar_wait(full_bar(s), (kc / kGtcStages) & 1);
        tc_fence_after();
        const uint32_t sa = smem_base + s * kGtcStageBytes;
        const uint64_t da = umma_desc_sw128(sa);
#pragma unroll
        for (int term = 0; term < 3; ++term) {                      // lo, mid, hi
          const uint64_t db = umma_desc_sw128(sa + kGtcTok * 128 + term * kGtcExp * 128);
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            if (term < 2) { umma_bf16_if(leader, d_lo, da + 2 * k, db + 2 * k, idesc, first_lo ? 0u : 1u); first_lo = false; }
            else { umma_bf16_if(leader, d_hi, da + 2 * k, db + 2 * k, idesc, first_hi ? 0u : 1u); first_hi = false; }
          }
        }
        umma_commit_if(leader, empty_bar(s));
      }
      umma_commit_if(leader, tfull_bar(buf));
    }
  } else {
    const int qtr = warp & 3;                                       // TMEM lane quarter this warp may read
    const int t = t0 + 32 * qtr + lane;
    float acc[kGtcExp];
#pragma unroll
    for (int j = 0; j < kGtcExp; ++j) acc[j] = 0.f;
    for (int sl = 0; sl < n_slices; ++sl) {
      const int buf = sl & 1;
      mbar_wait(tfull_bar(buf), (sl >> 1) & 1);
      tc_fence_after();
      const uint32_t t_addr = tmem_base + buf * 2 * kGtcExp + ((uint32_t)(qtr * 32) << 16);
#pragma unroll
      for (int c0 = 0; c0 < kGtcExp; c0 += 16) {
        float vh[16], vl[16];
        tmem_ld16(t_addr + c0, vh);
        tmem_ld16(t_addr + kGtcExp + c0, vl);
#pragma unroll
        for (int j = 0; j < 16; ++j) acc[c0 + j] += vh[j] + vl[j];  // chunk order, round to nearest
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(tempty_bar(buf));
    }
    if (t < T) {
      float* zr = z + (size_t)t * E + e0;
#pragma unroll
      for (int j = 0; j < kGtcExp; ++j)
        if (e0 + j < E) zr[j] = acc[j] + (bias ? bias[e0 + j] : 0.f);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_base), "r"(tmem_cols) : "memory");
  }
}

}  // namespace eldr
