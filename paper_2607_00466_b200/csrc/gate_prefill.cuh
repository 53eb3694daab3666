// a1 for PREFILL-shaped calls of eldr_moe_gate_topk (hundreds to thousands of tokens: where the paper captures
// its signatures): z[t,e] = sum_h x[t,h] * Wg[e,h] (+ bias[e]) as a register-tiled fp32 GEMM
// on the CUDA cores.  fp32 FMA on purpose (DESIGN.md reading: bf16 x is exact in fp32, Wg is fp32; no TF32 / bf16
// MMA, which would flip near-tie selections), so the bound is the fp32 ALU peak, not the tensor pipe.
//
//   tile 128 tokens x 128 experts x 16 h per CTA (256 threads, 8 x 8 accumulators each), operands staged
//   transposed in shared memory ([h][token], [h][expert]) so that a thread's 8 + 8 operands are four LDS.128 per
//   64 FMA; the next chunk's global loads are in flight while the current one is multiplied.
//   split-K: H is cut into S slices of AT MOST 256 h -- one fp32 accumulator over all of H = 2048 drifts to 1.6e-5
//   from the fp64 logits (measured), past the 1e-5 near-tie threshold, while 256-wide slices stay at a few 1e-6
//   like the decode path's per-lane partial sums (a second in-register accumulator level costs 64 registers and
//   half the occupancy: measured 20 % slower); the slices also fill the 148 SMs.  Slice s writes its partial
//   logits to zp[s]; topk_splitk_kernel adds the S partials IN SLICE ORDER (deterministic), stores the
//   final logits in zp[0] (= the z the ABI documents) and runs the same warp top-k (+signature) as the decode path.
#pragma once
#include "gate_route.cuh"

namespace eldr {

constexpr int kGpBM = 128, kGpBN = 128, kGpBK = 16, kGpThreads = 256;

__global__ void __launch_bounds__(kGpThreads)
gate_logits_tiled_kernel(const uint16_t* __restrict__ x, const float* __restrict__ gate_w,
                         const float* __restrict__ gate_bias, float* __restrict__ zp, int T, int H, int E,
                         int k_per_slice) {
  __shared__ __align__(16) float As[2][kGpBK][kGpBM];
  __shared__ __align__(16) float Bs[2][kGpBK][kGpBN];
  const int tid = threadIdx.x;
  const int m0 = blockIdx.x * kGpBM, n0 = blockIdx.y * kGpBN, slice = blockIdx.z;
  const int kbeg = slice * k_per_slice, n_it = k_per_slice / kGpBK;
  // loader roles: row = tid / 2 (token or expert of the tile), half = tid % 2 (8 of the 16 h of the chunk)
  const int lrow = tid >> 1, lhalf = tid & 1;
  const bool a_ok = m0 + lrow < T, b_ok = n0 + lrow < E;
  const uint16_t* xa = x + (size_t)(a_ok ? m0 + lrow : 0) * H + kbeg + lhalf * 8;
  const float* wb = gate_w + (size_t)(b_ok ? n0 + lrow : 0) * H + kbeg + lhalf * 8;
  uint4 ra = make_uint4(0u, 0u, 0u, 0u);
  float4 rb0 = make_float4(0.f, 0.f, 0.f, 0.f), rb1 = rb0;
  auto gload = [&](int it) {
    if (a_ok) ra = __ldg(reinterpret_cast<const uint4*>(xa + (size_t)it * kGpBK));
    if (b_ok) {
      rb0 = __ldg(reinterpret_cast<const float4*>(wb + (size_t)it * kGpBK));
      rb1 = __ldg(reinterpret_cast<const float4*>(wb + (size_t)it * kGpBK + 4));
    }
  };
  auto sstore = [&](int buf) {
    const int kk = lhalf * 8;
    const int col = lrow ^ (lhalf << 4);            // rows 8..15 of a chunk live 16 columns over: the two halves of a warp
                                                    // (same lrow, other lhalf) no longer store to the same bank
    As[buf][kk + 0][col] = bf16_lo(ra.x); As[buf][kk + 1][col] = bf16_hi(ra.x);
    As[buf][kk + 2][col] = bf16_lo(ra.y); As[buf][kk + 3][col] = bf16_hi(ra.y);
    As[buf][kk + 4][col] = bf16_lo(ra.z); As[buf][kk + 5][col] = bf16_hi(ra.z);
    As[buf][kk + 6][col] = bf16_lo(ra.w); As[buf][kk + 7][col] = bf16_hi(ra.w);
    Bs[buf][kk + 0][col] = rb0.x; Bs[buf][kk + 1][col] = rb0.y; Bs[buf][kk + 2][col] = rb0.z; Bs[buf][kk + 3][col] = rb0.w;
    Bs[buf][kk + 4][col] = rb1.x; Bs[buf][kk + 5][col] = rb1.y; Bs[buf][kk + 6][col] = rb1.z; Bs[buf][kk + 7][col] = rb1.w;
  };
  const int ty = tid >> 4, tx = tid & 15;          // rows ty*8.., columns tx*8..
  float acc[8][8];
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 8; ++j) acc[i][j] = 0.f;

  gload(0);
  sstore(0);
  __syncthreads();
  for (int it = 0; it < n_it; ++it) {
    const int buf = it & 1;
    if (it + 1 < n_it) gload(it + 1);               // in flight during the multiply
#pragma unroll
    for (int kk = 0; kk < kGpBK; ++kk) {
      const int sw = (kk & 8) << 1;                 // the store-side swizzle, a compile-time constant per kk
      const float4 a0 = *reinterpret_cast<const float4*>(&As[buf][kk][(ty * 8) ^ sw]);
      const float4 a1 = *reinterpret_cast<const float4*>(&As[buf][kk][((ty * 8) ^ sw) + 4]);
      const float4 b0 = *reinterpret_cast<const float4*>(&Bs[buf][kk][(tx * 8) ^ sw]);
      const float4 b1 = *reinterpret_cast<const float4*>(&Bs[buf][kk][((tx * 8) ^ sw) + 4]);
      const float av[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
      const float bv[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[i][j] = fmaf(av[i], bv[j], acc[i][j]);
    }
    if (it + 1 < n_it) {
      sstore(buf ^ 1);                              // the other buffer was last read one iteration ago
      __syncthreads();
    }
  }
  float* zs = zp + (size_t)slice * T * E;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const int t = m0 + ty * 8 + i;
    if (t >= T) continue;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const int e = n0 + tx * 8 + j;
      if (e < E) zs[(size_t)t * E + e] = acc[i][j] + ((slice == 0 && gate_bias) ? gate_bias[e] : 0.f);
    }
  }
}

// Adds the split-K partials in slice order into zp[0] and runs the warp top-k (+signature): warp per token.
__global__ void __launch_bounds__(256) topk_splitk_kernel(TopkArgs a, float* __restrict__ zp, int n_slices) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int t = blockIdx.x * 8 + warp;
  if (t >= a.T) return;
  const size_t TE = (size_t)a.T * a.E;
  float* zrow = zp + (size_t)t * a.E;
  if (n_slices > 1) {
    for (int e = lane; e < a.E; e += 32) {
      // all partials of this logit requested before the first add (a dependent chain of loads costs one L2 round
      // trip per slice); the adds stay in slice order
      float v[8];
      const int n8 = min(n_slices, 8);
#pragma unroll
      for (int p = 0; p < 8; ++p) v[p] = p < n8 ? __ldcg(zp + (size_t)p * TE + (size_t)t * a.E + e) : 0.f;
      float s = v[0];
#pragma unroll
      for (int p = 1; p < 8; ++p) s += v[p];
      for (int p = 8; p < n_slices; ++p) s += __ldcg(zp + (size_t)p * TE + (size_t)t * a.E + e);
      zrow[e] = s;
    }
    __syncwarp();
  }
  int id; float w;
  warp_topk(zrow, a.E, a.k, a.renorm, lane, id, w);
  if (lane < a.k) {
    a.ids[(size_t)t * a.k + lane] = id;
    a.w[(size_t)t * a.k + lane] = w;
    sig_add(a.sig_req, a.sig_block, a.token_req ? a.token_req[t] : -1, a.token_block ? a.token_block[t] : -1,
            a.L, a.layer, a.E, id);
  }
}

}  // namespace eldr
