// CUDA-core GEMV expert FFN for very small tokens-per-expert counts (north_star: "Tensor cores ... are used only where
// tokens-per-expert fill a tile, with a CUDA-core GEMV path otherwise").  Selectable with
// ELDR_OPT_FFN_PATH = ELDR_FFN_GEMV on the staged path; NOT the default: measured against the tcgen05 swap-AB kernels it
// is never faster, not even at one token per expert (profiles/r2_gemv_vs_tcgen05.md) -- the tensor-core path leaves
// the SM's issue slots to the TMA producers, this one spends them on loads and FMAs.
//
// One persistent CTA per SM, 32 warps.  A work unit is the same row tile as in the tensor-core kernels (MODE 0: 64
// intermediate indices = 64 rows of w1 + the same 64 of w3; MODE 1: 128 rows of w2).  The expert's token rows (at most
// kGemvTok per pass) sit in shared memory as bf16; a warp owns whole weight rows: its lanes sweep the row in 16-byte
// chunks (8 bf16, coalesced 512 bytes per warp instruction, L1 bypassed, four chunks in flight per lane), multiply
// each chunk with the matching chunk of every token in fp32, and a butterfly reduction finishes the dot products.
// Same arithmetic contract as the other paths: bf16 operands, fp32 accumulation, h rounded once to bf16, y fp32.
#pragma once
#include "device_utils.cuh"
#include "ffn_stream.cuh"   // FfnArgs

namespace eldr {

constexpr int kGemvThreads = 1024;
constexpr int kGemvTok = 8;            // tokens per pass (accumulators per lane: kGemvTok, twice that in MODE 0)

__device__ __forceinline__ void gemv_fma8(const uint4& w, const uint4& x, float& acc) {
  acc = fmaf(bf16_lo(w.x), bf16_lo(x.x), acc); acc = fmaf(bf16_hi(w.x), bf16_hi(x.x), acc);
  acc = fmaf(bf16_lo(w.y), bf16_lo(x.y), acc); acc = fmaf(bf16_hi(w.y), bf16_hi(x.y), acc);
  acc = fmaf(bf16_lo(w.z), bf16_lo(x.z), acc); acc = fmaf(bf16_hi(w.z), bf16_hi(x.z), acc);
  acc = fmaf(bf16_lo(w.w), bf16_lo(x.w), acc); acc = fmaf(bf16_hi(w.w), bf16_hi(x.w), acc);
}

template <int MODE>
__global__ void __launch_bounds__(kGemvThreads, 1)
ffn_gemv_kernel(const uint16_t* __restrict__ w, const uint16_t* __restrict__ w_shared, const uint16_t* __restrict__ xin,
                const FfnArgs a) {
  extern __shared__ __align__(16) uint8_t gemv_smem[];          // [kGemvTok][K] bf16
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  pdl_launch_dependents();
  pdl_wait();
  const int n_work = *a.n_work;
  const int total_tiles = n_work * a.tiles_per_expert;
  const int K = a.K, kvec = K >> 3;                              // 16-byte chunks per row
  const uint4* xs = reinterpret_cast<const uint4*>(gemv_smem);
  int staged_ent = -1, staged_n0 = -1;
  for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
    const int ent = tile / a.tiles_per_expert, rt = tile - ent * a.tiles_per_expert;
    const int4 wk = a.work[ent];
    const bool shared = wk.x >= a.E;
    const uint16_t* wbase = (shared ? w_shared : w) + (size_t)(shared ? wk.x - a.E : wk.x) * a.rows_per_expert * K;
    const int xrow0 = (MODE == 0) ? wk.y : wk.z;
    for (int n0 = 0; n0 < wk.w; n0 += kGemvTok) {
      const int m = min(kGemvTok, wk.w - n0);
      if (ent != staged_ent || n0 != staged_n0) {
        __syncthreads();                                         // the previous pass's readers are done
        uint4* dst = reinterpret_cast<uint4*>(gemv_smem);
        for (int i = threadIdx.x; i < kGemvTok * kvec; i += kGemvThreads) {
          const int t = i / kvec, c = i - t * kvec;
          dst[i] = t < m ? ld_nc_v4(xin + (size_t)(xrow0 + n0 + t) * K + (size_t)c * 8) : make_uint4(0u, 0u, 0u, 0u);
        }
        __syncthreads();
        staged_ent = ent; staged_n0 = n0;
      }
      const int rows_in_tile = MODE == 0 ? 64 : 128;
      for (int r = warp; r < rows_in_tile; r += kGemvThreads / 32) {
        const int row = rt * rows_in_tile + r;                   // MODE 0: intermediate index i; MODE 1: output row
        if (MODE == 1 && row >= a.H) break;
        if (MODE == 0 && row >= a.I) break;                       // I not a multiple of 64: the last tile is partial
        const uint4* w0 = reinterpret_cast<const uint4*>(wbase + (size_t)row * K);
        const uint4* w1 = reinterpret_cast<const uint4*>(wbase + (size_t)(row + a.I) * K);     // MODE 0: the w3 row
        float acc0[kGemvTok], acc1[kGemvTok];
#pragma unroll
        for (int t = 0; t < kGemvTok; ++t) { acc0[t] = 0.f; acc1[t] = 0.f; }
        for (int c0 = lane; c0 < kvec; c0 += 128) {
          uint4 wa[4], wb[4];
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int c = c0 + 32 * u;
            wa[u] = c < kvec ? ld_nc_v4(w0 + c) : make_uint4(0u, 0u, 0u, 0u);
            if (MODE == 0) wb[u] = c < kvec ? ld_nc_v4(w1 + c) : make_uint4(0u, 0u, 0u, 0u);
          }
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int c = c0 + 32 * u;
            if (c < kvec) {
#pragma unroll
              for (int t = 0; t < kGemvTok; ++t) {
                if (t < m) {
                  const uint4 xv = xs[t * kvec + c];
                  gemv_fma8(wa[u], xv, acc0[t]);
                  if (MODE == 0) gemv_fma8(wb[u], xv, acc1[t]);
                }
              }
            }
          }
        }
#pragma unroll
        for (int t = 0; t < kGemvTok; ++t) {
          if (t < m) {
            float s0 = acc0[t], s1 = acc1[t];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
              s0 += __shfl_xor_sync(0xffffffffu, s0, o);
              if (MODE == 0) s1 += __shfl_xor_sync(0xffffffffu, s1, o);
            }
            if (lane == 0) {
              if (MODE == 0) a.h_out[(size_t)(wk.z + n0 + t) * a.I + row] = f32_to_bf16_rn(silu_f(s0) * s1);
              else a.y_out[(size_t)(wk.z + n0 + t) * a.H + row] = s0;
            }
          }
        }
      }
    }
  }
}

}  // namespace eldr
