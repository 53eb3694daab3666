// Grouped SwiGLU expert FFN: weight-streaming kernels ("each step
// fetches the weights of every expert the batch activates").
//
// One persistent CTA per SM.  A producer warp streams 128-row x 64-column bf16 weight tiles (16 KiB) of the
// ACTIVE experts only through an NSTAGE-deep TMA + mbarrier ring (SWIZZLE_128B), together with the matching
// 64-column slice of the expert's gathered token rows.  Eight consumer warps read 16-byte fragments straight
// out of the swizzled tiles and feed mma.sync.m16n8k16 (bf16 x bf16 -> fp32): weights are the M=16 operand,
// tokens the N=8 operand.  The k index inside every 32-column group is permuted identically for A and B
// (thread q owns columns 8q..8q+7), so each fragment is ONE conflict-free 16-byte shared load -- no ldmatrix,
// no transposes.  Rows are visited in the order rho = (0,4,1,5,2,6,3,7) so that the two rows touched by one
// quarter-warp phase land in disjoint bank groups under the 128-byte swizzle.
//
// MODE 0 (w1/w3): warp w pairs 8 rows of W1 with the same 8 rows of W3 in one M=16 tile, so silu(g)*u is
//                 formed in registers; writes h (bf16) per sorted pair.
// MODE 1 (w2):    warp w owns 16 rows of W2; writes y (fp32) per sorted pair for the ordered combine.
#pragma once
#include "device_utils.cuh"

namespace eldr {

constexpr int kFfnStages = 8;
constexpr int kFfnKC = 64;                      // columns per stage (128 bytes of bf16)
constexpr int kFfnTileRows = 128;               // weight rows per stage
constexpr int kFfnWBytes = kFfnTileRows * 128;  // 16 KiB
constexpr int kFfnXRows = 64;                   // token rows per pass (8 n-tiles)
constexpr int kFfnXBox = 16;                    // token rows per TMA box
constexpr int kFfnXBytes = kFfnXRows * 128;     // 8 KiB
constexpr int kFfnStageBytes = kFfnWBytes + kFfnXBytes;
constexpr int kFfnConsumerWarps = 8;
constexpr int kFfnThreads = (kFfnConsumerWarps + 1) * 32;
constexpr size_t kFfnSmemBytes = (size_t)kFfnStages * kFfnStageBytes + 1024 /*align*/ + 256 /*barriers*/;

struct FfnArgs {
  const int4* work;        // {expert, x_row0, out_row0, m}; mode 1 reads its B rows (h) at out_row0
  const int32_t* n_work;
  int E;                   // routed experts (expert >= E => shared expert expert-E)
  int K;                   // reduction length: H (mode 0) or I (mode 1)
  int rows_per_expert;     // 2I (mode 0) or H (mode 1)
  int I;                   // intermediate size
  int H;
  int tiles_per_expert;    // I/64 (mode 0) or ceil(H/128) (mode 1)
  uint16_t* h_out;         // mode 0: [rows, I] bf16
  float* y_out;            // mode 1: [rows, H] fp32
};

template <int MODE>
__global__ void __launch_bounds__(kFfnThreads, 1)
ffn_stream_kernel(const __grid_constant__ CUtensorMap tm_w, const __grid_constant__ CUtensorMap tm_ws,
                  const __grid_constant__ CUtensorMap tm_x, const FfnArgs a) {
  extern __shared__ uint8_t smem_dyn[];
  const uint32_t smem_base = (smem_u32(smem_dyn) + 1023u) & ~1023u;     // SWIZZLE_128B atoms: 1024-byte aligned
  const uint32_t bar_base = smem_base + kFfnStages * kFfnStageBytes;
  auto full_bar = [&](int s) { return bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return bar_base + 8u * (kFfnStages + s); };

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < kFfnStages; ++s) {
      mbar_init(full_bar(s), 1);
      mbar_init(empty_bar(s), kFfnConsumerWarps);
    }
    mbar_fence_init();
  }
  __syncthreads();
  pdl_launch_dependents();
  pdl_wait();

  const int n_work = *a.n_work;
  const int total_tiles = n_work * a.tiles_per_expert;
  const int k_iters = a.K / kFfnKC;
  uint32_t it = 0;     // ring position, advanced identically by producer and consumers

  if (warp == kFfnConsumerWarps) {
    // ===================================================================== TMA producer (one lane)
    if (lane == 0) {
      tma_prefetch_desc(&tm_w);
      tma_prefetch_desc(&tm_x);
      const uint64_t pol_stream = l2_policy_evict_first();   // weights: read exactly once
      const uint64_t pol_keep = l2_policy_evict_last();      // activations: re-read by every row tile
      for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
        const int ent = tile / a.tiles_per_expert, rt = tile - ent * a.tiles_per_expert;
        const int4 wk = a.work[ent];
        const bool shared = wk.x >= a.E;
        const CUtensorMap* tmw = shared ? &tm_ws : &tm_w;
        const int wrow0 = (shared ? wk.x - a.E : wk.x) * a.rows_per_expert;
        for (int n0 = 0; n0 < wk.w; n0 += kFfnXRows) {
          const int n_here = min(kFfnXRows, wk.w - n0);
          const int n_box = (n_here + kFfnXBox - 1) / kFfnXBox;
          const uint32_t tx = kFfnWBytes + n_box * (kFfnXBox * 128);
          for (int kc = 0; kc < k_iters; ++kc, ++it) {
            const int s = it % kFfnStages;
            mbar_wait(empty_bar(s), ((it / kFfnStages) & 1) ^ 1);
            const uint32_t dst = smem_base + s * kFfnStageBytes;
            mbar_arrive_expect_tx(full_bar(s), tx);
            if (MODE == 0) {
              tma_load_2d(dst, tmw, kc * kFfnKC, wrow0 + rt * 64, full_bar(s), pol_stream);
              tma_load_2d(dst + 8192, tmw, kc * kFfnKC, wrow0 + a.I + rt * 64, full_bar(s), pol_stream);
            } else {
              tma_load_2d(dst, tmw, kc * kFfnKC, wrow0 + rt * 128, full_bar(s), pol_stream);
            }
            for (int b = 0; b < n_box; ++b)
              tma_load_2d(dst + kFfnWBytes + b * (kFfnXBox * 128), &tm_x, kc * kFfnKC,
                          (MODE == 0 ? wk.y : wk.z) + n0 + b * kFfnXBox, full_bar(s), pol_keep);
          }
        }
      }
    }
    return;
  }

  // ========================================================================= consumers (8 warps)
  const int g = lane >> 2, q = lane & 3;
  const int rho = (g >> 1) + ((g & 1) << 2);            // (0,4,1,5,2,6,3,7)
  const int rowA0 = (MODE == 0) ? (8 * warp + rho) : (16 * warp + rho);
  const int rowA1 = (MODE == 0) ? (64 + 8 * warp + rho) : (16 * warp + 8 + rho);
  const uint32_t offA0 = rowA0 * 128, offA1 = rowA1 * 128;
  const uint32_t sw0 = ((uint32_t)(q ^ rho)) << 4;          // chunk (q)   ^ (row & 7)
  const uint32_t sw1 = ((uint32_t)((4 + q) ^ rho)) << 4;    // chunk (4+q) ^ (row & 7)

  for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
    const int ent = tile / a.tiles_per_expert, rt = tile - ent * a.tiles_per_expert;
    const int4 wk = a.work[ent];
    for (int n0 = 0; n0 < wk.w; n0 += kFfnXRows) {
      const int n_here = min(kFfnXRows, wk.w - n0);
      const int nt = (n_here + 7) >> 3;
      float acc[8][4];
#pragma unroll
      for (int j = 0; j < 8; ++j) { acc[j][0] = acc[j][1] = acc[j][2] = acc[j][3] = 0.f; }

      for (int kc = 0; kc < k_iters; ++kc, ++it) {
        const int s = it % kFfnStages;
        mbar_wait(full_bar(s), (it / kFfnStages) & 1);
        const uint32_t sA = smem_base + s * kFfnStageBytes;
        const uint32_t sX = sA + kFfnWBytes + rho * 128;
#pragma unroll
        for (int half = 0; half < 2; ++half) {
          const uint32_t sw = half ? sw1 : sw0;
          const uint4 A0 = lds_v4(sA + offA0 + sw);
          const uint4 A1 = lds_v4(sA + offA1 + sw);
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            if (j < nt) {
              const uint4 B = lds_v4(sX + j * 1024 + sw);
              mma_bf16_16816(acc[j], A0.x, A1.x, A0.y, A1.y, B.x, B.y);
              mma_bf16_16816(acc[j], A0.z, A1.z, A0.w, A1.w, B.z, B.w);
            }
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(empty_bar(s));
      }

      // ------------------------------------------------------------------------------ epilogue
      // C fragment: c0/c1 = row g (tile row rowA0), tokens 2q / 2q+1 of the n-tile; c2/c3 = row g+8 (rowA1).
      // n-tile column n was loaded by the thread group with g == n, i.e. token row 8j + rho(n):
      // rho(2q) = q, rho(2q+1) = q + 4.
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        if (j < nt) {
          const int tok0 = n0 + 8 * j + q, tok1 = tok0 + 4;
          if (MODE == 0) {
            const int i = rt * 64 + 8 * warp + rho;
            if (tok0 < wk.w)
              a.h_out[(size_t)(wk.z + tok0) * a.I + i] = f32_to_bf16_rn(silu_f(acc[j][0]) * acc[j][2]);
            if (tok1 < wk.w)
              a.h_out[(size_t)(wk.z + tok1) * a.I + i] = f32_to_bf16_rn(silu_f(acc[j][1]) * acc[j][3]);
          } else {
            const int r0 = rt * 128 + 16 * warp + rho, r1 = r0 + 8;
            if (tok0 < wk.w) {
              if (r0 < a.H) a.y_out[(size_t)(wk.z + tok0) * a.H + r0] = acc[j][0];
              if (r1 < a.H) a.y_out[(size_t)(wk.z + tok0) * a.H + r1] = acc[j][2];
            }
            if (tok1 < wk.w) {
              if (r0 < a.H) a.y_out[(size_t)(wk.z + tok1) * a.H + r0] = acc[j][1];
              if (r1 < a.H) a.y_out[(size_t)(wk.z + tok1) * a.H + r1] = acc[j][3];
            }
          }
        }
      }
    }
  }
}

// ----------------------------------------------------------------------------------------------
// Plain CUDA-core path for shapes the TMA path does not take (H or I not a multiple of 64).  Correct for
// any H, I multiple of 8; not a performance path.  One CTA per streamed expert; thread per output row.
// ----------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) ffn13_plain_kernel(const uint16_t* __restrict__ w13,
                                                          const uint16_t* __restrict__ shared_w13,
                                                          const uint16_t* __restrict__ x_perm, FfnArgs a) {
  pdl_launch_dependents();
  pdl_wait();
  if ((int)blockIdx.x >= *a.n_work) return;
  const int4 wk = a.work[blockIdx.x];
  const bool shared = wk.x >= a.E;
  const uint16_t* wb = (shared ? shared_w13 : w13) + (size_t)(shared ? wk.x - a.E : wk.x) * 2 * a.I * a.H;
  for (int i = blockIdx.y * 128 + threadIdx.x; i < a.I; i += gridDim.y * 128) {
    const uint16_t* r1 = wb + (size_t)i * a.H;
    const uint16_t* r3 = wb + (size_t)(a.I + i) * a.H;
    for (int n = 0; n < wk.w; ++n) {
      const uint16_t* xr = x_perm + (size_t)(wk.y + n) * a.H;
      float gsum = 0.f, usum = 0.f;
      for (int c = 0; c < a.H; ++c) {
        const float xv = bf16_lo(xr[c]);
        gsum = fmaf(bf16_lo(r1[c]), xv, gsum);
        usum = fmaf(bf16_lo(r3[c]), xv, usum);
      }
      a.h_out[(size_t)(wk.z + n) * a.I + i] = f32_to_bf16_rn(silu_f(gsum) * usum);
    }
  }
}

__global__ void __launch_bounds__(128) ffn2_plain_kernel(const uint16_t* __restrict__ w2,
                                                         const uint16_t* __restrict__ shared_w2,
                                                         const uint16_t* __restrict__ h, FfnArgs a) {
  pdl_launch_dependents();
  pdl_wait();
  if ((int)blockIdx.x >= *a.n_work) return;
  const int4 wk = a.work[blockIdx.x];
  const bool shared = wk.x >= a.E;
  const uint16_t* wb = (shared ? shared_w2 : w2) + (size_t)(shared ? wk.x - a.E : wk.x) * a.H * a.I;
  for (int r = blockIdx.y * 128 + threadIdx.x; r < a.H; r += gridDim.y * 128) {
    const uint16_t* row = wb + (size_t)r * a.I;
    for (int n = 0; n < wk.w; ++n) {
      const uint16_t* hr = h + (size_t)(wk.z + n) * a.I;
      float acc = 0.f;
      for (int i = 0; i < a.I; ++i) acc = fmaf(bf16_lo(row[i]), bf16_lo(hr[i]), acc);
      a.y_out[(size_t)(wk.z + n) * a.H + r] = acc;
    }
  }
}

}  // namespace eldr
