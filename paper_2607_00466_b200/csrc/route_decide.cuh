// expert signature -> routing decision (PAPER.md:196-203 steps 2-4 of "Four steps build
// s_r": IDF reweight, layer mask, Eq. 2 normalisation; PAPER.md:239 locality-band routing).
//
//   route_sims_kernel   one CTA per request r, one warp per centroid k (strided): a single pass over the kept
//                       (layer, expert) cells accumulates  x.c,  |x|^2  and  |c|^2  in fp32, x = count * idf;
//                       sims[r,k] = x.c / (|x| |c|)   (0 if either vector is all zero).  Inputs are read once per
//                       (r,k); the request's row (L*E counts, <= 24 KiB) stays in L1/L2 across the K warps.
//   route_pick_kernel   ONE warp walks the requests in index order -- each decision sees the loads left by the
//                       previous ones ("updated as requests are dispatched") -- lanes stride over the workers:
//                       s* by redux-style max, band = {k : s_k >= s* - tau}, pick = smallest load, then larger
//                       similarity, then lower index; loads live in shared memory and are written back once.
// Latency-bound by construction (R*K*L*E*4 bytes of centroid reads from L2, a serial chain of R picks).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace eldr {

constexpr int kRouteMaxWorkers = 1024;

__global__ void __launch_bounds__(256)
route_sims_kernel(const int32_t* __restrict__ counts, const float* __restrict__ idf,
                  const uint8_t* __restrict__ layer_mask, const float* __restrict__ centroids, float* __restrict__ sims,
                  int L, int E, int K) {
  const int r = blockIdx.x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5;
  const size_t D = (size_t)L * E;
  const int32_t* crow = counts + (size_t)r * D;
  for (int k = warp; k < K; k += n_warps) {
    const float* cen = centroids + (size_t)k * D;
    float dot = 0.f, xn = 0.f, cn = 0.f;
    for (int l = 0; l < L; ++l) {
      if (!layer_mask[l]) continue;                      // warp-uniform
      const size_t base = (size_t)l * E;
      for (int e = lane; e < E; e += 32) {
        const float x = (float)crow[base + e] * idf[base + e];
        const float c = cen[base + e];
        dot = fmaf(x, c, dot);
        xn = fmaf(x, x, xn);
        cn = fmaf(c, c, cn);
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      dot += __shfl_xor_sync(0xffffffffu, dot, o);
      xn += __shfl_xor_sync(0xffffffffu, xn, o);
      cn += __shfl_xor_sync(0xffffffffu, cn, o);
    }
    if (lane == 0) sims[(size_t)r * K + k] = (xn > 0.f && cn > 0.f) ? dot / (sqrtf(xn) * sqrtf(cn)) : 0.f;
  }
}

// better(a, b): a precedes b in (load ascending, similarity descending, index ascending)
__device__ __forceinline__ bool route_better(int la, float sa, int ka, int lb, float sb, int kb) {
  if (la != lb) return la < lb;
  if (sa != sb) return sa > sb;
  return ka < kb;
}

__global__ void __launch_bounds__(32)
route_pick_kernel(const float* __restrict__ sims, int32_t* __restrict__ loads, int32_t* __restrict__ worker,
                  int R, int K, float tau) {
  __shared__ int32_t s_load[kRouteMaxWorkers];
  const int lane = threadIdx.x;
  for (int k = lane; k < K; k += 32) s_load[k] = loads[k];
  __syncwarp();
  for (int r = 0; r < R; ++r) {
    const float* s = sims + (size_t)r * K;
    float best = -2.f;
    for (int k = lane; k < K; k += 32) best = fmaxf(best, s[k]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) best = fmaxf(best, __shfl_xor_sync(0xffffffffu, best, o));
    const float edge = best - tau;
    int pl = 0x7fffffff, pk = 0x7fffffff;
    float ps = -2.f;
    for (int k = lane; k < K; k += 32) {
      const float sk = s[k];
      if (sk >= edge && route_better(s_load[k], sk, k, pl, ps, pk)) { pl = s_load[k]; ps = sk; pk = k; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const int ol = __shfl_xor_sync(0xffffffffu, pl, o);
      const float os = __shfl_xor_sync(0xffffffffu, ps, o);
      const int ok = __shfl_xor_sync(0xffffffffu, pk, o);
      if (route_better(ol, os, ok, pl, ps, pk)) { pl = ol; ps = os; pk = ok; }
    }
    if (lane == 0) {
      worker[r] = pk;
      s_load[pk] += 1;
    }
    __syncwarp();
  }
  for (int k = lane; k < K; k += 32) loads[k] = s_load[k];
}

}  // namespace eldr
