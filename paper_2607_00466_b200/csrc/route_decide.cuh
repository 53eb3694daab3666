// expert signature -> routing decision (PAPER.md:196-203 steps 2-4 of "Four steps build
// s_r": IDF reweight, layer mask, Eq. 2 normalisation; PAPER.md:239 locality-band routing).
//
//   route_sims_kernel   one CTA per request r, one warp per centroid k (strided): a single pass over the kept
//                       (layer, expert) cells accumulates  x.c,  |x|^2  and  |c|^2  in fp32, x = count * idf;
//                       sims[r,k] = x.c / (|x| |c|)   (0 if either vector is all zero).  Inputs are read once per
//                       (r,k); the request's row (L*E counts, <= 24 KiB) stays in L1/L2 across the K warps.
//   route_pick_kernel   similarities staged through shared memory by the whole CTA; ONE warp walks the requests
//                       in index order -- each decision sees the loads left by the previous ones ("updated as requests are dispatched") -- lanes stride over the workers:
//                       s* by redux-style max, band = {k : s_k >= s* - tau}, pick = smallest load, then larger
//                       similarity, then lower index; loads live in shared memory and are written back once.
// Latency-bound by construction (R*K*L*E*4 bytes of centroid reads from L2, a serial chain of R picks).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace eldr {

constexpr int kRouteMaxWorkers = 1024;

constexpr int kRouteMaxLayers = 256;
constexpr int kRouteStageCells = 12288;       // kept (layer, expert) cells whose x = count * idf is staged in shared memory (48 KiB)

__global__ void __launch_bounds__(256)
route_sims_kernel(const int32_t* __restrict__ counts, const float* __restrict__ idf,
                  const uint8_t* __restrict__ layer_mask, const float* __restrict__ centroids, float* __restrict__ sims,
                  int L, int E, int K) {
  // compact list of the kept layers, built once per CTA: the cell loop below has no dependent mask load and
  // keeps four independent (count, idf, centroid) triples in flight per lane
  __shared__ int s_kept[kRouteMaxLayers];
  __shared__ uint8_t s_mask[kRouteMaxLayers];
  __shared__ int s_nkept;
  for (int l = threadIdx.x; l < L; l += blockDim.x) s_mask[l] = layer_mask[l];     // one round trip, not L of them
  __syncthreads();
  if (threadIdx.x == 0) {
    int n = 0;
    for (int l = 0; l < L; ++l)
      if (s_mask[l]) s_kept[n++] = l;
    s_nkept = n;
  }
  __syncthreads();
  const int r = blockIdx.x;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5;
  const size_t D = (size_t)L * E;
  const int32_t* crow = counts + (size_t)r * D;
  const int n_cells = s_nkept * E;
  // x = count * idf over the kept cells, once per CTA (when it fits), and |x|^2 with it
  extern __shared__ float s_x[];
  const bool staged = n_cells <= kRouteStageCells;
  if (staged) {
    for (int i0 = threadIdx.x; i0 < n_cells; i0 += 8 * blockDim.x) {      // eight (count, idf) pairs in flight per thread
      int cv[8];
      float wv[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int i = i0 + u * blockDim.x;
        cv[u] = 0; wv[u] = 0.f;
        if (i < n_cells) {
          const int j = i / E;
          const size_t cell = (size_t)s_kept[j] * E + (i - j * E);
          cv[u] = __ldg(crow + cell);
          wv[u] = __ldg(idf + cell);
        }
      }
#pragma unroll
      for (int u = 0; u < 8; ++u) {
        const int i = i0 + u * blockDim.x;
        if (i < n_cells) s_x[i] = (float)cv[u] * wv[u];
      }
    }
    __syncthreads();
  }
  // blockIdx.y selects a group of n_warps centroids: one warp per centroid, sixteen cells in flight per lane
  for (int k = blockIdx.y * n_warps + warp; k < K; k += gridDim.y * n_warps) {
    const float* cen = centroids + (size_t)k * D;
    float dot = 0.f, xn = 0.f, cn = 0.f;
    for (int i0 = lane; i0 < n_cells; i0 += 512) {
      float x[16], c[16];
#pragma unroll
      for (int u = 0; u < 16; ++u) {
        const int i = i0 + 32 * u;
        x[u] = 0.f; c[u] = 0.f;
        if (i < n_cells) {
          const int j = i / E;
          const size_t cell = (size_t)s_kept[j] * E + (i - j * E);
          x[u] = staged ? s_x[i] : (float)__ldg(crow + cell) * __ldg(idf + cell);
          c[u] = __ldg(cen + cell);
        }
      }
#pragma unroll
      for (int u = 0; u < 16; ++u) {
        dot = fmaf(x[u], c[u], dot);
        xn = fmaf(x[u], x[u], xn);
        cn = fmaf(c[u], c[u], cn);
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

// order-preserving map float -> uint32 (-0 folded onto +0 so that equal values have equal keys)
__device__ __forceinline__ uint32_t route_order_key(float f) {
  const uint32_t b = __float_as_uint(f + 0.0f);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float route_from_order_key(uint32_t k) {
  return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}

constexpr int kRoutePickThreads = 256;
constexpr int kRoutePickChunkReq = 1024;
constexpr int kRouteSimChunk = 8192;          // similarities staged in shared memory per chunk of requests (32 KiB)

__global__ void __launch_bounds__(kRoutePickThreads)
route_pick_kernel(const float* __restrict__ sims, int32_t* __restrict__ loads, int32_t* __restrict__ worker,
                  int R, int K, float tau) {
  __shared__ int32_t s_load[kRouteMaxWorkers];
  __shared__ float s_sim[kRouteSimChunk];
  __shared__ int32_t s_worker[kRoutePickChunkReq];   // picks of the chunk: no global store inside the serial chain
  const int tid = threadIdx.x, lane = tid & 31;
  for (int k = tid; k < K; k += kRoutePickThreads) s_load[k] = loads[k];
  const int per = min(kRouteSimChunk / K, kRoutePickChunkReq);   // requests per chunk (K <= 1024 -> at least 8)
  for (int r0 = 0; r0 < R; r0 += per) {
    const int rn = min(per, R - r0);
    __syncthreads();                             // previous chunk consumed (and s_load ready the first time)
    for (int i = tid; i < rn * K; i += kRoutePickThreads) s_sim[i] = sims[(size_t)r0 * K + i];   // coalesced, all in flight
    __syncthreads();
    if (tid < 32) {
      for (int rr = 0; rr < rn; ++rr) {
        const float* s = s_sim + rr * K;
        // four hardware warp reductions per request instead of a twenty-shuffle tuple reduction (the chain of R
        // picks is serial, so its length is the latency): s*, then among the band the smallest load, among those
        // the largest similarity, among those the lowest index
        uint32_t bkey = 0u;
        for (int k = lane; k < K; k += 32) bkey = max(bkey, route_order_key(s[k]));
        const float best = route_from_order_key(__reduce_max_sync(0xffffffffu, bkey));
        const float edge = best - tau;
        uint32_t ml = 0xffffffffu;
        for (int k = lane; k < K; k += 32)
          if (s[k] >= edge) ml = min(ml, (uint32_t)s_load[k]);
        ml = __reduce_min_sync(0xffffffffu, ml);
        uint32_t mk = 0u;
        for (int k = lane; k < K; k += 32)
          if (s[k] >= edge && (uint32_t)s_load[k] == ml) mk = max(mk, route_order_key(s[k]));
        mk = __reduce_max_sync(0xffffffffu, mk);
        uint32_t pk_u = 0xffffffffu;
        for (int k = lane; k < K; k += 32)
          if (s[k] >= edge && (uint32_t)s_load[k] == ml && route_order_key(s[k]) == mk) { pk_u = (uint32_t)k; break; }
        const int pk = (int)__reduce_min_sync(0xffffffffu, pk_u);
        if (lane == 0) {
          s_worker[rr] = pk;
          s_load[pk] += 1;
        }
        __syncwarp();
      }
    }
    __syncthreads();
    for (int i = tid; i < rn; i += kRoutePickThreads) worker[r0 + i] = s_worker[i];
  }
  __syncthreads();
  for (int k = tid; k < K; k += kRoutePickThreads) loads[k] = s_load[k];
}

}  // namespace eldr
