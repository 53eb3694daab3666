// The whole decode step of one MoE layer in ONE persistent launch (PAPER.md:79
// "the gate partitions the batch among experts ... each step fetches the weights of every expert the batch
// activates"; PAPER.md:198/:253 signature counts).  One CTA per SM, 8 warps.
//
//   G  gate GEMV: GT-token x 8-expert logit tiles spread over the grid (GT = 8 / 16 / 32 for T <= 64 / 128 / 256: one
//      round of tiles).  fp32 FMA on CUDA cores; a warp owns 2 experts x GT/2 tokens, gate rows are requested 8 float4
//      deep per row BEFORE the x tile is staged so both latencies overlap.  Each tile publishes an epoch flag.
//   K  top-k: the CTA that owns token group g polls the group's tile flags, runs a redux-based warp top-k
//      (+ fused signature increments) and publishes ids and weights as epoch-tagged 64-bit words.
//   R  routing, redundantly in EVERY CTA from the tagged ids: membership bitmasks -> counts -> offsets ->
//      union-compacted work list (shared experts first; the weights producer starts streaming here) -> token<->position
//      maps, all in shared memory.  No second election, no route/gather kernels, no work list in HBM.
//      CTA 0 also writes the routing outputs of the C ABI (active list, n_active, cnt/off/perm/pair_pos).
//   F  expert FFN on tcgen05 + TMEM, swap-AB (weights = M=128 operand, the expert's tokens = N operand).  Per
//      phase (A: w1/w3 tiles, B: w2 tiles) the tile list is entry-major.  Schedule (PieceWalker, below): a phase with
//      at least one round of gridDim.x tiles runs WHOLE tiles -- CTA c's first tile is tile c, further ones are drawn
//      from a global counter by its weights producer (SMs get unequal shares of a saturated HBM, so fast SMs draw
//      more), the tiles past the last whole round go whole to as many CTAs while the others move on; a phase shorter
//      than one round is a STATIC stream-K schedule: the flattened sequence of 16 KiB weight stages (tile-major,
//      k-chunk minor) is cut into gridDim.x equal contiguous ranges.  A tile cut by a range boundary is finished by the
//      CTA that owns its k=0 end: the other owner(s) -- which reach the tile FIRST, at the start of their range -- park
//      raw fp32 accumulators in a scratch slot and raise a flag; the head owner adds them in ascending CTA order (a
//      fixed order: results are run-to-run bit-identical whichever CTA computed a whole tile).  Weights: TMA
//      (SWIZZLE_128B, evict_first).  Activations: TMA too -- tile::gather4 pulls the expert's token rows straight
//      from x (A; wide batches: 16-row boxes of an expert-sorted copy of x written at the start of the phase), 16-row
//      boxes read h (B) -- into the swizzled K-major B tile.  Phase B waits on per-tile epoch flags of the expert's h
//      tiles (release/acquire through L2, proxy fences around the TMA reads).  Phase A never waits on phase B and first
//      pieces never wait on anything, so there is no cycle.  Because whole tiles finish in work-list order, B's first
//      rounds find their h long finished: no pipeline drain at the hand-over when the union is large.
//      The B-tile rows per stage adapt to the batch's largest tokens-per-expert count, so small-m steps get a
//      deeper weight ring (more bytes in flight).
//   C  flag-driven ordered combine (no grid barrier): out[t] = sum_j w[t,j]*y[pos(t,j)] (+ shared) in slot order, one
//      RNE rounding to bf16, each (token, 128-column tile) as soon as its y tiles are flagged.
//
// Nothing needs zeroing by the host: flags compare against the step's epoch (device_utils.cuh: a full-period sequence
// state kept in the workspace, salted with the workspace address); the state lives in the workspace and is
// bumped by the last CTA to leave the step (the launch is CUDA-graph capturable; a workspace of arbitrary initial
// contents works up to a 2^-32 flag collision).
#pragma once
#include "device_utils.cuh"
#include "ffn_umma.cuh"
#include "gate_route.cuh"

namespace eldr {

constexpr int kFusedThreads = 256;
constexpr int kFusedMaxT = 256;
constexpr int kNPCap = 128;               // token columns per accumulator pass (TMEM: 2 x 128 columns)
constexpr int kMaxStages = 12;
constexpr int kClaimSlots = 4;            // claimed-tile ring: weights producer -> the seven consumer warps

// sync region (uint32 words) at the START of the layer workspace
constexpr int kSyncGen = 0;
constexpr int kSyncCntReady = 1;                // CTA 0 zeroed this step's tile counters
constexpr int kSyncTileCnt = 2;                 // [2] next unclaimed data-parallel tile of phase A / B
constexpr int kSyncExit = 4;                    // CTAs that have left the step (zeroed by CTA 0 with the tile counters; the last one bumps the generation)
constexpr int kSyncXReady = 32;                 // [256]     per CTA "my rows of the expert-sorted copy of x are written"
constexpr int kSyncGroup = kSyncXReady + 256;     // [32]      per token group "ids/weights written"
constexpr int kSyncTile = kSyncGroup + 32;      // [32][32]  gate logit tile written
constexpr int kSyncPartial = kSyncTile + 1024;  // [4][256]  per (sub-phase, CTA) "partial accumulators parked"
constexpr int kSyncHReady = kSyncPartial + 1024; // [(E+ns)*2*tilesA] per phase-A tile "h tile written", then
                                                 // [(E+ns)*2*tilesB] per phase-B tile "y tile written"

// Tagged ids: one 64-bit word {epoch : 32 | four expert ids, one byte each : 32} per (token, group of four top-k
// slots), written by the token group's owner after its top-k and polled by every CTA.  Tag and payload arrive in one
// atomic 8-byte access, so the routing input needs no flag, no release and no second L2 round trip.  (The same
// scheme for the logits was measured slower than tile flags + plain loads and is not used.)
constexpr int kIdWordsPerTok = 4;         // kMaxTopK / 4
__host__ __device__ inline size_t fused_ydone_word_offset(int E, int ns, int I) {
  return (size_t)kSyncHReady + (size_t)(E + ns) * 2 * ((I + 63) / 64);
}
__host__ __device__ inline size_t fused_idt_word_offset(int E, int ns, int I, int H) {
  return (fused_ydone_word_offset(E, ns, I) + (size_t)(E + ns) * 2 * ((H + 127) / 128) + 1) & ~(size_t)1;
}
// Tagged weights: {epoch : 32 | fp32 weight : 32} per (token, slot), written by the top-k owner and polled by the
// warp that combines the token -- value and tag in one atomic word, so the combine needs no fence for them.
__host__ __device__ inline size_t fused_wtag_word_offset(int E, int ns, int I, int H) {
  return fused_idt_word_offset(E, ns, I, H) + (size_t)kFusedMaxT * kIdWordsPerTok * 2;
}
__host__ __device__ inline size_t fused_sync_words(int E, int ns, int I, int H) {
  return fused_wtag_word_offset(E, ns, I, H) + (size_t)kFusedMaxT * 16 * 2;
}
__host__ __device__ inline size_t fused_partial_bytes(int n_cta) {
  return (size_t)4 * n_cta * 128 * kNPCap * 4;
}

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
  unsigned long long* idt;     // [T][4] tagged top-k ids (inside the sync region)
  unsigned long long* wtag;    // [T][16] tagged top-k weights (inside the sync region)
  float* partial;              // [4][gridDim.x][128][kNPCap] fp32 scratch of the stream-K fix-up
  uint16_t* xs;                // [T*k (+T), H] bf16: x rows in expert-sorted position order (wide batches only)
  uint16_t* hbuf;              // [T*(k+ns), I] bf16
  float* ybuf;                 // [T*(k+ns), H] fp32
  uint16_t* out;               // [T,H] bf16
  int stage_area;              // bytes of shared memory cut into ring stages (multiple of 1024; set by the host)
  int ring_bytes;              // cap on the bytes the ring keeps in flight (<= stage_area)
  int dp_min_rounds;           // hybrid schedule: data-parallel part only if a phase has at least this many tile rounds
  int sk_split_pct;            // small unions (whole phase stream-K): share of the accumulator passes in the first expert group
  int xs_min_np;               // experts with this many token columns or more (np, padded to 16): phase A reads the sorted copy of x
  int sk_max_split;            // large unions: at most this many pieces per tile of a stream-K remainder (0: cut over the whole grid)
  int head_first;              // static ranges: head piece first and parked, split tiles finished by the owner of their last stage
};

#ifdef ELDR_TRACE
__device__ __forceinline__ unsigned long long gtime() {
  unsigned long long t_;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_));
  return t_;
}
#define FSTAMP(id) do { g_trace[(blockIdx.x & 4095) * 16 + (id)] = gtime(); } while (0)
#define FVALUE(id, v) do { g_trace[(blockIdx.x & 4095) * 16 + (id)] = (unsigned long long)(v); } while (0)
#define FVALUE2(id, v) do { g_trace[((blockIdx.x + 2048) & 4095) * 16 + (id)] = (unsigned long long)(v); } while (0)
#define FSTAMP2(id) do { g_trace[((blockIdx.x + 2048) & 4095) * 16 + (id)] = gtime(); } while (0)
#define FTIMED(acc, stmt) do { const long long c0_ = clock64(); stmt; acc += clock64() - c0_; } while (0)
#define FSTAMP3(id) do { g_trace[((blockIdx.x + 1024) & 4095) * 16 + (id)] = gtime(); } while (0)
#define FADD3(id, v) do { g_trace[((blockIdx.x + 1024) & 4095) * 16 + (id)] += (unsigned long long)(v); } while (0)
#define FADD4(id, v) do { g_trace[((blockIdx.x + 3072) & 4095) * 16 + (id)] += (unsigned long long)(v); } while (0)
#else
#define FADD4(id, v) do {} while (0)
#define FSTAMP3(id) do {} while (0)
#define FADD3(id, v) do {} while (0)
#define FSTAMP2(id) do {} while (0)
#define FVALUE2(id, v) do {} while (0)
#define FTIMED(acc, stmt) do { stmt; } while (0)
#define FSTAMP(id) do {} while (0)
#define FVALUE(id, v) do {} while (0)
#endif

__device__ __forceinline__ void flag_release(uint32_t* p, uint32_t v) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" :: "l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t flag_acquire(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ uint32_t flag_relaxed(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void fence_acq_rel_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
// One warp waits until flags[0..n) all equal epoch.  Every lane keeps all of its flags' (relaxed) loads in flight
// together -- a chain of acquire loads costs one L2 round trip per flag -- and one fence after the last successful
// poll gives the acquire.  A short sleep between polls keeps 148 pollers from saturating the flags' L2 slice.
// Traps instead of hanging.
__device__ __forceinline__ void warp_wait_flags(const uint32_t* flags, int n, uint32_t epoch, int lane) {
  uint32_t spins = 0;
  for (;;) {
    bool ok = true;
    for (int i0 = 0; i0 < n; i0 += 256) {
      uint32_t v[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const int i = i0 + lane + 32 * j;
        v[j] = (i < n) ? flag_relaxed(flags + i) : epoch;
      }
#pragma unroll
      for (int j = 0; j < 8; ++j) ok = ok && (v[j] == epoch);
    }
    if (__all_sync(0xffffffffu, ok)) break;
    __nanosleep(40);
    if (++spins > (1u << 24)) __trap();
  }
  fence_acq_rel_gpu();
  __syncwarp();
}
__device__ __forceinline__ bool warp_test_flags(const uint32_t* flags, int n, uint32_t epoch, int lane) {
  bool ok = true;
  for (int i = lane; i < n; i += 32) ok = ok && (flag_acquire(flags + i) == epoch);
  return __all_sync(0xffffffffu, ok);
}

__device__ __forceinline__ void st_relaxed_u64(unsigned long long* p, unsigned long long v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" :: "l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" :: "n"(N) : "memory"); }
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ------------------------------------------------------------------------------------ G: one logit tile
// GT tokens (token tile g) x 8 experts (tile et).  Warp w: experts 2*(w&3), 2*(w&3)+1 of the tile, tokens
// (GT/2)*(w>>2)..+GT/2-1.  GT = 8 for T <= 64; 16 / 32 for T <= 128 / 256 so that the whole gate stays ONE round of
// tiles over the grid (8-token tiles took 2 / 4 rounds of ~4 us there).  GT is a template parameter of the whole
// kernel: the wider tiles live in their own instantiations and do not perturb the code generated for T <= 64.
template <int GT>
__device__ __forceinline__ void fused_gate_tile(const FusedArgs& a, int et, int g, uint8_t* smem_raw, uint32_t gbar,
                                                uint32_t gpar) {
  constexpr int TW = GT / 2;              // tokens per warp
  const int T = a.tk.T, H = a.H, E = a.tk.E;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int t0 = g * GT;
  const int ep = warp & 3, th = warp >> 2;
  const int e0 = et * kGateExp + 2 * ep, e1 = e0 + 1;
  const int q_per_row = H >> 2;
  constexpr int kDepth = 8;                    // float4 per gate row requested before the x tile is staged (16: no faster, measured)
  const float4* wrow0 = reinterpret_cast<const float4*>(a.gate_w + (size_t)(e0 < E ? e0 : 0) * H);
  const float4* wrow1 = reinterpret_cast<const float4*>(a.gate_w + (size_t)(e1 < E ? e1 : 0) * H);
  const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
  float4 wa[kDepth], wb[kDepth];
#pragma unroll
  for (int u = 0; u < kDepth; ++u) {
    const int c4 = lane + 32 * u;
    wa[u] = (c4 < q_per_row) ? __ldg(wrow0 + c4) : zero4;
    wb[u] = (c4 < q_per_row) ? __ldg(wrow1 + c4) : zero4;
  }
  uint4* xs4 = reinterpret_cast<uint4*>(smem_raw);
  const int vec_per_row = H >> 3;
  const int n_vec = GT * vec_per_row;
  __syncthreads();                       // the previous tile's readers are done with the x tile
  if (GT > 8) {
    // wide tiles (64 / 128 KiB of x): the tile's token rows are contiguous in x -- ONE bulk copy by the TMA engine
    // instead of four register round trips per thread (T = 256: gate tiles done 11.5 us after the start)
    const int rows = min(GT, T - t0);
    if (tid == 0) {
      const uint32_t bytes = (uint32_t)rows * (uint32_t)H * 2u;
      mbar_arrive_expect_tx(gbar, bytes);
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                   :: "r"(smem_u32(smem_raw)), "l"(a.x + (size_t)t0 * H), "r"(bytes), "r"(gbar) : "memory");
    }
    for (int v = rows * vec_per_row + tid; v < n_vec; v += kFusedThreads) xs4[v] = make_uint4(0u, 0u, 0u, 0u);
    mbar_wait(gbar, gpar);
  } else
  for (int v0 = 0; v0 < n_vec; v0 += 8 * kFusedThreads) {
    uint4 val[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const int v = v0 + tid + j * kFusedThreads;
      const int t = v / vec_per_row, c = v - t * vec_per_row;
      val[j] = make_uint4(0u, 0u, 0u, 0u);
      if (v < n_vec && t0 + t < T) val[j] = __ldcg(reinterpret_cast<const uint4*>(a.x + (size_t)(t0 + t) * H + (size_t)c * 8));
    }
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const int v = v0 + tid + j * kFusedThreads;
      if (v < n_vec) xs4[v] = val[j];
    }
  }
  __syncthreads();
  float acc0[TW], acc1[TW];
#pragma unroll
  for (int t = 0; t < TW; ++t) { acc0[t] = 0.f; acc1[t] = 0.f; }
  const uint2* xs2 = reinterpret_cast<const uint2*>(smem_raw) + (size_t)(TW * th) * q_per_row;
  for (int base = 0; base < q_per_row; base += 32 * kDepth) {
    if (base > 0) {
#pragma unroll
      for (int u = 0; u < kDepth; ++u) {
        const int c4 = base + lane + 32 * u;
        wa[u] = (c4 < q_per_row) ? __ldg(wrow0 + c4) : zero4;
        wb[u] = (c4 < q_per_row) ? __ldg(wrow1 + c4) : zero4;
      }
    }
#pragma unroll
    for (int u = 0; u < kDepth; ++u) {
      const int c4 = base + lane + 32 * u;
      if (c4 < q_per_row) {
#pragma unroll
        for (int t = 0; t < TW; ++t) {
          const uint2 xv = xs2[t * q_per_row + c4];
          const float x0 = bf16_lo(xv.x), x1 = bf16_hi(xv.x), x2 = bf16_lo(xv.y), x3 = bf16_hi(xv.y);
          float s0 = acc0[t], s1 = acc1[t];
          s0 = fmaf(wa[u].x, x0, s0); s1 = fmaf(wb[u].x, x0, s1);
          s0 = fmaf(wa[u].y, x1, s0); s1 = fmaf(wb[u].y, x1, s1);
          s0 = fmaf(wa[u].z, x2, s0); s1 = fmaf(wb[u].z, x2, s1);
          s0 = fmaf(wa[u].w, x3, s0); s1 = fmaf(wb[u].w, x3, s1);
          acc0[t] = s0; acc1[t] = s1;
        }
      }
    }
  }
#pragma unroll
  for (int t = 0; t < TW; ++t) {
    float s0 = acc0[t], s1 = acc1[t];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      s0 += __shfl_xor_sync(0xffffffffu, s0, o);
      s1 += __shfl_xor_sync(0xffffffffu, s1, o);
    }
    acc0[t] = s0; acc1[t] = s1;
  }
  if (lane == 0) {
    float* z = const_cast<float*>(a.tk.z);
    const float b0 = (a.gate_bias && e0 < E) ? a.gate_bias[e0] : 0.f;
    const float b1 = (a.gate_bias && e1 < E) ? a.gate_bias[e1] : 0.f;
#pragma unroll
    for (int t = 0; t < TW; ++t) {
      const int tt = t0 + TW * th + t;
      if (tt < T) {
        if (e0 < E) z[(size_t)tt * E + e0] = acc0[t] + b0;
        if (e1 < E) z[(size_t)tt * E + e1] = acc1[t] + b1;
      }
    }
  }
}

// Shared-memory gate tile (every tile that fits the ring area: all of T > 64, and 8-token tiles up to H ~ 4300): the x
// tile AND the tile's eight gate rows are brought into shared memory by two bulk copies, and a warp owns 4 experts x
// GT/4 tokens (the register-staged tile below: 2 x GT/2 with the gate rows in registers).  Measured at T = 64: every
// config-2 point 1.2-1.5 us faster (one L2 round trip for everything instead of rows -> x -> second half of the rows).
// Every converted x value now feeds four FMAs instead of two (the bf16 -> fp32 conversions run on the ALU pipe at half
// the FMA rate and were half of the tile's issue time at GT = 32), and no gate-row load sits between two halves of the
// K loop.  The per-lane summation order (column = lane + 32 j, ascending) is the narrow tile's: same logits, bit for bit.
template <int GT>
__device__ __forceinline__ void fused_gate_tile_wide(const FusedArgs& a, int et, int g, uint8_t* smem_raw, uint32_t gbar,
                                                     uint32_t gpar) {
  constexpr int TW = GT / 4;              // tokens per warp
  const int T = a.tk.T, H = a.H, E = a.tk.E;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int t0 = g * GT;
  const int eq = warp & 1, tg = warp >> 1;
  const int e0 = et * kGateExp;
  const int q_per_row = H >> 2;
  const int rows = min(GT, T - t0), n_e = min(kGateExp, E - e0);
  uint8_t* w_smem = smem_raw + (size_t)GT * H * 2;
  __syncthreads();                       // the previous tile's readers are done with the tile
  if (tid == 0) {
    const uint32_t xb = (uint32_t)rows * (uint32_t)H * 2u, wb = (uint32_t)n_e * (uint32_t)H * 4u;
    mbar_arrive_expect_tx(gbar, xb + wb);
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(smem_u32(smem_raw)), "l"(a.x + (size_t)t0 * H), "r"(xb), "r"(gbar) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(smem_u32(w_smem)), "l"(a.gate_w + (size_t)e0 * H), "r"(wb), "r"(gbar) : "memory");
  }
  {
    uint4* xs4 = reinterpret_cast<uint4*>(smem_raw);
    const int vec_per_row = H >> 3;
    for (int v = rows * vec_per_row + tid; v < GT * vec_per_row; v += kFusedThreads) xs4[v] = make_uint4(0u, 0u, 0u, 0u);
    uint4* ws4 = reinterpret_cast<uint4*>(w_smem);
    for (int v = n_e * q_per_row + tid; v < kGateExp * q_per_row; v += kFusedThreads) ws4[v] = make_uint4(0u, 0u, 0u, 0u);
  }
  mbar_wait(gbar, gpar);
  __syncthreads();
  float acc[4][TW];
#pragma unroll
  for (int e = 0; e < 4; ++e)
#pragma unroll
    for (int t = 0; t < TW; ++t) acc[e][t] = 0.f;
  const float4* wv = reinterpret_cast<const float4*>(w_smem) + (size_t)(4 * eq) * q_per_row;
  const uint2* xs2 = reinterpret_cast<const uint2*>(smem_raw) + (size_t)(TW * tg) * q_per_row;
  for (int c4 = lane; c4 < q_per_row; c4 += 32) {
    float4 w4[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) w4[e] = wv[(size_t)e * q_per_row + c4];
#pragma unroll
    for (int t = 0; t < TW; ++t) {
      const uint2 xv = xs2[t * q_per_row + c4];
      const float x0 = bf16_lo(xv.x), x1 = bf16_hi(xv.x), x2 = bf16_lo(xv.y), x3 = bf16_hi(xv.y);
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        float s = acc[e][t];
        s = fmaf(w4[e].x, x0, s);
        s = fmaf(w4[e].y, x1, s);
        s = fmaf(w4[e].z, x2, s);
        s = fmaf(w4[e].w, x3, s);
        acc[e][t] = s;
      }
    }
  }
#pragma unroll
  for (int e = 0; e < 4; ++e)
#pragma unroll
    for (int t = 0; t < TW; ++t) {
      float s = acc[e][t];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
      acc[e][t] = s;
    }
  if (lane == 0) {
    float* z = const_cast<float*>(a.tk.z);
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const int ee = e0 + 4 * eq + e;
      if (ee < E) {
        const float b = a.gate_bias ? a.gate_bias[ee] : 0.f;
#pragma unroll
        for (int t = 0; t < TW; ++t) {
          const int tt = t0 + TW * tg + t;
          if (tt < T) z[(size_t)tt * E + ee] = acc[e][t] + b;
        }
      }
    }
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
  if (!renorm) {
    uint32_t m = key[0];
#pragma unroll
    for (int i = 1; i < NV; ++i) m = max(m, key[i]);
    const float zmax = f32_from_order_key(__reduce_max_sync(0xffffffffu, m));
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
  uint32_t stage_base;     // stage_area bytes cut into S stages of [16 KiB weights | np*128 B activations]
  uint32_t bar_base;       // full[kMaxStages], empty[kMaxStages], tfull[2], tempty[2], cfull[4], cempty[4]
  uint32_t tmem_slot;
  volatile int32_t* claim; // [kClaimSlots] claimed data-parallel tile ids (-1 = part finished)
  int4* work;              // [E+ns] {expert, x_row0, out_row0, m}
  int32_t* cumpass;        // [E+ns+1] exclusive scan of accumulator passes per work entry
  int32_t* meta;           // [8] {n_work, np, S, total passes}
  uint16_t* tok_of_pos;    // [T*k (+T)]
  uint16_t* pos_of_pair;   // [T*k]
  uint8_t* ids8;           // [T*k] expert id of each pair (E <= 256)
  uint8_t* route_scratch;  // mask [E][W], pref [E][W], ent [E], off [E+1], scan totals [32] (part a -> part b, combine)
};

// Bytes of everything except the stage ring (barriers, routing tables); the host gives the ring what is left.
__host__ __device__ inline size_t fused_smem_fixed_bytes(int E, int ns, int T, int k) {
  const size_t W = (T + 31) / 32;
  size_t o = 512;                                        // barriers + claim ring + tmem slot
  o += (size_t)(E + ns) * 16;
  o += ((size_t)(E + ns + 1) * 4 + 15) / 16 * 16;
  o += 32;
  o += (((size_t)T * k + T) * 2 + 15) / 16 * 16;
  o += ((size_t)T * k * 2 + 15) / 16 * 16;
  o += ((size_t)T * k + 15) / 16 * 16;
  o += ((size_t)E * W * 8 + (size_t)(2 * E + 1 + 32) * 4 + 15) / 16 * 16;   // route scratch: mask, pref, ent, off, scan totals
  return o + 1024;                                       // alignment slack
}

// ------------------------------------------------------------------------------ R (part a): union + work list
// Scratch (mask, pref, s_ent, s_off, s_blk) has its own shared-memory region: part b still reads it while the weights
// producer is already filling the stage ring.  All 256 threads take part: thread e owns expert e (E <= 256) -- its
// count from the membership words, then one block-wide scan (warp shuffles + eight warp totals) gives the offsets
// and, through a ballot, the slot of every active expert in the union-compacted work list.  (The one-warp scan of
// round 1 cost 2.5 us of the serial prelude.)
__device__ __forceinline__ void fused_route_a(const FusedArgs& a, const FusedSmem& sm, uint8_t* scratch, bool is_cta0) {
  const int T = a.tk.T, E = a.tk.E, k = a.tk.k, ns = a.n_shared;
  const int W = (T + 31) >> 5;
  uint32_t* mask = reinterpret_cast<uint32_t*>(scratch);     // [E][W]
  uint32_t* pref = mask + (size_t)E * W;                      // [E][W]
  int32_t* s_ent = reinterpret_cast<int32_t*>(pref + (size_t)E * W);   // [E] work-list entry of expert e (-1: inactive)
  int32_t* s_off = s_ent + E;                                 // [E+1]
  int32_t* s_blk = s_off + E + 1;                             // [32] warp totals of the block scans
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const bool do_sig = is_cta0 && a.force_routing;

  // (the membership masks were zeroed in the kernel's prologue, before the gate)
  if (a.force_routing) {
    // ids were given: bring them into the shared-memory table the tagged-ids poll would have filled
    for (int p = tid; p < T * k; p += kFusedThreads) {
      const int id = min(max(__ldcg(a.tk.ids + p), 0), E - 1);
      sm.ids8[p] = (uint8_t)id;
      if (do_sig) {
        const int t = p / k;
        sig_add(a.tk.sig_req, a.tk.sig_block, a.tk.token_req ? a.tk.token_req[t] : -1,
                a.tk.token_block ? a.tk.token_block[t] : -1, a.tk.L, a.tk.layer, E, id);
      }
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) FSTAMP2(4);
  for (int p = tid; p < T * k; p += kFusedThreads) {
    const int t = p / k;
    atomicOr(&mask[(int)sm.ids8[p] * W + (t >> 5)], 1u << (t & 31));
  }
  __syncthreads();
  if (threadIdx.x == 0) FSTAMP2(5);
  // thread e: count of expert e and the per-word prefixes the position maps need
  int c = 0;
  if (tid < E) {
    for (int w = 0; w < W; ++w) {
      pref[tid * W + w] = c;
      c += __popc(mask[tid * W + w]);
    }
  }
  const uint32_t act_ballot = __ballot_sync(0xffffffffu, c > 0);
  int cinc = c;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int cv = __shfl_up_sync(0xffffffffu, cinc, o);
    if (lane >= o) cinc += cv;
  }
  const int wmax = (int)__reduce_max_sync(0xffffffffu, (unsigned)c);
  if (lane == 31) { s_blk[warp] = cinc; s_blk[8 + warp] = __popc(act_ballot); s_blk[16 + warp] = wmax; }
  __syncthreads();
  if (threadIdx.x == 0) FSTAMP2(6);
  int cbase = 0, abase = 0, total = 0, n_act = 0, cmax = 0;
#pragma unroll
  for (int w = 0; w < kFusedThreads / 32; ++w) {
    const int cw = s_blk[w], aw = s_blk[8 + w];
    if (w < warp) { cbase += cw; abase += aw; }
    total += cw; n_act += aw;
    cmax = max(cmax, s_blk[16 + w]);
  }
  if (ns) cmax = T;
  const int n_work = n_act + ns;
  if (tid < E) {
    const int coff = cbase + cinc - c;
    const int aoff = abase + __popc(act_ballot & ((1u << lane) - 1u));
    s_off[tid] = coff;
    // Work-list order: the SHARED experts first, then the active routed experts in id order.  The shared experts
    // take every token, so their tiles are the widest (128 columns per pass) and every token's combine needs them:
    // first in the list they are whole tiles of the first rounds -- never split between SMs, h and y ready early --
    // and the tail of each phase is the narrow routed experts, whose fix-ups and epilogues are cheap.  (Shared last:
    // config-5 shape, T = 256: the last 35 us of the step were 128-column fix-ups and a combine that could not start.)
    s_ent[tid] = c > 0 ? aoff + ns : -1;
    if (is_cta0) { a.off[tid] = coff; a.cnt[tid] = c; }
    if (c > 0) {
      const int4 wk = make_int4(tid, coff, coff, c);
      sm.work[aoff + ns] = wk;
      if (is_cta0) { a.active[aoff] = tid; a.work[aoff + ns] = wk; }
    }
    if (is_cta0 && tid >= n_act) a.active[tid] = -1;
  }
  if (tid < ns) {
    const int4 wk = make_int4(E + tid, T * k, T * k + tid * T, T);
    sm.work[tid] = wk;
    if (is_cta0) a.work[tid] = wk;
  }
  if (tid == 0) {
    const int np = (min(cmax, kNPCap) + 15) & ~15;
    s_off[E] = total;
    sm.meta[0] = n_work;
    sm.meta[1] = np;
    sm.meta[2] = min(kMaxStages, max(min(a.stage_area, a.ring_bytes), 3 * (kUmmaWBytes + np * 128)) / (kUmmaWBytes + np * 128));
    if (is_cta0) { a.off[E] = total; *a.n_active = n_act; *a.n_work = n_work; }
  }
  // accumulator passes per entry (1 unless an expert got more than kNPCap tokens) and their exclusive scan
  if (cmax <= kNPCap) {
    // every entry fits one accumulator pass (the usual decode case): the pass table is the identity
    for (int ent = tid; ent <= n_work; ent += kFusedThreads) sm.cumpass[ent] = ent;
    if (tid == 0) sm.meta[3] = n_work;
    __syncthreads();
  } else {
    __syncthreads();                                 // the work list is complete
    // entries <= E + ns <= 264: thread `tid` takes entry tid, thread 0..7 also entry 256 + tid; two-level scan again
    const int ps0 = tid < n_work ? (sm.work[tid].w + kNPCap - 1) / kNPCap : 0;
    int pinc = ps0;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int pv = __shfl_up_sync(0xffffffffu, pinc, o);
      if (lane >= o) pinc += pv;
    }
    if (lane == 31) s_blk[24 + warp] = pinc;
    __syncthreads();
    int pbase = 0, ptot = 0;
#pragma unroll
    for (int w = 0; w < kFusedThreads / 32; ++w) {
      const int pw_ = s_blk[24 + w];
      if (w < warp) pbase += pw_;
      ptot += pw_;
    }
    if (tid < n_work) sm.cumpass[tid] = pbase + pinc - ps0;
    if (tid == 0) {
      int run = ptot;
      for (int ent = kFusedThreads; ent < n_work; ++ent) {          // at most ns = 8 entries past the block
        sm.cumpass[ent] = run;
        run += (sm.work[ent].w + kNPCap - 1) / kNPCap;
      }
      sm.cumpass[n_work] = run;
      sm.meta[3] = run;
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) FSTAMP2(7);
}

// ---------------------------------------------------------------------- R (part b): token <-> position maps
__device__ __forceinline__ void fused_route_b(const FusedArgs& a, const FusedSmem& sm, uint8_t* scratch, bool is_cta0,
                                              int tid, int nthr) {
  const int T = a.tk.T, E = a.tk.E, k = a.tk.k, ns = a.n_shared;
  const int W = (T + 31) >> 5;
  const uint32_t* mask = reinterpret_cast<const uint32_t*>(scratch);
  const uint32_t* pref = mask + (size_t)E * W;
  const int32_t* s_off = reinterpret_cast<const int32_t*>(pref + (size_t)E * W) + E;
  for (int p = tid; p < T * k; p += nthr) {
    const int t = p / k;
    const int e = sm.ids8[p];
    const int rank = pref[e * W + (t >> 5)] + __popc(mask[e * W + (t >> 5)] & ((1u << (t & 31)) - 1u));
    const int pos = s_off[e] + rank;
    sm.tok_of_pos[pos] = (uint16_t)t;
    sm.pos_of_pair[p] = (uint16_t)pos;
    if (is_cta0) { a.perm[pos] = p; a.pair_pos[p] = pos; }
  }
  if (ns)
    for (int t = tid; t < T; t += nthr) sm.tok_of_pos[T * k + t] = (uint16_t)t;
}

// -------------------------------------------------------------------------------- F: stream-K piece walker
// Phase ph (0: w1/w3, 1: w2): tiles = (work entry, pass, row tile), flattened entry-major; each tile has `kit`
// k-chunks (stages).  CTA c owns stages [c*P/G, (c+1)*P/G).  A piece = the part of one tile inside that range.
struct Piece {
  int tile, k0, k1, ent, pass, rt;
};
// Schedule, decided PER PHASE from its tile count n (tile list entry-major, so experts come in order), R0 = the
// largest multiple of gridDim.x <= n:
//   n >= min_rounds * G (default: at least one whole round):
//     part 0 ("data-parallel"): tiles [0, R0) whole -- the first one of CTA c is tile c, the following ones are drawn
//             from the phase's counter -- no split, no fix-up, and experts FINISH IN ORDER over the phase;
//     part 1 (remainder): tiles [R0, n) cut over at most max_split CTAs per tile (default 1: whole tiles on n - R0
//             CTAs); the other CTAs go straight on to the next phase / the combine.  Measured: every further piece of
//             a tile costs more (park, publish, the finisher's serial adds) than the idle SMs of a partial round --
//             |U| = 128: 205.8 us with the remainder cut over the whole grid, 197.4 with whole tiles.
//   n < min_rounds * G: the whole phase is one static stream-K cut (equal contiguous stage ranges over the grid).
// Sub-phase order A0 A1 B0 B1: B0 starts on the first experts, whose h tiles were all produced in A0 (several
// microseconds earlier), so the w1/w3 -> w2 hand-over costs no pipeline drain; B1 needs the last experts, finished
// a whole B0 earlier.
struct PieceWalker {
  int tpe, kit;          // row tiles per (entry, pass); k-chunks per tile
  long long g, hi, P;    // remainder part: current / end stage of this CTA, total stages
  long long hi_walk;     // end of the ascending walk (the head piece, emitted first, is cut off)
  bool head_first, head_pending;
  int ent;               // cursor into cumpass
  const int32_t* cumpass;
  int tile0;             // remainder part: first tile (R0)
  int dp_tile, dp_end, G;
  int Gs;                // CTAs that share the static (stream-K) part: 0 .. Gs-1, the others skip it
  bool dp;
  __device__ __forceinline__ void init(int sp, int tilesA, int tilesB, int kitA, int kitB, int total_pass,
                                       const int32_t* cp, int cta, int G_, int min_rounds, int split_pct, bool head_first_, int max_split) {
    const int ph = sp >> 1;
    head_first = head_first_;
    tpe = ph == 0 ? tilesA : tilesB;
    kit = ph == 0 ? kitA : kitB;
    G = G_;
    Gs = G_;
    const int n_tiles = total_pass * tpe;
    ent = 0;
    cumpass = cp;
    dp_tile = cta;
    if (n_tiles / G >= min_rounds) {
      // a phase with at least min_rounds whole rounds of tiles (decided per phase): whole rounds, then the remainder
      const int R0 = (n_tiles / G) * G;
      dp = (sp & 1) == 0;
      dp_end = R0;
      tile0 = R0;
      P = (long long)(n_tiles - R0) * kit;
      // a remainder of few tiles is not cut over the whole grid: every further piece of a tile is one more parked
      // partial the tile's finisher adds in series (config-5 shape: 16 tiles over 148 CTAs = nine pieces per tile, the
      // finishers 25 us behind); at most max_split pieces per tile, the other CTAs go straight on to the next part
      if (max_split > 0 && R0 > 0) Gs = min(G, max(1, (n_tiles - R0) * max_split));
    } else {
      // small union (phase A shorter than min_rounds rounds of tiles): the accumulator passes -- experts, in order --
      // are cut into two groups and the sub-phases run A(g0) A(g1) B(g0) B(g1), each a static stream-K cut of its own
      // stage sequence.  B(g0) starts on h tiles that were finished a whole A(g1) earlier and B(g1) on tiles finished a
      // whole B(g0) earlier, so the w1/w3 -> w2 hand-over no longer drains the pipeline (with one stream-K cut per
      // phase every expert had an h tile finished in the last microsecond of A: the activation producers idled a
      // median 8 us at |U| = 16).  The decision needs n_active, so it is taken here, in the kernel.
      const int p_split = min(total_pass, (total_pass * split_pct + 50) / 100);
      const int t_lo = (sp & 1) ? p_split * tpe : 0, t_hi = (sp & 1) ? n_tiles : p_split * tpe;
      dp = false;
      dp_end = 0;
      tile0 = t_lo;
      P = (long long)(t_hi - t_lo) * kit;
    }
    g = cta < Gs ? P * cta / Gs : 0;
    hi = cta < Gs ? P * (cta + 1) / Gs : 0;
    hi_walk = hi;
    head_pending = head_first && !dp;
  }
  // data-parallel part: `claimed` is the tile this CTA drew from the phase's counter (ascending per CTA), or
  // anything >= dp_end / negative when the part is exhausted.  Remainder part: `claimed` is ignored.
  __device__ __forceinline__ bool next(Piece& p, int claimed) {
    if (dp) {
      if (claimed < 0 || claimed >= dp_end) return false;
      p.tile = claimed;
      p.k0 = 0;
      p.k1 = kit;
    } else {
      // Static range [g, hi) of the stage sequence, ascending by default.  Optional piece order (head_first,
      // ELDR_OPT_HEAD_FIRST): the HEAD of the tile the range ends in comes first and is parked at once; then the tail of
      // the tile the range starts in -- finished here with the previous CTA's parked head -- then the whole tiles, so
      // that no range ends on a fix-up.  (Per-CTA traces show the CTAs whose range ends in a short head piece raising
      // their last h flags ~6 us after the others; but with the fix-ups moved to the start of the sub-phase the step
      // got 5 us SLOWER at |U| = 16 / 32 -- kept as a parity-tested option, off by default.)
      if (head_pending) {
        head_pending = false;
        if (g < hi) {
          const long long t_last = (hi - 1) / kit;
          if (hi % kit != 0 && t_last != g / kit) {
            p.tile = tile0 + (int)t_last;
            p.k0 = 0;
            p.k1 = (int)(hi - t_last * kit);
            hi_walk = t_last * kit;
            ent = 0;
            const int cpi_h = p.tile / tpe;
            p.rt = p.tile - cpi_h * tpe;
            int e2 = 0;
            while (cumpass[e2 + 1] <= cpi_h) ++e2;
            p.ent = e2;
            p.pass = cpi_h - cumpass[e2];
            return true;
          }
        }
      }
      if (g >= hi_walk) return false;
      const int lt = (int)(g / kit);                 // tile index inside the remainder
      p.tile = tile0 + lt;
      p.k0 = (int)(g - (long long)lt * kit);
      p.k1 = (int)min((long long)kit, p.k0 + (hi_walk - g));
      g += p.k1 - p.k0;
    }
    const int cpi = p.tile / tpe;
    p.rt = p.tile - cpi * tpe;
    while (cumpass[ent + 1] <= cpi) ++ent;
    p.ent = ent;
    p.pass = cpi - cumpass[ent];
    return true;
  }
};

// ------------------------------------------------------------------------------ C: flag-driven combine
template <int KMAX>
__device__ __forceinline__ void fused_combine(const FusedArgs& a, const FusedSmem& sm, const uint32_t* ydone, uint32_t epoch,
                                              int n_work, int tilesB, int cta, int G, int warp, int lane) {
  const int T = a.tk.T, E = a.tk.E, k = a.tk.k, H = a.H, ns = a.n_shared;
  {
    const int32_t* s_ent = reinterpret_cast<const int32_t*>(sm.route_scratch + (size_t)E * ((T + 31) >> 5) * 8);
    const int q_per_row = H >> 2;
    const int n_units = T * tilesB;
    // Two units per iteration: both units' flag polls, then both units' k row loads, are in flight together (one
    // unit at a time cost a poll + fence + load round trip each: 13 us of combine at T = 256).
    const int u_step = G * (kFusedThreads / 32);
    for (int u0 = cta * (kFusedThreads / 32) + warp; u0 < n_units; u0 += 2 * u_step) {
      int t_[2], rt_[2], pos_[2], fl_[2];
      float wt_[2];
      const unsigned long long* wsrc_[2];
      bool have_[2];
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        const int u = u0 + q * u_step;
        have_[q] = u < n_units;
        const int uu = have_[q] ? u : u0;
        const int t = uu / tilesB, rt = uu - t * tilesB;
        t_[q] = t; rt_[q] = rt; pos_[q] = 0; fl_[q] = -1; wt_[q] = 0.f; wsrc_[q] = nullptr;
        if (have_[q]) {
          if (lane < k) {
            const int ent = s_ent[sm.ids8[t * k + lane]];
            pos_[q] = sm.pos_of_pair[t * k + lane];
            fl_[q] = (sm.cumpass[ent] + (pos_[q] - sm.work[ent].y) / kNPCap) * tilesB + rt;
            if (a.force_routing) wt_[q] = __ldcg(a.tk.w + t * k + lane);
            else wsrc_[q] = a.wtag + (size_t)t * kMaxTopK + lane;
          } else if (lane < k + ns) {
            const int ent = lane - k;                       // shared experts lead the work list
            pos_[q] = T * k + (lane - k) * T + t;
            fl_[q] = (sm.cumpass[ent] + t / kNPCap) * tilesB + rt;
            wt_[q] = 1.0f;
          }
        }
      }
      bool f_ok[2] = {fl_[0] < 0, fl_[1] < 0}, w_ok[2] = {wsrc_[0] == nullptr, wsrc_[1] == nullptr};
      for (uint32_t spins = 0;; ++spins) {
        uint32_t fv[2] = {0u, 0u};
        unsigned long long wv[2] = {0ull, 0ull};
#pragma unroll
        for (int q = 0; q < 2; ++q) {
          if (!f_ok[q]) fv[q] = flag_relaxed(ydone + fl_[q]);
          if (!w_ok[q]) wv[q] = ld_relaxed_u64(wsrc_[q]);       // written by the top-k owner in the prelude: up on the first look
        }
#pragma unroll
        for (int q = 0; q < 2; ++q) {
          if (!f_ok[q]) f_ok[q] = fv[q] == epoch;
          if (!w_ok[q] && (uint32_t)(wv[q] >> 32) == epoch) { w_ok[q] = true; wt_[q] = __uint_as_float((uint32_t)wv[q]); }
        }
        if (__all_sync(0xffffffffu, f_ok[0] && f_ok[1] && w_ok[0] && w_ok[1])) break;
        __nanosleep(250);
        if (spins > (1u << 22)) __trap();
      }
      fence_acq_rel_gpu();
      __syncwarp();
      float4 v[2][KMAX];
      float wj[2][KMAX];
      bool in_[2];
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        const int c4 = rt_[q] * 32 + lane;
        in_[q] = have_[q] && c4 < q_per_row;
#pragma unroll
        for (int j = 0; j < KMAX; ++j)
          if (j < k) {
            const int pj = __shfl_sync(0xffffffffu, pos_[q], j);
            wj[q][j] = __shfl_sync(0xffffffffu, wt_[q], j);
            if (in_[q]) v[q][j] = __ldcg(reinterpret_cast<const float4*>(a.ybuf + (size_t)pj * H + (size_t)c4 * 4));
          }
      }
#pragma unroll
      for (int q = 0; q < 2; ++q) {
        const int c4 = rt_[q] * 32 + lane;
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        if (in_[q]) {
#pragma unroll
          for (int j = 0; j < KMAX; ++j)
            if (j < k) {
              acc.x = fmaf(wj[q][j], v[q][j].x, acc.x); acc.y = fmaf(wj[q][j], v[q][j].y, acc.y);
              acc.z = fmaf(wj[q][j], v[q][j].z, acc.z); acc.w = fmaf(wj[q][j], v[q][j].w, acc.w);
            }
        }
        for (int s_ = 0; s_ < ns; ++s_) {
          const int ps = __shfl_sync(0xffffffffu, pos_[q], k + s_);
          if (in_[q]) {
            const float4 sv = __ldcg(reinterpret_cast<const float4*>(a.ybuf + (size_t)ps * H + (size_t)c4 * 4));
            acc.x += sv.x; acc.y += sv.y; acc.z += sv.z; acc.w += sv.w;
          }
        }
        if (in_[q]) {
          uint2 o;
          o.x = (uint32_t)f32_to_bf16_rn(acc.x) | ((uint32_t)f32_to_bf16_rn(acc.y) << 16);
          o.y = (uint32_t)f32_to_bf16_rn(acc.z) | ((uint32_t)f32_to_bf16_rn(acc.w) << 16);
          *reinterpret_cast<uint2*>(a.out + (size_t)t_[q] * H + (size_t)c4 * 4) = o;
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------------------- the kernel
// GT: tokens per gate tile (8 / 16 / 32 for T <= 64 / 128 / 256).  GW: the gate tile staged in shared memory (always for
// GT > 8; for GT = 8 whenever it fits the ring area, else the register-staged tile).  Template parameters, not run-time
// branches: with both tile kinds inlined into one kernel every config-2 point lost the microsecond the new tile gains.
template <int GT, bool GW = true>
__global__ void __launch_bounds__(kFusedThreads, 1)
moe_fused_kernel(const __grid_constant__ CUtensorMap tm_w13, const __grid_constant__ CUtensorMap tm_sw13,
                 const __grid_constant__ CUtensorMap tm_w2, const __grid_constant__ CUtensorMap tm_sw2,
                 const __grid_constant__ CUtensorMap tm_x, const __grid_constant__ CUtensorMap tm_xs,
                 const __grid_constant__ CUtensorMap tm_h, const FusedArgs a) {
  extern __shared__ uint8_t smem_dyn[];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int G = gridDim.x, cta = blockIdx.x;
  const int T = a.tk.T, E = a.tk.E, k = a.tk.k, H = a.H, I = a.I, ns = a.n_shared;

  FusedSmem sm;
  {
    const uint32_t base = (smem_u32(smem_dyn) + 1023u) & ~1023u;
    uint8_t* gen = smem_dyn + (base - smem_u32(smem_dyn));
    sm.stage_base = base;
    size_t o = (size_t)a.stage_area;
    sm.bar_base = base + (uint32_t)o;
    sm.tmem_slot = base + (uint32_t)o + 496;
    sm.claim = reinterpret_cast<volatile int32_t*>(gen + o + 320);
    o += 512;
    sm.work = reinterpret_cast<int4*>(gen + o);
    o += (size_t)(E + ns) * 16;
    sm.cumpass = reinterpret_cast<int32_t*>(gen + o);
    o += ((size_t)(E + ns + 1) * 4 + 15) / 16 * 16;
    sm.meta = reinterpret_cast<int32_t*>(gen + o);
    o += 32;
    sm.tok_of_pos = reinterpret_cast<uint16_t*>(gen + o);
    o += (((size_t)T * k + T) * 2 + 15) / 16 * 16;
    sm.pos_of_pair = reinterpret_cast<uint16_t*>(gen + o);
    o += ((size_t)T * k * 2 + 15) / 16 * 16;
    sm.ids8 = gen + o;
    o += ((size_t)T * k + 15) / 16 * 16;
    sm.route_scratch = gen + o;
  }
  uint8_t* scratch = smem_dyn + (sm.stage_base - smem_u32(smem_dyn));     // stage area, generic pointer
  auto full_bar = [&](int s) { return sm.bar_base + 8u * s; };
  auto empty_bar = [&](int s) { return sm.bar_base + 8u * (kMaxStages + s); };
  auto tfull_bar = [&](int b) { return sm.bar_base + 8u * (2 * kMaxStages + b); };
  auto tempty_bar = [&](int b) { return sm.bar_base + 8u * (2 * kMaxStages + 2 + b); };
  auto cfull_bar = [&](int b) { return sm.bar_base + 8u * (2 * kMaxStages + 4 + b); };
  auto cempty_bar = [&](int b) { return sm.bar_base + 8u * (2 * kMaxStages + 4 + kClaimSlots + b); };

  // ------------------------------------------------------------- prologue (overlaps the previous kernel's tail)
  if (tid == 0) FSTAMP2(8);
  if (tid == 0) {
    for (int s = 0; s < kMaxStages; ++s) { mbar_init(full_bar(s), 2); mbar_init(empty_bar(s), 1); }
    for (int b = 0; b < 2; ++b) { mbar_init(tfull_bar(b), 1); mbar_init(tempty_bar(b), 4); }
    for (int b = 0; b < kClaimSlots; ++b) { mbar_init(cfull_bar(b), 1); mbar_init(cempty_bar(b), 7); }
    mbar_init(sm.bar_base + 400u, 1);                 // x tile of the wide gate tiles (bulk copy)
    mbar_fence_init();
    tma_prefetch_desc(&tm_w13);
    tma_prefetch_desc(&tm_w2);
    tma_prefetch_desc(&tm_x);
    tma_prefetch_desc(&tm_xs);
    tma_prefetch_desc(&tm_h);
  }
  constexpr uint32_t tmem_cols = 2 * kNPCap;
  if (warp == 6) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(sm.tmem_slot), "r"(tmem_cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(sm.tmem_slot));
  {
    // routing membership masks [E][W]: zeroed here, long before the ids arrive (ordered by the barriers in between)
    uint32_t* mask0 = reinterpret_cast<uint32_t*>(sm.route_scratch);
    for (int i = tid; i < E * ((T + 31) >> 5); i += kFusedThreads) mask0[i] = 0u;
  }
  if (tid == 0) FSTAMP(0);
  pdl_launch_dependents();
  pdl_wait();
  if (tid == 0) FSTAMP(1);

  const uint32_t gen_next = epoch_next_state(__ldcg(a.sync + kSyncGen));
  const uint32_t epoch = epoch_of_state(gen_next, a.sync);
  if (cta == 0 && tid == 0) {
    // this step's tile counters (the previous grid has completed: pdl_wait above)
    a.sync[kSyncTileCnt] = 0u;
    a.sync[kSyncTileCnt + 1] = 0u;
    a.sync[kSyncExit] = 0u;
    flag_release(a.sync + kSyncCntReady, epoch);
  }

  // ------------------------------------------------------------------------------ G + K: gate and top-k
  SigPending sig_pend{nullptr, 0u, 0u};     // this lane's signature increment of the step, saturation check deferred to the end
  if (!a.force_routing) {
    const int n_et = (E + kGateExp - 1) / kGateExp, n_gr = (T + kGateTok - 1) / kGateTok;
    const int n_tiles = n_et * ((T + GT - 1) / GT);
    uint32_t gpar = 0;
    for (int tile = cta; tile < n_tiles; tile += G, gpar ^= 1u) {
      const int g = tile / n_et, et = tile - g * n_et;
      // (the register-staged tile only where the shared-memory one does not fit: 8-token tiles at H > ~4300)
      if constexpr (GT > 8 || GW) fused_gate_tile_wide<GT>(a, et, g, scratch, sm.bar_base + 400u, gpar);
      else fused_gate_tile<GT>(a, et, g, scratch, sm.bar_base + 400u, gpar);
      __syncthreads();
      if (tid == 0) flag_release(a.sync + kSyncTile + g * 32 + et, epoch);    // cumulative over the barrier
    }
    if (tid == 0) FSTAMP2(12);
    // owner of token group g: waits for the group's logit tiles, warp w runs the top-k of token 8g + w and writes the
    // ABI outputs, the signature increments and the tagged ids words every CTA routes from
    for (int g = ((cta - n_tiles % G) + G) % G; g < n_gr; g += G) {     // owner(g) = (n_tiles + g) % G: CTAs without a gate tile first
      if (warp == 0) warp_wait_flags(a.sync + kSyncTile + (g * kGateTok / GT) * 32, n_et, epoch, lane);
      __syncthreads();
      const int t = g * kGateTok + warp;
      if (t < T) {
        int id; float w;
        warp_topk_redux(a.tk.z + (size_t)t * E, E, k, a.tk.renorm, lane, id, w);
        const uint32_t b = lane < k ? (uint32_t)id : 0u;
        const uint32_t packed = b | (__shfl_down_sync(0xffffffffu, b, 1) << 8) | (__shfl_down_sync(0xffffffffu, b, 2) << 16) |
                                (__shfl_down_sync(0xffffffffu, b, 3) << 24);
        if ((lane & 3) == 0 && lane < k)
          st_relaxed_u64(a.idt + (size_t)t * kIdWordsPerTok + (lane >> 2), ((unsigned long long)epoch << 32) | packed);
        if (lane < k) {
          a.tk.ids[(size_t)t * k + lane] = id;
          a.tk.w[(size_t)t * k + lane] = w;
          st_relaxed_u64(a.wtag + (size_t)t * kMaxTopK + lane, ((unsigned long long)epoch << 32) | __float_as_uint(w));
          sig_add_finish(sig_pend);          // (a second group of this owner: T <= 256 never has one)
          sig_pend = sig_add_begin(a.tk.sig_req, a.tk.sig_block, a.tk.token_req ? a.tk.token_req[t] : -1,
                                   a.tk.token_block ? a.tk.token_block[t] : -1, a.tk.L, a.tk.layer, E, id);
        }
      }
    }
    if (tid == 0) FSTAMP2(13);
    // every CTA: poll the tagged ids of all tokens into the shared-memory id table
    {
      const int wpt = (k + 3) >> 2;
      const int n_words = T * wpt;
      for (int i = tid; i < n_words; i += kFusedThreads) {
        const int t = i / wpt, q = i - t * wpt;
        const unsigned long long* src = a.idt + (size_t)t * kIdWordsPerTok + q;
        unsigned long long v = ld_relaxed_u64(src);
        uint32_t spins = 0;
        while ((uint32_t)(v >> 32) != epoch) {
          __nanosleep(40);
          v = ld_relaxed_u64(src);
          if (++spins > (1u << 24)) __trap();
        }
#pragma unroll
        for (int j = 0; j < 4; ++j)
          if (4 * q + j < k) sm.ids8[t * k + 4 * q + j] = (uint8_t)min((int)((v >> (8 * j)) & 0xffu), E - 1);
      }
    }
    __syncthreads();
    if (tid == 0) FSTAMP2(14);
  }

  // ------------------------------------------------------------------------------------------ R: routing
  fused_route_a(a, sm, sm.route_scratch, cta == 0);
  if (tid == 0) FSTAMP2(15);
  if (warp != 4) {
    // the weights producer (warp 4) is already streaming; everyone else finishes the position maps
    fused_route_b(a, sm, sm.route_scratch, cta == 0, warp < 4 ? tid : tid - 32, kFusedThreads - 32);
    asm volatile("bar.sync 2, 224;" ::: "memory");
  }

  // ------------------------------------------------------------------------------------------ F: expert FFN
  const int n_work = sm.meta[0];
  const int NP = sm.meta[1], S = sm.meta[2], total_pass = sm.meta[3];
  // Wide batches (some expert has xs_min_np token columns or more): phase A reads its activations from an
  // expert-sorted copy of x, sixteen rows per TMA instruction, instead of gathering the token rows four per
  // instruction from x for every stage -- at 64-128 tokens per expert the gather instructions, not the bytes, bound
  // phase A (measured: T = 256, |U| = 32: 110.6 -> 99.0 us with plain boxes).  CTA c copies rows c, c + G, ... (one
  // warp per 4-KiB row) while its weights producer fills the ring, then raises its flag; the activation producers
  // wait for all G flags once.  Narrow batches keep the gather: few instructions per stage and no extra hand-over.
  const bool use_xs = NP >= a.xs_min_np;
  if (use_xs && warp != 4) {
    const int n_rows = T * k + (ns ? T : 0);
    const int w7 = warp < 4 ? warp : warp - 1;
    const int vec = H >> 3;                                     // 16-byte chunks per row
    for (int pos = cta + G * w7; pos < n_rows; pos += G * 7) {
      const uint4* src = reinterpret_cast<const uint4*>(a.x + (size_t)sm.tok_of_pos[pos] * H);
      uint4* dst = reinterpret_cast<uint4*>(a.xs + (size_t)pos * H);
      for (int c0 = lane; c0 < vec; c0 += 256) {
        uint4 v[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) v[j] = (c0 + 32 * j < vec) ? __ldcg(src + c0 + 32 * j) : make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
        for (int j = 0; j < 8; ++j)
          if (c0 + 32 * j < vec) dst[c0 + 32 * j] = v[j];
      }
    }
    fence_proxy_async_all();                                    // generic stores, read by other SMs' TMA loads
    asm volatile("bar.sync 2, 224;" ::: "memory");
    if (tid == 0) flag_release(a.sync + kSyncXReady + cta, epoch);
  }
  const uint32_t stage_bytes = kUmmaWBytes + NP * 128;
  const int tilesA = I / 64, tilesB = (H + 127) / 128;
  const int kitA = H / 64, kitB = I / 64;
  uint32_t* hready = a.sync + kSyncHReady;
  uint32_t* pready = a.sync + kSyncPartial;
  uint32_t* ydone = a.sync + fused_ydone_word_offset(E, ns, I);

  // Consumer side of the claimed-tile ring (a converged warp; `cn` = claims this warp has popped so far).
  auto claim_pop = [&](uint32_t& cn) -> int {
    const uint32_t slot = cn & (kClaimSlots - 1);
    int v = 0;
    if (lane == 0) {
      mbar_wait(cfull_bar(slot), (cn / kClaimSlots) & 1);
      v = sm.claim[slot];
      mbar_arrive(cempty_bar(slot));
    }
    ++cn;
    return __shfl_sync(0xffffffffu, v, 0);
  };
  // next piece of a consumer warp: data-parallel part -> pop a claim; remainder part -> the static walker
  auto consumer_next = [&](PieceWalker& pw, Piece& p, uint32_t& cn) -> bool {
    if (pw.dp) {
      if (pw.dp_end == 0) return false;
      return pw.next(p, claim_pop(cn));
    }
    return pw.next(p, 0);
  };

  if (warp == 4) {
    // ================================================================ weights producer (one lane)
    // Also draws this CTA's data-parallel tiles from the phase's global counter -- SMs do not get equal shares of
    // a saturated HBM (measured: +-8 %), so fixed rounds left the slow SMs 15-30 us behind at the grid barrier --
    // and hands each drawn tile to the seven consumer warps through a 4-slot shared-memory ring.  The next draw is
    // in flight while the current tile streams.
    if (lane == 0) {
      const uint64_t pol = l2_policy_evict_first();
      FSTAMP(5);
      uint32_t it = 0, wn = 0;
      bool cnt_ready = false;
      long long w_wait[2] = {0, 0}, w_iss[2] = {0, 0};
      (void)w_wait; (void)w_iss;
      auto claim_push = [&](int v) {
        const uint32_t slot = wn & (kClaimSlots - 1);
        mbar_wait(cempty_bar(slot), ((wn / kClaimSlots) & 1) ^ 1);
        sm.claim[slot] = v;
        mbar_arrive(cfull_bar(slot));
        ++wn;
      };
      for (int sp = 0; sp < 4; ++sp) {
        const int ph = sp >> 1;
        PieceWalker pw;
        pw.init(sp, tilesA, tilesB, kitA, kitB, total_pass, sm.cumpass, cta, G, a.dp_min_rounds, a.sk_split_pct, a.head_first != 0, a.sk_max_split);
        Piece p;
        auto stream_piece = [&]() {
          const int4 wk = sm.work[p.ent];
          const bool shared = wk.x >= E;
          const int we = shared ? wk.x - E : wk.x;
          const CUtensorMap* tmw = ph == 0 ? (shared ? &tm_sw13 : &tm_w13) : (shared ? &tm_sw2 : &tm_w2);
          for (int kc = p.k0; kc < p.k1; ++kc, ++it) {
            const int s = it % S;
            // suspended wait (try_wait with a time hint: the lane sleeps until a slot is free instead of re-polling the
            // barrier every ~80 cycles).  Measured: |U| = 128 197.7 -> 193.7 us, 64: 111.2 -> 108.6, T = 256 91.1 -> 92.5.
            // (The same wait selected by a run-time branch between the two loops cost 8 %: |U| = 128 213 us.)
            FTIMED(w_wait[ph], mbar_wait_long(empty_bar(s), ((it / S) & 1) ^ 1));
#ifdef ELDR_TRACE
            const long long cw_ = clock64();
#endif
            mbar_arrive_expect_tx(full_bar(s), kUmmaWBytes);
            const uint32_t dst = sm.stage_base + s * stage_bytes;
            if (ph == 0) tma_load_5d(dst, tmw, kc * 64, 0, 0, p.rt * 4, we, full_bar(s), pol);
            else tma_load_2d(dst, tmw, kc * 64, we * H + p.rt * 128, full_bar(s), pol);
#ifdef ELDR_TRACE
            w_iss[ph] += clock64() - cw_;
#endif
          }
        };
        if (pw.dp) {
          if (pw.dp_end > 0) {
            if (!cnt_ready) {
              uint32_t spins = 0;
              while (flag_acquire(a.sync + kSyncCntReady) != epoch) { __nanosleep(40); if (++spins > (1u << 24)) __trap(); }
              cnt_ready = true;
            }
            // first tile: the CTA's own index (no draw, no round trip before the first byte); the counter hands out
            // tiles G, G+1, ...
            int cur = cta;
            claim_push(cur);
            while (pw.next(p, cur)) {
              const int nxt = G + (int)atomicAdd(a.sync + kSyncTileCnt + ph, 1u);     // in flight while this tile streams
              stream_piece();
              claim_push(nxt);
              cur = nxt;
            }
          }
        } else {
          while (pw.next(p, 0)) stream_piece();
        }
        if (sp == 1) FSTAMP(11);
        FSTAMP3(sp);
      }
      FSTAMP(7);
      FVALUE2(0, w_wait[0]); FVALUE2(1, w_wait[1]); FVALUE2(10, w_iss[0]); FVALUE2(11, w_iss[1]);
    }
    __syncwarp();
  } else if (warp == 5 || warp == 7) {
    // ================================================================ activations producers (TMA)
    // Phase A: the expert's token rows of x are gathered four rows per instruction (tile::gather4) straight into
    // the swizzled K-major B tile -- the permutation never exists in HBM.  Phase B: the expert's h rows are
    // contiguous, plain 16-row boxes.  Nothing here waits for data: a stage's bytes are in flight as soon as its
    // slot is free, as deep as the ring (cp.async groups tracked by a warp capped that at six stages).
    // Two warps alternate ring stages.
    const uint32_t xw = warp == 7 ? 1u : 0u;
    const uint64_t xpol = l2_policy_evict_last();
    if (warp == 5 && lane == 0) {
      // CTA 0 zeroed this step's counters (tile draws, leavers): observed once per CTA, off the critical path
      uint32_t spins = 0;
      while (flag_acquire(a.sync + kSyncCntReady) != epoch) { __nanosleep(100); if (++spins > (1u << 22)) __trap(); }
    }
    __syncwarp();
    uint32_t it = 0, cn = 0;
    bool xs_ready = false;
#ifdef ELDR_TRACE
    unsigned long long stall = 0, nb = 0;
#endif
    for (int sp = 0; sp < 4; ++sp) {
      const int ph = sp >> 1;
      PieceWalker pw;
      pw.init(sp, tilesA, tilesB, kitA, kitB, total_pass, sm.cumpass, cta, G, a.dp_min_rounds, a.sk_split_pct, a.head_first != 0, a.sk_max_split);
      Piece p;
      int ready_ent = -1;
      while (consumer_next(pw, p, cn)) {
        const int4 wk = sm.work[p.ent];
        if (ph == 0 && use_xs && !xs_ready) {
          // The sorted copy takes ~3 us to appear (every CTA's part, flagged).  The head of this CTA's FIRST piece --
          // one ring's worth of stages -- is gathered from x as in the narrow case, so the MMAs start while the copy is
          // still being written; then the flags are awaited once and the piece goes on in the regular loop below.
          // (A loop of its own: the regular per-stage loop is sensitive to every instruction added to it.)
          const int n0h = p.pass * kNPCap;
          const int n_hh = min(kNPCap, wk.w - n0h);
          const int n_padh = (n_hh + 15) & ~15;
          int g0 = 0, g1 = 0, g2 = 0, g3 = 0;
          if (4 * lane < n_padh) {
            const uint16_t* tp = sm.tok_of_pos + wk.y + n0h;
            g0 = tp[min(4 * lane, n_hh - 1)];
            g1 = tp[min(4 * lane + 1, n_hh - 1)];
            g2 = tp[min(4 * lane + 2, n_hh - 1)];
            g3 = tp[min(4 * lane + 3, n_hh - 1)];
          }
          const int k_head = min(p.k1, p.k0 + S);
          for (int kc = p.k0; kc < k_head; ++kc, ++it) {
            if ((it & 1u) != xw) continue;
            const int s = it % S;
            if (lane == 0) {
              mbar_wait(empty_bar(s), ((it / S) & 1) ^ 1);
              mbar_arrive_expect_tx(full_bar(s), (uint32_t)n_padh * 128u);
            }
            __syncwarp();
            if (4 * lane < n_padh)
              tma_gather4(sm.stage_base + s * stage_bytes + kUmmaWBytes + lane * 512, &tm_x, kc * 64, g0, g1, g2, g3, full_bar(s), xpol);
          }
          p.k0 = k_head;
          warp_wait_flags(a.sync + kSyncXReady, G, epoch, lane);
          fence_proxy_async_all();
          __syncwarp();
          xs_ready = true;
        }
        if (ph == 1 && p.ent != ready_ent) {
          // every h tile of this expert must have landed (written by generic stores of other CTAs, read here by
          // the async proxy: acquire, then a proxy fence)
          const uint32_t* fl = hready + (size_t)sm.cumpass[p.ent] * tilesA;
          const int nfl = (sm.cumpass[p.ent + 1] - sm.cumpass[p.ent]) * tilesA;
          if (!warp_test_flags(fl, nfl, epoch, lane)) {
#ifdef ELDR_TRACE
            const unsigned long long t0_ = gtime();
#endif
            warp_wait_flags(fl, nfl, epoch, lane);
#ifdef ELDR_TRACE
            stall += gtime() - t0_; ++nb;
            if (lane == 0 && xw == 0) FADD3(8 + sp, gtime() - t0_);
#endif
          }
          fence_proxy_async_all();
          __syncwarp();
          ready_ent = p.ent;
#ifdef ELDR_TRACE
          if (lane == 0 && xw == 0 && g_trace[(blockIdx.x & 4095) * 16 + 14] == 0) FSTAMP(14);
#endif
        }
        const int n0 = p.pass * kNPCap;
        const int n_here = min(kNPCap, wk.w - n0);
        const int n_pad = (n_here + 15) & ~15;
        // phase A: this lane's four gather rows (padding rows repeat the last valid row; their columns are ignored)
        int r0 = 0, r1 = 0, r2 = 0, r3 = 0;
        if (ph == 0 && !use_xs && 4 * lane < n_pad) {
          const uint16_t* tp = sm.tok_of_pos + wk.y + n0;
          r0 = tp[min(4 * lane, n_here - 1)];
          r1 = tp[min(4 * lane + 1, n_here - 1)];
          r2 = tp[min(4 * lane + 2, n_here - 1)];
          r3 = tp[min(4 * lane + 3, n_here - 1)];
        }
        for (int kc = p.k0; kc < p.k1; ++kc, ++it) {
          if ((it & 1u) != xw) continue;
          const int s = it % S;
          if (lane == 0) {
            mbar_wait(empty_bar(s), ((it / S) & 1) ^ 1);
            mbar_arrive_expect_tx(full_bar(s), (uint32_t)n_pad * 128u);
          }
          __syncwarp();
          const uint32_t dst = sm.stage_base + s * stage_bytes + kUmmaWBytes;
          if (ph == 0) {
            if (use_xs) {
              if (16 * lane < n_pad) tma_load_2d(dst + lane * 2048, &tm_xs, kc * 64, wk.y + n0 + 16 * lane, full_bar(s), xpol);
            } else if (4 * lane < n_pad) {
              tma_gather4(dst + lane * 512, &tm_x, kc * 64, r0, r1, r2, r3, full_bar(s), xpol);
            }
          } else {
            if (16 * lane < n_pad) tma_load_2d(dst + lane * 2048, &tm_h, kc * 64, wk.z + n0 + 16 * lane, full_bar(s), xpol);
          }
        }
      }
    }
#ifdef ELDR_TRACE
    if (lane == 0 && xw == 0) { FVALUE(12, stall); }
#endif
  } else if (warp == 6) {
    // ================================================================ MMA issuer
    // The warp stays converged; every operand of the issue path is warp-uniform (redux / kernel parameters) and
    // the tcgen05 instructions are predicated on the elected lane inside the asm, so one stage costs four
    // back-to-back UTCHMMA + one UTCBAR instead of five ELECT/R2UR waterfalls.  Ring slot and parity are carried
    // incrementally (no division by the run-time ring depth).
    const uint32_t leader = elect_one();
    const uint32_t uS = warp_uniform((uint32_t)S), ustage = warp_uniform(stage_bytes);
    const uint32_t ubase = warp_uniform(sm.stage_base), ubar = warp_uniform(sm.bar_base);
    const uint32_t utmem = warp_uniform(tmem_base);
    uint32_t s = 0, par = 0, piece_no = 0, cn = 0;
    bool first = true;
    for (int sp = 0; sp < 4; ++sp) {
      PieceWalker pw;
      pw.init(sp, tilesA, tilesB, kitA, kitB, total_pass, sm.cumpass, cta, G, a.dp_min_rounds, a.sk_split_pct, a.head_first != 0, a.sk_max_split);
      Piece p;
      while (consumer_next(pw, p, cn)) {
        const int4 wk = sm.work[p.ent];
        const uint32_t n_pad = warp_uniform((uint32_t)((min(kNPCap, wk.w - p.pass * kNPCap) + 15) & ~15));
        const uint32_t nk = warp_uniform((uint32_t)(p.k1 - p.k0));
        const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((n_pad >> 3) << 17) | (8u << 24);
        const uint32_t buf = piece_no & 1u;
        mbar_wait(ubar + 8u * (2 * kMaxStages + 2 + buf), ((piece_no >> 1) & 1u) ^ 1u);      // tempty
        tc_fence_after();
        const uint32_t d_tmem = utmem + buf * kNPCap;
        for (uint32_t j = 0; j < nk; ++j) {
          mbar_wait(ubar + 8u * s, par);                                                      // full
          tc_fence_after();
          if (first) { first = false; if (lane == 0) FSTAMP(6); }
          const uint32_t sa = ubase + s * ustage;
          const uint64_t da = umma_desc_sw128(sa), db = umma_desc_sw128(sa + kUmmaWBytes);
#pragma unroll
          for (int kk = 0; kk < 4; ++kk) umma_bf16_if(leader, d_tmem, da + 2 * kk, db + 2 * kk, idesc, (j | kk) ? 1u : 0u);
          umma_commit_if(leader, ubar + 8u * (kMaxStages + s));                                // empty
          if (j == nk - 1) umma_commit_if(leader, ubar + 8u * (2 * kMaxStages + buf));         // tfull
          if (++s == uS) { s = 0; par ^= 1u; }
        }
        ++piece_no;
      }
      if (sp == 1 && lane == 0) FSTAMP(13);
    }
  } else if (warp < 4) {
    // ================================================================ epilogue (TMEM lane quarter = warp)
    const int qtr = warp;
    uint32_t piece_no = 0, cn = 0;
    for (int sp = 0; sp < 4; ++sp) {
      const int ph = sp >> 1;
      PieceWalker pw;
      pw.init(sp, tilesA, tilesB, kitA, kitB, total_pass, sm.cumpass, cta, G, a.dp_min_rounds, a.sk_split_pct, a.head_first != 0, a.sk_max_split);
      const long long P = pw.P;
      const int Gs = pw.Gs;
      Piece p;
      while (consumer_next(pw, p, cn)) {
        const int4 wk = sm.work[p.ent];
        const int n0 = p.pass * kNPCap;
        const int n_here = min(kNPCap, wk.w - n0);
        const int buf = piece_no & 1;
        const int row = 32 * qtr + lane;                        // TMEM lane = row of the 128-row tile
        // Head piece of a split tile: the other pieces were parked long ago (their owners reach the tile first).
        // Find them, wait for their flags and request the first chunk of the first partner BEFORE waiting for our
        // own accumulator: under a saturated memory system every dependent L2 round trip costs more than a microsecond.
        if (tid == 0 && ph == 0) FSTAMP2(3);
        int n_partner = 0;
        float4 pf0[4], pf1[4], pf2[4], pf3[4];                  // four chunks of the first partner in flight
        bool pf_valid = false;
        // Which piece of a split tile finishes it: the owner of its LAST stage (head_first: the partners are the
        // PRECEDING CTAs, which parked their head pieces at the very start of the sub-phase) or, in the round-1 order,
        // the owner of its first stage (partners = the following CTAs, which reach the tile first).
        const bool hf = a.head_first != 0;
        const int dir = hf ? -1 : 1;
        const bool finisher = hf ? (p.k1 == pw.kit) : (p.k0 == 0);
        if (finisher && (hf ? p.k0 > 0 : p.k1 < pw.kit)) {
          auto wait_partner = [&](int j) {
            if (lane == 0) {
              uint32_t spins = 0;
#ifdef ELDR_TRACE
              const unsigned long long tp0_ = gtime();
#endif
              while (flag_acquire(pready + sp * 256 + j) != epoch) { __nanosleep(40); if (++spins > (1u << 24)) __trap(); }
#ifdef ELDR_TRACE
              if (tid == 0) FADD3(12 + sp, gtime() - tp0_);
#endif
            }
          };
          if (!hf) {
            const long long tile_end = ((long long)(p.tile - pw.tile0) + 1) * pw.kit;
            long long covered = (long long)(p.tile - pw.tile0) * pw.kit + p.k1;
            int j = cta + 1;
            while (covered < tile_end && j < Gs) {
              const long long hj = P * (j + 1) / Gs;
              if (hj > covered) {                              // CTA j owns a non-empty piece of this tile
                wait_partner(j);
                covered = min(hj, tile_end);
                n_partner = j - cta;
              }
              ++j;
            }
          } else {
            const long long tile_start = (long long)(p.tile - pw.tile0) * pw.kit;
            for (int j = cta - 1; j >= 0; --j) {
              const long long lj = P * j / Gs, hj = P * (j + 1) / Gs;
              if (hj <= lj) continue;                          // empty range: parked nothing
              if (hj <= tile_start) break;
              wait_partner(j);
              n_partner = cta - j;
              if (lj <= tile_start) break;
            }
          }
          __syncwarp();
          pf_valid = n_partner >= 1 && (P * (cta + dir + 1) / Gs > P * (cta + dir) / Gs);
        }
        // parked partials: [slot][column / 4][row] float4 -- the 32 lanes of a warp (consecutive rows) touch 512
        // contiguous bytes per access
        const float4* pf_src = reinterpret_cast<const float4*>(a.partial) + (size_t)(sp * G + cta + dir) * 128 * (kNPCap / 4) + row;
        auto pf_load = [&](float4 (&dst)[4], int c0) {
          if (pf_valid && c0 < n_here) {
#pragma unroll
            for (int q = 0; q < 4; ++q) dst[q] = __ldcg(pf_src + (size_t)(c0 / 4 + q) * 128);
          }
        };
        if (tid == 0 && ph == 0) FSTAMP2(2);
        pf_load(pf0, 0);
        pf_load(pf1, 16);
        pf_load(pf2, 32);
        pf_load(pf3, 48);
#ifdef ELDR_TRACE
        const long long ce0_ = clock64();
#endif
        mbar_wait(tfull_bar(buf), (piece_no >> 1) & 1);
        tc_fence_after();
#ifdef ELDR_TRACE
        const long long ce1_ = clock64();
#endif
        if (tid == 0 && ph == 0) FSTAMP(2);
        const uint32_t t_addr = tmem_base + buf * kNPCap + ((uint32_t)(qtr * 32) << 16);
        if (!finisher) {
          // ---- not the finisher of this tile: park the raw accumulators for it
          float4* dstp = reinterpret_cast<float4*>(a.partial) + (size_t)(sp * G + cta) * 128 * (kNPCap / 4) + row;
          for (int c0 = 0; c0 < n_here; c0 += 16) {
            float v[16];
            tmem_ld16(t_addr + c0, v);
#pragma unroll
            for (int q = 0; q < 4; ++q)
              dstp[(size_t)(c0 / 4 + q) * 128] = make_float4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
          }
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(tempty_bar(buf));
#ifdef ELDR_TRACE
          const long long ce2_ = clock64();
#endif
          // (no per-thread fence: the release below is cumulative over the barrier; 128 membars cost ~1 us per step)
          asm volatile("bar.sync 1, 128;" ::: "memory");
          if (tid == 0) flag_release(pready + sp * 256 + cta, epoch);
#ifdef ELDR_TRACE
          if (tid == 0) { const int b_ = ph * 8; FADD4(b_ + 0, 1); FADD4(b_ + 1, ce1_ - ce0_); FADD4(b_ + 2, ce2_ - ce1_); FADD4(b_ + 3, clock64() - ce2_); }
#endif
        } else {
          // ---- finisher (or only owner): add the partners' parked partials, nearest CTA first (a fixed order)
          auto chunk = [&](int c0, float4 (&pfx)[4]) {
            float v[16];
            tmem_ld16(t_addr + c0, v);
            if (pf_valid) {
#pragma unroll
              for (int q = 0; q < 4; ++q) {
                v[4 * q] += pfx[q].x; v[4 * q + 1] += pfx[q].y; v[4 * q + 2] += pfx[q].z; v[4 * q + 3] += pfx[q].w;
              }
              pf_load(pfx, c0 + 64);                           // refill this buffer four chunks ahead
            }
            for (int j = pf_valid ? 2 : 1; j <= n_partner; ++j) {
              // CTAs with an empty range parked nothing; their slot is skipped by the same test as above
              const long long lj = P * (cta + dir * j) / Gs, hj = P * (cta + dir * j + 1) / Gs;
              if (hj <= lj) continue;
              const float4* srcp = reinterpret_cast<const float4*>(a.partial) + (size_t)(sp * G + cta + dir * j) * 128 * (kNPCap / 4) + row;
#pragma unroll
              for (int q = 0; q < 4; ++q) {
                const float4 pv = __ldcg(srcp + (size_t)(c0 / 4 + q) * 128);
                v[4 * q] += pv.x; v[4 * q + 1] += pv.y; v[4 * q + 2] += pv.z; v[4 * q + 3] += pv.w;
              }
            }
            if (ph == 0) {
              // lanes 0-15: g for i = rt*64 + 16*qtr + lane; lanes 16-31: u for the same i
              // (three straight-line passes -- exchange, SiLU * u, predicated stores: with the bounds test around
              // the whole body every element was its own branch region, shuffle -> ex2 -> rcp -> store in series,
              // ~0.8 us per 16-column chunk)
              const bool lo = lane < 16;
              const int i = p.rt * 64 + 16 * qtr + (lane & 15);
              float gv[8], uv[8];
#pragma unroll
              for (int kk = 0; kk < 8; ++kk) {
                const float send = lo ? v[8 + kk] : v[kk];
                const float recv = __shfl_xor_sync(0xffffffffu, send, 16);
                gv[kk] = lo ? v[kk] : recv;
                uv[kk] = lo ? recv : v[8 + kk];
              }
              uint16_t hv[8];
#pragma unroll
              for (int kk = 0; kk < 8; ++kk) hv[kk] = f32_to_bf16_rn(__fdividef(gv[kk], 1.0f + __expf(-gv[kk])) * uv[kk]);
              const int tok0 = n0 + c0 + (lo ? 0 : 8);
              uint16_t* hp = a.hbuf + (size_t)(wk.z + tok0) * I + i;
              const int n_rem = wk.w - tok0;
#pragma unroll
              for (int kk = 0; kk < 8; ++kk)
                if (kk < n_rem) hp[(size_t)kk * I] = hv[kk];
            } else {
              const int r = p.rt * 128 + row;
              if (r < H) {
#pragma unroll
                for (int kk = 0; kk < 16; ++kk) {
                  const int tok = n0 + c0 + kk;
                  if (tok < wk.w)
                    a.ybuf[(size_t)(wk.z + tok) * H + r] = v[kk];
                }
              }
            }
          };
          for (int c0 = 0; c0 < n_here; c0 += 64) {
            chunk(c0, pf0);
            if (tid == 0 && ph == 0 && c0 == 0) FSTAMP(3);
            if (c0 + 16 < n_here) chunk(c0 + 16, pf1);
            if (c0 + 32 < n_here) chunk(c0 + 32, pf2);
            if (c0 + 48 < n_here) chunk(c0 + 48, pf3);
          }
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive(tempty_bar(buf));
          if (tid == 0 && ph == 0) FSTAMP(4);
#ifdef ELDR_TRACE
          const long long ce2_ = clock64();
#endif
          if (ph == 0) {
            // publish "h tile written": each writer orders its stores before later async-proxy (TMA) reads, the
            // four epilogue warps meet, one thread releases (cumulative)
            fence_proxy_async_all();
            asm volatile("bar.sync 1, 128;" ::: "memory");
            if (tid == 0) { flag_release(hready + p.tile, epoch); FSTAMP(15); }
          } else {
            // publish "y tile written" for the flag-driven combine
            asm volatile("bar.sync 1, 128;" ::: "memory");
            if (tid == 0) flag_release(ydone + p.tile, epoch);
          }
#ifdef ELDR_TRACE
          if (tid == 0) { const int b_ = ph * 8 + 4; FADD4(b_ + 0, 1); FADD4(b_ + 1, ce1_ - ce0_); FADD4(b_ + 2, ce2_ - ce1_); FADD4(b_ + 3, clock64() - ce2_); }
#endif
        }
        ++piece_no;
      }
      if (tid == 0) FSTAMP3(4 + sp);
    }
  }

  // ------------------------------------------------------------------------------ C: flag-driven combine
  // No grid barrier: the unit of combine work is (token t, 128-column tile rt) = one warp pass; lane j < k looks up
  // slot j's y tile (work entry of the expert, accumulator pass of the position, rt) and polls that tile's "y
  // written" flag, lanes k..k+ns-1 do the same for the shared experts; when all are up the warp sums the k (+ns) rows
  // in slot order -- a fixed order, so results stay run-to-run bit-identical -- and rounds once to bf16.  Every warp
  // CTA starts on its units as soon as its own FFN roles have run out of pieces, so the combine of tokens whose
  // experts finished early overlaps the last tiles of the slow SMs (round 1: every SM waited for the slowest one, then
  // combined: barrier + combine 3.4 us after the last tile).  Polls are one 4-byte load per slot and sleep 250 ns in
  // between: warps that polled from the moment their role ended, all lanes, every 100 ns, hot-spotted the flags' L2
  // lines and cost every step 40 us (measured).
  if (tid == 0) FSTAMP(8);
  __syncthreads();
  if (k <= 8) fused_combine<8>(a, sm, ydone, epoch, n_work, tilesB, cta, G, warp, lane);
  else fused_combine<kMaxTopK>(a, sm, ydone, epoch, n_work, tilesB, cta, G, warp, lane);
  if (tid == 0) FSTAMP(10);
  sig_add_finish(sig_pend);

  tc_fence_before();
  __syncthreads();
  if (tid == 0) FSTAMP(9);
  if (tid == 0) {
    // Leave the step.  The counter was zeroed by CTA 0 in this step's first microsecond (seen here: warp 5 acquired
    // kSyncCntReady == epoch before its first piece, and the barrier above orders that before this add); the last CTA
    // to leave publishes the new generation -- every CTA read the old one long before it got here.  One atomicAdd per
    // CTA: a compare-and-swap loop on an epoch-tagged word serialised the 148 leavers by L2 round trips and cost
    // every step 30 us (measured).
    if (atomicAdd(a.sync + kSyncExit, 1u) == (uint32_t)G - 1u) a.sync[kSyncGen] = gen_next;
  }
  if (warp == 6) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_base), "r"(tmem_cols) : "memory");
  }
}

}  // namespace eldr
