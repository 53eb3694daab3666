// Grouped SwiGLU expert FFN with MXFP4 expert weights ("GPT-OSS-120B (128 experts,
// top-4, mxfp4)").  Format (readings in DESIGN.md 2, the oracle's: oracle/mxfp4.py): FP4 E2M1 codes, two per byte
// (element 2i in the low nibble), one E8M0 scale byte per 32 elements of the contraction axis, value =
// e2m1(code) * 2^(scale - 127).  Every decoded value is exactly a bf16 number, and the activations stay bf16, so the
// layer is BY DEFINITION the plain layer on the decoded weights: the kernel streams the packed bytes from HBM
// (17/64 of the bf16 bytes), decodes them to bf16 in registers, stores the decoded tile into TENSOR MEMORY
// (tcgen05.st) and issues the swap-AB MMAs with the A operand read from TMEM -- nothing is approximated, the
// activations are not quantised.  (Round 2's first version wrote the decoded tiles to shared memory: decoded data is
// four times the packed bytes, written once and read once by the tensor core -- at HBM speed that alone is ~180 bytes
// per clock against the 128 bytes per clock of an SM's shared memory.  TMEM ring: 1.49 -> 1.75 TB/s of packed bytes.)
//
// One persistent CTA per SM, 11 warps:
//   warp 0   TMA producer, packed weights: 128 rows x 128 bytes (256 codes per row = FOUR 64-element k-chunks) per RAW
//            stage (16 KiB, SWIZZLE_128B; MODE 0: 64 rows of w1 + the same 64 rows of w3), L2 evict_first.  (A first
//            version fetched one k-chunk = 32 bytes per row per stage: 32-byte pieces of 1440-byte rows ran HBM at
//            1.2 TB/s even with the decode switched off.)
//   warp 1   TMA producer, activations (as ffn_umma.cuh)
//   warp 2   MMA issuer: 4 x tcgen05.mma (M=128, N=n_pad, K=16; A = 8 TMEM columns of the decoded ring, B = shared
//            memory descriptor) per stage, fp32 accumulators in TMEM
//   warps 3-6  epilogue: TMEM -> SiLU*mul -> h (MODE 0) / y (MODE 1)
//   warps 7-10 decoders: thread r owns row r of the 128-row tile.  Per k-chunk it reads 32 raw bytes of its row and the
//            row's two scale bytes (the eight scale bytes of a raw stage are fetched three raw stages ahead with 4-byte
//            cp.async into a per-thread ring: the scale rows are K/32 bytes long, neither 16-byte aligned nor
//            TMA-addressable), decodes 64 codes with two
//            byte-permute look-ups per four codes (magnitudes 0, .5, 1, 1.5, 2, 3, 4, 6 need five distinct bf16 bytes),
//            ORs in the signs, multiplies by the scale as a bf16x2 power of two (exact) and stores its 16 columns
//            (32 bf16) of the tile row = TMEM lane it owns (a warp reaches the lanes of its quarter, warp % 4); MODE 0
//            rows land in the 4 x [16 rows of w1 | 16 of w3] order the SiLU*mul epilogue expects.  20 operations per 8 codes, 14-16 of them on the ALU pipe (byte permutes,
//            logic): 8192 codes per stage -> ~256 SM cycles of ALU-pipe time against ~180 cycles a 4 KiB stage lasts
//            at HBM speed, so the decode -- not HBM -- bounds this kernel (measured 1.5 TB/s of packed bytes, 2.2 TB/s
//            with the decode switched off; every role's loop nest is written out with incremental ring cursors
//            because a generic per-stage walker with run-time modulos alone held it at 0.9 TB/s).
#pragma once
#include <cuda_bf16.h>

#include "ffn_umma.cuh"

namespace eldr {

#ifndef ELDR_MX_PARTS
#define ELDR_MX_PARTS 2
#endif
constexpr int kMxParts = ELDR_MX_PARTS;        // decoder threads per tile row (each decodes 64 / kMxParts codes per stage)
constexpr int kMxDecWarps = 4 * kMxParts;
constexpr int kMxThreads = (7 + kMxDecWarps) * 32;
constexpr int kMxRawBytes = 128 * 128;         // packed codes of one raw stage: 128 rows x 4 k-chunks
constexpr int kMxRawChunks = 4;                // 64-element k-chunks per raw stage
constexpr int kMxATmemCol = 256;               // first TMEM column of the decoded-tile ring (accumulators: 2 x np <= 256 columns)
constexpr int kMxMaxStages = 8;                // decoded-tile ring: 8 x 32 columns
constexpr int kMxScaleAhead = 3;               // raw stages of scale prefetch per decoder thread (16-byte slot each)

struct MxArgs {
  FfnArgs f;
  const uint8_t* scales;      // [E * rows_per_expert, K/32]
  int np, stages, raw_stages, act_stages;
};

// Three rings: RAW packed codes (HBM latency: deep in bytes), decoded bf16 weight tiles (on-chip hand-over: shallow),
// activations (L2 latency: their own ring -- sharing the weight tiles' four stages bounded the pipeline at four stages
// per L2 round trip, 1.2 TB/s).
__host__ __device__ inline size_t mx_smem_bytes(int np, int stages, int raw_stages, int act_stages) {
  (void)stages;                                  // decoded tiles live in TMEM, not in shared memory
  return (size_t)act_stages * np * 128 + (size_t)raw_stages * kMxRawBytes +
         (size_t)kMxScaleAhead * kMxDecWarps * 32 * 16 + 1024 + 1024;
}

// 8 codes (one 32-bit word, element j in nibble j) -> 8 bf16 values scaled by `sc` (bf16x2, both halves 2^(b-127)),
// in the K-SLOT ORDER e0 e4 | e1 e5 | e2 e6 | e3 e7 (kMxSlot: slot j of a group of eight holds element kMxSlot[j]).
// An E2M1 code s|ee|m placed as a bf16 with exponent field ee and top mantissa bit m IS the code's value times 2^-126
// -- for ee = 0 a bf16 subnormal, m * 2^-127: the subnormal code 0.5 needs no special case -- so a code pair becomes
// a bf16x2 with one mask, one integer multiply (x * (2^a + 2^b) = two shifted copies: exponent/mantissa and sign
// each land on their bit positions) and one mask; the masks pick nibbles j and j+4 of the word, which lie exactly 16
// bits apart: no shifts.  Then one exact bf16x2 multiply by 2^126 x the block scale.  Per word 9 logic
// operations (ALU pipe) + 4 integer multiplies + 4 bf16x2 multiplies (FMA pipe); the byte-permute look-up it replaces
// took 16 on the ALU pipe, which bounds this kernel (ncu: ALU 59 % busy at 1.6 TB/s, FMA 15 %).  The contraction does
// not care about the order of its terms as long as BOTH operands use it: the activation rows are stored in the same
// slot order (gather_x_kernel, the MODE 0 epilogue).
// `sc` = bf16x2 of 2^(b-1) (the 2^126 folded in) for scale bytes b <= 128; larger scales (`wide`, weights beyond 2^1 per
// unit code: not seen in practice) take the two multiplies 2^126, 2^(b-127).
__device__ __forceinline__ uint4 mx_decode8(uint32_t w, __nv_bfloat162 sc, bool wide) {
  const uint32_t k126 = 0x7E807E80u;                          // bf16x2 (2^126, 2^126)
  const __nv_bfloat162 c126 = *reinterpret_cast<const __nv_bfloat162*>(&k126);
  const uint32_t w8 = w >> 8;
  uint32_t o[4];
  o[0] = ((w & 0x000F000Fu) * 0x1040u) & 0x81C081C0u;         // nibbles 0, 4: value << 6, sign << 12
  o[1] = ((w & 0x00F000F0u) * 0x0104u) & 0x81C081C0u;         // nibbles 1, 5: value << 2, sign << 8
  o[2] = ((w8 & 0x000F000Fu) * 0x1040u) & 0x81C081C0u;        // nibbles 2, 6
  o[3] = ((w8 & 0x00F000F0u) * 0x0104u) & 0x81C081C0u;        // nibbles 3, 7
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    __nv_bfloat162 v = *reinterpret_cast<__nv_bfloat162*>(&o[k]);
    if (wide) v = __hmul2(v, c126);
    v = __hmul2(v, sc);
    o[k] = *reinterpret_cast<uint32_t*>(&v);
  }
  return make_uint4(o[0], o[1], o[2], o[3]);
}
// slot of element e inside its group of eight (inverse of the slot order above)
__host__ __device__ __forceinline__ int mx_slot_of(int e) { return (e & ~7) | ((e & 3) << 1) | ((e >> 2) & 1); }

// Walks this CTA's (tile, pass, k-chunk) stages in the order every role uses.
struct MxWalker {
  const FfnArgs* a;
  int tile, total, step, np, k_iters, kstep;
  int ent, rt, we, m, n0, kc;
  bool live;
  __device__ __forceinline__ void load_tile() {
    live = tile < total;
    if (!live) return;
    ent = tile / a->tiles_per_expert;
    rt = tile - ent * a->tiles_per_expert;
    const int4 wk = a->work[ent];
    we = wk.x;
    m = wk.w;
    n0 = 0;
    kc = 0;
  }
  __device__ __forceinline__ void init(const FfnArgs* a_, int total_, int np_, int k_iters_, int kstep_ = 1) {
    a = a_; total = total_; np = np_; k_iters = k_iters_; kstep = kstep_;
    tile = blockIdx.x; step = gridDim.x;
    load_tile();
  }
  __device__ __forceinline__ void next() {
    kc += kstep;
    if (kc < k_iters) return;
    kc = 0;
    n0 += np;
    if (n0 < m) return;
    tile += step;
    load_tile();
  }
};

template <int MODE>
__global__ void __launch_bounds__(kMxThreads, 1)
ffn_mx_kernel(const __grid_constant__ CUtensorMap tm_codes, const __grid_constant__ CUtensorMap tm_x16,
              const __grid_constant__ CUtensorMap tm_x64, const MxArgs a) {
  extern __shared__ uint8_t smem_dyn[];
  const uint32_t smem_base = (smem_u32(smem_dyn) + 1023u) & ~1023u;
  uint8_t* smem_gen = smem_dyn + (smem_base - smem_u32(smem_dyn));
  const int NP = a.np, S = a.stages, RS = a.raw_stages, AS = a.act_stages;
  const uint32_t act_bytes = NP * 128;
  const uint32_t act_base = smem_base;
  const uint32_t raw_base = act_base + AS * act_bytes;
  const uint32_t sc_base = raw_base + RS * kMxRawBytes;             // [kMxScaleAhead][128] x 16 bytes
  const uint32_t bar_base = sc_base + kMxScaleAhead * kMxDecWarps * 32 * 16;
  auto wfull_bar = [&](int s) { return bar_base + 8u * s; };
  auto wempty_bar = [&](int s) { return bar_base + 8u * (S + s); };
  auto rfull_bar = [&](int s) { return bar_base + 8u * (2 * S + s); };
  auto rempty_bar = [&](int s) { return bar_base + 8u * (2 * S + RS + s); };
  auto tfull_bar = [&](int b) { return bar_base + 8u * (2 * S + 2 * RS + b); };
  auto tempty_bar = [&](int b) { return bar_base + 8u * (2 * S + 2 * RS + 2 + b); };
  auto afull_bar = [&](int s) { return bar_base + 8u * (2 * S + 2 * RS + 4 + s); };
  auto aempty_bar = [&](int s) { return bar_base + 8u * (2 * S + 2 * RS + 4 + AS + s); };
  const uint32_t tmem_slot = bar_base + 8u * (2 * S + 2 * RS + 4 + 2 * AS);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(wfull_bar(s), kMxDecWarps); mbar_init(wempty_bar(s), 1); }
    for (int s = 0; s < AS; ++s) { mbar_init(afull_bar(s), 1); mbar_init(aempty_bar(s), 1); }
    for (int s = 0; s < RS; ++s) { mbar_init(rfull_bar(s), 1); mbar_init(rempty_bar(s), kMxDecWarps); }
    for (int b = 0; b < 2; ++b) { mbar_init(tfull_bar(b), 1); mbar_init(tempty_bar(b), 4); }
    mbar_fence_init();
  }
  // TMEM: accumulators (2 x NP columns) at column 0, the ring of decoded weight tiles (S stages x 32 columns: 128 rows
  // x 64 bf16, two per 32-bit column) from column kMxATmemCol on.  All 512 columns: one CTA per SM.
  const uint32_t tmem_cols = 512;
  if (warp == 2) {
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

  const FfnArgs& f = a.f;
  const int n_work = *f.n_work;
  const int total_tiles = n_work * f.tiles_per_expert;
  const int k_iters = f.K / 64;
  const int kbytes = f.K / 2;                       // packed bytes per weight row

  if (warp == 0) {
    // ================================================================ packed-weights producer
    if (lane == 0) {
      tma_prefetch_desc(&tm_codes);
      const uint64_t pol = l2_policy_evict_first();
      MxWalker w;
      w.init(&f, total_tiles, NP, k_iters, kMxRawChunks);
      for (uint32_t it = 0; w.live; w.next(), ++it) {
        const int rs = it % RS;
        mbar_wait(rempty_bar(rs), ((it / RS) & 1) ^ 1);
        mbar_arrive_expect_tx(rfull_bar(rs), kMxRawBytes);
        const uint32_t dst = raw_base + rs * kMxRawBytes;
        if (MODE == 0) {
          const int row0 = w.we * f.rows_per_expert + w.rt * 64;
          tma_load_2d(dst, &tm_codes, w.kc * 32, row0, rfull_bar(rs), pol);
          tma_load_2d(dst + kMxRawBytes / 2, &tm_codes, w.kc * 32, row0 + f.I, rfull_bar(rs), pol);
        } else {
          tma_load_2d(dst, &tm_codes, w.kc * 32, w.we * f.rows_per_expert + w.rt * 128, rfull_bar(rs), pol);
        }
      }
    }
  } else if (warp == 1) {
    // ================================================================ activations producer
    if (lane == 0) {
      tma_prefetch_desc(&tm_x16);
      const uint64_t pol = l2_policy_evict_last();
      // (loop nest written out, ring cursor carried incrementally: a 4 KiB stage lasts ~180 cycles at HBM speed, so a
      // single-lane role has ~40 instructions per stage to spend)
      uint32_t as = 0, apar = 1;
      for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
        const int ent = tile / f.tiles_per_expert;
        const int4 wk = f.work[ent];
        const int xrow0 = (MODE == 0) ? wk.y : wk.z;
        for (int n0 = 0; n0 < wk.w; n0 += NP) {
          const int n_pad = (min(NP, wk.w - n0) + 15) & ~15;
          const bool big = n_pad > 48;
          const int n_box = big ? (n_pad + 63) / 64 : n_pad / 16;
          const uint32_t box_bytes = big ? 64 * 128 : 16 * 128;
          const CUtensorMap* tmx = big ? &tm_x64 : &tm_x16;
          const int row = xrow0 + n0, rstep = big ? 64 : 16;
          for (int kc = 0; kc < k_iters; ++kc) {
            mbar_wait(aempty_bar(as), apar);
            mbar_arrive_expect_tx(afull_bar(as), n_box * box_bytes);
            const uint32_t dst = act_base + as * act_bytes;
            for (int b = 0; b < n_box; ++b)
              tma_load_2d(dst + b * box_bytes, tmx, kc * 64, row + b * rstep, afull_bar(as), pol);
            if (++as == (uint32_t)AS) { as = 0; apar ^= 1u; }
          }
        }
      }
    }
  } else if (warp == 2) {
    // ================================================================ MMA issuer
    // The warp stays converged; operands of the issue path are warp-uniform and the tcgen05 instructions are
    // predicated on the elected lane inside the asm (no ELECT / R2UR waterfall per instruction).
    const uint32_t leader = elect_one();
    const uint32_t uS = warp_uniform((uint32_t)S), uAS = warp_uniform((uint32_t)AS);
    const uint32_t ubar = warp_uniform(bar_base), ua = warp_uniform(act_base), uab = warp_uniform(act_bytes);
    const uint32_t utmem = warp_uniform(tmem_base);
    uint32_t unit = 0, ws_ = 0, wpar = 0, as = 0, apar = 0;
    for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
      const int ent = tile / f.tiles_per_expert;
      const int m_tok = f.work[ent].w;
      for (int n0 = 0; n0 < m_tok; n0 += NP, ++unit) {
        const uint32_t n_pad = warp_uniform((uint32_t)((min(NP, m_tok - n0) + 15) & ~15));
        const uint32_t idesc = (1u << 4) | (1u << 7) | (1u << 10) | ((n_pad >> 3) << 17) | (8u << 24);
        const uint32_t buf = unit & 1u;
        mbar_wait(ubar + 8u * (2 * uS + 2 * RS + 2 + buf), ((unit >> 1) & 1u) ^ 1u);       // tempty
        tc_fence_after();
        const uint32_t d_tmem = utmem + buf * NP;
        for (int kc = 0; kc < k_iters; ++kc) {
          mbar_wait(ubar + 8u * (2 * uS + 2 * RS + 4 + as), apar);                          // afull
          mbar_wait(ubar + 8u * ws_, wpar);                                                 // wfull
          tc_fence_after();
          const uint32_t a_tmem = utmem + kMxATmemCol + ws_ * 32u;
          const uint64_t db = umma_desc_sw128(ua + as * uab);
#pragma unroll
          for (int k = 0; k < 4; ++k) umma_bf16_ts_if(leader, d_tmem, a_tmem + 8u * k, db + 2 * k, idesc, (kc | k) ? 1u : 0u);
          umma_commit_if(leader, ubar + 8u * (uS + ws_));                                   // wempty
          umma_commit_if(leader, ubar + 8u * (2 * uS + 2 * RS + 4 + uAS + as));             // aempty
          if (kc == k_iters - 1) umma_commit_if(leader, ubar + 8u * (2 * uS + 2 * RS + buf));   // tfull
          if (++ws_ == uS) { ws_ = 0; wpar ^= 1u; }
          if (++as == uAS) { as = 0; apar ^= 1u; }
        }
      }
    }
  } else if (warp < 7) {
    // ================================================================ epilogue (TMEM lane quarter = warp & 3)
    const int qtr = warp & 3;
    uint32_t unit = 0;
    for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
      const int ent = tile / f.tiles_per_expert, rt = tile - ent * f.tiles_per_expert;
      const int4 wk = f.work[ent];
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
            const bool lo = lane < 16;
            const int i = rt * 64 + 16 * qtr + (lane & 15);
#pragma unroll
            for (int k = 0; k < 8; ++k) {
              const float send = lo ? v[8 + k] : v[k];
              const float recv = __shfl_xor_sync(0xffffffffu, send, 16);
              const float gv = lo ? v[k] : recv;
              const float uv = lo ? recv : v[8 + k];
              const int tok = n0 + c0 + (lo ? k : 8 + k);
              if (tok < wk.w) f.h_out[(size_t)(wk.z + tok) * f.I + mx_slot_of(i)] = f32_to_bf16_rn(silu_f(gv) * uv);   // K-slot order of the w2 decode
            }
          } else {
            const int r = rt * 128 + 32 * qtr + lane;
            if (r < f.H) {
#pragma unroll
              for (int k = 0; k < 16; ++k) {
                const int tok = n0 + c0 + k;
                if (tok < wk.w) f.y_out[(size_t)(wk.z + tok) * f.H + r] = v[k];
              }
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(tempty_bar(buf));
      }
    }
  } else {
    // ================================================================ decoders: tile row d, part `part` of its 64 codes.
    // kMxParts threads share a row so that each SM sub-partition holds several decoder warps: one warp per
    // sub-partition ran the ~300 dependent-ish ALU instructions of a stage at ~3 cycles each (ncu: 1.4 IPC, 0.9 TB/s).
    // A warp reaches only the TMEM lanes of its quarter (warp % 4): thread -> tile row d = 32 * (warp % 4) + lane.
    const int dt = threadIdx.x - 7 * 32;
    const int d = 32 * (warp & 3) + lane, part = (warp - 7) >> 2;
    const int kscale = f.K / 32;                     // scale bytes per weight row
    const size_t scale_total = (size_t)f.E * f.rows_per_expert * kscale;
    // row of this thread inside the expert's weight matrix, as a function of the row tile
    auto grow = [&](int rt) -> int {
      if (MODE == 0) {
        const int g = d >> 5, j = d & 31;
        return (j < 16 ? 0 : f.I) + rt * 64 + g * 16 + (j & 15);
      }
      return min(rt * 128 + d, f.rows_per_expert - 1);          // rows past H are never read back
    };
    const int src_row = MODE == 0 ? (((d & 31) < 16 ? 0 : 64) + (d >> 5) * 16 + (d & 15)) : d;
    const uint32_t my_sc = sc_base + dt * 16;        // every decoder thread keeps its own copy of its row's scale bytes
    const uint4* my_sc_gen = reinterpret_cast<const uint4*>(smem_gen + (sc_base - smem_base)) + dt;
    // Copy the three aligned 4-byte words that hold this thread's eight scale bytes of the walker's RAW stage
    // (row offset + 8 * raw index is only 2-byte aligned); returns the byte offset of the first one inside them.
    auto fetch_scales = [&](const MxWalker& w, uint32_t slot) -> uint32_t {
      const size_t off = ((size_t)w.we * f.rows_per_expert + grow(w.rt)) * kscale + (size_t)w.kc * 2;
      const size_t al = off & ~(size_t)3;
      const uint32_t dst = my_sc + slot * (kMxDecWarps * 32 * 16);
      if (al + 12 <= scale_total) {
#pragma unroll
        for (int q = 0; q < 3; ++q)
          asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" :: "r"(dst + 4 * q), "l"(a.scales + al + 4 * q) : "memory");
      } else {                                       // the tensor's last bytes: no three aligned words inside it
        for (int q = 0; q < 12; ++q) {
          const uint8_t v = (al + q < scale_total) ? a.scales[al + q] : (uint8_t)127;
          asm volatile("st.shared.u8 [%0], %1;" :: "r"(dst + q), "r"((uint32_t)v) : "memory");
        }
      }
      return (uint32_t)(off & 3);
    };
    // The loop nest is written out (tile -> accumulator pass -> raw stage -> k-chunk) with ring cursors carried
    // incrementally: a generic per-stage walker plus run-time modulos cost ~500 instructions per stage per thread --
    // more than the decode itself (ncu: 1850 warp instructions per 4 KiB stage).
    MxWalker wf;                                     // scale prefetch cursor, one step = one raw stage
    wf.init(&f, total_tiles, NP, k_iters, kMxRawChunks);
    uint32_t sh_bits = 0;                            // 2 bits per prefetched raw stage: byte offset of its scales in the fetched words
    for (int j = 0; j < kMxScaleAhead; ++j) {
      if (wf.live) { sh_bits |= fetch_scales(wf, j) << (2 * j); wf.next(); }
      asm volatile("cp.async.commit_group;" ::: "memory");
    }
    constexpr int NW = 8 / kMxParts;                  // 32-bit words (8 codes each) per thread per stage
    static_assert(NW == 4 || NW == 8, "a decoder thread stores whole groups of 16 TMEM columns");
    const int n_raw = (k_iters + kMxRawChunks - 1) / kMxRawChunks;
    const uint32_t rx = src_row & 7;
    const uint32_t raw_row0 = raw_base + src_row * 128;
    const uint32_t a_row0 = tmem_base + kMxATmemCol + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)(4 * NW * part);
    const uint32_t sc_stride = kMxDecWarps * 32;      // uint4 per scale slot
    uint32_t ws_ = 0, wpar = 1, rs = 0, rpar = 0, slot = 0;
    for (int tile = blockIdx.x; tile < total_tiles; tile += gridDim.x) {
      const int ent = tile / f.tiles_per_expert;
      const int m_tok = f.work[ent].w;
      for (int n0 = 0; n0 < m_tok; n0 += NP) {
        for (int rk = 0; rk < n_raw; ++rk) {
          asm volatile("cp.async.wait_group %0;" :: "n"(kMxScaleAhead - 1) : "memory");
          const uint4 sw = my_sc_gen[slot * sc_stride];
          const uint32_t sh = (sh_bits & 3u) * 8u;
          sh_bits >>= 2;
          const uint32_t sc_lo = __funnelshift_r(sw.x, sw.y, sh), sc_hi = __funnelshift_r(sw.y, sw.z, sh);
          if (wf.live) { sh_bits |= fetch_scales(wf, slot) << (2 * (kMxScaleAhead - 1)); wf.next(); }
          asm volatile("cp.async.commit_group;" ::: "memory");
          if (++slot == kMxScaleAhead) slot = 0;
          mbar_wait(rfull_bar(rs), rpar);
          const uint32_t raw_row = raw_row0 + rs * kMxRawBytes;
          const int nsub = min(kMxRawChunks, k_iters - rk * kMxRawChunks);
#pragma unroll
          for (int sub = 0; sub < kMxRawChunks; ++sub) {
            if (sub < nsub) {
              const uint32_t sb = (sub < 2 ? sc_lo : sc_hi) >> (16 * (sub & 1));
              const uint32_t sbyte = (NW * part >= 4 ? (sb >> 8) : sb) & 0xffu;      // my codes lie in one 32-element block when NW <= 4
              // multiplier bits: exponent field b + 126 (= 2^(b-1), the decode's 2^126 folded in) while that is a finite
              // bf16, else b (= 2^(b-127)) and the decode multiplies by 2^126 itself
              auto mul_bits = [](uint32_t b) -> uint32_t { return (b <= 128u ? b + 126u : b) << 7; };
              const bool wide0 = (sb & 0xffu) > 128u, wide1 = ((sb >> 8) & 0xffu) > 128u, widem = sbyte > 128u;
              const uint32_t s0 = mul_bits(sb & 0xffu), s1 = mul_bits((sb >> 8) & 0xffu), sm_ = mul_bits(sbyte);
              const uint32_t p0 = s0 | (s0 << 16), p1 = s1 | (s1 << 16), pm = sm_ | (sm_ << 16);
              const __nv_bfloat162 sc0 = *reinterpret_cast<const __nv_bfloat162*>(&p0);
              const __nv_bfloat162 sc1 = *reinterpret_cast<const __nv_bfloat162*>(&p1);
              const __nv_bfloat162 scm = *reinterpret_cast<const __nv_bfloat162*>(&pm);
              // my raw bytes: logical offset 32 * sub + 4 * NW * part inside the 128-byte row (SWIZZLE_128B)
              uint32_t wd[NW];
              const uint32_t lo = 32u * sub + 4u * NW * part;
              const uint32_t addr = raw_row + ((((lo >> 4) ^ rx) << 4) | (lo & 15u));
              if (NW == 8) {
                const uint4 q0 = lds_v4(addr), q1 = lds_v4(raw_row + ((((lo >> 4) + 1) ^ rx) << 4));
                wd[0] = q0.x; wd[1 % NW] = q0.y; wd[2 % NW] = q0.z; wd[3 % NW] = q0.w;
                wd[4 % NW] = q1.x; wd[5 % NW] = q1.y; wd[6 % NW] = q1.z; wd[7 % NW] = q1.w;
              } else if (NW == 4) {
                const uint4 q0 = lds_v4(addr);
                wd[0] = q0.x; wd[1 % NW] = q0.y; wd[2 % NW] = q0.z; wd[3 % NW] = q0.w;
              } else {
                asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(wd[0]), "=r"(wd[1 % NW]) : "r"(addr));
              }
              // decode into registers, then straight into this row's TMEM lane: 4 columns (8 bf16) per word
              uint4 o[NW];
#pragma unroll
              for (int i = 0; i < NW; ++i)
                o[i] = mx_decode8(wd[i], NW == 8 ? (i < 4 ? sc0 : sc1) : scm, NW == 8 ? (i < 4 ? wide0 : wide1) : widem);
              mbar_wait(wempty_bar(ws_), wpar);
              tc_fence_after();
              const uint32_t a_addr = a_row0 + ws_ * 32u;
#pragma unroll
              for (int i = 0; i < NW; i += 4)
                tmem_st16(a_addr + 4u * i, o[i], o[(i + 1) % NW], o[(i + 2) % NW], o[(i + 3) % NW]);
              asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
              tc_fence_before();
              __syncwarp();
              if (lane == 0) mbar_arrive(wfull_bar(ws_));
              if (++ws_ == (uint32_t)S) { ws_ = 0; wpar ^= 1u; }
            }
          }
          __syncwarp();
          if (lane == 0) mbar_arrive(rempty_bar(rs));
          if (++rs == (uint32_t)RS) { rs = 0; rpar ^= 1u; }
        }
      }
    }
    asm volatile("cp.async.wait_all;" ::: "memory");
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_base), "r"(tmem_cols) : "memory");
  }
}

}  // namespace eldr
