// C ABI of the B200 decode-MoE layer (include/eldr_moe.h): argument validation, workspace carving, TMA
// descriptor construction and kernel launches.  No device allocation, no host synchronisation (except the
// *_host entry point, synchronous by contract).
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdio>
#include <cstring>
#include <atomic>
#include <mutex>

#include "eldr_moe.h"
#include "ffn_stream.cuh"
#include "ffn_umma.cuh"
#include "ffn_umma2.cuh"
#include "ffn_mx.cuh"
#include "ffn_gemv.cuh"
#include "fit_host.cuh"
#include "gate_route.cuh"
#include "gate_prefill.cuh"
#include "gate_tc.cuh"
#include "moe_fused.cuh"
#include "route_decide.cuh"
#include "route_prefill.cuh"

namespace {

using namespace eldr;

// Process-wide tuning knobs (eldr_moe_set_option).  Relaxed atomics: a call reads each knob once, so a concurrent
// set_option from another host thread changes whole calls, never half of one.
std::atomic<int> g_ffn_pair{1};   // prefill-shaped calls: cta_group::2 FFN tiles over SM pairs (ELDR_OPT_FFN_PAIR)
std::atomic<int> g_ffn_path{ELDR_FFN_TCGEN05};
std::atomic<int> g_pdl{1};
std::atomic<int> g_step_path{ELDR_STEP_AUTO};
std::atomic<int> g_ring_kb{208};
std::atomic<int> g_dp_min_rounds{1};
std::atomic<int> g_sk_split_pct{0};
std::atomic<int> g_coop{1};
std::atomic<int> g_head_first{0};
std::atomic<int> g_xs_min_np{48};
std::atomic<int> g_gate_tc{1};
std::atomic<int> g_sk_max_split{1};

// Scratch of eldr_moe_gate_topk_static (the entry point that allocates nothing): the gate logits z [T,E] fp32.  File
// scope, so every GPU that loads the library holds these bytes until the process exits.  In HOST code this name is a
// host-side stand-in, not a device address: the entry point asks cudaGetSymbolAddress for the device address, once per
// device, and hands that to the kernels.
static __device__ __align__(256) unsigned char g_static_scratch[ELDR_STATIC_SCRATCH_BYTES];

thread_local char g_err[256] = "";
thread_local int g_launches = 0;

// optional per-kernel event timing (eldr_moe_profile_enable)
thread_local bool g_prof_on = false;
thread_local cudaEvent_t g_prof_ev[ELDR_PROFILE_SLOTS + 1];
thread_local bool g_prof_ev_made = false;
thread_local int g_prof_mark[ELDR_PROFILE_SLOTS + 1];   // event index recorded before kernel slot i (-1: not run)
thread_local int g_prof_n = 0;

void prof_begin() {
  if (!g_prof_on) return;
  if (!g_prof_ev_made) {
    for (auto& e : g_prof_ev) cudaEventCreate(&e);
    g_prof_ev_made = true;
  }
  for (auto& m : g_prof_mark) m = -1;
  g_prof_n = 0;
}
// record "kernel `slot` starts here" (slot == ELDR_PROFILE_SLOTS: end of the call)
void prof_mark(int slot, cudaStream_t st) {
  if (!g_prof_on) return;
  cudaEventRecord(g_prof_ev[g_prof_n], st);
  g_prof_mark[slot] = g_prof_n++;
}

bool cuda_ok(cudaError_t e, const char* what) {
  if (e == cudaSuccess) return true;
  snprintf(g_err, sizeof(g_err), "%s: %s", what, cudaGetErrorString(e));
  return false;
}
bool launch_ok(const char* what) {
  ++g_launches;
  return cuda_ok(cudaGetLastError(), what);
}

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

constexpr int kDecodeMaxT = 1024;     // single-CTA routing (route_phases); above it the chunked routing kernels
constexpr int kPrefillMaxT = 16384;   // eldr_moe_decode_layer: largest prefill-shaped T

// Split-K slices of the prefill-shaped gate GEMM (gate_prefill.cuh): the fewest slices of at most 256 h; 0 when the
// shape does not take that path.
int gate_slices(const eldr_moe_shape_t* s, int T) {
  if (T < 2048 || s->hidden % kGpBK != 0) return 0;
  const int chunks = s->hidden / kGpBK;
  for (int c = 1; c <= 64; ++c)
    if (chunks % c == 0 && s->hidden / c <= 256) return c;
  return 0;
}
inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

int32_t check_shape(const eldr_moe_shape_t* s) {
  if (!s) return ELDR_ERR_INVALID_ARG;
  if (s->hidden < 8 || s->hidden % 8 || s->inter < 8 || s->inter % 8) return ELDR_ERR_INVALID_ARG;
  if (s->n_experts < 1 || s->n_experts > kMaxExperts) return ELDR_ERR_INVALID_ARG;
  if (s->top_k < 1 || s->top_k > s->n_experts || s->top_k > kMaxTopK) return ELDR_ERR_INVALID_ARG;
  if (s->n_shared < 0 || s->n_shared > 8) return ELDR_ERR_INVALID_ARG;
  if (s->n_layers < 1) return ELDR_ERR_INVALID_ARG;
  if (s->kv_block_size < 1 || s->kv_block_size > 127) return ELDR_ERR_INVALID_ARG;
  return ELDR_OK;
}

void make_layout(const eldr_moe_shape_t* s, int T, eldr_moe_ws_layout_t* L) {
  const size_t H = s->hidden, I = s->inter, E = s->n_experts, k = s->top_k, ns = s->n_shared;
  const size_t Tz = T > 0 ? T : 1;
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t r = o; o = align_up(o + bytes, 256); return r; };
  // epoch flags first, at a T-independent offset and size: the fused kernel keeps its generation word there
  const size_t sync_staged = ((size_t)((kFusedMaxT > (int)Tz ? kFusedMaxT : Tz) + kGateTok - 1) / kGateTok * ((E + kGateExp - 1) / kGateExp + 2) + 2) * 4;
  const size_t sync_fused = fused_sync_words((int)E, (int)ns, (int)I, (int)H) * 4;
  L->sync = take(align_up(sync_fused, 256) + sync_staged);   // [fused | staged]: never aliased (both derive epochs)
  const int zs = gate_slices(s, T);
  // prefill-shaped gate: one partial logit tensor per slice (CUDA-core split-K) or the logits + the three-term bf16
  // split of the gate weights behind them (tensor-core gate: gate_tc.cuh), whichever is larger
  const size_t z_cuda = Tz * E * 4 * (zs > 1 ? zs : 1);
  const size_t z_tc = (T >= 2048 && H % 64 == 0) ? align_up(Tz * E * 4, 1024) + 3 * E * H * 2 : 0;
  L->z = take(z_cuda > z_tc ? z_cuda : z_tc);
  L->cnt = take(align_up(E * 4, 256) + (Tz > (size_t)kDecodeMaxT ? (Tz + kRouteChunk - 1) / kRouteChunk * E * 4 : 0));   // + cnt_blk
  L->off = take((E + 1) * 4);
  L->perm = take(Tz * k * 4);
  L->pair_pos = take(Tz * k * 4);
  L->work = take((E + ns) * 16);
  L->n_work = take(4);
  L->x_perm = take((Tz * k + Tz) * H * 2);
  L->h = take(Tz * (k + ns) * I * 2);
  L->y = take(Tz * (k + ns) * H * 4);
  L->partial = take(T <= kFusedMaxT ? fused_partial_bytes(256) : 256);   // stream-K fix-up slots of the fused kernel (grid <= 256 CTAs); unused above its T limit
  L->total = o;
}

// staging block appended to the layer workspace by eldr_moe_decode_layer_host
struct HostStage { size_t x, req, blk, out, ids, w, active, n_active, total; };
void make_host_stage(const eldr_moe_shape_t* s, int T, size_t base, HostStage* S) {
  const size_t H = s->hidden, E = s->n_experts, k = s->top_k, Tz = T > 0 ? T : 1;
  size_t o = base;
  auto take = [&](size_t bytes) { size_t r = o; o = align_up(o + bytes, 256); return r; };
  S->x = take(Tz * H * 2); S->req = take(Tz * 4); S->blk = take(Tz * 4); S->out = take(Tz * H * 2);
  S->ids = take(Tz * k * 4); S->w = take(Tz * k * 4); S->active = take(E * 4); S->n_active = take(4);
  S->total = o;
}

// Per-DEVICE state: cudaFuncSetAttribute is a per-device setting and the SM count / co-residency of the persistent
// grid are properties of the device the call runs on, so everything cached here is keyed by the device ordinal.
constexpr int kMaxDevices = 64;
enum { kAttrFused = 0, kAttrRouteBig, kAttrUmma, kAttrPair, kAttrStream, kAttrRouteSims, kAttrGateLogits, kAttrGateRoute,
       kAttrRouteOnly, kAttrMx, kAttrSigLayers, kAttrGemv, kAttrGateTc, kAttrCount };
struct DevState {
  std::atomic<int> sms{0};
  std::atomic<int> fused_ok{-1};          // -1 unknown, 0 the persistent grid cannot be co-resident, 1 it can
  std::atomic<int> coop_pdl_ok{-1};       // -1 unknown, 1 cooperative + programmatic launch compose on this driver, 0 they do not
  std::atomic<void*> static_scratch{nullptr};   // device address of g_static_scratch on this device (cudaGetSymbolAddress)
  std::atomic<bool> attr[kAttrCount];
  DevState() { for (auto& a : attr) a.store(false); }
};
DevState g_dev[kMaxDevices];

int current_device() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) dev = 0;
  return dev;
}
int num_sms() {
  DevState& d = g_dev[current_device()];
  int n = d.sms.load(std::memory_order_relaxed);
  if (n == 0) {
    cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, current_device());
    if (n <= 0) n = 148;
    d.sms.store(n, std::memory_order_relaxed);
  }
  return n;
}
// cudaFuncAttributeMaxDynamicSharedMemorySize, once per (device, kernel family)
template <typename F>
bool once_per_device(int which, F&& set) {
  DevState& d = g_dev[current_device()];
  if (d.attr[which].load(std::memory_order_acquire)) return true;
  if (!set()) return false;
  d.attr[which].store(true, std::memory_order_release);
  return true;
}

// ---------------------------------------------------------------------------- TMA descriptors
typedef CUresult (*encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                    CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                    CUtensorMapFloatOOBfill);

encode_tiled_fn get_encode_fn() {
  static encode_tiled_fn fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<encode_tiled_fn>(p);
  });
  return fn;
}

// bf16 [rows, cols] row-major, box = box_rows x 64 columns (128 bytes), SWIZZLE_128B, OOB reads give zeros.
// Descriptors are pure functions of (ptr, rows, cols, box_rows); a small cache avoids re-encoding the
// static weight descriptors every step.
// The cache is a 4-way set-associative table of 1024 slots hashed on (device, pointer, shape): a 48-layer stack holds
// 96 weight descriptors plus the activations' (the 64-slot round-robin list of round 1 cycled and missed on every
// lookup there).  Within a set the oldest entry is replaced.
struct TmapKey { const void* p; uint64_t rows, cols; uint32_t box_rows, kind; int dev; };
struct TmapSlot { TmapKey k; CUtensorMap m; uint64_t stamp; bool used; };
constexpr int kTmSets = 256, kTmWays = 4;
std::mutex g_tm_mu;
TmapSlot g_tm_cache[kTmSets * kTmWays];
uint64_t g_tm_clock = 0;

inline bool tm_same(const TmapKey& a, const TmapKey& b) {
  return a.p == b.p && a.rows == b.rows && a.cols == b.cols && a.box_rows == b.box_rows && a.kind == b.kind && a.dev == b.dev;
}
inline int tm_set(const TmapKey& k) {
  uint64_t h = reinterpret_cast<uintptr_t>(k.p) * 0x9E3779B97F4A7C15ull;
  h ^= (k.rows * 0xC2B2AE3D27D4EB4Full) ^ (k.cols << 17) ^ ((uint64_t)k.box_rows << 7) ^ ((uint64_t)k.kind << 3) ^ (uint64_t)k.dev;
  h ^= h >> 29;
  return (int)(h % kTmSets);
}
bool tmap_lookup(const TmapKey& k, CUtensorMap* out) {
  std::lock_guard<std::mutex> lk(g_tm_mu);
  TmapSlot* set = g_tm_cache + tm_set(k) * kTmWays;
  for (int w = 0; w < kTmWays; ++w)
    if (set[w].used && tm_same(set[w].k, k)) {
      set[w].stamp = ++g_tm_clock;
      *out = set[w].m;
      return true;
    }
  return false;
}
void tmap_store(const TmapKey& k, const CUtensorMap& m) {
  std::lock_guard<std::mutex> lk(g_tm_mu);
  TmapSlot* set = g_tm_cache + tm_set(k) * kTmWays;
  int victim = 0;
  for (int w = 0; w < kTmWays; ++w) {
    if (!set[w].used) { victim = w; break; }
    if (set[w].stamp < set[victim].stamp) victim = w;
  }
  set[victim].k = k;
  set[victim].m = m;
  set[victim].stamp = ++g_tm_clock;
  set[victim].used = true;
}

// bf16 [rows, cols] row-major, box = box_rows x 64 columns (128 bytes), SWIZZLE_128B, OOB reads give zeros.
bool make_tmap(CUtensorMap* out, const void* ptr, uint64_t rows, uint64_t cols, uint32_t box_rows) {
  const TmapKey key{ptr, rows, cols, box_rows, 2, current_device()};
  if (tmap_lookup(key, out)) return true;
  encode_tiled_fn fn = get_encode_fn();
  if (!fn) { snprintf(g_err, sizeof(g_err), "cuTensorMapEncodeTiled entry point not found"); return false; }
  cuuint64_t gdim[2] = {cols, rows};
  cuuint64_t gstride[1] = {cols * 2};
  cuuint32_t box[2] = {64, box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(ptr), gdim, gstride, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { snprintf(g_err, sizeof(g_err), "cuTensorMapEncodeTiled failed: %d", (int)r); return false; }
  tmap_store(key, *out);
  return true;
}

// uint8 [rows, row_bytes] row-major, box = box_rows x 128 bytes, SWIZZLE_128B (packed MXFP4 codes: 256 codes per row per box)
bool make_tmap_u8(CUtensorMap* out, const void* ptr, uint64_t rows, uint64_t row_bytes, uint32_t box_rows) {
  const TmapKey key{ptr, rows, row_bytes, box_rows, 8, current_device()};
  if (tmap_lookup(key, out)) return true;
  encode_tiled_fn fn = get_encode_fn();
  if (!fn) { snprintf(g_err, sizeof(g_err), "cuTensorMapEncodeTiled entry point not found"); return false; }
  cuuint64_t gdim[2] = {row_bytes, rows};
  cuuint64_t gstride[1] = {row_bytes};
  cuuint32_t box[2] = {128, box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void*>(ptr), gdim, gstride, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { snprintf(g_err, sizeof(g_err), "cuTensorMapEncodeTiled(u8) failed: %d", (int)r); return false; }
  tmap_store(key, *out);
  return true;
}

// w13 [n_exp, 2I, H] viewed as 5-D (col, row-in-16, branch{w1,w3}, 16-row group, expert) so that ONE box of
// (64 cols, 16 rows, 2 branches, 4 groups) lands in shared memory as 4 x [16 rows of w1 | same 16 rows of w3].
bool make_tmap_w13_5d(CUtensorMap* out, const void* ptr, uint64_t n_exp, uint64_t I, uint64_t H) {
  // (I is part of the key: two weight tensors of the same total row count and different I that the allocator placed at
  // the same address -- one freed, the next allocated -- must not share a descriptor: found by a fuzz run)
  const TmapKey key{ptr, n_exp * 2 * I, H | (I << 32), 16, 5, current_device()};
  if (tmap_lookup(key, out)) return true;
  encode_tiled_fn fn = get_encode_fn();
  if (!fn) { snprintf(g_err, sizeof(g_err), "cuTensorMapEncodeTiled entry point not found"); return false; }
  cuuint64_t gdim[5] = {H, 16, 2, I / 16, n_exp};
  cuuint64_t gstride[4] = {H * 2, I * H * 2, 16 * H * 2, 2 * I * H * 2};
  cuuint32_t box[5] = {64, 16, 2, 4, 1};
  cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  CUresult r = fn(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 5, const_cast<void*>(ptr), gdim, gstride, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { snprintf(g_err, sizeof(g_err), "cuTensorMapEncodeTiled(5d) failed: %d", (int)r); return false; }
  tmap_store(key, *out);
  return true;
}

// Launch with the programmatic-dependent-launch attribute: the kernel may start (prologue: barrier init, TMEM
// allocation, descriptor prefetch) while its predecessor drains; it calls griddepcontrol.wait before touching
// the predecessor's outputs.  Profiling events between kernels disable the overlap by construction.
template <typename... KArgs, typename... Args>
cudaError_t launch_dep(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = (g_pdl.load() && !g_prof_on) ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// Same, as thread-block clusters of two CTAs (an SM pair for tcgen05 cta_group::2); grid.x must be even.
template <typename... KArgs, typename... Args>
cudaError_t launch_dep_pair(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 2;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = (g_pdl.load() && !g_prof_on) ? 2 : 1;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// The fused step: cooperative launch (all CTAs co-resident or the launch fails) plus, when allowed, the
// programmatic-dependent-launch attribute.  Whether the two attributes compose is found out once per device: if the
// first launch with both is rejected as an invalid configuration, the kernel is launched cooperatively without PDL
// from then on.
template <typename... KArgs, typename... Args>
cudaError_t launch_fused(void (*kernel)(KArgs...), DevState& dv, dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeCooperative;
  attr[0].val.cooperative = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  const bool want_pdl = g_pdl.load() && !g_prof_on;
  if (!g_coop.load()) {
    // ELDR_OPT_COOPERATIVE = 0: plain launch (+ PDL).  For a GPU this process has to itself: nothing else can hold an
    // SM, the occupancy check above has shown that the grid fits, and consecutive steps overlap their launch latency.
    cfg.attrs = attr + 1;
    cfg.numAttrs = want_pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
  }
  int both = dv.coop_pdl_ok.load(std::memory_order_relaxed);
  if (want_pdl && both != 0) {
    cfg.numAttrs = 2;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
    if (e == cudaSuccess || both == 1) { dv.coop_pdl_ok.store(1, std::memory_order_relaxed); return e; }
    if (e != cudaErrorInvalidValue && e != cudaErrorNotSupported && e != cudaErrorInvalidConfiguration) return e;
    cudaGetLastError();
    dv.coop_pdl_ok.store(0, std::memory_order_relaxed);
  }
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

template <typename K>
bool set_smem(K kernel, size_t bytes) {
  return cuda_ok(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes),
                 "cudaFuncSetAttribute(smem)");
}

int32_t launch_gate_logits(const eldr_moe_shape_t* s, int T, const eldr_bf16* x, const float* gate_w,
                           const float* gate_bias, float* z, cudaStream_t st) {
  const size_t smem = (size_t)kGateTok * s->hidden * 2;
  if (smem > 200 * 1024) return ELDR_ERR_UNSUPPORTED;
  if (smem > 48 * 1024 && !once_per_device(kAttrGateLogits, [] { return set_smem(gate_logits_kernel, 200 * 1024); })) return ELDR_ERR_CUDA;
  dim3 grid((s->n_experts + kGateExp - 1) / kGateExp, (T + kGateTok - 1) / kGateTok);
  gate_logits_kernel<<<grid, 256, smem, st>>>(x, gate_w, gate_bias, z, T, s->hidden, s->n_experts);
  return launch_ok("gate_logits_kernel") ? ELDR_OK : ELDR_ERR_CUDA;
}

// a1-a3 as separate launches (eldr_moe_gate_topk and the prefill-shaped layer): logits, then warp top-k + signature.
int32_t launch_gate_topk(const eldr_moe_shape_t* s, int T, const eldr_bf16* x, const float* gate_w,
                         const float* gate_bias, float* z, size_t z_bytes, const TopkArgs& a, cudaStream_t st) {
  // prefill-shaped, H a multiple of 64: the tensor-core gate (three exact bf16 terms per fp32 weight, 256-wide K slices
  // summed in fp32: gate_tc.cuh); the three-term split of the weights lives behind z in the workspace
  const size_t z_sz = align_up((size_t)T * s->n_experts * 4, 1024);
  const size_t split_sz = (size_t)3 * s->n_experts * s->hidden * 2;
  if (g_gate_tc.load() && T >= 2048 && s->hidden % 64 == 0 && z_bytes >= z_sz + split_sz) {
    uint16_t* wsplit = reinterpret_cast<uint16_t*>(reinterpret_cast<uint8_t*>(z) + z_sz);
    const int n = s->n_experts * s->hidden;
    gate_split_kernel<<<(n + 255) / 256, 256, 0, st>>>(gate_w, wsplit, n);
    if (!launch_ok("gate_split_kernel")) return ELDR_ERR_CUDA;
    CUtensorMap tm_x, tm_w;
    if (!make_tmap(&tm_x, x, (uint64_t)T, s->hidden, kGtcTok)) return ELDR_ERR_CUDA;
    if (!make_tmap(&tm_w, wsplit, (uint64_t)3 * s->n_experts, s->hidden, kGtcExp)) return ELDR_ERR_CUDA;
    if (!once_per_device(kAttrGateTc, [] { return set_smem(gate_logits_tc_kernel, kGtcSmemBytes); })) return ELDR_ERR_CUDA;
    launch_dep(gate_logits_tc_kernel, dim3((s->n_experts + kGtcExp - 1) / kGtcExp, (T + kGtcTok - 1) / kGtcTok), dim3(kGtcThreads),
               (size_t)kGtcSmemBytes, st, tm_x, tm_w, gate_bias, z, T, s->hidden, s->n_experts);
    if (!launch_ok("gate_logits_tc_kernel")) return ELDR_ERR_CUDA;
    topk_kernel<<<(T + 7) / 8, 256, 0, st>>>(a);
    return launch_ok("topk_kernel") ? ELDR_OK : ELDR_ERR_CUDA;
  }
  const int S = gate_slices(s, T);
  if (S > 0 && z_bytes >= (size_t)S * T * s->n_experts * 4) {
    // prefill-shaped: register-tiled fp32 GEMM, split-K into the fewest slices of at most 256 h (accuracy, see
    // gate_prefill.cuh); taken when the workspace holds the S partial logit tensors
    gate_logits_tiled_kernel<<<dim3((T + kGpBM - 1) / kGpBM, (s->n_experts + kGpBN - 1) / kGpBN, S), kGpThreads, 0, st>>>(
        x, gate_w, gate_bias, z, T, s->hidden, s->n_experts, s->hidden / S);
    if (!launch_ok("gate_logits_tiled_kernel")) return ELDR_ERR_CUDA;
    topk_splitk_kernel<<<(T + 7) / 8, 256, 0, st>>>(a, z, S);
    return launch_ok("topk_splitk_kernel") ? ELDR_OK : ELDR_ERR_CUDA;
  }
  const int32_t rc = launch_gate_logits(s, T, x, gate_w, gate_bias, z, st);
  if (rc != ELDR_OK) return rc;
  topk_kernel<<<(T + 7) / 8, 256, 0, st>>>(a);
  return launch_ok("topk_kernel") ? ELDR_OK : ELDR_ERR_CUDA;
}

}  // namespace

extern "C" {

#ifdef ELDR_TRACE
void eldr_debug_read_trace(unsigned long long* h) {
  cudaDeviceSynchronize();
  cudaMemcpyFromSymbol(h, eldr::g_trace, sizeof(unsigned long long) * 4096 * 16);
}
void eldr_debug_clear_trace(void) {
  cudaDeviceSynchronize();
  void* p = nullptr;
  cudaGetSymbolAddress(&p, eldr::g_trace);
  cudaMemset(p, 0, sizeof(unsigned long long) * 4096 * 16);
}
#endif

const char* eldr_status_string(int32_t st) {
  switch (st) {
    case ELDR_OK: return "ok";
    case ELDR_ERR_INVALID_ARG: return "invalid argument";
    case ELDR_ERR_UNSUPPORTED: return "unsupported shape";
    case ELDR_ERR_WORKSPACE_SMALL: return "workspace too small";
    case ELDR_ERR_CUDA: return "CUDA error";
    default: return "unknown status";
  }
}

const char* eldr_last_cuda_error(void) { return g_err; }

int32_t eldr_moe_set_option(int32_t key, int32_t value) {
  if (key == ELDR_OPT_FFN_PATH && (value == ELDR_FFN_MMA_SYNC || value == ELDR_FFN_TCGEN05 || value == ELDR_FFN_GEMV)) {
    g_ffn_path = value;
    return ELDR_OK;
  }
  if (key == ELDR_OPT_FFN_PAIR && value >= 0 && value <= 2) {
    g_ffn_pair = value;
    return ELDR_OK;
  }
  if (key == ELDR_OPT_PDL && (value == 0 || value == 1)) {
    g_pdl = value;
    return ELDR_OK;
  }
  if (key == ELDR_OPT_STEP_PATH && (value == ELDR_STEP_STAGED || value == ELDR_STEP_FUSED || value == ELDR_STEP_AUTO)) {
    g_step_path = value;
    return ELDR_OK;
  }
  if (key == ELDR_OPT_RING_KB && value >= 32 && value <= 208) {
    g_ring_kb = value;
    return ELDR_OK;
  }
  if (key == ELDR_OPT_DP_MIN_ROUNDS && value >= 1 && value <= (1 << 20)) {
    g_dp_min_rounds = value;
    return ELDR_OK;
  }
  if (key == ELDR_OPT_SK_MAX_SPLIT && value >= 0 && value <= 64) {
    g_sk_max_split = value;
    return ELDR_OK;
  }
  if (key == ELDR_OPT_GATE_TC && (value == 0 || value == 1)) {
    g_gate_tc = value;
    return ELDR_OK;
  }
  if (key == ELDR_OPT_XS_MIN_NP && value >= 16 && value <= 144) {
    g_xs_min_np = value;
    return ELDR_OK;
  }
  if (key == ELDR_OPT_HEAD_FIRST && (value == 0 || value == 1)) {
    g_head_first = value;
    return ELDR_OK;
  }
  if (key == ELDR_OPT_COOPERATIVE && (value == 0 || value == 1)) {
    g_coop = value;
    return ELDR_OK;
  }
  if (key == ELDR_OPT_SK_SPLIT_PCT && value >= 0 && value <= 100) {
    g_sk_split_pct = value;
    return ELDR_OK;
  }
  return ELDR_ERR_INVALID_ARG;
}

int32_t eldr_moe_profile_enable(int32_t on) {
  g_prof_on = on != 0;
  return ELDR_OK;
}

int32_t eldr_moe_profile_read(float* h_ms) {
  if (!h_ms) return ELDR_ERR_INVALID_ARG;
  for (int i = 0; i < ELDR_PROFILE_SLOTS; ++i) h_ms[i] = 0.f;
  if (!g_prof_ev_made || g_prof_n < 2 || g_prof_mark[ELDR_PROFILE_SLOTS] < 0) return ELDR_ERR_INVALID_ARG;
  if (!cuda_ok(cudaEventSynchronize(g_prof_ev[g_prof_mark[ELDR_PROFILE_SLOTS]]), "profile sync")) return ELDR_ERR_CUDA;
  for (int i = 0; i < ELDR_PROFILE_SLOTS; ++i) {
    if (g_prof_mark[i] < 0) continue;
    // the next recorded event after this kernel's start marks its end
    if (!cuda_ok(cudaEventElapsedTime(&h_ms[i], g_prof_ev[g_prof_mark[i]], g_prof_ev[g_prof_mark[i] + 1]), "profile elapsed"))
      return ELDR_ERR_CUDA;
  }
  return ELDR_OK;
}
int32_t eldr_moe_last_launch_count(void) { return g_launches; }

size_t eldr_moe_workspace_bytes(const eldr_moe_shape_t* shape, int32_t max_T) {
  if (check_shape(shape) != ELDR_OK || max_T < 0) return 0;
  eldr_moe_ws_layout_t L;
  make_layout(shape, max_T, &L);
  return L.total;
}

size_t eldr_moe_workspace_bytes_host(const eldr_moe_shape_t* shape, int32_t max_T) {
  if (check_shape(shape) != ELDR_OK || max_T < 0) return 0;
  eldr_moe_ws_layout_t L;
  make_layout(shape, max_T, &L);
  HostStage S;
  make_host_stage(shape, max_T, L.total, &S);
  return S.total;
}

int32_t eldr_moe_workspace_layout(const eldr_moe_shape_t* shape, int32_t T, eldr_moe_ws_layout_t* layout) {
  if (check_shape(shape) != ELDR_OK || T < 0 || !layout) return ELDR_ERR_INVALID_ARG;
  make_layout(shape, T, layout);
  return ELDR_OK;
}

int32_t eldr_moe_gate_topk(const eldr_moe_shape_t* s, int32_t layer, int32_t T, const eldr_bf16* x,
                           const float* gate_w, const float* gate_bias, int32_t* topk_ids, float* topk_w,
                           const int32_t* token_req, const int32_t* token_block, int32_t* sig_req,
                           int8_t* sig_block, void* workspace, size_t workspace_bytes, eldr_stream_t stream) {
  g_launches = 0;
  int32_t rc = check_shape(s);
  if (rc != ELDR_OK) return rc;
  if (T < 0 || layer < 0 || layer >= s->n_layers) return ELDR_ERR_INVALID_ARG;
  if (T == 0) return ELDR_OK;
  if (!x || !gate_w || !topk_ids || !topk_w || !workspace) return ELDR_ERR_INVALID_ARG;
  if (!aligned16(x) || !aligned16(gate_w) || !aligned16(workspace) || !aligned16(sig_block)) return ELDR_ERR_INVALID_ARG;
  if (workspace_bytes < align_up((size_t)T * s->n_experts * 4, 256)) return ELDR_ERR_WORKSPACE_SMALL;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  float* z = static_cast<float*>(workspace);
  TopkArgs a{z, topk_ids, topk_w, token_req, token_block, sig_req, sig_block,
             T, s->n_experts, s->top_k, s->n_layers, layer, s->renormalize};
  return launch_gate_topk(s, T, x, gate_w, gate_bias, z, workspace_bytes, a, st);
}

int32_t eldr_moe_gate_topk_static(const eldr_moe_shape_t* s, int32_t layer, int32_t T, const eldr_bf16* x,
                                  const float* gate_w, const float* gate_bias, int32_t* topk_ids, float* topk_w,
                                  const int32_t* token_req, const int32_t* token_block, int32_t* sig_req,
                                  int8_t* sig_block, eldr_stream_t stream) {
  g_launches = 0;
  int32_t rc = check_shape(s);
  if (rc != ELDR_OK) return rc;
  if (T < 0 || layer < 0 || layer >= s->n_layers) return ELDR_ERR_INVALID_ARG;
  if (T == 0) return ELDR_OK;
  if (!x || !gate_w || !topk_ids || !topk_w) return ELDR_ERR_INVALID_ARG;
  if (!aligned16(x) || !aligned16(gate_w) || !aligned16(sig_block)) return ELDR_ERR_INVALID_ARG;
  const size_t z_bytes = (size_t)T * s->n_experts * 4;
  if (z_bytes > (size_t)ELDR_STATIC_SCRATCH_BYTES) {
    snprintf(g_err, sizeof(g_err), "eldr_moe_gate_topk_static: T * n_experts * 4 = %zu bytes of logits exceed the static scratch (%u bytes)",
             z_bytes, (unsigned)ELDR_STATIC_SCRATCH_BYTES);
    return ELDR_ERR_WORKSPACE_SMALL;
  }
  // device address of the file-scope array: resolved once per device, with that device current (it is: the call runs
  // on the current device).  No allocation: the array is part of the loaded module.
  DevState& dv = g_dev[current_device()];
  void* scratch = dv.static_scratch.load(std::memory_order_acquire);
  if (!scratch) {
    if (!cuda_ok(cudaGetSymbolAddress(&scratch, g_static_scratch), "cudaGetSymbolAddress(g_static_scratch)")) return ELDR_ERR_CUDA;
    dv.static_scratch.store(scratch, std::memory_order_release);
  }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  float* z = static_cast<float*>(scratch);
  TopkArgs a{z, topk_ids, topk_w, token_req, token_block, sig_req, sig_block,
             T, s->n_experts, s->top_k, s->n_layers, layer, s->renormalize};
  // z_bytes = one logit tensor: every element of z[0 .. T*E) is written by the logits kernel before the top-k reads it,
  // so nothing left by an earlier call is ever read and nothing has to be cleared
  return launch_gate_topk(s, T, x, gate_w, gate_bias, z, z_bytes, a, st);
}

int32_t eldr_moe_decode_layer(const eldr_moe_shape_t* s, int32_t layer, int32_t T, const eldr_bf16* x,
                              const float* gate_w, const float* gate_bias, const eldr_bf16* w13,
                              const eldr_bf16* w2, const eldr_bf16* shared_w13, const eldr_bf16* shared_w2,
                              eldr_bf16* out, int32_t* topk_ids, float* topk_w, int32_t force_routing,
                              int32_t* active_experts, int32_t* n_active, const int32_t* token_req,
                              const int32_t* token_block, int32_t* sig_req, int8_t* sig_block,
                              void* workspace, size_t workspace_bytes, eldr_stream_t stream) {
  g_launches = 0;
  int32_t rc = check_shape(s);
  if (rc != ELDR_OK) return rc;
  if (T < 0 || layer < 0 || layer >= s->n_layers) return ELDR_ERR_INVALID_ARG;
  if (T == 0) return ELDR_OK;
  if (T > kPrefillMaxT) return ELDR_ERR_UNSUPPORTED;
  if (!x || !w13 || !w2 || !out || !topk_ids || !topk_w || !active_experts || !n_active || !workspace)
    return ELDR_ERR_INVALID_ARG;
  if (!force_routing && !gate_w) return ELDR_ERR_INVALID_ARG;
  if (s->n_shared > 0 && (!shared_w13 || !shared_w2)) return ELDR_ERR_INVALID_ARG;
  if (!aligned16(x) || !aligned16(gate_w) || !aligned16(w13) || !aligned16(w2) || !aligned16(shared_w13) ||
      !aligned16(shared_w2) || !aligned16(out) || !aligned16(workspace) || !aligned16(sig_block))
    return ELDR_ERR_INVALID_ARG;
  eldr_moe_ws_layout_t L;
  make_layout(s, T, &L);
  if (workspace_bytes < L.total) return ELDR_ERR_WORKSPACE_SMALL;

  cudaStream_t st = static_cast<cudaStream_t>(stream);
  uint8_t* ws = static_cast<uint8_t*>(workspace);
  const int H = s->hidden, I = s->inter, E = s->n_experts, k = s->top_k, ns = s->n_shared;
  float* z = reinterpret_cast<float*>(ws + L.z);
  int32_t* perm = reinterpret_cast<int32_t*>(ws + L.perm);
  int32_t* pair_pos = reinterpret_cast<int32_t*>(ws + L.pair_pos);
  int4* work = reinterpret_cast<int4*>(ws + L.work);
  int32_t* n_work = reinterpret_cast<int32_t*>(ws + L.n_work);
  uint16_t* x_perm = reinterpret_cast<uint16_t*>(ws + L.x_perm);
  uint16_t* hbuf = reinterpret_cast<uint16_t*>(ws + L.h);
  float* ybuf = reinterpret_cast<float*>(ws + L.y);

  // ------------------------------------------------------------------ whole step in one persistent launch
  // AUTO = the one-launch step whenever the shape allows it.  (Round 1 sent layers with shared experts and T >= 224 to
  // the staged path; with the expert-sorted copy of x and the shared experts first in the work list the one-launch
  // step is faster there too: config-5 shape, T = 256: 223.6 vs 258.6 us.)
  const int step_path = g_step_path.load();
  const bool want_fused = step_path == ELDR_STEP_FUSED || step_path == ELDR_STEP_AUTO;
  const int ffn_path = g_ffn_path.load();
  if (want_fused && ffn_path == ELDR_FFN_TCGEN05 && H % 64 == 0 && I % 64 == 0 &&
      T <= kFusedMaxT && num_sms() <= 256) {
    FusedArgs fa;
    fa.x = x; fa.gate_w = gate_w; fa.gate_bias = gate_bias;
    fa.tk = TopkArgs{z, topk_ids, topk_w, token_req, token_block, sig_req, sig_block,
                     T, E, k, s->n_layers, layer, s->renormalize};
    fa.force_routing = force_routing ? 1 : 0;
    fa.n_shared = ns; fa.H = H; fa.I = I;
    fa.cnt = reinterpret_cast<int32_t*>(ws + L.cnt);
    fa.off = reinterpret_cast<int32_t*>(ws + L.off);
    fa.perm = perm; fa.pair_pos = pair_pos; fa.work = work; fa.n_work = n_work;
    fa.active = active_experts; fa.n_active = n_active;
    fa.sync = reinterpret_cast<uint32_t*>(ws + L.sync);
    fa.idt = reinterpret_cast<unsigned long long*>(fa.sync + fused_idt_word_offset(E, ns, I, H));
    fa.wtag = reinterpret_cast<unsigned long long*>(fa.sync + fused_wtag_word_offset(E, ns, I, H));
    fa.hbuf = hbuf; fa.ybuf = ybuf; fa.out = out;
    fa.partial = reinterpret_cast<float*>(ws + L.partial);
    const size_t smem_max = 227 * 1024;
    const size_t fixed = fused_smem_fixed_bytes(E, ns, T, k);
    const int gate_tok = T <= 64 ? 8 : (T <= 128 ? 16 : 32);      // gate tile height: one round of tiles over the grid
    // the gate tile borrows the ring's area: x rows, and for the wide tiles the eight fp32 gate rows too
    const size_t gate_area_wide = (size_t)gate_tok * H * 2 + (size_t)kGateExp * H * 4;
    const bool gate_wide8 = gate_tok == 8 && fixed < smem_max && gate_area_wide <= (smem_max - fixed) / 1024 * 1024;
    const size_t gate_area = (gate_tok > 8 || gate_wide8) ? gate_area_wide : (size_t)gate_tok * H * 2;
    const size_t min_area = (size_t)3 * (kUmmaWBytes + kNPCap * 128) > gate_area ? (size_t)3 * (kUmmaWBytes + kNPCap * 128) : gate_area;
    fa.stage_area = fixed < smem_max ? (int)((smem_max - fixed) / 1024 * 1024) : 0;
    fa.ring_bytes = g_ring_kb.load() * 1024;
    fa.dp_min_rounds = g_dp_min_rounds.load();
    fa.sk_split_pct = g_sk_split_pct.load();
    fa.head_first = g_head_first.load();
    fa.xs_min_np = g_xs_min_np.load();
    fa.sk_max_split = g_sk_max_split.load();
    fa.xs = x_perm;
    const size_t smem = fixed + fa.stage_area;
    if ((size_t)fa.stage_area >= min_area) {
      CUtensorMap tm_w13, tm_sw13, tm_w2, tm_sw2, tm_x, tm_xs, tm_h;
      if (!make_tmap(&tm_x, x, (uint64_t)T, H, 1)) return ELDR_ERR_CUDA;                       // gather4: 1-row box
      if (!make_tmap(&tm_xs, x_perm, (uint64_t)T * k + (ns ? T : 0), H, 16)) return ELDR_ERR_CUDA;   // wide batches: expert-sorted copy
      if (!make_tmap(&tm_h, hbuf, (uint64_t)T * (k + ns), I, 16)) return ELDR_ERR_CUDA;
      if (!make_tmap_w13_5d(&tm_w13, w13, E, I, H)) return ELDR_ERR_CUDA;
      if (!make_tmap(&tm_w2, w2, (uint64_t)E * H, I, 128)) return ELDR_ERR_CUDA;
      if (ns) {
        if (!make_tmap_w13_5d(&tm_sw13, shared_w13, ns, I, H)) return ELDR_ERR_CUDA;
        if (!make_tmap(&tm_sw2, shared_w2, (uint64_t)ns * H, I, 128)) return ELDR_ERR_CUDA;
      } else {
        tm_sw13 = tm_w13;
        tm_sw2 = tm_w2;
      }
      if (!once_per_device(kAttrFused, [] {
            return set_smem(moe_fused_kernel<8, true>, 227 * 1024) && set_smem(moe_fused_kernel<8, false>, 227 * 1024) &&
                   set_smem(moe_fused_kernel<16, true>, 227 * 1024) && set_smem(moe_fused_kernel<32, true>, 227 * 1024);
          })) return ELDR_ERR_CUDA;
      auto kern = gate_tok == 8 ? (gate_wide8 ? moe_fused_kernel<8, true> : moe_fused_kernel<8, false>)
                                : (gate_tok == 16 ? moe_fused_kernel<16, true> : moe_fused_kernel<32, true>);
      // The persistent grid's CTAs wait on one another (tile flags, tagged ids, h / y flags): they must all be
      // resident.  (1) Once per device: the occupancy calculator must grant one CTA of this size on every SM, else the
      // call takes the staged path (no grid-wide waits there).  (2) Every launch is a COOPERATIVE launch: the driver
      // starts the grid only when all of its CTAs can be co-resident -- also next to kernels of other streams or
      // under an SM partition (MPS, green contexts) -- and fails the launch otherwise instead of letting resident CTAs
      // spin on CTAs that have no SM.
      DevState& dv = g_dev[current_device()];
      int fused_ok = dv.fused_ok.load(std::memory_order_relaxed);
      if (fused_ok < 0) {
        int per_sm = 0;
        if (!cuda_ok(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kFusedThreads, 227 * 1024), "occupancy(moe_fused_kernel)"))
          return ELDR_ERR_CUDA;
        int coop = 0;
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, current_device());
        fused_ok = (per_sm >= 1 && coop) ? 1 : 0;
        dv.fused_ok.store(fused_ok, std::memory_order_relaxed);
      }
      if (fused_ok == 1) {
        prof_begin();
        prof_mark(0, st);
        const cudaError_t le = launch_fused(kern, dv, dim3(num_sms()), dim3(kFusedThreads), smem, st, tm_w13, tm_sw13, tm_w2, tm_sw2, tm_x, tm_xs, tm_h, fa);
        if (le == cudaErrorCooperativeLaunchTooLarge) {
          // the device cannot hold the grid right now (partitioned SMs): not an error of the call -- staged path
          cudaGetLastError();
          if (g_step_path.load() == ELDR_STEP_FUSED) { snprintf(g_err, sizeof(g_err), "moe_fused_kernel: grid cannot be co-resident"); return ELDR_ERR_UNSUPPORTED; }
        } else {
          ++g_launches;
          if (!cuda_ok(le, "moe_fused_kernel") || !cuda_ok(cudaGetLastError(), "moe_fused_kernel")) return ELDR_ERR_CUDA;
          prof_mark(ELDR_PROFILE_SLOTS, st);
          return ELDR_OK;
        }
      } else if (g_step_path.load() == ELDR_STEP_FUSED) {
        snprintf(g_err, sizeof(g_err), "moe_fused_kernel: one CTA per SM is not available on this device");
        return ELDR_ERR_UNSUPPORTED;
      }
    }
  }

  prof_begin();
  RouteArgs ra;
  ra.tk = TopkArgs{z, topk_ids, topk_w, token_req, token_block, sig_req, sig_block,
                   T, E, k, s->n_layers, layer, s->renormalize};
  ra.force_routing = force_routing ? 1 : 0;
  ra.n_shared = ns;
  ra.H = H;
  ra.cnt = reinterpret_cast<int32_t*>(ws + L.cnt);
  ra.off = reinterpret_cast<int32_t*>(ws + L.off);
  ra.perm = perm;
  ra.pair_pos = pair_pos;
  ra.work = work;
  ra.n_work = n_work;
  ra.active = active_experts;
  ra.n_active = n_active;
  const int W = (T + 31) / 32;
  const size_t route_smem = (size_t)E * W * 8 + (size_t)(2 * E + 1) * 4;
  if (T > kDecodeMaxT) {
    // prefill-shaped: gate GEMM + top-k/signature as their own launches, then the chunked
    // counting sort (route_prefill.cuh)
    if (!force_routing) {
      prof_mark(0, st);
      rc = launch_gate_topk(s, T, x, gate_w, gate_bias, z, L.cnt - L.z, ra.tk, st);
      if (rc != ELDR_OK) return rc;
    }
    RouteBigArgs rb{ra, reinterpret_cast<int32_t*>(ws + L.cnt + align_up((size_t)E * 4, 256)), force_routing ? 1 : 0};
    const int n_chunks = (T + kRouteChunk - 1) / kRouteChunk;
    const size_t big_smem = route_big_smem_bytes(E);
    if (!once_per_device(kAttrRouteBig, [] {
          return set_smem(route_count_kernel, route_big_smem_bytes(kMaxExperts)) &&
                 set_smem(route_scatter_kernel, route_big_smem_bytes(kMaxExperts));
        })) return ELDR_ERR_CUDA;
    prof_mark(1, st);
    route_count_kernel<<<n_chunks, kRouteBigThreads, big_smem, st>>>(rb);
    if (!launch_ok("route_count_kernel")) return ELDR_ERR_CUDA;
    route_scatter_kernel<<<n_chunks, kRouteBigThreads, big_smem, st>>>(rb);
    if (!launch_ok("route_scatter_kernel")) return ELDR_ERR_CUDA;
  } else if (!force_routing) {
    // a1-a4 in one launch: gate GEMV tiles; last CTA of a token group runs its top-k (+signature);
    // last group runs the permutation / union compaction
    GateRouteArgs ga;
    ga.x = x; ga.gate_w = gate_w; ga.gate_bias = gate_bias; ga.r = ra;
    ga.sync = reinterpret_cast<uint32_t*>(ws + L.sync + align_up(fused_sync_words(E, ns, I, H) * 4, 256));
    size_t smem = (size_t)kGateTok * H * 2;
    if (route_smem > smem) smem = route_smem;
    if (smem > 200 * 1024) return ELDR_ERR_UNSUPPORTED;
    if (smem > 48 * 1024 && !once_per_device(kAttrGateRoute, [] { return set_smem(gate_topk_route_kernel, 200 * 1024); })) return ELDR_ERR_CUDA;
    dim3 grid((E + kGateExp - 1) / kGateExp, (T + kGateTok - 1) / kGateTok);
    prof_mark(0, st);
    gate_topk_route_kernel<<<grid, 256, smem, st>>>(ga);
    if (!launch_ok("gate_topk_route_kernel")) return ELDR_ERR_CUDA;
  } else {
    if (route_smem > 48 * 1024 && !once_per_device(kAttrRouteOnly, [] { return set_smem(route_only_kernel, 200 * 1024); })) return ELDR_ERR_CUDA;
    prof_mark(1, st);
    route_only_kernel<<<1, 1024, route_smem, st>>>(ra);
    if (!launch_ok("route_only_kernel")) return ELDR_ERR_CUDA;
  }
  // gather token rows in expert-sorted order (+ plain copy for the shared experts)
  const int x_rows = T * k + (ns ? T : 0);
  const int out_rows = T * (k + ns);
  // (Gathering inside the w1/w3 kernel by TMA tile::gather4, as the fused decode kernel does, was measured for the
  // prefill-shaped calls and rejected: 256 single-row requests per stage instead of four boxes made w1/w3 3.7x slower.)
  prof_mark(2, st);
  launch_dep(gather_x_kernel, dim3((x_rows + 7) / 8), dim3(256), 0, st, x, perm, x_perm, T, H, k, x_rows, 0);
  if (!launch_ok("gather_x_kernel")) return ELDR_ERR_CUDA;

  // a5/a6: grouped SwiGLU FFN over the active experts
  const int max_work = (E < T * k ? E : T * k) + ns;
  FfnArgs f13{work, n_work, E, H, 2 * I, I, H, I / 64, hbuf, nullptr};
  FfnArgs f2{work, n_work, E, I, H, I, H, (H + 127) / 128, nullptr, ybuf};
  const int sms = num_sms();
  int g13 = max_work * f13.tiles_per_expert; if (g13 > sms) g13 = sms;
  int g2 = max_work * f2.tiles_per_expert; if (g2 > sms) g2 = sms;
  if (ffn_path == ELDR_FFN_GEMV) {
    // CUDA-core GEMV path (comparison path for tiny tokens-per-expert counts: profiles/r2_gemv_vs_tcgen05.md)
    const size_t smem13 = (size_t)kGemvTok * H * 2, smem2 = (size_t)kGemvTok * I * 2;
    if (smem13 > 200 * 1024 || smem2 > 200 * 1024) return ELDR_ERR_UNSUPPORTED;
    if ((smem13 > 48 * 1024 || smem2 > 48 * 1024) && !once_per_device(kAttrGemv, [] {
          return set_smem(ffn_gemv_kernel<0>, 200 * 1024) && set_smem(ffn_gemv_kernel<1>, 200 * 1024);
        })) return ELDR_ERR_CUDA;
    f13.tiles_per_expert = (I + 63) / 64;
    g13 = max_work * f13.tiles_per_expert; if (g13 > sms) g13 = sms;
    prof_mark(3, st);
    launch_dep(ffn_gemv_kernel<0>, dim3(g13), dim3(kGemvThreads), smem13, st, w13, shared_w13, x_perm, f13);
    if (!launch_ok("ffn_gemv_kernel<w13>")) return ELDR_ERR_CUDA;
    prof_mark(4, st);
    launch_dep(ffn_gemv_kernel<1>, dim3(g2), dim3(kGemvThreads), smem2, st, w2, shared_w2, hbuf, f2);
    if (!launch_ok("ffn_gemv_kernel<w2>")) return ELDR_ERR_CUDA;
  } else if (H % 64 == 0 && I % 64 == 0 && ffn_path == ELDR_FFN_TCGEN05) {
    // tcgen05 + TMEM path: weights are the M=128 operand, the expert's tokens the N operand
    CUtensorMap tm_w13, tm_sw13, tm_x16, tm_x64, tm_w2, tm_sw2, tm_h16, tm_h64;
    if (!make_tmap_w13_5d(&tm_w13, w13, E, I, H)) return ELDR_ERR_CUDA;
    if (!make_tmap(&tm_w2, w2, (uint64_t)E * H, I, 128)) return ELDR_ERR_CUDA;
    if (ns) {
      if (!make_tmap_w13_5d(&tm_sw13, shared_w13, ns, I, H)) return ELDR_ERR_CUDA;
      if (!make_tmap(&tm_sw2, shared_w2, (uint64_t)ns * H, I, 128)) return ELDR_ERR_CUDA;
    } else {
      tm_sw13 = tm_w13;
      tm_sw2 = tm_w2;
    }
    if (!make_tmap(&tm_x16, x_perm, (uint64_t)x_rows, H, 16)) return ELDR_ERR_CUDA;
    if (!make_tmap(&tm_x64, x_perm, (uint64_t)x_rows, H, 64)) return ELDR_ERR_CUDA;
    if (!make_tmap(&tm_h16, hbuf, (uint64_t)out_rows, I, 16)) return ELDR_ERR_CUDA;
    if (!make_tmap(&tm_h64, hbuf, (uint64_t)out_rows, I, 64)) return ELDR_ERR_CUDA;
    UmmaCfg cfg;
    // token columns per accumulator pass (an expert receives at most T tokens); prefill-shaped calls take the widest
    // MMA (N = 256: each 16 KiB weight stage is reused by 256 tokens, TMEM 2 x 256 columns)
    cfg.np = T <= 64 ? 64 : (T <= kDecodeMaxT ? 128 : 256);
    cfg.stages = T <= 64 ? 8 : (T <= kDecodeMaxT ? 6 : 4);
    const size_t smem = (size_t)cfg.stages * (kUmmaWBytes + cfg.np * 128) + 1024 + 256;
    if (!once_per_device(kAttrUmma, [] {
          const size_t mx = 8 * (kUmmaWBytes + 64 * 128) + 1024 + 256;
          return set_smem(ffn_umma_kernel<0>, mx) && set_smem(ffn_umma_kernel<1>, mx);
        })) return ELDR_ERR_CUDA;
    f13.tiles_per_expert = I / 64;
    // auto: from 256 tokens per expert on average (half of the experts then need a second 256-token pass and the pass-
    // level unit list pays): T = 4096 on the Qwen shape 0.605 vs 0.632 ms; below it single-CTA tiles win (T = 3072:
    // 0.462 vs 0.528 ms, T = 3584: 0.510 vs 0.524 ms)
    const int ffn_pair = g_ffn_pair.load();
    const bool pair_pays = ffn_pair == 2 || (ffn_pair == 1 && (size_t)T * k >= (size_t)256 * E);
    if (T > kDecodeMaxT && pair_pays && I % 128 == 0 && H % 256 == 0 && sms >= 2) {
      // prefill-shaped: M = 256 tiles over SM pairs (ffn_umma2.cuh), six 32 KiB stages per CTA
      const int stages = 6;
      const size_t smem2 = (size_t)stages * kPairStageBytes + 1024 + 256 + (size_t)(2 * max_work + 2) * 4 + 16;
      if (!once_per_device(kAttrPair, [stages] {
            const size_t mx2 = (size_t)stages * kPairStageBytes + 1024 + 256 + (size_t)(2 * (256 + 64) + 4) * 4 + 16;
            return set_smem(ffn_umma2_kernel<0>, mx2) && set_smem(ffn_umma2_kernel<1>, mx2);
          })) return ELDR_ERR_CUDA;
      const int grid2 = sms & ~1;
      prof_mark(3, st);
      launch_dep_pair(ffn_umma2_kernel<0>, dim3(grid2), dim3(kUmmaThreads), smem2, st, tm_w13, tm_sw13, tm_x16, tm_x64, f13, stages, max_work + 1);
      if (!launch_ok("ffn_umma2_kernel<w13>")) return ELDR_ERR_CUDA;
      prof_mark(4, st);
      launch_dep_pair(ffn_umma2_kernel<1>, dim3(grid2), dim3(kUmmaThreads), smem2, st, tm_w2, tm_sw2, tm_h16, tm_h64, f2, stages, max_work + 1);
      if (!launch_ok("ffn_umma2_kernel<w2>")) return ELDR_ERR_CUDA;
    } else {
      prof_mark(3, st);
      launch_dep(ffn_umma_kernel<0>, dim3(g13), dim3(kUmmaThreads), smem, st, tm_w13, tm_sw13, tm_x16, tm_x64, f13, cfg);
      if (!launch_ok("ffn_umma_kernel<w13>")) return ELDR_ERR_CUDA;
      prof_mark(4, st);
      launch_dep(ffn_umma_kernel<1>, dim3(g2), dim3(kUmmaThreads), smem, st, tm_w2, tm_sw2, tm_h16, tm_h64, f2, cfg);
      if (!launch_ok("ffn_umma_kernel<w2>")) return ELDR_ERR_CUDA;
    }
  } else if (H % 64 == 0 && I % 64 == 0) {
    // legacy tensor-core path (mma.sync), kept selectable for comparison
    CUtensorMap tm_w13, tm_sw13, tm_x, tm_w2, tm_sw2, tm_h;
    if (!make_tmap(&tm_w13, w13, (uint64_t)E * 2 * I, H, 64)) return ELDR_ERR_CUDA;
    if (!make_tmap(&tm_w2, w2, (uint64_t)E * H, I, 128)) return ELDR_ERR_CUDA;
    if (ns) {
      if (!make_tmap(&tm_sw13, shared_w13, (uint64_t)ns * 2 * I, H, 64)) return ELDR_ERR_CUDA;
      if (!make_tmap(&tm_sw2, shared_w2, (uint64_t)ns * H, I, 128)) return ELDR_ERR_CUDA;
    } else {
      tm_sw13 = tm_w13;
      tm_sw2 = tm_w2;
    }
    if (!make_tmap(&tm_x, x_perm, (uint64_t)x_rows, H, kFfnXBox)) return ELDR_ERR_CUDA;
    if (!make_tmap(&tm_h, hbuf, (uint64_t)out_rows, I, kFfnXBox)) return ELDR_ERR_CUDA;
    if (!once_per_device(kAttrStream, [] {
          return set_smem(ffn_stream_kernel<0>, kFfnSmemBytes) && set_smem(ffn_stream_kernel<1>, kFfnSmemBytes);
        })) return ELDR_ERR_CUDA;
    prof_mark(3, st);
    launch_dep(ffn_stream_kernel<0>, dim3(g13), dim3(kFfnThreads), kFfnSmemBytes, st, tm_w13, tm_sw13, tm_x, f13);
    if (!launch_ok("ffn_stream_kernel<w13>")) return ELDR_ERR_CUDA;
    prof_mark(4, st);
    launch_dep(ffn_stream_kernel<1>, dim3(g2), dim3(kFfnThreads), kFfnSmemBytes, st, tm_w2, tm_sw2, tm_h, f2);
    if (!launch_ok("ffn_stream_kernel<w2>")) return ELDR_ERR_CUDA;
  } else {
    dim3 g13(max_work, (I + 127) / 128), g2(max_work, (H + 127) / 128);
    prof_mark(3, st);
    launch_dep(ffn13_plain_kernel, g13, dim3(128), 0, st, w13, shared_w13, x_perm, f13);
    if (!launch_ok("ffn13_plain_kernel")) return ELDR_ERR_CUDA;
    prof_mark(4, st);
    launch_dep(ffn2_plain_kernel, g2, dim3(128), 0, st, w2, shared_w2, hbuf, f2);
    if (!launch_ok("ffn2_plain_kernel")) return ELDR_ERR_CUDA;
  }
  // a7: weighted combine
  prof_mark(5, st);
  launch_dep(k <= 8 ? combine_kernel<8> : combine_kernel<kMaxTopK>, dim3((T * (H / 4) + 255) / 256), dim3(256), 0, st,
             ybuf, topk_w, pair_pos, out, T, H, k, ns);
  if (!launch_ok("combine_kernel")) return ELDR_ERR_CUDA;
  prof_mark(ELDR_PROFILE_SLOTS, st);
  return ELDR_OK;
}

int32_t eldr_moe_decode_layer_mxfp4(const eldr_moe_shape_t* s, int32_t layer, int32_t T, const eldr_bf16* x,
                                    const float* gate_w, const float* gate_bias, const uint8_t* w13_codes,
                                    const uint8_t* w13_scales, const uint8_t* w2_codes, const uint8_t* w2_scales,
                                    eldr_bf16* out, int32_t* topk_ids, float* topk_w, int32_t force_routing,
                                    int32_t* active_experts, int32_t* n_active, const int32_t* token_req,
                                    const int32_t* token_block, int32_t* sig_req, int8_t* sig_block,
                                    void* workspace, size_t workspace_bytes, eldr_stream_t stream) {
  g_launches = 0;
  int32_t rc = check_shape(s);
  if (rc != ELDR_OK) return rc;
  if (T < 0 || layer < 0 || layer >= s->n_layers) return ELDR_ERR_INVALID_ARG;
  if (T == 0) return ELDR_OK;
  if (!x || !w13_codes || !w13_scales || !w2_codes || !w2_scales || !out || !topk_ids || !topk_w || !active_experts ||
      !n_active || !workspace) return ELDR_ERR_INVALID_ARG;
  if (!force_routing && !gate_w) return ELDR_ERR_INVALID_ARG;
  if (!aligned16(x) || !aligned16(gate_w) || !aligned16(w13_codes) || !aligned16(w13_scales) || !aligned16(w2_codes) ||
      !aligned16(w2_scales) || !aligned16(out) || !aligned16(workspace) || !aligned16(sig_block)) return ELDR_ERR_INVALID_ARG;
  // decode-shaped calls, no shared experts, whole 64-element k-chunks (two 32-element scale blocks each)
  if (T > kDecodeMaxT || s->n_shared != 0 || s->hidden % 64 || s->inter % 64) return ELDR_ERR_UNSUPPORTED;
  eldr_moe_ws_layout_t L;
  make_layout(s, T, &L);
  if (workspace_bytes < L.total) return ELDR_ERR_WORKSPACE_SMALL;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  uint8_t* ws = static_cast<uint8_t*>(workspace);
  const int H = s->hidden, I = s->inter, E = s->n_experts, k = s->top_k;
  float* z = reinterpret_cast<float*>(ws + L.z);
  int32_t* perm = reinterpret_cast<int32_t*>(ws + L.perm);
  int32_t* pair_pos = reinterpret_cast<int32_t*>(ws + L.pair_pos);
  int4* work = reinterpret_cast<int4*>(ws + L.work);
  int32_t* n_work = reinterpret_cast<int32_t*>(ws + L.n_work);
  uint16_t* x_perm = reinterpret_cast<uint16_t*>(ws + L.x_perm);
  uint16_t* hbuf = reinterpret_cast<uint16_t*>(ws + L.h);
  float* ybuf = reinterpret_cast<float*>(ws + L.y);
  prof_begin();
  RouteArgs ra;
  ra.tk = TopkArgs{z, topk_ids, topk_w, token_req, token_block, sig_req, sig_block, T, E, k, s->n_layers, layer, s->renormalize};
  ra.force_routing = force_routing ? 1 : 0;
  ra.n_shared = 0;
  ra.H = H;
  ra.cnt = reinterpret_cast<int32_t*>(ws + L.cnt);
  ra.off = reinterpret_cast<int32_t*>(ws + L.off);
  ra.perm = perm; ra.pair_pos = pair_pos; ra.work = work; ra.n_work = n_work;
  ra.active = active_experts; ra.n_active = n_active;
  const int W = (T + 31) / 32;
  const size_t route_smem = (size_t)E * W * 8 + (size_t)(2 * E + 1) * 4;
  if (!force_routing) {
    GateRouteArgs ga;
    ga.x = x; ga.gate_w = gate_w; ga.gate_bias = gate_bias; ga.r = ra;
    ga.sync = reinterpret_cast<uint32_t*>(ws + L.sync + align_up(fused_sync_words(E, 0, I, H) * 4, 256));
    size_t smem = (size_t)kGateTok * H * 2;
    if (route_smem > smem) smem = route_smem;
    if (smem > 200 * 1024) return ELDR_ERR_UNSUPPORTED;
    if (smem > 48 * 1024 && !once_per_device(kAttrGateRoute, [] { return set_smem(gate_topk_route_kernel, 200 * 1024); })) return ELDR_ERR_CUDA;
    dim3 grid((E + kGateExp - 1) / kGateExp, (T + kGateTok - 1) / kGateTok);
    prof_mark(0, st);
    gate_topk_route_kernel<<<grid, 256, smem, st>>>(ga);
    if (!launch_ok("gate_topk_route_kernel")) return ELDR_ERR_CUDA;
  } else {
    if (route_smem > 48 * 1024 && !once_per_device(kAttrRouteOnly, [] { return set_smem(route_only_kernel, 200 * 1024); })) return ELDR_ERR_CUDA;
    prof_mark(1, st);
    route_only_kernel<<<1, 1024, route_smem, st>>>(ra);
    if (!launch_ok("route_only_kernel")) return ELDR_ERR_CUDA;
  }
  const int x_rows = T * k;
  prof_mark(2, st);
  launch_dep(gather_x_kernel, dim3((x_rows + 7) / 8), dim3(256), 0, st, x, perm, x_perm, T, H, k, x_rows, 1);
  if (!launch_ok("gather_x_kernel")) return ELDR_ERR_CUDA;

  const int max_work = E < T * k ? E : T * k;
  MxArgs m13, m2;
  m13.f = FfnArgs{work, n_work, E, H, 2 * I, I, H, I / 64, hbuf, nullptr};
  m2.f = FfnArgs{work, n_work, E, I, H, I, H, (H + 127) / 128, nullptr, ybuf};
  m13.scales = w13_scales;
  m2.scales = w2_scales;
  m13.np = m2.np = T <= 64 ? 64 : 128;
  m13.stages = m2.stages = kMxMaxStages;               // decoded tiles: TMEM ring
  m13.raw_stages = m2.raw_stages = 8;
  m13.act_stages = m2.act_stages = T <= 64 ? 8 : 4;
  const size_t smem = mx_smem_bytes(m13.np, m13.stages, m13.raw_stages, m13.act_stages);
  if (!once_per_device(kAttrMx, [] {
        const size_t a_ = mx_smem_bytes(64, kMxMaxStages, 8, 8), b_ = mx_smem_bytes(128, kMxMaxStages, 8, 4);
        const size_t mx = a_ > b_ ? a_ : b_;
        return set_smem(ffn_mx_kernel<0>, mx) && set_smem(ffn_mx_kernel<1>, mx);
      })) return ELDR_ERR_CUDA;
  CUtensorMap tm_c13, tm_c2, tm_x16, tm_x64, tm_h16, tm_h64;
  if (!make_tmap_u8(&tm_c13, w13_codes, (uint64_t)E * 2 * I, (uint64_t)H / 2, 64)) return ELDR_ERR_CUDA;
  if (!make_tmap_u8(&tm_c2, w2_codes, (uint64_t)E * H, (uint64_t)I / 2, 128)) return ELDR_ERR_CUDA;
  if (!make_tmap(&tm_x16, x_perm, (uint64_t)x_rows, H, 16)) return ELDR_ERR_CUDA;
  if (!make_tmap(&tm_x64, x_perm, (uint64_t)x_rows, H, 64)) return ELDR_ERR_CUDA;
  if (!make_tmap(&tm_h16, hbuf, (uint64_t)x_rows, I, 16)) return ELDR_ERR_CUDA;
  if (!make_tmap(&tm_h64, hbuf, (uint64_t)x_rows, I, 64)) return ELDR_ERR_CUDA;
  const int sms = num_sms();
  int g13 = max_work * m13.f.tiles_per_expert; if (g13 > sms) g13 = sms;
  int g2 = max_work * m2.f.tiles_per_expert; if (g2 > sms) g2 = sms;
  prof_mark(3, st);
  launch_dep(ffn_mx_kernel<0>, dim3(g13), dim3(kMxThreads), smem, st, tm_c13, tm_x16, tm_x64, m13);
  if (!launch_ok("ffn_mx_kernel<w13>")) return ELDR_ERR_CUDA;
  prof_mark(4, st);
  launch_dep(ffn_mx_kernel<1>, dim3(g2), dim3(kMxThreads), smem, st, tm_c2, tm_h16, tm_h64, m2);
  if (!launch_ok("ffn_mx_kernel<w2>")) return ELDR_ERR_CUDA;
  prof_mark(5, st);
  launch_dep(k <= 8 ? combine_kernel<8> : combine_kernel<kMaxTopK>, dim3((T * (H / 4) + 255) / 256), dim3(256), 0, st,
             ybuf, topk_w, pair_pos, out, T, H, k, 0);
  if (!launch_ok("combine_kernel")) return ELDR_ERR_CUDA;
  prof_mark(ELDR_PROFILE_SLOTS, st);
  return ELDR_OK;
}

// ids / weights of the step copied from device memory into MAPPED pinned host buffers by one small block (a
// kernel in the stream costs ~3 us; two cudaMemcpyAsync of 2 KB each cost ~12 us of stream time).
__global__ void mirror_to_host_kernel(const int32_t* __restrict__ ids, int32_t* __restrict__ h_ids,
                                      const float* __restrict__ w, float* __restrict__ h_w, int n) {
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    if (h_ids) h_ids[i] = ids[i];
    if (h_w) h_w[i] = w[i];
  }
}

int32_t eldr_moe_decode_layer_host(const eldr_moe_shape_t* s, int32_t layer, int32_t T, const eldr_bf16* h_x,
                                   const float* gate_w, const float* gate_bias, const eldr_bf16* w13,
                                   const eldr_bf16* w2, const eldr_bf16* shared_w13, const eldr_bf16* shared_w2,
                                   eldr_bf16* h_out, int32_t* h_topk_ids, float* h_topk_w, int32_t* h_n_active,
                                   const int32_t* h_token_req, const int32_t* h_token_block, int32_t* sig_req,
                                   int8_t* sig_block, void* workspace, size_t workspace_bytes,
                                   eldr_stream_t stream) {
  int32_t rc = check_shape(s);
  if (rc != ELDR_OK) return rc;
  if (T < 0) return ELDR_ERR_INVALID_ARG;
  if (T == 0) return ELDR_OK;
  if (!h_x || !h_out || !workspace) return ELDR_ERR_INVALID_ARG;
  eldr_moe_ws_layout_t L;
  make_layout(s, T, &L);
  HostStage S;
  make_host_stage(s, T, L.total, &S);
  if (workspace_bytes < S.total) return ELDR_ERR_WORKSPACE_SMALL;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  uint8_t* ws = static_cast<uint8_t*>(workspace);
  const size_t H = s->hidden, k = s->top_k;
  // Pinned (page-locked, mapped) host buffers are used in place by the kernels: the small inputs (token maps) are
  // read and out / n_active are written straight through the mapping, so the step is one host-to-device copy
  // (x, which the kernels read many times), the launch, one small block that mirrors ids / weights (which the
  // kernels read back, so they stay in device memory) into the mapped buffers, and one synchronisation.
  // Pageable buffers fall back to staged copies.
  auto mapped = [](const void* h) -> void* {
    if (!h) return nullptr;
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, h) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return (at.type == cudaMemoryTypeHost && at.devicePointer && aligned16(at.devicePointer)) ? at.devicePointer : nullptr;
  };
  int32_t* d_req = static_cast<int32_t*>(mapped(h_token_req));
  int32_t* d_blk = static_cast<int32_t*>(mapped(h_token_block));
  eldr_bf16* d_out = static_cast<eldr_bf16*>(mapped(h_out));
  // ids / weights: the staged kernels read them back (routing, combine), so there they stay in device memory and a
  // small block mirrors them into the mapped buffers; the one-launch step never reads them back (its CTAs route from
  // the tagged words in the workspace), so when that is the path this call is expected to take its top-k owners write
  // them straight through the mapping and the mirror launch is dropped.  (If the launch falls back to the staged
  // kernels after all -- the grid cannot be co-resident -- those read the mapped memory: slower, still correct.)
  const int sp_ = g_step_path.load();
  const bool expect_fused = (sp_ == ELDR_STEP_FUSED || sp_ == ELDR_STEP_AUTO) && g_ffn_path.load() == ELDR_FFN_TCGEN05 &&
                            s->hidden % 64 == 0 && s->inter % 64 == 0 && T <= kFusedMaxT && num_sms() <= 256 &&
                            g_dev[current_device()].fused_ok.load(std::memory_order_relaxed) == 1;
  int32_t* d_ids = expect_fused ? static_cast<int32_t*>(mapped(h_topk_ids)) : nullptr;
  float* d_w = expect_fused ? static_cast<float*>(mapped(h_topk_w)) : nullptr;
  int32_t* d_na = static_cast<int32_t*>(mapped(h_n_active));
  if (!cuda_ok(cudaMemcpyAsync(ws + S.x, h_x, (size_t)T * H * 2, cudaMemcpyHostToDevice, st), "H2D x")) return ELDR_ERR_CUDA;
  if (h_token_req && !d_req) {
    if (!cuda_ok(cudaMemcpyAsync(ws + S.req, h_token_req, (size_t)T * 4, cudaMemcpyHostToDevice, st), "H2D req")) return ELDR_ERR_CUDA;
    d_req = reinterpret_cast<int32_t*>(ws + S.req);
  }
  if (h_token_block && !d_blk) {
    if (!cuda_ok(cudaMemcpyAsync(ws + S.blk, h_token_block, (size_t)T * 4, cudaMemcpyHostToDevice, st), "H2D blk")) return ELDR_ERR_CUDA;
    d_blk = reinterpret_cast<int32_t*>(ws + S.blk);
  }
  rc = eldr_moe_decode_layer(s, layer, T, reinterpret_cast<eldr_bf16*>(ws + S.x), gate_w, gate_bias, w13, w2,
                             shared_w13, shared_w2, d_out ? d_out : reinterpret_cast<eldr_bf16*>(ws + S.out),
                             d_ids ? d_ids : reinterpret_cast<int32_t*>(ws + S.ids),
                             d_w ? d_w : reinterpret_cast<float*>(ws + S.w), 0,
                             reinterpret_cast<int32_t*>(ws + S.active),
                             d_na ? d_na : reinterpret_cast<int32_t*>(ws + S.n_active),
                             d_req, d_blk, sig_req, sig_block, workspace, L.total, stream);
  if (rc != ELDR_OK) return rc;
  if (!d_out && !cuda_ok(cudaMemcpyAsync(h_out, ws + S.out, (size_t)T * H * 2, cudaMemcpyDeviceToHost, st), "D2H out")) return ELDR_ERR_CUDA;
  int32_t* m_ids = d_ids ? nullptr : static_cast<int32_t*>(mapped(h_topk_ids));
  float* m_w = d_w ? nullptr : static_cast<float*>(mapped(h_topk_w));
  if (m_ids || m_w) {
    mirror_to_host_kernel<<<1, 256, 0, st>>>(reinterpret_cast<const int32_t*>(ws + S.ids), m_ids,
                                             reinterpret_cast<const float*>(ws + S.w), m_w, (int)(T * k));
    if (!cuda_ok(cudaGetLastError(), "mirror_to_host_kernel")) return ELDR_ERR_CUDA;
  }
  if (h_topk_ids && !m_ids && !d_ids && !cuda_ok(cudaMemcpyAsync(h_topk_ids, ws + S.ids, (size_t)T * k * 4, cudaMemcpyDeviceToHost, st), "D2H ids")) return ELDR_ERR_CUDA;
  if (h_topk_w && !m_w && !d_w && !cuda_ok(cudaMemcpyAsync(h_topk_w, ws + S.w, (size_t)T * k * 4, cudaMemcpyDeviceToHost, st), "D2H w")) return ELDR_ERR_CUDA;
  if (h_n_active && !d_na && !cuda_ok(cudaMemcpyAsync(h_n_active, ws + S.n_active, 4, cudaMemcpyDeviceToHost, st), "D2H n_active")) return ELDR_ERR_CUDA;
  if (!cuda_ok(cudaStreamSynchronize(st), "stream sync")) return ELDR_ERR_CUDA;
  return ELDR_OK;
}

int32_t eldr_signature_accumulate(const eldr_moe_shape_t* s, int32_t layer, int32_t T, const int32_t* topk_ids,
                                  const int32_t* token_req, const int32_t* token_block, int32_t* sig_req,
                                  int8_t* sig_block, eldr_stream_t stream) {
  g_launches = 0;
  int32_t rc = check_shape(s);
  if (rc != ELDR_OK) return rc;
  if (T < 0 || layer < 0 || layer >= s->n_layers) return ELDR_ERR_INVALID_ARG;
  if (T == 0) return ELDR_OK;
  if (!topk_ids || !aligned16(sig_block)) return ELDR_ERR_INVALID_ARG;
  const long long pairs = (long long)T * s->top_k;
  sig_accumulate_kernel<<<(unsigned)((pairs + 255) / 256), 256, 0, static_cast<cudaStream_t>(stream)>>>(
      topk_ids, token_req, token_block, sig_req, sig_block, T, s->n_experts, s->top_k, s->n_layers, layer);
  return launch_ok("sig_accumulate_kernel") ? ELDR_OK : ELDR_ERR_CUDA;
}

int32_t eldr_signature_accumulate_layers(const eldr_moe_shape_t* s, int32_t layer0, int32_t n_layers, int32_t T,
                                         const int32_t* topk_ids, const int32_t* token_req, const int32_t* token_block,
                                         int32_t* sig_req, int8_t* sig_block, eldr_stream_t stream) {
  g_launches = 0;
  int32_t rc = check_shape(s);
  if (rc != ELDR_OK) return rc;
  if (T < 0 || n_layers < 0 || layer0 < 0 || layer0 + n_layers > s->n_layers) return ELDR_ERR_INVALID_ARG;
  if (T == 0 || n_layers == 0) return ELDR_OK;
  if (!topk_ids || !aligned16(sig_block)) return ELDR_ERR_INVALID_ARG;
  const int E = s->n_experts;
  const size_t smem = (size_t)E * 4 + (size_t)(kSigChunk + 4) * ((E + 3) / 4) * 4;
  if (smem > 48 * 1024 && !once_per_device(kAttrSigLayers, [] { return set_smem(sig_accumulate_layers_kernel, 100 * 1024); })) return ELDR_ERR_CUDA;
  sig_accumulate_layers_kernel<<<dim3((T + kSigChunk - 1) / kSigChunk, n_layers), 256, smem, static_cast<cudaStream_t>(stream)>>>(
      topk_ids, token_req, token_block, sig_req, sig_block, T, E, s->top_k, s->n_layers, layer0);
  return launch_ok("sig_accumulate_layers_kernel") ? ELDR_OK : ELDR_ERR_CUDA;
}

int32_t eldr_signature_reset_blocks(const eldr_moe_shape_t* s, const int32_t* block_ids, int32_t n,
                                    int8_t* sig_block, eldr_stream_t stream) {
  g_launches = 0;
  int32_t rc = check_shape(s);
  if (rc != ELDR_OK) return rc;
  if (n < 0) return ELDR_ERR_INVALID_ARG;
  if (n == 0) return ELDR_OK;
  if (!block_ids || !sig_block || !aligned16(sig_block)) return ELDR_ERR_INVALID_ARG;
  sig_reset_kernel<<<n, 256, 0, static_cast<cudaStream_t>(stream)>>>(block_ids, sig_block,
                                                                    s->n_layers * s->n_experts);
  return launch_ok("sig_reset_kernel") ? ELDR_OK : ELDR_ERR_CUDA;
}

int32_t eldr_signature_readout(const eldr_moe_shape_t* s, const int32_t* block_ids, const int32_t* req_off,
                               int32_t n_req, const int8_t* sig_block, int32_t* sig_out, eldr_stream_t stream) {
  g_launches = 0;
  int32_t rc = check_shape(s);
  if (rc != ELDR_OK) return rc;
  if (n_req < 0) return ELDR_ERR_INVALID_ARG;
  if (n_req == 0) return ELDR_OK;
  if (!block_ids || !req_off || !sig_block || !sig_out) return ELDR_ERR_INVALID_ARG;
  const int cells = s->n_layers * s->n_experts;
  const int per_thread = (cells % 16 == 0) ? 16 : 1;
  const int want = (cells / per_thread + 255) / 256;
  dim3 grid(want < 64 ? (want > 0 ? want : 1) : 64, n_req);
  sig_readout_kernel<<<grid, 256, 0, static_cast<cudaStream_t>(stream)>>>(block_ids, req_off, sig_block, sig_out,
                                                                       cells);
  return launch_ok("sig_readout_kernel") ? ELDR_OK : ELDR_ERR_CUDA;
}

int32_t eldr_route_decide(const eldr_moe_shape_t* s, int32_t R, int32_t K, const int32_t* sig_req, const float* idf,
                          const uint8_t* layer_mask, const float* centroids, int32_t* loads, float tau,
                          int32_t* worker, float* sims, eldr_stream_t stream) {
  g_launches = 0;
  int32_t rc = check_shape(s);
  if (rc != ELDR_OK) return rc;
  if (R < 0 || K < 1 || K > kRouteMaxWorkers || !(tau >= 0.f)) return ELDR_ERR_INVALID_ARG;
  if (s->n_layers > kRouteMaxLayers) return ELDR_ERR_UNSUPPORTED;
  if (R == 0) return ELDR_OK;
  if (!sig_req || !idf || !layer_mask || !centroids || !loads || !worker || !sims) return ELDR_ERR_INVALID_ARG;
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  if (!once_per_device(kAttrRouteSims, [] { return set_smem(route_sims_kernel, kRouteStageCells * 4); })) return ELDR_ERR_CUDA;
  route_sims_kernel<<<dim3(R, (K + 7) / 8 < 16 ? (K + 7) / 8 : 16), 256, kRouteStageCells * 4, st>>>(sig_req, idf, layer_mask, centroids, sims, s->n_layers, s->n_experts, K);
  if (!launch_ok("route_sims_kernel")) return ELDR_ERR_CUDA;
  route_pick_kernel<<<1, kRoutePickThreads, 0, st>>>(sims, loads, worker, R, K, tau);
  return launch_ok("route_pick_kernel") ? ELDR_OK : ELDR_ERR_CUDA;
}

// ------------------------------------------------------------------------------- offline fit (host)
int32_t eldr_fit_idf(const int32_t* h_counts, int32_t N, int32_t L, int32_t E, double* h_idf) {
  if (!h_counts || !h_idf || N < 1 || L < 1 || E < 1) return ELDR_ERR_INVALID_ARG;
  eldr_fit::idf_table(h_counts, N, L, E, h_idf);
  return ELDR_OK;
}

int32_t eldr_fit_layer_mask(const int32_t* h_counts, const double* h_idf, const double* h_decode_p, int32_t N, int32_t L,
                            int32_t E, const int32_t* h_pairs, int32_t P, int32_t* h_order, double* h_cum_rho,
                            int32_t* h_n_star, uint8_t* h_mask) {
  if (!h_counts || !h_idf || !h_decode_p || !h_pairs || !h_order || !h_cum_rho || !h_n_star || !h_mask) return ELDR_ERR_INVALID_ARG;
  if (N < 2 || L < 1 || E < 1 || P < 2) return ELDR_ERR_INVALID_ARG;
  for (int p = 0; p < 2 * P; ++p)
    if (h_pairs[p] < 0 || h_pairs[p] >= N) return ELDR_ERR_INVALID_ARG;
  eldr_fit::greedy_layer_mask(h_counts, h_idf, h_decode_p, N, L, E, h_pairs, P, h_order, h_cum_rho, h_n_star, h_mask);
  return ELDR_OK;
}

int32_t eldr_fit_balanced_assign(const double* h_cost, int32_t N, int32_t K, int32_t cap, int32_t* h_assign, double* h_total) {
  if (!h_cost || !h_assign || N < 1 || K < 1 || cap < 1 || (long long)K * cap < N) return ELDR_ERR_INVALID_ARG;
  const double t = eldr_fit::balanced_assign(h_cost, N, K, cap, h_assign);
  if (h_total) *h_total = t;
  return ELDR_OK;
}

int32_t eldr_fit_kmeans_balanced(const double* h_sig, int32_t N, int32_t d, int32_t K, const int32_t* h_init_idx,
                                 int32_t max_iter, double* h_centroids, int32_t* h_assign, int32_t* h_steps, double* h_total) {
  if (!h_sig || !h_init_idx || !h_centroids || !h_assign || !h_steps || !h_total) return ELDR_ERR_INVALID_ARG;
  if (N < 1 || d < 1 || K < 1 || K > N || max_iter < 1) return ELDR_ERR_INVALID_ARG;
  for (int k = 0; k < K; ++k)
    if (h_init_idx[k] < 0 || h_init_idx[k] >= N) return ELDR_ERR_INVALID_ARG;
  eldr_fit::kmeans_balanced(h_sig, N, d, K, h_init_idx, max_iter, h_centroids, h_assign, h_steps, h_total);
  return ELDR_OK;
}

}  // extern "C"
