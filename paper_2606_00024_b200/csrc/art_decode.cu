// ART decode attention for B200 (sm_100a): host side and C ABI (include/art_decode.h).
//
// Two kernels sit behind the ABI, both walking the eligible KV blocks in the paper's order with the
// exact sequential termination semantics of Algorithm 1:
//   art_decode_tc.cuh    bf16 KV, head_dim 128: TMA tensor loads, tcgen05.mma with TMEM accumulators
//   art_decode_simt.cuh  fp32 KV, head_dim 64:  TMA bulk loads, CUDA-core FMAs (1e-5 tolerance rules out TF32)
// The ART-off entry point is the same kernel template with the detector compiled out.
#include <array>
#include <cstdio>
#include <cstdlib>
#include <map>
#include <mutex>
#include <utility>
#include "art_decode_simt.cuh"
#include "art_decode_pc.cuh"
#include "art_host_util.cuh"
#include "art_launch.h"
#include "art_policy.cuh"
#ifdef ART_DEBUG
#include "art_debug.cuh"
#endif

namespace art {

// ----------------------------------------------------------------------------- host side

// kernels are instantiated for 1, 2, 4, 8 heads per group; other group sizes run the next one up with padding heads
static inline int padded_group(int g) { return g <= 1 ? 1 : (g <= 2 ? 2 : (g <= 4 ? 4 : 8)); }
static inline int qlen_of(const art_desc_t* d) { return d->q_len > 1 ? d->q_len : 1; }
// rows a group carries through its walk: one per (query token, head) pair (reading R15)
static inline int rows_of(const art_desc_t* d) { return (d->num_q_heads / d->num_kv_heads) * qlen_of(d); }

struct LaunchPlan { int C, stages, mslots; uint32_t smem; };

// dispatch over (G, MODE) with a generic functor f(mode_constant, G_constant)
template <typename F>
static int dispatch(int G, int mode, F&& f) {
#define ART_CASE_G(GG)                                                                                   \
  if (G == GG) {                                                                                         \
    if (mode == 0) return f(std::integral_constant<int, 0>{}, std::integral_constant<int, GG>{});        \
    if (mode == 1) return f(std::integral_constant<int, 1>{}, std::integral_constant<int, GG>{});        \
    return f(std::integral_constant<int, 2>{}, std::integral_constant<int, GG>{});                       \
  }
  ART_CASE_G(1) ART_CASE_G(2) ART_CASE_G(4) ART_CASE_G(8)
#undef ART_CASE_G
  return ART_ERR_SHAPE;
}

// ---- TMA tensor maps over the paged caches (bf16 path).  cuTensorMapEncodeTiled is a driver entry point;
// it is fetched through the runtime so the library has no link-time dependency on libcuda.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_tiled_fn() {
  static const EncodeTiledFn fn = [] {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q = cudaDriverEntryPointSymbolNotFound;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess) { cudaGetLastError(); f = nullptr; }
    return reinterpret_cast<EncodeTiledFn>(f);
  }();
  return fn;
}

// One box = 64 token rows x 64 bf16 (128 bytes), 128-byte swizzle: exactly the canonical shared-memory
// layout tcgen05.mma reads (K-major for K_t, MN-major for V_t^T).  Coordinates are (d, c1, c2):
//   HND cache[page][head][token][d]:  dims (128, 64 tokens, page*Hkv + head)
//   NHD cache[page][token][head][d]:  dims (128, Hkv, page*64 + token)
// The outermost extent is not known to the ABI (the cache is the caller's); it is set to 2^30.
static bool encode_cache_map(CUtensorMap* tm, const void* base, int layout, int Hkv, bool whole);
// Encoding a tensor map is a driver call; a decode loop passes the same caches every step, so the last few maps
// are remembered (keyed by base pointer, layout, Hkv: everything the map depends on).
// whole: one box = the whole 64 x 128 tile of a block (rank 4: [d % 64][token][d / 64][page, head]), so a tile is ONE copy
// instruction (static-cluster kernel); otherwise rank 3 with a box of 64 x 64 (two copies per tile; persistent kernel)
static bool make_cache_map(CUtensorMap* tm, const void* base, int layout, int Hkv, bool whole = false) {
  if (whole) layout |= 256;
  struct Entry { const void* base; int layout, Hkv; CUtensorMap tm; };
  static std::mutex mu;
  static Entry cache[8];
  static int n = 0, next = 0;
  {
    std::lock_guard<std::mutex> lock(mu);
    for (int i = 0; i < n; ++i)
      if (cache[i].base == base && cache[i].layout == layout && cache[i].Hkv == Hkv) { *tm = cache[i].tm; return true; }
  }
  if (!encode_cache_map(tm, base, layout & 255, Hkv, whole)) return false;
  std::lock_guard<std::mutex> lock(mu);
  cache[next] = Entry{base, layout, Hkv, *tm};
  next = (next + 1) % 8; if (n < 8) ++n;
  return true;
}
static bool encode_cache_map(CUtensorMap* tm, const void* base, int layout, int Hkv, bool whole) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return false;
  if (whole) {
    // shared-memory image = [d / 64][token][64 elements]: the two 64-column halves one after the other, each 64 rows x 128 B
    cuuint64_t dims[4]; cuuint64_t strides[3]; cuuint32_t box[4] = {64, 64, 2, 1}; cuuint32_t es[4] = {1, 1, 1, 1};
    if (layout == ART_LAYOUT_HND) {                          // [page * Hkv + head][token][d]
      dims[0] = 64; dims[1] = 64; dims[2] = 2; dims[3] = 1ull << 30;
      strides[0] = 256; strides[1] = 128; strides[2] = 256ull * 64;
    } else {                                                 // [page * 64 + token][head][d]
      dims[0] = 64; dims[1] = 1ull << 30; dims[2] = 2; dims[3] = static_cast<cuuint64_t>(Hkv);
      strides[0] = 256ull * Hkv; strides[1] = 128; strides[2] = 256;
    }
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(base), dims, strides, box, es,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
  }
  cuuint64_t dims[3]; cuuint64_t strides[2]; cuuint32_t box[3]; cuuint32_t es[3] = {1, 1, 1};
  if (layout == ART_LAYOUT_HND) {
    dims[0] = 128; dims[1] = 64; dims[2] = 1ull << 30;
    strides[0] = 256; strides[1] = 256ull * 64;
    box[0] = 64; box[1] = 64; box[2] = 1;
  } else {
    dims[0] = 128; dims[1] = static_cast<cuuint64_t>(Hkv); dims[2] = 1ull << 30;
    strides[0] = 256; strides[1] = 256ull * Hkv;
    box[0] = 64; box[1] = 1; box[2] = 64;
  }
  return enc(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, es,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

static int validate(const art_desc_t* d, const void* q, const void* k, const void* v, const int32_t* bt,
                    const int32_t* elig, const int32_t* sl, const art_thresholds_t* th, const void* out,
                    const void* stop, bool host_variant) {
  if (!d || !q || !k || !v || !bt || !sl || !out || !stop) return ART_ERR_NULL;
  if (d->batch < 0 || d->num_q_heads <= 0 || d->num_kv_heads <= 0 || d->max_blocks_per_seq < 0) return ART_ERR_SHAPE;
  if (d->num_q_heads % d->num_kv_heads != 0) return ART_ERR_SHAPE;
  const int G = d->num_q_heads / d->num_kv_heads;
  if (G > 8) return ART_ERR_SHAPE;
  if (d->q_len < 0 || d->q_len > 8 || G * qlen_of(d) > 8) return ART_ERR_SHAPE;
  if (d->dtype == ART_DTYPE_BF16 && (d->max_blocks_per_seq >= (1 << 24) || d->max_eligible >= (1 << 24))) return ART_ERR_SHAPE;   // a step number is 24 bits
  if (d->block_tokens != ART_BLOCK_TOKENS) return ART_ERR_SHAPE;
  if (d->dtype != ART_DTYPE_F32 && d->dtype != ART_DTYPE_BF16) return ART_ERR_DTYPE;
  if (d->head_dim != 64 && d->head_dim != 128) return ART_ERR_SHAPE;
  if (!((d->dtype == ART_DTYPE_F32 && d->head_dim == 64) || (d->dtype == ART_DTYPE_BF16 && d->head_dim == 128))) return ART_ERR_DTYPE;
  if (d->kv_layout != ART_LAYOUT_HND && d->kv_layout != ART_LAYOUT_NHD) return ART_ERR_SHAPE;
  if (d->policy < ART_POLICY_DENSE || d->policy > ART_POLICY_LIST) return ART_ERR_SHAPE;
  if (d->policy == ART_POLICY_LIST) {
    if (!elig || !d->eligible_counts) return ART_ERR_NULL;
    if (d->max_eligible < 0) return ART_ERR_SHAPE;
  }
  if (d->policy == ART_POLICY_SINK_WINDOW && (d->sink_tokens < 0 || d->window_tokens < 0)) return ART_ERR_SHAPE;
  if (d->split < ART_SPLIT_PERSISTENT(16) || d->split > 16) return ART_ERR_SHAPE;
  if (d->split < 0 && d->dtype != ART_DTYPE_BF16) return ART_ERR_DTYPE;
  if (d->dtype == ART_DTYPE_F32 && d->split > 0 && (d->split & (d->split - 1))) return ART_ERR_SHAPE;
  if (!(d->sm_scale >= 0.f) || isinf(d->sm_scale)) return ART_ERR_SHAPE;
  if (th) {
    if (th->patience < 1) return ART_ERR_SHAPE;
    if (th->probe_dim != 0 && th->probe_dim != 32 && th->probe_dim != d->head_dim) return ART_ERR_SHAPE;
    if (isnan(th->tau) || isnan(th->phi)) return ART_ERR_SHAPE;
  }
  if ((reinterpret_cast<uintptr_t>(k) & 15u) || (reinterpret_cast<uintptr_t>(v) & 15u)) return ART_ERR_ALIGN;
  if (!host_variant && (reinterpret_cast<uintptr_t>(q) & 15u)) return ART_ERR_ALIGN;
  if (host_variant && d->blocks_loaded) return ART_ERR_SHAPE;
  return ART_OK;
}

static int check_arch() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return ART_ERR_CUDA; }
  int major = 0;
  if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) { cudaGetLastError(); return ART_ERR_CUDA; }
  return major == 10 ? ART_OK : ART_ERR_ARCH;
}

static int mode_of(const art_desc_t* d, const art_thresholds_t* th) {
  if (!th) return 0;
  return (th->probe_dim == 0 || th->probe_dim == d->head_dim) ? 2 : 1;
}

// ---- which bf16 kernel a descriptor selects (include/art_decode.h, art_desc_t.split):
//   1..16                 static clusters: one cluster of that many CTAs per group
//   ART_SPLIT_DYNAMIC     persistent clusters, the library's cluster size;  ART_SPLIT_PERSISTENT(cl): clusters of cl
//   0                     the library decides (see route())
struct Route { bool persistent; int want; };               // want: cluster size asked for, 0 = the library's choice
static inline Route route_of_split(const art_desc_t* d) {
  if (d->dtype != ART_DTYPE_BF16 || d->split >= 0) return {false, d->split};
  return {true, d->split == ART_SPLIT_DYNAMIC ? 0 : -d->split - 1};
}

// shared-memory plan of the static-cluster kernels (fp32 CUDA-core kernel; legacy bf16 kernel)
static LaunchPlan plan_for(bool tensor_core, int G, int PW, bool art, int C) {
  LaunchPlan pl;
  pl.C = C;
  if (tensor_core) {
    const bool two_per_sm = !art || PW == 32;
    const uint32_t budget = two_per_sm ? kSmemTwoPerSm : static_cast<uint32_t>(kMaxSmem);
    pl.stages = two_per_sm ? 3 : tc::kMaxStages;
    pl.mslots = art ? 16 : 0;
    auto total = [&]() { return tc::make_smem_map(G, PW, pl.stages, pl.mslots, art).total; };
    if (art && total() > budget) pl.mslots = kScanBatch;           // the mailbox must hold one scan batch
    while (pl.stages > 2 && total() > budget) --pl.stages;
    pl.smem = total();
    return pl;
  }
  pl.mslots = art ? (4 * C < 8 ? 8 : (4 * C > 32 ? 32 : 4 * C)) : 0;
  pl.stages = 6;
  auto total = [&](int stages) { return simt::make_smem_map(G, PW, stages, pl.mslots, art).total; };
  while (pl.stages > 2 && total(pl.stages) > static_cast<uint32_t>(kMaxSmem)) --pl.stages;
  pl.smem = total(pl.stages);
  return pl;
}

// shared-memory plan of the persistent-cluster kernel (detector off): two CTAs per SM, a 3-stage ring each
struct PcPlan { int stages; uint32_t smem; };
static PcPlan plan_pc(int G) {
  PcPlan pl;
  pl.stages = 3;
  while (pl.stages > 2 && pc::make_smem_map_p(G, pl.stages).total > kSmemTwoPerSm) --pl.stages;
  pl.smem = pc::make_smem_map_p(G, pl.stages).total;
  return pl;
}

// The occupancy calculator counts a kernel that allocates tensor memory as one CTA per SM, whatever it
// allocates; the hardware runs two of ours side by side (256 of the SM's 512 columns each; checked with a
// timestamp probe).  This twin has the same launch shape and no tcgen05 code: it is only ever passed to the
// occupancy calculator, never launched.
__global__ void __launch_bounds__(tc::kThreads, 2) tc_occupancy_twin(int* sink) {
  extern __shared__ uint8_t twin_smem[];
  if (sink) *sink = twin_smem[0];
}

static int occupancy_tc(int G, int mode, int C, uint32_t smem) {
  switch (G) { case 1: return occupancy_tc_g1(mode, C, smem); case 2: return occupancy_tc_g2(mode, C, smem);
               case 4: return occupancy_tc_g4(mode, C, smem); default: return occupancy_tc_g8(mode, C, smem); }
}
// clusters of size C that can be co-resident, cached per (device, kernel class, shared memory size)
// kind: 0 = fp32 CUDA-core kernel, 1 = bf16 tensor-core kernels (static clusters; persistent clusters: mode 0)
static int cluster_capacity(int kind, int G, int mode, int C, uint32_t smem) {
  static std::mutex mu;
  static std::map<std::array<int, 4>, int> cache;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return 0; }
  const bool twin = kind != 0 && mode != 2;
  const std::array<int, 4> key = {dev, twin ? -1 : kind * 100 + G * 4 + mode, C, static_cast<int>(smem)};
  std::lock_guard<std::mutex> lock(mu);
  auto it = cache.find(key);
  if (it != cache.end()) return it->second;
  int fit;
  if (twin) fit = max_active_clusters(tc_occupancy_twin, tc::kThreads, C, smem);
  else if (kind == 1) fit = occupancy_tc(G, mode, C, smem);
  else
    fit = dispatch(G, mode, [&](auto m, auto gg) {
      return max_active_clusters(simt::art_decode_kernel<float, 64, decltype(gg)::value, decltype(m)::value>, simt::kThreads, C, smem);
    });
  cache[key] = fit;
  return fit;
}

// Static-cluster kernels: the largest C (<= 16) whose clusters for ALL groups can be co-resident, so every
// group streams from the first cycle; never more CTAs than a group could have blocks.
static int choose_split(const art_desc_t* d, int mode, int want, int* C_out) {
  const int G = padded_group(rows_of(d));
  const int groups = d->batch * d->num_kv_heads;
  const bool art = mode != 0;
  const int PW = mode == 2 ? d->head_dim : 32;
  const bool tensor_core = d->dtype == ART_DTYPE_BF16;
  if (want != 0) { *C_out = want; return ART_OK; }
  int maxT = d->policy == ART_POLICY_LIST ? d->max_eligible : d->max_blocks_per_seq;
  if (d->policy == ART_POLICY_SINK_WINDOW) {
    const int sw = (d->sink_tokens + 63) / 64 + (d->window_tokens + 63) / 64 + 1;
    maxT = sw < maxT ? sw : maxT;
  }
  int best = 1;
  for (int C = 16; C >= 2; --C) {
    if (C > maxT) continue;
    if (!tensor_core && (C & (C - 1))) continue;
    const LaunchPlan pl = plan_for(tensor_core, G, PW, art, C);
    const int fit = cluster_capacity(tensor_core ? 1 : 0, G, mode, C, pl.smem);
    if (fit >= groups && fit > 0) { best = C; break; }
  }
  *C_out = best;
  return ART_OK;
}

// Persistent clusters (detector off): cluster size CL and the number of clusters NC = min(co-resident clusters, groups).
// The library's own choice is clusters of ONE CTA: measured on configs[3] (1024 groups of ~65 blocks), 355 us against
// 372 / 363 us with clusters of 2 / 4 and 368 us with static one-CTA clusters (profiles/r02_sweeps.md); larger
// clusters exist for callers whose groups are few and uneven (the tail of the call is then shared inside a cluster).
static int choose_pc(int G, int want, int groups, const PcPlan& pl, int* CL_out, int* NC_out) {
  const int CL = want > 0 ? want : 1;
  const int fit = cluster_capacity(1, G, 0, CL, pl.smem);
  if (fit <= 0) return ART_ERR_CUDA;
  *CL_out = CL; *NC_out = fit < groups ? fit : groups;
  return ART_OK;
}

// steps a CTA of a persistent cluster claims per atomic on its cluster's board
static int pc_claim() { return 4; }

#if defined(ART_WATCHDOG) || defined(ART_DEBUG)
// debugging builds: a pinned, device-mapped word that a wait which never ends writes before it traps; it survives
// the death of the context, so the test harness can print where the kernel was stuck (art_debug_watchdog())
static unsigned long long* g_watchdog_host = nullptr;
static unsigned long long* watchdog_word() {
  static unsigned long long* dev = [] {
    unsigned long long* h = nullptr; unsigned long long* dptr = nullptr;
    if (cudaHostAlloc(&h, 512, cudaHostAllocMapped) != cudaSuccess) { cudaGetLastError(); return dptr; }
    for (int i = 0; i < 64; ++i) h[i] = 0ull;
    if (cudaHostGetDevicePointer(&dptr, h, 0) != cudaSuccess) { cudaGetLastError(); return static_cast<unsigned long long*>(nullptr); }
    g_watchdog_host = h;
    return dptr;
  }();
  return dev;
}
#endif

// static bf16 clusters, detector on: how far the loads of a group may run ahead of its last decided step.  Every CTA of
// the cluster keeps its ring full (stages) plus two blocks per CTA on their way through P.V / mailbox / scan (+ 4).
// ART_RUNAHEAD overrides it for measurements (0 = no limit, the behaviour of round 1).
static int static_run_ahead(int C, int stages) {
  static const int env = [] { const char* e = getenv("ART_RUNAHEAD"); return e ? atoi(e) : -1; }();
  if (env >= 0) return env;
  return C * (stages + 2) + 4;
}

// workspace of the persistent-cluster kernel: one partial state (m, l, acc) per (group, CTA of a cluster)
static size_t pc_part_bytes(int groups, int G) {
  return static_cast<size_t>(groups) * pc::kMaxCL * static_cast<size_t>(G * (tc::kD + 2)) * 4u;
}
static size_t ws_bytes_for(const art_desc_t* d) {
  if (d->dtype != ART_DTYPE_BF16 || d->num_kv_heads <= 0 || d->num_q_heads % d->num_kv_heads || rows_of(d) > 8) return 0;
  return pc_part_bytes(d->batch * d->num_kv_heads, padded_group(rows_of(d))) + 256;
}

static int run(const art_desc_t* d, const void* q, const void* k, const void* v, const int32_t* bt,
               const int32_t* elig, const int32_t* elig_counts, const int32_t* sl, const art_thresholds_t* th,
               float* out, int32_t* stop, int32_t* blocks_loaded, void* workspace, size_t workspace_bytes,
               cudaStream_t stream) {
  const int groups = d->batch * d->num_kv_heads;
  if (groups == 0) return ART_OK;
  const int G = padded_group(rows_of(d));
  const int mode = mode_of(d, th);
  const int PW = mode == 2 ? d->head_dim : 32;
  const bool tensor_core = d->dtype == ART_DTYPE_BF16;
  // Static clusters are the default: every group streams from the first cycle and, with the detector on, the decision
  // loop of a group never leaves its cluster.  Persistent clusters that pull groups from a queue (detector off; they
  // need the caller's workspace) run only when split < 0 asks for them: since the S-MMA / P.V-MMA operand traffic was
  // halved, waves of one-CTA static clusters are as fast on many short groups (configs[3]: 340 / 330 us against
  // 338 / 336 us).
  Route rt = route_of_split(d);
  if (rt.persistent && mode != 0) rt = {false, 0};         // persistent clusters exist for the detector-off path only
  const size_t pc_need = tensor_core ? pc_part_bytes(groups, G) : 0;
  const bool ws_ok = workspace && workspace_bytes >= pc_need && !(reinterpret_cast<uintptr_t>(workspace) & 255u);
  int C_static = 1;
  if (!rt.persistent) {
    int rc = choose_split(d, mode, rt.want, &C_static);
    if (rc != ART_OK) return rc;
  }
  const bool persistent = rt.persistent;

  Params p = {};
  p.q = q; p.k = static_cast<const uint8_t*>(k); p.v = static_cast<const uint8_t*>(v);
  p.block_table = bt; p.elig = elig; p.elig_counts = elig_counts; p.seq_lens = sl;
  p.out = out; p.stop_block = stop; p.blocks_loaded = blocks_loaded;
  p.batch = d->batch; p.Hq = d->num_q_heads; p.Hkv = d->num_kv_heads;
  p.Gh = d->num_q_heads / d->num_kv_heads; p.qlen = qlen_of(d); p.Gr = p.Gh * p.qlen;
  for (int r = 0; r < p.Gr; ++r) p.cuts |= static_cast<uint32_t>(p.qlen - 1 - r / p.Gh) << (4 * r);
  p.max_blocks = d->max_blocks_per_seq; p.max_elig = d->max_eligible;
  p.policy = d->policy; p.layout = d->kv_layout; p.sink = d->sink_tokens; p.window = d->window_tokens;
  const int64_t row = kRowBytes;
  if (d->kv_layout == ART_LAYOUT_HND) {
    p.token_stride = row; p.head_stride = row * kBlockTokens; p.page_stride = p.head_stride * d->num_kv_heads;
  } else {
    p.head_stride = row; p.token_stride = row * d->num_kv_heads; p.page_stride = p.token_stride * kBlockTokens;
  }
  const float scale = d->sm_scale > 0.f ? d->sm_scale : 1.0f / sqrtf(static_cast<float>(d->head_dim));
  p.scale_log2 = scale * 1.4426950408889634f;
  if (th) { p.tau = th->tau; p.phi = th->phi; p.patience = th->patience; }
#ifdef ART_DEBUG
  debug::art_validate_inputs_kernel<<<groups, 128, 0, stream>>>(p, d->num_pages, watchdog_word() ? watchdog_word() + 4 : nullptr);
  if (cudaGetLastError() != cudaSuccess) return ART_ERR_CUDA;
#endif

  cudaError_t e;
  if (persistent) {
    const PcPlan pl = plan_pc(G);
    int CL = 1, NC = 1;
    int rc = choose_pc(G, rt.want, groups, pl, &CL, &NC);
    if (rc != ART_OK) return rc;
    if (!ws_ok) return ART_ERR_WORKSPACE;
    p.stages = pl.stages; p.mbox_slots = 0; p.dyn = 1;
    pc::PcParams pp = {};
    pp.b = p; pp.n_groups = groups; pp.NC = NC; pp.part = static_cast<float*>(workspace);
    pp.claim = pc_claim();
    pp.dbg = nullptr;
#ifdef ART_WATCHDOG
    pp.dbg = watchdog_word();
#endif
    CUtensorMap tmK, tmV;
    if (!make_cache_map(&tmK, k, d->kv_layout, d->num_kv_heads) || !make_cache_map(&tmV, v, d->kv_layout, d->num_kv_heads))
      return ART_ERR_CUDA;
    if (blocks_loaded && cudaMemsetAsync(blocks_loaded, 0, sizeof(int32_t) * groups, stream) != cudaSuccess) { cudaGetLastError(); return ART_ERR_CUDA; }
    const bool mt = p.qlen > 1;
    int r;
    switch (G) {
      case 1: r = launch_pc_g1(mt, NC, CL, pl.smem, stream, pp, tmK, tmV); break;
      case 2: r = launch_pc_g2(mt, NC, CL, pl.smem, stream, pp, tmK, tmV); break;
      case 4: r = launch_pc_g4(mt, NC, CL, pl.smem, stream, pp, tmK, tmV); break;
      default: r = launch_pc_g8(mt, NC, CL, pl.smem, stream, pp, tmK, tmV); break;
    }
    e = static_cast<cudaError_t>(r);
  } else {
    const int C = C_static;
    const LaunchPlan pl = plan_for(tensor_core, G, PW, mode != 0, C);
    p.stages = pl.stages; p.mbox_slots = pl.mslots;
    p.dyn = 0;                                               // static clusters deal their steps round-robin
    p.run_ahead = (tensor_core && mode != 0) ? static_run_ahead(C, pl.stages) : 0;
    if (tensor_core) {
#ifdef ART_TRACE
      if (workspace && workspace_bytes >= (1u << 20)) { cudaMemsetAsync(workspace, 0, 1u << 20, stream); p.trace = static_cast<uint8_t*>(workspace); }
#endif
      CUtensorMap tmK, tmV;
      if (!make_cache_map(&tmK, k, d->kv_layout, d->num_kv_heads, true) || !make_cache_map(&tmV, v, d->kv_layout, d->num_kv_heads, true))
        return ART_ERR_CUDA;
      const bool mt = p.qlen > 1;
      int r;
      switch (G) {
        case 1: r = launch_tc_g1(mode, mt, groups, C, pl.smem, stream, p, tmK, tmV); break;
        case 2: r = launch_tc_g2(mode, mt, groups, C, pl.smem, stream, p, tmK, tmV); break;
        case 4: r = launch_tc_g4(mode, mt, groups, C, pl.smem, stream, p, tmK, tmV); break;
        default: r = launch_tc_g8(mode, mt, groups, C, pl.smem, stream, p, tmK, tmV); break;
      }
      e = static_cast<cudaError_t>(r);
    } else {
      e = static_cast<cudaError_t>(dispatch(G, mode, [&](auto m, auto gg) {
        return static_cast<int>(launch_cluster(simt::art_decode_kernel<float, 64, decltype(gg)::value, decltype(m)::value>,
                                               simt::kThreads, groups, C, pl.smem, stream, p));
      }));
    }
  }
  if (e != cudaSuccess) { cudaGetLastError(); return ART_ERR_CUDA; }
  return ART_OK;
}

// ---- host entry point: one gather kernel instead of up to five small copies.  The per-step inputs (q, tables,
// lists: ~100 KB) are read straight out of the caller's PINNED buffers over PCIe, 16 bytes per thread.
struct StageSegs { const uint8_t* src[5]; uint8_t* dst[5]; uint32_t wide[5]; uint32_t first[6]; };   // first[i]: units before segment i; unit = 16 B (wide) or 4 B
__global__ void __launch_bounds__(256) art_stage_inputs_kernel(const StageSegs sg) {
  const uint32_t u = blockIdx.x * blockDim.x + threadIdx.x;
  if (u >= sg.first[5]) return;
  int i = 0;
#pragma unroll
  for (int k = 1; k < 5; ++k) i += (u >= sg.first[k]) ? 1 : 0;
  const uint32_t off = u - sg.first[i];
  if (sg.wide[i]) reinterpret_cast<uint4*>(sg.dst[i])[off] = reinterpret_cast<const uint4*>(sg.src[i])[off];
  else reinterpret_cast<uint32_t*>(sg.dst[i])[off] = reinterpret_cast<const uint32_t*>(sg.src[i])[off];
}

// device-accessible alias of a pinned host buffer (nullptr if the buffer is pageable or unknown to the runtime)
static const uint8_t* pinned_alias(const void* host) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, host) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  return (a.type == cudaMemoryTypeHost && a.devicePointer) ? static_cast<const uint8_t*>(a.devicePointer) : nullptr;
}

}  // namespace art

// ----------------------------------------------------------------------------- C ABI

extern "C" {

int art_decode_attention(const art_desc_t* desc, const void* q, const void* k_cache, const void* v_cache,
                         const int32_t* block_table, const int32_t* eligible_blocks, const int32_t* seq_lens,
                         const art_thresholds_t* thresholds, float* out, int32_t* stop_block,
                         void* workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!thresholds) return ART_ERR_NULL;
  int rc = art::validate(desc, q, k_cache, v_cache, block_table, eligible_blocks, seq_lens, thresholds, out, stop_block, false);
  if (rc != ART_OK) return rc;
  if ((rc = art::check_arch()) != ART_OK) return rc;
  return art::run(desc, q, k_cache, v_cache, block_table, eligible_blocks, desc->eligible_counts, seq_lens,
                  thresholds, out, stop_block, desc->blocks_loaded, workspace, workspace_bytes,
                  static_cast<cudaStream_t>(cuda_stream));
}

int art_decode_attention_off(const art_desc_t* desc, const void* q, const void* k_cache, const void* v_cache,
                             const int32_t* block_table, const int32_t* eligible_blocks, const int32_t* seq_lens,
                             float* out, int32_t* stop_block, void* workspace, size_t workspace_bytes,
                             void* cuda_stream) {
  int rc = art::validate(desc, q, k_cache, v_cache, block_table, eligible_blocks, seq_lens, nullptr, out, stop_block, false);
  if (rc != ART_OK) return rc;
  if ((rc = art::check_arch()) != ART_OK) return rc;
  return art::run(desc, q, k_cache, v_cache, block_table, eligible_blocks, desc->eligible_counts, seq_lens,
                  nullptr, out, stop_block, desc->blocks_loaded, workspace, workspace_bytes,
                  static_cast<cudaStream_t>(cuda_stream));
}

// device scratch layout of the host variant: q | block_table | seq_lens | eligible | counts | out | stop
struct HostLayout { size_t q, bt, sl, el, ec, out, stop, kws, total; };
static HostLayout host_layout(const art_desc_t* d) {
  auto up = [](size_t x) { return (x + 255) & ~static_cast<size_t>(255); };
  HostLayout h; size_t off = 0;
  const size_t esz = d->dtype == ART_DTYPE_F32 ? 4 : 2;
  const size_t B = d->batch, Hq = static_cast<size_t>(d->num_q_heads) * art::qlen_of(d), Hkv = d->num_kv_heads, D = d->head_dim;   // Hq: query rows per sequence
  h.q = off; off = up(off + B * Hq * D * esz);
  h.bt = off; off = up(off + B * static_cast<size_t>(d->max_blocks_per_seq) * 4);
  h.sl = off; off = up(off + B * 4);
  h.el = off; off = up(off + (d->policy == ART_POLICY_LIST ? B * Hkv * static_cast<size_t>(d->max_eligible) * 4 : 0));
  h.ec = off; off = up(off + (d->policy == ART_POLICY_LIST ? B * Hkv * 4 : 0));
  h.out = off; off = up(off + B * Hq * D * 4);
  h.stop = off; off = up(off + B * Hkv * 4);
  h.kws = off; off = up(off + art::ws_bytes_for(d));        // scratch of the dynamically scheduled kernel
  h.total = off;
  return h;
}

size_t art_workspace_bytes(const art_desc_t* desc) {
  if (!desc || desc->batch < 0 || desc->num_q_heads <= 0 || desc->num_kv_heads <= 0 || desc->head_dim <= 0 ||
      desc->max_blocks_per_seq < 0 || desc->max_eligible < 0) return 0;
  if (desc->num_q_heads % desc->num_kv_heads) return 0;
  return host_layout(desc).total;
}

int art_decode_attention_host(const art_desc_t* desc, const void* q_host, const void* k_cache, const void* v_cache,
                              const int32_t* block_table_host, const int32_t* eligible_blocks_host,
                              const int32_t* seq_lens_host, const art_thresholds_t* thresholds, float* out_host,
                              int32_t* stop_block_host, void* workspace, size_t workspace_bytes, void* cuda_stream) {
  int rc = art::validate(desc, q_host, k_cache, v_cache, block_table_host, eligible_blocks_host, seq_lens_host,
                         thresholds, out_host, stop_block_host, true);
  if (rc != ART_OK) return rc;
  const HostLayout h = host_layout(desc);
  if (!workspace || workspace_bytes < h.total || (reinterpret_cast<uintptr_t>(workspace) & 255u)) return ART_ERR_WORKSPACE;
  if ((rc = art::check_arch()) != ART_OK) return rc;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  uint8_t* ws = static_cast<uint8_t*>(workspace);
  const size_t esz = desc->dtype == ART_DTYPE_F32 ? 4 : 2;
  const size_t B = desc->batch, Hq = static_cast<size_t>(desc->num_q_heads) * art::qlen_of(desc), Hkv = desc->num_kv_heads, D = desc->head_dim;
  if (B == 0) return ART_OK;
  bool ok = true;
  {
    const bool list = desc->policy == ART_POLICY_LIST;
    const void* srcs[5] = {q_host, block_table_host, seq_lens_host, list ? eligible_blocks_host : nullptr, list ? desc->eligible_counts : nullptr};
    const size_t offs[5] = {h.q, h.bt, h.sl, h.el, h.ec};
    const size_t bytes[5] = {B * Hq * D * esz, B * static_cast<size_t>(desc->max_blocks_per_seq) * 4, B * 4,
                             list ? B * Hkv * static_cast<size_t>(desc->max_eligible) * 4 : 0, list ? B * Hkv * 4 : 0};
    // gather with one kernel when every buffer is pinned (16 bytes per thread where address and size allow it, else
    // 4 bytes: every size here is a multiple of 4), else fall back to one copy per buffer
    art::StageSegs sg = {};
    bool gather = true;
    uint32_t total = 0;
    for (int i = 0; i < 5; ++i) {
      sg.first[i] = total;
      sg.dst[i] = ws + offs[i]; sg.src[i] = nullptr; sg.wide[i] = 0;
      if (bytes[i] == 0) continue;
      const uint8_t* alias = art::pinned_alias(srcs[i]);
      if (!alias || (reinterpret_cast<uintptr_t>(alias) & 3u)) { gather = false; break; }
      sg.src[i] = alias;
      sg.wide[i] = (!(reinterpret_cast<uintptr_t>(alias) & 15u) && !(bytes[i] & 15u)) ? 1u : 0u;
      total += static_cast<uint32_t>(bytes[i] / (sg.wide[i] ? 16 : 4));
    }
    sg.first[5] = total;
    if (gather && total > 0) {
      art::art_stage_inputs_kernel<<<(total + 255) / 256, 256, 0, st>>>(sg);
      ok &= cudaGetLastError() == cudaSuccess;
    } else {
      for (int i = 0; i < 5; ++i)
        if (bytes[i]) ok &= cudaMemcpyAsync(ws + offs[i], srcs[i], bytes[i], cudaMemcpyHostToDevice, st) == cudaSuccess;
    }
  }
  if (!ok) { cudaGetLastError(); return ART_ERR_CUDA; }
  // Results: if the caller's buffers are pinned (device-accessible under UVA) the kernel writes them directly, which
  // saves two copies on the critical path of a decode step; otherwise they are staged and copied back.
  float* out_dev = reinterpret_cast<float*>(ws + h.out);
  int32_t* stop_dev = reinterpret_cast<int32_t*>(ws + h.stop);
  bool direct = false;
  {
    cudaPointerAttributes ao, as;
    if (cudaPointerGetAttributes(&ao, out_host) == cudaSuccess && cudaPointerGetAttributes(&as, stop_block_host) == cudaSuccess &&
        ao.type == cudaMemoryTypeHost && as.type == cudaMemoryTypeHost && ao.devicePointer && as.devicePointer) {
      out_dev = static_cast<float*>(ao.devicePointer); stop_dev = static_cast<int32_t*>(as.devicePointer); direct = true;
    } else {
      cudaGetLastError();
    }
  }
  rc = art::run(desc, ws + h.q, k_cache, v_cache, reinterpret_cast<const int32_t*>(ws + h.bt),
                reinterpret_cast<const int32_t*>(ws + h.el), reinterpret_cast<const int32_t*>(ws + h.ec),
                reinterpret_cast<const int32_t*>(ws + h.sl), thresholds, out_dev, stop_dev, nullptr,
                ws + h.kws, h.total - h.kws, st);
  if (rc != ART_OK) return rc;
  if (!direct) {
    ok &= cudaMemcpyAsync(out_host, ws + h.out, B * Hq * D * 4, cudaMemcpyDeviceToHost, st) == cudaSuccess;
    ok &= cudaMemcpyAsync(stop_block_host, ws + h.stop, B * Hkv * 4, cudaMemcpyDeviceToHost, st) == cudaSuccess;
  }
  ok &= cudaStreamSynchronize(st) == cudaSuccess;
  if (!ok) { cudaGetLastError(); return ART_ERR_CUDA; }
  return ART_OK;
}

// ----------------------------------------------------------------------------- base-policy list (A1's input)

int art_topk_blocks(const art_desc_t* d, const void* q, const void* k_cache, const int32_t* block_table,
                    const int32_t* seq_lens, int32_t top_k, float* block_scores, int32_t* eligible_blocks,
                    int32_t* eligible_counts, void* cuda_stream) {
  if (!d || !q || !k_cache || !block_table || !seq_lens || !block_scores || !eligible_blocks || !eligible_counts) return ART_ERR_NULL;
  if (d->batch < 0 || d->num_q_heads <= 0 || d->num_kv_heads <= 0 || d->num_q_heads % d->num_kv_heads) return ART_ERR_SHAPE;
  if (d->num_q_heads / d->num_kv_heads > 8 || d->q_len < 0 || art::rows_of(d) > 8) return ART_ERR_SHAPE;   // q_len = m: the last token scores (R15)
  const int G = art::padded_group(d->num_q_heads / d->num_kv_heads);
  if (d->block_tokens != ART_BLOCK_TOKENS) return ART_ERR_SHAPE;
  if (!((d->dtype == ART_DTYPE_F32 && d->head_dim == 64) || (d->dtype == ART_DTYPE_BF16 && d->head_dim == 128))) return ART_ERR_DTYPE;
  if (d->kv_layout != ART_LAYOUT_HND && d->kv_layout != ART_LAYOUT_NHD) return ART_ERR_SHAPE;
  if (top_k < 0 || top_k > d->max_eligible) return ART_ERR_SHAPE;
  if (d->max_blocks_per_seq <= 0 || d->max_blocks_per_seq > art::policy::kMaxSortBlocks) return ART_ERR_SHAPE;
  if ((reinterpret_cast<uintptr_t>(q) & 15u) || (reinterpret_cast<uintptr_t>(k_cache) & 15u)) return ART_ERR_ALIGN;
  int rc = art::check_arch();
  if (rc != ART_OK) return rc;
  const int groups = d->batch * d->num_kv_heads;
  if (groups == 0) return ART_OK;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);

  art::policy::ScoreParams sp = {};
  sp.q = q; sp.k = static_cast<const uint8_t*>(k_cache); sp.block_table = block_table; sp.seq_lens = seq_lens;
  sp.scores = block_scores; sp.batch = d->batch; sp.Hq = d->num_q_heads; sp.Hkv = d->num_kv_heads; sp.Gr = d->num_q_heads / d->num_kv_heads;
  sp.max_blocks = d->max_blocks_per_seq; sp.layout = d->kv_layout; sp.qlen = art::qlen_of(d);
  const int64_t row = art::kRowBytes;
  if (d->kv_layout == ART_LAYOUT_HND) { sp.token_stride = row; sp.head_stride = row * art::kBlockTokens; sp.page_stride = sp.head_stride * d->num_kv_heads; }
  else { sp.head_stride = row; sp.token_stride = row * d->num_kv_heads; sp.page_stride = sp.token_stride * art::kBlockTokens; }
  const dim3 grid(static_cast<unsigned>(groups), static_cast<unsigned>((d->max_blocks_per_seq + art::policy::kScoreWarps - 1) / art::policy::kScoreWarps));
  const dim3 block(art::policy::kScoreWarps * 32);
#define ART_SCORE_CASE(GG)                                                                                          \
  if (G == GG) {                                                                                                    \
    if (d->dtype == ART_DTYPE_BF16) art::policy::art_block_scores_kernel<__nv_bfloat16, 128, GG><<<grid, block, 0, st>>>(sp); \
    else art::policy::art_block_scores_kernel<float, 64, GG><<<grid, block, 0, st>>>(sp);                            \
  }
  ART_SCORE_CASE(1) ART_SCORE_CASE(2) ART_SCORE_CASE(4) ART_SCORE_CASE(8)
#undef ART_SCORE_CASE
  if (cudaGetLastError() != cudaSuccess) return ART_ERR_CUDA;

  art::policy::TopkParams tp = {};
  tp.scores = block_scores; tp.seq_lens = seq_lens; tp.lists = eligible_blocks; tp.counts = eligible_counts;
  tp.Hkv = d->num_kv_heads; tp.max_blocks = d->max_blocks_per_seq; tp.max_elig = d->max_eligible; tp.top_k = top_k;
  int n = 1;
  while (n < d->max_blocks_per_seq) n <<= 1;
  art::policy::art_topk_kernel<<<groups, 256, static_cast<size_t>(n) * 8, st>>>(tp);
  if (cudaGetLastError() != cudaSuccess) return ART_ERR_CUDA;
  return ART_OK;
}

// the launch shape run() would use, given a workspace of art_workspace_bytes(desc): cluster size, and the number of
// persistent clusters (0 = static clusters, one per group)
static int query_shape(const art_desc_t* desc, int art_on, int* C_out, int* NC_out) {
  if (!desc) return ART_ERR_NULL;
  if (desc->num_q_heads <= 0 || desc->num_kv_heads <= 0 || desc->num_q_heads % desc->num_kv_heads) return ART_ERR_SHAPE;
  if (desc->num_q_heads / desc->num_kv_heads > 8 || desc->q_len < 0 || art::rows_of(desc) > 8) return ART_ERR_SHAPE;
  if (!((desc->dtype == ART_DTYPE_F32 && desc->head_dim == 64) || (desc->dtype == ART_DTYPE_BF16 && desc->head_dim == 128))) return ART_ERR_DTYPE;
  if (desc->split < ART_SPLIT_PERSISTENT(16) || desc->split > 16 || (desc->split < 0 && desc->dtype != ART_DTYPE_BF16)) return ART_ERR_SHAPE;
  int rc = art::check_arch();
  if (rc != ART_OK) return rc;
  const int mode = art_on == 2 ? 2 : (art_on ? 1 : 0);                 // 2: detector on the full output (probe_dim = 0 or d)
  const int groups = desc->batch * desc->num_kv_heads > 0 ? desc->batch * desc->num_kv_heads : 1;
  art::Route rt = art::route_of_split(desc);
  int C = 1;
  if (!rt.persistent) {
    rc = art::choose_split(desc, mode, rt.want, &C);
    if (rc != ART_OK) return rc;
  } else if (mode != 0) {                                  // persistent clusters exist for the detector-off path only
    rt = {false, 0};
    rc = art::choose_split(desc, mode, 0, &C);
    if (rc != ART_OK) return rc;
  }
  *C_out = C; *NC_out = 0;
  if (rt.persistent) {
    const int G = art::padded_group(art::rows_of(desc));
    rc = art::choose_pc(G, rt.want, groups, art::plan_pc(G), C_out, NC_out);
  }
  return rc;
}

int art_query_split(const art_desc_t* desc, int art_on) {
  int C = 0, NC = 0;
  const int rc = query_shape(desc, art_on, &C, &NC);
  return rc == ART_OK ? C : rc;
}

int art_query_clusters(const art_desc_t* desc, int art_on) {
  int C = 0, NC = 0;
  const int rc = query_shape(desc, art_on, &C, &NC);
  return rc == ART_OK ? NC : rc;
}

const char* art_status_string(int status) {
  switch (status) {
    case ART_OK: return "ok";
    case ART_ERR_NULL: return "a required pointer is NULL";
    case ART_ERR_SHAPE: return "unsupported or inconsistent shape / parameter";
    case ART_ERR_DTYPE: return "unsupported dtype / head_dim combination";
    case ART_ERR_ALIGN: return "q / k_cache / v_cache must be 16-byte aligned";
    case ART_ERR_WORKSPACE: return "workspace missing, misaligned or too small";
    case ART_ERR_ARCH: return "device is not compute capability 10.x (sm_100)";
    case ART_ERR_CUDA: return "CUDA runtime or launch error";
    case ART_ERR_SCRATCH_LIMIT: return "problem needs more scratch than the library's built-in array (ART_STATIC_SCRATCH_BYTES)";
    default: return "unknown status";
  }
}

int art_version(void) { return ART_VERSION; }

#ifdef ART_WATCHDOG
unsigned long long art_debug_watchdog(void) { return art::g_watchdog_host ? art::g_watchdog_host[0] : 0ull; }
#endif
#ifdef ART_DEBUG
// (code << 48 | b << 32 | g << 24 | index) of the first violation art_validate_inputs_kernel found, 0 if none; *value gets
// the offending value.  The word lives in pinned host memory: it can be read after the trap has killed the context.
unsigned long long art_debug_last_violation(unsigned long long* value) {
  if (!art::g_watchdog_host) return 0ull;
  if (value) *value = art::g_watchdog_host[6];
  return art::g_watchdog_host[5];
}
#endif

}  // extern "C"
