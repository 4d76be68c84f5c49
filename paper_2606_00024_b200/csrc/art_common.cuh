// Shared device-side pieces of the ART decode-attention kernels (sm_100a): launch parameters,
// PTX wrappers (mbarrier, TMA bulk copies, cluster / distributed shared memory) and the
// traversal order of the eligible KV blocks.
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include <math.h>
#include <type_traits>

#include "art_decode.h"

namespace art {

constexpr int kBlockTokens = 64;
constexpr int kRowBytes = 256;                    // one token row of one head: d * sizeof(T)
constexpr int kTileBytes = kBlockTokens * kRowBytes;   // 16 KiB: K or V tile of one block
constexpr int kStageBytes = 2 * kTileBytes;       // K + V
constexpr int kMaxSmem = 232448;                  // 227 KiB usable per CTA on sm_100
constexpr int kSmemTwoPerSm = 115712;              // (228 KiB - 2 x 1 KiB reserved) / 2: two CTAs share an SM
constexpr float kNegInf = -INFINITY;

struct Params {
  const void* q;
  const uint8_t* k;
  const uint8_t* v;
  const int32_t* block_table;
  const int32_t* elig;
  const int32_t* elig_counts;
  const int32_t* seq_lens;
  float* out;
  int32_t* stop_block;
  int32_t* blocks_loaded;
  int32_t batch, Hq, Hkv;
  int32_t Gr;                                        // real rows per group (q_len * Hq / Hkv); kernels are built for the next power of two
  int32_t Gh, qlen;                                  // heads per query token of a group (Hq / Hkv), query tokens m (R15); row = i * Gh + h
  uint32_t cuts;                                     // 4 bits per row: m - 1 - i, the most recent tokens row i may not see; 0 when m == 1
  int32_t max_blocks, max_elig;
  int32_t policy, layout, sink, window;
  int64_t page_stride, head_stride, token_stride;   // bytes
  float scale_log2;                                  // sm_scale * log2(e)
  float tau, phi;
  int32_t patience;
  int32_t stages, mbox_slots;
  int32_t dyn;                                       // 1 in the persistent-cluster kernel (steps claimed at run time); static clusters deal round-robin
  int32_t run_ahead;                                 // bf16 cluster kernel, detector on: loads of step t are issued once step t - run_ahead is decided (0 = no limit)
#ifdef ART_TRACE
  uint8_t* trace;
#endif
};

#ifdef ART_TRACE   // debugging aid (never in the shipped build): timestamped events of the first CTAs
constexpr int kTraceCtas = 8, kTraceRoles = 6, kTraceEvents = 1024;
__device__ __forceinline__ unsigned long long trace_now() {
  unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t;
}
struct Tracer {      // roles claim one of kTraceCtas trace slots when they first have something to say
  uint8_t* region; ulonglong2* buf; int n, role; volatile int* share;
  __device__ __forceinline__ void init(uint8_t* base, size_t off, int role_, volatile int* share_) {
    region = base + off; buf = nullptr; n = 0; role = role_; share = share_;
  }
  __device__ __forceinline__ void ev(int code, int a, int b) {
    if (region == nullptr) return;
    if (!buf) {
      int slot;
      if (role != 0) { slot = *share - 1; if (slot < 0) return; }            // every other role follows its producer
      else {
        if (n < 0) return;
        slot = atomicAdd(reinterpret_cast<int*>(region) + role, 1);
        if (role == 0) *share = slot < kTraceCtas ? slot + 1 : 0;
        if (slot >= kTraceCtas) { n = -1; return; }
      }
      if (slot >= kTraceCtas) return;
      buf = reinterpret_cast<ulonglong2*>(region + 256) + (slot * kTraceRoles + role) * kTraceEvents;
    }
    if (n >= 0 && n < kTraceEvents) { buf[n++] = make_ulonglong2(trace_now(), (static_cast<unsigned long long>(code) << 48) | (static_cast<unsigned long long>(a & 0xffffff) << 24) | static_cast<unsigned long long>(b & 0xffffff)); }
  }
};
#endif

// ----------------------------------------------------------------------------- PTX wrappers

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r;
}
__device__ __forceinline__ uint32_t cluster_nctarank() {
  uint32_t r; asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r)); return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t mapa(uint32_t addr, uint32_t rank) {
  uint32_t r; asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank)); return r;
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive_remote(uint32_t cluster_bar) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" :: "r"(cluster_bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile("{\n\t.reg .pred p;\n\t"
               "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
               "selp.u32 %0, 1, 0, p;\n\t}"
               : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0;
}
// non-blocking probe of a phase (try_wait may suspend the thread for a while before answering "no")
__device__ __forceinline__ bool mbar_test_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile("{\n\t.reg .pred p;\n\t"
               "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
               "selp.u32 %0, 1, 0, p;\n\t}"
               : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0;
}
__device__ __forceinline__ bool mbar_try_wait_cluster(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile("{\n\t.reg .pred p;\n\t"
               "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
               "selp.u32 %0, 1, 0, p;\n\t}"
               : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  while (!mbar_try_wait(bar, parity)) {}
}
__device__ __forceinline__ void fence_mbar_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
// TMA 1-D bulk copy global -> this CTA's shared memory, completion on an mbarrier.
__device__ __forceinline__ void tma_load_1d(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               :: "r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void st_cluster_f32(uint32_t cluster_addr, float v) {
  asm volatile("st.shared::cluster.f32 [%0], %1;" :: "r"(cluster_addr), "f"(v) : "memory");
}
__device__ __forceinline__ void st_cluster_release_s32(uint32_t cluster_addr, int v) {
  asm volatile("st.release.cluster.shared::cluster.s32 [%0], %1;" :: "r"(cluster_addr), "r"(v) : "memory");
}
__device__ __forceinline__ float ld_cluster_f32(uint32_t cluster_addr) {
  float v; asm volatile("ld.shared::cluster.f32 %0, [%1];" : "=f"(v) : "r"(cluster_addr) : "memory"); return v;
}
__device__ __forceinline__ int ld_cluster_s32(uint32_t cluster_addr) {
  int v; asm volatile("ld.shared::cluster.s32 %0, [%1];" : "=r"(v) : "r"(cluster_addr) : "memory"); return v;
}
__device__ __forceinline__ int ld_acquire_ctrl(uint32_t addr) {
  int v; asm volatile("ld.acquire.cluster.shared::cta.s32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory"); return v;
}
__device__ __forceinline__ int ld_volatile_s32(uint32_t addr) {
  int v; asm volatile("ld.volatile.shared::cta.s32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory"); return v;
}
__device__ __forceinline__ void st_volatile_s32(uint32_t addr, int v) {
  asm volatile("st.volatile.shared::cta.s32 [%0], %1;" :: "r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
  uint4 r; asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr));
  return r;
}
__device__ __forceinline__ uint2 lds64(uint32_t addr) {
  uint2 r; asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(r.x), "=r"(r.y) : "r"(addr));
  return r;
}
__device__ __forceinline__ float lds_f32(uint32_t addr) {
  float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr)); return v;
}
__device__ __forceinline__ float fast_exp2(float x) {       // ex2.approx: exp2(-inf) = +0
  float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y;
}

// ----------------------------------------------------------------------------- traversal (A1)

// Traversal order of the eligible blocks (SINK_WINDOW per reading R3).
struct Trav {
  int T;        // number of steps
  int nb;       // blocks holding tokens < L
  int sb;       // blocks holding sink tokens
  int wb;       // first block holding window tokens (== nb if none)
  int policy;
  const int32_t* list;
};

__device__ __forceinline__ Trav make_trav(const Params& p, int b, int g, int L) {
  Trav tr;
  tr.policy = p.policy; tr.list = nullptr;
  tr.nb = (L + kBlockTokens - 1) / kBlockTokens; tr.sb = 0; tr.wb = tr.nb;
  if (p.policy == ART_POLICY_LIST) {
    tr.list = p.elig + (static_cast<int64_t>(b) * p.Hkv + g) * p.max_elig;
    tr.T = p.elig_counts[b * p.Hkv + g];
  } else if (p.policy == ART_POLICY_SINK_WINDOW) {
    const int s_eff = min(max(p.sink, 0), L);
    tr.sb = (s_eff + kBlockTokens - 1) / kBlockTokens;
    const int w0 = L - min(max(p.window, 0), L);           // first window token
    tr.wb = (w0 < L) ? w0 / kBlockTokens : tr.nb;
    if (tr.sb > 0) tr.T = (tr.wb <= tr.sb) ? tr.nb : 1 + (tr.nb - tr.wb) + (tr.sb - 1);
    else tr.T = tr.nb - tr.wb;
  } else {
    tr.T = tr.nb;
  }
  if (L <= 0 && p.policy != ART_POLICY_LIST) tr.T = 0;
  return tr;
}

// logical block id visited at 1-based step t
__device__ __forceinline__ int trav_block(const Trav& tr, int t) {
  if (tr.policy == ART_POLICY_LIST) return tr.list[t - 1];
  if (tr.policy == ART_POLICY_SINK_WINDOW && tr.sb > 0) {
    if (t == 1) return 0;                                   // the sink block is never skipped (R3)
    const int k = t - 2;
    if (tr.wb <= tr.sb) return tr.nb - 1 - k;
    const int n1 = tr.nb - tr.wb;
    return (k < n1) ? tr.nb - 1 - k : tr.sb - 1 - (k - n1);
  }
  return (tr.policy == ART_POLICY_SINK_WINDOW ? tr.nb : tr.T) - t;   // most recent first
}

__device__ __forceinline__ uint64_t range_mask(int lo, int hi) {     // bits [lo, hi) of 64
  lo = max(lo, 0); hi = min(hi, 64);
  if (hi <= lo) return 0ull;
  const uint64_t upper = (hi >= 64) ? ~0ull : ((1ull << hi) - 1ull);
  return upper & ~((1ull << lo) - 1ull);
}

// which of the block's 64 tokens are eligible (partial last block, sink / window edges; R8)
__device__ __forceinline__ uint64_t block_mask(const Params& p, int L, int blk) {
  if (blk < 0) return 0ull;
  const int64_t j0 = static_cast<int64_t>(blk) * kBlockTokens;
  if (j0 >= L) return 0ull;
  const int base = static_cast<int>(j0);
  if (p.policy == ART_POLICY_SINK_WINDOW) {
    const int s_eff = min(max(p.sink, 0), L);
    const int w0 = L - min(max(p.window, 0), L);
    return range_mask(0, s_eff - base) | range_mask(w0 - base, L - base);
  }
  return range_mask(0, L - base);
}

}  // namespace art
