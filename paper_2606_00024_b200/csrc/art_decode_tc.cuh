// ART decode attention, Blackwell tensor-core kernel (bf16 KV, head_dim 128): tcgen05 + TMEM + TMA.
//
// One thread-block CLUSTER of C CTAs per query group (sequence b, KV head g); traversal steps
// t = 1..T are dealt round-robin, CTA c owns steps c+1, c+1+C, ...  Two CTAs fit on
// one SM (3-stage ring, 256 TMEM columns each), so one SM always has ~6 KV blocks in flight.  Inside a
// CTA one 64-token KV block is one pipeline item, handled by specialised warps that meet only through
// mbarriers, each warp waiting on ONE barrier at a time:
//
//   producer (warp 8)      A1/A2  resolves block -> page, issues 2 TMA tensor copies (one per tile: rank-4 map, the image
//                                 in shared memory is two 64-column boxes, 128-byte swizzle) into the ring of stages
//   S-MMA    (warp 9, 1 thr) A3   S[token, head] = K_t . Q^T : tcgen05.mma M128 N16 K16, ONE per k-step: the 64
//                                 tokens are M rows 0-63 (even blocks; TMEM lanes 0-63) or rows 64-127 (odd
//                                 blocks: the operand starts 64 rows below the tile; lanes 64-127).  What an MMA
//                                 costs here is reading its A operand (128 rows x 32 B) from shared memory, so
//                                 the K tile is read twice per block, not four times as in round 1
//   softmax  (warps 4-7)   A4     a PAIR of warps owns a block (warps 4, 5: even blocks; 6, 7: odd blocks), one
//                                 token per thread; the two halves exchange their maxima through shared memory
//                                 and one 64-thread named barrier.  p = 2^(s - m_blk) relative to the BLOCK
//                                 maximum (the warps are stateless), split into bf16 hi + lo (~16 mantissa
//                                 bits, so the probe of P~V_t is accurate to ~1e-5 and the criterion does not
//                                 flip) and written to shared memory as the B operand of the P.V MMA
//   PV-MMA   (warp 10, 1 thr) A5   PV[d, head] = V_t^T . P^T : tcgen05.mma M128 N16 K16 x 4, N = (hi of 8 heads | lo of 8 heads)
//   fold     (warps 0-3)   A5/A6  one thread per output coordinate: tcgen05.ld of P~V_t; publishes the step
//                                 summary (m_blk, block sum, probe components of P~V_t) to the cluster
//                                 leader's mailbox (st.async + mbarrier complete_tx, no fences) and merges
//                                 P~V_t into the running (m, l, acc) only once the leader has decided that
//                                 step t <= t*
//   scan     (warp 11, leader CTA) A6/A7/A9  replays Algorithm 1 (Eq. 2-3) sequentially
//                                 over the step summaries (art_scan.cuh), broadcasts progress / t*
//
// The block-local P~V_t of up to 8 steps per CTA wait UNFOLDED in tensor memory, so loads, MMAs and
// softmax never wait for the sequential decision; blocks with step > t* are simply never folded, which
// makes the result equal to the sequential algorithm's for any C.
#pragma once
#include <cuda.h>   // CUtensorMap (type only: the encoder is fetched through the runtime, no -lcuda)

#include "art_common.cuh"
#include "art_scan.cuh"

namespace art {
namespace tc {

#ifdef ART_TRACE
#define TC_TRACE_INIT(tr, role) Tracer tr; tr.init(p.trace, 0, role, reinterpret_cast<volatile int*>(smem + sm.misc + 20))
#define TC_TRACE(tr, code, a, b) tr.ev(code, a, b)
#else
#define TC_TRACE_INIT(tr, role)
#define TC_TRACE(tr, code, a, b)
#endif

constexpr int kThreads = 384;
// Fold and softmax warps must sit at warp % 4 == TMEM lane quadrant.  The single-thread roles and the scan warp
// get the highest warp ids: the SM's schedulers favour them, and their latency is what the pipeline feels.
constexpr int kWarpFold0 = 0, kWarpSoftmax0 = 4, kWarpProducer = 8, kWarpMmaS = 9, kWarpMmaPV = 10, kWarpScan = 11;
constexpr int kD = 128;                      // head_dim
constexpr int kUmmaN = 16;                   // MMA N: the group's heads padded to 16
constexpr int kSSlots = 4;                   // S accumulators: one per softmax warp, 2 x 16 TMEM columns
constexpr int kSCols = 2 * kUmmaN;
constexpr int kPVSlots = 8;                  // unfolded P~V_t results (16 TMEM columns each)
constexpr int kSCols1 = kUmmaN;              // static-cluster kernel: an S accumulator is 16 columns (64 tokens on the lanes)
constexpr int kTmemCols = 256;               // S + 8 x 16 (allocations are powers of two); two CTAs share the SM's 512 columns
constexpr int kIterSlots = 16;               // softmax -> fold hand-over ring; >= kPVSlots + max stages
constexpr int kMaxStages = 6;
// P^T (hi, lo) buffers: one per ring stage, except for G = 8 with the detector on, where shared memory only has room for two (block i
// then uses buffer i & 1, free again once P~V_(i-2) is complete)
// ring of the step numbers of the items in flight (>= stages + kPVSlots entries; 12 where every byte counts)
__host__ __device__ constexpr int item_ring(int G, bool art32) { return (G == 8 && art32) ? 12 : 16; }
// softmax -> fold hand-over ring of the static-cluster kernel: per block [m_blk | block sum of tokens 0-31 | of tokens 32-63] x G
__host__ __device__ constexpr int iter_ring(int G, bool art32) { return (G == 8 && art32) ? 12 : kIterSlots; }
__host__ __device__ constexpr int p_bufs(int G, int stages, bool art32) { return (G == 8 && art32) ? 2 : stages; }
constexpr int kBoxBytes = 8192;              // one TMA box: 64 rows x 128 bytes
constexpr int kFront = 12288;                // mapped bytes the S MMA may read below a K tile (3 x 32 rows)
// Q^T as B operand (K-major, no swizzle): [16 d-chunks of 8][rows][16 B], chunk stride 128 B.  Rows 8-15 of
// a chunk alias rows 0-7 of the next one: they only feed accumulator columns >= 8, which nobody reads.
constexpr int kQLbo = 128, kQSbo = 128, kQBytes = 16 * kQLbo + 128;
static_assert(kIterSlots >= kPVSlots + kMaxStages, "IterSlot ring too short");

// P^T as B operand: [8 token-chunks of 8][rows][16 B]; chunk stride 16 G + 16 B puts the 4 chunks a warp
// writes at once into distinct banks; rows >= G alias later chunks (unread accumulator columns).
__host__ __device__ constexpr int p_lbo(int G) { return 16 * G + 16; }
__host__ __device__ constexpr int p_buf_bytes(int G) { return 7 * p_lbo(G) + 128; }

struct SmemMap {
  uint32_t qb, pb, slots, xch, items, sinfo, mbox, bars, misc, ring, total;
  uint32_t full0, empty0, pfull0, sfull0, sfree0, pvfull0, pvfree0, done0, mbox0, nbars;
};

// Offsets from the (1024-byte aligned) dynamic shared memory base.  The small buffers come first: the S MMA
// reads up to kFront bytes below its K tile (rows that only feed unused accumulator lanes).
__host__ __device__ inline SmemMap make_smem_map(int G, int PW, int stages, int mslots, bool art) {
  SmemMap m;
  uint32_t off = 0;
  m.qb = off; off += kQBytes;
  m.pb = off; off += static_cast<uint32_t>(p_bufs(G, stages, art && PW == 32)) * 2u * p_buf_bytes(G);
  m.slots = off; off += static_cast<uint32_t>(iter_ring(G, art && PW == 32)) * 3u * G * 4u;
  m.xch = off; off += 8u * G * 4u;        // block maxima of the two token halves: [pair][parity][half][G]
  m.items = off; off += static_cast<uint32_t>(item_ring(G, art && PW == 32)) * 4u;
  m.sinfo = off; off += static_cast<uint32_t>(stages) * 8u;
  off = (off + 15u) & ~15u;                // mailbox rows are written with 16-byte st.async
  m.mbox = off; off += art ? static_cast<uint32_t>(mslots) * G * (2 + PW) * 4u : 0u;
  off = (off + 15u) & ~15u;
  m.bars = off;
  uint32_t n = 0;
  m.full0 = n; n += stages; m.empty0 = n; n += stages; m.pfull0 = n; n += stages;
  m.sfull0 = n; n += kSSlots; m.sfree0 = n; n += kSSlots;
  m.pvfull0 = n; n += kPVSlots; m.pvfree0 = n; n += kPVSlots;
  m.done0 = n; n += 2;
  m.mbox0 = n; n += art ? mslots : 0;
  m.nbars = n;
  off += n * 8u;
  m.misc = off; off += 24u;              // ctrl, loaded, tmem_ptr, next_step (leader), n_total
  off = (off + 1023u) & ~1023u;
  if (off < static_cast<uint32_t>(kFront)) off = kFront;
  m.ring = off; off += static_cast<uint32_t>(stages) * kStageBytes;
  m.total = off;
  return m;
}
constexpr uint32_t kCtrl = 0, kNTotal = 4, kLoaded = 8, kTmemPtr = 12;   // (ctrl, n_total) are read as one 8-byte word

// An entry of the item ring: the step number in the low 24 bits and, for multi-token queries (R15), the causal
// code of the step's block above them: e = L - 64 * blk (tokens of the sequence from the start of this block on)
// when the causal cut of some row can reach into the block (1 <= e <= 70: a row loses at most 7 tokens), else 0.
// Row r then sees token `tok` of the block iff tok + cut_r < e.
constexpr int kItemShift = 24, kItemStep = (1 << kItemShift) - 1;
__device__ __forceinline__ int causal_code(const Params& p, int L, int blk) {
  const int e = L - blk * kBlockTokens;
  return (e >= 1 && e < kBlockTokens + 7) ? e : 0;
}

// ----------------------------------------------------------------------------- tcgen05 / TMA wrappers

__device__ __forceinline__ void tma_load_box(uint32_t dst, const CUtensorMap* tm, int c0, int c1, int c2, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
               :: "r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}
// a whole 64 x 128 tile with ONE instruction (rank-4 map [d % 64][token][d / 64][page, head]; the image in shared memory is the
// two 64-column boxes one after the other): HND (0, 0, 0, page * Hkv + head), NHD (0, page * 64, 0, head)
__device__ __forceinline__ void tma_load_tile(uint32_t dst, const CUtensorMap* tm, int ca, int cb, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %2, %4}], [%5];"
               :: "r"(dst), "l"(tm), "r"(0), "r"(ca), "r"(cb), "r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(smem_dst), "r"(ncols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// D[tmem] (+)= A[smem desc] . B[smem desc], bf16 inputs, fp32 accumulate; issued by ONE thread
__device__ __forceinline__ void umma_bf16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
               "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
               :: "r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate) : "memory");
}
// arrive on an mbarrier once every tcgen05.mma this thread issued so far has completed
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(bar) : "memory");
}
template <int N> __device__ __forceinline__ void tmem_ld(uint32_t taddr, float (&r)[N]);
template <> __device__ __forceinline__ void tmem_ld<1>(uint32_t taddr, float (&r)[1]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%1];" : "=f"(r[0]) : "r"(taddr) : "memory");
}
template <> __device__ __forceinline__ void tmem_ld<2>(uint32_t taddr, float (&r)[2]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0,%1}, [%2];" : "=f"(r[0]), "=f"(r[1]) : "r"(taddr) : "memory");
}
template <> __device__ __forceinline__ void tmem_ld<4>(uint32_t taddr, float (&r)[4]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];"
               : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]) : "r"(taddr) : "memory");
}
template <> __device__ __forceinline__ void tmem_ld<8>(uint32_t taddr, float (&r)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]), "=f"(r[4]), "=f"(r[5]), "=f"(r[6]), "=f"(r[7])
               : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ float warp_max_f32(float x) {
  float y; asm volatile("redux.sync.max.f32 %0, %1, 0xffffffff;" : "=f"(y) : "f"(x)); return y;
}

// shared-memory matrix descriptors (sm_100 format: version 1 at bit 46, layout type at bits 61-63)
constexpr uint64_t kDescSw128 = (2ull << 61) | (1ull << 46);
constexpr uint64_t kDescNoSw = (1ull << 46);
__device__ __forceinline__ constexpr uint64_t desc_strides(uint32_t lbo_bytes, uint32_t sbo_bytes) {
  return (static_cast<uint64_t>(lbo_bytes >> 4) << 16) | (static_cast<uint64_t>(sbo_bytes >> 4) << 32);
}
__device__ __forceinline__ uint64_t desc_addr(uint32_t smem_addr) { return static_cast<uint64_t>((smem_addr & 0x3ffffu) >> 4); }
// instruction descriptor: fp32 accumulate, bf16 A and B, N = 16, M = 128; bit 15 = A is MN-major
constexpr uint32_t kIdescS = (1u << 4) | (1u << 7) | (1u << 10) | ((kUmmaN >> 3) << 17) | ((128u >> 4) << 24);
constexpr uint32_t kIdescPV = kIdescS | (1u << 15);

// asynchronous store into a cluster peer's shared memory; completes bytes on the peer's mbarrier (no fences)
template <int N> __device__ __forceinline__ void st_async_vec(uint32_t cluster_addr, const float* v, uint32_t cluster_bar);
template <> __device__ __forceinline__ void st_async_vec<1>(uint32_t a, const float* v, uint32_t m) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.f32 [%0], %1, [%2];" :: "r"(a), "f"(v[0]), "r"(m) : "memory");
}
template <> __device__ __forceinline__ void st_async_vec<2>(uint32_t a, const float* v, uint32_t m) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f32 [%0], {%1,%2}, [%3];"
               :: "r"(a), "f"(v[0]), "f"(v[1]), "r"(m) : "memory");
}
template <> __device__ __forceinline__ void st_async_vec<4>(uint32_t a, const float* v, uint32_t m) {
  asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.f32 [%0], {%1,%2,%3,%4}, [%5];"
               :: "r"(a), "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]), "r"(m) : "memory");
}
template <> __device__ __forceinline__ void st_async_vec<8>(uint32_t a, const float* v, uint32_t m) {
  st_async_vec<4>(a, v, m); st_async_vec<4>(a + 16u, v + 4, m);
}
// progress word (ctrl): a stand-alone value, so relaxed accesses are enough
__device__ __forceinline__ void st_cluster_relaxed_s32(uint32_t cluster_addr, int v) {
  asm volatile("st.relaxed.cluster.shared::cluster.s32 [%0], %1;" :: "r"(cluster_addr), "r"(v) : "memory");
}
__device__ __forceinline__ int ld_ctrl_relaxed(uint32_t addr) {
  int v; asm volatile("ld.relaxed.cluster.shared::cta.s32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory"); return v;
}
// the progress word and the number of items the producer will issue, in one load (x = ctrl, y = n_total)
__device__ __forceinline__ int2 ld_ctrl_ntotal(uint32_t addr) {
  int2 v; asm volatile("ld.relaxed.cluster.shared::cta.v2.s32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr) : "memory"); return v;
}

// Sum G per-lane values over the 32 lanes with a transposing butterfly (G-1 + 5-log2(G) ... shuffles instead
// of 5 G): afterwards v[0] of lane l holds the total of value head_of_lane32<G>(l).
template <int N, int MASK>
struct Reduce32 {
  static __device__ __forceinline__ void run(float* v, int lane) {
    if constexpr (N > 1) {
      constexpr int n = N / 2;
      const bool up = (lane & MASK) != 0;
#pragma unroll
      for (int i = 0; i < n; ++i) {
        const float keep = up ? v[i + n] : v[i];
        const float send = up ? v[i] : v[i + n];
        v[i] = keep + __shfl_xor_sync(0xffffffffu, send, MASK);
      }
      if constexpr (MASK > 1) Reduce32<n, MASK / 2>::run(v, lane);
    } else {
      v[0] += __shfl_xor_sync(0xffffffffu, v[0], MASK);
      if constexpr (MASK > 1) Reduce32<1, MASK / 2>::run(v, lane);
    }
  }
};
template <int G> __device__ __forceinline__ int head_of_lane32(int lane) {
  int h = 0;
  if constexpr (G >= 2) h += ((lane >> 4) & 1) * (G / 2);
  if constexpr (G >= 4) h += ((lane >> 3) & 1) * (G / 4);
  if constexpr (G >= 8) h += ((lane >> 2) & 1) * (G / 8);
  return h;
}

// ----------------------------------------------------------------------------- the kernel

// MODE 0: ART off.  MODE 1: ART on, probe = 32 coordinates k*(d/32).  MODE 2: ART on, probe = all d.
// MT: multi-token queries (reading R15) -- rows are (query token, head) pairs and the most recent tokens are cut
// row by row; compiled apart so that plain decode carries none of it.
template <int G, int MODE, bool MT = false>
__global__ void __launch_bounds__(kThreads, (MODE == 2) ? 1 : 2)
art_decode_tc_kernel(const Params p, const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV) {
  constexpr bool ART = MODE != 0;
  constexpr int PW = (MODE == 2) ? kD : 32;          // probe width m
  constexpr int NP = kPVSlots, NS = kSSlots;
  constexpr int LBO_P = p_lbo(G), PBUF = p_buf_bytes(G);
  constexpr bool kTwoPBufs = (G == 8 && MODE == 1);
  constexpr uint32_t kSummaryBytes = (2 + PW) * G * 4;   // mailbox row block of one step: [2 + PW][G] floats

  extern __shared__ __align__(1024) uint8_t smem[];
  const int S = p.stages, M = p.mbox_slots;
  const SmemMap sm = make_smem_map(G, PW, S, M, ART);
  const uint32_t sbase = smem_u32(smem);
  if ((sbase & 1023u) != 0u) __trap();               // the 128-byte swizzle pattern is address based
  const uint32_t bars = sbase + sm.bars;
  auto bar = [&](uint32_t idx) { return bars + idx * 8u; };
  const uint32_t a_ctrl = sbase + sm.misc + kCtrl, a_loaded = sbase + sm.misc + kLoaded, a_tmem = sbase + sm.misc + kTmemPtr;
  constexpr int kIterN = iter_ring(G, MODE == 1);
  float* slots = reinterpret_cast<float*>(smem + sm.slots);   // block i: slots + (i % kIterN) * 3 G = [m_blk | sum lo half | sum hi half][G]
  float* xch = reinterpret_cast<float*>(smem + sm.xch);
  unsigned long long* sinfo = reinterpret_cast<unsigned long long*>(smem + sm.sinfo);   // [S] token masks
  float* mbox = reinterpret_cast<float*>(smem + sm.mbox);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int C = static_cast<int>(cluster_nctarank());
  const int rank = static_cast<int>(cluster_ctarank());
  const int group = blockIdx.x / C;
  const int b = group / p.Hkv, g = group % p.Hkv;
  const int L = p.seq_lens[b];
  const Trav tr = make_trav(p, b, g, L);
  const int Tn = tr.T;
  const int n_c = (Tn > rank) ? (Tn - rank + C - 1) / C : 0;   // steps of this CTA when they are dealt round-robin
  const int n_lim = n_c;                                      // items this CTA will process unless Algorithm 1 fires first
  constexpr int kItemT = item_ring(G, MODE == 1);
  int* item_t = reinterpret_cast<int*>(smem + sm.items);      // step number of item i (i mod kItemT)
  auto item_step = [](int v) { return MT ? (v & kItemStep) : v; };
  const uint32_t a_ntotal = sbase + sm.misc + kNTotal;

#ifdef ART_TRACE
  unsigned long long* cta_times = p.trace ? reinterpret_cast<unsigned long long*>(p.trace + 256 + static_cast<size_t>(kTraceCtas) * kTraceRoles * kTraceEvents * 16) + 4 * blockIdx.x : nullptr;
  if (tid == 0 && cta_times) cta_times[0] = trace_now();
#endif
  // ---- one-time setup: barriers, tensor memory, Q^T
  if (tid == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(bar(sm.full0 + s), 1); mbar_init(bar(sm.empty0 + s), 1); mbar_init(bar(sm.pfull0 + s), 64); }
    for (int s = 0; s < NS; ++s) { mbar_init(bar(sm.sfull0 + s), 1); mbar_init(bar(sm.sfree0 + s), 2); }
    for (int s = 0; s < NP; ++s) { mbar_init(bar(sm.pvfull0 + s), 1); mbar_init(bar(sm.pvfree0 + s), 4); }
    mbar_init(bar(sm.done0), 1); mbar_init(bar(sm.done0 + 1), 1);
    if (ART) {
      for (int s = 0; s < M; ++s) {
        mbar_init(bar(sm.mbox0 + s), 1);
        if (rank == 0 && s < Tn) mbar_arrive_expect_tx(bar(sm.mbox0 + s), kSummaryBytes);   // armed for steps 1..M
      }
    }
    st_volatile_s32(a_ctrl, 0); st_volatile_s32(a_loaded, 0);
    st_volatile_s32(a_ntotal, 0x7fffffff); st_volatile_s32(sbase + sm.misc + 20, 0);
    fence_mbar_init();
  }
  if (warp == kWarpMmaPV) tmem_alloc(a_tmem, kTmemCols);
  {
    // row = i * Gh + h: head h of the group for query token i (R15; one token: row == head)
    const __nv_bfloat16* qp = reinterpret_cast<const __nv_bfloat16*>(p.q) + (static_cast<int64_t>(b) * p.qlen * p.Hq + g * p.Gh) * kD;
    for (int idx = tid; idx < 8 * kD; idx += kThreads) {       // rows >= G: zeros (rows 8-15 alias, see kQLbo)
      const int row = idx / kD, dc = idx % kD;
      const __nv_bfloat16 v = (row < p.Gr) ? qp[((row / p.Gh) * p.Hq + row % p.Gh) * kD + dc] : __float2bfloat16_rn(0.f);
      *reinterpret_cast<__nv_bfloat16*>(smem + sm.qb + (dc >> 3) * kQLbo + row * 16 + (dc & 7) * 2) = v;
    }
    if (tid < 64) reinterpret_cast<__nv_bfloat16*>(smem + sm.qb + 16 * kQLbo)[tid] = __float2bfloat16_rn(0.f);
    uint4* pz = reinterpret_cast<uint4*>(smem + sm.pb);        // P^T rows are read before they are first written
    for (int idx = tid; idx < p_bufs(G, S, MODE == 1) * 2 * PBUF / 16; idx += kThreads) pz[idx] = make_uint4(0u, 0u, 0u, 0u);
  }
  fence_proxy_async();          // Q^T written by threads, read by the tensor core
  tc_fence_before();
  cluster_sync_all();           // barriers of every CTA of the cluster are live before any remote store
  tc_fence_after();
  const uint32_t tmem_base = static_cast<uint32_t>(ld_volatile_s32(a_tmem));
  const uint32_t tmem_S = tmem_base, tmem_PV = tmem_base + NS * kSCols1;

  // "fired and step t lies beyond t*": every wait that could otherwise never end checks this
  auto beyond_stop = [&](int t) -> bool {
    if constexpr (!ART) return false;
    const int c = ld_ctrl_relaxed(a_ctrl);
    return c < 0 && t > -c;
  };
  // A7, bounded run-ahead: the loads of step t are issued only once step t - run_ahead has been decided, so that at most
  // run_ahead blocks per group are loaded and then discarded when Algorithm 1 fires.  False if step t lies beyond t*.
  auto may_issue = [&](int t) -> bool {
    if constexpr (!ART) return true;
    if (p.run_ahead <= 0) return !beyond_stop(t);
    for (;;) {
      const int c = ld_ctrl_relaxed(a_ctrl);
      if (c < 0) return t <= -c;
      if (c >= t - p.run_ahead) return true;
    }
  };
  // Every issued item runs through all roles (one beyond t* is dropped by the fold warps), so every wait below is a plain
  // blocking wait.  When Algorithm 1 fires before the producer has issued its n_lim items, the producer publishes the number it
  // did issue (n_total) and sends ONE more, empty item down the pipeline (END): a role that wakes up for item i >= n_total
  // hands the wake-up on to the next role and leaves.  Nothing polls, and the roles leave as soon as the last real item is
  // through (a wait that also polled "no further item" noticed it only when its try_wait timed out, microseconds later).
  auto is_end = [&](int i) -> bool {
    if constexpr (!ART) return false;
    return i >= ld_volatile_s32(a_ntotal);
  };

  // fold warps: this thread's output coordinate and the running (un-normalised) state; read by the epilogue
  const int fq = warp & 3;
  const int d = fq * 32 + lane;                               // output coordinate == TMEM lane
  float acc[G], m_tot[G], l_tot[G];
#pragma unroll
  for (int h = 0; h < G; ++h) { acc[h] = 0.f; m_tot[h] = kNegInf; l_tot[h] = 0.f; }

  if (warp == kWarpProducer) {
    // ===================================================== A1 + A2: resolve blocks, issue TMA loads
    int it_issued = 0, loaded = 0, stage = 0;
    TC_TRACE_INIT(trc, 0);
    uint32_t ph = 0;                                          // (it / S) & 1
    {
      // ---- steps dealt round-robin: CTA c owns steps c+1, c+1+C, ...; 32 of them are resolved at a time
      auto step_of = [&](int i) { return i * C + rank + 1; };
      bool stop = false;
      for (int i0 = 0; i0 < n_c && !stop; i0 += 32) {
        const int i = i0 + lane;
        unsigned long long mask = 0ull; int c1 = 0, c2 = 0, ec = 0;
        if (i < n_c) {
          const int blk = trav_block(tr, step_of(i));
          mask = block_mask(p, L, blk);
          if constexpr (MT) ec = causal_code(p, L, blk);
          if (mask) {
            const int page = p.block_table[static_cast<int64_t>(b) * p.max_blocks + blk];
            if (p.layout == ART_LAYOUT_HND) { c1 = 0; c2 = page * p.Hkv + g; }     // [page*Hkv + head][token][d]
            else { c1 = page * kBlockTokens; c2 = g; }                             // [page*64 + token][head][d]
          }
        }
        const int cnt = min(32, n_c - i0);
        for (int kk = 0; kk < cnt; ++kk) {
          const int it = i0 + kk, t = step_of(it);
          const unsigned long long mask_k = __shfl_sync(0xffffffffu, mask, kk);
          const int c1_k = __shfl_sync(0xffffffffu, c1, kk), c2_k = __shfl_sync(0xffffffffu, c2, kk);
          int ec_k = 0;
          if constexpr (MT) ec_k = __shfl_sync(0xffffffffu, ec, kk);
          if (!may_issue(t)) { stop = true; break; }           // A7: stop issuing prefetch once fired; bounded run-ahead
          if (it >= S) mbar_wait(bar(sm.empty0 + stage), ph ^ 1u);                // slot released?
          if (lane == 0) {
            TC_TRACE(trc, 1, group, t);
            const uint32_t fb = bar(sm.full0 + stage);
            const uint32_t dst = sbase + sm.ring + stage * kStageBytes;
            item_t[it % kItemT] = t | (ec_k << kItemShift);
            sinfo[stage] = mask_k;
            if (mask_k == 0ull) {
              mbar_arrive(fb);                                 // nothing to load: an all-masked step
            } else {
              mbar_arrive_expect_tx(fb, kStageBytes);
              tma_load_tile(dst, &tmK, c1_k, c2_k, fb);
              tma_load_tile(dst + 2 * kBoxBytes, &tmV, c1_k, c2_k, fb);
            }
          }
          if (mask_k != 0ull) ++loaded;
          it_issued = it + 1;
          if (++stage == S) { stage = 0; ph ^= 1u; }
        }
      }
    }
    if (lane == 0) st_volatile_s32(a_ntotal, it_issued);
    if (lane == 0) st_volatile_s32(a_loaded, loaded);
#ifdef ART_TRACE
    if (lane == 0 && cta_times) cta_times[2] = trace_now();
#endif
    // drain: tensor copies still in flight must land before the CTA reuses the ring or exits (H5)
    for (int j = max(0, it_issued - S); j < it_issued; ++j) mbar_wait(bar(sm.full0 + j % S), (j / S) & 1);
    // END: stopped early, the other roles wait for item it_issued.  It is issued like an all-masked step (its stage must be free:
    // every role has then seen the stage's previous phase), after n_total says that it is not a real one.
    if (ART && it_issued < n_c) {
      if (it_issued >= S) mbar_wait(bar(sm.empty0 + stage), ph ^ 1u);
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(sm.full0 + stage));
    }
  } else if (warp == kWarpMmaS) {
    // ===================================================== A3: S = K_t Q^T, rows = tokens, columns = heads
    if (lane == 0) {
      const uint64_t dK = kDescSw128 | desc_strides(16, 1024);         // K tile, K-major, 128-B swizzle
      const uint64_t dQ = kDescNoSw | desc_strides(kQLbo, kQSbo);
      const uint32_t qb = sbase + sm.qb;
      int st = 0; uint32_t ph = 0;
      TC_TRACE_INIT(trm, 3);
      for (int i = 0; i < n_lim; ++i) {
        const int q = i & (NS - 1);
        mbar_wait(bar(sm.full0 + st), ph);
        if (is_end(i)) {                                      // wake both softmax pairs (their next blocks are i and i + 1)
          for (int j = 0; j < 2; ++j) {
            const int ii = i + j, qq = ii & (NS - 1);
            if (ii >= NS) mbar_wait(bar(sm.sfree0 + qq), ((ii / NS) - 1) & 1);
            umma_commit(bar(sm.sfull0 + qq));
          }
          break;
        }
        TC_TRACE(trm, 2, i, 0);
        if (i >= NS) mbar_wait(bar(sm.sfree0 + q), ((i / NS) - 1) & 1);
        TC_TRACE(trm, 10, i, 0);
        tc_fence_after();
        // M = 128 rows are read starting at the tile (even blocks: tokens 0-63 -> TMEM lanes 0-63) or 64 token rows
        // BELOW it (odd blocks: tokens 0-63 -> lanes 64-127).  The other 64 rows are whatever lies next to the tile
        // and only feed lanes nobody reads.
        const uint32_t kt = sbase + sm.ring + st * kStageBytes - (i & 1) * kBoxBytes;
        const uint32_t dcol = tmem_S + q * kSCols1;
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {                      // 8 x 16 = head_dim
          const uint32_t ka = kt + (ks >> 2) * kBoxBytes + (ks & 3) * 32;
          umma_bf16(dcol, dK | desc_addr(ka), dQ | desc_addr(qb + ks * 2 * kQLbo), kIdescS, ks > 0);
        }
        umma_commit(bar(sm.sfull0 + q));
        if (++st == S) { st = 0; ph ^= 1u; }
      }
      umma_commit(bar(sm.done0));                             // every MMA retired before TMEM is released
      mbar_wait(bar(sm.done0), 0);
    }
  } else if (warp == kWarpMmaPV) {
    // ===================================================== A5: P~V_t = V_t^T P^T, rows = d, columns = heads
    if (lane == 0) {
      const uint64_t dV = kDescSw128 | desc_strides(kBoxBytes, 1024);  // V tile as V^T: MN-major, 128-B swizzle
      // P^T (hi) and P^T (lo) are ONE B operand of N = 16 rows: rows 0-7 = hi of heads 0-7, rows 8-15 = lo (the stride
      // between the two 8-row groups is the distance of the lo buffer), so P~V_t costs 4 MMAs: accumulator columns
      // 0-7 = V^T hi, 8-15 = V^T lo, added by whoever reads them (an MMA costs what its A operand costs to read)
      const uint64_t dP = kDescNoSw | desc_strides(LBO_P, PBUF);
      int st = 0; uint32_t ph = 0;
      TC_TRACE_INIT(trv, 5);
      for (int i = 0; i < n_lim; ++i) {
        const int ps = i & (NP - 1);
        mbar_wait(bar(sm.pfull0 + st), ph);
        if (is_end(i)) break;
        TC_TRACE(trv, 6, i, 0);
        if (i >= NP) mbar_wait(bar(sm.pvfree0 + ps), ((i / NP) - 1) & 1);
        TC_TRACE(trv, 11, i, 0);
        tc_fence_after();
        const uint32_t vt = sbase + sm.ring + st * kStageBytes + 2 * kBoxBytes;
        const uint32_t pb = sbase + sm.pb + (kTwoPBufs ? (i & 1) : st) * 2 * PBUF;
#pragma unroll
        for (int ks = 0; ks < 4; ++ks)                        // 4 x 16 = tokens of the block; p = hi + lo side by side
          umma_bf16(tmem_PV + ps * kUmmaN, dV | desc_addr(vt + ks * 2048),
                    dP | desc_addr(pb + ks * 2 * LBO_P), kIdescPV, ks > 0);
        umma_commit(bar(sm.empty0 + st));                     // K/V stage and its P buffer are free again
        umma_commit(bar(sm.pvfull0 + ps));
        if (++st == S) { st = 0; ph ^= 1u; }
      }
      umma_commit(bar(sm.done0 + 1));
      mbar_wait(bar(sm.done0 + 1), 0);
    }
  } else if (warp >= kWarpSoftmax0 && warp < kWarpSoftmax0 + 4) {
    // ===================================================== A4: block-local softmax, one token per thread, two warps per block
    const int q = warp - kWarpSoftmax0;                       // TMEM lane quadrant == warp % 4
    const int pair = q >> 1, half = q & 1;                    // the pair owns blocks i = pair (mod 2); this warp tokens 32 half + lane
    const int tok = half * 32 + lane;
    const uint32_t tq = static_cast<uint32_t>(q * 32) << 16;
    int st = pair % S;                                        // ring stage of block i
    TC_TRACE_INIT(trx, 4);
    for (int i = pair; i < n_lim; i += 2) {
      const int sslot = i & (NS - 1);
      mbar_wait(bar(sm.sfull0 + sslot), (i / NS) & 1);
      if constexpr (ART) {
        const int nt = ld_volatile_s32(a_ntotal);
        if (i >= nt) {                                        // END: the pair that owns the END item hands it on to the P.V issuer
          if (i == nt) mbar_arrive(bar(sm.pfull0 + st));
          break;
        }
      }
      if (q == 0 && lane == 0) TC_TRACE(trx, 3, i, 0);
      tc_fence_after();
      float sv[G];
      tmem_ld<G>(tmem_S + sslot * kSCols1 + tq, sv);
      tmem_ld_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(sm.sfree0 + sslot));
      // P^T buffer i & 1 is read by the P.V MMA of block i - 2: wait until that one is complete
      if (kTwoPBufs && i >= 2) mbar_wait(bar(sm.pvfull0 + ((i - 2) & (NP - 1))), ((i - 2) / NP) & 1);
      const unsigned long long vmask = sinfo[st];             // written before the loads the S MMA waited for
      const bool v0 = (vmask >> tok) & 1ull;
      float mb[G];
      int ec = 0;
      if constexpr (MT) ec = item_t[i % kItemT] >> kItemShift;
#pragma unroll
      for (int h = 0; h < G; ++h) {
        bool vis = v0;                                        // masked tokens: weight 0 (R8); their K may be NaN
        if (MT && ec != 0) vis = vis && tok < ec - static_cast<int>((p.cuts >> (4 * h)) & 15u);   // R15: causal cut row by row
        sv[h] = vis ? sv[h] * p.scale_log2 : kNegInf;
        mb[h] = warp_max_f32(sv[h]);
      }
      {
        // block maximum = max over the two halves: through shared memory and the pair's named barrier.  The area is
        // double-buffered by block parity: a warp can be at most one block ahead of its partner at the barrier.
        float* xw = xch + (((pair * 2 + ((i >> 1) & 1)) * 2) + half) * G;
        const float* xr = xch + (((pair * 2 + ((i >> 1) & 1)) * 2) + (half ^ 1)) * G;
        float mine = mb[0];
#pragma unroll
        for (int h = 1; h < G; ++h) mine = (lane == h) ? mb[h] : mine;
        if (lane < G) xw[lane] = mine;
        asm volatile("bar.sync %0, 64;" :: "r"(2 + pair) : "memory");   // named barriers 2, 3 (0: __syncthreads, 1: fold warps of the persistent kernel)
#pragma unroll
        for (int h = 0; h < G; ++h) mb[h] = fmaxf(mb[h], xr[h]);
      }
      uint8_t* pb0 = smem + sm.pb + (kTwoPBufs ? (i & 1) : st) * 2 * PBUF + (half * 4 + (lane >> 3)) * LBO_P + (lane & 7) * 2;   // token `tok`, row 0, hi
      float ls[G];
#pragma unroll
      for (int h = 0; h < G; ++h) {
        const float p0 = (sv[h] != kNegInf) ? fast_exp2(sv[h] - mb[h]) : 0.f;
        const __nv_bfloat16 h0 = __float2bfloat16_rn(p0);
        const __nv_bfloat16 l0 = __float2bfloat16_rn(p0 - __bfloat162float(h0));
        *reinterpret_cast<__nv_bfloat16*>(pb0 + h * 16) = h0;
        *reinterpret_cast<__nv_bfloat16*>(pb0 + h * 16 + PBUF) = l0;
        ls[h] = __bfloat162float(h0) + __bfloat162float(l0);  // the weight the tensor core really uses
      }
      if (vmask != ~0ull && !v0) {                            // masked V rows may hold NaN: 0 * NaN would poison P~V
        uint4* vr = reinterpret_cast<uint4*>(smem + sm.ring + st * kStageBytes + 2 * kBoxBytes);
#pragma unroll
        for (int c = 0; c < 8; ++c) { vr[tok * 8 + c] = make_uint4(0u, 0u, 0u, 0u); vr[tok * 8 + c + kBoxBytes / 16] = make_uint4(0u, 0u, 0u, 0u); }
      }
      // sum of this half's weights per head: lane l ends up with the total of head head_of_lane32(l)
      Reduce32<G, 16>::run(ls, lane);
      {
        const int hh = head_of_lane32<G>(lane);
        float mine = mb[0];
#pragma unroll
        for (int h = 1; h < G; ++h) mine = (hh == h) ? mb[h] : mine;
        float* slot = slots + (i % kIterN) * 3 * G;
        if ((lane & (32 / G - 1)) == 0) { if (half == 0) slot[hh] = mine; slot[(1 + half) * G + hh] = ls[0]; }
      }
      fence_proxy_async();                                    // P^T (and V fixes) visible to the tensor core
      mbar_arrive(bar(sm.pfull0 + st));
      if (q == 0 && lane == 0) TC_TRACE(trx, 9, i, 0);
      st += 2; while (st >= S) st -= S;
    }
  } else if (warp < kWarpFold0 + 4) {
    // ===================================================== A5 / A6: publish step summaries, merge P~V_t
    const uint32_t tlane = static_cast<uint32_t>(fq * 32) << 16;
    TC_TRACE_INIT(trf, 1);
    auto release_pv = [&](int i) {                           // the tensor-memory slot of item i is free again
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(sm.pvfree0 + (i & (NP - 1))));
    };
    // merge block i (its P~V_t is relative to its own block maximum) into the running state
    auto fold = [&](int i) {
      if (tid == 0) TC_TRACE(trf, 20, i, 0);
      tc_fence_after();
      float pv[G], pvl[G];
      tmem_ld<G>(tmem_PV + tlane + (i & (NP - 1)) * kUmmaN, pv);
      tmem_ld<G>(tmem_PV + tlane + (i & (NP - 1)) * kUmmaN + 8, pvl);
      tmem_ld_wait();
      if (tid == 0) TC_TRACE(trf, 21, i, 0);
#pragma unroll
      for (int h = 0; h < G; ++h) pv[h] += pvl[h];            // hi + lo halves of p
      const float* sl = slots + (i % kIterN) * 3 * G;
#pragma unroll
      for (int h = 0; h < G; ++h) {                           // branch-free, so that the heads' chains overlap
        const float mr = sl[h];
        const bool some = mr != kNegInf;                      // a block with no valid token changes nothing
        const float mn = fmaxf(m_tot[h], mr);
        const float a = (m_tot[h] == mn) ? 1.f : fast_exp2(m_tot[h] - mn);
        const float bb = some ? fast_exp2(mr - mn) : 0.f;
        acc[h] = some ? fmaf(a, acc[h], bb * pv[h]) : acc[h];
        l_tot[h] = some ? fmaf(a, l_tot[h], bb * (sl[G + h] + sl[2 * G + h])) : l_tot[h];
        m_tot[h] = mn;
      }
      if (tid == 0) TC_TRACE(trf, 22, i, 0);
      release_pv(i);
      if (tid == 0) TC_TRACE(trf, 5, i, item_step(item_t[i % kItemT]));
    };
    if constexpr (!ART) {
      for (int i = 0; i < n_lim; ++i) {
        mbar_wait(bar(sm.pvfull0 + (i & (NP - 1))), (i / NP) & 1);
        fold(i);
      }
    } else {
      int pub = 0, fld = 0;
      bool pub_ready = false;                                 // P~V of block `pub` is complete in tensor memory
      int t_fld = 0, t_pub = 0;                               // steps of items fld (valid while fld < pub) and pub (valid while pub_ready)
      // the thread that ships (m_blk, block sum) of a step: not one of warp 0's, whose lanes ship probe values first
      const bool ml_thread = (tid == 97);
      while (fld < n_lim) {
        const int2 cn = ld_ctrl_ntotal(a_ctrl);
        const int c = cn.x, ntot = cn.y;
        if (fld >= ntot) break;
        // ---- merge the oldest unfolded block once the decision for the steps before it is known; one that
        //      lies beyond t* is dropped (its tensor-memory slot is released, nothing is merged)
        if (fld < pub) {
          if (c < 0 && t_fld > -c) { release_pv(fld); ++fld; t_fld = item_step(item_t[fld % kItemT]); continue; }
          if (c < 0 || c >= t_fld - 1) { fold(fld); ++fld; t_fld = item_step(item_t[fld % kItemT]); continue; }
        }
        // ---- publish the summary of the next finished block (never waits for a decision on itself)
        if (pub < ntot && pub < n_lim && pub - fld < NP) {
          if (!pub_ready) {
            const uint32_t pvb = bar(sm.pvfull0 + (pub & (NP - 1)));
            const uint32_t par = (pub / NP) & 1;
            pub_ready = (fld == pub) ? mbar_try_wait(pvb, par) : mbar_test_wait(pvb, par);
            if (pub_ready) { t_pub = item_step(item_t[pub % kItemT]); if (tid == 0) TC_TRACE(trf, 7, pub, 0); }
          }
          if (pub_ready && c < 0) { ++pub; pub_ready = false; continue; }   // fired: an unpublished step lies beyond t*
          if (pub_ready && c >= t_pub - M) {                  // mailbox slot free: step t - M has been scanned
            const int t = t_pub;
            const int slot_i = (t - 1) & (M - 1);
            const uint32_t row0 = mapa(sbase + sm.mbox + static_cast<uint32_t>(slot_i) * kSummaryBytes, 0);
            const uint32_t mb = mapa(bar(sm.mbox0 + slot_i), 0);
            tc_fence_after();
            float pv[G], pvl[G];
            tmem_ld<G>(tmem_PV + tlane + (pub & (NP - 1)) * kUmmaN, pv);
            tmem_ld<G>(tmem_PV + tlane + (pub & (NP - 1)) * kUmmaN + 8, pvl);
            if (ml_thread) {                                  // (overlaps the tensor-memory loads)
              const float* sl = slots + (pub % kIterN) * 3 * G;
              float ml[2 * G];
#pragma unroll
              for (int h = 0; h < G; ++h) { ml[h] = sl[h]; ml[G + h] = sl[G + h] + sl[2 * G + h]; }
              st_async_vec<G>(row0, ml, mb);
              st_async_vec<G>(row0 + G * 4u, ml + G, mb);
            }
            tmem_ld_wait();
            if (tid == 0) TC_TRACE(trf, 23, pub, 0);
#pragma unroll
            for (int h = 0; h < G; ++h) pv[h] += pvl[h];
            if (MODE == 2 || (d & 3) == 0) {
              const int pi = (MODE == 2) ? d : (d >> 2);      // probe coordinate k*(d/32)  (R1)
              st_async_vec<G>(row0 + (2 + pi) * G * 4u, pv, mb);
            }
            if (tid == 0) { TC_TRACE(trf, 4, pub, t); TC_TRACE(trf, 13, t, c < 0 ? 0 : c); }
            if (fld == pub) t_fld = t;
            ++pub; pub_ready = false;
            continue;
          }
        }
      }
    }
  } else if (ART && warp == kWarpScan && rank == 0) {
    // ===================================================== A6 + A7 + A9: Algorithm 1 over step summaries
    using Scan = ScanCore<G, PW>;
    constexpr int LPH = Scan::LPH, CPL = Scan::CPL;
    const int h = lane / LPH, sub = lane % LPH;
    Scan sc; sc.init(); sc.g_real = p.Gr;
    TC_TRACE_INIT(trs, 2);
    const uint32_t mb_lane = sbase + sm.mbox + h * 4u;         // this lane's head column of a mailbox row block
    int t_stop = 0;
    int t = 1;
    const int mshift = 31 - __clz(M);                         // M is a power of two
    // a batch takes at most half of the mailbox, so that the other half can fill while it is decided (M = 8 for eight rows
    // per group: batches of 4; a batch of 8 there made publishers and scan take turns: 2.5 -> 3.0 steps/us for a cluster of 4)
    const int nmax = (M / 2 < kScanBatch) ? M / 2 : kScanBatch;
    while (t <= Tn) {
      const int i0 = t - 1;                                   // 0-based step index of the batch head
      mbar_wait(bar(sm.mbox0 + (i0 & (M - 1))), (i0 >> mshift) & 1);
      if (lane == 0) TC_TRACE(trs, 14, t, 0);
      // how many of the following steps have arrived as well (lane k probes step t + k)
      int n = 1;
      {
        bool ok = false;
        if (lane >= 1 && lane < kScanBatch && t + lane <= Tn)
          ok = mbar_test_wait(bar(sm.mbox0 + ((i0 + lane) & (M - 1))), ((i0 + lane) >> mshift) & 1);
        const uint32_t bits = __ballot_sync(0xffffffffu, ok) | 1u;
        n = __ffs(~bits) - 1;
        n = n > nmax ? nmax : n;
        __syncwarp();                                         // the probing lane's acquire covers the whole warp
      }
      const int fired = sc.batch(n, lane, p.tau, p.phi, p.patience,
        [&](int k, bool live, float& mt, float& lt) {
          const uint32_t a = mb_lane + static_cast<uint32_t>((i0 + k) & (M - 1)) * kSummaryBytes;
          const float m_ = lds_f32(a), l_ = lds_f32(a + G * 4u);     // a slot that is not part of the batch
          mt = live ? m_ : kNegInf; lt = live ? l_ : 0.f;            // may hold anything: select, never use
        },
        [&](int k, bool live, float (&pv)[CPL]) {
          const uint32_t a = mb_lane + static_cast<uint32_t>((i0 + k) & (M - 1)) * kSummaryBytes + (2 + sub) * G * 4u;
#pragma unroll
          for (int j = 0; j < CPL; ++j) { const float v = lds_f32(a + LPH * j * G * 4u); pv[j] = live ? v : 0.f; }
        });
      __syncwarp();
      if (fired < 0 && lane < n && t + lane + M <= Tn)        // re-arm the consumed slots for steps t + k + M
        mbar_arrive_expect_tx(bar(sm.mbox0 + ((i0 + lane) & (M - 1))), kSummaryBytes);
      __syncwarp();
      const int t_last = fired >= 0 ? t + fired : t + n - 1;
      if (lane == 0) TC_TRACE(trs, 8, (group << 12) | t, n);
      if (lane < C) st_cluster_relaxed_s32(mapa(a_ctrl, lane), fired >= 0 ? -t_last : t_last);
      if (fired >= 0) { t_stop = t_last; break; }
      t += n;
    }
    if (lane == 0) p.stop_block[group] = t_stop ? t_stop : Tn;               // t* (R9)
  }

  // ===================================================== A8 / A9: combine the partial states, write out
  tc_fence_before();
  __syncthreads();                                            // ring is free: all loads drained, all MMAs retired
  float* cta = reinterpret_cast<float*>(smem + sm.ring);
  float* cta_m = cta + G * kD;
  float* cta_l = cta_m + G;
  if (warp < kWarpFold0 + 4) {
#pragma unroll
    for (int h = 0; h < G; ++h) {
      cta[h * kD + d] = acc[h];
      if (d == 0) { cta_m[h] = m_tot[h]; cta_l[h] = l_tot[h]; }
    }
  }
  cluster_sync_all();
  if (rank == 0) {
    for (int o = tid; o < G * kD; o += kThreads) {
      const int h = o / kD;
      float mx = kNegInf;
      for (int c = 0; c < C; ++c) mx = fmaxf(mx, ld_cluster_f32(mapa(smem_u32(&cta_m[h]), c)));
      float a = 0.f, l = 0.f;
      for (int c = 0; c < C; ++c) {
        const float mc = ld_cluster_f32(mapa(smem_u32(&cta_m[h]), c));
        const float f = (mc == kNegInf) ? 0.f : fast_exp2(mc - mx);
        a = fmaf(f, ld_cluster_f32(mapa(smem_u32(&cta[o]), c)), a);
        l = fmaf(f, ld_cluster_f32(mapa(smem_u32(&cta_l[h]), c)), l);
      }
      if (h < p.Gr)                                             // Alg. 1 l.18; row h = query token h / Gh, head h % Gh
        p.out[((static_cast<int64_t>(b) * p.qlen + h / p.Gh) * p.Hq + g * p.Gh + h % p.Gh) * kD + (o - h * kD)] = (l > 0.f) ? a / l : 0.f;
    }
    if (tid == 0) {
      if (!ART) p.stop_block[group] = Tn;
      if (p.blocks_loaded) {
        int tot = 0;
        for (int c = 0; c < C; ++c) tot += ld_cluster_s32(mapa(a_loaded, c));
        p.blocks_loaded[group] = tot;
      }
    }
  }
  cluster_sync_all();                                         // peers' shared memory stays alive until read
  if (warp == kWarpMmaPV) { tc_fence_after(); tmem_dealloc(tmem_base, kTmemCols); }
#ifdef ART_TRACE
  if (tid == 0 && cta_times) cta_times[1] = trace_now();
#endif
}

}  // namespace tc
}  // namespace art
