// ART decode attention, Blackwell tensor-core kernel (bf16 KV, head_dim 128): tcgen05 + TMEM + TMA.
//
// One thread-block CLUSTER of C CTAs per query group (sequence b, KV head g); traversal steps
// t = 1..T are dealt round-robin, CTA c owns steps c+1, c+1+C, ...  Inside a CTA
// one 64-token KV block is one pipeline item, handled by specialised warps that only meet through
// mbarriers:
//
//   producer  (warp 0)     A1/A2  resolves block -> page, issues 4 TMA tensor boxes (K, V: two
//                                 64-column halves each, 128-byte swizzle) into a ring of stages
//   MMA       (warp 1, 1 thread)  A3  S[token, head]  = K_t . Q^T      tcgen05.mma M128 N16 K16 x8
//                                 A5  PV[d, head]     = V_t^T . P^T    tcgen05.mma M128 N16 K16 x8
//                                 both with fp32 accumulators in TENSOR MEMORY
//   softmax   (warps 4-7)  A4     two groups of two warps (even / odd blocks), one thread per token:
//                                 tcgen05.ld S, running max, p = 2^(s-m); p is split into bf16 hi + lo
//                                 (keeps ~16 mantissa bits, so the probe of P~V_t is accurate to ~1e-5
//                                 and the criterion does not flip) and written to shared memory as the
//                                 B operand of the P.V MMA.  Each group is its own online-softmax stream.
//   fold      (warps 8-11) A5/A6  one thread per output coordinate: tcgen05.ld P~V_t, publishes the
//                                 step summary (reference max, block sum, probe components of P~V_t)
//                                 to the cluster leader's mailbox (st.async + mbarrier complete_tx, no
//                                 fences), and folds P~V_t into the running accumulator only once the
//                                 leader has decided that step t <= t*
//   scan      (warp 2, leader CTA)  A6/A7/A9  replays Algorithm 1 (Eq. 2-3)
//                                 sequentially over the step summaries, broadcasts progress / t*
//
// The block-local P~V_t of up to 16 steps wait UNFOLDED in tensor memory (16 x 16 columns), so the
// loads, the MMAs and the softmax never wait for the sequential decision; blocks with step > t* are
// simply never folded, which makes the result equal to the sequential algorithm's for any C.
#pragma once
#include <cuda.h>   // CUtensorMap (type only: the encoder is fetched through the runtime, no -lcuda)

#include "art_common.cuh"

namespace art {
namespace tc {

constexpr int kThreads = 384;
constexpr int kWarpProducer = 0, kWarpMma = 1, kWarpScan = 2, kWarpTmem = 3, kWarpSoftmax0 = 4, kWarpFold0 = 8;
constexpr int kD = 128;                      // head_dim
constexpr int kUmmaN = 16;                   // MMA N: the group's heads padded to 16
constexpr int kSSlots = 4;                   // S accumulators in flight (16 TMEM columns each)
constexpr int kPVSlots = 16;                 // unfolded P~V_t results (16 TMEM columns each)
constexpr int kTmemCols = 512;
constexpr int kBoxBytes = 8192;              // one TMA box: 64 rows x 128 bytes
constexpr int kQLbo = 256, kQSbo = 128;      // Q^T as B operand: [16 d-chunks][16 rows][16 B]
constexpr int kQBytes = 16 * kQLbo;
constexpr int kPLbo = 272, kPSbo = 128;      // P^T as B operand: [8 token-chunks][16 rows][16 B] (+16 B pad:
constexpr int kPBufBytes = 2304;             //   the 4 chunks a warp writes fall into distinct banks)

struct IterSlot {            // what softmax hands to fold for one block (ring of kPVSlots)
  float alpha[8];            // 2^(m_old - m_new): rescale of everything its stream folded before this block
  float mref[8];             // m_new: reference exponent of this block's p (log2 domain)
  float lsum[2][8];          // per softmax warp: sum of the block's (rounded) p
};

struct SmemMap {
  uint32_t qb, pb, slots, sinfo, xchg, mbox, bars, misc, ring, total;
  uint32_t full0, empty0, sfull0, sfree0, pfull0, pvfull0, pvfree0, xchg0, done0, mbox0, nbars;
};

// Offsets from a 1024-byte aligned base.  The small buffers come first: the S MMA of odd blocks reads
// 8 KiB below its K tile (rows that only feed unused accumulator lanes), which must be mapped memory.
__host__ __device__ inline SmemMap make_smem_map(int G, int PW, int stages, int mslots, bool art) {
  SmemMap m;
  uint32_t off = 0;
  m.qb = off; off += kQBytes;
  m.pb = off; off += static_cast<uint32_t>(stages) * 2u * kPBufBytes;
  m.slots = off; off += kPVSlots * static_cast<uint32_t>(sizeof(IterSlot));
  m.sinfo = off; off += static_cast<uint32_t>(stages) * 16u;
  m.xchg = off; off += 2u * 2u * 2u * 8u * 4u;
  m.mbox = off; off += art ? static_cast<uint32_t>(mslots) * G * (2 + PW) * 4u : 0u;
  off = (off + 15u) & ~15u;
  m.bars = off;
  uint32_t n = 0;
  m.full0 = n; n += stages; m.empty0 = n; n += stages; m.pfull0 = n; n += stages;
  m.sfull0 = n; n += kSSlots; m.sfree0 = n; n += kSSlots;
  m.pvfull0 = n; n += kPVSlots; m.pvfree0 = n; n += kPVSlots;
  m.xchg0 = n; n += 4; m.done0 = n; n += 1;
  m.mbox0 = n; n += art ? mslots : 0;
  m.nbars = n;
  off += n * 8u;
  m.misc = off; off += 128u;             // ctrl, loaded, tmem_ptr, cta_m[8], cta_l[8]
  off = (off + 1023u) & ~1023u;
  if (off < 8192u) off = 8192u;
  m.ring = off; off += static_cast<uint32_t>(stages) * kStageBytes;
  m.total = off + 1024u;                 // + slack: the base is aligned to 1024 B at run time
  return m;
}
constexpr uint32_t kCtrl = 0, kLoaded = 4, kTmemPtr = 8, kCtaM = 32, kCtaL = 64;

// ----------------------------------------------------------------------------- tcgen05 / TMA wrappers

__device__ __forceinline__ void tma_load_box(uint32_t dst, const CUtensorMap* tm, int c0, int c1, int c2, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
               :: "r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
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

// ----------------------------------------------------------------------------- the kernel

// MODE 0: ART off.  MODE 1: ART on, probe = 32 coordinates k*(d/32).  MODE 2: ART on, probe = all d.
template <int G, int MODE>
__global__ void __launch_bounds__(kThreads, 1)
art_decode_tc_kernel(const Params p, const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV) {
  constexpr bool ART = MODE != 0;
  constexpr int PW = (MODE == 2) ? kD : 32;          // probe width m
  constexpr int NP = kPVSlots, NS = kSSlots;
  constexpr uint32_t kSummaryBytes = (2 + PW) * G * 4;   // mailbox row block of one step: [2 + PW][G] floats
  static_assert((NP & (NP - 1)) == 0 && (NS & (NS - 1)) == 0, "slot rings are indexed with masks");

  extern __shared__ uint8_t smem_raw[];
  const int S = p.stages, M = p.mbox_slots;
  const SmemMap sm = make_smem_map(G, PW, S, M, ART);
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  uint8_t* smem = smem_raw + (sbase - smem_u32(smem_raw));
  const uint32_t bars = sbase + sm.bars;
  auto bar = [&](uint32_t idx) { return bars + idx * 8u; };
  const uint32_t a_ctrl = sbase + sm.misc + kCtrl, a_loaded = sbase + sm.misc + kLoaded, a_tmem = sbase + sm.misc + kTmemPtr;
  IterSlot* slots = reinterpret_cast<IterSlot*>(smem + sm.slots);
  unsigned long long* sinfo = reinterpret_cast<unsigned long long*>(smem + sm.sinfo);   // [S][2]: mask, pad
  float* xchg = reinterpret_cast<float*>(smem + sm.xchg);                               // [group][parity][warp][8]
  float* mbox = reinterpret_cast<float*>(smem + sm.mbox);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int C = static_cast<int>(cluster_nctarank());
  const int rank = static_cast<int>(cluster_ctarank());
  const int group = blockIdx.x / C;
  const int b = group / p.Hkv, g = group % p.Hkv;
  const int L = p.seq_lens[b];
  const Trav tr = make_trav(p, b, g, L);
  const int Tn = tr.T;
  const int n_c = (Tn > rank) ? (Tn - rank + C - 1) / C : 0;   // steps owned by this CTA

  // ---- one-time setup: barriers, tensor memory, Q^T and the zero padding rows of P^T
  if (tid == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(bar(sm.full0 + s), 1); mbar_init(bar(sm.empty0 + s), 1); mbar_init(bar(sm.pfull0 + s), 64); }
    for (int s = 0; s < NS; ++s) { mbar_init(bar(sm.sfull0 + s), 1); mbar_init(bar(sm.sfree0 + s), 2); }
    for (int s = 0; s < NP; ++s) { mbar_init(bar(sm.pvfull0 + s), 1); mbar_init(bar(sm.pvfree0 + s), 4); }
    for (int s = 0; s < 4; ++s) mbar_init(bar(sm.xchg0 + s), 2);
    mbar_init(bar(sm.done0), 1);
    if (ART) {
      for (int s = 0; s < M; ++s) {
        mbar_init(bar(sm.mbox0 + s), 1);
        if (rank == 0 && s < Tn) mbar_arrive_expect_tx(bar(sm.mbox0 + s), kSummaryBytes);   // armed for steps 1..M
      }
    }
    st_volatile_s32(a_ctrl, 0); st_volatile_s32(a_loaded, 0);
    fence_mbar_init();
  }
  if (warp == kWarpTmem) tmem_alloc(a_tmem, kTmemCols);
  {
    const __nv_bfloat16* qp = reinterpret_cast<const __nv_bfloat16*>(p.q) + (static_cast<int64_t>(b) * p.Hq + g * G) * kD;
    for (int idx = tid; idx < 16 * kD; idx += kThreads) {
      const int row = idx / kD, dc = idx % kD;
      const __nv_bfloat16 v = (row < G) ? qp[row * kD + dc] : __float2bfloat16_rn(0.f);
      *reinterpret_cast<__nv_bfloat16*>(smem + sm.qb + (dc >> 3) * kQLbo + row * 16 + (dc & 7) * 2) = v;
    }
    uint4* pz = reinterpret_cast<uint4*>(smem + sm.pb);
    for (int idx = tid; idx < S * 2 * kPBufBytes / 16; idx += kThreads) pz[idx] = make_uint4(0u, 0u, 0u, 0u);
  }
  fence_proxy_async();          // Q^T / P^T padding written by threads, read by the tensor core
  tc_fence_before();
  cluster_sync_all();           // barriers of every CTA of the cluster are live before any remote store
  tc_fence_after();
  const uint32_t tmem_base = static_cast<uint32_t>(ld_volatile_s32(a_tmem));
  const uint32_t tmem_S = tmem_base, tmem_PV = tmem_base + NS * kUmmaN;

  // "fired and step t lies beyond t*": every wait that could otherwise never end checks this
  auto beyond_stop = [&](int t) -> bool {
    if constexpr (!ART) return false;
    const int c = ld_ctrl_relaxed(a_ctrl);
    return c < 0 && t > -c;
  };
  auto wait_or_stop = [&](uint32_t baddr, uint32_t parity, int t) -> bool {
    while (!mbar_try_wait(baddr, parity)) { if (beyond_stop(t)) return false; }
    return true;
  };
  auto step_of = [&](int i) { return i * C + rank + 1; };

  // fold warps: this thread's output coordinate and the running (un-normalised) state of the two
  // softmax streams (even / odd blocks); read by the epilogue
  const int fq = (warp - kWarpFold0) & 3;
  const int d = fq * 32 + lane;                               // output coordinate == TMEM lane
  float acc0[G], acc1[G], m0[G], m1[G], l0[G], l1[G];
#pragma unroll
  for (int h = 0; h < G; ++h) { acc0[h] = acc1[h] = 0.f; m0[h] = m1[h] = kNegInf; l0[h] = l1[h] = 0.f; }

  if (warp == kWarpProducer) {
    // ===================================================== A1 + A2: resolve blocks, issue TMA loads
    int it_issued = 0, loaded = 0, stage = 0;
    uint32_t ph = 0;                                          // (it / S) & 1
    bool stop = false;
    for (int i0 = 0; i0 < n_c && !stop; i0 += 32) {
      const int i = i0 + lane;
      unsigned long long mask = 0ull; int c1 = 0, c2 = 0;
      if (i < n_c) {
        const int blk = trav_block(tr, step_of(i));
        mask = block_mask(p, L, blk);
        if (mask) {
          const int page = p.block_table[static_cast<int64_t>(b) * p.max_blocks + blk];
          if (p.layout == ART_LAYOUT_HND) { c1 = 0; c2 = page * p.Hkv + g; }     // [page*Hkv + head][token][d]
          else { c1 = g; c2 = page * kBlockTokens; }                             // [page*64 + token][head][d]
        }
      }
      const int cnt = min(32, n_c - i0);
      for (int kk = 0; kk < cnt; ++kk) {
        const int it = i0 + kk, t = step_of(it);
        const unsigned long long mask_k = __shfl_sync(0xffffffffu, mask, kk);
        const int c1_k = __shfl_sync(0xffffffffu, c1, kk), c2_k = __shfl_sync(0xffffffffu, c2, kk);
        if (it >= S && !wait_or_stop(bar(sm.empty0 + stage), ph ^ 1u, t)) stop = true;   // slot released?
        if (!stop && beyond_stop(t)) stop = true;            // A7: stop issuing prefetch once fired
        if (stop) break;
        if (lane == 0) {
          const uint32_t fb = bar(sm.full0 + stage);
          const uint32_t dst = sbase + sm.ring + stage * kStageBytes;
          sinfo[stage * 2] = mask_k;
          if (mask_k == 0ull) {
            mbar_arrive(fb);                                 // nothing to load: an all-masked step
          } else {
            mbar_arrive_expect_tx(fb, kStageBytes);
            tma_load_box(dst, &tmK, 0, c1_k, c2_k, fb);
            tma_load_box(dst + kBoxBytes, &tmK, 64, c1_k, c2_k, fb);
            tma_load_box(dst + 2 * kBoxBytes, &tmV, 0, c1_k, c2_k, fb);
            tma_load_box(dst + 3 * kBoxBytes, &tmV, 64, c1_k, c2_k, fb);
          }
        }
        if (mask_k != 0ull) ++loaded;
        it_issued = it + 1;
        if (++stage == S) { stage = 0; ph ^= 1u; }
      }
    }
    if (lane == 0) st_volatile_s32(a_loaded, loaded);
    // drain: tensor copies still in flight must land before the CTA reuses the ring or exits (H5)
    for (int j = max(0, it_issued - S); j < it_issued; ++j) mbar_wait(bar(sm.full0 + j % S), (j / S) & 1);
  } else if (warp == kWarpMma) {
    // ===================================================== A3 + A5: the two MMAs of every block
    if (lane == 0) {
      const uint64_t dK = kDescSw128 | desc_strides(16, 1024);         // K tile, K-major, 128-B swizzle
      const uint64_t dV = kDescSw128 | desc_strides(kBoxBytes, 1024);  // V tile as V^T: MN-major, 128-B swizzle
      const uint64_t dQ = kDescNoSw | desc_strides(kQLbo, kQSbo);
      const uint64_t dP = kDescNoSw | desc_strides(kPLbo, kPSbo);
      const uint32_t qb = sbase + sm.qb;
      int si = 0, pi = 0;                                     // next block whose S / P.V MMAs are to be issued
      int s_st = 0, p_st = 0; uint32_t s_ph = 0, p_ph = 0;    // their ring stage and (i / S) & 1
      while (pi < n_c) {
        bool did = false;
        if (si < n_c && mbar_try_wait(bar(sm.full0 + s_st), s_ph) &&
            (si < NS || mbar_try_wait(bar(sm.sfree0 + (si & (NS - 1))), ((si / NS) - 1) & 1))) {
          // S = K_t Q^T: rows = tokens, columns = heads.  M = 128 rows are read starting 8 KiB BELOW the K tile
          // for odd blocks, so their 64 tokens land in TMEM lanes 64-127 (softmax group 1); the other 64 rows
          // are whatever lies next to the tile and only feed lanes nobody reads.
          tc_fence_after();
          const uint32_t kt = sbase + sm.ring + s_st * kStageBytes - ((si & 1) ? kBoxBytes : 0);
#pragma unroll
          for (int ks = 0; ks < 8; ++ks)                      // 8 x 16 = head_dim
            umma_bf16(tmem_S + (si & (NS - 1)) * kUmmaN, dK | desc_addr(kt + (ks >> 2) * kBoxBytes + (ks & 3) * 32),
                      dQ | desc_addr(qb + ks * 2 * kQLbo), kIdescS, ks > 0);
          umma_commit(bar(sm.sfull0 + (si & (NS - 1))));
          ++si; if (++s_st == S) { s_st = 0; s_ph ^= 1u; }
          did = true;
        }
        if (pi < si && mbar_try_wait(bar(sm.pfull0 + p_st), p_ph) &&
            (pi < NP || mbar_try_wait(bar(sm.pvfree0 + (pi & (NP - 1))), ((pi / NP) - 1) & 1))) {
          // P~V_t = V_t^T P^T: rows = d, columns = heads; p = hi + lo
          tc_fence_after();
          const uint32_t vt = sbase + sm.ring + p_st * kStageBytes + 2 * kBoxBytes;
          const uint32_t pb = sbase + sm.pb + p_st * 2 * kPBufBytes;
#pragma unroll
          for (int part = 0; part < 2; ++part)
#pragma unroll
            for (int ks = 0; ks < 4; ++ks)                    // 4 x 16 = tokens of the block
              umma_bf16(tmem_PV + (pi & (NP - 1)) * kUmmaN, dV | desc_addr(vt + ks * 2048),
                        dP | desc_addr(pb + part * kPBufBytes + ks * 2 * kPLbo), kIdescPV, (part | ks) > 0);
          umma_commit(bar(sm.empty0 + p_st));                 // K/V stage and its P buffer are free again
          umma_commit(bar(sm.pvfull0 + (pi & (NP - 1))));
          ++pi; if (++p_st == S) { p_st = 0; p_ph ^= 1u; }
          did = true;
        }
        if (!did && beyond_stop(step_of(pi))) break;          // every block <= t* has had both MMAs
      }
      umma_commit(bar(sm.done0));                             // every MMA retired before TMEM is released
      mbar_wait(bar(sm.done0), 0);
    }
  } else if (warp >= kWarpSoftmax0 && warp < kWarpSoftmax0 + 4) {
    // ===================================================== A4: online softmax, one thread per token
    const int grp = (warp - kWarpSoftmax0) >> 1;              // stream: even / odd blocks
    const int wq = (warp - kWarpSoftmax0) & 1;                // which 32 tokens of the block
    const int tok = wq * 32 + lane;
    const uint32_t tlane = static_cast<uint32_t>((warp - kWarpSoftmax0) * 32) << 16;   // TMEM lane quadrant == warp % 4
    float m_run[G];
#pragma unroll
    for (int h = 0; h < G; ++h) m_run[h] = kNegInf;
    int s = grp % S; uint32_t ph = (grp / S) & 1;             // ring stage and (i / S) & 1 of block i
    for (int i = grp, k = 0; i < n_c; i += 2, ++k) {
      const int t = step_of(i);
      if (!wait_or_stop(bar(sm.sfull0 + (i & (NS - 1))), (i / NS) & 1, t)) break;
      tc_fence_after();
      float sc[G];
      tmem_ld<G>(tmem_S + tlane + (i & (NS - 1)) * kUmmaN, sc);
      tmem_ld_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(sm.sfree0 + (i & (NS - 1))));
      const unsigned long long vmask = sinfo[s * 2];          // written before the loads the S MMA waited for
      if (i >= NP && !wait_or_stop(bar(sm.pvfree0 + (i & (NP - 1))), ((i / NP) - 1) & 1, t)) break;   // IterSlot reuse
      const bool valid = (vmask >> tok) & 1ull;
      float wmax[G];
#pragma unroll
      for (int h = 0; h < G; ++h) {
        sc[h] = valid ? sc[h] * p.scale_log2 : kNegInf;       // masked tokens: weight 0 (R8); their K may be NaN
        wmax[h] = warp_max_f32(sc[h]);
      }
      float* xw = xchg + (((grp * 2 + (k & 1)) * 2) + wq) * 8;
#pragma unroll
      for (int h = 0; h < G; ++h) if (lane == h) xw[h] = wmax[h];
      __syncwarp();
      const uint32_t xb = bar(sm.xchg0 + grp * 2 + (k & 1));
      if (lane == 0) mbar_arrive(xb);
      if (!wait_or_stop(xb, (k >> 1) & 1, t)) break;
      const float* xo = xchg + (((grp * 2 + (k & 1)) * 2) + (wq ^ 1)) * 8;
      __nv_bfloat16* pbh = reinterpret_cast<__nv_bfloat16*>(smem + sm.pb + s * 2 * kPBufBytes + (tok >> 3) * kPLbo + (tok & 7) * 2);
      __nv_bfloat16* pbl = reinterpret_cast<__nv_bfloat16*>(reinterpret_cast<uint8_t*>(pbh) + kPBufBytes);
      IterSlot& slot = slots[i & (NP - 1)];
      float ls[G];
#pragma unroll
      for (int h = 0; h < G; ++h) {
        const float m_new = fmaxf(m_run[h], fmaxf(wmax[h], xo[h]));
        const float pj = (valid && m_new != kNegInf) ? fast_exp2(sc[h] - m_new) : 0.f;
        const __nv_bfloat16 hi = __float2bfloat16_rn(pj);
        const __nv_bfloat16 lo = __float2bfloat16_rn(pj - __bfloat162float(hi));
        pbh[h * 8] = hi; pbl[h * 8] = lo;                     // row h, 16 bytes per row
        ls[h] = __bfloat162float(hi) + __bfloat162float(lo);  // the weight the tensor core really uses
        if (lane == 0 && wq == 0) { slot.mref[h] = m_new; slot.alpha[h] = (m_new == kNegInf) ? 1.f : fast_exp2(m_run[h] - m_new); }
        m_run[h] = m_new;
      }
      if (vmask != ~0ull && !valid) {                         // masked V rows may hold NaN: 0 * NaN would poison P~V
        uint4* vr = reinterpret_cast<uint4*>(smem + sm.ring + s * kStageBytes + 2 * kBoxBytes + tok * 128);
#pragma unroll
        for (int c = 0; c < 8; ++c) { vr[c] = make_uint4(0u, 0u, 0u, 0u); vr[c + kBoxBytes / 16] = make_uint4(0u, 0u, 0u, 0u); }
      }
#pragma unroll
      for (int o = 16; o >= 1; o >>= 1)
#pragma unroll
        for (int h = 0; h < G; ++h) ls[h] += __shfl_xor_sync(0xffffffffu, ls[h], o);
#pragma unroll
      for (int h = 0; h < G; ++h) if (lane == h) slot.lsum[wq][h] = ls[h];
      fence_proxy_async();                                    // P^T (and V fixes) visible to the tensor core
      mbar_arrive(bar(sm.pfull0 + s));
      s += 2; if (s >= S) { s -= S; ph ^= 1u; }
    }
    (void)ph;
  } else if (warp >= kWarpFold0) {
    // ===================================================== A5 / A6: publish step summaries, fold P~V_t
    const uint32_t tlane = static_cast<uint32_t>(fq * 32) << 16;
    int pub = 0, fld = 0;
    while (fld < n_c) {
      const int c = ART ? ld_ctrl_relaxed(a_ctrl) : 0;
      if (ART && c < 0 && step_of(fld) > -c) break;           // everything from here on lies beyond t*
      if constexpr (ART) {
        // ---- publish the summary of the next finished block (does not wait for any decision)
        if (pub < n_c && pub - fld < NP && mbar_try_wait(bar(sm.pvfull0 + (pub & (NP - 1))), (pub / NP) & 1)) {
          const int t = step_of(pub);
          const int slot_i = (t - 1) % M;
          bool dead = false;                                  // mailbox slot free: step t - M has been scanned
          while (true) {
            const int cc = ld_ctrl_relaxed(a_ctrl);
            if (cc < 0) { dead = true; break; }
            if (cc >= t - M) break;
          }
          if (!dead) {
            tc_fence_after();
            float pv[G];
            tmem_ld<G>(tmem_PV + tlane + (pub & (NP - 1)) * kUmmaN, pv);
            tmem_ld_wait();
            const IterSlot& sl = slots[pub & (NP - 1)];
            const uint32_t row0 = mapa(sbase + sm.mbox + static_cast<uint32_t>(slot_i) * kSummaryBytes, 0);
            const uint32_t mb = mapa(bar(sm.mbox0 + slot_i), 0);
            if (MODE == 2 || (d & 3) == 0) {
              const int pi = (MODE == 2) ? d : (d >> 2);      // probe coordinate k*(d/32)  (R1)
              st_async_vec<G>(row0 + (2 + pi) * G * 4u, pv, mb);
            }
            if (d == 1) {
              float ml[2 * G];
#pragma unroll
              for (int h = 0; h < G; ++h) { ml[h] = sl.mref[h]; ml[G + h] = sl.lsum[0][h] + sl.lsum[1][h]; }
              st_async_vec<G>(row0, ml, mb);
              st_async_vec<G>(row0 + G * 4u, ml + G, mb);
            }
          }
          ++pub;
          continue;
        }
        if (fld >= pub) continue;
        if (!(c < 0 || c >= step_of(fld) - 1)) continue;      // decision for the steps before it not known yet
      } else {
        if (!mbar_try_wait(bar(sm.pvfull0 + (fld & (NP - 1))), (fld / NP) & 1)) continue;
      }
      // ---- fold block `fld` into its stream: it is part of the result (step <= t*)
      tc_fence_after();
      float pv[G];
      tmem_ld<G>(tmem_PV + tlane + (fld & (NP - 1)) * kUmmaN, pv);
      tmem_ld_wait();
      const IterSlot& sl = slots[fld & (NP - 1)];
      const bool odd = fld & 1;
#pragma unroll
      for (int h = 0; h < G; ++h) {
        const float a = sl.alpha[h], lb = sl.lsum[0][h] + sl.lsum[1][h], mr = sl.mref[h];
        const float an = fmaf(a, odd ? acc1[h] : acc0[h], pv[h]);
        const float ln = fmaf(a, odd ? l1[h] : l0[h], lb);
        if (odd) { acc1[h] = an; l1[h] = ln; m1[h] = mr; } else { acc0[h] = an; l0[h] = ln; m0[h] = mr; }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(sm.pvfree0 + (fld & (NP - 1))));
      ++fld;
    }
  } else if (ART && warp == kWarpScan && rank == 0) {
    // ===================================================== A6 + A7 + A9: Algorithm 1 over step summaries
    constexpr int LPH = 32 / G;                               // lanes per head
    constexpr int CPL = PW / LPH;                             // probe components per lane
    const int h = lane / LPH, sub = lane % LPH;
    float m_run = kNegInf, l_run = 0.f, x[CPL];
#pragma unroll
    for (int j = 0; j < CPL; ++j) x[j] = 0.f;                 // x^(0) = 0 (Alg. 1 l.1)
    int cnt = 0, t_stop = 0;                                  // c^(0) = 0 (l.2)
    int slot_i = 0; uint32_t mph = 0;                         // (t - 1) % M and ((t - 1) / M) & 1
    for (int t = 1; t <= Tn; ++t) {
      mbar_wait(bar(sm.mbox0 + slot_i), mph);
      const float* mb = mbox + static_cast<size_t>(slot_i) * (2 + PW) * G;
      const float mt = mb[h], lt = mb[G + h];
      float pv[CPL];
#pragma unroll
      for (int j = 0; j < CPL; ++j) pv[j] = mb[(2 + sub + LPH * j) * G + h];
      __syncwarp();
      if (lane == 0 && t + M <= Tn) mbar_arrive_expect_tx(bar(sm.mbox0 + slot_i), kSummaryBytes);   // re-arm for step t + M
      // streaming update in recurrence form: x^(t) - x^(t-1) = (l_t / A_t) P(u^(t) - o^(t-1))
      // (PAPER.md:320, :361), with l_t u^(t) = P~V_t and everything relative to the running max.
      float sdd = 0.f, sad = 0.f, saa = 0.f, sbb = 0.f;
      if (mt != kNegInf) {                                    // a step with no valid token changes nothing (R8)
        const float mn = fmaxf(m_run, mt);
        const float al = fast_exp2(m_run - mn), be = fast_exp2(mt - mn);
        const float l_new = fmaf(al, l_run, be * lt);
        const float r = (l_new > 0.f) ? be / l_new : 0.f;
#pragma unroll
        for (int j = 0; j < CPL; ++j) {
          const float dlt = r * fmaf(-lt, x[j], pv[j]);
          const float xn = x[j] + dlt;
          sdd = fmaf(dlt, dlt, sdd); sad = fmaf(x[j], dlt, sad); saa = fmaf(x[j], x[j], saa); sbb = fmaf(xn, xn, sbb);
          x[j] = xn;
        }
        m_run = mn; l_run = l_new;
      } else {
#pragma unroll
        for (int j = 0; j < CPL; ++j) { saa = fmaf(x[j], x[j], saa); }
        sbb = saa;
      }
#pragma unroll
      for (int msk = LPH / 2; msk >= 1; msk >>= 1) {
        sdd += __shfl_xor_sync(0xffffffffu, sdd, msk); sad += __shfl_xor_sync(0xffffffffu, sad, msk);
        saa += __shfl_xor_sync(0xffffffffu, saa, msk); sbb += __shfl_xor_sync(0xffffffffu, sbb, msk);
      }
      // Eq. 2: d_scale = ||dx||; d_direction = 1 - cos(x_new, x_old), evaluated as
      // (|a|^2 |d|^2 - (a.d)^2) / (|a||b| (|a||b| + a.b)) to avoid the cancellation in 1 - cos.
      const float d_scale = sqrtf(sdd);
      float d_dir = 1.f;                                      // zero norm => cos := 0 (R4)
      if (saa > 0.f && sbb > 0.f) {
        const float nanb = sqrtf(saa) * sqrtf(sbb);
        const float ab = saa + sad;
        if (ab > 0.f) d_dir = fmaxf(fmaf(saa, sdd, -sad * sad), 0.f) / (nanb * (nanb + ab));
        else d_dir = 1.f - ab / nanb;
      }
      const bool stable_h = (d_scale < p.tau) && (d_dir < p.phi);            // strict (R5)
      const bool stable = __all_sync(0xffffffffu, stable_h);                 // AND over the group's heads (R2)
      cnt = stable ? cnt + 1 : 0;                                            // Eq. 3
      const bool fire = cnt >= p.patience;
      if (lane < C) st_cluster_relaxed_s32(mapa(a_ctrl, lane), fire ? -t : t);
      if (fire) { t_stop = t; break; }
      if (++slot_i == M) { slot_i = 0; mph ^= 1u; }
    }
    if (lane == 0) p.stop_block[group] = t_stop ? t_stop : Tn;               // t* (R9)
  }

  // ===================================================== A8 / A9: combine the partial states, write out
  tc_fence_before();
  __syncthreads();                                            // ring is free: all loads drained, all MMAs retired
  float* cta = reinterpret_cast<float*>(smem + sm.ring);
  float* cta_m = reinterpret_cast<float*>(smem + sm.misc + kCtaM);
  float* cta_l = reinterpret_cast<float*>(smem + sm.misc + kCtaL);
  if (warp >= kWarpFold0) {
#pragma unroll
    for (int h = 0; h < G; ++h) {                             // the CTA's two streams -> one partial state
      const float mx = fmaxf(m0[h], m1[h]);
      const float f0 = (m0[h] == kNegInf) ? 0.f : fast_exp2(m0[h] - mx), f1 = (m1[h] == kNegInf) ? 0.f : fast_exp2(m1[h] - mx);
      cta[h * kD + d] = fmaf(f0, acc0[h], f1 * acc1[h]);
      if (d == 0) { cta_m[h] = mx; cta_l[h] = fmaf(f0, l0[h], f1 * l1[h]); }
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
      p.out[(static_cast<int64_t>(b) * p.Hq + g * G) * kD + o] = (l > 0.f) ? a / l : 0.f;   // Alg. 1 l.18
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
  if (warp == kWarpTmem) { tc_fence_after(); tmem_dealloc(tmem_base, kTmemCols); }
}

}  // namespace tc
}  // namespace art
