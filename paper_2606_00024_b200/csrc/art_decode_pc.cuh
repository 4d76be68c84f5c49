// ART decode attention, bf16 KV / head_dim 128: PERSISTENT CLUSTERS with run-time scheduling (tcgen05 + TMEM + TMA).
//
// The grid is NC thread-block clusters of CL CTAs (CL up to 16, two CTAs per SM), launched once and resident for the
// whole call.  Cluster c owns the query groups c, c + NC, c + 2 NC, ...  Nothing inside a cluster is bound:
//
//   * a CTA that needs work OPENS the next group of its cluster (it becomes the group's HOME: its scan warp replays
//     Algorithm 1 for the group) or, when the cluster has no unopened group left, JOINS the open group of its cluster
//     with the most remaining steps per worker.  CTAs freed by a group that terminated early therefore stream for the
//     groups that still run, and the last long group of a cluster is served by all CL CTAs;
//   * traversal steps t = 1..T are CLAIMED one at a time from the group's counter on the cluster's
//     board (rank 0's shared memory, atom.shared::cluster); with the detector on, the TMA loads of step t are issued
//     only once step t - R has been decided, R = run-ahead per worker x workers: this bounds the blocks that are
//     loaded and then discarded when Algorithm 1 fires (A7) to the blocks in flight;
//   * one 64-token KV block is one pipeline ITEM, handled by specialised warps that meet through mbarriers exactly as
//     in art_decode_tc.cuh (TMA -> S = K Q^T -> block-local softmax -> P~V = V^T P^T with P split hi + lo), its
//     block-local result waiting UNFOLDED in tensor memory until the decision for its step is known;
//   * the step summary (m_t, l_t, probe of P~V_t) stays in the shared memory of the CTA that computed it; the home's
//     scan warp is told where (one word per step, st.shared::cluster) and PULLS it over distributed shared memory.
//     Every word of a summary carries, in its lowest mantissa bit, the parity of the slot's generation, so the reader
//     needs no fence: a word is either the previous generation's or final (a 4-byte store is single-copy atomic);
//   * the scan warp (art_scan_chunk.cuh) decides up to 8 steps per chunk and broadcasts the progress word to the
//     cluster; fold warps merge P~V_t into the CTA's partial state for t <= t* only, drop the others;
//   * a CTA that leaves a group flushes its partial (m, l, acc) to the workspace; whoever completes the count of
//     folded steps combines the partial states (flash-decoding merge) and writes `out` (A8/A9).
//
// Steps beyond t* are never folded and the scan consumes summaries in step order whoever computed them, so the
// result is the sequential algorithm's for any CL and any schedule.  Deadlock freedom: DESIGN.md section 6.
#pragma once
#include "art_decode_tc.cuh"
#include "art_scan_chunk.cuh"

namespace art {
namespace pc {

using namespace tc;

constexpr int kMaxCL = 16;
constexpr int kHS = 2 * kMaxCL;              // home slots of a cluster: two per CTA (a CTA opens its next group while the last one drains)
constexpr int kNR = 64;                      // notice ring per home slot; the run-ahead window never exceeds it
constexpr int kItemsRing = 32;               // item descriptors; >= stages + kPVSlots + the four END items
constexpr int kLock = -(1 << 20);            // board.nact while a slot is being (re)opened
constexpr int kMinJoin = 4;                  // a group with fewer unclaimed steps is not worth a Q reload and a partial state
static_assert(kItemsRing >= kPVSlots + kMaxStages + 4, "item ring too short");

struct PcParams {
  Params b;
  int32_t n_groups, NC;
  float* part;                               // workspace: partial states [group][rank][G * (kD + 2)]
  int32_t rw;                                // run-ahead per worker (steps issued beyond the last decided one)
  int32_t nsum;                              // summary slots per CTA (<= kPVSlots)
  int32_t claim;                             // steps claimed per atomic (a chunk of consecutive steps)
  uint32_t nap;                              // nanoseconds a polling warp sleeps between two looks
  unsigned long long* dbg;                   // ART_WATCHDOG: where a wait that never ended reports itself
  unsigned long long* stats;                 // ART_PC_STATS: cycle counters (device memory)
};

enum { ITEM_DATA = 0, ITEM_FLUSH = 1, ITEM_END = 2 };
// meta: bits 0-4 home slot, 5 Q buffer, 6-7 kind, 8-14 generation of the slot's group
struct Item { int tcode; int meta; unsigned long long mask; };   // FLUSH: tcode = blocks loaded in the visit, mask = group
__device__ __forceinline__ int item_hs(int meta) { return meta & 31; }
__device__ __forceinline__ int item_q(int meta) { return (meta >> 5) & 1; }
__device__ __forceinline__ int item_kind(int meta) { return (meta >> 6) & 3; }
__device__ __forceinline__ int item_gen(int meta) { return (meta >> 8) & 127; }

// progress word of a home slot, broadcast to every CTA of the cluster: [gen:7][fired:1][t:24]
__device__ __forceinline__ int ctrl_word(int gen, bool fired, int t) { return (gen << 25) | (fired ? (1 << 24) : 0) | t; }

struct BoardEntry { int next, T, nact, group, gen, pad0, pad1, pad2; };        // rank 0: one per home slot
struct HomeInfo { unsigned long long done; int group, T, gen, loaded; unsigned joined; int pad; };   // home CTA: one per local slot

struct SmemMapP {
  uint32_t qb, pb, slots, items, sums, tags, stab, hinfo, ctrl, board, bars, misc, ring, total;
  uint32_t full0, empty0, pfull0, sfull0, sfree0, pvfull0, pvfree0, done0, nbars;
};
// summary of one step: [G * PW] probe values (lane l of the scan warp owns floats l*CPL .. l*CPL + CPL - 1), then (m, l) x G
__host__ __device__ constexpr uint32_t sum_bytes(int G, int PW) { return static_cast<uint32_t>(G * (PW + 2) * 4); }

__host__ __device__ inline SmemMapP make_smem_map_p(int G, int PW, int stages, int nsum, bool art) {
  SmemMapP m;
  uint32_t off = 0;
  m.qb = off; off += 2u * kQBytes;
  m.pb = off; off += static_cast<uint32_t>(p_bufs(G, stages, art && PW == 32)) * 2u * p_buf_bytes(G);
  m.slots = off; off += kIterSlots * static_cast<uint32_t>(2 * G) * 4u;           // per item: m_blk[G], block sum[G]
  m.items = off; off += kItemsRing * static_cast<uint32_t>(sizeof(Item));
  off = (off + 15u) & ~15u;
  m.sums = off; off += art ? static_cast<uint32_t>(nsum) * sum_bytes(G, PW) : 0u;
  m.tags = off; off += art ? 2u * kNR * 4u : 0u;
  m.stab = off; off += art ? 2u * 4u * kNR : 0u;                 // per-step results of the four scanning warps
  off = (off + 15u) & ~15u;
  m.hinfo = off; off += 2u * static_cast<uint32_t>(sizeof(HomeInfo));
  m.ctrl = off; off += kHS * 4u;
  m.board = off; off += kHS * static_cast<uint32_t>(sizeof(BoardEntry)) + 16u;    // + next_local
  m.bars = off;
  uint32_t n = 0;
  m.full0 = n; n += stages; m.empty0 = n; n += stages; m.pfull0 = n; n += stages;
  m.sfull0 = n; n += kSSlots; m.sfree0 = n; n += kSSlots;
  m.pvfull0 = n; n += kPVSlots; m.pvfree0 = n; n += kPVSlots;
  m.done0 = n; n += 2;
  m.nbars = n;
  off += n * 8u;
  m.misc = off; off += 32u + 4u * kPVSlots;
  off = (off + 1023u) & ~1023u;
  if (off < static_cast<uint32_t>(kFront)) off = kFront;
  m.ring = off; off += static_cast<uint32_t>(stages) * kStageBytes;
  m.total = off;
  return m;
}
constexpr uint32_t kMTmem = 0, kMOpen = 4, kMScanExit = 8, kMFlag = 12, kMJoined = 16, kMPubCnt = 32;   // + kPVSlots publish counters

// ----------------------------------------------------------------------------- small PTX helpers

__device__ __forceinline__ int atom_add_cluster(uint32_t a, int v) {           // relaxed
  int r; asm volatile("atom.relaxed.cluster.shared::cluster.add.s32 %0, [%1], %2;" : "=r"(r) : "r"(a), "r"(v) : "memory"); return r;
}
// release = MEMBAR.ALL.GPU + atom (about a microsecond under load); acquire = atom + CCTL.IVALL (cheap): every
// atomic below carries exactly the ordering its use needs
__device__ __forceinline__ int atom_add_cluster_acquire(uint32_t a, int v) {
  int r; asm volatile("atom.acquire.cluster.shared::cluster.add.s32 %0, [%1], %2;" : "=r"(r) : "r"(a), "r"(v) : "memory"); return r;
}
__device__ __forceinline__ int atom_add_cluster_release(uint32_t a, int v) {
  int r; asm volatile("atom.release.cluster.shared::cluster.add.s32 %0, [%1], %2;" : "=r"(r) : "r"(a), "r"(v) : "memory"); return r;
}
__device__ __forceinline__ int atom_cas_cluster_acquire(uint32_t a, int cmp, int v) {
  int r; asm volatile("atom.acquire.cluster.shared::cluster.cas.b32 %0, [%1], %2, %3;" : "=r"(r) : "r"(a), "r"(cmp), "r"(v) : "memory"); return r;
}
__device__ __forceinline__ unsigned atom_or_cluster(uint32_t a, unsigned v) {
  unsigned r; asm volatile("atom.relaxed.cluster.shared::cluster.or.b32 %0, [%1], %2;" : "=r"(r) : "r"(a), "r"(v) : "memory"); return r;
}
__device__ __forceinline__ unsigned long long atom_add64_cluster_acqrel(uint32_t a, unsigned long long v) {
  unsigned long long r;
  asm volatile("atom.acq_rel.cluster.shared::cluster.add.u64 %0, [%1], %2;" : "=l"(r) : "r"(a), "l"(v) : "memory"); return r;
}
__device__ __forceinline__ int ld_cluster_relaxed_s32(uint32_t a) {
  int v; asm volatile("ld.relaxed.cluster.shared::cluster.s32 %0, [%1];" : "=r"(v) : "r"(a) : "memory"); return v;
}
__device__ __forceinline__ int ld_cluster_acquire_s32(uint32_t a) {
  int v; asm volatile("ld.acquire.cluster.shared::cluster.s32 %0, [%1];" : "=r"(v) : "r"(a) : "memory"); return v;
}
__device__ __forceinline__ uint32_t ld_cluster_u32(uint32_t a) {
  uint32_t v; asm volatile("ld.relaxed.cluster.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory"); return v;
}
template <int N> __device__ __forceinline__ void ld_cluster_vec(uint32_t a, uint32_t (&r)[N]) {
  if constexpr (N == 1) {
    asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(r[0]) : "r"(a) : "memory");
  } else if constexpr (N == 2) {
    asm volatile("ld.shared::cluster.v2.u32 {%0,%1}, [%2];" : "=r"(r[0]), "=r"(r[1]) : "r"(a) : "memory");
  } else {
    static_assert(N % 4 == 0, "vector width");
#pragma unroll
    for (int i = 0; i < N; i += 4)
      asm volatile("ld.shared::cluster.v4.u32 {%0,%1,%2,%3}, [%4];"
                   : "=r"(r[i]), "=r"(r[i + 1]), "=r"(r[i + 2]), "=r"(r[i + 3]) : "r"(a + 4u * i) : "memory");
  }
}
__device__ __forceinline__ void fence_cluster() { asm volatile("fence.acq_rel.cluster;" ::: "memory"); }
__device__ __forceinline__ void named_bar_sync(int id, int threads) { asm volatile("bar.sync %0, %1;" :: "r"(id), "r"(threads) : "memory"); }
__device__ __forceinline__ void nsleep(unsigned ns) { asm volatile("nanosleep.u32 %0;" :: "r"(ns)); }
__device__ __forceinline__ unsigned long long gtime() { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }

// A wait that does not end within two seconds is a scheduling bug: report where and trap, so that the call fails
// instead of hanging the device.  Compiled in with -DART_WATCHDOG (the test build); free otherwise.
#ifdef ART_WATCHDOG
struct Watch {
  unsigned long long t0; unsigned long long* dbg; int code;
  __device__ __forceinline__ Watch(unsigned long long* d, int c) : t0(gtime()), dbg(d), code(c) {}
  __device__ __forceinline__ void poll(int a = 0, int b = 0) {
    if (gtime() - t0 > (code == 7 || code == 8 ? 1000000000ull : 2000000000ull)) {
      if (dbg && atomicCAS(dbg + 2, 0ull, 1ull) == 0ull) { dbg[1] = (static_cast<unsigned long long>(static_cast<unsigned>(a)) << 32) | static_cast<unsigned>(b); dbg[0] = (static_cast<unsigned long long>(code) << 48) | (static_cast<unsigned long long>(blockIdx.x) << 32) | (static_cast<unsigned>(a) & 0xffffu) << 16 | (static_cast<unsigned>(b) & 0xffffu); __threadfence_system(); }
      __trap();
    }
  }
};
#define ART_WATCH(name, code) Watch name(pp.dbg, code)
#define ART_WATCH_POLL(name, ...) name.poll(__VA_ARGS__)
#else
#define ART_WATCH(name, code)
#define ART_WATCH_POLL(name, ...)
#endif

#ifdef ART_PC_STATS
#define ART_STAT_ADD(i, v) do { if (pp.stats && lane == 0) atomicAdd(pp.stats + (i), static_cast<unsigned long long>(v)); } while (0)
#define ART_STAT_T(name) const long long name = clock64()
#define ART_STAT_SET(name) name = clock64()
#else
#define ART_STAT_SET(name)
#define ART_STAT_ADD(i, v)
#define ART_STAT_T(name)
#endif

// self-validating words: the lowest mantissa bit carries the generation parity of the slot; -inf travels as -1e30
__device__ __forceinline__ uint32_t tag_word(float v, uint32_t par) { return (__float_as_uint(v) & ~1u) | par; }
constexpr float kNegBig = -1e30f;

// ----------------------------------------------------------------------------- the kernel

template <int G, int MODE, bool MT = false>
__global__ void __launch_bounds__(kThreads, (MODE == 2) ? 1 : 2)
art_decode_pc_kernel(const PcParams pp, const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV) {
  constexpr bool ART = MODE != 0;
  constexpr int PW = (MODE == 2) ? kD : 32;
  constexpr int NP = kPVSlots, NS = kSSlots;
  constexpr int LBO_P = p_lbo(G), PBUF = p_buf_bytes(G);
  constexpr bool kTwoPBufs = (G == 8 && MODE == 1);
  constexpr uint32_t SUMB = sum_bytes(G, PW);
  constexpr int PF = G * (kD + 2);                       // floats of one partial state
  constexpr int GW = G >= 8 ? 2 : 1;                     // heads per scanning warp (the fold warps of the home CTA scan)
  using Scan = ChunkScan<GW, PW>;
  const Params& p = pp.b;

  extern __shared__ __align__(1024) uint8_t smem[];
  const int S = p.stages, NSUM = pp.nsum;
  const SmemMapP sm = make_smem_map_p(G, PW, S, NSUM, ART);
  const uint32_t sbase = smem_u32(smem);
  if ((sbase & 1023u) != 0u) __trap();
  const uint32_t bars = sbase + sm.bars;
  auto bar = [&](uint32_t idx) { return bars + idx * 8u; };
  float* slots = reinterpret_cast<float*>(smem + sm.slots);   // [item & 15][2 G]: block maximum (log2 domain), block sum
  volatile Item* items = reinterpret_cast<volatile Item*>(smem + sm.items);
  const uint32_t a_misc = sbase + sm.misc;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int CL = static_cast<int>(cluster_nctarank());
  const int rank = static_cast<int>(cluster_ctarank());
  const int cidx = blockIdx.x / CL;
  const int n_local = (pp.n_groups > cidx) ? (pp.n_groups - cidx + pp.NC - 1) / pp.NC : 0;   // groups cidx, cidx + NC, ...
  const int n_init = n_local < CL ? n_local : CL;        // opened before the cluster starts: CTA r opens local group r

  // addresses on the cluster's board (rank 0) and in a home CTA
  auto board_at = [&](int hs, int field) { return mapa(sbase + sm.board + static_cast<uint32_t>(hs) * 32u + field * 4u, 0); };
  const uint32_t a_next_local = mapa(sbase + sm.board + kHS * 32u, 0);
  auto hinfo_at = [&](int hs, uint32_t byte_off) { return mapa(sbase + sm.hinfo + static_cast<uint32_t>(hs & 1) * 32u + byte_off, hs >> 1); };
  enum { B_NEXT = 0, B_T = 1, B_NACT = 2, B_GROUP = 3, B_GEN = 4 };
  constexpr uint32_t H_DONE = 0, H_GROUP = 8, H_T = 12, H_GEN = 16, H_LOADED = 20, H_JOINED = 24;

  // ---- one-time setup
  if (tid == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(bar(sm.full0 + s), 1); mbar_init(bar(sm.empty0 + s), 1); mbar_init(bar(sm.pfull0 + s), 32); }
    for (int s = 0; s < NS; ++s) { mbar_init(bar(sm.sfull0 + s), 1); mbar_init(bar(sm.sfree0 + s), 1); }
    for (int s = 0; s < NP; ++s) { mbar_init(bar(sm.pvfull0 + s), 1); mbar_init(bar(sm.pvfree0 + s), 4); }
    mbar_init(bar(sm.done0), 1); mbar_init(bar(sm.done0 + 1), 1);
    st_volatile_s32(a_misc + kMOpen, 0); st_volatile_s32(a_misc + kMScanExit, 0); st_volatile_s32(a_misc + kMFlag, 0);
    for (int s = 0; s < kPVSlots; ++s) st_volatile_s32(a_misc + kMPubCnt + 4u * s, 0);
    fence_mbar_init();
  }
  for (int i = tid; i < kHS; i += kThreads) {
    reinterpret_cast<int*>(smem + sm.ctrl)[i] = 0;
    int* e = reinterpret_cast<int*>(smem + sm.board + i * 32);
    e[B_NEXT] = 0; e[B_T] = 0; e[B_NACT] = 0; e[B_GROUP] = -1; e[B_GEN] = 0;
  }
  if (tid == 0) *reinterpret_cast<int*>(smem + sm.board + kHS * 32) = n_init;
  if (tid < 16) reinterpret_cast<int*>(smem + sm.hinfo)[tid] = 0;
  if (warp == kWarpMmaPV) tmem_alloc(a_misc + kMTmem, kTmemCols);
  {
    if (tid < 64) {                                          // the zero rows behind each Q^T buffer
      reinterpret_cast<__nv_bfloat16*>(smem + sm.qb + 16 * kQLbo)[tid] = __float2bfloat16_rn(0.f);
      reinterpret_cast<__nv_bfloat16*>(smem + sm.qb + kQBytes + 16 * kQLbo)[tid] = __float2bfloat16_rn(0.f);
    }
    uint4* qz = reinterpret_cast<uint4*>(smem + sm.qb);      // rows >= Gr stay zero for the whole launch
    for (int idx = tid; idx < 2 * kQBytes / 16; idx += kThreads) qz[idx] = make_uint4(0u, 0u, 0u, 0u);
    uint4* pz = reinterpret_cast<uint4*>(smem + sm.pb);      // P^T rows are read before they are first written
    for (int idx = tid; idx < p_bufs(G, S, MODE == 1) * 2 * PBUF / 16; idx += kThreads) pz[idx] = make_uint4(0u, 0u, 0u, 0u);
  }
  fence_proxy_async();
  tc_fence_before();
  cluster_sync_all();                                        // boards and barriers of every CTA are live
  tc_fence_after();
  const uint32_t tmem_base = static_cast<uint32_t>(ld_volatile_s32(a_misc + kMTmem));
  const uint32_t tmem_S = tmem_base, tmem_PV = tmem_base + NS * kSCols;

  // fold warps: output coordinate and running (un-normalised) partial state of the current visit
  const int fq = warp & 3;
  const int d = fq * 32 + lane;

  // decoded progress word of (home slot, generation): last decided step, fired?
  auto read_ctrl = [&](int hs, int gen, bool& fired) -> int {
    const int c = ld_ctrl_relaxed(sbase + sm.ctrl + static_cast<uint32_t>(hs) * 4u);
    if ((static_cast<unsigned>(c) >> 25) != static_cast<unsigned>(gen)) { fired = false; return 0; }
    fired = (c >> 24) & 1;
    return c & 0xffffff;
  };

  // ===================================================== scheduling state of the producer warp (open / join / claim)
  int it = 0, stage = 0; uint32_t ph = 0;
  int my_gen = 0;                                          // groups this CTA has opened
  int nvisit = 0;                                          // visits that issued at least one item
  int q_last[2] = {-1, -1};                                // last item that reads Q buffer 0 / 1
  bool more_local = n_local > n_init;
  // the visit
  bool have = false;
  int v_hs = 0, v_gen = 0, v_group = 0, v_T = 0, v_b = 0, v_g = 0, v_L = 0, v_loaded = 0, v_items = 0, v_qsel = 0;
  Trav v_tr = {};

  auto wait_empty = [&]() {                               // the stage this item will use is free again
    if (it >= S) mbar_wait(bar(sm.empty0 + stage), ph ^ 1u);
  };
  auto advance = [&]() { ++it; if (++stage == S) { stage = 0; ph ^= 1u; } };
  auto push_marker = [&](int kind, int tcode, int meta_extra, unsigned long long payload) {
    wait_empty();
    if (lane == 0) {
      items[it % kItemsRing].tcode = tcode; items[it % kItemsRing].meta = (kind << 6) | meta_extra; items[it % kItemsRing].mask = payload;
      if (kind == ITEM_END)                               // one END per softmax warp: only the first takes a stage
        for (int j = 1; j < NS; ++j) { items[(it + j) % kItemsRing].tcode = 0; items[(it + j) % kItemsRing].meta = (ITEM_END << 6); items[(it + j) % kItemsRing].mask = 0ull; }
      mbar_arrive(bar(sm.full0 + stage));
    }
    __syncwarp();
    advance();
  };
  // group -> geometry
  auto set_group = [&](int group) {
    v_group = group; v_b = group / p.Hkv; v_g = group % p.Hkv; v_L = p.seq_lens[v_b];
    v_tr = make_trav(p, v_b, v_g, v_L); v_T = v_tr.T;
  };
  // become the home of local group i (lane-uniform); false if the group is empty (handled here)
  auto open_group = [&](int i, bool before_start) -> bool {
    set_group(cidx + i * pp.NC);
    if (v_T == 0) {                                        // no eligible block: out = 0, t* = 0
      for (int o = lane; o < p.Gr * kD; o += 32) {
        const int h = o / kD;
        p.out[((static_cast<int64_t>(v_b) * p.qlen + h / p.Gh) * p.Hq + v_g * p.Gh + h % p.Gh) * kD + (o - h * kD)] = 0.f;
      }
      if (lane == 0) p.stop_block[v_group] = 0;
      return false;
    }
    const int hsl = my_gen & 1;
    v_hs = rank * 2 + hsl; v_gen = my_gen & 127;
    if (lane == 0) {
      ART_WATCH(wd, 1);
      while (atom_cas_cluster_acquire(board_at(v_hs, B_NACT), 0, kLock) != 0) { nsleep(64); ART_WATCH_POLL(wd, v_hs, my_gen); }
    }
    __syncwarp();
    if constexpr (ART) {                                   // nobody is left who could still write a notice of the slot's last group
      uint32_t* tg = reinterpret_cast<uint32_t*>(smem + sm.tags) + hsl * kNR;
      for (int i2 = lane; i2 < kNR; i2 += 32) tg[i2] = 0u;
      uint32_t* sb = reinterpret_cast<uint32_t*>(smem + sm.stab) + hsl * kNR;      // four scanning warps x kNR bytes
      for (int i2 = lane; i2 < kNR; i2 += 32) sb[i2] = 0u;
    }
    if (lane == 0) {
      HomeInfo* hi = reinterpret_cast<HomeInfo*>(smem + sm.hinfo) + hsl;
      hi->done = ART ? 0ull : (static_cast<unsigned long long>(v_T + 1) << 32);
      hi->group = v_group; hi->T = v_T; hi->gen = v_gen; hi->loaded = 0; hi->joined = 0u;
      asm volatile("st.relaxed.cluster.shared::cluster.s32 [%0], %1;" :: "r"(board_at(v_hs, B_NEXT)), "r"(0) : "memory");
      asm volatile("st.relaxed.cluster.shared::cluster.s32 [%0], %1;" :: "r"(board_at(v_hs, B_T)), "r"(v_T) : "memory");
      asm volatile("st.relaxed.cluster.shared::cluster.s32 [%0], %1;" :: "r"(board_at(v_hs, B_GROUP)), "r"(v_group) : "memory");
      asm volatile("st.relaxed.cluster.shared::cluster.s32 [%0], %1;" :: "r"(board_at(v_hs, B_GEN)), "r"(v_gen) : "memory");
    }
    __syncwarp();
    if (lane == 0) {
      // open, one worker (this CTA); releases all of the above (before the start the cluster barrier does that)
      if (before_start) atom_add_cluster(board_at(v_hs, B_NACT), 1 - kLock);
      else atom_add_cluster_release(board_at(v_hs, B_NACT), 1 - kLock);
      if constexpr (ART) asm volatile("st.release.cta.shared::cta.s32 [%0], %1;" :: "r"(a_misc + kMOpen), "r"(my_gen + 1) : "memory");
    }
    __syncwarp();
    ++my_gen;
    return true;
  };
  // the home slot this CTA would open next is free (every worker of the group that used it last has left)
  auto slot_free = [&]() -> bool {
    if (my_gen < 2) return true;
    int v = 0;
    if (lane == 0) v = ld_cluster_relaxed_s32(board_at(rank * 2 + (my_gen & 1), B_NACT));
    return __shfl_sync(0xffffffffu, v, 0) == 0;
  };
  // join the open group of the cluster with the most unclaimed steps per worker; false if there is none
  auto join_group = [&]() -> bool {
    int score = 0, e_next = 0, e_T = 0, e_nact = 0, e_group = -1, e_gen = 0;
    if (lane < 2 * CL) {
      e_next = ld_cluster_relaxed_s32(board_at(lane, B_NEXT)); e_T = ld_cluster_relaxed_s32(board_at(lane, B_T));
      e_nact = ld_cluster_relaxed_s32(board_at(lane, B_NACT)); e_group = ld_cluster_relaxed_s32(board_at(lane, B_GROUP));
      e_gen = ld_cluster_relaxed_s32(board_at(lane, B_GEN));
      bool fired = false;
      if constexpr (ART) read_ctrl(lane, e_gen, fired);
      const int rem = (e_nact > 0 && e_group >= 0 && !fired) ? e_T - e_next : 0;
      if (rem >= kMinJoin) score = (rem << 4) / (e_nact + 1) + 1;
    }
    int best = score, who = lane;
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) {
      const int ob = __shfl_xor_sync(0xffffffffu, best, m), ow = __shfl_xor_sync(0xffffffffu, who, m);
      if (ob > best || (ob == best && ow < who)) { best = ob; who = ow; }
    }
    if (best == 0) return false;
    int ok = 0, T2 = 0, grp = 0, gen2 = 0;
    if (lane == 0) {
      const int old = atom_add_cluster_acquire(board_at(who, B_NACT), 1);       // pin: the slot cannot be reopened under us
      T2 = ld_cluster_relaxed_s32(board_at(who, B_T)); grp = ld_cluster_relaxed_s32(board_at(who, B_GROUP));
      gen2 = ld_cluster_relaxed_s32(board_at(who, B_GEN));
      const int nx = ld_cluster_relaxed_s32(board_at(who, B_NEXT));
      ok = (old > 0 && grp >= 0 && nx < T2) ? 1 : 0;
      if (!ok) atom_add_cluster(board_at(who, B_NACT), -1);
    }
    ok = __shfl_sync(0xffffffffu, ok, 0);
    if (!ok) return true;                                  // lost a race: look again
    v_hs = who; v_gen = __shfl_sync(0xffffffffu, gen2, 0);
    set_group(__shfl_sync(0xffffffffu, grp, 0));
    have = true;
    return true;
  };
  // leave the current group without having issued an item for it
  auto leave_quietly = [&]() { if (lane == 0) atom_add_cluster(board_at(v_hs, B_NACT), -1); __syncwarp(); };

  if (warp == kWarpProducer && rank < n_init) have = open_group(rank, true);
  // every CTA's first group is on the board before anybody looks for a group to join
  cluster_sync_all();
  if (warp == kWarpProducer && rank >= n_init && n_init > 0) {
    // the CTAs that opened nothing start as workers of the cluster's first groups, dealt round-robin: no search
    const int home = rank % n_init;
    set_group(cidx + home * pp.NC);
    if (v_T >= kMinJoin) {                                  // (an empty or tiny first group: look for work the usual way)
      v_hs = home * 2; v_gen = 0;
      if (lane == 0) atom_add_cluster(board_at(v_hs, B_NACT), 1);
      __syncwarp();
      have = true;
    }
  }

  if (warp == kWarpProducer) {
    // ===================================================== A1 + A2: claim steps, resolve blocks, issue TMA loads
    for (;;) {
      if (!have) {
        if (more_local && slot_free()) {
          int i = 0;
          if (lane == 0) i = atom_add_cluster(a_next_local, 1);
          i = __shfl_sync(0xffffffffu, i, 0);
          if (i < n_local) { have = open_group(i, false); if (!have) continue; }
          else more_local = false;
        }
        if (!have) {
          if (!join_group()) {
            if (!more_local) break;                          // nothing to open, nothing to join: done
            nsleep(200);                                     // our next slot is still draining
            continue;
          }
          if (!have) continue;
        }
        v_loaded = 0; v_items = 0;
      }
      // ---- the visit: claim steps until the group has none left (or Algorithm 1 has fired)
      const uint32_t a_next = board_at(v_hs, B_NEXT), a_nact = board_at(v_hs, B_NACT);
      // steps are claimed a chunk of `claim` consecutive steps at a time, one chunk ahead of the one being issued,
      // so the round trip to the board is never waited for
      const int K = pp.claim;
      int ch_t = 0, ch_left = 0, nx = 0, nactB = 1;
      auto claim_chunk = [&]() {
        if (lane == 0) { nx = atom_add_cluster(a_next, K) + 1; if constexpr (ART) nactB = ld_cluster_relaxed_s32(a_nact); }
      };
      auto next_step = [&]() -> int {
        if (ch_left == 0) { ch_t = __shfl_sync(0xffffffffu, nx, 0); ch_left = K; if (ch_t <= v_T) claim_chunk(); }
        --ch_left;
        return ch_t++;
      };
      auto resolve = [&](int t, bool& valid, unsigned long long& mask, int& page, int& ec) {
        bool fired = false;
        if constexpr (ART) read_ctrl(v_hs, v_gen, fired);
        valid = t <= v_T && !fired;
        mask = 0ull; page = 0; ec = 0;
        if (valid) {
          const int blk = trav_block(v_tr, t);
          mask = block_mask(p, v_L, blk);
          if constexpr (MT) ec = causal_code(p, v_L, blk);
          if (mask) page = p.block_table[static_cast<int64_t>(v_b) * p.max_blocks + blk];
        }
      };
      claim_chunk();
      int tA = next_step();
      bool validA; unsigned long long maskA; int pageA, ecA;
      resolve(tA, validA, maskA, pageA, ecA);
      while (validA) {
        const int tN = next_step();
        bool validB; unsigned long long maskB; int pageB, ecB;
        resolve(tN, validB, maskB, pageB, ecB);
        if constexpr (ART) {
          // A7 / run-ahead: the loads of step t go out once step t - R is decided (R grows with the workers of the group)
          int R = pp.rw * max(__shfl_sync(0xffffffffu, nactB, 0), 1);
          R = R > kNR ? kNR : R;
          bool fired = false;
          ART_WATCH(wd, 2);
          ART_STAT_T(tg0);
          while (read_ctrl(v_hs, v_gen, fired) < tA - R && !fired) { nsleep(pp.nap); ART_WATCH_POLL(wd, v_hs, tA); }
          ART_STAT_T(tg1);
          ART_STAT_ADD(8, tg1 - tg0); ART_STAT_ADD(10, 1);
          if (fired) break;                                  // t > t*: nothing of this group is loaded any more
        }
        if (v_items == 0) {
          // first item of the visit: this group's Q^T goes into the Q buffer that the visit before last used
          v_qsel = nvisit & 1;
          if (q_last[v_qsel] >= 0 && q_last[v_qsel] > it - S) mbar_wait(bar(sm.empty0 + q_last[v_qsel] % S), (q_last[v_qsel] / S) & 1);
          const __nv_bfloat16* qp = reinterpret_cast<const __nv_bfloat16*>(p.q) + (static_cast<int64_t>(v_b) * p.qlen * p.Hq + v_g * p.Gh) * kD;
          for (int c = lane; c < p.Gr * (kD / 8); c += 32) {  // 16-byte chunks: row r, columns 8 c8 .. 8 c8 + 7
            const int row = c / (kD / 8), c8 = c % (kD / 8);
            const uint4 val = *reinterpret_cast<const uint4*>(qp + ((row / p.Gh) * p.Hq + row % p.Gh) * kD + c8 * 8);
            *reinterpret_cast<uint4*>(smem + sm.qb + v_qsel * kQBytes + c8 * kQLbo + row * 16) = val;
          }
          fence_proxy_async();                               // written by threads, read by the tensor core
          __syncwarp();
          ++nvisit;
        }
        ART_STAT_T(te0);
        wait_empty();
        ART_STAT_T(te1);
        ART_STAT_ADD(9, te1 - te0);
        if (lane == 0) {
          const uint32_t fb = bar(sm.full0 + stage);
          const uint32_t dst = sbase + sm.ring + stage * kStageBytes;
          items[it % kItemsRing].tcode = tA | (ecA << kItemShift);
          items[it % kItemsRing].meta = v_hs | (v_qsel << 5) | (ITEM_DATA << 6) | (v_gen << 8);
          items[it % kItemsRing].mask = maskA;
          if (maskA == 0ull) {
            mbar_arrive(fb);                                 // nothing to load: an all-masked step
          } else {
            int c1, c2;
            if (p.layout == ART_LAYOUT_HND) { c1 = 0; c2 = pageA * p.Hkv + v_g; }
            else { c1 = v_g; c2 = pageA * kBlockTokens; }
            mbar_arrive_expect_tx(fb, kStageBytes);
            tma_load_box(dst, &tmK, 0, c1, c2, fb);
            tma_load_box(dst + kBoxBytes, &tmK, 64, c1, c2, fb);
            tma_load_box(dst + 2 * kBoxBytes, &tmV, 0, c1, c2, fb);
            tma_load_box(dst + 3 * kBoxBytes, &tmV, 64, c1, c2, fb);
          }
        }
        __syncwarp();
        if (maskA != 0ull) ++v_loaded;
        q_last[v_qsel] = it;
        ++v_items;
        advance();
        tA = tN; validA = validB; maskA = maskB; pageA = pageB; ecA = ecB;
      }
      // ---- the group has no step left for us: flush our partial state (the fold warps leave the group for us)
      if (v_items > 0) push_marker(ITEM_FLUSH, v_loaded, v_hs | (v_gen << 8), static_cast<unsigned long long>(v_group));
      else leave_quietly();
      have = false;
    }
    push_marker(ITEM_END, 0, 0, 0ull);
    if (lane == 0) st_volatile_s32(a_misc + kMScanExit, 1);
  } else if (warp == kWarpMmaS) {
    // ===================================================== A3: S = K_t Q^T, rows = tokens, columns = heads
    if (lane == 0) {
      const uint64_t dK = kDescSw128 | desc_strides(16, 1024);
      const uint64_t dQ = kDescNoSw | desc_strides(kQLbo, kQSbo);
      int st = 0; uint32_t ph = 0;
      for (int i = 0;; ++i) {
        const int q = i & (NS - 1);
        mbar_wait(bar(sm.full0 + st), ph);
        const int meta = items[i % kItemsRing].meta;
        const int kind = item_kind(meta);
        if (kind == ITEM_END) {                              // wake every softmax warp once more; each finds its END item
          for (int j = 0; j < NS; ++j) {
            const int ii = i + j, qq = ii & (NS - 1);
            if (ii >= NS) mbar_wait(bar(sm.sfree0 + qq), ((ii / NS) - 1) & 1);
            umma_commit(bar(sm.sfull0 + qq));
          }
          break;
        }
        if (i >= NS) mbar_wait(bar(sm.sfree0 + q), ((i / NS) - 1) & 1);
        if (kind == ITEM_DATA) {
          tc_fence_after();
          const uint32_t qb = sbase + sm.qb + item_q(meta) * kQBytes;
          const uint32_t kt = sbase + sm.ring + st * kStageBytes - q * 4096;
          const uint32_t dcol = tmem_S + q * kSCols;
#pragma unroll
          for (int ks = 0; ks < 8; ++ks) {
            const uint32_t ka = kt + (ks >> 2) * kBoxBytes + (ks & 3) * 32;
            const uint64_t bq = dQ | desc_addr(qb + ks * 2 * kQLbo);
            umma_bf16(dcol, dK | desc_addr(ka), bq, kIdescS, ks > 0);
            umma_bf16(dcol + kUmmaN, dK | desc_addr(ka + 4096), bq, kIdescS, ks > 0);
          }
        }
        umma_commit(bar(sm.sfull0 + q));
        if (++st == S) { st = 0; ph ^= 1u; }
      }
      umma_commit(bar(sm.done0));
      mbar_wait(bar(sm.done0), 0);
    }
  } else if (warp == kWarpMmaPV) {
    // ===================================================== A5: P~V_t = V_t^T P^T, rows = d, columns = heads
    if (lane == 0) {
      const uint64_t dV = kDescSw128 | desc_strides(kBoxBytes, 1024);
      const uint64_t dP = kDescNoSw | desc_strides(LBO_P, 128);
      int st = 0; uint32_t ph = 0;
      for (int i = 0;; ++i) {
        const int ps = i & (NP - 1);
        mbar_wait(bar(sm.pfull0 + st), ph);
        const int kind = item_kind(items[i % kItemsRing].meta);
        if (i >= NP) mbar_wait(bar(sm.pvfree0 + ps), ((i / NP) - 1) & 1);
        if (kind == ITEM_DATA) {
          tc_fence_after();
          const uint32_t vt = sbase + sm.ring + st * kStageBytes + 2 * kBoxBytes;
          const uint32_t pb = sbase + sm.pb + (kTwoPBufs ? (i & 1) : st) * 2 * PBUF;
#pragma unroll
          for (int part = 0; part < 2; ++part)
#pragma unroll
            for (int ks = 0; ks < 4; ++ks)
              umma_bf16(tmem_PV + ps * kUmmaN, dV | desc_addr(vt + ks * 2048),
                        dP | desc_addr(pb + part * PBUF + ks * 2 * LBO_P), kIdescPV, (part | ks) > 0);
        }
        umma_commit(bar(sm.empty0 + st));
        umma_commit(bar(sm.pvfull0 + ps));
        if (kind == ITEM_END) break;
        if (++st == S) { st = 0; ph ^= 1u; }
      }
      umma_commit(bar(sm.done0 + 1));
      mbar_wait(bar(sm.done0 + 1), 0);
    }
  } else if (warp >= kWarpSoftmax0 && warp < kWarpSoftmax0 + 4) {
    // ===================================================== A4: block-local softmax, two tokens per thread
    const int q = warp - kWarpSoftmax0;
    const uint32_t taddr = tmem_S + q * kSCols + (static_cast<uint32_t>(q * 32) << 16);
    int st = q % S;
    // ---- home duty (ART on).  The softmax warps are idle most of the time and carry no state from item to item, so
    //      they replay Algorithm 1 for the group this CTA opened: warp w scans heads w GW .. w GW + GW - 1
    //      (art_scan_chunk.cuh) and leaves one byte per step in `stab`; warp 0 also walks the patience counter over
    //      those bytes and broadcasts the progress word.  One call does at most one chunk; true if it did something.
      constexpr int LPH = Scan::LPH, CPL = Scan::CPL, NBK = Scan::NBK, STRIDE = Scan::STRIDE;
      constexpr int NSW = G / GW;                             // warps that have heads to scan
      const int fw = warp - kWarpSoftmax0;                    // softmax warp w scans heads w GW .. w GW + GW - 1
      const int sub = lane % LPH, h_scan = fw * GW + lane / LPH;   // the head this lane scans
      const bool owner = (sub % STRIDE) == 0;
      const int own_k = sub / STRIDE;
      const bool i_scan = fw < NSW && fw * GW < p.Gr;         // this warp has at least one real head
      const int nsw_real = (p.Gr + GW - 1) / GW;              // warps whose bytes the decider waits for
      int sg = 0;                                             // groups of this home CTA already scanned
      bool scanning = false;
      int s_t = 1, s_T = 0, s_gen = 0, s_group = 0, s_hs = 0; // the group being scanned: next step, ...
      int d_t = 0, d_cnt = 0;                                 // warp 0: last decided step, c^(t)
      Scan sc; sc.init(true);
      // a chunk whose summaries are on their way over distributed shared memory (issued at the top of an iteration,
      // looked at after the item work of the same iteration: the round trip hides behind it)
      int pend_n = 0;
      long long pend_t0 = 0; (void)pend_t0;
      uint32_t pend_word = 0u, pend_ml[2] = {0u, 0u}, pend_raw[NBK][CPL];
      auto issue_pull = [&]() {
        const uint32_t wk_own = __shfl_sync(0xffffffffu, pend_word, own_k);
        if (owner && own_k < pend_n)
          ld_cluster_vec<2>(mapa(sbase + sm.sums + (wk_own & 7u) * SUMB, (wk_own >> 4) & 15u) + static_cast<uint32_t>(G * PW + 2 * h_scan) * 4u, pend_ml);
#pragma unroll
        for (int k = 0; k < NBK; ++k) {
          const uint32_t wk = __shfl_sync(0xffffffffu, pend_word, k);
          if (k < pend_n) ld_cluster_vec<CPL>(mapa(sbase + sm.sums + (wk & 7u) * SUMB, (wk >> 4) & 15u) + static_cast<uint32_t>(h_scan * PW + sub * CPL) * 4u, pend_raw[k]);
        }
      };
      // which of the next NBK steps have arrived (lane k looks at step first + k)?  Issue the loads of their summaries.
      auto poll_and_pull = [&](int first) {
        const uint32_t tg = sbase + sm.tags + static_cast<uint32_t>(s_hs & 1) * kNR * 4u;
        bool ok = false;
        pend_word = 0u;
        if (lane < NBK && first + lane <= s_T) {
          pend_word = static_cast<uint32_t>(ld_volatile_s32(tg + static_cast<uint32_t>((first + lane - 1) % kNR) * 4u));
          ok = (pend_word >> 8) == static_cast<uint32_t>(first + lane);
        }
        pend_n = __ffs(~__ballot_sync(0xffffffffu, ok)) - 1;
        if (pend_n > 0) { issue_pull(); ART_STAT_SET(pend_t0); }
      };
      auto scan_duty = [&]() -> bool {
        bool progress = false;
        // ---- (3) home duty
        if (!scanning) {
          int oc;
          asm volatile("ld.acquire.cta.shared::cta.s32 %0, [%1];" : "=r"(oc) : "r"(a_misc + kMOpen) : "memory");
          if (oc > sg) {
            const HomeInfo* hi = reinterpret_cast<const HomeInfo*>(smem + sm.hinfo) + (sg & 1);
            s_group = *reinterpret_cast<const volatile int*>(&hi->group); s_T = *reinterpret_cast<const volatile int*>(&hi->T);
            s_gen = *reinterpret_cast<const volatile int*>(&hi->gen);
            s_hs = rank * 2 + (sg & 1); s_t = 1; d_t = 0; d_cnt = 0;
            sc.init(h_scan < p.Gr);
            scanning = true;
          }
        }
        if (scanning) {
          const int hsl = s_hs & 1;
          bool fin_seen;
          const int g_dec = read_ctrl(s_hs, s_gen, fin_seen);
          fin_seen = fin_seen || g_dec >= s_T;
          if (fin_seen) { scanning = false; pend_n = 0; ++sg; progress = true; }
          else if (i_scan && pend_n == 0 && s_t <= s_T) { poll_and_pull(s_t); progress = pend_n > 0; }
          else if (pend_n > 0) {
            // ---- (3b) the chunk's summaries are here.  A word whose parity bit is the slot's previous generation's
            //      (written by another warp of the producing CTA a moment later): pull again.
            int n = pend_n;
            const uint32_t wk_own = __shfl_sync(0xffffffffu, pend_word, own_k);
            const bool has_own = owner && own_k < n;
            uint32_t bad = has_own ? ((pend_ml[0] ^ (wk_own >> 3)) | (pend_ml[1] ^ (wk_own >> 3))) : 0u;
            float pv[NBK][CPL];
#pragma unroll
            for (int k = 0; k < NBK; ++k) {
              const uint32_t pk = __shfl_sync(0xffffffffu, pend_word, k) >> 3;
#pragma unroll
              for (int j = 0; j < CPL; ++j) {
                if (k < n) { bad |= pend_raw[k][j] ^ pk; pv[k][j] = __uint_as_float(pend_raw[k][j]); }
                else pv[k][j] = 0.f;
              }
            }
            if (__any_sync(0xffffffffu, (bad & 1u) != 0u)) {
              if (fw == 0) ART_STAT_ADD(4, 1);
              issue_pull();                                   // (if Algorithm 1 has fired meanwhile, fin_seen ends this next time round)
            } else {
              float m_own = kNegInf, l_own = 0.f;
              if (has_own) { m_own = __uint_as_float(pend_ml[0]); l_own = __uint_as_float(pend_ml[1]); if (m_own <= -1e29f) m_own = kNegInf; }
              if (n > 1 && !sc.spread_ok(m_own, owner)) {     // exponents too far apart for one reference: one step at a time
                n = 1;
                if (own_k >= 1) { m_own = kNegInf; l_own = 0.f; }
#pragma unroll
                for (int k = 1; k < NBK; ++k)
#pragma unroll
                  for (int j = 0; j < CPL; ++j) pv[k][j] = 0.f;
              }
              // the next chunk's summaries travel while this one is scanned
              const int first = s_t;
              s_t += n;
              pend_n = 0;
              if (s_t <= s_T) poll_and_pull(s_t);
              ART_STAT_T(tc0);
              const uint32_t bits = sc.chunk(n, lane, p.tau, p.phi, m_own, l_own, pv);
              ART_STAT_T(tc1);
              if (fw == 0) { ART_STAT_ADD(0, 1); ART_STAT_ADD(1, n); ART_STAT_ADD(2, tc0 - pend_t0); ART_STAT_ADD(3, tc1 - tc0); }
              // one byte per step: [lap tag : 7][stable : 1]
              if (lane < n) {
                const int s = first + lane;
                const uint32_t byte = (static_cast<uint32_t>(((s - 1) / kNR) % 127 + 1) << 1) | ((bits >> lane) & 1u);
                *reinterpret_cast<volatile uint8_t*>(smem + sm.stab + (hsl * 4 + fw) * kNR + (s - 1) % kNR) = static_cast<uint8_t>(byte);
              }
            }
            progress = true;
          }
          if (fw == 0 && !fin_seen) {
            // ---- the patience counter (Eq. 3) over the steps every scanning warp has finished
            bool valid = false, stable = true;
            const int s = d_t + 1 + lane;
            if (lane < 16 && s <= s_T) {
              const uint32_t want = static_cast<uint32_t>(((s - 1) / kNR) % 127 + 1);
              valid = true;
              for (int w = 0; w < nsw_real; ++w) {
                const uint32_t b8 = *reinterpret_cast<volatile uint8_t*>(smem + sm.stab + (hsl * 4 + w) * kNR + (s - 1) % kNR);
                valid = valid && (b8 >> 1) == want;
                stable = stable && (b8 & 1u);
              }
            }
            const int nv = __ffs(~__ballot_sync(0xffffffffu, valid)) - 1;
            if (nv > 0) {
              const uint32_t sb = __ballot_sync(0xffffffffu, stable);
              int fired_at = 0;
              for (int k = 0; k < nv && !fired_at; ++k) {
                d_cnt = ((sb >> k) & 1u) ? d_cnt + 1 : 0;     // Eq. 3
                if (d_cnt >= p.patience) fired_at = d_t + 1 + k;
              }
              d_t = fired_at ? fired_at : d_t + nv;
              const uint32_t a_c = sbase + sm.ctrl + static_cast<uint32_t>(s_hs) * 4u;
              if (fired_at || d_t >= s_T) {
                // t* is known: record it, let the last flusher recognise itself, THEN release the final progress word
                if (lane == 0) {
                  p.stop_block[s_group] = d_t;               // t* (R9)
                  asm volatile("red.relaxed.cluster.shared::cluster.add.u64 [%0], %1;" :: "r"(hinfo_at(s_hs, H_DONE)), "l"(static_cast<unsigned long long>(d_t + 1) << 32) : "memory");
                }
                __syncwarp();
                if (lane < CL) st_cluster_release_s32(mapa(a_c, lane), ctrl_word(s_gen, fired_at != 0, d_t));
              } else if (lane < CL) {
                st_cluster_relaxed_s32(mapa(a_c, lane), ctrl_word(s_gen, false, d_t));
              }
              progress = true;
            }
          }
        }
        return progress;
      };
      // true once no group is left for this CTA to scan
      auto scan_all_done = [&]() -> bool {
        if (scanning || !ld_volatile_s32(a_misc + kMScanExit)) return false;
        int oc;
        asm volatile("ld.acquire.cta.shared::cta.s32 %0, [%1];" : "=r"(oc) : "r"(a_misc + kMOpen) : "memory");
        return oc <= sg;
      };
    for (int i = q;; i += NS) {
      if constexpr (ART) {
        ART_WATCH(wds, 7);
        while (!mbar_test_wait(bar(sm.sfull0 + q), (i / NS) & 1)) { if (!scan_duty()) nsleep(pp.nap); if (scanning) ART_WATCH_POLL(wds, s_t, (d_t << 8) | (pend_n << 4) | (scanning ? 1 : 0) | (q << 1)); }
      } else {
        mbar_wait(bar(sm.sfull0 + q), (i / NS) & 1);
      }
      const int kind = item_kind(items[i % kItemsRing].meta);
      if (kind == ITEM_END) {
        // the END item that owns a stage is the first of the four; only its warp hands it on to the P.V issuer
        if (item_kind(items[(i + kItemsRing - 1) % kItemsRing].meta) != ITEM_END || i == 0) mbar_arrive(bar(sm.pfull0 + st));
        if constexpr (ART) {                                  // no item left; the group(s) this CTA opened may still run
          ART_WATCH(wde, 8);
          while (!scan_all_done()) { if (!scan_duty()) nsleep(pp.nap); ART_WATCH_POLL(wde, s_t, (d_t << 8) | (pend_n << 4) | (scanning ? 1 : 0) | (q << 1)); }
        }
        break;
      }
      if (kind != ITEM_DATA) {                               // a marker: nothing to compute
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(sm.sfree0 + q));
        mbar_arrive(bar(sm.pfull0 + st));
        st += NS; while (st >= S) st -= S;
        continue;
      }
      tc_fence_after();
      float s0[G], s1[G];
      tmem_ld<G>(taddr, s0);
      tmem_ld<G>(taddr + kUmmaN, s1);
      tmem_ld_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(sm.sfree0 + q));
      if (kTwoPBufs && i >= 2) mbar_wait(bar(sm.pvfull0 + ((i - 2) & (NP - 1))), ((i - 2) / NP) & 1);
      const unsigned long long vmask = items[i % kItemsRing].mask;
      const bool v0 = (vmask >> lane) & 1ull, v1 = (vmask >> (lane + 32)) & 1ull;
      float mb[G];
      int ec = 0;
      if constexpr (MT) ec = items[i % kItemsRing].tcode >> kItemShift;
      if (MT && ec != 0) {                                    // R15: the most recent tokens are cut row by row
#pragma unroll
        for (int h = 0; h < G; ++h) {
          const int lim = ec - static_cast<int>((p.cuts >> (4 * h)) & 15u);
          s0[h] = (v0 && lane < lim) ? s0[h] * p.scale_log2 : kNegInf;
          s1[h] = (v1 && lane + 32 < lim) ? s1[h] * p.scale_log2 : kNegInf;
          mb[h] = warp_max_f32(fmaxf(s0[h], s1[h]));
        }
      } else {
#pragma unroll
        for (int h = 0; h < G; ++h) {
          s0[h] = v0 ? s0[h] * p.scale_log2 : kNegInf;        // masked tokens: weight 0 (R8); their K may be NaN
          s1[h] = v1 ? s1[h] * p.scale_log2 : kNegInf;
          mb[h] = warp_max_f32(fmaxf(s0[h], s1[h]));
        }
      }
      uint8_t* pb0 = smem + sm.pb + (kTwoPBufs ? (i & 1) : st) * 2 * PBUF + (lane >> 3) * LBO_P + (lane & 7) * 2;
      float ls[G];
#pragma unroll
      for (int h = 0; h < G; ++h) {
        const float p0 = (v0 && mb[h] != kNegInf) ? fast_exp2(s0[h] - mb[h]) : 0.f;
        const float p1 = (v1 && mb[h] != kNegInf) ? fast_exp2(s1[h] - mb[h]) : 0.f;
        const __nv_bfloat16 h0 = __float2bfloat16_rn(p0), h1 = __float2bfloat16_rn(p1);
        const __nv_bfloat16 l0 = __float2bfloat16_rn(p0 - __bfloat162float(h0)), l1 = __float2bfloat16_rn(p1 - __bfloat162float(h1));
        *reinterpret_cast<__nv_bfloat16*>(pb0 + h * 16) = h0;
        *reinterpret_cast<__nv_bfloat16*>(pb0 + h * 16 + 4 * LBO_P) = h1;
        *reinterpret_cast<__nv_bfloat16*>(pb0 + h * 16 + PBUF) = l0;
        *reinterpret_cast<__nv_bfloat16*>(pb0 + h * 16 + PBUF + 4 * LBO_P) = l1;
        ls[h] = (__bfloat162float(h0) + __bfloat162float(l0)) + (__bfloat162float(h1) + __bfloat162float(l1));
      }
      if (vmask != ~0ull) {                                   // masked V rows may hold NaN: 0 * NaN would poison P~V
        uint4* vr = reinterpret_cast<uint4*>(smem + sm.ring + st * kStageBytes + 2 * kBoxBytes);
        if (!v0) {
#pragma unroll
          for (int c = 0; c < 8; ++c) { vr[lane * 8 + c] = make_uint4(0u, 0u, 0u, 0u); vr[lane * 8 + c + kBoxBytes / 16] = make_uint4(0u, 0u, 0u, 0u); }
        }
        if (!v1) {
#pragma unroll
          for (int c = 0; c < 8; ++c) { vr[(lane + 32) * 8 + c] = make_uint4(0u, 0u, 0u, 0u); vr[(lane + 32) * 8 + c + kBoxBytes / 16] = make_uint4(0u, 0u, 0u, 0u); }
        }
      }
      Reduce32<G, 16>::run(ls, lane);
      {
        const int hh = head_of_lane32<G>(lane);
        float mine = mb[0];
#pragma unroll
        for (int h = 1; h < G; ++h) mine = (hh == h) ? mb[h] : mine;
        float* slot = slots + (i & (kIterSlots - 1)) * 2 * G;
        if ((lane & (32 / G - 1)) == 0) { slot[hh] = mine; slot[G + hh] = ls[0]; }
      }
      fence_proxy_async();
      mbar_arrive(bar(sm.pfull0 + st));
      st += NS; while (st >= S) st -= S;
    }
  } else if (warp < kWarpFold0 + 4) {
    // ===================================================== A5 / A6 / A8 / A9: publish summaries, merge P~V_t, flush, combine
    const uint32_t tlane = static_cast<uint32_t>(fq * 32) << 16;
    float acc[G], m_tot[G], l_tot[G];
    int nfold = 0;
    auto reset_state = [&]() {
#pragma unroll
      for (int h = 0; h < G; ++h) { acc[h] = 0.f; m_tot[h] = kNegInf; l_tot[h] = 0.f; }
      nfold = 0;
    };
    reset_state();
    auto release_pv = [&](int i) {
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(sm.pvfree0 + (i & (NP - 1))));
    };
    auto fold = [&](int i) {
      tc_fence_after();
      float pv[G];
      tmem_ld<G>(tmem_PV + tlane + (i & (NP - 1)) * kUmmaN, pv);
      tmem_ld_wait();
      const float* sl = slots + (i & (kIterSlots - 1)) * 2 * G;
#pragma unroll
      for (int h = 0; h < G; ++h) {
        const float mr = sl[h];
        if (mr != kNegInf) {                                  // a block with no valid token changes nothing
          const float mn = fmaxf(m_tot[h], mr);
          const float a = fast_exp2(m_tot[h] - mn), bb = fast_exp2(mr - mn);
          acc[h] = fmaf(a, acc[h], bb * pv[h]);
          l_tot[h] = fmaf(a, l_tot[h], bb * sl[G + h]);
          m_tot[h] = mn;
        }
      }
      ++nfold;
      release_pv(i);
    };
    // out[row h] = our own partial state (registers) merged with the flushed partial states of the CTAs in `others`
    // (flash-decoding merge).  The partial states are read a few at a time with every load of a
    // batch in flight at once: the combine sits on the tail of the call.
    auto combine = [&](int group, unsigned others, int T) {
      const int b = group / p.Hkv, g = group % p.Hkv;
      constexpr int CH = G <= 2 ? 4 : (G <= 4 ? 3 : 2);
      float mx[G], a[G], l[G];
#pragma unroll
      for (int h = 0; h < G; ++h) { mx[h] = m_tot[h]; a[h] = acc[h]; l[h] = l_tot[h]; }
      unsigned js = others;
      while (js) {
        const float* pc[CH];
#pragma unroll
        for (int k = 0; k < CH; ++k) {
          pc[k] = nullptr;
          if (js) { pc[k] = pp.part + (static_cast<size_t>(group) * CL + (__ffs(js) - 1)) * PF; js &= js - 1; }
        }
        float mc[CH][G], lc[CH][G], ac[CH][G];
#pragma unroll
        for (int k = 0; k < CH; ++k)
#pragma unroll
          for (int h = 0; h < G; ++h) {
            mc[k][h] = pc[k] ? __ldcg(pc[k] + G * kD + h) : kNegInf;
            lc[k][h] = pc[k] ? __ldcg(pc[k] + G * kD + G + h) : 0.f;
            ac[k][h] = pc[k] ? __ldcg(pc[k] + h * kD + d) : 0.f;
          }
#pragma unroll
        for (int k = 0; k < CH; ++k)
#pragma unroll
          for (int h = 0; h < G; ++h) {
            if (mc[k][h] != kNegInf) {
              const float mn = fmaxf(mx[h], mc[k][h]);
              const float f0 = fast_exp2(mx[h] - mn), f1 = fast_exp2(mc[k][h] - mn);
              a[h] = fmaf(f0, a[h], f1 * ac[k][h]);
              l[h] = fmaf(f0, l[h], f1 * lc[k][h]);
              mx[h] = mn;
            }
          }
      }
#pragma unroll
      for (int h = 0; h < G; ++h)
        if (h < p.Gr)                                         // Alg. 1 l.18; row h = query token h / Gh, head h % Gh
          p.out[((static_cast<int64_t>(b) * p.qlen + h / p.Gh) * p.Hq + g * p.Gh + h % p.Gh) * kD + d] = (l[h] > 0.f) ? a[h] / l[h] : 0.f;
      if (!ART && d == 0) p.stop_block[group] = T;
    };
    // End of a visit: hand the partial state over, combine if we are the last, leave the group.
    //   done word of the group (home CTA): low half = steps folded AND flushed so far, high half = t* + 1 once known.
    //   Whoever brings the low half to t* combines.  A CTA that finds itself the group's only worker ever (nobody
    //   else is working on it, nobody has flushed, all t* steps are in its registers) skips the round trip.
    auto flush = [&](int tcode, int meta, unsigned long long payload) {
      const int hs = item_hs(meta), group = static_cast<int>(payload);
      if (warp == kWarpFold0 && lane == 0) {
        int flag = 0;                                         // 0: not ours to combine; 1: alone; >= 2: last of several, t* + 1
        if (p.blocks_loaded && tcode > 0) atomicAdd(p.blocks_loaded + group, tcode);
        if (nfold > 0) {
          const int nact = ld_cluster_relaxed_s32(board_at(hs, B_NACT));
          const unsigned jn = ld_cluster_u32(hinfo_at(hs, H_JOINED));
          unsigned long long dn;
          asm volatile("ld.relaxed.cluster.shared::cluster.u64 %0, [%1];" : "=l"(dn) : "r"(hinfo_at(hs, H_DONE)) : "memory");
          if (nact == 1 && jn == 0u && static_cast<unsigned>(dn) == 0u && static_cast<unsigned>(dn >> 32) == static_cast<unsigned>(nfold) + 1u) flag = 1;
        }
        st_volatile_s32(a_misc + kMFlag, flag);
        st_volatile_s32(a_misc + kMJoined, 0);
      }
      named_bar_sync(1, 128);
      int flag = ld_volatile_s32(a_misc + kMFlag);
      if (flag == 0 && nfold > 0) {
        float* part = pp.part + (static_cast<size_t>(group) * CL + rank) * PF;
#pragma unroll
        for (int h = 0; h < G; ++h) {
          part[h * kD + d] = acc[h];
          if (d == 0) { part[G * kD + h] = m_tot[h]; part[G * kD + G + h] = l_tot[h]; }
        }
        named_bar_sync(1, 128);                               // every thread's part is written ...
        if (warp == kWarpFold0 && lane == 0) {
          const unsigned before = atom_or_cluster(hinfo_at(hs, H_JOINED), 1u << rank);
          // ... and released by this one atomic (cumulative over the barrier); acquire: the partial states of the others
          const unsigned long long old = atom_add64_cluster_acqrel(hinfo_at(hs, H_DONE), static_cast<unsigned long long>(nfold));
          const unsigned long long tot = old + static_cast<unsigned long long>(nfold);
          const unsigned hi = static_cast<unsigned>(tot >> 32), lo = static_cast<unsigned>(tot);
          if (hi != 0u && lo == hi - 1u) {                    // every step <= t* is folded and flushed: we combine
            st_volatile_s32(a_misc + kMJoined, static_cast<int>((before | ld_cluster_u32(hinfo_at(hs, H_JOINED))) & ~(1u << rank)));
            st_volatile_s32(a_misc + kMFlag, static_cast<int>(hi));      // >= 2: t* + 1
          }
        }
        named_bar_sync(1, 128);
        flag = ld_volatile_s32(a_misc + kMFlag);
      }
      if (flag) combine(group, static_cast<unsigned>(ld_volatile_s32(a_misc + kMJoined)), flag == 1 ? nfold : flag - 1);
      named_bar_sync(1, 128);                                 // flag and mask are read by all before the next flush rewrites them
      // leave; the release orders our notices before a re-opening of the slot can clear its notice ring
      if (warp == kWarpFold0 && lane == 0) { if constexpr (ART) atom_add_cluster_release(board_at(hs, B_NACT), -1); else atom_add_cluster(board_at(hs, B_NACT), -1); }
      reset_state();
    };

    if constexpr (!ART) {
      for (int i = 0;; ++i) {
        mbar_wait(bar(sm.pvfull0 + (i & (NP - 1))), (i / NP) & 1);
        const int meta = items[i % kItemsRing].meta;
        const int kind = item_kind(meta);
        if (kind == ITEM_DATA) { fold(i); continue; }
        if (kind == ITEM_END) break;
        flush(items[i % kItemsRing].tcode, meta, items[i % kItemsRing].mask);
        release_pv(i);
      }
    } else {
      // ---- ART on: (1) merge or drop the oldest finished item once its step is decided, (2) write the summary of the
      //      next finished item and tell its group's home.  Neither waits for the other.
      constexpr int LPH = Scan::LPH, CPL = Scan::CPL;
      int pub = 0, fld = 0;
      bool pub_ready = false, items_done = false;
      ART_WATCH(wd, 3);
      while (!items_done) {
        bool progress = false;
        // ---- (1) the oldest unfolded item
        if (!items_done && fld < pub) {
          const int meta = items[fld % kItemsRing].meta;
          const int kind = item_kind(meta);
          if (kind == ITEM_DATA) {
            bool fired;
            const int tdec = read_ctrl(item_hs(meta), item_gen(meta), fired);
            const int tf = items[fld % kItemsRing].tcode & kItemStep;
            if (fired && tf > tdec) { release_pv(fld); ++fld; progress = true; }
            else if (tdec >= tf) { fold(fld); ++fld; progress = true; }   // decided: the scan has read this step's summary
          } else if (kind == ITEM_FLUSH) {
            flush(items[fld % kItemsRing].tcode, meta, items[fld % kItemsRing].mask);
            release_pv(fld); ++fld; progress = true;
          } else {
            items_done = true;                                // END: only the home duty may be left
          }
        }
        // ---- (2) the next finished item: write its summary, tell the group's home where it is
        if (!items_done && pub - fld < NSUM) {
          const uint32_t pvb = bar(sm.pvfull0 + (pub & (NP - 1)));
          const uint32_t par = (pub / NP) & 1;
          if (!pub_ready) pub_ready = (fld == pub) ? mbar_try_wait(pvb, par) : mbar_test_wait(pvb, par);
          if (pub_ready) {
            const int meta = items[pub % kItemsRing].meta;
            if (item_kind(meta) == ITEM_DATA) {
              const int hs = item_hs(meta), t = items[pub % kItemsRing].tcode & kItemStep;
              const int sslot = pub % NSUM;
              const uint32_t gpar = static_cast<uint32_t>(pub / NSUM) & 1u;
              tc_fence_after();
              float pv[G];
              tmem_ld<G>(tmem_PV + tlane + (pub & (NP - 1)) * kUmmaN, pv);
              tmem_ld_wait();
              uint32_t* sw = reinterpret_cast<uint32_t*>(smem + sm.sums + sslot * SUMB);
              if (MODE == 2 || (d & 3) == 0) {
                const int pi = (MODE == 2) ? d : (d >> 2);    // probe coordinate k * (d / 32)  (R1)
#pragma unroll
                for (int h = 0; h < G; ++h) sw[h * PW + (pi % LPH) * CPL + pi / LPH] = tag_word(pv[h], gpar);
              }
              if (d == 1) {
                const float* sl = slots + (pub & (kIterSlots - 1)) * 2 * G;
#pragma unroll
                for (int h = 0; h < G; ++h) {
                  sw[G * PW + 2 * h] = tag_word(fmaxf(sl[h], kNegBig), gpar);
                  sw[G * PW + 2 * h + 1] = tag_word(sl[G + h], gpar);
                }
              }
              __syncwarp();
              // the notice: step number, producing CTA, slot, parity; sent by the warp that finishes last
              if (lane == 0) {
                const int prev = atomicAdd(reinterpret_cast<int*>(smem + sm.misc + kMPubCnt) + sslot, 1);
                if ((prev & 3) == 3) {
                  const uint32_t word = (static_cast<uint32_t>(t) << 8) | (static_cast<uint32_t>(rank) << 4) | (gpar << 3) | static_cast<uint32_t>(sslot);
                  const uint32_t dst = mapa(sbase + sm.tags + (static_cast<uint32_t>(hs & 1) * kNR + static_cast<uint32_t>((t - 1) % kNR)) * 4u, hs >> 1);
                  asm volatile("st.relaxed.cluster.shared::cluster.u32 [%0], %1;" :: "r"(dst), "r"(word) : "memory");
                }
              }
            }
            ++pub; pub_ready = false; progress = true;
          }
        }
        if (!progress && fld < pub) { nsleep(pp.nap); ART_WATCH_POLL(wd, items[fld % kItemsRing].tcode, ld_ctrl_relaxed(sbase + sm.ctrl + static_cast<uint32_t>(item_hs(items[fld % kItemsRing].meta)) * 4u)); }
      }
    }
  }

  // ===================================================== every role is done; peers may still read our shared memory
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  if (warp == kWarpMmaPV) { tc_fence_after(); tmem_dealloc(tmem_base, kTmemCols); }
}

}  // namespace pc
}  // namespace art
