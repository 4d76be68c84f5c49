// ART decode attention, bf16 KV / head_dim 128, DETECTOR OFF: persistent clusters with run-time scheduling
// (tcgen05 + TMEM + TMA).  Runs when the caller asks for it (art_desc_t.split < 0) and behind
// art_decode_attention_off_static.  Built for many short groups (configs[3]), where one short-lived cluster per group runs
// in several waves, each CTA paying for its own start-up (tensor-memory allocation, cluster barriers, Q staging) and
// tail; since the MMA operand traffic was halved the static one-CTA clusters are as fast there.
//
// The grid is NC thread-block clusters of CL CTAs (two CTAs per SM), launched once and resident for the whole call.
// Cluster c owns the query groups c, c + NC, c + 2 NC, ...  Nothing inside a cluster is bound:
//
//   * a CTA that needs work OPENS the next group of its cluster (it becomes the group's HOME) or, when the cluster has
//     no unopened group left, JOINS the open group of its cluster with the most unclaimed steps per worker: at the tail
//     of the call the CTAs that ran out of groups stream for the groups that are still open;
//   * traversal steps t = 1..T are CLAIMED a few at a time from the group's counter on the cluster's
//     board (rank 0's shared memory, atom.shared::cluster), one claim ahead of the step being issued;
//   * one 64-token KV block is one pipeline ITEM, handled by specialised warps that meet through mbarriers exactly as
//     in art_decode_tc.cuh (TMA -> S = K Q^T -> block-local softmax -> P~V = V^T P^T with P split hi + lo -> merge into
//     the CTA's running (m, l, acc)); marker items travel through the same pipeline to end a visit or the call, so
//     every role waits on barriers only and nothing polls;
//   * a CTA that leaves a group flushes its partial (m, l, acc) to the workspace; whoever completes the group's count of
//     folded steps combines the partial states (flash-decoding merge) and writes `out` (A8/A9).  A CTA that was the
//     group's only worker writes `out` straight from its registers.
//
// With the detector ON the library always uses the static clusters of art_decode_tc.cuh: three persistent variants
// were built and measured in round 2 (summaries pulled over DSMEM, pushed into a home mailbox, scanned by one or by
// four warps); none came within 25 % of the static clusters (DESIGN.md section 6.5.2 has the numbers and the reasons).
#pragma once
#include "art_decode_tc.cuh"

namespace art {
namespace pc {

using namespace tc;

constexpr int kMaxCL = 16;
constexpr int kHS = 2 * kMaxCL;              // home slots of a cluster: two per CTA (a CTA opens its next group while the last one drains)
constexpr int kItemsRing = 32;               // item descriptors; >= stages + kPVSlots + the four END items
constexpr int kLock = -(1 << 20);            // board.nact while a slot is being (re)opened
constexpr int kMinJoin = 4;                  // a group with fewer unclaimed steps is not worth a Q reload and a partial state
static_assert(kItemsRing >= kPVSlots + kMaxStages + 4, "item ring too short");

struct PcParams {
  Params b;
  int32_t n_groups, NC;
  float* part;                               // workspace: partial states [group][rank][G * (kD + 2)]
  int32_t claim;                             // steps claimed per atomic (a chunk of consecutive steps)
  unsigned long long* dbg;                   // ART_WATCHDOG: where a wait that never ended reports itself
};

enum { ITEM_DATA = 0, ITEM_FLUSH = 1, ITEM_END = 2 };
// meta: bits 0-4 home slot, 5 Q buffer, 6-7 kind
struct Item { int tcode; int meta; unsigned long long mask; };   // FLUSH: tcode = blocks loaded in the visit, mask = group
__device__ __forceinline__ int item_hs(int meta) { return meta & 31; }
__device__ __forceinline__ int item_q(int meta) { return (meta >> 5) & 1; }
__device__ __forceinline__ int item_kind(int meta) { return (meta >> 6) & 3; }

struct HomeInfo { unsigned long long done; int group, T, gen, loaded; unsigned joined; int pad; };   // home CTA: one per local slot

struct SmemMapP {
  uint32_t qb, pb, slots, xch, items, hinfo, board, bars, misc, ring, total;
  uint32_t full0, empty0, pfull0, sfull0, sfree0, pvfull0, pvfree0, done0, nbars;
};

__host__ __device__ inline SmemMapP make_smem_map_p(int G, int stages) {
  SmemMapP m;
  uint32_t off = 0;
  m.qb = off; off += 2u * kQBytes;
  m.pb = off; off += static_cast<uint32_t>(stages) * 2u * p_buf_bytes(G);
  m.slots = off; off += kIterSlots * static_cast<uint32_t>(3 * G) * 4u;           // per item: m_blk[G], block sum of tokens 0-31 [G], of tokens 32-63 [G]
  m.xch = off; off += 8u * G * 4u;                                                // block maxima of the two token halves: [pair][parity][half][G]
  m.items = off; off += kItemsRing * static_cast<uint32_t>(sizeof(Item));
  off = (off + 15u) & ~15u;
  m.hinfo = off; off += 2u * static_cast<uint32_t>(sizeof(HomeInfo));
  m.board = off; off += kHS * 32u + 16u;                         // rank 0: {next, T, nact, group, gen} per home slot, + next_local
  m.bars = off;
  uint32_t n = 0;
  m.full0 = n; n += stages; m.empty0 = n; n += stages; m.pfull0 = n; n += stages;
  m.sfull0 = n; n += kSSlots; m.sfree0 = n; n += kSSlots;
  m.pvfull0 = n; n += kPVSlots; m.pvfree0 = n; n += kPVSlots;
  m.done0 = n; n += 2;
  m.nbars = n;
  off += n * 8u;
  m.misc = off; off += 32u;
  off = (off + 1023u) & ~1023u;
  if (off < static_cast<uint32_t>(kFront)) off = kFront;
  m.ring = off; off += static_cast<uint32_t>(stages) * kStageBytes;
  m.total = off;
  return m;
}
constexpr uint32_t kMTmem = 0, kMFlag = 12, kMJoined = 16;

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
__device__ __forceinline__ uint32_t ld_cluster_u32(uint32_t a) {
  uint32_t v; asm volatile("ld.relaxed.cluster.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory"); return v;
}
__device__ __forceinline__ void named_bar_sync(int id, int threads) { asm volatile("bar.sync %0, %1;" :: "r"(id), "r"(threads) : "memory"); }
__device__ __forceinline__ void nsleep(unsigned ns) { asm volatile("nanosleep.u32 %0;" :: "r"(ns)); }
__device__ __forceinline__ unsigned long long gtime() { unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }

// A wait that does not end within two seconds is a scheduling bug: report where and trap, so that the call fails
// instead of hanging the device.  Compiled in with -DART_WATCHDOG (a debugging build); free otherwise.
#ifdef ART_WATCHDOG
struct Watch {
  unsigned long long t0; unsigned long long* dbg; int code;
  __device__ __forceinline__ Watch(unsigned long long* d, int c) : t0(gtime()), dbg(d), code(c) {}
  __device__ __forceinline__ void poll(int a = 0, int b = 0) {
    if (gtime() - t0 > 2000000000ull) {
      if (dbg) { dbg[0] = (static_cast<unsigned long long>(code) << 48) | (static_cast<unsigned long long>(blockIdx.x) << 32) | (static_cast<unsigned>(a) & 0xffffu) << 16 | (static_cast<unsigned>(b) & 0xffffu); __threadfence_system(); }
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

// ----------------------------------------------------------------------------- the kernel

template <int G, bool MT = false>
__global__ void __launch_bounds__(kThreads, 2)
art_decode_pc_kernel(const PcParams pp, const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV) {
  constexpr int NP = kPVSlots, NS = kSSlots;
  constexpr int LBO_P = p_lbo(G), PBUF = p_buf_bytes(G);
  constexpr int PF = G * (kD + 2);                       // floats of one partial state
  const Params& p = pp.b;

  extern __shared__ __align__(1024) uint8_t smem[];
  const int S = p.stages;
  const SmemMapP sm = make_smem_map_p(G, S);
  const uint32_t sbase = smem_u32(smem);
  if ((sbase & 1023u) != 0u) __trap();
  const uint32_t bars = sbase + sm.bars;
  auto bar = [&](uint32_t idx) { return bars + idx * 8u; };
  float* slots = reinterpret_cast<float*>(smem + sm.slots);   // [item & 15][3 G]: block maximum (log2 domain), block sums of the two token halves
  float* xch = reinterpret_cast<float*>(smem + sm.xch);
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
  enum { B_NEXT = 0, B_T = 1, B_NACT = 2, B_GROUP = 3 };
  constexpr uint32_t H_DONE = 0, H_JOINED = 24;

  // ---- one-time setup
  if (tid == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(bar(sm.full0 + s), 1); mbar_init(bar(sm.empty0 + s), 1); mbar_init(bar(sm.pfull0 + s), 64); }
    for (int s = 0; s < NS; ++s) { mbar_init(bar(sm.sfull0 + s), 1); mbar_init(bar(sm.sfree0 + s), 2); }
    for (int s = 0; s < NP; ++s) { mbar_init(bar(sm.pvfull0 + s), 1); mbar_init(bar(sm.pvfree0 + s), 4); }
    mbar_init(bar(sm.done0), 1); mbar_init(bar(sm.done0 + 1), 1);
    st_volatile_s32(a_misc + kMFlag, 0);
    fence_mbar_init();
  }
  for (int i = tid; i < kHS; i += kThreads) {
    int* e = reinterpret_cast<int*>(smem + sm.board + i * 32);
    e[B_NEXT] = 0; e[B_T] = 0; e[B_NACT] = 0; e[B_GROUP] = -1;
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
    for (int idx = tid; idx < S * 2 * PBUF / 16; idx += kThreads) pz[idx] = make_uint4(0u, 0u, 0u, 0u);
  }
  fence_proxy_async();
  tc_fence_before();
  cluster_sync_all();                                        // boards and barriers of every CTA are live
  tc_fence_after();
  const uint32_t tmem_base = static_cast<uint32_t>(ld_volatile_s32(a_misc + kMTmem));
  const uint32_t tmem_S = tmem_base, tmem_PV = tmem_base + NS * kSCols1;

  // fold warps: output coordinate and running (un-normalised) partial state of the current visit
  const int fq = warp & 3;
  const int d = fq * 32 + lane;

  // ===================================================== scheduling state of the producer warp (open / join / claim)
  int it = 0, stage = 0; uint32_t ph = 0;
  int my_gen = 0;                                          // groups this CTA has opened
  int nvisit = 0;                                          // visits that issued at least one item
  int q_last[2] = {-1, -1};                                // last item that reads Q buffer 0 / 1
  bool more_local = n_local > n_init;
  // the visit
  bool have = false;
  int v_hs = 0, v_group = 0, v_T = 0, v_b = 0, v_g = 0, v_L = 0, v_loaded = 0, v_items = 0, v_qsel = 0;
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
    v_hs = rank * 2 + hsl;
    if (lane == 0) {
      ART_WATCH(wd, 1);
      while (atom_cas_cluster_acquire(board_at(v_hs, B_NACT), 0, kLock) != 0) { nsleep(64); ART_WATCH_POLL(wd, v_hs, my_gen); }
    }
    __syncwarp();
    if (lane == 0) {
      HomeInfo* hi = reinterpret_cast<HomeInfo*>(smem + sm.hinfo) + hsl;
      hi->done = static_cast<unsigned long long>(v_T + 1) << 32;   // high half: T + 1; low half: steps folded and flushed so far
      hi->group = v_group; hi->T = v_T; hi->gen = my_gen; hi->loaded = 0; hi->joined = 0u;
      asm volatile("st.relaxed.cluster.shared::cluster.s32 [%0], %1;" :: "r"(board_at(v_hs, B_NEXT)), "r"(0) : "memory");
      asm volatile("st.relaxed.cluster.shared::cluster.s32 [%0], %1;" :: "r"(board_at(v_hs, B_T)), "r"(v_T) : "memory");
      asm volatile("st.relaxed.cluster.shared::cluster.s32 [%0], %1;" :: "r"(board_at(v_hs, B_GROUP)), "r"(v_group) : "memory");
    }
    __syncwarp();
    if (lane == 0) {
      // open, one worker (this CTA); releases all of the above (before the start the cluster barrier does that)
      if (before_start) atom_add_cluster(board_at(v_hs, B_NACT), 1 - kLock);
      else atom_add_cluster_release(board_at(v_hs, B_NACT), 1 - kLock);
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
    int score = 0, e_next = 0, e_T = 0, e_nact = 0, e_group = -1;
    if (lane < 2 * CL) {
      e_next = ld_cluster_relaxed_s32(board_at(lane, B_NEXT)); e_T = ld_cluster_relaxed_s32(board_at(lane, B_T));
      e_nact = ld_cluster_relaxed_s32(board_at(lane, B_NACT)); e_group = ld_cluster_relaxed_s32(board_at(lane, B_GROUP));
      const int rem = (e_nact > 0 && e_group >= 0) ? e_T - e_next : 0;
      if (rem >= kMinJoin) score = (rem << 4) / (e_nact + 1) + 1;
    }
    int best = score, who = lane;
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) {
      const int ob = __shfl_xor_sync(0xffffffffu, best, m), ow = __shfl_xor_sync(0xffffffffu, who, m);
      if (ob > best || (ob == best && ow < who)) { best = ob; who = ow; }
    }
    if (best == 0) return false;
    int ok = 0, T2 = 0, grp = 0;
    if (lane == 0) {
      const int old = atom_add_cluster_acquire(board_at(who, B_NACT), 1);       // pin: the slot cannot be reopened under us
      T2 = ld_cluster_relaxed_s32(board_at(who, B_T)); grp = ld_cluster_relaxed_s32(board_at(who, B_GROUP));
      const int nx = ld_cluster_relaxed_s32(board_at(who, B_NEXT));
      ok = (old > 0 && grp >= 0 && nx < T2) ? 1 : 0;
      if (!ok) atom_add_cluster(board_at(who, B_NACT), -1);
    }
    ok = __shfl_sync(0xffffffffu, ok, 0);
    if (!ok) return true;                                  // lost a race: look again
    v_hs = who;
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
      v_hs = home * 2;
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
      const uint32_t a_next = board_at(v_hs, B_NEXT);
      // steps are claimed a chunk of `claim` consecutive steps at a time, one chunk ahead of the one being issued,
      // so the round trip to the board is never waited for
      const int K = pp.claim;
      int ch_t = 0, ch_left = 0, nx = 0;
      auto claim_chunk = [&]() {
        if (lane == 0) nx = atom_add_cluster(a_next, K) + 1;
      };
      auto next_step = [&]() -> int {
        if (ch_left == 0) { ch_t = __shfl_sync(0xffffffffu, nx, 0); ch_left = K; if (ch_t <= v_T) claim_chunk(); }
        --ch_left;
        return ch_t++;
      };
      auto resolve = [&](int t, bool& valid, unsigned long long& mask, int& page, int& ec) {
        valid = t <= v_T;
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
        wait_empty();
        if (lane == 0) {
          const uint32_t fb = bar(sm.full0 + stage);
          const uint32_t dst = sbase + sm.ring + stage * kStageBytes;
          items[it % kItemsRing].tcode = tA | (ecA << kItemShift);
          items[it % kItemsRing].meta = v_hs | (v_qsel << 5) | (ITEM_DATA << 6);
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
      if (v_items > 0) push_marker(ITEM_FLUSH, v_loaded, v_hs, static_cast<unsigned long long>(v_group));
      else leave_quietly();
      have = false;
    }
    push_marker(ITEM_END, 0, 0, 0ull);
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
          // one M128 MMA per k-step: tokens on lanes 0-63 (even items) or 64-127 (odd items), see art_decode_tc.cuh
          const uint32_t kt = sbase + sm.ring + st * kStageBytes - (i & 1) * kBoxBytes;
          const uint32_t dcol = tmem_S + q * kSCols1;
#pragma unroll
          for (int ks = 0; ks < 8; ++ks) {
            const uint32_t ka = kt + (ks >> 2) * kBoxBytes + (ks & 3) * 32;
            umma_bf16(dcol, dK | desc_addr(ka), dQ | desc_addr(qb + ks * 2 * kQLbo), kIdescS, ks > 0);
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
      const uint64_t dP = kDescNoSw | desc_strides(LBO_P, PBUF);   // rows 0-7 = hi, rows 8-15 = lo (art_decode_tc.cuh)
      int st = 0; uint32_t ph = 0;
      for (int i = 0;; ++i) {
        const int ps = i & (NP - 1);
        mbar_wait(bar(sm.pfull0 + st), ph);
        const int kind = item_kind(items[i % kItemsRing].meta);
        if (i >= NP) mbar_wait(bar(sm.pvfree0 + ps), ((i / NP) - 1) & 1);
        if (kind == ITEM_DATA) {
          tc_fence_after();
          const uint32_t vt = sbase + sm.ring + st * kStageBytes + 2 * kBoxBytes;
          const uint32_t pb = sbase + sm.pb + st * 2 * PBUF;
#pragma unroll
          for (int ks = 0; ks < 4; ++ks)
            umma_bf16(tmem_PV + ps * kUmmaN, dV | desc_addr(vt + ks * 2048),
                      dP | desc_addr(pb + ks * 2 * LBO_P), kIdescPV, ks > 0);
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
    // ===================================================== A4: block-local softmax, one token per thread, two warps per item
    const int q = warp - kWarpSoftmax0;                       // TMEM lane quadrant
    const int pair = q >> 1, half = q & 1;                    // the pair owns items i = pair (mod 2); this warp tokens 32 half + lane
    const int tok = half * 32 + lane;
    const uint32_t tq = static_cast<uint32_t>(q * 32) << 16;
    int st = pair % S;
    for (int i = pair;; i += 2) {
      const int sslot = i & (NS - 1);
      mbar_wait(bar(sm.sfull0 + sslot), (i / NS) & 1);
      const int kind = item_kind(items[i % kItemsRing].meta);
      if (kind == ITEM_END) {
        // the END item that owns a stage is the first of the run; only its pair hands it on to the P.V issuer
        if (item_kind(items[(i + kItemsRing - 1) % kItemsRing].meta) != ITEM_END || i == 0) mbar_arrive(bar(sm.pfull0 + st));
        break;
      }
      if (kind != ITEM_DATA) {                               // a marker: nothing to compute
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(sm.sfree0 + sslot));
        mbar_arrive(bar(sm.pfull0 + st));
        st += 2; while (st >= S) st -= S;
        continue;
      }
      tc_fence_after();
      float sv[G];
      tmem_ld<G>(tmem_S + sslot * kSCols1 + tq, sv);
      tmem_ld_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(sm.sfree0 + sslot));
      const unsigned long long vmask = items[i % kItemsRing].mask;
      const bool v0 = (vmask >> tok) & 1ull;
      float mb[G];
      int ec = 0;
      if constexpr (MT) ec = items[i % kItemsRing].tcode >> kItemShift;
#pragma unroll
      for (int h = 0; h < G; ++h) {
        bool vis = v0;                                        // masked tokens: weight 0 (R8); their K may be NaN
        if (MT && ec != 0) vis = vis && tok < ec - static_cast<int>((p.cuts >> (4 * h)) & 15u);   // R15: causal cut row by row
        sv[h] = vis ? sv[h] * p.scale_log2 : kNegInf;
        mb[h] = warp_max_f32(sv[h]);
      }
      {
        // block maximum over the two halves (shared memory + the pair's named barrier; double-buffered by item parity)
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
      uint8_t* pb0 = smem + sm.pb + st * 2 * PBUF + (half * 4 + (lane >> 3)) * LBO_P + (lane & 7) * 2;
      float ls[G];
#pragma unroll
      for (int h = 0; h < G; ++h) {
        const float p0 = (sv[h] != kNegInf) ? fast_exp2(sv[h] - mb[h]) : 0.f;
        const __nv_bfloat16 h0 = __float2bfloat16_rn(p0);
        const __nv_bfloat16 l0 = __float2bfloat16_rn(p0 - __bfloat162float(h0));
        *reinterpret_cast<__nv_bfloat16*>(pb0 + h * 16) = h0;
        *reinterpret_cast<__nv_bfloat16*>(pb0 + h * 16 + PBUF) = l0;
        ls[h] = __bfloat162float(h0) + __bfloat162float(l0);
      }
      if (vmask != ~0ull && !v0) {                            // masked V rows may hold NaN: 0 * NaN would poison P~V
        uint4* vr = reinterpret_cast<uint4*>(smem + sm.ring + st * kStageBytes + 2 * kBoxBytes);
#pragma unroll
        for (int c = 0; c < 8; ++c) { vr[tok * 8 + c] = make_uint4(0u, 0u, 0u, 0u); vr[tok * 8 + c + kBoxBytes / 16] = make_uint4(0u, 0u, 0u, 0u); }
      }
      Reduce32<G, 16>::run(ls, lane);
      {
        const int hh = head_of_lane32<G>(lane);
        float mine = mb[0];
#pragma unroll
        for (int h = 1; h < G; ++h) mine = (hh == h) ? mb[h] : mine;
        float* slot = slots + (i & (kIterSlots - 1)) * 3 * G;
        if ((lane & (32 / G - 1)) == 0) { if (half == 0) slot[hh] = mine; slot[(1 + half) * G + hh] = ls[0]; }
      }
      fence_proxy_async();
      mbar_arrive(bar(sm.pfull0 + st));
      st += 2; while (st >= S) st -= S;
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
      float pv[G], pvl[G];
      tmem_ld<G>(tmem_PV + tlane + (i & (NP - 1)) * kUmmaN, pv);
      tmem_ld<G>(tmem_PV + tlane + (i & (NP - 1)) * kUmmaN + 8, pvl);
      tmem_ld_wait();
#pragma unroll
      for (int h = 0; h < G; ++h) pv[h] += pvl[h];            // hi + lo halves of p
      const float* sl = slots + (i & (kIterSlots - 1)) * 3 * G;
#pragma unroll
      for (int h = 0; h < G; ++h) {
        const float mr = sl[h];
        if (mr != kNegInf) {                                  // a block with no valid token changes nothing
          const float mn = fmaxf(m_tot[h], mr);
          const float a = fast_exp2(m_tot[h] - mn), bb = fast_exp2(mr - mn);
          acc[h] = fmaf(a, acc[h], bb * pv[h]);
          l_tot[h] = fmaf(a, l_tot[h], bb * (sl[G + h] + sl[2 * G + h]));
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
      if (d == 0) p.stop_block[group] = T;
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
      if (warp == kWarpFold0 && lane == 0) atom_add_cluster(board_at(hs, B_NACT), -1);
      reset_state();
    };

    for (int i = 0;; ++i) {
      mbar_wait(bar(sm.pvfull0 + (i & (NP - 1))), (i / NP) & 1);
      const int meta = items[i % kItemsRing].meta;
      const int kind = item_kind(meta);
      if (kind == ITEM_DATA) { fold(i); continue; }
      if (kind == ITEM_END) break;
      flush(items[i % kItemsRing].tcode, meta, items[i % kItemsRing].mask);
      release_pv(i);
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
