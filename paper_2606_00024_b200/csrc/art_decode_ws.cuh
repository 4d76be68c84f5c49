// ART decode attention, bf16 / head_dim 128, DYNAMICALLY SCHEDULED tcgen05 kernel ("work-stealing" grid).
//
// art_decode_tc.cuh binds a query group to a fixed cluster of CTAs; once ART has stopped a group its SMs
// idle while the groups that run long keep only their own few CTAs (variant R of configs[1]: 49 % of the
// blocks skipped, 3 % faster).  Here the grid is PERSISTENT (one or two CTAs per SM) and nothing is bound:
//
//   * every group has a control block in global memory (L2): a claim counter `next_step`, the progress word
//     `ctrl` (last scanned step, or -t* once Algorithm 1 has fired), a worker count, a completion word;
//   * a CTA's PRODUCER warp joins a group that has unclaimed steps, claims traversal steps t one at a time
//     (atomicAdd, one claim ahead), resolves block -> page (A1) and issues the TMA loads (A2); when the group
//     has no step left it moves to the group with the most remaining work per worker;
//   * the item then runs through the same warp-specialised pipeline as in art_decode_tc.cuh (S-MMA, softmax,
//     PV-MMA, block-local results waiting unfolded in tensor memory);
//   * the FOLD warps publish the step summary (m_t, l_t, probe of P~V_t) into the group's mailbox in global
//     memory and merge P~V_t into the CTA's partial state only once step t <= t* is decided; when the CTA
//     leaves the group they flush the partial state to a per-group slot;
//   * every group is OPENED by the scan warp of some resident CTA, which then replays Algorithm 1
//      sequentially over the mailbox (art_scan.cuh), staging summaries into shared
//     memory with cp.async so that the L2 latency overlaps the arithmetic;
//   * whoever brings the group's completion word to "folded steps == t*" (the last flusher, or the scan
//     warp) combines the partial states and writes out / stop_block (A8/A9).
//
// Steps beyond t* are never folded, so the result is the sequential algorithm's whatever the schedule was.
// Deadlock freedom: a worker only joins groups that are open (their scanner is a RESIDENT CTA's warp) and
// leaves a group only when it is exhausted, which is permanent; see DESIGN.md "Scheduling".
#pragma once
#include "art_decode_tc.cuh"

namespace art {
namespace ws {

using namespace tc;

constexpr int kItemRing = 16;                // per-item info ring; >= kPVSlots + max stages
static_assert(kItemRing >= kPVSlots + kMaxStages, "item ring too short");

struct ItemInfo { int group, t, marker, pad; };   // marker = 1: end of a visit (no step, flush the partial state)
template <int G> struct IterSlotW { float mref[G], lsum[G]; };   // what softmax hands to fold for one block

// ---- global workspace: [header 64 B][ctl 64 B x groups][mailbox pay_bytes x M x groups] (zeroed per call)
// One step summary in the mailbox = (2 + PW) G floats: (m_t, l_t) pairs of the G heads, then PW probe values of
// head 0, of head 1, ...: the scan lane (head h, sub) reads its pair and its PW / LPH probe values as vectors.
//                        [partials part_floats x 4 B x Wmax x groups]
// Mailbox words are SELF-VALIDATING: the lowest mantissa bit of every float of a step summary carries the
// parity of the slot's generation ((t-1)/M + 1) & 1, so the reader needs neither a flag nor a fence: a word is
// either still the previous generation's (or the zero fill) or the final value (4-byte stores are atomic).
// Cost: 2^-23 relative on the probe values, far inside the criterion's error budget.
constexpr int kCtlInts = 16;
enum { C_NEXT = 0,      // steps claimed so far
       C_CTRL = 1,      // >= 0: steps 1..ctrl scanned, none fired;  < 0: fired, t* = -ctrl
       C_WORKERS = 2,   // CTAs currently working on the group
       C_OPENT = 3,     // 0: not opened yet; else T + 1
       C_NSLOTS = 4,    // partial-state slots handed out
       C_DONE = 6 };    // u64: low = steps folded and flushed, high = t_final + 1 once the scan has finished
enum { H_NEXT_GROUP = 0, H_OPENED = 1 };

struct WsView {
  uint8_t* base;
  uint32_t M, mshift, Wmax, pay_bytes, part_floats;
  uint64_t off_ctl, off_pay, off_part, off_trace;
};

struct WsLayout { WsView v; size_t total, zero_bytes; };
// one step summary, padded to the 16-byte granularity of bulk copies
__host__ __device__ constexpr int probe_off_of(int G) { return (2 * G + 3) & ~3; }   // floats: (m, l) pairs, padded to 16 B
__host__ __device__ constexpr uint32_t pay_bytes_of(int G, int PW) { return (static_cast<uint32_t>((probe_off_of(G) + PW * G) * 4) + 15u) & ~15u; }

#ifdef ART_TRACE
#define TRACE_INIT(tr, role) Tracer tr; tr.init(w.base, w.off_trace, role, reinterpret_cast<volatile int*>(smem + sm.misc + 16))
#define TRACE(tr, code, a, b) tr.ev(code, a, b)
#else
#define TRACE_INIT(tr, role)
#define TRACE(tr, code, a, b)
#endif

// Workers per group are capped where more of them stop paying (the scan of one group absorbs ~8 blocks/us)
// and so that the partial-state slots stay small when there are many groups.
inline WsLayout make_ws_layout(int groups, int G, int PW, bool art) {
  WsLayout l; WsView& v = l.v;
  auto up = [](size_t x) { return (x + 255) & ~static_cast<size_t>(255); };
  const int fair = (3 * 296 + groups - 1) / (groups > 0 ? groups : 1);
  const int cap = art ? 12 : 32;
  v.Wmax = static_cast<uint32_t>(fair < 2 ? 2 : (fair > cap ? cap : fair));
  v.M = groups <= 296 ? 64u : 16u;
  v.mshift = groups <= 296 ? 6u : 4u;
  v.pay_bytes = pay_bytes_of(G, PW);
  v.part_floats = static_cast<uint32_t>(G * (kD + 2));
  v.base = nullptr;
  size_t off = 64;
  v.off_ctl = off; off += static_cast<size_t>(groups) * kCtlInts * 4;
  off = up(off);
  v.off_pay = off; off = up(off + (art ? static_cast<size_t>(groups) * v.M * v.pay_bytes : 0));
  v.off_trace = off;
#ifdef ART_TRACE
  off = up(off + 256 + static_cast<size_t>(kTraceCtas) * kTraceRoles * kTraceEvents * 16 + 1024 * 16);   // + per-CTA (start, end)
#endif
  l.zero_bytes = off;
  v.off_part = off; off = up(off + static_cast<size_t>(groups) * v.Wmax * v.part_floats * 4);
  l.total = off;
  return l;
}

struct SmemMapW {
  uint32_t qb, pb, slots, items, sinfo, stg, bars, misc, ring, total;
  uint32_t full0, empty0, pfull0, sfull0, sfree0, pvfull0, pvfree0, done0, stg0, nbars;
};
__host__ __device__ inline SmemMapW make_smem_map_w(int G, int PW, int stages, int ms, bool art) {
  SmemMapW m;
  uint32_t off = 0;
  m.qb = off; off += kQBytes;
  m.pb = off; off += static_cast<uint32_t>(stages) * 2u * p_buf_bytes(G);
  m.slots = off; off += kIterSlots * static_cast<uint32_t>(G) * 8u;        // IterSlotW<G>
  m.items = off; off += kItemRing * static_cast<uint32_t>(sizeof(ItemInfo));
  m.sinfo = off; off += static_cast<uint32_t>(stages) * 8u;
  off = (off + 15u) & ~15u;
  m.stg = off; off += art ? static_cast<uint32_t>(ms) * pay_bytes_of(G, PW) : 0u;   // staged step summaries (cp.async)
  off = (off + 15u) & ~15u;
  m.bars = off;
  uint32_t n = 0;
  m.full0 = n; n += stages; m.empty0 = n; n += stages; m.pfull0 = n; n += stages;
  m.sfull0 = n; n += kSSlots; m.sfree0 = n; n += kSSlots;
  m.pvfull0 = n; n += kPVSlots; m.pvfree0 = n; n += kPVSlots;
  m.done0 = n; n += 2;
  m.stg0 = n; n += art ? 2 : 0;
  m.nbars = n;
  off += n * 8u;
  m.misc = off; off += 64u;              // tmem_ptr, n_total, fold broadcast words
  off = (off + 1023u) & ~1023u;
  if (off < static_cast<uint32_t>(kFront)) off = kFront;
  m.ring = off; off += static_cast<uint32_t>(stages) * kStageBytes;
  m.total = off;
  return m;
}
constexpr uint32_t kWTmemPtr = 0, kWNTotal = 4, kWSlot = 8, kWCompleter = 12;

// ----------------------------------------------------------------------------- global-memory helpers

__device__ __forceinline__ int ld_relaxed_gpu(const int* ptr) {
  int v; asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(ptr) : "memory"); return v;
}
__device__ __forceinline__ void st_relaxed_gpu(int* ptr, int v) {
  asm volatile("st.relaxed.gpu.global.s32 [%0], %1;" :: "l"(ptr), "r"(v) : "memory");
}
__device__ __forceinline__ void st_release_gpu(int* ptr, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" :: "l"(ptr), "r"(v) : "memory");
}
__device__ __forceinline__ void red_release_add(int* ptr, int v) {
  asm volatile("red.release.gpu.global.add.s32 [%0], %1;" :: "l"(ptr), "r"(v) : "memory");
}
__device__ __forceinline__ void fence_acq_rel_gpu() { asm volatile("fence.acq_rel.gpu;" ::: "memory"); }
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() {
  asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
}
// mailbox word = value with the generation parity in its lowest mantissa bit
__device__ __forceinline__ float tag_word(float x, uint32_t par) {
  return __uint_as_float((__float_as_uint(x) & ~1u) | par);
}
__device__ __forceinline__ uint32_t step_parity(int t, int mshift) {
  return static_cast<uint32_t>((((t - 1) >> mshift) + 1) & 1);
}
// shared-memory loads of the staged summaries: volatile + memory clobber, they must stay behind the cp.async wait
__device__ __forceinline__ float2 lds_v2(uint32_t addr) {
  float2 r; asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(r.x), "=f"(r.y) : "r"(addr) : "memory"); return r;
}
template <int N> __device__ __forceinline__ void lds_vec(uint32_t addr, float (&v)[N]) {
  if constexpr (N % 4 == 0) {
#pragma unroll
    for (int i = 0; i < N; i += 4)
      asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v[i]), "=f"(v[i + 1]), "=f"(v[i + 2]), "=f"(v[i + 3]) : "r"(addr + i * 4) : "memory");
  } else if constexpr (N == 2) {
    asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(v[0]), "=f"(v[1]) : "r"(addr) : "memory");
  } else {
#pragma unroll
    for (int i = 0; i < N; ++i) asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v[i]) : "r"(addr + i * 4) : "memory");
  }
}
constexpr float kEmptyMax = -1.0e30f;       // "no valid token" in the mailbox (-inf has no spare mantissa bit)
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" :: "r"(id), "r"(nthreads) : "memory");
}
template <int G> __device__ __forceinline__ void st_global_vec(float* dst, const float* v) {
  if constexpr (G == 1) { *dst = v[0]; }
  else if constexpr (G == 2) { *reinterpret_cast<float2*>(dst) = make_float2(v[0], v[1]); }
  else {
#pragma unroll
    for (int i = 0; i < G; i += 4) *reinterpret_cast<float4*>(dst + i) = make_float4(v[i], v[i + 1], v[i + 2], v[i + 3]);
  }
}

// A8 / A9: flash-decoding combine of the partial states flushed for `group`; called by the thread set that
// completed the group (all of its flushes are visible: fence after the completing atomic).
template <int G>
__device__ __forceinline__ void combine_group(const Params& p, const WsView& w, int group, int tid, int nthreads) {
  const int* c = reinterpret_cast<const int*>(w.base + w.off_ctl) + group * kCtlInts;
  int ns = __ldcg(c + C_NSLOTS);
  ns = ns > static_cast<int>(w.Wmax) ? static_cast<int>(w.Wmax) : ns;
  const float* part = reinterpret_cast<const float*>(w.base + w.off_part) + static_cast<size_t>(group) * w.Wmax * w.part_floats;
  const int b = group / p.Hkv, g = group % p.Hkv;
  float* out = p.out + (static_cast<int64_t>(b) * p.Hq + g * p.Gr) * kD;
  for (int o = tid; o < p.Gr * kD; o += nthreads) {
    const int h = o / kD;
    float mx = kNegInf;
#pragma unroll 4
    for (int s = 0; s < ns; ++s) mx = fmaxf(mx, __ldcg(part + s * w.part_floats + G * kD + h));
    float a = 0.f, l = 0.f;
#pragma unroll 4                                               // four slots' loads in flight together
    for (int s = 0; s < ns; ++s) {
      const float* ps = part + s * w.part_floats;
      const float mc = __ldcg(ps + G * kD + h);
      const float f = (mc == kNegInf) ? 0.f : fast_exp2(mc - mx);
      a = fmaf(f, __ldcg(ps + o), a);
      l = fmaf(f, __ldcg(ps + G * kD + G + h), l);
    }
    out[o] = (l > 0.f) ? a / l : 0.f;                         // Alg. 1 l.18
  }
}

}  // namespace ws
}  // namespace art
