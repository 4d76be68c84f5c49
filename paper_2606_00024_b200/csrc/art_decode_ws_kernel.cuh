// The dynamically scheduled kernel itself; data structures and helpers in art_decode_ws.cuh.
#pragma once
#include "art_decode_ws.cuh"

namespace art {
namespace ws {

// MODE 0: ART off.  MODE 1: ART on, probe = 32 coordinates k*(d/32).  MODE 2: ART on, probe = all d.
template <int G, int MODE>
__global__ void __launch_bounds__(kThreads, (MODE == 2) ? 1 : 2)
art_decode_ws_kernel(const Params p, const WsView w, const __grid_constant__ CUtensorMap tmK,
                     const __grid_constant__ CUtensorMap tmV) {
  constexpr bool ART = MODE != 0;
  constexpr int PW = (MODE == 2) ? kD : 32;
  constexpr int NP = kPVSlots, NS = kSSlots;
  constexpr int LBO_P = p_lbo(G), PBUF = p_buf_bytes(G);
  constexpr uint32_t kPayBytes = pay_bytes_of(G, PW);         // one step summary: (2 + PW) G floats, padded to 16 B
  constexpr int kPayFloats = static_cast<int>(kPayBytes / 4);
  constexpr int kProbeOff = probe_off_of(G);

  extern __shared__ __align__(1024) uint8_t smem[];
  const int S = p.stages, MS = p.mbox_slots;
  const SmemMapW sm = make_smem_map_w(G, PW, S, MS, ART);
  const uint32_t sbase = smem_u32(smem);
  if ((sbase & 1023u) != 0u) __trap();
  const uint32_t bars = sbase + sm.bars;
  auto bar = [&](uint32_t idx) { return bars + idx * 8u; };
  const uint32_t a_tmem = sbase + sm.misc + kWTmemPtr, a_ntotal = sbase + sm.misc + kWNTotal;
  const uint32_t a_slot = sbase + sm.misc + kWSlot, a_completer = sbase + sm.misc + kWCompleter;
  IterSlotW<G>* slots = reinterpret_cast<IterSlotW<G>*>(smem + sm.slots);
  ItemInfo* items = reinterpret_cast<ItemInfo*>(smem + sm.items);
  unsigned long long* sinfo = reinterpret_cast<unsigned long long*>(smem + sm.sinfo);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int groups = p.batch * p.Hkv;
  int* hdr = reinterpret_cast<int*>(w.base);
  int* ctl_base = reinterpret_cast<int*>(w.base + w.off_ctl);
  float* pay_base = reinterpret_cast<float*>(w.base + w.off_pay);
  float* part_base = reinterpret_cast<float*>(w.base + w.off_part);
  auto ctl = [&](int grp) { return ctl_base + grp * kCtlInts; };
  const int M = static_cast<int>(w.M), Wmax = static_cast<int>(w.Wmax);

#ifdef ART_TRACE
  unsigned long long* cta_times = reinterpret_cast<unsigned long long*>(w.base + w.off_trace + 256 + static_cast<size_t>(kTraceCtas) * kTraceRoles * kTraceEvents * 16) + 2 * blockIdx.x;
  if (tid == 0) cta_times[0] = trace_now();
#endif
  // ---- one-time setup
  if (tid == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(bar(sm.full0 + s), 1); mbar_init(bar(sm.empty0 + s), 1); mbar_init(bar(sm.pfull0 + s), 32); }
    for (int s = 0; s < NS; ++s) { mbar_init(bar(sm.sfull0 + s), 1); mbar_init(bar(sm.sfree0 + s), 1); }
    for (int s = 0; s < NP; ++s) { mbar_init(bar(sm.pvfull0 + s), 1); mbar_init(bar(sm.pvfree0 + s), 4); }
    mbar_init(bar(sm.done0), 1); mbar_init(bar(sm.done0 + 1), 1);
    if (ART) { mbar_init(bar(sm.stg0), 1); mbar_init(bar(sm.stg0 + 1), 1); }
    st_volatile_s32(a_ntotal, 0x7fffffff);
    st_volatile_s32(sbase + sm.misc + 16, 0);
    fence_mbar_init();
  }
  if (warp == kWarpMmaPV) tmem_alloc(a_tmem, kTmemCols);
  {
    uint4* qz = reinterpret_cast<uint4*>(smem + sm.qb);        // Q^T rows >= G stay zero for good
    for (int idx = tid; idx < kQBytes / 16; idx += kThreads) qz[idx] = make_uint4(0u, 0u, 0u, 0u);
    uint4* pz = reinterpret_cast<uint4*>(smem + sm.pb);        // P^T rows are read before they are first written
    for (int idx = tid; idx < S * 2 * PBUF / 16; idx += kThreads) pz[idx] = make_uint4(0u, 0u, 0u, 0u);
  }
  fence_proxy_async();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = static_cast<uint32_t>(ld_volatile_s32(a_tmem));
  const uint32_t tmem_S = tmem_base, tmem_PV = tmem_base + NS * kSCols;

  // waits that must end when the producer has issued its last item
  auto wait_or_end = [&](uint32_t baddr, uint32_t parity, int i) -> bool {
    while (!mbar_try_wait(baddr, parity)) { if (i >= ld_volatile_s32(a_ntotal)) return false; }
    return true;
  };

  if (warp == kWarpProducer) {
    // ===================================================== scheduling + A1 + A2
    int it = 0, stage = 0; uint32_t ph = 0;
    int last_marker = -1, visit = 0;
    TRACE_INIT(trc, 0);
    bool static_phase = true;
    auto issue = [&](int grp, int t, int marker, unsigned long long mask, int c1, int c2) {
      if (it >= S) mbar_wait(bar(sm.empty0 + stage), ph ^ 1u);
      if (lane == 0) {
        TRACE(trc, 1, grp, t);
        ItemInfo& ii = items[it & (kItemRing - 1)];
        ii.group = grp; ii.t = t; ii.marker = marker;
        sinfo[stage] = mask;
        const uint32_t fb = bar(sm.full0 + stage);
        const uint32_t dst = sbase + sm.ring + stage * kStageBytes;
        if (mask == 0ull) {
          mbar_arrive(fb);                                   // an all-masked step or a marker: nothing to load
        } else {
          mbar_arrive_expect_tx(fb, kStageBytes);
          tma_load_box(dst, &tmK, 0, c1, c2, fb);
          tma_load_box(dst + kBoxBytes, &tmK, 64, c1, c2, fb);
          tma_load_box(dst + 2 * kBoxBytes, &tmV, 0, c1, c2, fb);
          tma_load_box(dst + 3 * kBoxBytes, &tmV, 64, c1, c2, fb);
        }
      }
      ++it;
      if (++stage == S) { stage = 0; ph ^= 1u; }
    };
    // a group is worth joining if it is open, not fired, has unclaimed steps and room for a worker
    auto remaining = [&](const int4 v) -> int {
      if (v.w == 0 || v.y < 0 || v.z >= Wmax) return 0;
      const int r = (v.w - 1) - v.x;
      return r > 0 ? r : 0;
    };
    while (true) {
      // ---- pick a group: this CTA's static list first (group = blockIdx + k * gridDim), then the most
      //      remaining work per worker among all groups
      int gsel = -3;
      if (static_phase) {
        // few groups: CTA x starts on group x mod groups (an even spread), later picks are dynamic
        const int gs = (groups >= static_cast<int>(gridDim.x)) ? static_cast<int>(blockIdx.x) + visit * static_cast<int>(gridDim.x)
                                                               : (visit == 0 ? static_cast<int>(blockIdx.x) % groups : groups);
        if (gs >= groups) static_phase = false;
        else {
          int r = 0;
          for (int tries = 0; tries < 32 && r == 0; ++tries) {     // at start-up the opener may be a moment behind
            const int4 v = __ldcg(reinterpret_cast<const int4*>(ctl(gs)));
            r = remaining(v);
            if (v.w != 0) break;
            __nanosleep(100);
          }
          ++visit;
          if (r > 0) gsel = gs;
        }
      }
      if (gsel == -3) {
        unsigned long long best = 0ull;
        bool unopened = false;
#pragma unroll 4
        for (int base = 0; base < groups; base += 32) {
          const int gi = base + lane;
          if (gi < groups) {
            const int4 v = __ldcg(reinterpret_cast<const int4*>(ctl(gi)));
            unopened |= (v.w == 0);
            const int r = remaining(v);
            if (r > 0) {
              uint32_t hsh = (static_cast<uint32_t>(gi) * 2654435761u) ^ (blockIdx.x * 40503u + static_cast<uint32_t>(it) * 9973u);
              hsh ^= hsh >> 15; hsh *= 2246822519u; hsh ^= hsh >> 13;
              const float noise = 0.75f + 0.5f * static_cast<float>(hsh & 0xffffu) * (1.0f / 65536.0f);
              const float score = static_cast<float>(r) / static_cast<float>(v.z + 1) * noise;
              const unsigned long long key = (static_cast<unsigned long long>(__float_as_uint(score)) << 32) | static_cast<uint32_t>(gi);
              best = key > best ? key : best;
            }
          }
        }
#pragma unroll
        for (int m = 16; m >= 1; m >>= 1) {
          const unsigned long long o = __shfl_xor_sync(0xffffffffu, best, m);
          best = o > best ? o : best;
        }
        unopened = __any_sync(0xffffffffu, unopened);
        if (best != 0ull) gsel = static_cast<int>(best & 0xffffffffull);
        else if (!unopened && __ldcg(hdr + H_OPENED) >= groups) break;   // nothing left that needs this CTA
        else { __nanosleep(300); continue; }
      }
      // ---- admission: at most Wmax workers per group (never over-counted: compare-and-swap)
      int ok = 0;
      if (lane == 0) {
        int* wk = ctl(gsel) + C_WORKERS;
        int cur = ld_relaxed_gpu(wk);
        while (cur < Wmax) {
          const int old = atomicCAS(wk, cur, cur + 1);
          if (old == cur) { ok = 1; break; }
          cur = old;
        }
      }
      ok = __shfl_sync(0xffffffffu, ok, 0);
      if (!ok) continue;
      if (lane == 0) TRACE(trc, 2, gsel, ok);

      const int b = gsel / p.Hkv, g = gsel % p.Hkv;
      const int L = p.seq_lens[b];
      const Trav tr = make_trav(p, b, g, L);
      const int Tn = tr.T;
      int* c_next = ctl(gsel) + C_NEXT;
      int* c_ctrl = ctl(gsel) + C_CTRL;
      // The claim -> page lookup -> TMA chain is two dependent L2 round trips; it is software-pipelined so that
      // neither sits between "stage free" and "TMA issued": item A is resolved (its page lookup in flight since
      // the previous iteration), item B is claimed, and the claim for the item after B is issued now.
      int tB = 0, cB = 0;                                      // lane 0: claim B (possibly still in flight)
      if (lane == 0) { tB = atomicAdd(c_next, 1) + 1; cB = ld_relaxed_gpu(c_ctrl); }
      // Q^T may be overwritten once every S-MMA of the previous visit has retired: its marker's stage is empty
      if (last_marker >= 0 && it < last_marker + S)
        mbar_wait(bar(sm.empty0 + last_marker % S), static_cast<uint32_t>((last_marker / S) & 1));
      {
        const uint4* qp = reinterpret_cast<const uint4*>(reinterpret_cast<const __nv_bfloat16*>(p.q) +
                                                         (static_cast<int64_t>(b) * p.Hq + g * p.Gr) * kD);
        for (int idx = lane; idx < p.Gr * 16; idx += 32) {        // 16-byte chunk (row, 8 d) -> K-major core matrices
          const int row = idx >> 4, dc = idx & 15;
          *reinterpret_cast<uint4*>(smem + sm.qb + dc * kQLbo + row * 16) = qp[row * 16 + dc];
        }
        fence_proxy_async();
        __syncwarp();
      }
      // resolve a claimed step: validity, token mask, page (the load is left in flight)
      auto resolve = [&](int t, int c, bool& valid, unsigned long long& mask, int& page) {
        valid = !(t > Tn || (c < 0 && t > -c));                // exhausted, or beyond t* (A7: stop prefetching)
        mask = 0ull; page = 0;
        if (valid) {
          const int blk = trav_block(tr, t);
          mask = block_mask(p, L, blk);
          if (mask) page = p.block_table[static_cast<int64_t>(b) * p.max_blocks + blk];
        }
      };
      int tA_ = __shfl_sync(0xffffffffu, tB, 0), cA_ = __shfl_sync(0xffffffffu, cB, 0);
      bool validA; unsigned long long maskA; int pageA;
      resolve(tA_, cA_, validA, maskA, pageA);
      if (lane == 0) { tB = atomicAdd(c_next, 1) + 1; cB = ld_relaxed_gpu(c_ctrl); }
      int n_items = 0, loaded = 0;
      while (validA) {
        // B becomes known: start its page lookup, and claim the step after it
        const int tN = __shfl_sync(0xffffffffu, tB, 0), cN = __shfl_sync(0xffffffffu, cB, 0);
        bool validB; unsigned long long maskB; int pageB;
        resolve(tN, cN, validB, maskB, pageB);
        if (validB && lane == 0) { tB = atomicAdd(c_next, 1) + 1; cB = ld_relaxed_gpu(c_ctrl); }
        int c1 = 0, c2 = 0;
        if (maskA) {
          if (p.layout == ART_LAYOUT_HND) { c1 = 0; c2 = pageA * p.Hkv + g; }
          else { c1 = g; c2 = pageA * kBlockTokens; }
        }
        issue(gsel, tA_, 0, maskA, c1, c2);
        loaded += maskA != 0ull;
        ++n_items;
        tA_ = tN; validA = validB; maskA = maskB; pageA = pageB;
      }
      if (n_items > 0) { issue(gsel, 0, 1, 0ull, 0, 0); last_marker = it - 1; }
      if (lane == 0) {
        atomicSub(ctl(gsel) + C_WORKERS, 1);
        if (p.blocks_loaded && loaded) atomicAdd(p.blocks_loaded + gsel, loaded);
      }
    }
    if (lane == 0) { TRACE(trc, 3, it, 0); st_volatile_s32(a_ntotal, it); }
    // drain: tensor copies still in flight must land before the CTA exits (H5)
    for (int j = max(0, it - S); j < it; ++j) mbar_wait(bar(sm.full0 + j % S), (j / S) & 1);
  } else if (warp == kWarpMmaS) {
    // ===================================================== A3: S = K_t Q^T
    if (lane == 0) {
      const uint64_t dK = kDescSw128 | desc_strides(16, 1024);
      const uint64_t dQ = kDescNoSw | desc_strides(kQLbo, kQSbo);
      const uint32_t qb = sbase + sm.qb;
      int st = 0; uint32_t ph = 0;
      for (int i = 0;; ++i) {
        const int q = i & (NS - 1);
        if (!wait_or_end(bar(sm.full0 + st), ph, i)) break;
        if (i >= NS && !wait_or_end(bar(sm.sfree0 + q), ((i / NS) - 1) & 1, i)) break;
        tc_fence_after();
        const uint32_t kt = sbase + sm.ring + st * kStageBytes - q * 4096;
        const uint32_t dcol = tmem_S + q * kSCols;
#pragma unroll
        for (int ks = 0; ks < 8; ++ks) {
          const uint32_t ka = kt + (ks >> 2) * kBoxBytes + (ks & 3) * 32;
          const uint64_t bq = dQ | desc_addr(qb + ks * 2 * kQLbo);
          umma_bf16(dcol, dK | desc_addr(ka), bq, kIdescS, ks > 0);
          umma_bf16(dcol + kUmmaN, dK | desc_addr(ka + 4096), bq, kIdescS, ks > 0);
        }
        umma_commit(bar(sm.sfull0 + q));
        if (++st == S) { st = 0; ph ^= 1u; }
      }
      umma_commit(bar(sm.done0));
      mbar_wait(bar(sm.done0), 0);
    }
  } else if (warp == kWarpMmaPV) {
    // ===================================================== A5: P~V_t = V_t^T P^T
    if (lane == 0) {
      const uint64_t dV = kDescSw128 | desc_strides(kBoxBytes, 1024);
      const uint64_t dP = kDescNoSw | desc_strides(LBO_P, 128);
      int st = 0; uint32_t ph = 0;
      for (int i = 0;; ++i) {
        const int ps = i & (NP - 1);
        if (!wait_or_end(bar(sm.pfull0 + st), ph, i)) break;
        if (i >= NP && !wait_or_end(bar(sm.pvfree0 + ps), ((i / NP) - 1) & 1, i)) break;
        tc_fence_after();
        const uint32_t vt = sbase + sm.ring + st * kStageBytes + 2 * kBoxBytes;
        const uint32_t pb = sbase + sm.pb + st * 2 * PBUF;
#pragma unroll
        for (int part = 0; part < 2; ++part)
#pragma unroll
          for (int ks = 0; ks < 4; ++ks)
            umma_bf16(tmem_PV + ps * kUmmaN, dV | desc_addr(vt + ks * 2048),
                      dP | desc_addr(pb + part * PBUF + ks * 2 * LBO_P), kIdescPV, (part | ks) > 0);
        umma_commit(bar(sm.empty0 + st));
        umma_commit(bar(sm.pvfull0 + ps));
        if (++st == S) { st = 0; ph ^= 1u; }
      }
      umma_commit(bar(sm.done0 + 1));
      mbar_wait(bar(sm.done0 + 1), 0);
    }
  } else if (warp >= kWarpSoftmax0 && warp < kWarpSoftmax0 + 4) {
    // ===================================================== A4: block-local softmax (as in art_decode_tc.cuh)
    const int q = warp - kWarpSoftmax0;
    const uint32_t taddr = tmem_S + q * kSCols + (static_cast<uint32_t>(q * 32) << 16);
    int st = q % S;
    for (int i = q;; i += NS) {
      if (!wait_or_end(bar(sm.sfull0 + q), (i / NS) & 1, i)) break;
      tc_fence_after();
      float s0[G], s1[G];
      tmem_ld<G>(taddr, s0);
      tmem_ld<G>(taddr + kUmmaN, s1);
      tmem_ld_wait();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(sm.sfree0 + q));
      const unsigned long long vmask = sinfo[st];
      const bool v0 = (vmask >> lane) & 1ull, v1 = (vmask >> (lane + 32)) & 1ull;
      float mb[G];
#pragma unroll
      for (int h = 0; h < G; ++h) {
        s0[h] = v0 ? s0[h] * p.scale_log2 : kNegInf;
        s1[h] = v1 ? s1[h] * p.scale_log2 : kNegInf;
        mb[h] = warp_max_f32(fmaxf(s0[h], s1[h]));
      }
      uint8_t* pb0 = smem + sm.pb + st * 2 * PBUF + (lane >> 3) * LBO_P + (lane & 7) * 2;
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
        IterSlotW<G>& slot = slots[i & (kIterSlots - 1)];
        if ((lane & (32 / G - 1)) == 0) { slot.mref[hh] = mine; slot.lsum[hh] = ls[0]; }
      }
      fence_proxy_async();
      mbar_arrive(bar(sm.pfull0 + st));
      st += NS; while (st >= S) st -= S;
    }
  }
  else if (warp < kWarpFold0 + 4) {
    // ===================================================== A5 / A6: publish step summaries, merge P~V_t, flush
    const int fq = warp & 3;
    const int d = fq * 32 + lane;                             // output coordinate == TMEM lane
    const uint32_t tlane = static_cast<uint32_t>(fq * 32) << 16;
    float acc[G], m_tot[G], l_tot[G];
#pragma unroll
    for (int h = 0; h < G; ++h) { acc[h] = 0.f; m_tot[h] = kNegInf; l_tot[h] = 0.f; }
    int n_folded = 0;                                         // steps merged during the current visit
    TRACE_INIT(trf, 1);
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
      const IterSlotW<G>& sl = slots[i & (kIterSlots - 1)];
#pragma unroll
      for (int h = 0; h < G; ++h) {
        const float mr = sl.mref[h];
        if (mr != kNegInf) {                                  // a block with no valid token changes nothing (R8)
          const float mn = fmaxf(m_tot[h], mr);
          const float a = fast_exp2(m_tot[h] - mn), bb = fast_exp2(mr - mn);
          acc[h] = fmaf(a, acc[h], bb * pv[h]);
          l_tot[h] = fmaf(a, l_tot[h], bb * sl.lsum[h]);
          m_tot[h] = mn;
        }
      }
      release_pv(i);
      ++n_folded;
      if (tid == 0) TRACE(trf, 5, i, items[i & (kItemRing - 1)].t);
    };
    // End of a visit (all four fold warps arrive here with the same n_folded): hand the partial state to the
    // group; whoever completes the group combines (A8 / A9).
    auto flush = [&](int grp) {
      if (n_folded > 0) {
        int* cg = ctl(grp);
        if (tid == 0) st_volatile_s32(a_slot, atomicAdd(cg + C_NSLOTS, 1));
        named_bar_sync(1, 128);
        int slot = ld_volatile_s32(a_slot);
        slot = slot < Wmax ? slot : Wmax - 1;
        float* ps = part_base + (static_cast<size_t>(grp) * Wmax + slot) * w.part_floats;
#pragma unroll
        for (int h = 0; h < G; ++h) ps[h * kD + d] = acc[h];
        if (d == 0) {
#pragma unroll
          for (int h = 0; h < G; ++h) { ps[G * kD + h] = m_tot[h]; ps[G * kD + G + h] = l_tot[h]; }
        }
        __threadfence();
        named_bar_sync(1, 128);
        if (tid == 0) {
          const unsigned long long old = atomicAdd(reinterpret_cast<unsigned long long*>(cg + C_DONE),
                                                   static_cast<unsigned long long>(n_folded));
          const unsigned long long nw = old + static_cast<unsigned long long>(n_folded);
          const uint32_t lo = static_cast<uint32_t>(nw), hi = static_cast<uint32_t>(nw >> 32);
          const bool comp = ART ? (hi != 0u && lo == hi - 1u) : (lo == static_cast<uint32_t>(__ldcg(cg + C_OPENT) - 1));
          st_volatile_s32(a_completer, comp ? 1 : 0);
        }
        named_bar_sync(1, 128);
        if (tid == 0) TRACE(trf, 6, grp, n_folded);
        if (ld_volatile_s32(a_completer)) {
          __threadfence();
          combine_group<G>(p, w, grp, tid, 128);
          if (tid == 0) TRACE(trf, 7, grp, 0);
        }
      }
#pragma unroll
      for (int h = 0; h < G; ++h) { acc[h] = 0.f; m_tot[h] = kNegInf; l_tot[h] = 0.f; }
      n_folded = 0;
    };
    if constexpr (!ART) {
      for (int i = 0;; ++i) {
        if (!wait_or_end(bar(sm.pvfull0 + (i & (NP - 1))), (i / NP) & 1, i)) break;
        const ItemInfo ii = items[i & (kItemRing - 1)];
        if (ii.marker) { release_pv(i); flush(ii.group); }
        else fold(i);
      }
    } else {
      // One poll of a group's progress word costs an L2 round trip, so each poll is used for everything it
      // decides: every decided item is merged (or dropped) and every finished item whose mailbox slot is free is
      // published before the word is read again.
      int pub = 0, fld = 0;
      while (true) {
        const int ntot = ld_volatile_s32(a_ntotal);
        if (fld >= ntot) break;
        if (fld < pub && items[fld & (kItemRing - 1)].marker) {               // end of a visit
          release_pv(fld); flush(items[fld & (kItemRing - 1)].group); ++fld; continue;
        }
        // the group whose progress matters now: the oldest unfolded item's, else the next item to publish
        int gq = -1;
        bool pub_ready = false;
        if (pub < ntot && pub - fld < NP) {
          const uint32_t pvb = bar(sm.pvfull0 + (pub & (NP - 1)));
          const uint32_t par = (pub / NP) & 1;
          pub_ready = (fld == pub) ? mbar_try_wait(pvb, par) : mbar_test_wait(pvb, par);
        }
        if (fld < pub) gq = items[fld & (kItemRing - 1)].group;
        else if (pub_ready) gq = items[pub & (kItemRing - 1)].group;
        if (gq < 0) continue;
        if (fld == pub && items[pub & (kItemRing - 1)].marker) { ++pub; continue; }   // a marker has nothing to publish
        const int c = ld_relaxed_gpu(ctl(gq) + C_CTRL);
        // ---- merge (or drop) every item of this group that c decides
        while (fld < pub) {
          const ItemInfo ii = items[fld & (kItemRing - 1)];
          if (ii.marker || ii.group != gq) break;
          if (c < 0 && ii.t > -c) { release_pv(fld); ++fld; continue; }        // beyond t*: never folded
          if (c < 0 || c >= ii.t - 1) { fold(fld); ++fld; continue; }          // no stop before t  =>  t <= t*
          break;
        }
        // ---- publish every finished item of this group whose mailbox slot is free under c
        while (pub < ntot && pub - fld < NP) {
          const uint32_t pvb = bar(sm.pvfull0 + (pub & (NP - 1)));
          if (!mbar_test_wait(pvb, (pub / NP) & 1)) break;
          const ItemInfo ii = items[pub & (kItemRing - 1)];
          if (ii.marker) { ++pub; continue; }
          if (ii.group != gq) break;
          if (c < 0) { ++pub; continue; }                        // fired: an unpublished step lies beyond t*
          if (c < ii.t - M) break;                               // mailbox slot not free yet: step t - M unscanned
          const int slot_i = (ii.t - 1) & (M - 1);
          float* pay = pay_base + (static_cast<size_t>(ii.group) * M + slot_i) * kPayFloats;
          tc_fence_after();
          float pv[G];
          tmem_ld<G>(tmem_PV + tlane + (pub & (NP - 1)) * kUmmaN, pv);
          tmem_ld_wait();
          const uint32_t par = step_parity(ii.t, static_cast<int>(w.mshift));
          if (MODE == 2 || (d & 3) == 0) {
            const int pi = (MODE == 2) ? d : (d >> 2);          // probe coordinate k*(d/32)  (R1)
#pragma unroll
            for (int h = 0; h < G; ++h) pay[kProbeOff + h * PW + pi] = tag_word(pv[h], par);
          }
          if (d == 1) {
            const IterSlotW<G>& sl = slots[pub & (kIterSlots - 1)];
            float ml[2 * G];
#pragma unroll
            for (int h = 0; h < G; ++h) {
              ml[2 * h] = tag_word(sl.mref[h] == kNegInf ? kEmptyMax : sl.mref[h], par);
              ml[2 * h + 1] = tag_word(sl.lsum[h], par);
            }
            st_global_vec<2 * G>(pay, ml);
          }
          if (tid == 0) TRACE(trf, 4, pub, ii.t);
          ++pub;
        }
      }
    }
  } else if (warp == kWarpScan) {
    // ===================================================== open groups; A6 + A7: Algorithm 1 over step summaries
    using Scan = ScanCore<G, PW>;
    constexpr int LPH = Scan::LPH, CPL = Scan::CPL;
    const int h = lane / LPH, sub = lane % LPH;
    const int mshift = static_cast<int>(w.mshift);
    TRACE_INIT(trs, 2);
    uint32_t stg_phase = 0u;
    while (true) {
      int grp = 0;
      if (lane == 0) grp = atomicAdd(hdr + H_NEXT_GROUP, 1);
      grp = __shfl_sync(0xffffffffu, grp, 0);
      if (grp >= groups) break;
      const int b = grp / p.Hkv, g = grp % p.Hkv;
      const Trav tr = make_trav(p, b, g, p.seq_lens[b]);
      const int Tn = tr.T;
      if (Tn == 0) {                                          // empty group: zero row, stop_block 0
        float* out = p.out + (static_cast<int64_t>(b) * p.Hq + g * p.Gr) * kD;
        for (int o = lane; o < p.Gr * kD; o += 32) out[o] = 0.f;
      }
      if (lane == 0) {
        if (!ART || Tn == 0) p.stop_block[grp] = Tn;
        st_release_gpu(ctl(grp) + C_OPENT, Tn + 1);
        atomicAdd(hdr + H_OPENED, 1);
      }
      if constexpr (ART) {
        if (Tn == 0) continue;
        Scan sc; sc.init(); sc.g_real = p.Gr;
        int* c_ctrl = ctl(grp) + C_CTRL;
        const uint8_t* pay = reinterpret_cast<const uint8_t*>(pay_base + static_cast<size_t>(grp) * M * kPayFloats);
        // The mailbox is consumed in aligned blocks of kScanBatch steps through two staging halves: while block b
        // is validated and scanned out of one half, the bulk copy of block b + 1 (issued a block earlier) lands in
        // the other, so the L2 latency is off the sequential path whenever the workers are ahead of the scan.
        const int nblk = (Tn + kScanBatch - 1) / kScanBatch;
        auto fetch = [&](int blk) {                            // lane 0: mailbox block -> staging half blk & 1
          const int nb = min(kScanBatch, Tn - blk * kScanBatch);
          const uint32_t sb = bar(sm.stg0 + (blk & 1));
          mbar_arrive_expect_tx(sb, static_cast<uint32_t>(nb) * kPayBytes);
          tma_load_1d(sbase + sm.stg + static_cast<uint32_t>(blk & 1) * kScanBatch * kPayBytes,
                      pay + static_cast<size_t>((blk * kScanBatch) & (M - 1)) * kPayBytes, static_cast<uint32_t>(nb) * kPayBytes, sb);
        };
        if (lane == 0) { fetch(0); if (nblk > 1) fetch(1); }
        int blk = 0, o = 0, t_stop = 0;                        // current block, steps of it already scanned
        while (blk < nblk) {
          const int nb = min(kScanBatch, Tn - blk * kScanBatch);
          const uint32_t half = static_cast<uint32_t>(blk & 1);
          mbar_wait(bar(sm.stg0 + half), (stg_phase >> half) & 1u);
          stg_phase ^= 1u << half;
          const uint32_t sh = sbase + sm.stg + half * kScanBatch * kPayBytes;
          const int t_first = blk * kScanBatch + 1;
          // ---- a step has arrived when every word this warp will use carries its generation's parity
          const uint32_t par = step_parity(t_first, mshift);   // M is a multiple of the block: one generation per block
          uint32_t bad = 0u;
          constexpr int KC = (CPL <= 4) ? 4 : (CPL <= 8 ? 2 : 1);   // steps whose loads are in flight together
#pragma unroll
          for (int k0 = 0; k0 < kScanBatch; k0 += KC) {
            float2 ml[KC]; float pv[KC][CPL];
#pragma unroll
            for (int k = 0; k < KC; ++k) {
              ml[k] = lds_v2(sh + (k0 + k) * kPayBytes + h * 8u);
              lds_vec<CPL>(sh + (k0 + k) * kPayBytes + (kProbeOff + h * PW + sub * CPL) * 4u, pv[k]);
            }
#pragma unroll
            for (int k = 0; k < KC; ++k) {
              uint32_t x = (__float_as_uint(ml[k].x) ^ par) | (__float_as_uint(ml[k].y) ^ par);
#pragma unroll
              for (int j = 0; j < CPL; ++j) x |= __float_as_uint(pv[k][j]) ^ par;
              bad |= (x & 1u) << (k0 + k);
            }
          }
          bad = __reduce_or_sync(0xffffffffu, bad) | (1u << nb);
          bad >>= o;                                           // steps before o were scanned in an earlier round
          const int n = __ffs(bad) - 1;                        // run of complete steps starting at o
          if (lane == 0) TRACE(trs, 12, t_first + o, n);
          if (n > 0) {
            const uint32_t s0 = sh + static_cast<uint32_t>(o) * kPayBytes;
            const int fired = sc.batch(n, lane, p.tau, p.phi, p.patience,
              [&](int k, bool live, float& mt, float& lt) {
                const float2 ml = lds_v2(s0 + k * kPayBytes + h * 8u);       // beyond the half: unused garbage
                mt = (live && ml.x > -1.0e29f) ? ml.x : kNegInf; lt = live ? ml.y : 0.f;
              },
              [&](int k, bool live, float (&pv)[CPL]) {
                lds_vec<CPL>(s0 + k * kPayBytes + (kProbeOff + h * PW + sub * CPL) * 4u, pv);
#pragma unroll
                for (int j = 0; j < CPL; ++j) pv[j] = live ? pv[j] : 0.f;
              });
            __syncwarp();
            const int t_base = t_first + o;
            const int t_last = fired >= 0 ? t_base + fired : t_base + n - 1;
            if (lane == 0) { st_relaxed_gpu(c_ctrl, fired >= 0 ? -t_last : t_last); TRACE(trs, 8, t_base, n); }
            if (fired >= 0) { t_stop = t_last; break; }
            o += n;
          }
          if (o == nb) {                                       // block done: its half takes block blk + 2
            if (lane == 0 && blk + 2 < nblk) fetch(blk + 2);
            ++blk; o = 0;
          } else if (lane == 0) fetch(blk);                    // some step still missing: read the block again
        }
        // a copy may still be in flight into the other half (after a stop, or the prefetch of the last block)
        {
          const int pend = (t_stop != 0) ? blk + 1 : nblk;     // blocks > blk that were fetched but never waited for
          if (t_stop != 0 && pend < nblk) {
            const uint32_t half = static_cast<uint32_t>(pend & 1);
            mbar_wait(bar(sm.stg0 + half), (stg_phase >> half) & 1u);
            stg_phase ^= 1u << half;
          }
        }
        const int t_final = t_stop ? t_stop : Tn;              // t* (R9)
        int comp = 0;
        if (lane == 0) {
          p.stop_block[grp] = t_final;
          const unsigned long long old = atomicAdd(reinterpret_cast<unsigned long long*>(ctl(grp) + C_DONE),
                                                   static_cast<unsigned long long>(t_final + 1) << 32);
          comp = static_cast<uint32_t>(old) == static_cast<uint32_t>(t_final);
        }
        comp = __shfl_sync(0xffffffffu, comp, 0);
        if (comp) { __threadfence(); combine_group<G>(p, w, grp, lane, 32); }
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == kWarpMmaPV) { tc_fence_after(); tmem_dealloc(tmem_base, kTmemCols); }
#ifdef ART_TRACE
  if (tid == 0) cta_times[1] = trace_now();
#endif
}

}  // namespace ws
}  // namespace art
