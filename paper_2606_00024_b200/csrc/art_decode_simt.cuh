// ART decode attention, CUDA-core (SIMT) kernel: used for fp32 KV (head_dim 64), where the 1e-5
// output tolerance rules out TF32 tensor-core math.
//
// One thread-block CLUSTER of C CTAs per query group (sequence b, KV head g).  Traversal
// steps t = 1..T are dealt round-robin: CTA c owns steps c+1, c+1+C, ...
// Each CTA streams its blocks HBM -> shared memory with cp.async.bulk (TMA) into an
// mbarrier ring, and its 8 compute warps each run an independent online-softmax stream over
// 8 of the block's 64 tokens, keeping the block-local P~V_t SEPARATE
// ("pending") until the termination decision for the preceding steps is known.  Every step's
// summary (block max, block sum, the probe components of P~V_t; 2+m floats per head) goes
// through distributed shared memory to the cluster leader, whose scan warp replays the
// SEQUENTIAL criterion of Algorithm 1 (Eq. 2-3) in the recurrence form of
// PAPER.md:320/361 and broadcasts progress / the stop step t*.  Blocks with step > t* are
// discarded, so the result equals the sequential algorithm's for any C; the only cost is a
// bounded number of prefetched-then-discarded blocks, which are counted in blocks_loaded.
#pragma once
#include "art_common.cuh"
#include "art_scan.cuh"

namespace art {
namespace simt {

constexpr int kComputeWarps = 8;
constexpr int kProducerWarp = 8;
constexpr int kScanWarp = 9;                      // summaries + (leader) the sequential criterion
constexpr int kThreads = 320;

// ----------------------------------------------------------------------------- element types

template <typename T> struct Elem;
template <> struct Elem<float> {
  static constexpr int E16 = 4, E8 = 2;
  static __device__ __forceinline__ void cvt16(const uint4& r, float (&f)[4]) {
    f[0] = __uint_as_float(r.x); f[1] = __uint_as_float(r.y); f[2] = __uint_as_float(r.z); f[3] = __uint_as_float(r.w);
  }
  static __device__ __forceinline__ void cvt8(const uint2& r, float (&f)[2]) {
    f[0] = __uint_as_float(r.x); f[1] = __uint_as_float(r.y);
  }
};
template <> struct Elem<__nv_bfloat16> {
  static constexpr int E16 = 8, E8 = 4;
  static __device__ __forceinline__ void cvt16(const uint4& r, float (&f)[8]) {
    f[0] = __uint_as_float(r.x << 16); f[1] = __uint_as_float(r.x & 0xffff0000u);
    f[2] = __uint_as_float(r.y << 16); f[3] = __uint_as_float(r.y & 0xffff0000u);
    f[4] = __uint_as_float(r.z << 16); f[5] = __uint_as_float(r.z & 0xffff0000u);
    f[6] = __uint_as_float(r.w << 16); f[7] = __uint_as_float(r.w & 0xffff0000u);
  }
  static __device__ __forceinline__ void cvt8(const uint2& r, float (&f)[4]) {
    f[0] = __uint_as_float(r.x << 16); f[1] = __uint_as_float(r.x & 0xffff0000u);
    f[2] = __uint_as_float(r.y << 16); f[3] = __uint_as_float(r.y & 0xffff0000u);
  }
};
__device__ __forceinline__ float to_float(float x) { return x; }
__device__ __forceinline__ float to_float(__nv_bfloat16 x) { return __bfloat162float(x); }

// ----------------------------------------------------------------------------- warp helpers

// Sum N values over the 16 lanes of a half-warp with a transposing butterfly: while more than
// one value is left each step halves the value count; afterwards lane l holds, in v[0], the
// full sum of value head_of_lane(l).
template <int N, int MASK>
struct Reduce16 {
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
      if constexpr (MASK > 1) Reduce16<n, MASK / 2>::run(v, lane);
    } else {
      v[0] += __shfl_xor_sync(0xffffffffu, v[0], MASK);
      if constexpr (MASK > 1) Reduce16<1, MASK / 2>::run(v, lane);
    }
  }
};

template <int G> __device__ __forceinline__ int head_of_lane(int lane) {   // which value Reduce16 leaves in this lane
  int h = 0;
  if constexpr (G >= 2) h += ((lane >> 3) & 1) * (G / 2);
  if constexpr (G >= 4) h += ((lane >> 2) & 1) * (G / 4);
  if constexpr (G >= 8) h += ((lane >> 1) & 1) * (G / 8);
  return h;
}
template <int G> __device__ __forceinline__ constexpr int lane_of_head(int h) {   // first lane (0..15) holding head h
  int l = 0;
  if constexpr (G >= 2) l |= ((h / (G / 2)) & 1) << 3;
  if constexpr (G >= 4) l |= ((h / (G / 4)) & 1) << 2;
  if constexpr (G >= 8) l |= ((h / (G / 8)) & 1) << 1;
  return l;
}

// ----------------------------------------------------------------------------- shared memory map

struct StageInfo { unsigned long long mask; int blk; int pad; };

struct SmemMap {
  uint32_t ring, sumbuf, mbox, info, bars, misc, total;
  // barrier indices inside `bars` (8 bytes each)
  uint32_t full0, empty0, sumready0, sumfree0, mbox0;
};

__host__ __device__ inline SmemMap make_smem_map(int G, int PW, int stages, int mslots, bool art) {
  SmemMap m;
  uint32_t off = 0;
  m.ring = off; off += static_cast<uint32_t>(stages) * kStageBytes;
  const uint32_t row = static_cast<uint32_t>(G) * (2 + PW) * 4;
  m.sumbuf = off; off += art ? 2u * kComputeWarps * row : 0u;
  m.mbox = off; off += art ? static_cast<uint32_t>(mslots) * row : 0u;
  off = (off + 15u) & ~15u;
  m.info = off; off += static_cast<uint32_t>(stages) * 16u;
  m.bars = off;
  m.full0 = 0; m.empty0 = stages; m.sumready0 = 2 * stages; m.sumfree0 = 2 * stages + 2; m.mbox0 = 2 * stages + 4;
  off += (2u * stages + 4u + (art ? mslots : 0)) * 8u;
  m.misc = off; off += 64u + 16u * 4u;   // ctrl, n_issued, loaded, cta_m[8], cta_l[8]
  m.total = (off + 127u) & ~127u;
  return m;
}

// misc words
constexpr uint32_t kCtrl = 0, kIssued = 4, kLoaded = 8, kCtaM = 64, kCtaL = 96;

// ----------------------------------------------------------------------------- the kernel

// MODE 0: ART off.  MODE 1: ART on, probe = 32 coordinates k*(d/32).  MODE 2: ART on, probe = all d.
template <typename T, int D, int G, int MODE>
__global__ void __launch_bounds__(kThreads, 1) art_decode_kernel(const Params p) {
  constexpr bool ART = MODE != 0;
  constexpr int PW = (MODE == 2) ? D : 32;           // probe width m
  constexpr int E16 = Elem<T>::E16, E8 = Elem<T>::E8;
  constexpr int ROWF = 2 + PW;                       // summary floats per head: max, sum, probe
  static_assert(D * sizeof(T) == kRowBytes, "token row must be 256 bytes");
  static_assert(D / 32 == E8, "one probe coordinate per 8-byte chunk");

  extern __shared__ __align__(128) uint8_t smem[];
  const int S = p.stages, M = p.mbox_slots;
  const SmemMap sm = make_smem_map(G, PW, S, M, ART);
  const uint32_t sbase = smem_u32(smem);
  const uint32_t bars = sbase + sm.bars;
  auto bar = [&](uint32_t idx) { return bars + idx * 8u; };
  const uint32_t a_ctrl = sbase + sm.misc + kCtrl, a_issued = sbase + sm.misc + kIssued,
                 a_loaded = sbase + sm.misc + kLoaded;
  float* sumbuf = reinterpret_cast<float*>(smem + sm.sumbuf);
  float* mbox = reinterpret_cast<float*>(smem + sm.mbox);
  StageInfo* info = reinterpret_cast<StageInfo*>(smem + sm.info);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int C = static_cast<int>(cluster_nctarank());
  const int rank = static_cast<int>(cluster_ctarank());
  const int group = blockIdx.x / C;
  const int b = group / p.Hkv, g = group % p.Hkv;
  const int L = p.seq_lens[b];
  const Trav tr = make_trav(p, b, g, L);
  const int Tn = tr.T;
  const int n_c = (Tn > rank) ? (Tn - rank + C - 1) / C : 0;   // steps owned by this CTA

  if (tid == 0) {
    for (int s = 0; s < S; ++s) { mbar_init(bar(sm.full0 + s), 1); mbar_init(bar(sm.empty0 + s), kComputeWarps); }
    mbar_init(bar(sm.sumready0), kComputeWarps); mbar_init(bar(sm.sumready0 + 1), kComputeWarps);
    mbar_init(bar(sm.sumfree0), 1); mbar_init(bar(sm.sumfree0 + 1), 1);
    if (ART) for (int s = 0; s < M; ++s) mbar_init(bar(sm.mbox0 + s), 32);
    st_volatile_s32(a_ctrl, 0); st_volatile_s32(a_issued, 0x7fffffff); st_volatile_s32(a_loaded, 0);
    fence_mbar_init();
  }
  cluster_sync_all();   // barriers of every CTA of the cluster are live before any remote arrive

  // per-warp flash state (compute warps); declared here so the epilogue can see it
  float acc[G][E8], m_w[G], l_w[G];
#pragma unroll
  for (int h = 0; h < G; ++h) {
    m_w[h] = kNegInf; l_w[h] = 0.f;
#pragma unroll
    for (int e = 0; e < E8; ++e) acc[h][e] = 0.f;
  }

  // "fired and step t lies beyond t*": every wait that could otherwise hang forever checks this
  auto beyond_stop = [&](int t) -> bool {
    if constexpr (!ART) return false;
    const int c = ld_acquire_ctrl(a_ctrl);
    return c < 0 && t > -c;
  };

  if (warp == kProducerWarp) {
    // ===================================================== A1 + A2: resolve blocks, issue TMA loads
    int it_issued = 0, loaded = 0;
    bool stop = false;
    for (int i0 = 0; i0 < n_c && !stop; i0 += 32) {
      const int i = i0 + lane;
      int blk = -1; unsigned long long mask = 0ull; long long off = 0;
      if (i < n_c) {
        blk = trav_block(tr, i * C + rank + 1);
        mask = block_mask(p, L, blk);
        if (mask) {
          const int page = p.block_table[static_cast<int64_t>(b) * p.max_blocks + blk];
          off = static_cast<int64_t>(page) * p.page_stride + static_cast<int64_t>(g) * p.head_stride;
        }
      }
      const int cnt = min(32, n_c - i0);
      for (int kk = 0; kk < cnt; ++kk) {
        const int it = i0 + kk, stage = it % S, t = it * C + rank + 1;
        const int blk_k = __shfl_sync(0xffffffffu, blk, kk);
        const unsigned long long mask_k = __shfl_sync(0xffffffffu, mask, kk);
        const long long off_k = __shfl_sync(0xffffffffu, off, kk);
        if (it >= S) {                                       // slot must have been released
          const uint32_t par = ((it / S) - 1) & 1;
          while (!mbar_try_wait(bar(sm.empty0 + stage), par)) { if (beyond_stop(t)) { stop = true; break; } }
        }
        if (!stop && beyond_stop(t)) stop = true;            // A7: stop issuing prefetch once fired
        if (stop) break;
        const uint32_t fb = bar(sm.full0 + stage);
        const uint32_t dstK = sbase + sm.ring + stage * kStageBytes, dstV = dstK + kTileBytes;
        if (lane == 0) { info[stage].mask = mask_k; info[stage].blk = blk_k; }
        if (mask_k == 0ull) {
          if (lane == 0) mbar_arrive(fb);                    // nothing to load: an all-masked step
        } else if (p.layout == ART_LAYOUT_HND) {
          if (lane == 0) {
            mbar_arrive_expect_tx(fb, kStageBytes);
            tma_load_1d(dstK, p.k + off_k, kTileBytes, fb);
            tma_load_1d(dstV, p.v + off_k, kTileBytes, fb);
          }
          ++loaded;
        } else {                                             // NHD: one 256-byte row per (token)
          if (lane == 0) mbar_arrive_expect_tx(fb, kStageBytes);
          __syncwarp();
#pragma unroll
          for (int rr = 0; rr < 2; ++rr) {
            const int r = lane * 2 + rr;
            tma_load_1d(dstK + r * kRowBytes, p.k + off_k + r * p.token_stride, kRowBytes, fb);
            tma_load_1d(dstV + r * kRowBytes, p.v + off_k + r * p.token_stride, kRowBytes, fb);
          }
          ++loaded;
        }
        it_issued = it + 1;
      }
    }
    if (lane == 0) { st_volatile_s32(a_issued, it_issued); st_volatile_s32(a_loaded, loaded); }
    // drain: bulk copies still in flight must land before the CTA reuses the ring or exits (H5)
    for (int j = max(0, it_issued - S); j < it_issued; ++j) mbar_wait(bar(sm.full0 + j % S), (j / S) & 1);
  } else if (warp < kComputeWarps) {
    // ===================================================== A3-A5: scores, online softmax, P.V
    const int half = lane >> 4, c16 = lane & 15;
    float qreg[G][E16];                                      // this lane's 16-byte chunk of every head's q
    {
      // row h = query token h / Gh, head h % Gh of the group (R15; one query token: row == head)
      const T* qp = reinterpret_cast<const T*>(p.q) + (static_cast<int64_t>(b) * p.qlen * p.Hq + g * p.Gh) * D + c16 * E16;
#pragma unroll
      for (int h = 0; h < G; ++h)
#pragma unroll
        for (int e = 0; e < E16; ++e)                          // padding rows: q = 0
          qreg[h][e] = (h < p.Gr) ? to_float(qp[((h / p.Gh) * p.Hq + h % p.Gh) * D + e]) * p.scale_log2 : 0.f;
    }
    float pend[G][E8], pend_m[G], pend_l[G];
    bool have_pend = false; int pend_t = 0;
#pragma unroll
    for (int h = 0; h < G; ++h) { pend_m[h] = kNegInf; pend_l[h] = 0.f;
#pragma unroll
      for (int e = 0; e < E8; ++e) pend[h][e] = 0.f; }

    auto fold = [&](const float (&val)[G][E8], const float (&mt)[G], const float (&lt)[G]) {
#pragma unroll
      for (int h = 0; h < G; ++h) {
        const float mn = fmaxf(m_w[h], mt[h]);
        if (mn == kNegInf) continue;
        const float a = fast_exp2(m_w[h] - mn), bb = fast_exp2(mt[h] - mn);
        l_w[h] = a * l_w[h] + bb * lt[h];
#pragma unroll
        for (int e = 0; e < E8; ++e) acc[h][e] = a * acc[h][e] + bb * val[h][e];
        m_w[h] = mn;
      }
    };
    auto wait_decision = [&](int need) -> int {              // progress >= need, or fired
      int c;
      do { c = ld_acquire_ctrl(a_ctrl); } while (c >= 0 && c < need);
      return c;
    };

    for (int i = 0; i < n_c; ++i) {
      const int stage = i % S, t = i * C + rank + 1;
      {
        bool got = false;
        const uint32_t par = (i / S) & 1;
        while (true) {
          if (mbar_try_wait(bar(sm.full0 + stage), par)) { got = true; break; }
          if (ART && ld_volatile_s32(a_issued) <= i) break;   // the producer stopped before this step
        }
        if (!got) break;
      }
      const unsigned long long vmask = info[stage].mask;
      // R15: the row this lane ends up with after the reduction may not see the last `cut` tokens of the sequence;
      // e = tokens of the sequence from the start of this block on (cut == 0 for a single query token)
      const int row_lim = (L - info[stage].blk * kBlockTokens) - static_cast<int>((p.cuts >> (4 * head_of_lane<G>(lane))) & 15u);
      const uint32_t Kt = sbase + sm.ring + stage * kStageBytes, Vt = Kt + kTileBytes;

      // ---- A3: s = q.k / sqrt(d) (log2 domain) for this warp's 8 tokens; lane ends with head hl
      float sv[4];
#pragma unroll
      for (int pp = 0; pp < 4; ++pp) {
        const int r = warp * 8 + pp * 2 + half;
        float kv[E16];
        Elem<T>::cvt16(lds128(Kt + r * kRowBytes + c16 * 16), kv);
        float s[G];
#pragma unroll
        for (int h = 0; h < G; ++h) {
          float a = 0.f;
#pragma unroll
          for (int e = 0; e < E16; ++e) a = fmaf(qreg[h][e], kv[e], a);
          s[h] = a;
        }
        Reduce16<G, 8>::run(s, lane);
        sv[pp] = (((vmask >> r) & 1ull) && r < row_lim) ? s[0] : kNegInf;     // masked tokens: weight 0 (R8)
      }
      // ---- A4: block-local softmax over the warp's 8 tokens
      float mloc = fmaxf(fmaxf(sv[0], sv[1]), fmaxf(sv[2], sv[3]));
      mloc = fmaxf(mloc, __shfl_xor_sync(0xffffffffu, mloc, 16));
      float pr[4], lsum = 0.f;
#pragma unroll
      for (int pp = 0; pp < 4; ++pp) { pr[pp] = (sv[pp] == kNegInf) ? 0.f : fast_exp2(sv[pp] - mloc); lsum += pr[pp]; }
      lsum += __shfl_xor_sync(0xffffffffu, lsum, 16);
      float mt[G], lt[G];
#pragma unroll
      for (int h = 0; h < G; ++h) {
        mt[h] = __shfl_sync(0xffffffffu, mloc, lane_of_head<G>(h));
        lt[h] = __shfl_sync(0xffffffffu, lsum, lane_of_head<G>(h));
      }
      // ---- A5: P~V for the warp's 8 tokens; lane owns the 8-byte chunk `lane` of every row
      float nw[G][E8];
#pragma unroll
      for (int h = 0; h < G; ++h)
#pragma unroll
        for (int e = 0; e < E8; ++e) nw[h][e] = 0.f;
#pragma unroll
      for (int rr = 0; rr < 8; ++rr) {
        const int r = warp * 8 + rr;
        float ph[G];
#pragma unroll
        for (int h = 0; h < G; ++h) ph[h] = __shfl_sync(0xffffffffu, pr[rr >> 1], (rr & 1) * 16 + lane_of_head<G>(h));
        if ((vmask >> r) & 1ull) {                           // warp-uniform; masked rows may hold NaN
          float vv[E8];
          Elem<T>::cvt8(lds64(Vt + r * kRowBytes + lane * 8), vv);
#pragma unroll
          for (int h = 0; h < G; ++h)
#pragma unroll
            for (int e = 0; e < E8; ++e) nw[h][e] = fmaf(ph[h], vv[e], nw[h][e]);
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(sm.empty0 + stage));    // K/V tile consumed: slot free

      if constexpr (!ART) {
        fold(nw, mt, lt);
      } else {
        // ---- publish this warp's share of the step summary (max, sum, probe part of P~V)
        const int par = i & 1;
        bool discard = false;
        if (i >= 2) {
          const uint32_t ph2 = ((i >> 1) - 1) & 1;
          while (!mbar_try_wait(bar(sm.sumfree0 + par), ph2)) { if (beyond_stop(t)) { discard = true; break; } }
        }
        if (discard) break;                                  // t > t*: this block is not part of the result
        float* sb = sumbuf + static_cast<size_t>(par * kComputeWarps + warp) * G * ROWF;
#pragma unroll
        for (int h = 0; h < G; ++h) {
          if constexpr (MODE == 1) sb[h * ROWF + 2 + lane] = nw[h][0];      // coordinate lane*(d/32)  (R1)
          else {
#pragma unroll
            for (int e = 0; e < E8; ++e) sb[h * ROWF + 2 + lane * E8 + e] = nw[h][e];
          }
          if (lane == h) { sb[h * ROWF] = mt[h]; sb[h * ROWF + 1] = lt[h]; }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar(sm.sumready0 + par));
        // ---- fold the PREVIOUS block once the decision for everything before it is known
        if (have_pend) {
          const int c = wait_decision(pend_t - 1);
          have_pend = false;
          if (c < 0 && pend_t > -c) break;                   // previous (and so this) block lies beyond t*
          fold(pend, pend_m, pend_l);
          if (c < 0 && t > -c) break;
        }
#pragma unroll
        for (int h = 0; h < G; ++h) { pend_m[h] = mt[h]; pend_l[h] = lt[h];
#pragma unroll
          for (int e = 0; e < E8; ++e) pend[h][e] = nw[h][e]; }
        have_pend = true; pend_t = t;
      }
    }
    if (ART && have_pend) {
      const int c = wait_decision(pend_t - 1);
      if (!(c < 0 && pend_t > -c)) fold(pend, pend_m, pend_l);
    }
  } else if (ART && warp == kScanWarp) {
    // ===================================================== A6 + A7 + A9: summaries, sequential criterion
    constexpr int LPH = 32 / G;                              // lanes per head
    constexpr int CPL = PW / LPH;                            // probe components per lane
    const int h = lane / LPH, sub = lane % LPH;

    // merge the 8 warps' shares of local iteration i into one step summary (mt, lt, pv[])
    auto merge_local = [&](int i, int t, float& mt, float& lt, float (&pv)[CPL]) -> bool {
      const int par = i & 1;
      const uint32_t ph = (i >> 1) & 1;
      while (!mbar_try_wait(bar(sm.sumready0 + par), ph)) { if (beyond_stop(t)) return false; }
      const float* sb = sumbuf + static_cast<size_t>(par * kComputeWarps) * G * ROWF + h * ROWF;
      float mw[kComputeWarps];
      mt = kNegInf;
#pragma unroll
      for (int w = 0; w < kComputeWarps; ++w) { mw[w] = sb[w * G * ROWF]; mt = fmaxf(mt, mw[w]); }
      lt = 0.f;
#pragma unroll
      for (int j = 0; j < CPL; ++j) pv[j] = 0.f;
#pragma unroll
      for (int w = 0; w < kComputeWarps; ++w) {
        const float f = (mw[w] == kNegInf) ? 0.f : fast_exp2(mw[w] - mt);
        lt = fmaf(f, sb[w * G * ROWF + 1], lt);
#pragma unroll
        for (int j = 0; j < CPL; ++j) pv[j] = fmaf(f, sb[w * G * ROWF + 2 + sub + LPH * j], pv[j]);
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(bar(sm.sumfree0 + par));
      return true;
    };

    if (rank == 0) {
      // ---- leader: Algorithm 1's loop over steps, on summaries, in batches (art_scan.cuh).
      // The leader's own steps do not arrive by themselves: the scan warp moves each of them from the summary
      // buffers into its mailbox slot first, then every step of the group is read from the mailbox alike.
      using Scan = ScanCore<G, PW>;
      Scan sc; sc.init(); sc.g_real = p.Gr;
      int t = 1, t_stop = 0, own_next = 0;                   // own_next: next local iteration to move (step own_next * C + 1)
      while (t <= Tn) {
        while (own_next < n_c) {
          const int ts = own_next * C + 1;
          if (ts > t - 1 + M) break;                         // its slot still holds step ts - M, not scanned yet
          if (ts != t && !mbar_test_wait(bar(sm.sumready0 + (own_next & 1)), (own_next >> 1) & 1)) break;   // not finished: later
          float mt, lt, pv[CPL];
          merge_local(own_next, ts, mt, lt, pv);             // waits if the scan cannot go on without it (ts == t)
          float* mb = mbox + static_cast<size_t>((ts - 1) % M) * G * ROWF + h * ROWF;
          if (sub == 0) { mb[0] = mt; mb[1] = lt; }
#pragma unroll
          for (int j = 0; j < CPL; ++j) mb[2 + sub + LPH * j] = pv[j];
          mbar_arrive(bar(sm.mbox0 + (ts - 1) % M));         // 32 arrivals complete the slot, as for a remote step
          ++own_next;
        }
        // how many consecutive steps have arrived (lane k looks at step t + k); the first one is waited for
        while (!mbar_try_wait_cluster(bar(sm.mbox0 + (t - 1) % M), ((t - 1) / M) & 1)) {}
        int n;
        {
          bool ok = lane == 0;
          if (lane >= 1 && lane < kScanBatch && t + lane <= Tn && lane < M)
            ok = mbar_test_wait(bar(sm.mbox0 + (t - 1 + lane) % M), ((t - 1 + lane) / M) & 1);
          const uint32_t bits = __ballot_sync(0xffffffffu, ok);
          n = __ffs(~bits) - 1;
          n = n > kScanBatch ? kScanBatch : n;
        }
        for (int k = 1; k < n; ++k)                          // every lane acquires the slots it is about to read
          while (!mbar_try_wait_cluster(bar(sm.mbox0 + (t - 1 + k) % M), ((t - 1 + k) / M) & 1)) {}
        const int t0 = t - 1;
        const int fired = sc.batch(n, lane, p.tau, p.phi, p.patience,
          [&](int k, bool live, float& mt, float& lt) {
            const float* mb = mbox + static_cast<size_t>((t0 + k) % M) * G * ROWF + h * ROWF;
            const float m_ = mb[0], l_ = mb[1];
            mt = live ? m_ : kNegInf; lt = live ? l_ : 0.f;
          },
          [&](int k, bool live, float (&pv)[CPL]) {
            const float* mb = mbox + static_cast<size_t>((t0 + k) % M) * G * ROWF + h * ROWF;
#pragma unroll
            for (int j = 0; j < CPL; ++j) { const float v = mb[2 + sub + LPH * j]; pv[j] = live ? v : 0.f; }
          });
        __syncwarp();
        const int t_last = fired >= 0 ? t + fired : t + n - 1;
        // relaxed is enough: the value depends on the mailbox loads of these steps, so they have completed
        if (lane < C) asm volatile("st.relaxed.cluster.shared::cluster.s32 [%0], %1;" :: "r"(mapa(a_ctrl, lane)), "r"(fired >= 0 ? -t_last : t_last) : "memory");
        if (fired >= 0) { t_stop = t_last; break; }
        t += n;
      }
      if (lane == 0) p.stop_block[group] = t_stop ? t_stop : Tn;             // t* (R9)
    } else {
      // ---- other CTAs: ship each own step's summary to the leader's mailbox
      for (int i = 0; i < n_c; ++i) {
        const int t = i * C + rank + 1;
        float mt, lt, pv[CPL];
        if (!merge_local(i, t, mt, lt, pv)) break;
        bool dead = false;                                   // the slot must have been consumed: step t - M scanned
        while (true) {
          const int c = ld_acquire_ctrl(a_ctrl);
          if (c < 0) { dead = t > -c; break; }
          if (c >= t - M) break;
        }
        if (dead) break;
        const int slot = (t - 1) % M;
        const uint32_t row = sbase + sm.mbox + (static_cast<uint32_t>(slot) * G + h) * ROWF * 4u;
        const uint32_t rrow = mapa(row, 0);
        if (sub == 0) { st_cluster_f32(rrow, mt); st_cluster_f32(rrow + 4, lt); }
#pragma unroll
        for (int j = 0; j < CPL; ++j) st_cluster_f32(rrow + (2 + sub + LPH * j) * 4u, pv[j]);
        mbar_arrive_remote(mapa(bar(sm.mbox0 + slot), 0));   // release.cluster: this lane's stores first
      }
    }
  }

  // ===================================================== A8 / A9: combine partial states, write out
  __syncthreads();                                           // ring is free: all loads drained, all warps done
  float* part = reinterpret_cast<float*>(smem + sm.ring);    // [8][G][D] + pm[8][G] + pl[8][G] + cta[G][D]
  float* pm = part + kComputeWarps * G * D;
  float* pl = pm + kComputeWarps * G;
  float* cta = pl + kComputeWarps * G;
  if (warp < kComputeWarps) {
#pragma unroll
    for (int h = 0; h < G; ++h) {
#pragma unroll
      for (int e = 0; e < E8; ++e) part[(warp * G + h) * D + lane * E8 + e] = acc[h][e];
      if (lane == h) { pm[warp * G + h] = m_w[h]; pl[warp * G + h] = l_w[h]; }
    }
  }
  __syncthreads();
  float* cta_m = reinterpret_cast<float*>(smem + sm.misc + kCtaM);
  float* cta_l = reinterpret_cast<float*>(smem + sm.misc + kCtaL);
  for (int o = tid; o < G * D; o += kThreads) {
    const int h = o / D;
    float mx = kNegInf;
#pragma unroll
    for (int w = 0; w < kComputeWarps; ++w) mx = fmaxf(mx, pm[w * G + h]);
    float a = 0.f, l = 0.f;
#pragma unroll
    for (int w = 0; w < kComputeWarps; ++w) {
      const float f = (pm[w * G + h] == kNegInf) ? 0.f : fast_exp2(pm[w * G + h] - mx);
      a = fmaf(f, part[(w * G + h) * D + (o - h * D)], a);
      l = fmaf(f, pl[w * G + h], l);
    }
    cta[o] = a;
    if (o == h * D) { cta_m[h] = mx; cta_l[h] = l; }
  }
  cluster_sync_all();
  if (rank == 0) {
    for (int o = tid; o < G * D; o += kThreads) {
      const int h = o / D;
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
        p.out[((static_cast<int64_t>(b) * p.qlen + h / p.Gh) * p.Hq + g * p.Gh + h % p.Gh) * D + (o - h * D)] = (l > 0.f) ? a / l : 0.f;
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
  cluster_sync_all();                                        // peers' shared memory stays alive until read
}

}  // namespace simt
}  // namespace art
