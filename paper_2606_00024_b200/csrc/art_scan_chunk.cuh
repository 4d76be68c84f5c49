// Algorithm 1's stability criterion (Eq. 2) replayed over per-step summaries, a CHUNK
// of up to NBK consecutive steps at a time, by one warp for GW of the group's heads.  (The patience counter, Eq. 3
// PAPER.md:154, is an integer walk over the per-step results of all heads; it lives with the caller.)
//
// What a step contributes is the triple (m_t, l_t, P~V_t[idx]) per head: the block's reference exponent, its
// sum of weights relative to it and the probe coordinates of its un-normalised P.V.  The state
// carried from step to step is (M, A, x): the running reference, A_t relative to it and the probe of the
// normalised output x^(t) = o^(t)[idx].  Nothing in that chain is inherently serial:
//
//   * A_t is a prefix sum once every block sum is expressed against ONE reference Mc (the largest exponent of the
//     chunk and the carry): W_t = A 2^(M - Mc) + sum_{s <= t} l_s 2^(m_s - Mc), and the factor the recurrence needs,
//     r_t = 2^(m_t - M_t) / A_t, equals 2^(m_t - Mc) / W_t whatever M_t is.  The lanes that own the steps of a chunk
//     get W_t with a log-step shuffle scan;
//   * x^(t) = x^(t-1) + r_t (P~V_t - l_t x^(t-1)) is then a chain of two fused multiply-adds
//     per step and coordinate, carried in registers by the lanes that own the coordinates; the increment is formed
//     from the block-local P~V_t, never as a difference of two normalised outputs (fp32 cancellation);
//   * |dx|^2, x.dx, |x|^2 of every step are summed over the lanes of a head with one transposing butterfly, after
//     which lane (head h, step s) owns step s of head h and evaluates Eq. 2 for it; a ballot collects the steps.
//
// Lane layout: 32 lanes = GW heads x LPH lanes; lane `sub` of a head owns probe coordinates sub + LPH j (CPL of
// them) during the recurrence and step sub / STRIDE (if sub % STRIDE == 0) before and after it.
#pragma once
#include "art_common.cuh"

namespace art {

template <int GW, int PW>
struct ChunkScan {
  static constexpr int LPH = 32 / GW;                                  // lanes per head
  static constexpr int CPL = PW / LPH;                                 // probe coordinates per lane
  static constexpr int NBK_R = 16 / CPL < 1 ? 1 : 16 / CPL;            // P~V of a chunk: at most 16 registers per lane (it is held twice)
  static constexpr int NBK = NBK_R < 8 ? NBK_R : 8;                    // steps per chunk (<= 8 <= LPH)
  static constexpr int STRIDE = LPH / NBK;                             // lane distance between the owners of two steps
  static_assert(GW == 1 || GW == 2 || GW == 4 || GW == 8, "heads per warp");
  static_assert(PW % LPH == 0 && NBK >= 1 && (NBK & (NBK - 1)) == 0 && NBK <= LPH, "layout");

  float M, A;               // running reference exponent (log2 domain) and A_t relative to it, of this lane's head
  float x[CPL];             // x^(t) at this lane's coordinates
  bool real;                // this lane's head exists; padding heads (q = 0) never hold the decision back

  __device__ __forceinline__ void init(bool real_) {
    M = kNegInf; A = 0.f; real = real_;
#pragma unroll
    for (int j = 0; j < CPL; ++j) x[j] = 0.f;               // x^(0) = 0 (Alg. 1 l.1)
  }

  static __device__ __forceinline__ float sqrt_approx(float v) {
    float r; asm("sqrt.approx.f32 %0, %1;" : "=f"(r) : "f"(v)); return r;
  }
  // Eq. 2 for one head from the complete sums |dx|^2, x_old.dx, |x_old|^2: d_scale = ||dx||; d_direction =
  // 1 - cos(x_new, x_old) evaluated as (|a|^2 |d|^2 - (a.d)^2) / (|a||b| (|a||b| + a.b)), free of the cancellation in
  // 1 - cos; compared as num < phi * den.  |b|^2 = |a|^2 + 2 a.d + |d|^2.  Zero norm => cos := 0 (R4); strict '<' (R5).
  static __device__ __forceinline__ bool stable_head(float sdd, float sad, float saa, float tau, float phi) {
    const float sbb = fmaf(2.f, sad, saa) + sdd;
    const bool scale_ok = sqrt_approx(sdd) < tau;
    bool dir_ok = 1.f < phi;
    if (saa > 0.f && sbb > 0.f) {
      const float nanb = sqrt_approx(saa) * sqrt_approx(sbb);
      const float ab = saa + sad;
      if (ab > 0.f) dir_ok = fmaxf(fmaf(saa, sdd, -sad * sad), 0.f) < phi * (nanb * (nanb + ab));
      else dir_ok = (1.f - __fdividef(ab, nanb)) < phi;
    }
    return scale_ok && dir_ok;
  }

  // Sums s[k] over the LPH lanes of each head; afterwards s[0] of the lanes with sub / STRIDE == k holds the total of
  // step k.  (The transposing rounds pick the bits of k from the most significant one down.)
  template <int Q>
  static __device__ __forceinline__ void reduce(float (&s)[NBK][Q], int lane) {
    int cntk = NBK;
#pragma unroll
    for (int m = LPH / 2; m >= 1; m >>= 1) {
      if (cntk > 1) {                                        // transposing round: halve the number of steps held
        const int half = cntk / 2;
        const bool up = (lane & m) != 0;
#pragma unroll
        for (int i = 0; i < half; ++i)
#pragma unroll
          for (int q = 0; q < Q; ++q) {
            const float keep = up ? s[i + half][q] : s[i][q];
            const float send = up ? s[i][q] : s[i + half][q];
            s[i][q] = keep + __shfl_xor_sync(0xffffffffu, send, m);
          }
        cntk = half;
      } else {
#pragma unroll
        for (int q = 0; q < Q; ++q) s[0][q] += __shfl_xor_sync(0xffffffffu, s[0][q], m);
      }
    }
  }
  static __host__ __device__ constexpr int owner_sub(int k) { return k * STRIDE; }
  // mask of the GW lanes (one per head) that own step k
  static __device__ __forceinline__ uint32_t owner_mask(int k) {
    uint32_t need = 0;
#pragma unroll
    for (int h = 0; h < GW; ++h) need |= 1u << (h * LPH + owner_sub(k));
    return need;
  }

  // the widest spread of reference exponents (log2) a chunk may hold and still be scanned against ONE common
  // reference: beyond it the caller scans the steps one at a time (a chunk of one step is exact for any spread)
  static constexpr float kMaxSpread = 60.f;

  // Can the steps be scanned as one chunk?  m_own as for chunk().  (Same answer in every lane.)
  __device__ __forceinline__ bool spread_ok(float m_own, bool owner) const {
    float lo = (owner && m_own != kNegInf) ? m_own : INFINITY, hi = owner ? m_own : kNegInf;
    if (A > 0.f) { lo = fminf(lo, M); hi = fmaxf(hi, M); }
    return !__any_sync(0xffffffffu, hi - lo > kMaxSpread);       // inf - inf = NaN compares false: an empty side is fine
  }

  // One chunk of n (1..NBK) consecutive steps.
  //   m_own, l_own: (m_t, l_t) of the step this lane OWNS for its head (lane sub = k STRIDE <-> step k); (-inf, 0) for
  //                 k >= n and in lanes that own nothing
  //   pv[k][j]: P~V_t of step k at this lane's coordinates (zeros for k >= n)
  // Returns bit k = "every head of this warp is stable at step k" (Eq. 2 with AND over the heads, reading R2), k < n.
  // A step with no valid token (m = -inf) leaves the state unchanged but counts as a step.
  // Requires spread_ok() unless n == 1.
  __device__ __forceinline__ uint32_t chunk(int n, int lane, float tau, float phi, float m_own, float l_own,
                                            const float (&pv)[NBK][CPL]) {
    const int sub = lane % LPH, hbase = lane - sub;
    const bool owner = (sub % STRIDE) == 0;
    // ---- W_t (see the header): reference Mc, e_s = 2^(m_s - Mc), prefix sum over the owners, r_t = e_t / W_t
    float mc = owner ? m_own : kNegInf;
#pragma unroll
    for (int w = LPH / 2; w >= STRIDE; w >>= 1) mc = fmaxf(mc, __shfl_xor_sync(0xffffffffu, mc, w));   // over the owners (the other lanes' value is not used)
    mc = fmaxf(mc, M);
    const float e_own = (owner && m_own != kNegInf) ? fast_exp2(m_own - mc) : 0.f;
    float W = l_own * e_own;                                  // 0 in lanes that own nothing
#pragma unroll
    for (int off = STRIDE; off < LPH; off <<= 1) {
      const float q = __shfl_up_sync(0xffffffffu, W, off, LPH);
      if (sub >= off) W += q;
    }
    W += (M == kNegInf) ? 0.f : A * fast_exp2(M - mc);
    const float r_own = (e_own > 0.f) ? __fdividef(e_own, W) : 0.f;      // l_t r_t = l_t / A_t of PAPER.md:320
    M = mc;
    A = __shfl_sync(0xffffffffu, W, hbase + owner_sub(NBK - 1));   // the inclusive sum at the owner of the chunk's last step
    const float rl_own = r_own * l_own;
    // ---- the recurrence x^(t) = x^(t-1) + r_t (P~V_t - l_t x^(t-1)), |dx|^2 per step
    float x0[CPL];
#pragma unroll
    for (int j = 0; j < CPL; ++j) x0[j] = x[j];
    float sd[NBK][1];
#pragma unroll
    for (int k = 0; k < NBK; ++k) {
      const float rk = __shfl_sync(0xffffffffu, r_own, hbase + owner_sub(k));
      const float rlk = __shfl_sync(0xffffffffu, rl_own, hbase + owner_sub(k));
      float sdd = 0.f;
#pragma unroll
      for (int j = 0; j < CPL; ++j) {
        const float dlt = fmaf(rk, pv[k][j], -rlk * x[j]);
        sdd = fmaf(dlt, dlt, sdd);
        x[j] += dlt;
      }
      sd[k][0] = sdd;
    }
    reduce<1>(sd, lane);
    // A step can only be stable if every head passes the scale test (first half of Eq. 2); far from convergence none
    // does, and the two sums of the direction test are not needed at all.
    const float sdd_own = sd[0][0];
    const uint32_t scale_votes = __ballot_sync(0xffffffffu, !owner || !real || sqrt_approx(sdd_own) < tau);
    uint32_t cand = 0u;
#pragma unroll
    for (int k = 0; k < NBK; ++k) cand |= (k < n && (scale_votes & owner_mask(k)) == owner_mask(k)) ? (1u << k) : 0u;
    if (cand == 0u) return 0u;
    // ---- second pass from the chunk's initial x: x_old . dx and |x_old|^2 per step
    float sa[NBK][2];
    {
      float y[CPL];
#pragma unroll
      for (int j = 0; j < CPL; ++j) y[j] = x0[j];
#pragma unroll
      for (int k = 0; k < NBK; ++k) {
        const float rk = __shfl_sync(0xffffffffu, r_own, hbase + owner_sub(k));
        const float rlk = __shfl_sync(0xffffffffu, rl_own, hbase + owner_sub(k));
        float sad = 0.f, saa = 0.f;
#pragma unroll
        for (int j = 0; j < CPL; ++j) {
          const float dlt = fmaf(rk, pv[k][j], -rlk * y[j]);
          sad = fmaf(y[j], dlt, sad); saa = fmaf(y[j], y[j], saa);
          y[j] += dlt;
        }
        sa[k][0] = sad; sa[k][1] = saa;
      }
    }
    reduce<2>(sa, lane);
    const uint32_t votes = __ballot_sync(0xffffffffu, !owner || !real || stable_head(sdd_own, sa[0][0], sa[0][1], tau, phi));
    uint32_t out = 0u;
#pragma unroll
    for (int k = 0; k < NBK; ++k) out |= (k < n && (votes & owner_mask(k)) == owner_mask(k)) ? (1u << k) : 0u;
    return out;
  }
};

}  // namespace art
