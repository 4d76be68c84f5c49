// Algorithm 1's criterion and patience counter (Eq. 2; Eq. 3)
// replayed over per-step summaries, a CHUNK of up to NBK consecutive steps at a time, by one warp.
//
// What a step contributes is the triple (m_t, l_t, P~V_t[idx]) per head: the block's reference exponent, its
// sum of weights relative to it and the probe coordinates of its un-normalised P.V.  The state
// carried from step to step is (M, A, x): the running reference, A_t relative to it and the probe of the
// normalised output x^(t) = o^(t)[idx].  Nothing in that chain is inherently serial:
//
//   * (M_t, A_t) is a prefix "sum" under the associative merge (m1,l1)+(m2,l2) = (max, l1 2^(m1-max) + l2 2^(m2-max))
//     -- the flash-decoding combine -- so the lanes that own the steps of a chunk get it with a log-step
//     shuffle scan; r_t = 2^(m_t - M_t) / A_t follows per lane;
//   * x^(t) = x^(t-1) + r_t (P~V_t - l_t x^(t-1)) is then a chain of ONE fused multiply-add
//     pair per step and coordinate, carried in registers by the lanes that own the coordinates; the increment
//     is formed from the block-local P~V_t, never as a difference of two normalised outputs (fp32 cancellation);
//   * |dx|^2, x.dx, |x|^2 of every step are summed over the lanes of a head with one transposing butterfly, after
//     which lane (head h, step s) owns step s of head h, evaluates Eq. 2 for it, and a ballot brings the G heads
//     together (AND over the heads, reading R2); the patience counter (Eq. 3) is an integer walk over the ballot.
//
// Lane layout: 32 lanes = G heads x LPH lanes; lane `sub` of a head owns probe coordinates sub + LPH j (CPL of
// them) during the recurrence and step sub / STRIDE (if sub % STRIDE == 0) before and after it.
#pragma once
#include "art_common.cuh"

namespace art {

template <int G, int PW>
struct ChunkScan {
  static constexpr int LPH = 32 / G;                                   // lanes per head
  static constexpr int CPL = PW / LPH;                                 // probe coordinates per lane
  static constexpr int NBK0 = LPH < 8 ? LPH : 8;                       // steps per chunk (probe width 32)
  static constexpr int NBK = (PW == 32) ? NBK0 : (NBK0 >= 4 ? NBK0 / 4 : 1);   // wider probes: keep NBK * CPL <= 32 registers
  static constexpr int STRIDE = LPH / NBK;                             // lane distance between the owners of two steps
  static_assert(G == 1 || G == 2 || G == 4 || G == 8, "group size");
  static_assert(PW % LPH == 0 && NBK >= 1 && (NBK & (NBK - 1)) == 0, "layout");

  float M, A;               // running reference exponent (log2 domain) and A_t relative to it, of this lane's head
  float x[CPL];             // x^(t) at this lane's coordinates
  int cnt;                  // c^(t)
  int g_real;               // heads that exist; padding heads (q = 0) never hold the decision back

  __device__ __forceinline__ void init(int g_real_) {
    M = kNegInf; A = 0.f; cnt = 0; g_real = g_real_;          // c^(0) = 0 (Alg. 1 l.2)
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

  // Sums s[k] over the LPH lanes of each head; afterwards s[0] of lane sub = k * STRIDE holds the total of step k.
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
  // The butterfly above leaves step k in the lanes whose bit pattern over the transposing rounds spells k from the
  // most significant round down: with NBK = 2^r steps and rounds m = LPH/2, LPH/4, ... the first r rounds pick the
  // bits of k, highest first, so step k ends in the lanes with (sub / STRIDE) == k.
  static __host__ __device__ constexpr int owner_sub(int k) { return k * STRIDE; }
  // mask of the G lanes (one per head) that own step k
  static __device__ __forceinline__ uint32_t owner_mask(int k) {
    uint32_t need = 0;
#pragma unroll
    for (int h = 0; h < G; ++h) need |= 1u << (h * LPH + owner_sub(k));
    return need;
  }

  // One chunk of n (1..NBK) consecutive steps.
  //   ml: (m_t, l_t) of the step this lane OWNS for its head (lane sub = k STRIDE <-> step k); (-inf, 0) for k >= n
  //       and in lanes that own nothing
  //   pv[k][j]: P~V_t of step k at this lane's coordinates (zeros for k >= n)
  // Returns the 0-based index within the chunk of the step at which the criterion fired (c >= patience,
  // PAPER.md:157), or -1.  A step with no valid token (m = -inf) leaves the state unchanged but counts as a step.
  __device__ __forceinline__ int chunk(int n, int lane, float tau, float phi, int patience, float m_own, float l_own,
                                       const float (&pv)[NBK][CPL]) {
    const int sub = lane % LPH, hbase = lane - sub;
    const bool owner = (sub % STRIDE) == 0 && (sub / STRIDE) < NBK;
    // ---- (M_t, A_t): inclusive scan of the merge over the owners of the chunk's steps, then the carry in front
    float pm = owner ? m_own : kNegInf, pl = owner ? l_own : 0.f;
#pragma unroll
    for (int off = 1; off < NBK; off <<= 1) {
      const float qm = __shfl_up_sync(0xffffffffu, pm, off * STRIDE, LPH);
      const float ql = __shfl_up_sync(0xffffffffu, pl, off * STRIDE, LPH);
      if (sub >= off * STRIDE) {
        const float mx = fmaxf(pm, qm);
        const float a = (pm == mx) ? 1.f : fast_exp2(pm - mx);      // -inf - -inf never evaluated: pm == mx first
        const float b = (qm == mx) ? 1.f : fast_exp2(qm - mx);
        pl = fmaf(a, pl, b * ql); pm = mx;
      }
    }
    float r_own = 0.f;
    {
      const float mx = fmaxf(pm, M);
      const float a = (pm == mx) ? 1.f : fast_exp2(pm - mx);
      const float b = (M == mx) ? 1.f : fast_exp2(M - mx);
      const float At = fmaf(a, pl, b * A);                           // A_t relative to M_t = mx
      if (m_own != kNegInf && owner) r_own = __fdividef(fast_exp2(m_own - mx), At);   // l_t / A_t = r_t l_t
      // carry out: the state after the chunk's last step sits in the owner of step NBK - 1
      const int last = hbase + owner_sub(NBK - 1);
      M = __shfl_sync(0xffffffffu, mx, last);
      A = __shfl_sync(0xffffffffu, At, last);
    }
    // ---- the recurrence x^(t) = x^(t-1) + r_t (P~V_t - l_t x^(t-1)), |dx|^2 per step
    float x0[CPL];
#pragma unroll
    for (int j = 0; j < CPL; ++j) x0[j] = x[j];
    float sd[NBK][1];
    float rk[NBK], lk[NBK];
#pragma unroll
    for (int k = 0; k < NBK; ++k) {
      rk[k] = __shfl_sync(0xffffffffu, r_own, hbase + owner_sub(k));
      lk[k] = __shfl_sync(0xffffffffu, l_own, hbase + owner_sub(k));
    }
#pragma unroll
    for (int k = 0; k < NBK; ++k) {
      float sdd = 0.f;
#pragma unroll
      for (int j = 0; j < CPL; ++j) {
        const float dlt = rk[k] * fmaf(-lk[k], x[j], pv[k][j]);
        sdd = fmaf(dlt, dlt, sdd);
        x[j] += dlt;
      }
      sd[k][0] = sdd;
    }
    reduce<1>(sd, lane);
    // A step can only be stable if every head passes the scale test (first half of Eq. 2); far from convergence none
    // does, and the two sums of the direction test are not needed at all.
    const uint32_t scale_votes = __ballot_sync(0xffffffffu, !owner || sqrt_approx(sd[0][0]) < tau || (lane / LPH) >= g_real);
    uint32_t cand = 0u;
#pragma unroll
    for (int k = 0; k < NBK; ++k) cand |= (k < n && (scale_votes & owner_mask(k)) == owner_mask(k)) ? (1u << k) : 0u;
    if (cand == 0u) { cnt = 0; return -1; }                   // nobody stable: the counter is back at 0 (Eq. 3); n >= 1
    // ---- second pass from the chunk's initial x: x_old . dx and |x_old|^2 per step
    float sa[NBK][2];
    {
      float y[CPL];
#pragma unroll
      for (int j = 0; j < CPL; ++j) y[j] = x0[j];
#pragma unroll
      for (int k = 0; k < NBK; ++k) {
        float sad = 0.f, saa = 0.f;
#pragma unroll
        for (int j = 0; j < CPL; ++j) {
          const float dlt = rk[k] * fmaf(-lk[k], y[j], pv[k][j]);
          sad = fmaf(y[j], dlt, sad); saa = fmaf(y[j], y[j], saa);
          y[j] += dlt;
        }
        sa[k][0] = sad; sa[k][1] = saa;
      }
    }
    reduce<2>(sa, lane);
    const uint32_t votes = __ballot_sync(0xffffffffu, !owner || stable_head(sd[0][0], sa[0][0], sa[0][1], tau, phi) ||
                                                          (lane / LPH) >= g_real);
    int fired = -1;
#pragma unroll
    for (int k = 0; k < NBK; ++k) {
      const bool stable = (votes & owner_mask(k)) == owner_mask(k);       // AND over the group's heads (R2)
      const int c_new = stable ? cnt + 1 : 0;                               // Eq. 3
      const bool live = k < n && fired < 0;
      cnt = live ? c_new : cnt;
      fired = (live && c_new >= patience) ? k : fired;
    }
    return fired;
  }
};

}  // namespace art
