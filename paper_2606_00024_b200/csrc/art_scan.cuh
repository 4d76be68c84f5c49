// The sequential part of ART: Algorithm 1's criterion and patience counter (PAPER.md:101-133,
// Eq. 2, Eq. 3) replayed by ONE warp of the cluster leader over the per-step
// summaries (m_t = reference exponent, l_t = block sum, P~V_t at the probe coordinates).
//
// The cost of this warp per step bounds the rate at which a group can stream KV blocks.  The steps are walked in
// order here, but the walk is not inherently serial: only the short recurrence
//     x^(t) = x^(t-1) + (l_t / A_t) (u^(t)[idx] - x^(t-1))
// is carried from step to step (an affine map of x, so a run of steps could also be composed as a parallel prefix:
// DESIGN.md section 11, lead 2, has the measurement of that variant) and the patience counter is a walk over bits;
// everything else (norms, cross-lane sums, sqrt, divide, compare) is independent per step.  The warp therefore takes a BATCH of up to kScanBatch consecutive steps whose
// summaries have arrived, runs the recurrence over them back to back, reduces the 4 x batch partial sums
// with one transposing butterfly (each lane ends up owning one step), evaluates Eq. 2 for all steps of
// the batch in parallel lanes and then walks the patience counter.  The arithmetic per step is exactly
// the sequential algorithm's; a batch of one is the plain loop.
#pragma once
#include "art_common.cuh"

namespace art {

constexpr int kScanBatch = 8;

// Lane layout: the warp's 32 lanes are split into G groups of LPH = 32 / G lanes, one group per head of
// the query group; lane `sub` of a group owns probe components sub, sub + LPH, ...  (CPL of them).
template <int G, int PW>
struct ScanCore {
  static constexpr int LPH = 32 / G;
  static constexpr int CPL = PW / LPH;
  // steps a lane owns after the reduction of a batch of NB steps (1, or 2 when the head has fewer lanes than NB)
  template <int NB> static __host__ __device__ constexpr int kh() { return NB > LPH ? NB / LPH : 1; }
  static constexpr int KH = kh<kScanBatch>();
  static_assert(G == 1 || G == 2 || G == 4 || G == 8, "group size");
  static_assert(PW % LPH == 0, "probe width must split over the lanes of a head");

  float m_run, l_run;       // running reference exponent (log2 domain) and A_t relative to it
  float x[CPL];             // probe of the normalised output, x^(t)
  int cnt;                  // c^(t)
  int g_real = G;           // heads that exist; padding heads (q = 0) never hold the decision back

  __device__ __forceinline__ void init() {
    m_run = kNegInf; l_run = 0.f; cnt = 0;                // c^(0) = 0 (Alg. 1 l.2)
#pragma unroll
    for (int j = 0; j < CPL; ++j) x[j] = 0.f;             // x^(0) = 0 (Alg. 1 l.1)
  }

  // Sums s[k][q] over the LPH lanes of each head.  Afterwards s[j][q], j < KH, holds the complete sums of
  // step owned_step(lane) + j.
  template <int NB, int Q>
  static __device__ __forceinline__ void reduce(float (&s)[NB][Q], int lane) {
    constexpr int KH = kh<NB>();
    int cntk = NB;
#pragma unroll
    for (int m = LPH / 2; m >= 1; m >>= 1) {
      if (cntk > KH) {                                     // transposing round: halve the number of steps held
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
        for (int i = 0; i < KH; ++i)
#pragma unroll
          for (int q = 0; q < Q; ++q) s[i][q] += __shfl_xor_sync(0xffffffffu, s[i][q], m);
      }
    }
  }
  // lane (within its head's LPH lanes) that owns step k after reduce(), and the slot j it sits in
  template <int NB> static __host__ __device__ constexpr int owner_sub(int k) { return NB > LPH ? k / kh<NB>() : k * (LPH / NB); }
  template <int NB> static __host__ __device__ constexpr int owner_slot(int k) { return NB > LPH ? k % kh<NB>() : 0; }

  static __device__ __forceinline__ float sqrt_approx(float v) {
    float r; asm("sqrt.approx.f32 %0, %1;" : "=f"(r) : "f"(v)); return r;
  }
  // Eq. 2 for one head from the complete sums |dx|^2, x_old.dx, |x_old|^2: d_scale = ||dx||,
  // d_direction = 1 - cos(x_new, x_old) evaluated as (|a|^2 |d|^2 - (a.d)^2) / (|a||b| (|a||b| + a.b)), which
  // avoids the cancellation in 1 - cos; the quotient is compared as num < phi * den.  |b|^2 = |a|^2 + 2 a.d +
  // |d|^2.  Zero norm => cos := 0 (R4); strict '<' (R5).
  static __device__ __forceinline__ bool stable_head(const float (&s)[3], float tau, float phi) {
    const float sdd = s[0], sad = s[1], saa = s[2];
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

  // Processes n (1..kScanBatch) consecutive steps.  load_ml(k, mt, lt) / load_pv(k, pv) fetch the summary of
  // the k-th step of the batch for this lane's head / probe components; they are called for every k <
  // kScanBatch with `k < n` as a predicate (the code is branch-free so that the loads of all steps and the
  // independent parts of the arithmetic overlap; a missing step is an empty one and leaves the state as it is).
  // Returns the 0-based index within the batch of the step at which the criterion fired (c >= patience,
  // PAPER.md:157), or -1.
  template <int NB, bool FULL, typename LoadML, typename LoadPV>      // FULL: n == NB, nothing is predicated
  __device__ __forceinline__ int batch_n(int n, int lane, float tau, float phi, int patience, LoadML&& load_ml, LoadPV&& load_pv) {
    // ---- the scalar chain: reference exponent and A_t, r_t = 2^(m_t - m) / A_t
    float lt[NB], r[NB];
#pragma unroll
    for (int k = 0; k < NB; ++k) {
      float mt;
      load_ml(k, FULL || k < n, mt, lt[k]);                // (-inf, 0) when the predicate is false
      const float mn = fmaxf(m_run, mt);
      const float al = (m_run == mn) ? 1.f : fast_exp2(m_run - mn);
      const float be = (mt == kNegInf) ? 0.f : fast_exp2(mt - mn);   // a step with no valid token changes nothing (R8)
      const float l_new = fmaf(al, l_run, be * lt[k]);
      r[k] = (l_new > 0.f) ? __fdividef(be, l_new) : 0.f;
      m_run = mn; l_run = l_new;
    }
    // ---- the recurrence x^(t) = x^(t-1) + r_t (P~V_t - l_t x^(t-1))   (l_t u^(t) = P~V_t)
    float sd[NB][1], sa[NB][2];                              // |dx|^2; (x_old . dx, |x_old|^2)
#pragma unroll
    for (int k = 0; k < NB; ++k) {
      float pv[CPL];
      load_pv(k, FULL || k < n, pv);                       // zeros when the predicate is false
      float sdd = 0.f, sad = 0.f, saa = 0.f;
#pragma unroll
      for (int j = 0; j < CPL; ++j) {
        const float dlt = r[k] * fmaf(-lt[k], x[j], pv[j]);
        sdd = fmaf(dlt, dlt, sdd); sad = fmaf(x[j], dlt, sad); saa = fmaf(x[j], x[j], saa);
        x[j] += dlt;
      }
      sd[k][0] = sdd; sa[k][0] = sad; sa[k][1] = saa;
    }
    constexpr int KH = kh<NB>();
    // A step can only be stable if every head passes the scale test (first half of Eq. 2).  Far from convergence
    // none does, so |dx|^2 is summed over the lanes first and the two sums of the direction test only if needed:
    // two thirds of the shuffles of a batch are saved in the common case, nothing is computed twice.
    reduce<NB, 1>(sd, lane);
    uint32_t pass = 0u;
#pragma unroll
    for (int j = 0; j < KH; ++j) {
      const uint32_t v = __ballot_sync(0xffffffffu, sqrt_approx(sd[j][0]) < tau || (lane / LPH) >= g_real);
#pragma unroll
      for (int k = 0; k < NB; ++k) {
        if (owner_slot<NB>(k) != j) continue;
        uint32_t need = 0;
#pragma unroll
        for (int h = 0; h < G; ++h) need |= 1u << (h * LPH + owner_sub<NB>(k));
        pass |= ((FULL || k < n) && (v & need) == need) ? (1u << k) : 0u;
      }
    }
    if (pass == 0u) { cnt = (n > 0) ? 0 : cnt; return -1; }      // nobody stable: the counter is back at 0 (Eq. 3)
    reduce<NB, 2>(sa, lane);
    float s[KH][3];
#pragma unroll
    for (int j = 0; j < KH; ++j) { s[j][0] = sd[j][0]; s[j][1] = sa[j][0]; s[j][2] = sa[j][1]; }
    uint32_t votes[KH];
#pragma unroll
    for (int j = 0; j < KH; ++j) votes[j] = __ballot_sync(0xffffffffu, stable_head(s[j], tau, phi) || (lane / LPH) >= g_real);
    // far from convergence no step of the batch is stable: the counter is simply back at 0 (Eq. 3)
    bool any = false;
#pragma unroll
    for (int k = 0; k < NB; ++k) {
      uint32_t need = 0;
#pragma unroll
      for (int h = 0; h < G; ++h) need |= 1u << (h * LPH + owner_sub<NB>(k));
      any |= (FULL || k < n) && (votes[owner_slot<NB>(k)] & need) == need;
    }
    if (!any) { cnt = (n > 0) ? 0 : cnt; return -1; }
    int fired = -1;
#pragma unroll
    for (int k = 0; k < NB; ++k) {
      uint32_t need = 0;                                   // the lanes (one per head) that own step k
#pragma unroll
      for (int h = 0; h < G; ++h) need |= 1u << (h * LPH + owner_sub<NB>(k));
      const bool stable = (votes[owner_slot<NB>(k)] & need) == need;     // AND over the group's heads (R2)
      const int c_new = stable ? cnt + 1 : 0;              // Eq. 3
      const bool live = (FULL || k < n) && (fired < 0);
      cnt = live ? c_new : cnt;
      fired = (live && c_new >= patience) ? k : fired;
    }
    return fired;
  }
  // n <= kScanBatch steps: a half-size batch costs half, so short runs of arrived steps are decided sooner
  template <typename LoadML, typename LoadPV>
  __device__ __forceinline__ int batch(int n, int lane, float tau, float phi, int patience, LoadML&& load_ml, LoadPV&& load_pv) {
    if (n <= kScanBatch / 4) return batch_n<kScanBatch / 4, false>(n, lane, tau, phi, patience, load_ml, load_pv);
    if (n <= kScanBatch / 2) return batch_n<kScanBatch / 2, false>(n, lane, tau, phi, patience, load_ml, load_pv);
    if (n == kScanBatch) return batch_n<kScanBatch, true>(n, lane, tau, phi, patience, load_ml, load_pv);
    return batch_n<kScanBatch, false>(n, lane, tau, phi, patience, load_ml, load_pv);
  }
};

}  // namespace art
