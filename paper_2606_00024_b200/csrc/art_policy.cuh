// Base-policy side of the path: the "auxiliary index mapping for indirect addressing" of the
// scored policies built on the GPU, so that the eligible-block list need not come from the host.
//
//   art_block_scores_kernel   score[b, g, blk] = mean over the group's G heads and the block's valid tokens of
//                             q_h . k_j  =  (sum_h q_h) . (sum_j k_j) / (G n_valid).  HBM-bound: every K row of the
//                             cache is read once, 16 bytes per lane, one warp per block.
//   art_topk_kernel           per (b, g): the top_k blocks by DESCENDING score, ties -> lower block index first
//                             (reading R10): bitonic sort of (score, index) keys in shared memory.
#pragma once
#include "art_common.cuh"

namespace art {
namespace policy {

constexpr int kScoreWarps = 8;                 // blocks scored per CTA
constexpr int kMaxSortBlocks = 4096;           // candidates per group the top-k kernel sorts (32 KiB of keys)

struct ScoreParams {
  const void* q;
  const uint8_t* k;
  const int32_t* block_table;
  const int32_t* seq_lens;
  float* scores;                               // [B, Hkv, max_blocks]
  int32_t batch, Hq, Hkv, Gr, max_blocks, layout;   // Gr: real heads per group (the template G is its power-of-two ceiling)
  int32_t qlen;                                // query tokens per sequence (R15): the LAST one scores the blocks
  int64_t page_stride, head_stride, token_stride;   // bytes
};

template <typename T> struct Elem;
template <> struct Elem<float> {
  static constexpr int kPer16 = 4;
  static __device__ __forceinline__ void unpack(const uint4 v, float (&f)[4]) {
    f[0] = __uint_as_float(v.x); f[1] = __uint_as_float(v.y); f[2] = __uint_as_float(v.z); f[3] = __uint_as_float(v.w);
  }
};
template <> struct Elem<__nv_bfloat16> {
  static constexpr int kPer16 = 8;
  static __device__ __forceinline__ void unpack(const uint4 v, float (&f)[8]) {
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) { f[2 * i] = __uint_as_float(w[i] << 16); f[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u); }
  }
};

// One warp per (group, block).  A token row is 256 bytes = 16 chunks of 16 bytes; lane l reads chunk l % 16 of
// rows l / 16, l / 16 + 2, ...  (two rows per warp-wide load, fully coalesced) and keeps the matching 16 bytes of
// sum_h q_h in registers.
template <typename T, int D, int G>
__global__ void __launch_bounds__(kScoreWarps * 32) art_block_scores_kernel(const ScoreParams p) {
  constexpr int E = Elem<T>::kPer16;
  static_assert(D * sizeof(T) == kRowBytes, "a token row is 256 bytes");
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int group = blockIdx.x;
  const int b = group / p.Hkv, g = group % p.Hkv;
  const int blk = blockIdx.y * kScoreWarps + warp;
  const int L = p.seq_lens[b];
  const int nb = (L + kBlockTokens - 1) / kBlockTokens;
  if (blk >= p.max_blocks) return;
  float* out = p.scores + (static_cast<int64_t>(b) * p.Hkv + g) * p.max_blocks + blk;
  if (blk >= nb) { if (lane == 0) *out = kNegInf; return; }            // not a candidate
  const int chunk = lane & 15;
  float qs[E];
#pragma unroll
  for (int e = 0; e < E; ++e) qs[e] = 0.f;
  // q is [B, m, Hq, D]; the policy is the group's, computed as for the last query token (reading R15)
  const T* qp = reinterpret_cast<const T*>(p.q) + ((static_cast<int64_t>(b) * p.qlen + (p.qlen - 1)) * p.Hq + g * p.Gr) * D;
#pragma unroll
  for (int h = 0; h < G; ++h) {
    if (h >= p.Gr) break;
    float f[E];
    Elem<T>::unpack(*reinterpret_cast<const uint4*>(qp + h * D + chunk * E), f);
#pragma unroll
    for (int e = 0; e < E; ++e) qs[e] += f[e];
  }
  const int page = p.block_table[static_cast<int64_t>(b) * p.max_blocks + blk];
  const uint8_t* base = p.k + page * p.page_stride + g * p.head_stride + chunk * 16;
  const int n_valid = min(kBlockTokens, L - blk * kBlockTokens);
  float acc = 0.f;
#pragma unroll 8
  for (int r = lane >> 4; r < kBlockTokens; r += 2) {
    if (r < n_valid) {                                                 // rows >= L may hold anything (R8)
      float f[E];
      Elem<T>::unpack(__ldg(reinterpret_cast<const uint4*>(base + r * p.token_stride)), f);
#pragma unroll
      for (int e = 0; e < E; ++e) acc = fmaf(f[e], qs[e], acc);
    }
  }
#pragma unroll
  for (int m = 16; m >= 1; m >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, m);
  if (lane == 0) *out = acc / static_cast<float>(p.Gr * n_valid) + 0.f;   // + 0: -0 and +0 are the same score
}

struct TopkParams {
  const float* scores;                         // [B, Hkv, max_blocks]
  const int32_t* seq_lens;
  int32_t* lists;                              // [B, Hkv, max_elig]
  int32_t* counts;                             // [B, Hkv]
  int32_t Hkv, max_blocks, max_elig, top_k;
};

// key: larger = earlier in the list.  High word: the score mapped to an unsigned that orders like the float;
// low word: ~index, so that among equal scores the LOWER block index sorts first (R10).
__device__ __forceinline__ unsigned long long rank_key(float score, int idx) {
  uint32_t u = __float_as_uint(score);
  u = (u & 0x80000000u) ? ~u : (u | 0x80000000u);
  return (static_cast<unsigned long long>(u) << 32) | static_cast<uint32_t>(~static_cast<uint32_t>(idx));
}

// One CTA per (b, g): bitonic sort, descending, of n (padded to a power of two <= kMaxSortBlocks) keys.
__global__ void __launch_bounds__(256) art_topk_kernel(const TopkParams p) {
  extern __shared__ unsigned long long keys[];
  const int group = blockIdx.x;
  const int b = group / p.Hkv;
  const int L = p.seq_lens[b];
  const int nb = min((L + kBlockTokens - 1) / kBlockTokens, p.max_blocks);
  int n = 1;
  while (n < nb) n <<= 1;
  const float* sc = p.scores + static_cast<int64_t>(group) * p.max_blocks;
  for (int i = threadIdx.x; i < n; i += blockDim.x) keys[i] = (i < nb) ? rank_key(sc[i], i) : 0ull;   // padding sorts last
  __syncthreads();
  for (int size = 2; size <= n; size <<= 1) {
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      for (int i = threadIdx.x; i < (n >> 1); i += blockDim.x) {
        const int lo = 2 * i - (i & (stride - 1));          // partner pairs (lo, lo + stride)
        const int hi = lo + stride;
        const bool desc = (lo & size) == 0;                  // direction of this bitonic sequence
        const unsigned long long a = keys[lo], c = keys[hi];
        if ((a < c) == desc) { keys[lo] = c; keys[hi] = a; }
      }
      __syncthreads();
    }
  }
  const int k = min(p.top_k, nb);
  int32_t* out = p.lists + static_cast<int64_t>(group) * p.max_elig;
  for (int i = threadIdx.x; i < k; i += blockDim.x) out[i] = static_cast<int32_t>(~static_cast<uint32_t>(keys[i] & 0xffffffffull));
  if (threadIdx.x == 0) p.counts[group] = k;
}

}  // namespace policy
}  // namespace art
