// -DART_DEBUG builds only ("Errors": device-side contents are not validated in release builds; a debug
// build traps).  One small kernel in front of every attention launch walks what the call can reach and traps on
//   * seq_lens[b] < 0 or beyond max_blocks_per_seq * 64,
//   * a LIST count outside [0, max_eligible], a list entry outside [0, max_blocks_per_seq), a repeated list entry,
//   * a block_table entry outside [0, num_pages) for any block the traversal visits (when desc.num_pages is given).
// The offending (code, b, g, index, value) is left in a pinned host word first (art_debug_last_violation()).
#pragma once
#include "art_common.cuh"

namespace art {
namespace debug {

enum { V_SEQ_LEN = 1, V_COUNT = 2, V_LIST_RANGE = 3, V_LIST_DUP = 4, V_PAGE = 5 };

__global__ void __launch_bounds__(128) art_validate_inputs_kernel(const Params p, int num_pages, unsigned long long* report) {
  const int group = blockIdx.x, b = group / p.Hkv, g = group % p.Hkv;
  auto fail = [&](int code, int index, int value) {
    if (report && atomicCAS(report, 0ull, 1ull) == 0ull) {
      report[1] = (static_cast<unsigned long long>(code) << 48) | (static_cast<unsigned long long>(static_cast<unsigned>(b) & 0xffffu) << 32) |
                  (static_cast<unsigned long long>(static_cast<unsigned>(g) & 0xffu) << 24) | (static_cast<unsigned>(index) & 0xffffffu);
      report[2] = static_cast<unsigned long long>(static_cast<unsigned>(value));
      __threadfence_system();
    }
    __trap();
  };
  const int L = p.seq_lens[b];
  if (L < 0 || static_cast<long long>(L) > static_cast<long long>(p.max_blocks) * kBlockTokens) fail(V_SEQ_LEN, 0, L);
  int T;
  if (p.policy == ART_POLICY_LIST) {
    T = p.elig_counts[group];
    if (T < 0 || T > p.max_elig) fail(V_COUNT, 0, T);
  } else {
    T = make_trav(p, b, g, L).T;
  }
  const Trav tr = make_trav(p, b, g, L);
  for (int t = 1 + threadIdx.x; t <= T; t += blockDim.x) {
    const int blk = trav_block(tr, t);
    if (p.policy == ART_POLICY_LIST) {
      if (blk < 0 || blk >= p.max_blocks) fail(V_LIST_RANGE, t - 1, blk);
      for (int u = 1; u < t; ++u)                          // O(T^2): a debugging aid
        if (tr.list[u - 1] == blk) fail(V_LIST_DUP, t - 1, blk);
    }
    if (num_pages > 0 && block_mask(p, L, blk) != 0ull) {
      const int page = p.block_table[static_cast<int64_t>(b) * p.max_blocks + blk];
      if (page < 0 || page >= num_pages) fail(V_PAGE, blk, page);
    }
  }
}

}  // namespace debug
}  // namespace art
