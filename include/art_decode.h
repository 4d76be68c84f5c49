/*
 * art_decode.h -- C ABI of the B200 (sm_100a) ART decode-attention library.
 *
 * ART = Attention Run-time Termination, arXiv 2606.00024.  Citations are
 * "PAPER.md:<line>" (the extracted paper text) plus section / equation.
 *
 * What one call computes (Eq. 1; Algorithm 1;
 * PAPER.md:144 Eq. 2; Eq. 3; PAPER.md:171-173 traversal orders):
 * for every query group (sequence b, KV head g) = the G = Hq/Hkv query heads that
 * share one KV head, walk the eligible 64-token KV blocks in the policy's traversal
 * order; per block compute s = q k^T / sqrt(d), the online-softmax update and P V;
 * after each block evaluate the stability criterion on the probe x^(t) of the
 * NORMALISED intermediate output,
 *     d_scale = ||x^(t) - x^(t-1)||_2 < tau   and   d_direction = 1 - cos(x^(t), x^(t-1)) < phi
 * for ALL heads of the group, count consecutive stable steps, and stop loading KV
 * blocks once the count reaches `patience`.  out = o^(t*), stop_block = t*.
 * The readings taken where the paper is silent (probe = coordinates k*(d/32),
 * AND over heads, sink block first, zero-norm => d_direction = 1, strict '<') are
 * listed in DESIGN.md, "Readings".
 *
 * All functions are re-entrant; the library never allocates or frees device memory and never dereferences a
 * pointer after returning.  Its only global state are three mutex-guarded host-side caches of values that are
 * pure functions of their keys (kernel attributes already set, cluster occupancy, the last few tensor maps
 * keyed by cache base pointer / layout / Hkv).
 * Nothing here falls back to the CPU: on a device that is not sm_100 the calls
 * return ART_ERR_ARCH.
 */
#ifndef ART_DECODE_H_
#define ART_DECODE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ART_VERSION 122          /* 0.2.2: split = 0 always runs static clusters, which are bit-reproducible (same ABI);
                                    0.2.1: art_decode_attention_off_static (no caller workspace); 0.2.0: art_desc_t.num_pages,
                                    ART_SPLIT_PERSISTENT, art_query_clusters, art_hbm_read_probe */
#define ART_BLOCK_TOKENS 64      /* n: tokens per KV block = per cache page */
#define ART_SPLIT_DYNAMIC (-1)   /* art_desc_t.split: persistent clusters, cluster size chosen by the library (BF16, detector
                                    off; a call with the detector on runs the library's static clusters instead) */
#define ART_SPLIT_PERSISTENT(cl) (-1 - (cl))   /* same with clusters of cl = 1..16 CTAs */
#define ART_STATIC_SCRATCH_BYTES (32u << 20) /* size of the library's built-in scratch array (art_decode_attention_off_static) */
#define ART_PATIENCE_INF 2147483647 /* "p = infinity": detector runs, never fires (App. E) */

/* status codes: 0 = OK, negative = error.  No exceptions, no abort. */
enum {
  ART_OK = 0,
  ART_ERR_NULL = -1,      /* a required pointer is NULL */
  ART_ERR_SHAPE = -2,     /* Hq % Hkv != 0, G = Hq / Hkv > 8, q_len * G > 8, unsupported head_dim, block_tokens != 64,
                             negative sizes, split outside ART_SPLIT_PERSISTENT(16)..16, BF16 with max_blocks_per_seq
                             or max_eligible >= 2^24, policy/list mismatch, bad thresholds */
  ART_ERR_DTYPE = -3,     /* dtype / head_dim combination not built (built: F32 d=64, BF16 d=128) */
  ART_ERR_ALIGN = -4,     /* q / k_cache / v_cache not 16-byte aligned */
  ART_ERR_WORKSPACE = -5, /* workspace NULL, misaligned or too small where one is needed (the *_host entry point;
                             split < 0 on a detector-off call) */
  ART_ERR_ARCH = -6,      /* current device is not compute capability 10.x */
  ART_ERR_CUDA = -7,      /* a CUDA runtime call or the launch failed */
  ART_ERR_SCRATCH_LIMIT = -8 /* art_decode_attention_off_static: the problem needs more than ART_STATIC_SCRATCH_BYTES of
                             scratch; use art_decode_attention_off with a caller-provided workspace */
};

enum { ART_DTYPE_F32 = 0, ART_DTYPE_BF16 = 1 };          /* element type of q, k_cache, v_cache */
enum { ART_LAYOUT_HND = 0,  /* cache[page][kv_head][token][d]: one contiguous 16 KiB tile per (page, head) */
       ART_LAYOUT_NHD = 1 };/* cache[page][token][kv_head][d] */
enum { ART_POLICY_DENSE = 0,        /* all blocks, most recent first */
       ART_POLICY_SINK_WINDOW = 1,  /* tokens {j < sink} U {j >= L - window}; block 0 first, then
                                       descending (reading R3) */
       ART_POLICY_LIST = 2 };       /* eligible_blocks walked in the order given */

/* Problem description.  HOST memory, read during the call only. */
typedef struct art_desc {
  int32_t batch;               /* B */
  int32_t num_q_heads;         /* Hq */
  int32_t num_kv_heads;        /* Hkv; query head h uses KV head h / (Hq/Hkv); G = Hq / Hkv must be 1..8 (kernels are
                                  built for 1, 2, 4, 8: other sizes run the next one up with padding heads) */
  int32_t head_dim;            /* d: 64 (F32) or 128 (BF16) */
  int32_t block_tokens;        /* must be 64 */
  int32_t dtype;               /* ART_DTYPE_* */
  int32_t kv_layout;           /* ART_LAYOUT_* */
  int32_t policy;              /* ART_POLICY_* */
  int32_t max_blocks_per_seq;  /* row stride of block_table */
  int32_t sink_tokens;         /* SINK_WINDOW */
  int32_t window_tokens;       /* SINK_WINDOW */
  int32_t max_eligible;        /* row stride of eligible_blocks (LIST) */
  float sm_scale;              /* logit scale; 0 => 1/sqrt(d) (Eq. 1) */
  int32_t split;               /* how CTAs are bound to groups.
                                  1..16 (a power of two for F32): STATIC clusters, one thread-block cluster of that
                                  many CTAs per group, the steps of the group dealt over its CTAs.
                                  ART_SPLIT_DYNAMIC / ART_SPLIT_PERSISTENT(cl) (BF16, detector off): PERSISTENT clusters,
                                  as many as fit the GPU at once; each takes groups from a queue and its CTAs claim
                                  steps of whichever of the cluster's open groups has work left (needs `workspace`).
                                  A detector-on call with split < 0 runs static clusters of the library's choice.
                                  0 = the library decides: static clusters sized so that groups x CTAs fill the GPU
                                  (persistent clusters run only when split < 0 asks for them).
                                  Any value gives the same stop_block as the sequential algorithm. */
  int32_t q_len;               /* m: query tokens per sequence (speculative decode, the tail of a chunked
                                  prefill); 0 or 1 = plain decode.  The m tokens are the LAST m positions of the
                                  sequence (their K/V are in the cache and counted in seq_lens); query token i attends
                                  to the eligible tokens j <= L - m + i; the group walks its blocks once and the
                                  criterion is the AND over all m * G (token, head) rows (reading R15).
                                  m > 1 needs m * G <= 8; q and out are then [B, m, Hq, d]. */
  int32_t num_pages;           /* pages in k_cache / v_cache; 0 = not given.  Only read by debug builds of the library
                                  (-DART_DEBUG), which check every block_table entry a call can reach against it */
  const int32_t* eligible_counts; /* DEVICE [B*Hkv] number of list entries per group (LIST only) */
  int32_t* blocks_loaded;      /* optional DEVICE [B*Hkv] out: KV blocks whose loads were issued
                                  (processed + prefetched-then-discarded): "bytes actually read" / 32 KiB.
                                  BF16 with the detector on: blocks_loaded - stop_block <= C (stages + 3) + 4 for a
                                  group that stops early (C = art_query_split, stages = ring depth, 3 with the default
                                  probe: at most 28 blocks with clusters of 4), 0 for a group that runs to T
                                  (Appendix A.7) */
} art_desc_t;

/* Termination thresholds (tau = 1e-5, phi = 1e-3, p = 5).  HOST memory. */
typedef struct art_thresholds {
  float tau;          /* scale tolerance, compared as d_scale < tau (strict) */
  float phi;          /* direction tolerance, d_direction < phi (strict) */
  int32_t patience;   /* p >= 1; ART_PATIENCE_INF never fires */
  int32_t probe_dim;  /* m: 32 = coordinates k*(d/32) (default); 0 or d = all coordinates */
} art_thresholds_t;

/*
 * ART-on decode attention.  Enqueues on `cuda_stream` (a cudaStream_t, NULL = default
 * stream) and returns; results are valid once the stream has been synchronised.
 *
 *   q               DEVICE [B, Hq, d]            dtype elements, 16-B aligned ([B, m, Hq, d] when q_len = m > 1)
 *   k_cache,v_cache DEVICE paged caches (kv_layout), dtype elements, 16-B aligned
 *   block_table     DEVICE int32 [B, max_blocks_per_seq]  logical block -> physical page
 *   eligible_blocks DEVICE int32 [B, Hkv, max_eligible]   LOGICAL block ids, distinct, walked in the
 *                   order given; NULL unless policy == LIST
 *   seq_lens        DEVICE int32 [B]; tokens >= seq_lens[b] of the last block are masked
 *   thresholds      HOST
 *   out             DEVICE float32 [B, Hq, d]    o^(t*) (Alg. 1 l.18) ([B, m, Hq, d] when q_len = m > 1)
 *   stop_block      DEVICE int32 [B, Hkv]        t* = number of blocks processed, in [0, T];
 *                                                T if the criterion never fired
 *   workspace       DEVICE scratch, 256-B aligned, >= art_workspace_bytes(desc); only the persistent-cluster kernel
 *                   uses it (partial online-softmax states, [group][CTA of the cluster][G][d + 2] floats, written
 *                   before they are read: nothing needs zeroing).  May be NULL unless split < 0 on a detector-off
 *                   call (ART_ERR_WORKSPACE); split >= 0 runs static clusters, which need none
 *
 * seq_lens[b] == 0 or an empty list gives a zero output row and stop_block 0.
 * Reproducibility: stop_block is bit-deterministic for every schedule.  `out` is bit-reproducible with static
 * clusters (steps are dealt round-robin, every CTA merges its steps in order, the partial states are combined in rank
 * order); with persistent clusters CTAs claim steps at run time, which CTA folds which step depends on the run and
 * `out` agrees to fp32 rounding (<= 1e-5 relative) between runs.
 * Device-side contents (page ids in range, list entries valid and distinct, seq_lens within the table) are not
 * validated by the release build; a library built with -DART_DEBUG runs a checking kernel before every launch that
 * records the first violation and traps (tests/test_gpu_debug_build.py).
 */
int art_decode_attention(const art_desc_t* desc, const void* q, const void* k_cache,
                         const void* v_cache, const int32_t* block_table,
                         const int32_t* eligible_blocks, const int32_t* seq_lens,
                         const art_thresholds_t* thresholds, float* out, int32_t* stop_block,
                         void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * ART-off: the same kernel source with the detector compiled out (NOT "patience = inf").
 * out = o^(T) (Eq. 1 over the eligible tokens); stop_block[b, g] = T.
 */
int art_decode_attention_off(const art_desc_t* desc, const void* q, const void* k_cache,
                             const void* v_cache, const int32_t* block_table,
                             const int32_t* eligible_blocks, const int32_t* seq_lens,
                             float* out, int32_t* stop_block,
                             void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * ART-off on persistent clusters WITHOUT a caller workspace, for callers that cannot allocate device memory (code
 * under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Same computation, arguments and
 * results as art_decode_attention_off with split = ART_SPLIT_DYNAMIC (desc->split: 0 or negative; > 0 =
 * ART_ERR_SHAPE, static clusters need no scratch; BF16 only, else ART_ERR_DTYPE), but the partial online-softmax
 * states of the persistent-cluster kernel (art_static_scratch_needed(desc) = B x Hkv x 16 x padded rows x 130 floats,
 * rows = G x q_len padded to 1, 2, 4, 8) live in a file-scope device array of ART_STATIC_SCRATCH_BYTES = 32 MiB inside
 * the library, which every GPU that loads the library holds until the process exits (504 groups of 8 rows, 1008 groups
 * of 4).  A problem that needs more returns ART_ERR_SCRATCH_LIMIT before anything is launched.  The call and
 * everything under it calls no cudaMalloc / cudaFree / allocating library routine; the array's device address is taken
 * once per device (cudaGetSymbolAddress, with the calling thread's current device).
 * ALL calls on a device share the one array, which keeps the previous call's contents: the kernel writes every partial
 * state before it reads it, so nothing has to start at zero, but two calls that overlap on the GPU (different streams,
 * or graph branches that may run concurrently) RACE on it.  Serialise them, or use art_decode_attention_off with
 * separate workspaces.
 */
int art_decode_attention_off_static(const art_desc_t* desc, const void* q, const void* k_cache,
                                    const void* v_cache, const int32_t* block_table,
                                    const int32_t* eligible_blocks, const int32_t* seq_lens,
                                    float* out, int32_t* stop_block, void* cuda_stream);

/* ART_STATIC_SCRATCH_BYTES of the loaded library / scratch bytes this problem would need (0 on a bad desc).
 * Neither needs a CUDA device. */
size_t art_static_scratch_bytes(void);
size_t art_static_scratch_needed(const art_desc_t* desc);

/*
 * End-to-end variants for a serving loop: the per-step inputs (q, block_table,
 * eligible_blocks, eligible_counts, seq_lens) are HOST buffers (pinned for async
 * copies), copied to the device inside the call; out and stop_block are HOST buffers
 * filled before the call returns (the call synchronises the stream).  The KV caches
 * are decode STATE and stay DEVICE pointers.  Pinned inputs are gathered into the workspace by one small kernel
 * (pageable ones by one copy each).  If out / stop_block are pinned (device-accessible) the kernel writes
 * them directly, otherwise they are staged in the workspace and copied back.  desc->eligible_counts is then a HOST
 * pointer; desc->blocks_loaded must be NULL.  `thresholds == NULL` selects ART-off.
 * `workspace` is DEVICE scratch of at least art_workspace_bytes(desc).
 */
int art_decode_attention_host(const art_desc_t* desc, const void* q_host, const void* k_cache,
                              const void* v_cache, const int32_t* block_table_host,
                              const int32_t* eligible_blocks_host, const int32_t* seq_lens_host,
                              const art_thresholds_t* thresholds, float* out_host,
                              int32_t* stop_block_host, void* workspace, size_t workspace_bytes,
                              void* cuda_stream);

/*
 * Base-policy side (scored methods are walked importance-first through "an auxiliary index
 * mapping for indirect addressing"): builds that mapping on the device.
 *   block_scores[b, g, blk] = mean over the G query heads of the group and over the valid tokens (j < L) of block
 *                             blk of q_h . k_j (fp32); -inf for blocks at or beyond ceil(L / 64)
 *   eligible_blocks[b, g, :] = the min(top_k, ceil(L / 64)) blocks with the largest score, in DESCENDING score,
 *                             ties -> lower block index first (reading R10); eligible_counts[b, g] = their number
 * The outputs are what art_decode_attention takes with policy == LIST.  Uses desc->{batch, num_q_heads,
 * num_kv_heads, head_dim, block_tokens, dtype, kv_layout, max_blocks_per_seq (<= 4096), max_eligible (row stride
 * of eligible_blocks, >= top_k), q_len}.  With q_len = m > 1 (q is [B, m, Hq, d]) the LAST query token scores the blocks: the
 * policy's eligible set and order are the group's, computed as for the last token (reading R15).  q, k_cache,
 * block_table, seq_lens as above; block_scores DEVICE float32
 * [B, Hkv, max_blocks_per_seq]; eligible_blocks DEVICE int32 [B, Hkv, max_eligible]; eligible_counts DEVICE
 * int32 [B, Hkv].  Enqueues two kernels on cuda_stream and returns.  Entries beyond the count are not written.
 */
int art_topk_blocks(const art_desc_t* desc, const void* q, const void* k_cache, const int32_t* block_table,
                    const int32_t* seq_lens, int32_t top_k, float* block_scores, int32_t* eligible_blocks,
                    int32_t* eligible_counts, void* cuda_stream);

/* DEVICE scratch bytes that cover every entry point for this problem: the staging area of
 * art_decode_attention_host plus the partial states of the persistent-cluster kernel (BF16: groups x 16 x G x 130
 * floats).  0 on a bad desc.  Needs no CUDA device. */
size_t art_workspace_bytes(const art_desc_t* desc);

/* CTAs per cluster the library would launch for this descriptor (desc->split as given; needs a CUDA device):
 * art_on: 0 = detector off, 1 = probe of 32 coordinates, 2 = full-output detector (probe_dim = 0 or d).
 * <0 = error code. */
int art_query_split(const art_desc_t* desc, int art_on);

/* Number of persistent clusters the library would launch for this problem when given a workspace, 0 if the call
 * runs static clusters (one per group); art_on as above; needs a CUDA device.  <0 = error code. */
int art_query_clusters(const art_desc_t* desc, int art_on);

/* Measurement aid: streams the first floor(bytes / 32768) * 32768 bytes of the DEVICE buffer `buf`
 * (16-byte aligned) through shared memory with the access pattern of the attention kernels (32 KiB TMA bulk copies, a
 * 3-stage ring, two CTAs per SM) and no compute: the time of this call is the read-only HBM ceiling of the box the
 * attention kernels are compared with (bench.py: roofline.read_only_ceiling_gbs).  Enqueues on cuda_stream. */
int art_hbm_read_probe(const void* buf, size_t bytes, void* cuda_stream);

/* Human-readable text for a status code (static storage). */
const char* art_status_string(int status);

/* ART_VERSION of the loaded library. */
int art_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ART_DECODE_H_ */
