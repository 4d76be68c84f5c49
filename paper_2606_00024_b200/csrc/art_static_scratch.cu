// art_decode_attention_off_static: the detector-off decode attention on persistent clusters (art_decode_pc.cuh) for
// callers that cannot allocate device memory at all (CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc) and therefore cannot provide the `workspace` the persistent-cluster kernel needs for its partial
// online-softmax states.  Here that scratch is a file-scope device array of a fixed, modest size that every GPU which
// loads the library holds until the process exits.
//
// The array's NAME is a host-side stand-in in host code, not a device address: its address on the current device is
// taken once per device with cudaGetSymbolAddress (return code checked) and handed to the kernel through the existing
// entry point as its workspace.  Nothing in this file, and nothing on the path it calls, allocates or frees memory.
#include <cuda_runtime.h>

#include <mutex>

#include "art_decode.h"

namespace {

// partial states: [group][CTA of the cluster: 16][padded rows of the group][head_dim + 2] floats
__device__ __align__(256) unsigned char g_static_scratch[ART_STATIC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
void* g_scratch_ptr[kMaxDevices] = {};          // device address of g_static_scratch, per device ordinal

// the device address of the array on the CURRENT device (set-up: once per device), nullptr on error
void* scratch_on_current_device() {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) { cudaGetLastError(); return nullptr; }
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_ptr[dev]) {
    void* ptr = nullptr;
    if (cudaGetSymbolAddress(&ptr, g_static_scratch) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    g_scratch_ptr[dev] = ptr;
  }
  return g_scratch_ptr[dev];
}

inline int padded_rows(int rows) { return rows <= 1 ? 1 : (rows <= 2 ? 2 : (rows <= 4 ? 4 : 8)); }

}  // namespace

extern "C" {

size_t art_static_scratch_bytes(void) { return ART_STATIC_SCRATCH_BYTES; }

size_t art_static_scratch_needed(const art_desc_t* d) {
  if (!d || d->batch < 0 || d->num_kv_heads <= 0 || d->num_q_heads <= 0 || d->num_q_heads % d->num_kv_heads) return 0;
  const int rows = (d->num_q_heads / d->num_kv_heads) * (d->q_len > 1 ? d->q_len : 1);
  if (rows > 8) return 0;
  return static_cast<size_t>(d->batch) * static_cast<size_t>(d->num_kv_heads) * 16u *
         static_cast<size_t>(padded_rows(rows)) * (128u + 2u) * 4u;
}

int art_decode_attention_off_static(const art_desc_t* desc, const void* q, const void* k_cache, const void* v_cache,
                                    const int32_t* block_table, const int32_t* eligible_blocks,
                                    const int32_t* seq_lens, float* out, int32_t* stop_block, void* cuda_stream) {
  if (!desc) return ART_ERR_NULL;
  if (desc->dtype != ART_DTYPE_BF16) return ART_ERR_DTYPE;        // only the bf16 persistent-cluster kernel uses scratch
  if (desc->split > 0) return ART_ERR_SHAPE;                      // static clusters need no scratch: use art_decode_attention_off
  if (desc->num_kv_heads <= 0 || desc->num_q_heads <= 0 || desc->num_q_heads % desc->num_kv_heads || desc->batch < 0)
    return ART_ERR_SHAPE;
  const int rows = (desc->num_q_heads / desc->num_kv_heads) * (desc->q_len > 1 ? desc->q_len : 1);
  if (rows > 8) return ART_ERR_SHAPE;
  if (art_static_scratch_needed(desc) > ART_STATIC_SCRATCH_BYTES) return ART_ERR_SCRATCH_LIMIT;
  void* scratch = scratch_on_current_device();
  if (!scratch) return ART_ERR_CUDA;
  art_desc_t d = *desc;
  if (d.split == 0) d.split = ART_SPLIT_DYNAMIC;                  // always persistent clusters
  return art_decode_attention_off(&d, q, k_cache, v_cache, block_table, eligible_blocks, seq_lens, out, stop_block,
                                  scratch, ART_STATIC_SCRATCH_BYTES, cuda_stream);
}

}  // extern "C"
