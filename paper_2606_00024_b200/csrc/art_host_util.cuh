// Host-side launch helpers shared by the translation units of the library: per-kernel attribute caching, cluster
// launches, cluster occupancy.  Everything here is `static`: each translation unit keeps its own small caches,
// keyed by (device, kernel), of values that are pure functions of their keys.
#pragma once
#include <array>
#include <map>
#include <mutex>
#include <cuda_runtime.h>
#include <stdint.h>

namespace art {

static inline void set_cluster_attr(cudaLaunchAttribute* attr, int C) {
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = C; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
}

template <typename Kern>
static cudaError_t prepare_kernel_uncached(Kern kern, int C, uint32_t smem_bytes) {
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem_bytes));
  if (e != cudaSuccess) return e;
  // two CTAs per SM need the whole unified L1/shared array configured as shared memory
  e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, static_cast<int>(cudaSharedmemCarveoutMaxShared));
  if (e != cudaSuccess) return e;
  if (C > 8) e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
  return e;
}

// The attribute calls cost a few microseconds each on the host.  They are per-function state, so what has been set
// is remembered per (device, kernel): the dynamic shared memory limit only ever grows (a larger limit than a launch
// needs is harmless), the carveout preference and the non-portable cluster size are set once.
template <typename Kern>
static cudaError_t prepare_kernel(Kern kern, int C, uint32_t smem_bytes) {
  struct State { uint32_t smem = 0; bool nonportable = false; };
  static std::mutex mu;
  static std::map<std::array<uintptr_t, 2>, State> done;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return cudaGetLastError();
  const std::array<uintptr_t, 2> key = {static_cast<uintptr_t>(dev), reinterpret_cast<uintptr_t>(kern)};
  std::lock_guard<std::mutex> lock(mu);
  State& st = done[key];
  if (st.smem >= smem_bytes && (C <= 8 || st.nonportable)) return cudaSuccess;
  const uint32_t want = smem_bytes > st.smem ? smem_bytes : st.smem;
  cudaError_t e = prepare_kernel_uncached(kern, C > 8 || st.nonportable ? 16 : 1, want);
  if (e == cudaSuccess) { st.smem = want; st.nonportable = st.nonportable || C > 8; }
  return e;
}

// grid = clusters x C CTAs, one cluster dimension
template <typename Kern, typename... Args>
static cudaError_t launch_cluster(Kern kern, int threads, int clusters, int C, uint32_t smem_bytes, cudaStream_t stream,
                                  Args... args) {
  cudaError_t e = prepare_kernel(kern, C, smem_bytes);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(static_cast<unsigned>(clusters) * C, 1, 1);
  cfg.blockDim = dim3(threads, 1, 1);
  cfg.dynamicSmemBytes = smem_bytes;
  cfg.stream = stream;
  cudaLaunchAttribute attr[1];
  set_cluster_attr(attr, C);
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, args...);
}

template <typename Kern>
static int max_active_clusters(Kern kern, int threads, int C, uint32_t smem_bytes) {
  if (prepare_kernel(kern, C, smem_bytes) != cudaSuccess) { cudaGetLastError(); return 0; }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(C, 1, 1); cfg.blockDim = dim3(threads, 1, 1); cfg.dynamicSmemBytes = smem_bytes;
  cudaLaunchAttribute attr[1];
  set_cluster_attr(attr, C);
  cfg.attrs = attr; cfg.numAttrs = 1;
  int n = 0;
  if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess) { cudaGetLastError(); return 0; }
  return n;
}

}  // namespace art
