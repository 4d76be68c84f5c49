// Read-only streaming ceiling: what this box's HBM delivers to a kernel that only READS, with
// the same access pattern as the attention kernels (32 KiB pieces, TMA bulk copies into a 3-stage shared-memory ring,
// two CTAs per SM) and no compute at all.  MEASURED_PEAKS.json's hbm_gbs is a COPY (read + write); a read-only stream
// can run above it, so the attention kernels' fraction of peak is also reported against this number.
#include "art_common.cuh"
#include "art_host_util.cuh"

namespace art {
namespace probe {

constexpr int kStages = 3;
constexpr uint32_t kPiece = 32768;                       // one KV block of one head: K + V tile

__global__ void __launch_bounds__(32, 2) art_hbm_read_probe_kernel(const uint8_t* __restrict__ buf, unsigned long long pieces) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t sbase = smem_u32(smem);
  const uint32_t bars = sbase + kStages * kPiece;
  if (threadIdx.x == 0) {
    for (int s = 0; s < kStages; ++s) mbar_init(bars + 8u * s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    // pieces are dealt round-robin over the grid; every stage always has a copy in flight
    unsigned long long next = blockIdx.x;
    unsigned long long mine = pieces > blockIdx.x ? (pieces - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    unsigned long long issued = 0, done = 0;
    for (; issued < mine && issued < kStages; ++issued, next += gridDim.x) {
      const uint32_t b = bars + 8u * static_cast<uint32_t>(issued);
      mbar_arrive_expect_tx(b, kPiece);
      tma_load_1d(sbase + static_cast<uint32_t>(issued) * kPiece, buf + next * kPiece, kPiece, b);
    }
    for (; done < mine; ++done) {
      const uint32_t s = static_cast<uint32_t>(done % kStages);
      mbar_wait(bars + 8u * s, static_cast<uint32_t>((done / kStages) & 1));
      if (issued < mine) {
        mbar_arrive_expect_tx(bars + 8u * s, kPiece);
        tma_load_1d(sbase + s * kPiece, buf + next * kPiece, kPiece, bars + 8u * s);
        ++issued; next += gridDim.x;
      }
    }
  }
}

}  // namespace probe
}  // namespace art

extern "C" int art_hbm_read_probe(const void* buf, size_t bytes, void* cuda_stream) {
  using namespace art;
  if (!buf) return ART_ERR_NULL;
  if (reinterpret_cast<uintptr_t>(buf) & 15u) return ART_ERR_ALIGN;
  const unsigned long long pieces = bytes / probe::kPiece;
  if (pieces == 0) return ART_ERR_SHAPE;
  int dev = 0, major = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
      cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) { cudaGetLastError(); return ART_ERR_CUDA; }
  if (major != 10) return ART_ERR_ARCH;
  const uint32_t smem = probe::kStages * probe::kPiece + 64;
  if (prepare_kernel(probe::art_hbm_read_probe_kernel, 1, smem) != cudaSuccess) { cudaGetLastError(); return ART_ERR_CUDA; }
  probe::art_hbm_read_probe_kernel<<<2 * sms, 32, smem, static_cast<cudaStream_t>(cuda_stream)>>>(static_cast<const uint8_t*>(buf), pieces);
  if (cudaGetLastError() != cudaSuccess) return ART_ERR_CUDA;
  return ART_OK;
}
