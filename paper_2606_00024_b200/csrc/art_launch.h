// Launchers of the bf16 tensor-core kernels.  Each group size G is compiled in its own translation unit
// (art_pc_g<G>.cu, art_tc_g<G>.cu) so that the library builds in parallel; art_decode.cu dispatches on G.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include "art_common.cuh"

namespace art {
namespace pc { struct PcParams; }

// persistent-cluster kernel, detector off (art_decode_pc.cuh): NC clusters of CL CTAs; returns a cudaError_t as int
#define ART_DECL_PC(G) \
  int launch_pc_g##G(bool mt, int NC, int CL, uint32_t smem, cudaStream_t stream, const pc::PcParams& p, \
                     const CUtensorMap& tmK, const CUtensorMap& tmV);
ART_DECL_PC(1) ART_DECL_PC(2) ART_DECL_PC(4) ART_DECL_PC(8)
#undef ART_DECL_PC

// static-cluster kernel (art_decode_tc.cuh): one cluster of C CTAs per group
#define ART_DECL_TC(G) \
  int launch_tc_g##G(int mode, bool mt, int groups, int C, uint32_t smem, cudaStream_t stream, const Params& p, \
                     const CUtensorMap& tmK, const CUtensorMap& tmV);                                             \
  int occupancy_tc_g##G(int mode, int C, uint32_t smem);
ART_DECL_TC(1) ART_DECL_TC(2) ART_DECL_TC(4) ART_DECL_TC(8)
#undef ART_DECL_TC

}  // namespace art
