// Programmatic dependent launch between the kernels of one pvf_run (the deployment runs event by
// event under a sub-400 us budget, so for small batches the launch gaps and kernel prologues are a large share of the
// time).  A kernel launched with the attribute below may start while its predecessor on the stream is still running;
// everything it does before pdl_wait() -- barrier / TMEM set-up, staging of WEIGHTS (written at pvf_create, never by
// a kernel of the run) -- overlaps the predecessor's tail.  pdl_wait() returns when the predecessor grid has completed
// and its memory is visible; every kernel of the chain executes it (all threads) before touching anything a kernel of
// the same run wrote, so completion is transitive along the chain.  Without the attribute both calls are no-ops.
#pragma once
#include <cuda_runtime.h>

namespace pvf {

__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// cudaLaunchConfig_t with up to two attributes: programmatic stream serialization (pdl) and a cluster dimension.
struct PdlLaunch {
  cudaLaunchConfig_t cfg;
  cudaLaunchAttribute at[2];
  PdlLaunch(dim3 grid, dim3 block, size_t smem, cudaStream_t s, bool pdl, int cluster = 0) {
    cfg = cudaLaunchConfig_t{};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    int n = 0;
    if (cluster > 1) {
      at[n].id = cudaLaunchAttributeClusterDimension;
      at[n].val.clusterDim.x = (unsigned)cluster;
      at[n].val.clusterDim.y = 1;
      at[n].val.clusterDim.z = 1;
      ++n;
    }
    if (pdl) {
      at[n].id = cudaLaunchAttributeProgrammaticStreamSerialization;
      at[n].val.programmaticStreamSerializationAllowed = 1;
      ++n;
    }
    cfg.attrs = at;
    cfg.numAttrs = (unsigned)n;
  }
};

}  // namespace pvf
