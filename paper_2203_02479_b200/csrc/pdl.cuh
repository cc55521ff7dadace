// pdl.cuh -- programmatic dependent launch (sm_90+): the kernels of one plane-event are launched with
// cudaLaunchAttributeProgrammaticStreamSerialization, so the CTAs of kernel n+1 become resident while the last wave of
// kernel n drains, do their prologue and block in pdl_wait() until kernel n has completed and flushed.  The 17-20 us
// kernels of configs[1] otherwise lose a quarter of their time to ramp-up and tail.
//   * every kernel launched this way calls pdl_wait() before it reads or writes anything a predecessor touches, and
//     reads such data with plain loads: __ldg / ld.global.nc marks memory invariant for the kernel's lifetime, which lets
//     the compiler hoist the load above the wait (seen on configs[0]: S read before the raster had finished);
//   * a CTA calls pdl_trigger() only once no CTA of its own grid is still waiting to be scheduled (all CTAs of a
//     one-wave grid, else the CTAs of the last wave: blockIdx >= tail_from), so early dependents never take a slot
//     from their predecessor.
#pragma once
#include <cuda_runtime.h>

namespace wcsim {

__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// first linear block index of the last wave of a grid of `ctas` blocks when `resident` of them fit on the device
inline int pdl_tail_from(long long ctas, long long resident) { return ctas > resident ? (int)(ctas - resident) : 0; }

template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

} // namespace wcsim
