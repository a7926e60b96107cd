// pdl.h -- programmatic dependent launch: a kernel launched with pdl_launch may have its CTAs set up while
// the kernel before it in the stream drains, which takes ~2 us off every dependent launch (measured:
// nb_force at N = 16384, N_i = 256: 20.5 -> 16.8 us per call with the pair kernel and the reduction
// launched this way; N = 131072, N_i = 64: 25.9 -> 21.3 us).  The kernel MUST execute pdl_wait() before
// it touches anything an earlier kernel of the stream wrote or still reads; since every kernel launched
// this way waits at its start, completion is transitive along a chain of them.  None of them triggers
// its dependents early (no griddepcontrol.launch_dependents): a dependent grid never takes SM slots from
// a running one.  Launched without the attribute (graph capture of nb_steps' rounds) pdl_wait() is a no-op.
#pragma once
#include "nb_internal.h"

namespace nb {

__device__ __forceinline__ void pdl_wait()
{
#if NB_PDL
    asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
}

template <typename... KArgs, typename... Args>
cudaError_t pdl_launch(void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem, cudaStream_t s, Args&&... args)
{
#if NB_PDL
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
#else
    kernel<<<grid, block, smem, s>>>(static_cast<KArgs>(args)...);
    return cudaGetLastError();
#endif
}

}  // namespace nb
