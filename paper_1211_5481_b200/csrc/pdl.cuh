// Programmatic dependent launch (PDL) for the kernels of one generation (one stream, no host sync).
//
// A generation is a chain of short dependent kernels (W images -> fitness -> finalize -> GA step); at the small
// configurations (c0, c1, the paper-shaped n1) the gaps between them -- the previous grid draining, the next one being
// launched and running its prologue -- are a large part of the generation.  Every kernel of the chain is launched with
// cudaLaunchAttributeProgrammaticStreamSerialization and follows ONE rule:
//
//     nothing that another kernel writes is read, and nothing is written to global memory, before pdl_wait();
//     pdl_launch_dependents() comes after pdl_wait().
//
// pdl_wait() (griddepcontrol.wait) returns once the preceding grid of the stream has completed and its writes are visible;
// because every thread of every kernel passes its own wait before it can exit, completion is transitive along the chain.
// pdl_launch_dependents() lets the NEXT grid be launched (its blocks become resident where resources allow and park in
// their own wait) once every block of this grid has passed it: launch latency and prologue of kernel n+1 overlap kernel n.
// Both are no-ops for a kernel launched without the attribute.
#pragma once
#include <cuda_runtime.h>

namespace game {

__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// Launch `kernel` on `stream` with programmatic stream serialisation allowed (`pdl` = false: a plain launch).
template <typename... KArgs, typename... Args>
inline cudaError_t launch_chain(bool pdl, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream,
                                Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = pdl ? 1 : 0;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

}  // namespace game
