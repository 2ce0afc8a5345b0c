// Launch helper shared by the kernel files: programmatic dependent launch for small batches, and the
// first launch error of a call kept for the C-ABI layer (every cudaLaunchKernelEx result is checked).
#pragma once
#include <cuda_runtime.h>

namespace landau {

// first failed launch since the last take_launch_error() on this thread (cudaSuccess if none)
void note_launch_error(cudaError_t e);
cudaError_t take_launch_error();

// Programmatic dependent launch (small batches only, see launch_k): lets the next kernel of the chain be
// scheduled while this one runs; every kernel waits here for its predecessor's results before touching memory.
// Both instructions do nothing in a launch without the attribute.
__device__ __forceinline__ void pdl_prologue() {
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

template <class... KArgs, class... Args>
static void launch_k(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
    note_launch_error(cudaLaunchKernelEx(&cfg, kern, KArgs(args)...));
}
constexpr int PDL_MAX_NB = 8;   // launch-latency bound batches

}  // namespace landau
