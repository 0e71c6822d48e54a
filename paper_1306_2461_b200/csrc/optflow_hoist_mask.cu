// optflow_hoist_mask.cu -- of_solve_pair<R, true, true>: of_set_hoist together with of_set_mask (see optflow_hoist.cu).
#include "of_dispatch.cuh"

cudaError_t of_launch_solve_hoisted_masked(int R_, const SolveArgs &a, int sms, cudaStream_t st)
{
    cudaError_t e = cudaErrorInvalidValue;
    SolveArgs args_copy = a;
    void *args[] = {&args_copy};
    DISPATCH_R(R_, e = cudaLaunchCooperativeKernel((const void *)of_solve_pair<R, true, true>, dim3(sms), dim3(32 * SOLVE_WARPS), args,
                                                   (size_t)SolveSmem<R>::BYTES, st));
    return e;
}

cudaError_t of_setup_attrs_hoisted_masked(int R_, int smem_max)
{
    cudaError_t e = cudaErrorInvalidValue;
    DISPATCH_R(R_, e = cudaFuncSetAttribute(of_solve_pair<R, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max));
    return e;
}
