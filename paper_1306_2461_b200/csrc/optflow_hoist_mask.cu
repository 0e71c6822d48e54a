// optflow_hoist_mask.cu -- of_solve_pair<R, true, true>: of_set_hoist together with of_set_mask (see optflow_hoist.cu).
#include "of_dispatch.cuh"

cudaError_t of_launch_solve_hoisted_masked(int R_, const SolveArgs &a, int sms, cudaStream_t st)
{
    cudaError_t e = cudaErrorInvalidValue;
    SolveArgs args_copy = a;
    void *args[] = {&args_copy};
    DISPATCH_RB(R_, a.ww.box, e = cudaLaunchCooperativeKernel((const void *)of_solve_pair<R, true, true, BX>, dim3(sms), dim3(32 * SOLVE_WARPS), args,
                                                   (size_t)SolveSmem<R>::BYTES, st));
    return e;
}

cudaError_t of_setup_attrs_hoisted_masked(int R_, int smem_max)
{
    cudaError_t e = cudaErrorInvalidValue;
    for (int box = 0; box < 2; ++box) {
        DISPATCH_RB(R_, box, e = cudaFuncSetAttribute(of_solve_pair<R, true, true, BX>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max));
        if (e != cudaSuccess) return e;
    }
    return e;
}
