// optflow_hoist.cu -- the of_set_hoist instantiations of the persistent solve kernel without a mask, of_solve_pair<R, false, true>
// (of_solve.cuh), as a translation unit of their own: build.py compiles it in parallel with the others.  The masked ones,
// of_solve_pair<R, true, true>, are in optflow_hoist_mask.cu.  Nothing but the entry points of of_dispatch.cuh.
#include "of_dispatch.cuh"

cudaError_t of_launch_solve_hoisted(int R_, bool mk, const SolveArgs &a, int sms, cudaStream_t st)
{
    if (mk) return of_launch_solve_hoisted_masked(R_, a, sms, st);
    cudaError_t e = cudaErrorInvalidValue;
    SolveArgs args_copy = a;
    void *args[] = {&args_copy};
    DISPATCH_RB(R_, a.ww.box, e = cudaLaunchCooperativeKernel((const void *)of_solve_pair<R, false, true, BX>, dim3(sms), dim3(32 * SOLVE_WARPS), args,
                                                   (size_t)SolveSmem<R>::BYTES, st));
    return e;
}

cudaError_t of_setup_attrs_hoisted(int R_, int smem_max)
{
    cudaError_t e = cudaErrorInvalidValue;
    for (int box = 0; box < 2; ++box) {
        DISPATCH_RB(R_, box, e = cudaFuncSetAttribute(of_solve_pair<R, false, true, BX>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max));
        if (e != cudaSuccess) return e;
    }
    if (e == cudaSuccess) e = of_setup_attrs_hoisted_masked(R_, smem_max);
    return e;
}
