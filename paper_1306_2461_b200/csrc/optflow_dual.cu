// optflow_dual.cu -- the instantiations of the two-pair persistent solve kernel of_solve_dual<R, BX> (of_solve_dual.cuh) as a translation
// unit of their own: build.py compiles it in parallel with the others.  Nothing but the entry points of of_dispatch.cuh.
#include "of_dispatch.cuh"
#include "of_solve_dual.cuh"

cudaError_t of_launch_solve_dual(int R_, const SolveArgs &a0, const SolveArgs &a1, int sms, cudaStream_t st)
{
    cudaError_t e = cudaErrorInvalidValue;
    SolveArgs c0 = a0, c1 = a1;
    void *args[] = {&c0, &c1};
    DISPATCH_RB(R_, a0.ww.box, e = cudaLaunchCooperativeKernel((const void *)of_solve_dual<R, BX>, dim3(sms), dim3(32 * SOLVE_WARPS), args,
                                                               (size_t)SolveSmem<R>::BYTES, st));
    return e;
}

cudaError_t of_setup_attrs_dual(int R_, int smem_max)
{
    cudaError_t e = cudaErrorInvalidValue;
    for (int box = 0; box < 2; ++box) {
        DISPATCH_RB(R_, box, e = cudaFuncSetAttribute(of_solve_dual<R, BX>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max));
        if (e != cudaSuccess) return e;
    }
    return e;
}
