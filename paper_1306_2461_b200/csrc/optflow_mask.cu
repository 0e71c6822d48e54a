// optflow_mask.cu -- the of_set_mask instantiations (MK = true) of K2, K3 and the persistent solve kernel as a translation unit of
// their own: build.py compiles it in parallel with optflow.cu and optflow_hoist.cu.  Nothing but the entry points of of_dispatch.cuh.
#include "of_dispatch.cuh"

void of_launch_k2_masked(int R_, const K2Params &p, int grid, int threads, size_t smem, cudaStream_t st)
{
    DISPATCH_RB(R_, p.ww.box, (k2_products_hsum<R, true, BX><<<grid, threads, smem, st>>>(p)));
}

void of_launch_k3_masked(int R_, const CUtensorMap &tm, const K3Params &p, int grid, int threads, size_t smem, cudaStream_t st)
{
    DISPATCH_RB(R_, p.ww.box, (k3_vsum_solve<R, true, BX><<<grid, threads, smem, st>>>(tm, p)));
}

cudaError_t of_launch_solve_masked(int R_, const SolveArgs &a, int sms, cudaStream_t st)
{
    cudaError_t e = cudaErrorInvalidValue;
    SolveArgs args_copy = a;
    void *args[] = {&args_copy};
    DISPATCH_RB(R_, a.ww.box, e = cudaLaunchCooperativeKernel((const void *)of_solve_pair<R, true, false, BX>, dim3(sms), dim3(32 * SOLVE_WARPS), args,
                                                   (size_t)SolveSmem<R>::BYTES, st));
    return e;
}

cudaError_t of_setup_attrs_masked(int R_, int smem_max)
{
    cudaError_t e = cudaErrorInvalidValue;
    for (int box = 0; box < 2; ++box) {
        DISPATCH_RB(R_, box, {
            e = cudaFuncSetAttribute(k2_products_hsum<R, true, BX>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(k3_vsum_solve<R, true, BX>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max);
            if (e == cudaSuccess) e = cudaFuncSetAttribute(of_solve_pair<R, true, false, BX>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max);
        });
        if (e != cudaSuccess) return e;
    }
    return e;
}
