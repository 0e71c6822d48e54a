// of_common.cuh -- small shared definitions of the sm_100a kernels (no arithmetic of the method).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define OFK_MAX_R 16

// Profiling switches of the kernels (phases switched off one by one, profiles/r1_launch_overhead.md) exist in -DOF_PROFILE builds
// only: in the shipped build OF_DBG() is a compile-time 0 and the switches cost neither instructions nor registers.
#ifdef OF_PROFILE
#define OF_DBG(flags, bit) ((flags) & (bit))
#else
#define OF_DBG(flags, bit) 0
#endif

struct WinWeights { float w[2 * OFK_MAX_R + 1]; };   // w[t + R], t = -R..R; passed by value (param bank)

__device__ __forceinline__ int clampi(int i, int lo, int hi) { return max(lo, min(i, hi)); }

// Equal, contiguous share of n work items for CTA `cta` of `ncta` (n * ncta < 2^32).
__host__ __device__ __forceinline__ void cta_range(int n, int cta, int ncta, int &begin, int &end)
{
    begin = (int)((unsigned)n * (unsigned)cta / (unsigned)ncta);
    end = (int)((unsigned)n * (unsigned)(cta + 1) / (unsigned)ncta);
}

// packed fp32 pair FMA with a scalar weight (FFMA2 on sm_100a: half the issue slots of two FFMA)
__device__ __forceinline__ float2 fma2s(float w, float2 x, float2 acc) { return __ffma2_rn(x, make_float2(w, w), acc); }

// ---- obstacle masks (NEXT item f4; readings M1-M5 of DESIGN.md).  Built by the host in
// of_set_mask: per level a byte plane (pitch = the level's float pitch, 0 in the padding, 1 = fluid) and
// compacted work lists, so that a pass only visits tiles / tasks that hold or feed a fluid pixel and the
// remaining work is still split evenly over the CTAs.
struct K3Run { int t0, ntask, chunk_off, pad; };          // consecutive active tasks of one strip owned by one CTA;
                                                          // chunk_off = its first ring chunk, relative to the CTA's pass
struct K3Cta { int ent_b, ent_e, run_b, run_e, nchunks, pad0, pad1, pad2; };   // one CTA's share of a level
struct MaskDesc {                                         // all zero when no mask is set
    const uint8_t *mask;
    const int *k2_list;                                   // active K2 tiles, ascending
    const int2 *k3_ent;                                   // active K3 tasks, ascending: {task, first ring chunk rel. to the CTA's pass}
    const K3Run *k3_runs;
    const K3Cta *k3_cta;                                  // [number of CTAs]
    int k2_n, k3_n;
    const int *zero_list;                                 // level 0 only: K3 tasks without a fluid pixel (their outputs are zero-filled)
    int zero_n, pad;
};
