// of_common.cuh -- small shared definitions of the sm_100a kernels (no arithmetic of the method).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define OFK_MAX_R 16

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
