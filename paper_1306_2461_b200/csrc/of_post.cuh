// of_post.cuh -- on-device integral quantity of a velocity field (NEXT item f3 of the scope table; eq. 3,
// PAPER.md:127-131): the recirculation-bubble surface S_bubble = share of the available vectors whose
// longitudinal component is <= T_v, with T_v = (min + max)/2 of the MEAN field.  Three streaming kernels
// (4-5 B per pixel, grid-stride, float4 loads): running sum of fields, min/max of a field, thresholded
// count.  Integer atomics only (counts, ordered-integer min/max): results do not depend on the order of
// arrival, so they are bit-reproducible and compared exactly with the oracle.
#pragma once
#include "of_common.cuh"

__global__ void __launch_bounds__(256) kp_accumulate(float *__restrict__ sum, const float *__restrict__ f, size_t n)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) sum[i] += f[i];
}

// order-preserving map float -> unsigned (so that integer min/max = float min/max); NaN is skipped by the caller
__device__ __forceinline__ unsigned f2ord(float x)
{
    const unsigned u = __float_as_uint(x);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__host__ __device__ __forceinline__ float ord2f(unsigned o)
{
    const unsigned u = (o & 0x80000000u) ? (o & 0x7fffffffu) : ~o;
#ifdef __CUDA_ARCH__
    return __uint_as_float(u);
#else
    float f;
    memcpy(&f, &u, 4);
    return f;
#endif
}

__global__ void kp_minmax_init(unsigned *mm) { mm[0] = 0xffffffffu; mm[1] = 0u; }

// mm[0] = ordered min, mm[1] = ordered max over the pixels with valid != 0 (valid may be NULL)
__global__ void __launch_bounds__(256) kp_minmax(const float *__restrict__ f, const uint8_t *__restrict__ valid, size_t n, unsigned *mm)
{
    unsigned lo = 0xffffffffu, hi = 0u;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const float x = f[i];
        if (x == x && (valid == nullptr || valid[i])) {
            const unsigned o = f2ord(x);
            lo = min(lo, o);
            hi = max(hi, o);
        }
    }
    lo = __reduce_min_sync(0xffffffffu, lo);
    hi = __reduce_max_sync(0xffffffffu, hi);
    if ((threadIdx.x & 31) == 0) {
        atomicMin(mm, lo);
        atomicMax(mm + 1, hi);
    }
}

__global__ void kp_minmax_finish(const unsigned *mm, float *out) { out[0] = ord2f(mm[0]); out[1] = ord2f(mm[1]); }

// T_v = (min + max) / 2 of the MEAN field from the min / max of the running SUM of n fields, in fp32: 0.5f * (lo + hi) / n
__global__ void kp_threshold_finish(const unsigned *mm, float n_fields, float *out) { out[0] = 0.5f * (ord2f(mm[0]) + ord2f(mm[1])) / n_fields; }

// cnt[0] = available vectors with vx <= threshold, cnt[1] = available vectors (cnt zeroed before the launch)
// (threshold_dev != NULL: the threshold is read from device memory, so that no step of eq. 3 needs the host)
__global__ void __launch_bounds__(256) kp_bubble_count(const float *__restrict__ vx, const uint8_t *__restrict__ valid, size_t n,
                                                       float threshold, const float *__restrict__ threshold_dev, unsigned long long *cnt)
{
    if (threshold_dev != nullptr) threshold = threshold_dev[0];
    unsigned below = 0, total = 0;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const bool ok = valid == nullptr || valid[i];
        total += ok ? 1u : 0u;
        below += (ok && vx[i] <= threshold) ? 1u : 0u;
    }
    below = __reduce_add_sync(0xffffffffu, below);
    total = __reduce_add_sync(0xffffffffu, total);
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(cnt, (unsigned long long)below);
        atomicAdd(cnt + 1, (unsigned long long)total);
    }
}
