// of_kernels.cuh -- sm_100a device kernels of the dense optical-flow solve (arxiv/paper_1306_2461).
//
// Rows of the scope table:
//   K0 convert_frames        a1   uint8/uint16/fp32 frame -> fp32 internal plane (exact, no scaling)
//   K1 pyramid_down          a2   [1 4 6 4 1]/16 separable low-pass + 2x decimation, fused
//   K4 upsample_flow         a10  u_l = 2*bilinear(u_{l+1}; x/2, y/2)
//   K2 products_hsum         a4-a7 -> of_k2.cuh
//   K3 vsum_solve            a8-a9 -> of_k3.cuh
//
// All internal planes of a level share one pitch (multiple of 32 floats, rows 128-byte aligned).
// Shares no code with oracle/.
#pragma once
#include "of_common.cuh"

// ------------------------------------------------------------------------------------------------
// K0: frame conversion (row a1).  One thread per 4 pixels; src is dense (pitch == W), dst pitched.
// ------------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) k0_convert(const T *__restrict__ srcA, const T *__restrict__ srcB,
                                                  float *__restrict__ dstA, float *__restrict__ dstB,
                                                  int W, int H, int pitch)
{
    const T *__restrict__ src = blockIdx.z ? srcB : srcA;
    float *__restrict__ dst = blockIdx.z ? dstB : dstA;
    int x4 = (blockIdx.x * blockDim.x + threadIdx.x) * 4;
    int y = blockIdx.y;
    if (x4 >= W || src == nullptr) return;
    const T *s = src + (size_t)y * W + x4;
    float *d = dst + (size_t)y * pitch + x4;
    if (x4 + 3 < W) {
        float4 o;
        if (((reinterpret_cast<uintptr_t>(s)) & (4 * sizeof(T) - 1)) == 0) {
            if (sizeof(T) == 1) {
                uchar4 p = *reinterpret_cast<const uchar4 *>(s);
                o = make_float4((float)p.x, (float)p.y, (float)p.z, (float)p.w);
            } else if (sizeof(T) == 2) {
                ushort4 p = *reinterpret_cast<const ushort4 *>(s);
                o = make_float4((float)p.x, (float)p.y, (float)p.z, (float)p.w);
            } else {
                o = *reinterpret_cast<const float4 *>(s);
            }
        } else {
            o = make_float4((float)s[0], (float)s[1], (float)s[2], (float)s[3]);
        }
        *reinterpret_cast<float4 *>(d) = o;
    } else {
        for (int i = 0; x4 + i < W; ++i) d[i] = (float)s[i];
    }
}

// ------------------------------------------------------------------------------------------------
// K1: pyramid step (row a2; "reduced in size by a factor of 4"; D4, D5).
// CTA = 32 x K1_TH outputs; source patch (2*32+3) x (2*K1_TH+3) staged in shared memory with clamped indices,
// rows filtered first, then columns (same order as the definition).
// ------------------------------------------------------------------------------------------------
#define K1_TW 32                                   // (the index arithmetic below relies on K1_TW == 32)
#ifndef K1_TH
#define K1_TH 8
#endif
// T = float: level l -> l+1 of an fp32 pyramid.  T = uint8_t / uint16_t / float with cvtA/cvtB != NULL: the first
// step of a pair, fused with the frame conversion (row a1): the source is the raw dense frame (pitch == W) and
// every CTA also writes the fp32 level-0 plane for the core of its patch (each source pixel belongs to exactly
// one core), so the raw frame is read once and level 0 is never re-read by a separate conversion kernel.
template <typename T>
__global__ void __launch_bounds__(256) k1_pyramid_down(const T *__restrict__ srcA, const T *__restrict__ srcB,
                                                       float *__restrict__ dstA, float *__restrict__ dstB,
                                                       int W, int H, int spitch, int Wd, int Hd, int dpitch,
                                                       float *__restrict__ cvtA, float *__restrict__ cvtB, int cpitch)
{
    const T *__restrict__ src = blockIdx.z ? srcB : srcA;
    float *__restrict__ dst = blockIdx.z ? dstB : dstA;
    float *__restrict__ cvt = blockIdx.z ? cvtB : cvtA;
    __shared__ float patch[2 * K1_TH + 3][2 * K1_TW + 4];
    __shared__ float T_[2 * K1_TH + 3][K1_TW + 1];
    const int X0 = blockIdx.x * K1_TW, Y0 = blockIdx.y * K1_TH;
    const int sx0 = 2 * X0 - 2, sy0 = 2 * Y0 - 2;
    {   // 2-D walk over the patch (no division): thread (tx, ty) loads columns tx, tx+32, tx+64 of rows ty, ty+8, ty+16
        const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
#pragma unroll
        for (int r = ty; r < 2 * K1_TH + 3; r += 8) {
            const int sy = sy0 + r;
            const T *row = src + (size_t)clampi(sy, 0, H - 1) * spitch;
#pragma unroll
            for (int c = tx; c < 2 * K1_TW + 3; c += 32) {
                const int sx = sx0 + c;
                const float val = (float)__ldg(row + clampi(sx, 0, W - 1));
                patch[r][c] = val;
                if (cvt != nullptr && r >= 2 && r < 2 * K1_TH + 2 && c >= 2 && c < 2 * K1_TW + 2 && sx < W && sy < H)
                    cvt[(size_t)sy * cpitch + sx] = val;
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < (2 * K1_TH + 3) * K1_TW; i += 256) {
        int r = i >> 5, X = i & 31;
        const float *p = &patch[r][2 * X];
        float s = 0.0625f * p[0];
        s = fmaf(0.25f, p[1], s);
        s = fmaf(0.375f, p[2], s);
        s = fmaf(0.25f, p[3], s);
        s = fmaf(0.0625f, p[4], s);
        T_[r][X] = s;
    }
    __syncthreads();
    for (int i = threadIdx.x; i < K1_TW * K1_TH; i += 256) {
        const int X = i & (K1_TW - 1), Y = i / K1_TW;
        const int gx = X0 + X, gy = Y0 + Y;
        if (gx < Wd && gy < Hd) {
            float s = 0.0625f * T_[2 * Y][X];
            s = fmaf(0.25f, T_[2 * Y + 1][X], s);
            s = fmaf(0.375f, T_[2 * Y + 2][X], s);
            s = fmaf(0.25f, T_[2 * Y + 3][X], s);
            s = fmaf(0.0625f, T_[2 * Y + 4][X], s);
            dst[(size_t)gy * dpitch + gx] = s;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// K4: flow hand-down (row a10; "used as an initial estimate"; D6).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k4_upsample_flow(const float *__restrict__ uc, const float *__restrict__ vc,
                                                        int Wc, int Hc, int cpitch, float *__restrict__ u,
                                                        float *__restrict__ v, int W, int H, int pitch,
                                                        const uint8_t *__restrict__ mask)   // fine-level obstacle mask or NULL (M3)
{
    int x = blockIdx.x * 64 + (threadIdx.x & 63);
    int y = blockIdx.y * 4 + (threadIdx.x >> 6);
    if (x >= W || y >= H) return;
    int x0 = x >> 1, x1 = min(x0 + 1, Wc - 1), y0 = y >> 1, y1 = min(y0 + 1, Hc - 1);
    float fx = (x & 1) * 0.5f, fy = (y & 1) * 0.5f;
    size_t i00 = (size_t)y0 * cpitch + x0, i01 = (size_t)y0 * cpitch + x1;
    size_t i10 = (size_t)y1 * cpitch + x0, i11 = (size_t)y1 * cpitch + x1;
    float ut = (1.0f - fx) * __ldg(uc + i00) + fx * __ldg(uc + i01);
    float ub = (1.0f - fx) * __ldg(uc + i10) + fx * __ldg(uc + i11);
    float vt = (1.0f - fx) * __ldg(vc + i00) + fx * __ldg(vc + i01);
    float vb = (1.0f - fx) * __ldg(vc + i10) + fx * __ldg(vc + i11);
    const bool fluid = mask == nullptr || mask[(size_t)y * pitch + x] != 0;
    u[(size_t)y * pitch + x] = fluid ? 2.0f * ((1.0f - fy) * ut + fy * ub) : 0.f;
    v[(size_t)y * pitch + x] = fluid ? 2.0f * ((1.0f - fy) * vt + fy * vb) : 0.f;
}

