// of_kernels.cuh -- sm_100a device kernels of the dense optical-flow solve (arxiv/paper_1306_2461).
//
// Rows of the scope table:
//   K0 convert_frames        a1   uint8/uint16/fp32 frame -> fp32 internal plane (exact, no scaling)
//   K1 pyramid_down          a2   [1 4 6 4 1]/16 separable low-pass + 2x decimation, fused
//   K4 upsample_flow         a10  u_l = 2*bilinear(u_{l+1}; x/2, y/2)
//   K2 products_hsum         a4-a7 bilinear warp of I2, central differences of I1, It, five
//                                 products, horizontal window sum -> five planes
//   K3 vsum_solve            a8-a9 vertical window sum, damped 2x2 solve, clamp, in-place update
//
// All internal planes of a level share one pitch (multiple of 32 floats, rows 128-byte aligned).
// Shares no code with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define OFK_MAX_R 16

struct WinWeights { float w[2 * OFK_MAX_R + 1]; };   // w[t + R], t = -R..R; passed by value (param bank)

__device__ __forceinline__ int clampi(int i, int lo, int hi) { return max(lo, min(i, hi)); }

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
// CTA = 32x8 outputs; source patch (2*32+3) x (2*8+3) staged in shared memory with clamped indices,
// rows filtered first, then columns (same order as the definition).
// ------------------------------------------------------------------------------------------------
#define K1_TW 32
#define K1_TH 8
__global__ void __launch_bounds__(256) k1_pyramid_down(const float *__restrict__ srcA, const float *__restrict__ srcB,
                                                       float *__restrict__ dstA, float *__restrict__ dstB,
                                                       int W, int H, int spitch, int Wd, int Hd, int dpitch)
{
    const float *__restrict__ src = blockIdx.z ? srcB : srcA;
    float *__restrict__ dst = blockIdx.z ? dstB : dstA;
    __shared__ float patch[2 * K1_TH + 3][2 * K1_TW + 4];
    __shared__ float T[2 * K1_TH + 3][K1_TW + 1];
    const int X0 = blockIdx.x * K1_TW, Y0 = blockIdx.y * K1_TH;
    const int sx0 = 2 * X0 - 2, sy0 = 2 * Y0 - 2;
    for (int i = threadIdx.x; i < (2 * K1_TH + 3) * (2 * K1_TW + 3); i += 256) {
        int r = i / (2 * K1_TW + 3), c = i - r * (2 * K1_TW + 3);
        int sy = clampi(sy0 + r, 0, H - 1), sx = clampi(sx0 + c, 0, W - 1);
        patch[r][c] = __ldg(src + (size_t)sy * spitch + sx);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < (2 * K1_TH + 3) * K1_TW; i += 256) {
        int r = i / K1_TW, X = i - r * K1_TW;
        const float *p = &patch[r][2 * X];
        float s = 0.0625f * p[0];
        s = fmaf(0.25f, p[1], s);
        s = fmaf(0.375f, p[2], s);
        s = fmaf(0.25f, p[3], s);
        s = fmaf(0.0625f, p[4], s);
        T[r][X] = s;
    }
    __syncthreads();
    {
        int X = threadIdx.x & (K1_TW - 1), Y = threadIdx.x / K1_TW;
        int gx = X0 + X, gy = Y0 + Y;
        if (gx < Wd && gy < Hd) {
            float s = 0.0625f * T[2 * Y][X];
            s = fmaf(0.25f, T[2 * Y + 1][X], s);
            s = fmaf(0.375f, T[2 * Y + 2][X], s);
            s = fmaf(0.25f, T[2 * Y + 3][X], s);
            s = fmaf(0.0625f, T[2 * Y + 4][X], s);
            dst[(size_t)gy * dpitch + gx] = s;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// K4: flow hand-down (row a10; "used as an initial estimate"; D6).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k4_upsample_flow(const float *__restrict__ uc, const float *__restrict__ vc,
                                                        int Wc, int Hc, int cpitch, float *__restrict__ u,
                                                        float *__restrict__ v, int W, int H, int pitch)
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
    u[(size_t)y * pitch + x] = 2.0f * ((1.0f - fy) * ut + fy * ub);
    v[(size_t)y * pitch + x] = 2.0f * ((1.0f - fy) * vt + fy * vb);
}

// ------------------------------------------------------------------------------------------------
// The five products at one pixel (rows a4-a6).  D8: the integer part of the displacement is added
// to the integer pixel index (x+u is never formed in fp32); D9: gradients of I1, clamped; D10:
// It = I2w - I1 - Ix*u - Iy*v.
// ------------------------------------------------------------------------------------------------
struct Prod5 { float xx, xy, yy, xt, yt; };

__device__ __forceinline__ Prod5 pixel_products(const float *__restrict__ I1, const float *__restrict__ I2,
                                                const float *__restrict__ u, const float *__restrict__ v,
                                                int x, int y, int W, int H, int pitch)
{
    const size_t row = (size_t)y * pitch;
    const float uu = __ldg(u + row + x), vv = __ldg(v + row + x);
    float fu = floorf(uu), fv = floorf(vv);
    const float ax = uu - fu, ay = vv - fv;
    fu = fminf(fmaxf(fu, -1.0e9f), 1.0e9f);
    fv = fminf(fmaxf(fv, -1.0e9f), 1.0e9f);
    const int X = x + (int)fu, Y = y + (int)fv;
    const int xa = clampi(X, 0, W - 1), xb = clampi(X + 1, 0, W - 1);
    const size_t ra = (size_t)clampi(Y, 0, H - 1) * pitch, rb = (size_t)clampi(Y + 1, 0, H - 1) * pitch;
    const float top = (1.0f - ax) * __ldg(I2 + ra + xa) + ax * __ldg(I2 + ra + xb);
    const float bot = (1.0f - ax) * __ldg(I2 + rb + xa) + ax * __ldg(I2 + rb + xb);
    const float I2w = (1.0f - ay) * top + ay * bot;
    const float c = __ldg(I1 + row + x);
    const float Ix = 0.5f * (__ldg(I1 + row + min(x + 1, W - 1)) - __ldg(I1 + row + max(x - 1, 0)));
    const float Iy = 0.5f * (__ldg(I1 + (size_t)min(y + 1, H - 1) * pitch + x) -
                             __ldg(I1 + (size_t)max(y - 1, 0) * pitch + x));
    const float It = I2w - c - Ix * uu - Iy * vv;
    Prod5 p;
    p.xx = Ix * Ix; p.xy = Ix * Iy; p.yy = Iy * Iy; p.xt = Ix * It; p.yt = Iy * It;
    return p;
}

// ------------------------------------------------------------------------------------------------
// K2: warp + gradients + products + horizontal window sum (rows a4-a7).
// CTA = 128 x 16 outputs, 256 threads.  Phase 1: products on (128+2R) x 16 pixels -> shared memory
// (zero outside the image: D12).  Phase 2: each thread sums 8 adjacent outputs of one row for each
// field from registers (8+2R inputs -> 8(2R+1) FMAs).
// ------------------------------------------------------------------------------------------------
#define K2_TW 128
#define K2_TH 16
#define K2_SEG 8
template <int R> struct K2Cfg {
    static constexpr int PW = K2_TW + 2 * R;                       // product columns per row
    static constexpr int NL = (K2_SEG + 2 * R + 3) / 4;            // float4 loads per thread per field
    static constexpr int PITCH = K2_TW - K2_SEG + 4 * NL;          // smem row pitch (multiple of 4)
    static constexpr size_t SMEM = sizeof(float) * 5 * K2_TH * PITCH;
};

template <int R>
__global__ void __launch_bounds__(256) k2_products_hsum(const float *__restrict__ I1, const float *__restrict__ I2,
                                                        const float *__restrict__ u, const float *__restrict__ v,
                                                        float *__restrict__ S, size_t plane, int W, int H, int pitch,
                                                        const WinWeights ww)
{
    typedef K2Cfg<R> C;
    extern __shared__ float4 smem4[];
    float *sm = reinterpret_cast<float *>(smem4);
    const int x0 = blockIdx.x * K2_TW, y0 = blockIdx.y * K2_TH;

    for (int i = threadIdx.x; i < C::PW * K2_TH; i += 256) {
        const int r = i / C::PW, c = i - r * C::PW;
        const int gx = x0 - R + c, gy = y0 + r;
        Prod5 p = {0.f, 0.f, 0.f, 0.f, 0.f};
        if (gx >= 0 && gx < W && gy < H) p = pixel_products(I1, I2, u, v, gx, gy, W, H, pitch);
        float *d = sm + r * C::PITCH + c;
        d[0 * K2_TH * C::PITCH] = p.xx;
        d[1 * K2_TH * C::PITCH] = p.xy;
        d[2 * K2_TH * C::PITCH] = p.yy;
        d[3 * K2_TH * C::PITCH] = p.xt;
        d[4 * K2_TH * C::PITCH] = p.yt;
    }
    __syncthreads();

    const int r = threadIdx.x >> 4, seg = threadIdx.x & 15;
    const int gy = y0 + r, gx = x0 + seg * K2_SEG;
    if (gy >= H || gx >= pitch) return;
#pragma unroll 1
    for (int f = 0; f < 5; ++f) {
        float in[4 * C::NL];
        const float4 *src = reinterpret_cast<const float4 *>(sm + (f * K2_TH + r) * C::PITCH + seg * K2_SEG);
#pragma unroll
        for (int k = 0; k < C::NL; ++k) {
            float4 t = src[k];
            in[4 * k] = t.x; in[4 * k + 1] = t.y; in[4 * k + 2] = t.z; in[4 * k + 3] = t.w;
        }
        float acc[K2_SEG];
#pragma unroll
        for (int j = 0; j < K2_SEG; ++j) acc[j] = 0.f;
#pragma unroll
        for (int t = 0; t <= 2 * R; ++t)
#pragma unroll
            for (int j = 0; j < K2_SEG; ++j) acc[j] = fmaf(ww.w[t], in[j + t], acc[j]);
        float4 *dst = reinterpret_cast<float4 *>(S + f * plane + (size_t)gy * pitch + gx);
        dst[0] = make_float4(acc[0], acc[1], acc[2], acc[3]);
        dst[1] = make_float4(acc[4], acc[5], acc[6], acc[7]);
    }
}

// ------------------------------------------------------------------------------------------------
// K3: vertical window sum + damped 2x2 solve + update (rows a8-a9).
// CTA = 64 x 32 outputs, 256 threads.  Phase 1: (32+2R) rows x 64 columns of the five planes ->
// shared memory (zero outside the image: D12).  Phase 2: each thread owns one column and 8 rows:
// 8+2R inputs per field stream through registers into 8 accumulators; then the solve (D14, D15).
// ------------------------------------------------------------------------------------------------
#define K3_TW 64
#define K3_TH 32
#define K3_SEG 8
template <int R> struct K3Cfg {
    static constexpr int ROWS = K3_TH + 2 * R;
    static constexpr size_t SMEM = sizeof(float) * 5 * ROWS * K3_TW;
};

struct SolveParams { float eps_half; float max_step; };

template <int R>
__global__ void __launch_bounds__(256) k3_vsum_solve(const float *__restrict__ S, size_t plane,
                                                     const float *u_in, const float *v_in,   // may alias u_out, v_out
                                                     float *u_out, float *v_out, int out_pitch,
                                                     uint8_t *__restrict__ valid, float *__restrict__ det,
                                                     int W, int H, int pitch, const WinWeights ww, const SolveParams sp)
{
    typedef K3Cfg<R> C;
    extern __shared__ float4 smem4[];
    float *sm = reinterpret_cast<float *>(smem4);
    const int x0 = blockIdx.x * K3_TW, y0 = blockIdx.y * K3_TH;

    // phase 1: 16 float4 per row
    for (int i = threadIdx.x; i < 5 * C::ROWS * (K3_TW / 4); i += 256) {
        const int c4 = i & 15, rr = i >> 4;
        const int f = rr / C::ROWS, r = rr - f * C::ROWS;
        const int gy = y0 - R + r, gx = x0 + 4 * c4;
        float4 t = make_float4(0.f, 0.f, 0.f, 0.f);
        if (gy >= 0 && gy < H && gx < pitch)
            t = __ldg(reinterpret_cast<const float4 *>(S + f * plane + (size_t)gy * pitch + gx));
        reinterpret_cast<float4 *>(sm)[i] = t;
    }
    __syncthreads();

    const int c = threadIdx.x & 63, g = threadIdx.x >> 6;
    const int gx = x0 + c;
    if (gx >= W) return;
    float acc[5][K3_SEG];
#pragma unroll
    for (int f = 0; f < 5; ++f) {
#pragma unroll
        for (int j = 0; j < K3_SEG; ++j) acc[f][j] = 0.f;
        const float *col = sm + (f * C::ROWS + g * K3_SEG) * K3_TW + c;
#pragma unroll
        for (int r = 0; r < K3_SEG + 2 * R; ++r) {
            const float val = col[r * K3_TW];
#pragma unroll
            for (int j = 0; j < K3_SEG; ++j) {
                const int t = r - j;
                if (t >= 0 && t <= 2 * R) acc[f][j] = fmaf(ww.w[t], val, acc[f][j]);
            }
        }
    }
#pragma unroll
    for (int j = 0; j < K3_SEG; ++j) {
        const int gy = y0 + g * K3_SEG + j;
        if (gy >= H) break;
        const size_t k = (size_t)gy * pitch + gx;
        const float a = acc[0][j], b = acc[1][j], cc = acc[2][j], p = acc[3][j], q = acc[4][j];
        const float uu = u_in[k], vv = v_in[k];
        const float tr = a + cc;
        float du = 0.f, dv = 0.f;
        if (tr > 0.f) {
            const float lam = sp.eps_half * tr;
            const float A = a + lam, Cc = cc + lam;
            const float D = A * Cc - b * b;
            const float rp = -(p + a * uu + b * vv);
            const float rq = -(q + b * uu + cc * vv);
            du = (Cc * rp - b * rq) / D;
            dv = (A * rq - b * rp) / D;
            du = fminf(fmaxf(du, -sp.max_step), sp.max_step);
            dv = fminf(fmaxf(dv, -sp.max_step), sp.max_step);
        }
        const size_t ko = (size_t)gy * out_pitch + gx;
        u_out[ko] = uu + du;
        v_out[ko] = vv + dv;
        if (valid) valid[(size_t)gy * W + gx] = tr > 0.f ? 1 : 0;
        if (det) det[k] = a * cc - b * b;
    }
}
