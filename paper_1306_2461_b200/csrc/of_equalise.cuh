// of_equalise.cuh -- local equalisation pre-filter fused with the frame conversion (NEXT item f1 of the
// scope table; eq. 2; readings E1-E5 in DESIGN.md):
//     In(x,y) = (I - local mean) / local standard deviation   over the in-image part of a (2r+1)^2 box,
//     0 where the local variance is not positive.
// Replaces K0 when of_set_equalisation(h, r > 0): reads the raw uint8 / uint16 / float frame once and
// writes the normalised fp32 level-0 plane.  CTA = 64 x 32 outputs; the raw patch with its halo is staged
// in shared memory, then two separable box passes (rows, columns) of the sums of I and I^2.  Integer
// frames are summed in integer arithmetic (uint32 / uint64), so n*sum(I^2) - sum(I)^2 is exact and the
// flat-neighbourhood decision (variance > 0) is the same as the fp64 oracle's; float frames use fp64 sums.
#pragma once
#include "of_common.cuh"

#define EQ_TW 64
#define EQ_TH 32

template <typename T> struct EqAcc { typedef unsigned int S1; typedef unsigned long long S2; };
template <> struct EqAcc<uint8_t> { typedef unsigned int S1; typedef unsigned int S2; };       // 33^2 * 255^2 < 2^32
template <> struct EqAcc<float> { typedef double S1; typedef double S2; };

#define EQ_HS (EQ_TW + 1)                                   // row stride of the row-sum arrays (odd: spreads the banks)

__host__ __device__ inline size_t eq_smem_bytes(int r, size_t elem)
{
    const size_t pw = EQ_TW + 2 * r, ph = EQ_TH + 2 * r;
    const size_t s1 = elem == 4 ? 8 : 4, s2 = elem == 1 ? 4 : 8;           // sizeof(EqAcc<T>::S1), sizeof(EqAcc<T>::S2)
    return (ph * (pw + 8) * elem + 15) / 16 * 16 + ph * EQ_HS * (s1 + s2) + 16;  // patch (rows of up to pw + 8 values: word-aligned staging) + row sums
}

// RT = the radius as a compile-time constant (the paper's 5: every loop unrolls) or 0 = run-time radius r_arg.
template <typename T, int RT = 0>
__global__ void __launch_bounds__(256) k0_equalise(const T *__restrict__ srcA, const T *__restrict__ srcB,
                                                   float *__restrict__ dstA, float *__restrict__ dstB,
                                                   int W, int H, int pitch, int r_arg)
{
    const int r = RT ? RT : r_arg;
    typedef typename EqAcc<T>::S1 S1;
    typedef typename EqAcc<T>::S2 S2;
    const T *__restrict__ src = blockIdx.z ? srcB : srcA;
    float *__restrict__ dst = blockIdx.z ? dstB : dstA;
    if (src == nullptr) return;
    extern __shared__ __align__(16) unsigned char eq_smem[];
    const int pw = EQ_TW + 2 * r, ph = EQ_TH + 2 * r;
    S2 *h2 = reinterpret_cast<S2 *>(eq_smem);                         // [ph][EQ_HS] row sums of I^2
    S1 *h1 = reinterpret_cast<S1 *>(h2 + (size_t)ph * EQ_HS + (sizeof(S2) == 4 ? (ph & 1) : 0));   // [ph][EQ_HS] row sums of I (8-byte aligned)
    T *patch = reinterpret_cast<T *>(h1 + (size_t)ph * EQ_HS);        // [ph][pw] raw values, 0 outside the image
    const int x0 = blockIdx.x * EQ_TW, y0 = blockIdx.y * EQ_TH;
    // 8-bit frames whose rows are whole words are staged a word at a time: patch row = 80 bytes = columns x0-8 .. x0+71 (20 aligned
    // 4-byte loads instead of 74 byte loads), value (gx, gy) at patch[py * pws + pofs + (gx - x0 + r)]
    const bool vec = sizeof(T) == 1 && r <= 8 && (W & 3) == 0 && (reinterpret_cast<uintptr_t>(src) & 3) == 0;
    const int pws = vec ? EQ_TW + 16 : pw, pofs = vec ? 8 - r : 0;
    if (vec) {
        constexpr int NWORD = (EQ_TW + 16) / 4;
        unsigned *pw32 = reinterpret_cast<unsigned *>(patch);
        for (int i = threadIdx.x; i < ph * NWORD; i += 256) {
            const int py = i / NWORD, wx = i - py * NWORD;
            const int gy = y0 - r + py, gx = x0 - 8 + 4 * wx;
            unsigned word = 0u;
            if (gy >= 0 && gy < H && gx >= 0 && gx < W) word = __ldg(reinterpret_cast<const unsigned *>(src + (size_t)gy * W + gx));
            pw32[i] = word;
        }
    } else {
        for (int py = threadIdx.x >> 5; py < ph; py += 8) {           // a warp per patch row: coalesced, no divisions
            const int gy = y0 - r + py;
            const bool row_ok = gy >= 0 && gy < H;
            const T *srow = src + (size_t)gy * W;
            for (int px = threadIdx.x & 31; px < pw; px += 32) {
                const int gx = x0 - r + px;
                patch[py * pw + px] = (row_ok && gx >= 0 && gx < W) ? __ldg(srow + gx) : T(0);
            }
        }
    }
    __syncthreads();
    // pass 1, along rows: one thread per (patch row, 8 adjacent outputs).  Integer frames slide the box
    // (add the entering value, subtract the leaving one: exact in integers); float frames re-sum every box.
    for (int i = threadIdx.x; i < ph * (EQ_TW / 8); i += 256) {
        const int py = i / (EQ_TW / 8), x8 = (i - py * (EQ_TW / 8)) * 8;
        const T *p = patch + py * pws + pofs + x8;
        S1 s = 0;
        S2 s2 = 0;
#pragma unroll
        for (int d = 0; d <= 2 * r; ++d) {
            const S1 v = (S1)p[d];
            s += v;
            s2 += (S2)v * (S2)v;
        }
        h1[py * EQ_HS + x8] = s;
        h2[py * EQ_HS + x8] = s2;
#pragma unroll
        for (int k = 1; k < 8; ++k) {
            if (sizeof(T) == 4) {
                s = 0;
                s2 = 0;
                for (int d = 0; d <= 2 * r; ++d) {
                    const S1 v = (S1)p[k + d];
                    s += v;
                    s2 += (S2)v * (S2)v;
                }
            } else {
                const S1 a = (S1)p[k + 2 * r], b = (S1)p[k - 1];
                s += a - b;
                s2 += (S2)a * (S2)a - (S2)b * (S2)b;
            }
            h1[py * EQ_HS + x8 + k] = s;
            h2[py * EQ_HS + x8 + k] = s2;
        }
    }
    __syncthreads();
    // pass 2, along columns: one thread per (column, 8 adjacent rows), same sliding rule; then normalise
    {
        const int x = threadIdx.x & (EQ_TW - 1), y8 = (threadIdx.x / EQ_TW) * 8;
        const int gx = x0 + x;
        S1 s = 0;
        S2 s2 = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const int y = y8 + k, gy = y0 + y;
            if (k == 0 || sizeof(T) == 4) {
                s = 0;
                s2 = 0;
#pragma unroll
                for (int d = 0; d <= 2 * r; ++d) {
                    s += h1[(y + d) * EQ_HS + x];
                    s2 += h2[(y + d) * EQ_HS + x];
                }
            } else {
                s += h1[(y + 2 * r) * EQ_HS + x] - h1[(y - 1) * EQ_HS + x];
                s2 += h2[(y + 2 * r) * EQ_HS + x] - h2[(y - 1) * EQ_HS + x];
            }
            if (gx >= W || gy >= H) continue;
            const int n = (min(gx + r, W - 1) - max(gx - r, 0) + 1) * (min(gy + r, H - 1) - max(gy - r, 0) + 1);
            const T c = patch[(y + r) * pws + pofs + x + r];
            float out;
            if (sizeof(T) == 1 && r <= 5) {                                // 8-bit frames, box of at most 11 x 11: every term fits 32 bits
                const unsigned ns2 = (unsigned)n * (unsigned)s2, ss = (unsigned)s * (unsigned)s;   // <= 121 * 121 * 255^2 < 2^30
                const int top = (int)c * n - (int)s;
                out = ns2 > ss ? (float)top * rsqrtf((float)(ns2 - ss)) : 0.f;   // the same integers, hence the same floats, as the 64-bit form
            } else if (sizeof(T) == 4) {                                          // float frames: fp64 moments
                const double num = (double)n * (double)s2 - (double)s * (double)s;
                out = num > 0.0 ? (float)(((double)c * n - (double)s) / sqrt(num)) : 0.f;
            } else {                                                       // integer frames: exact numerators
                const long long num = (long long)n * (long long)s2 - (long long)s * (long long)s;
                const long long top = (long long)c * n - (long long)s;
                out = num > 0 ? (float)top * rsqrtf((float)num) : 0.f;      // MUFU.RSQ, <= 2 ulp; the zero decision is exact
            }
            dst[(size_t)gy * pitch + gx] = out;
        }
    }
}
