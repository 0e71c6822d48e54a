// of_k3.cuh -- K3: vertical window sum + damped 2x2 solve + in-place (u,v) update (rows a8-a9 of the
// scope table; BASELINE.json:5 "(3) Vertical-sum+solve kernel"; readings D11-D15 of DESIGN.md).
//
// Persistent, one CTA per SM, TMA-fed ring (sm_100a):
//   * the image is cut into 64-column strips x 8-row blocks = "tasks"; task order is strip-major and
//     every CTA owns an equal, contiguous run of tasks (grid = number of SMs, no tail wave);
//   * the five horizontally summed planes are ONE 3-D tensor (x, y, field); a chunk = box of
//     64 x 8 x 5 floats (10 KB) fetched by a single cp.async.bulk.tensor into a shared-memory ring of
//     2*NW + NC - 1 chunks; rows above/below the image are zero-filled by the TMA unit, which IS the
//     zero extension of the window (D12) -- no border code;
//   * step s: NW warps each take one task (8 rows x 64 columns; lane = 2 adjacent columns) while the
//     chunks of step s+1 are in flight; one mbarrier per step parity, one __syncthreads per step;
//   * per lane: (8+2R) LDS.64 per field feed 8*(2R+1) FFMA2 (packed fp32 pair FMA, scalar weight);
//     then the damped 2x2 solve on the pair (D14), clamp (D15), update, validity byte.
// Direct (2R+1)-tap sums, fixed order, no atomics: bit-reproducible (H8), no cancellation (H2).
#pragma once
#include "of_common.cuh"
#include <cuda.h>

#define K3_CHUNK_BYTES (64 * 8 * 5 * 4)
#define K3_MAX_NW 9

template <int R> struct K3Geom {
    static constexpr int NIN = 8 + 2 * R;                // input rows per task
    static constexpr int NC = (NIN + 7) / 8;             // chunks spanned by one task
    __host__ __device__ static constexpr int ring(int nw) { return 2 * nw + NC - 1; }
    __host__ __device__ static constexpr int smem_bytes(int nw) { return ring(nw) * K3_CHUNK_BYTES + 64; }
};

struct SolveParams { float eps_half; float max_step; };

struct K3Params {
    const float *u_in, *v_in;        // may alias u_out, v_out (same pitch when aliased)
    float *u_out, *v_out;
    uint8_t *valid;                  // dense H x W bytes or NULL
    float *det;                      // pitched plane or NULL
    int W, H, pitch, out_pitch;
    int nrb, ntasks;                 // row blocks per strip; ntasks = nstrips * nrb
    WinWeights ww;
    SolveParams sp;
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap *tm, int x, int y, int z, uint32_t bar)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(dst), "l"(tm), "r"(x), "r"(y), "r"(z), "r"(bar) : "memory");
}

// a - b on a pair with one packed instruction
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return fma2s(-1.0f, b, a); }

// Damped 2x2 solve on a pair of pixels (D14, D15): returns the increment, the validity flags and the
// undamped determinant.  tr = a + c is a sum of non-negative terms, so tr > 0 is precision-independent.
__device__ __forceinline__ void k3_solve_pair(float2 a, float2 b, float2 c, float2 p, float2 q, float2 u, float2 v,
                                              const SolveParams sp, float2 &du, float2 &dv, float2 &tr, float2 &det)
{
    tr = __fadd2_rn(a, c);
    const float2 lam = __fmul2_rn(tr, make_float2(sp.eps_half, sp.eps_half));
    const float2 A = __fadd2_rn(a, lam), C = __fadd2_rn(c, lam);
    const float2 bb = __fmul2_rn(b, b);
    const float2 D = sub2(__fmul2_rn(A, C), bb);
    det = sub2(__fmul2_rn(a, c), bb);
    const float2 sp_ = __ffma2_rn(b, v, __ffma2_rn(a, u, p));       // -rp
    const float2 sq_ = __ffma2_rn(c, v, __ffma2_rn(b, u, q));       // -rq
    const float2 nu = sub2(__fmul2_rn(b, sq_), __fmul2_rn(C, sp_)); // C*rp - b*rq
    const float2 nv = sub2(__fmul2_rn(b, sp_), __fmul2_rn(A, sq_)); // A*rq - b*rp
    const float2 inv = make_float2(__fdividef(1.0f, D.x), __fdividef(1.0f, D.y));
    du = __fmul2_rn(nu, inv);
    dv = __fmul2_rn(nv, inv);
    const float ms = sp.max_step;
    du.x = tr.x > 0.f ? fminf(fmaxf(du.x, -ms), ms) : 0.f;
    du.y = tr.y > 0.f ? fminf(fmaxf(du.y, -ms), ms) : 0.f;
    dv.x = tr.x > 0.f ? fminf(fmaxf(dv.x, -ms), ms) : 0.f;
    dv.y = tr.y > 0.f ? fminf(fmaxf(dv.y, -ms), ms) : 0.f;
}

template <int R>
__global__ void __launch_bounds__(32 * K3_MAX_NW, 1) k3_vsum_solve(const __grid_constant__ CUtensorMap tmS, const K3Params p)
{
    typedef K3Geom<R> G;
    extern __shared__ __align__(1024) unsigned char k3_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, NW = blockDim.x >> 5;
    const int RING = G::ring(NW);
    const uint32_t ring0 = smem_u32(k3_smem);
    const uint32_t bar0 = ring0 + RING * K3_CHUNK_BYTES;
    if (threadIdx.x == 0) {
        mbar_init(bar0, 1);
        mbar_init(bar0 + 8, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int W = p.W, H = p.H, pitch = p.pitch, nrb = p.nrb;
    const int t_begin = (int)((long long)p.ntasks * blockIdx.x / gridDim.x);
    const int t_end = (int)((long long)p.ntasks * (blockIdx.x + 1) / gridDim.x);
    uint32_t g = 0;                                                   // step counter: barrier g&1, parity (g>>1)&1

    for (int t = t_begin; t < t_end;) {
        const int strip = t / nrb, rb0 = t - strip * nrb;
        const int ntask = min(nrb - rb0, t_end - t);
        const int total = ntask + G::NC - 1;                           // chunks of this segment
        const int x0 = strip * 64, yc0 = 8 * rb0 - R;                  // chunk c holds rows yc0+8c .. +7
        const int nsteps = (ntask + NW - 1) / NW;
        if (threadIdx.x == 0) {
            const int n = min(NW + G::NC - 1, total);
            const uint32_t bar = bar0 + 8 * (g & 1);
            mbar_expect_tx(bar, n * K3_CHUNK_BYTES);
            for (int c = 0; c < n; ++c) tma_load_3d(ring0 + (c % RING) * K3_CHUNK_BYTES, &tmS, x0, yc0 + 8 * c, 0, bar);
        }
        for (int s = 0; s < nsteps; ++s, ++g) {
            if (threadIdx.x == 0 && s + 1 < nsteps) {
                const int c_lo = NW * (s + 1) + G::NC - 1, c_hi = min(c_lo + NW, total);
                const uint32_t bar = bar0 + 8 * ((g + 1) & 1);
                mbar_expect_tx(bar, (c_hi - c_lo) * K3_CHUNK_BYTES);
                for (int c = c_lo; c < c_hi; ++c) tma_load_3d(ring0 + (c % RING) * K3_CHUNK_BYTES, &tmS, x0, yc0 + 8 * c, 0, bar);
            }
            const int task = s * NW + warp;
            const int gx = x0 + 2 * lane, gy0 = 8 * (rb0 + task);
            const bool active = task < ntask && gx < W;
            // this lane's field values (issued before the wait: their latency hides behind it)
            float2 uu[8], vv[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                uu[j] = make_float2(0.f, 0.f);
                vv[j] = make_float2(0.f, 0.f);
                if (active && gy0 + j < H) {
                    uu[j] = *reinterpret_cast<const float2 *>(p.u_in + (size_t)(gy0 + j) * pitch + gx);
                    vv[j] = *reinterpret_cast<const float2 *>(p.v_in + (size_t)(gy0 + j) * pitch + gx);
                }
            }
            mbar_wait(bar0 + 8 * (g & 1), (g >> 1) & 1);
            if (active) {
                const unsigned char *cb[G::NC];
#pragma unroll
                for (int k = 0; k < G::NC; ++k) cb[k] = k3_smem + ((task + k) % RING) * K3_CHUNK_BYTES + lane * 8;
                float2 acc[5][8];
#pragma unroll
                for (int f = 0; f < 5; ++f)
#pragma unroll
                    for (int j = 0; j < 8; ++j) acc[f][j] = make_float2(0.f, 0.f);
#pragma unroll
                for (int r = 0; r < G::NIN; ++r) {
#pragma unroll
                    for (int f = 0; f < 5; ++f) {
                        const float2 val = *reinterpret_cast<const float2 *>(cb[r >> 3] + f * 2048 + (r & 7) * 256);
#pragma unroll
                        for (int j = 0; j < 8; ++j)
                            if (r - j >= 0 && r - j <= 2 * R) acc[f][j] = fma2s(p.ww.w[r - j], val, acc[f][j]);
                    }
                }
                const bool pair_ok = gx + 1 < W;
                const bool vec_out = (p.out_pitch & 1) == 0 && pair_ok;
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int gy = gy0 + j;
                    if (gy < H) {
                        float2 du, dv, tr, det;
                        k3_solve_pair(acc[0][j], acc[1][j], acc[2][j], acc[3][j], acc[4][j], uu[j], vv[j], p.sp, du, dv, tr, det);
                        const float2 un = __fadd2_rn(uu[j], du), vn = __fadd2_rn(vv[j], dv);
                        float *uo = p.u_out + (size_t)gy * p.out_pitch + gx, *vo = p.v_out + (size_t)gy * p.out_pitch + gx;
                        if (vec_out) {
                            *reinterpret_cast<float2 *>(uo) = un;
                            *reinterpret_cast<float2 *>(vo) = vn;
                        } else {
                            uo[0] = un.x; vo[0] = vn.x;
                            if (pair_ok) { uo[1] = un.y; vo[1] = vn.y; }
                        }
                        if (p.valid) {
                            uint8_t *m = p.valid + (size_t)gy * W + gx;
                            m[0] = tr.x > 0.f ? 1 : 0;
                            if (pair_ok) m[1] = tr.y > 0.f ? 1 : 0;
                        }
                        if (p.det) {
                            float *d = p.det + (size_t)gy * pitch + gx;
                            d[0] = det.x;
                            if (pair_ok) d[1] = det.y;
                        }
                    }
                }
            }
            __syncthreads();
        }
        t += ntask;
    }
}
