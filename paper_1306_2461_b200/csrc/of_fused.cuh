// of_fused.cuh -- one iteration of a COARSE pyramid level inside the CTA: K2 (warp, gradients, It, five products, horizontal window
// sum) and K3 (vertical window sum, damped 2x2 solve, update) back to back on a tile that fits in shared memory (rows a4-a9 of the
// scope table; "coarse-to-fine": the coarse levels of the pyramid; a further level should cost ~2 %).
//
// Why: at 320x256 or 640x512 a CTA's share of a pass is a few hundred to a few thousand pixels, so the two-pass form spends its time
// in two grid barriers (~1.4 us each) and two pipeline fills per iteration (level 2 of config 3: 8.4 us per iteration for 0.9 us of
// bytes).  Here a CTA owns one tile of tw x th outputs, forms the products of the tile plus its window halo (RL columns, RT rows on
// each side; the halo is recomputed by the neighbours, which is cheap at this size), sums them horizontally and vertically out of
// shared memory and solves: one grid barrier per iteration.  Because the neighbours read the OLD field in their halo while this CTA
// writes the NEW one, the field is double buffered (u, v <-> u2, v2; the buffer an iteration starts from is chosen so that the last
// one ends in u, v).
//
// Every value is formed by the same functions and the same order of taps as in of_k2.cuh / of_k3.cuh (products: k2_load,
// k2_task_gather, k2_task_products; sums: left to right, top to bottom; solve: k3_solve_store), so the result is bit-identical to
// the two-pass form, which of_set_persistent(0) still runs (tests/test_gpu_parity.py).  The five summed planes of such a level
// stay in shared memory.
#pragma once
#include "of_k2.cuh"
#include "of_k3.cuh"
#include <type_traits>

template <int R> struct FusedGeom {
    static constexpr int RL = K2Geom<R>::RL, OFF = K2Geom<R>::OFF, NIN = K2Geom<R>::NIN;
    static constexpr int RT = (R + 1) / 2 * 2;                                   // vertical halo in whole row pairs
    static constexpr int NINV = K3_SEG + 2 * R;                                  // input rows of a vertical task
    __host__ __device__ static constexpr int pw(int tw) { return tw + 2 * RL; }   // product columns
    __host__ __device__ static constexpr int ph(int th) { return th + 2 * RT; }   // product rows (even)
    __host__ __device__ static constexpr int bb(int tw) { return pw(tw) * 10; }   // bytes of one (field, row pair) block (layout of of_k2.cuh)
    __host__ __device__ static constexpr int prod_bytes(int tw, int th) { return (5 * (ph(th) / 2) * bb(tw) + 127) / 128 * 128; }
    __host__ __device__ static constexpr int hs_bytes(int tw, int th) { return 5 * ph(th) * tw * 4; }
    __host__ __device__ static constexpr int smem_bytes(int tw, int th) { return prod_bytes(tw, th) + hs_bytes(tw, th); }
};

struct FusedParams {
    const float *I1, *I2;
    const float *u_in, *v_in;              // field this iteration starts from (pitch `pitch`)
    float *u_out, *v_out;                  // field it writes (pitch `out_pitch`)
    uint8_t *valid;                        // level 0, last iteration: validity bytes and undamped determinant, else NULL
    float *det;
    int W, H, pitch, out_pitch;
    int tw, th, tiles_x, ntiles;           // tile t -> (t % tiles_x, t / tiles_x)
    WinWeights ww;
    SolveParams sp;
    int zero_uv;
    const uint8_t *mask;                   // obstacle mask of the level (pitch `pitch`; MK instantiation only): zero weight in the windows, no vector (M2, M3)
};

// Vertical window sums + solve + update of one tile out of the horizontally summed rows `hs` ([field][PH rows][tw]).
template <int R, int SEG, bool BX, bool MK>
__device__ __forceinline__ void fused_vsolve(const FusedParams &p, const K3Params &p3, const float *hs, int x0, int y0, int tid, int nthr)
{
    typedef FusedGeom<R> G;
    const int tw = p.tw, W = p.W, H = p.H, PH = G::ph(p.th);
    const int ncp = tw >> 1, nrb = p.th / SEG, ntask_v = ncp * nrb;
    for (int k = tid; k < ntask_v; k += nthr) {
        const int rb = k / ncp, c = k - rb * ncp;
        const int gx = x0 + 2 * c, gy0 = y0 + SEG * rb;
        if (gx >= W || gy0 >= H) continue;
        const int nrows = min(SEG, H - gy0);
        const float *ui = p.u_in + (size_t)gy0 * p.pitch + gx, *vi = p.v_in + (size_t)gy0 * p.pitch + gx;
        float2 uu[SEG], vv[SEG];
        unsigned mk[SEG];
#pragma unroll
        for (int j = 0; j < SEG; ++j) {
            const int jj = min(j, nrows - 1) * p.pitch;
            mk[j] = 0x0101u;
            if (MK) mk[j] = __ldg(reinterpret_cast<const unsigned short *>(p.mask + (size_t)gy0 * p.pitch + gx + jj));
            uu[j] = !p.zero_uv ? __ldcg(reinterpret_cast<const float2 *>(ui + jj)) : make_float2(0.f, 0.f);
            vv[j] = !p.zero_uv ? __ldcg(reinterpret_cast<const float2 *>(vi + jj)) : make_float2(0.f, 0.f);
        }
        float2 acc[5][SEG], core[5];
#pragma unroll
        for (int f = 0; f < 5; ++f) {
            core[f] = make_float2(0.f, 0.f);
#pragma unroll
            for (int j = 0; j < SEG; ++j) acc[f][j] = make_float2(0.f, 0.f);
        }
        // summed row r of the task is image row gy0 - R + r = buffer row SEG*rb + (RT - R) + r; rows top to bottom as in k3_phase
        const float *col = hs + (size_t)(SEG * rb + (G::RT - R)) * tw + 2 * c;
        auto sum_rows = [&](auto box) {
            constexpr bool BOX = decltype(box)::value;
#pragma unroll
            for (int r = 0; r < SEG + 2 * R; ++r)
#pragma unroll
                for (int f = 0; f < 5; ++f)
                    win_vrow<R, SEG, BOX>(p.ww, r, *reinterpret_cast<const float2 *>(col + (size_t)(f * PH + r) * tw), acc[f], core[f]);
#pragma unroll
            for (int f = 0; f < 5; ++f) win_vfinish<SEG, BOX>(acc[f], core[f]);
        };
        sum_rows(std::integral_constant<bool, BX>());
        k3_solve_store<MK, SEG>(p3, acc, uu, vv, mk, gx, gy0, nrows);
    }
}

// One iteration of a level by the CTAs of the grid: CTA `cta` runs tiles cta, cta + ncta, ...  All threads of the CTA take part;
// `smem` is the CTA's dynamic shared memory (at least FusedGeom<R>::smem_bytes(tw, th) bytes).
// (__forceinline__ on purpose: as a __noinline__ function it spills and costs 4 us per iteration.)
// MK = an obstacle mask is set (p.mask): masked products and outputs exactly as in the MK instantiations of K2 / K3; every tile is run.
template <int R, bool BX, bool MK = false>
__device__ __forceinline__ void fused_iteration(const FusedParams &p, unsigned char *smem, int cta, int ncta)
{
    typedef FusedGeom<R> G;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int tw = p.tw, th = p.th, W = p.W, H = p.H;
    const int PW = G::pw(tw), PH = G::ph(th), half = PW >> 1, nrpf = PH >> 1, BB = G::bb(tw), nseg = tw >> 3;
    char *const prod = reinterpret_cast<char *>(smem);
    float *const hs = reinterpret_cast<float *>(smem + G::prod_bytes(tw, th));
    K2Params p2 = {};
    p2.I1 = p.I1; p2.I2 = p.I2; p2.u = p.u_in; p2.v = p.v_in; p2.W = W; p2.H = H; p2.pitch = p.pitch; p2.zero_uv = p.zero_uv; p2.mask = p.mask;
    K3Params p3 = {};
    p3.u_in = p.u_in; p3.v_in = p.v_in; p3.u_out = p.u_out; p3.v_out = p.v_out; p3.valid = p.valid; p3.det = p.det;
    p3.W = W; p3.H = H; p3.pitch = p.pitch; p3.out_pitch = p.out_pitch; p3.sp = p.sp; p3.zero_uv = p.zero_uv;

    for (int t = cta; t < p.ntiles; t += ncta) {
        const int ty = t / p.tiles_x, tx = t - ty * p.tiles_x;
        const int x0 = tx * tw, y0 = ty * th;
        // ---------------- products of (tw + 2 RL) x (th + 2 RT) pixels, 2 x 2 per lane task, {row y, row y+1} interleaved per column
        const int ntask = half * nrpf;
        // The field values of a thread's first FUSED_AHEAD tasks are requested before the first task is worked on, so that a task
        // waits for one L2 round trip (I1, then the gather of I2) instead of two (as in the wide tiles of of_k2.cuh).
        constexpr int FUSED_AHEAD = 4;
        float2 pu0[FUSED_AHEAD], pu1[FUSED_AHEAD], pv0[FUSED_AHEAD], pv1[FUSED_AHEAD];
#pragma unroll
        for (int a = 0; a < FUSED_AHEAD; ++a) {
            pu0[a] = pu1[a] = pv0[a] = pv1[a] = make_float2(0.f, 0.f);
            const int k = tid + a * nthr;
            const int rp = k / half, cp = k - rp * half;
            const int x = x0 - G::RL + 2 * cp, y = y0 - G::RT + 2 * rp;
            if (k < ntask && !p.zero_uv && x >= 0 && x < W && y >= 0 && y < H) {
                const int i0 = y * p.pitch + x, d1 = y + 1 < H ? p.pitch : 0;
                const float *qu = ptr_at(p.u_in, i0), *qv = ptr_at(p.v_in, i0);
                pu0[a] = __ldcg(reinterpret_cast<const float2 *>(qu));
                pu1[a] = __ldcg(reinterpret_cast<const float2 *>(ptr_at(qu, d1)));
                pv0[a] = __ldcg(reinterpret_cast<const float2 *>(qv));
                pv1[a] = __ldcg(reinterpret_cast<const float2 *>(ptr_at(qv, d1)));
            }
        }
        auto products_task = [&](int k, bool have_uv, float2 u0, float2 u1, float2 v0, float2 v1) {
            const int rp = k / half, cp = k - rp * half;
            const int x = x0 - G::RL + 2 * cp, y = y0 - G::RT + 2 * rp;      // x, y even; a row pair never straddles row 0
            float4 o[5];
            if (x >= 0 && x < W && y >= 0 && y < H) {
                K2In in;
                if (have_uv) {
                    in = k2_load<MK, false>(p2, x, y);
                    in.u0 = u0; in.u1 = u1; in.v0 = v0; in.v1 = v1;
                } else {
                    in = k2_load<MK>(p2, x, y);
                }
                K2Tap tp[4];
                k2_task_gather(p2, in, x, y, tp);
                k2_task_products<MK>(p2, in, x, y, tp, o);
            } else {
#pragma unroll
                for (int f = 0; f < 5; ++f) o[f] = make_float4(0.f, 0.f, 0.f, 0.f);
            }
            char *d = prod + rp * BB + cp * 16 + (cp >> 2) * 16;
#pragma unroll
            for (int f = 0; f < 5; ++f) *reinterpret_cast<float4 *>(d + f * nrpf * BB) = o[f];
        };
#pragma unroll
        for (int a = 0; a < FUSED_AHEAD; ++a)
            if (tid + a * nthr < ntask) products_task(tid + a * nthr, true, pu0[a], pu1[a], pv0[a], pv1[a]);
        for (int k = tid + FUSED_AHEAD * nthr; k < ntask; k += nthr) products_task(k, false, make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f), make_float2(0.f, 0.f));
        __syncthreads();
        // ---------------- horizontal window sums: lane task = 8 outputs x 2 rows of one field
        const int ntask_h = 5 * nrpf * nseg;
        for (int k = tid; k < ntask_h; k += nthr) {
            const int f = k / (nrpf * nseg), rem = k - f * (nrpf * nseg);
            const int rp = rem / nseg, sg = rem - rp * nseg;
            const char *src = prod + (f * nrpf + rp) * BB + sg * 80;
            float2 in[G::NIN];
#pragma unroll
            for (int q = 0; q < G::NIN / 2; ++q) {
                const float4 v4 = *reinterpret_cast<const float4 *>(src + 16 * q + 16 * (q >> 2));
                in[2 * q] = make_float2(v4.x, v4.y);
                in[2 * q + 1] = make_float2(v4.z, v4.w);
            }
            float2 acc[8];
            win_hsum8<R, G::OFF, G::NIN, BX>(p.ww, in, acc);
            float *d0 = hs + (size_t)(f * PH + 2 * rp) * tw + 8 * sg;
            *reinterpret_cast<float4 *>(d0) = make_float4(acc[0].x, acc[1].x, acc[2].x, acc[3].x);
            *reinterpret_cast<float4 *>(d0 + 4) = make_float4(acc[4].x, acc[5].x, acc[6].x, acc[7].x);
            *reinterpret_cast<float4 *>(d0 + tw) = make_float4(acc[0].y, acc[1].y, acc[2].y, acc[3].y);
            *reinterpret_cast<float4 *>(d0 + tw + 4) = make_float4(acc[4].y, acc[5].y, acc[6].y, acc[7].y);
        }
        __syncthreads();
        // ---------------- vertical window sums + solve + update: lane task = 2 columns x K3_SEG rows (shorter tasks on small tiles, so
        // that every thread has one, were measured slower: 14.2 against 12.5 us per iteration at 640x512)
        fused_vsolve<R, K3_SEG, BX, MK>(p, p3, hs, x0, y0, tid, nthr);
        __syncthreads();                                   // the buffers are reused by the CTA's next tile
    }
}
