// of_k2s.cuh -- K2, streaming form: bilinear warp of I2 + central differences of I1 + It + five products + horizontal window sum
// (rows a4-a7 of the scope table; BASELINE.json:5 "(2) Per-iteration warp+gradient+product kernel: it reads I1 and I2 ... through
// TMA- or shared-memory-staged tiles with halos, bilinearly samples I2 at x+u, ... and does the horizontal window sum in shared
// memory before writing the five fields"; PAPER.md:57-61 for the method step; readings D8-D12 of DESIGN.md).
//
// One CTA per SM, K2S_WORKERS worker warps + one producer warp, no block barrier inside a pass.
//   * A level is cut into column strips of TW = 128 outputs; a UNIT is one strip x RU = 4 rows.  Units are numbered strip by strip,
//     top to bottom, and every CTA owns an equal, contiguous range of them, so consecutive units of a CTA are vertical neighbours.
//   * The PRODUCER lane walks the CTA's units in order and stages their inputs with bulk tensor copies (TMA; rows and columns
//     outside the image arrive zero-filled):
//       - per unit an "A slot": u, v (one 3-D box over (x, y, plane)) and I1 rows y0-1 .. y0+RU (2-D box), both with the product
//         halo of RL columns;
//       - a ring of I2 rows shared by the units of a strip: a unit's window is rows y0-HYR .. y0+RU+HYR and columns
//         x0-RL-HX .. x0+TW+RL+HX, so consecutive units add RU new rows (one box); a row is loaded once per CTA run.
//     It grants a unit to the workers (mbarrier `ready`) once all its copies have landed, and reuses a slot / ring rows only after
//     the product tasks that read them have finished (mbarrier `pdone`, confirmed in unit order).
//   * The WORKERS pull tasks from one in-order ticket counter: P(i, r) = the five products of 32 lane tasks (2 x 2 pixels each) of
//     unit i (+ halo columns) into a shared-memory product buffer; H012(i), H34(i) = the horizontal window sums of fields 0-2 / 3-4 of unit i, written to the
//     five planes.  Every wait of a task is on tasks with smaller tickets (or on the producer, which waits on smaller tickets
//     only), so the queue cannot deadlock; which warp runs a task does not change its arithmetic (H8: bit-reproducible).
//   * P gathers I2 from the shared-memory window: x + floor(u) is formed on integers/exact floats (D8), clamp-to-edge exactly as
//     in of_k2.cuh; a 2x2 cell that leaves the staged window falls back to a global read of the same pixels, so the
//     result never depends on the window size.
//   * H: lane = 8 outputs x 2 rows: (8+2RL)/2 LDS.128 + 8*(2R+1) FFMA2 per field, direct (2R+1)-tap sums in a fixed order
//     (H2: no running sums, zero stays zero).
// The arithmetic of every value (expression trees, tap order) is that of of_k2.cuh, which the masked instantiations still use.
#pragma once
#include "of_k2.cuh"
#include "of_async.cuh"

#ifndef K2S_WORKERS
#define K2S_WORKERS 11
#endif
#ifdef K2S_PROFILE                                 // throw-away instrumentation of a debugging build: cycles per category, printed by two CTAs
#include <cstdio>
#define K2S_T(var) const long long var = clock64()
#define K2S_ACC(acc, a, b) acc += (b) - (a)
#else
#define K2S_T(var)
#define K2S_ACC(acc, a, b)
#endif

template <int R> struct K2S {
    static constexpr int RL = (R + 3) / 4 * 4, OFF = RL - R, NIN = 8 + 2 * RL;
    static constexpr int TW = 128, RU = 4, NRP = RU / 2, NSEG = TW / 8;       // unit = 128 x 4 outputs = 16 segments x 2 row pairs (32 H lanes)
    static constexpr int PW = TW + 2 * RL;                                     // product columns of a unit: x0-RL .. x0+TW+RL-1
    static constexpr int HALF = PW / 2, NTASK = HALF * NRP;                    // column pairs; P lane tasks (2 x 2 pixels)
    static constexpr int NROUND = (NTASK + 31) / 32;
    static constexpr int BB = PW * 10;                                         // one (field, row pair) block: 8 B per column + 16 B per 8 columns
    static constexpr int PROD_STRIDE = (5 * NRP * BB + 127) / 128 * 128;
    static constexpr int HX = 16, HYR = 8;                                     // I2 window halo beyond the product columns / the unit's rows
    static constexpr int PWB = PW + 2 * HX;                                    // staged I2 row: columns x0-RL-HX ..
    static constexpr int WROWS = RU + 2 * HYR + 1;                             // rows of a unit's I2 window: y0-HYR .. y0+RU+HYR
    static constexpr int WPAD = (WROWS + RU - 1) / RU * RU - WROWS;            // extra rows on top of a run's first window (whole boxes)
    static constexpr int I2BOX_BYTES = RU * PWB * 4;
    static constexpr int NB = 11, NU = 2 * NB, LAG = 2;                 // product buffers; unit slots of the barriers (> NGRP + LU: never the limit of the run-ahead); P-to-H lag
    static constexpr int DATA_MAX = 225280;                                    // bytes below the barrier area (= the K3 ring, of_k3.cuh)
    static constexpr int NBOX0 = (WROWS + WPAD) / RU;                          // boxes of a run's first window
    static constexpr int LU = (2 * HYR + RU) / RU;                             // a box loaded for unit i is last read by unit i + LU
    static constexpr int NGRP = (DATA_MAX - NB * PROD_STRIDE) / I2BOX_BYTES, NRING = NGRP * RU;   // I2 ring boxes / rows
    static constexpr int RING_OFF = NB * PROD_STRIDE;
    static constexpr int DATA_BYTES = RING_OFF + NRING * PWB * 4;
    // barrier area (offsets relative to its base): tfull[NU] ready[NU] pdone[NU] pfree[NB] | udesc[NU] | ticket counter
    static constexpr int BAR_TFULL = 0, BAR_READY = 8 * NU, BAR_PDONE = 16 * NU, BAR_PFREE = 24 * NU, DESC_OFF = 24 * NU + 8 * NB,
                         TICKET_OFF = DESC_OFF + 4 * NU, LASTUSER_OFF = TICKET_OFF + 16, BAR_BYTES = LASTUSER_OFF + 4 * NGRP;
    static_assert(NB > LAG, "pipeline depths");
    static_assert(NGRP >= NBOX0 + LU + 1, "I2 ring too short");
    static_assert(NTASK <= 32 * NROUND && NSEG * NRP == 32, "lane layout");
    static_assert(PWB <= 256, "TMA box limit");
    static_assert(I2BOX_BYTES % 128 == 0, "TMA destination alignment");
};

struct K2SMaps {                                   // tensor maps of one level, in global memory (encoded once in of_create)
    CUtensorMap i2[2];                             // pyramid slot s as I2: 2-D (x, y), box PWB x RU
};

struct K2SParams {
    const K2SMaps *maps;
    int s2;                                        // pyramid slot used as I2
    const float *I1, *I2, *u, *v;                  // I2: for the global fallback of the gather
    float *S;
    size_t plane;
    int W, H, pitch;
    int nuy, nunits;                               // units per strip; units of the level (unit g -> strip g / nuy, row block g % nuy)
    unsigned long long nuy_magic;                  // ceil(2^40 / nuy)
    WinWeights ww;
    int zero_uv;                                   // 1 = the field is identically zero and is not read
    int f_first;                                   // HO only: first plane formed by this pass (3 = IxIt, IyIt only)
};

template <int R> struct K2SSmem {
    unsigned char *data;
    uint32_t data0, bar0;
    int *desc, *ticket, *last_user;
    __device__ __forceinline__ K2SSmem(unsigned char *d, unsigned char *bars)
        : data(d), data0(smem_u32(d)), bar0(smem_u32(bars)), desc(reinterpret_cast<int *>(bars + K2S<R>::DESC_OFF)),
          ticket(reinterpret_cast<int *>(bars + K2S<R>::TICKET_OFF)), last_user(reinterpret_cast<int *>(bars + K2S<R>::LASTUSER_OFF)) {}
};

// Thread 0 of the CTA, once per kernel, followed by fence.mbarrier_init + __syncthreads.
template <int R> __device__ __forceinline__ void k2s_init_barriers(const K2SSmem<R> &sm)
{
    typedef K2S<R> G;
    for (int j = 0; j < G::NU; ++j) {
        mbar_init(sm.bar0 + G::BAR_TFULL + 8 * j, 1);
        mbar_init(sm.bar0 + G::BAR_PDONE + 8 * j, G::NROUND);           // one arrival per product round
    }
    for (int j = 0; j < G::NB; ++j) mbar_init(sm.bar0 + G::BAR_PFREE + 8 * j, 5);   // one arrival per field
    *sm.ticket = 0;
}

// ---------------------------------------------------------------------------------------------------------------- producer
// unit g -> (strip, row block) without a division: strip = (g * nuy_magic) >> 40, nuy_magic = ceil(2^40 / nuy) (exact for g * nuy < 2^40)
__device__ __forceinline__ void k2s_unit_xy(const K2SParams &p, int g, int &s, int &j)
{
    s = (int)(((unsigned long long)(unsigned)g * p.nuy_magic) >> 40);
    j = g - s * p.nuy;
}

// One lane.  `ub` = units this CTA has processed in earlier passes of the same kernel (keeps slot / parity bookkeeping continuous).
// It walks the CTA's units in order; the copies of unit i complete on mbarrier tfull[i], on which the product tasks wait themselves.
// All bookkeeping is incremental (no division, one shared-memory word per box): a single thread runs this loop.  A wait here is
// always for product tasks of units whose copies have already been issued, so it cannot deadlock.
template <int R>
__device__ __forceinline__ void k2s_produce(const K2SParams &p, const K2SSmem<R> &sm, int u_begin, int n, uint32_t ub)
{
    typedef K2S<R> G;
    const CUtensorMap *tm2 = &p.maps->i2[p.s2];
    for (int g = 0; g < G::NGRP; ++g) sm.last_user[g] = -1;
    int s, j;
    k2s_unit_xy(p, u_begin, s, j);
    int gi = 0;                                      // ring box (group of RU rows) the next copy goes to
    int wrow = 0;                                    // ring row of the first row (y0 - HYR) of the unit's window
    int run_last = 0;
    int confirmed = -1;                              // product tasks of the units <= confirmed are known to be finished
    uint32_t ci = ub % G::NU, cpar = (ub / G::NU) & 1;   // barrier slot / parity of unit confirmed + 1
    uint32_t ii = ci;                                    // ... of unit ip
    long long pr_wait = 0;
    (void)pr_wait;
    K2S_T(pr_begin);
    for (int ip = 0; ip < n; ++ip) {
        const bool new_run = (ip == 0) || (j == 0);
        const int nbox = new_run ? G::NBOX0 : 1;
        // the descriptor / barrier slot of unit ip - NU is re-used: the product tasks of the units ip - NU .. ip - NU + LU wait on
        // that mbarrier (their windows hold rows copied for it) and must all be past their wait before it starts another phase:
        // an mbarrier only tells the parity of its current phase, so a waiter that is two phases late would wait for ever
        int m = ip - G::NU + G::LU;
        {
            int g2 = gi;
            for (int b = 0; b < nbox; ++b) { m = max(m, sm.last_user[g2]); g2 = g2 + 1 == G::NGRP ? 0 : g2 + 1; }
        }
        K2S_T(c0);
        while (confirmed < m) {                      // the units that read the rows (and the slot) this issue overwrites
            mbar_wait(sm.bar0 + G::BAR_PDONE + 8 * ci, cpar);
            ++confirmed;
            if (++ci == G::NU) { ci = 0; cpar ^= 1; }
        }
        K2S_T(c1);
        K2S_ACC(pr_wait, c0, c1);
        const int x0 = s * G::TW, y0 = j * G::RU;
        const uint32_t bar = sm.bar0 + G::BAR_TFULL + 8 * ii;
        int r0;
        if (new_run) {
            run_last = min(n - 1, ip + (p.nuy - 1 - j));
            r0 = y0 - G::HYR - G::WPAD;
            wrow = gi * G::RU + G::WPAD;
            if (wrow >= G::NRING) wrow -= G::NRING;
        } else {
            r0 = y0 + G::HYR + 1;
        }
        sm.desc[ii] = wrow;                          // ring row of image row y0 - HYR (published by the arrive below)
        mbar_expect_tx(bar, (uint32_t)(nbox * G::I2BOX_BYTES));
        for (int b = 0; b < nbox; ++b, r0 += G::RU) {
            tma_load_2d(sm.data0 + G::RING_OFF + gi * G::I2BOX_BYTES, tm2, x0 - G::RL - G::HX, r0, bar);
            // last unit of this run whose window (rows y0'-HYR .. y0'+RU+HYR) holds one of the rows of this box
            sm.last_user[gi] = min(run_last, ip + (new_run ? b : G::LU));
            gi = gi + 1 == G::NGRP ? 0 : gi + 1;
        }
        wrow += G::RU;
        if (wrow >= G::NRING) wrow -= G::NRING;
        if (++ii == G::NU) ii = 0;
        if (++j == p.nuy) { j = 0; ++s; }
    }
#ifdef K2S_PROFILE
    if ((blockIdx.x == 0 || blockIdx.x == 77) && p.zero_uv == 0 && p.W >= 1024)
        printf("[k2s] cta %d producer units %d total %lld | confirm waits %lld\n", blockIdx.x, n, clock64() - pr_begin, pr_wait);
#endif
}

// ---------------------------------------------------------------------------------------------------------------- P task
// Round r of unit g: 32 lane tasks of 2 x 2 pixels.  k2s_products_load requests this lane's I1 / u / v values straight from global
// memory (8-byte loads, coalesced across the warp); it is called one task ahead, so that the L2 round trip is covered by the task
// in between.  k2s_products_task does the rest.
template <int R>
__device__ __forceinline__ K2In k2s_products_load(const K2SParams &p, int lane, int g, int r)
{
    typedef K2S<R> G;
    int s, j;
    k2s_unit_xy(p, g, s, j);
    const int k = lane + 32 * r;
    const int rp = k >= G::HALF ? 1 : 0, cp = k - rp * G::HALF;
    const int x = s * G::TW - G::RL + 2 * cp, y = j * G::RU + 2 * rp;
    K2In in = {};
    if (!(k < G::NTASK && x >= 0 && x < p.W && y < p.H)) return in;
    const int x0 = s * G::TW, y0 = j * G::RU;
    if (x0 - G::RL >= 1 && x0 + G::TW + G::RL + 2 <= p.W && y0 >= 1 && y0 + G::RU + 2 <= p.H) {
        // interior unit (decided per warp): no clamp-to-edge anywhere in its halo, one index and constant offsets
        const int pitch = p.pitch, i0 = y * pitch + x;
        const float *c = ptr_at(p.I1, i0);
        in.cm = __ldg(reinterpret_cast<const float2 *>(c - pitch));
        in.c0 = __ldg(reinterpret_cast<const float2 *>(c));
        in.c1 = __ldg(reinterpret_cast<const float2 *>(c + pitch));
        in.c2 = __ldg(reinterpret_cast<const float2 *>(c + 2 * pitch));
        in.l0 = __ldg(c - 1); in.q0 = __ldg(c + 2);
        in.l1 = __ldg(c + pitch - 1); in.q1 = __ldg(c + pitch + 2);
        if (!p.zero_uv) {
            const float *pu = ptr_at(p.u, i0), *pv = ptr_at(p.v, i0);
            in.u0 = __ldcg(reinterpret_cast<const float2 *>(pu)); in.u1 = __ldcg(reinterpret_cast<const float2 *>(pu + pitch));
            in.v0 = __ldcg(reinterpret_cast<const float2 *>(pv)); in.v1 = __ldcg(reinterpret_cast<const float2 *>(pv + pitch));
        }
        in.m0 = in.m1 = 0x0101u;
        return in;
    }
    K2Params pw = {};
    pw.I1 = p.I1; pw.u = p.u; pw.v = p.v; pw.W = p.W; pw.H = p.H; pw.pitch = p.pitch; pw.zero_uv = p.zero_uv;
    return k2_load<false>(pw, x, y);
}

template <int R, bool HO>
__device__ __forceinline__ void k2s_products_task(const K2SParams &p, const K2SSmem<R> &sm, int lane, int g, uint32_t q, int r, const K2In &in, long long *prof)
{
    typedef K2S<R> G;
    int s, j;
    k2s_unit_xy(p, g, s, j);
    const int x0 = s * G::TW, y0 = j * G::RU, xs = x0 - G::RL;
    const int W = p.W, H = p.H;
    const int f_first = HO ? p.f_first : 0;
    const int k = lane + 32 * r;
    const int rp = k >= G::HALF ? 1 : 0, cp = k - rp * G::HALF;
    const int x = xs + 2 * cp, y = y0 + 2 * rp;
    const bool act = k < G::NTASK && x >= 0 && x < W && y < H;
    K2Params pw = {};
    pw.W = W; pw.H = H;
    const uint32_t qu = q % G::NU, qb = q % G::NB;
    K2S_T(c0);
    // the window of unit q holds rows copied for units q - LU .. q (older ones of the same run; a unit of an earlier run or pass has
    // long completed): lanes 0 .. LU each wait on one of those mbarriers
    if (lane <= G::LU && q >= (uint32_t)lane) {
        const uint32_t ql = q - (uint32_t)lane;
        mbar_wait(sm.bar0 + G::BAR_TFULL + 8 * (ql % G::NU), (ql / G::NU) & 1);
    }
    __syncwarp();
    K2S_T(c1);
    if (q >= (uint32_t)G::NB) mbar_wait(sm.bar0 + G::BAR_PFREE + 8 * qb, (q / G::NB - 1) & 1);
    K2S_T(c2);
    K2S_ACC(prof[1], c0, c1); K2S_ACC(prof[2], c1, c2);
    const int slot_lo = sm.desc[qu];
    const uint32_t ring = sm.data0 + G::RING_OFF;
    char *buf = reinterpret_cast<char *>(sm.data) + qb * G::PROD_STRIDE;
    const int wx0 = xs - G::HX, wy0 = y0 - G::HYR;
    float4 o[5];
#pragma unroll
    for (int f = 0; f < 5; ++f) o[f] = make_float4(0.f, 0.f, 0.f, 0.f);
    K2Tap t[4];
    const float uu[4] = {in.u0.x, in.u1.x, in.u0.y, in.u1.y}, vv[4] = {in.v0.x, in.v1.x, in.v0.y, in.v1.y};
    // ---- fast path: every cell of the round lies inside the image (no clamp: Xc = X, the fraction is u - floor(u), the
    // expressions of k2_gather reduce to these bit for bit) and inside the staged window, and the window does not wrap in the ring
    int Xi[4], Yi[4];
    bool ok = true;
    {
        const int ixlo = max(0, wx0), ixr = min(W - 2, wx0 + G::PWB - 2) - ixlo;          // allowed cell origins (inclusive)
        const int iylo = max(0, wy0), iyr = min(H - 2, wy0 + G::WROWS - 2) - iylo;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float fu = floorf(uu[e]), fv = floorf(vv[e]);
            t[e].ax = uu[e] - fu; t[e].ay = vv[e] - fv;
            Xi[e] = x + (e >> 1) + __float2int_rn(fu); Yi[e] = y + (e & 1) + __float2int_rn(fv);
            ok = ok && (unsigned)(Xi[e] - ixlo) <= (unsigned)ixr && (unsigned)(Yi[e] - iylo) <= (unsigned)iyr;
        }
        ok = ok || !act;
    }
    if (__all_sync(0xffffffffu, ok)) {
        if (act) {
            const uint32_t base = ring + (uint32_t)(((slot_lo - wy0) * G::PWB - wx0) * 4);
            if (slot_lo + G::WROWS <= G::NRING) {                        // the window is contiguous in the ring
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const uint32_t a0 = base + (uint32_t)(Yi[e] * G::PWB + Xi[e]) * 4u;
                    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(t[e].i00) : "r"(a0));
                    asm volatile("ld.shared.f32 %0, [%1+4];" : "=f"(t[e].i01) : "r"(a0));
                    asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(t[e].i10) : "r"(a0), "n"(G::PWB * 4));
                    asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(t[e].i11) : "r"(a0), "n"(G::PWB * 4 + 4));
                }
            } else {                                                     // it wraps: rows from ring row NRING on live at the start
                const int ywrap = wy0 + (G::NRING - slot_lo);            // first image row that has wrapped
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const uint32_t a0 = base + (uint32_t)(Yi[e] * G::PWB + Xi[e]) * 4u;
                    const uint32_t b0 = a0 - (Yi[e] >= ywrap ? (uint32_t)(G::NRING * G::PWB * 4) : 0u);
                    const uint32_t b1 = a0 - (Yi[e] + 1 >= ywrap ? (uint32_t)(G::NRING * G::PWB * 4) : 0u);
                    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(t[e].i00) : "r"(b0));
                    asm volatile("ld.shared.f32 %0, [%1+4];" : "=f"(t[e].i01) : "r"(b0));
                    asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(t[e].i10) : "r"(b1), "n"(G::PWB * 4));
                    asm volatile("ld.shared.f32 %0, [%1+%2];" : "=f"(t[e].i11) : "r"(b1), "n"(G::PWB * 4 + 4));
                }
            }
        }
    } else if (act) {
        // ---- general path: clamp-to-edge as in k2_gather (of_k2.cuh); a cell that leaves the staged window is read from global memory (H4)
        const float Wm2f = (float)(W - 2), Hm2f = (float)(H - 2), xf = (float)x, yf = (float)y;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const float fu = floorf(uu[e]), fv = floorf(vv[e]);
            const float Xf = (xf + (float)(e >> 1)) + fu, Yf = (yf + (float)(e & 1)) + fv;
            const float Xc = fminf(fmaxf(Xf, 0.f), Wm2f), Yc = fminf(fmaxf(Yf, 0.f), Hm2f);
            t[e].ax = __saturatef((uu[e] - fu) + (Xf - Xc));
            t[e].ay = __saturatef((vv[e] - fv) + (Yf - Yc));
            const int X = __float2int_rn(Xc), Y = __float2int_rn(Yc);
            if ((unsigned)(X - wx0) <= (unsigned)(G::PWB - 2) && (unsigned)(Y - wy0) <= (unsigned)(G::WROWS - 2)) {
                int rr = slot_lo + (Y - wy0);
                rr -= rr >= G::NRING ? G::NRING : 0;
                const int rr1 = rr + 1 == G::NRING ? 0 : rr + 1;
                const uint32_t a0 = ring + (uint32_t)(rr * G::PWB + (X - wx0)) * 4u, a1 = ring + (uint32_t)(rr1 * G::PWB + (X - wx0)) * 4u;
                asm volatile("ld.shared.f32 %0, [%1];" : "=f"(t[e].i00) : "r"(a0));
                asm volatile("ld.shared.f32 %0, [%1+4];" : "=f"(t[e].i01) : "r"(a0));
                asm volatile("ld.shared.f32 %0, [%1];" : "=f"(t[e].i10) : "r"(a1));
                asm volatile("ld.shared.f32 %0, [%1+4];" : "=f"(t[e].i11) : "r"(a1));
            } else {
                const float *p0 = ptr_at(p.I2, Y * p.pitch + X);
                const float *p1 = ptr_at(p0, p.pitch);
                t[e].i00 = __ldg(p0); t[e].i01 = __ldg(p0 + 1); t[e].i10 = __ldg(p1); t[e].i11 = __ldg(p1 + 1);
            }
        }
    }
    if (act) k2_task_products<false>(pw, in, x, y, t, o);
    if (k < G::NTASK) {
        char *d = buf + rp * G::BB + cp * 16 + (cp >> 2) * 16;
#pragma unroll
        for (int f = 0; f < 5; ++f)
            if (f >= f_first) *reinterpret_cast<float4 *>(d + f * G::NRP * G::BB) = o[f];
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(sm.bar0 + G::BAR_PDONE + 8 * qu, 1);
    K2S_T(c3);
    K2S_ACC(prof[3], c2, c3);
}

// ---------------------------------------------------------------------------------------------------------------- H task
// Field f of unit g (or nothing, `skip`: a plane this pass does not form): horizontal window sums from the product buffer to the plane.
template <int R, bool BX>
__device__ __forceinline__ void k2s_hsum_task(const K2SParams &p, const K2SSmem<R> &sm, int lane, int g, uint32_t q, int f, bool skip, long long *prof)
{
    typedef K2S<R> G;
    int s, j;
    k2s_unit_xy(p, g, s, j);
    const int x0 = s * G::TW, y0 = j * G::RU;
    const uint32_t qb = q % G::NB;
    K2S_T(c0);
    mbar_wait(sm.bar0 + G::BAR_PDONE + 8 * (q % G::NU), (q / G::NU) & 1);
    K2S_T(c1);
    K2S_ACC(prof[4], c0, c1);
    if (!skip) {
        const int h_seg = lane % G::NSEG, h_rp = lane / G::NSEG;
        const int gx = x0 + 8 * h_seg, gy = y0 + 2 * h_rp;
        const char *src = reinterpret_cast<const char *>(sm.data) + qb * G::PROD_STRIDE + (f * G::NRP + h_rp) * G::BB + h_seg * 80;
        float2 in[G::NIN];
#pragma unroll
        for (int k = 0; k < G::NIN / 2; ++k) {
            const float4 v = *reinterpret_cast<const float4 *>(src + 16 * k + 16 * (k >> 2));
            in[2 * k] = make_float2(v.x, v.y);
            in[2 * k + 1] = make_float2(v.z, v.w);
        }
        float2 acc[8];
        win_hsum8<R, G::OFF, G::NIN, BX>(p.ww, in, acc);
        if (gx < p.pitch) {
            float *d0 = p.S + f * p.plane + (size_t)gy * p.pitch + gx;
            if (gy < p.H) {
                *reinterpret_cast<float4 *>(d0) = make_float4(acc[0].x, acc[1].x, acc[2].x, acc[3].x);
                *reinterpret_cast<float4 *>(d0 + 4) = make_float4(acc[4].x, acc[5].x, acc[6].x, acc[7].x);
            }
            if (gy + 1 < p.H) {
                *reinterpret_cast<float4 *>(d0 + p.pitch) = make_float4(acc[0].y, acc[1].y, acc[2].y, acc[3].y);
                *reinterpret_cast<float4 *>(d0 + p.pitch + 4) = make_float4(acc[4].y, acc[5].y, acc[6].y, acc[7].y);
            }
        }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(sm.bar0 + G::BAR_PFREE + 8 * qb, 1);
    K2S_T(c2);
    K2S_ACC(prof[5], c1, c2);
}

// ---------------------------------------------------------------------------------------------------------------- the pass
// One K2 pass over a level by the CTA that owns units [u_begin, u_end).  Warps 0 .. K2S_WORKERS-1 work, warp K2S_WORKERS produces.
// *sm.ticket must be 0 on entry (CTA-synchronised); the caller resets it after the pass and adds u_end - u_begin to `ub`.
template <int R, bool HO, bool BX>
__device__ __forceinline__ void k2s_phase(const K2SParams &p, const K2SSmem<R> &sm, int warp, int lane, int u_begin, int u_end, uint32_t ub)
{
    typedef K2S<R> G;
    const int n = u_end - u_begin;
    if (n <= 0) return;
    if (warp == K2S_WORKERS) {
        if (lane == 0) k2s_produce<R>(p, sm, u_begin, n, ub);
        __syncwarp();
        return;
    }
    constexpr int NK = G::NROUND + 5;                                      // tickets per unit: its product rounds, then one sum task per field
    const int total = NK * (n + G::LAG);
    const int f_first = HO ? p.f_first : 0;
    long long prof[6] = {0, 0, 0, 0, 0, 0};          // ticket, wait ready, wait pfree, products, wait pdone, sums (K2S_PROFILE only)
    (void)prof;
    K2S_T(p_begin);
    // Tickets are dealt round-robin (warp w runs tickets w, w + K2S_WORKERS, ...): no shared counter, and a warp knows its next
    // ticket, so the global loads of its next product task are in flight while it runs the current one.  Every warp runs its
    // tickets in increasing order and every wait is on smaller tickets, so the smallest unfinished ticket can always proceed.
    // (two tickets per trip with two input buffers: a register copy of prefetched values would wait for the loads.)
    auto preload = [&](int t, K2In &in) {
        const int i = t / NK, kind = t - NK * i;
        if (t < total && kind < G::NROUND && i < n) in = k2s_products_load<R>(p, lane, u_begin + i, kind);
    };
    auto run = [&](int t, const K2In &in) {
        const int i = t / NK, kind = t - NK * i;
        if (kind < G::NROUND) {
            if (i < n) k2s_products_task<R, HO>(p, sm, lane, u_begin + i, ub + (uint32_t)i, kind, in, prof);
        } else {
            const int ih = i - G::LAG, f = kind - G::NROUND;
            if (ih >= 0 && ih < n) k2s_hsum_task<R, BX>(p, sm, lane, u_begin + ih, ub + (uint32_t)ih, f, f < f_first, prof);
        }
    };
    K2In in_a = {}, in_b = {};
    preload(warp, in_a);
#ifdef K2S_PROFILE
    long long tl_s[40], tl_e[40];
    int tl_n = 0;
#define K2S_RUN(tt, inn) do { const long long a_ = clock64(); run(tt, inn); if (tl_n < 40) { tl_s[tl_n] = a_ - p_begin; tl_e[tl_n] = clock64() - p_begin; ++tl_n; } } while (0)
#else
#define K2S_RUN(tt, inn) run(tt, inn)
#endif
    for (int t = warp; t < total; t += 2 * K2S_WORKERS) {
        preload(t + K2S_WORKERS, in_b);
        K2S_RUN(t, in_a);
        if (t + K2S_WORKERS >= total) break;
        preload(t + 2 * K2S_WORKERS, in_a);
        K2S_RUN(t + K2S_WORKERS, in_b);
    }
#ifdef K2S_PROFILE
    if (lane == 0 && blockIdx.x == 77 && p.zero_uv == 0 && p.W >= 1024)
        for (int e = 0; e < tl_n; ++e) printf("[tl] %d %d %lld %lld\n", warp, warp + e * K2S_WORKERS, tl_s[e], tl_e[e]);
#endif
#ifdef K2S_PROFILE
    if (lane == 0 && (blockIdx.x == 0 || blockIdx.x == 77) && p.zero_uv == 0 && p.W >= 1024)
        printf("[k2s] cta %d warp %d units %d total %lld | ticket %lld wait_ready %lld wait_pfree %lld products %lld wait_pdone %lld sums %lld\n", blockIdx.x, warp, n,
               clock64() - p_begin, prof[0], prof[1], prof[2], prof[3], prof[4], prof[5]);
#endif
}

// Stand-alone launch of one K2 pass (of_set_persistent(0), of_run_step): the same pass function as in the persistent solve kernel.
template <int R, bool BX>
__global__ void __launch_bounds__(32 * (K2S_WORKERS + 1), 1) k2s_products_hsum(const K2SParams p)
{
    extern __shared__ __align__(1024) unsigned char k2s_smem_[];
    const K2SSmem<R> sm(k2s_smem_, k2s_smem_ + K2S<R>::DATA_MAX);
    if (threadIdx.x == 0) {
        k2s_init_barriers<R>(sm);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    int ub, ue;
    cta_range(p.nunits, blockIdx.x, gridDim.x, ub, ue);
    k2s_phase<R, false, BX>(p, sm, threadIdx.x >> 5, threadIdx.x & 31, ub, ue, 0u);
}
