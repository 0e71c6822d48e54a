// of_k3.cuh -- K3: vertical window sum + damped 2x2 solve + in-place (u,v) update (rows a8-a9 of the
// scope table; BASELINE.json:5 "(3) Vertical-sum+solve kernel"; readings D11-D15 of DESIGN.md).
//
// Persistent, warp-specialised, one CTA per SM (sm_100a):
//   * the image is cut into 64-column strips x K3_SEG-row blocks = "tasks"; task order is strip-major and
//     every CTA owns an equal, contiguous run of tasks (grid = number of SMs, no tail wave);
//   * the five horizontally summed planes are ONE 3-D tensor (x, y, field); a chunk = box of
//     64 x K3_SEG x 5 floats (5 KB) fetched by a single cp.async.bulk.tensor into a shared-memory ring;
//     rows above/below the image are zero-filled by the TMA unit, which IS the zero extension of the
//     window (D12) -- no border code;
//   * one PRODUCER warp issues the CTA's chunks, its 32 lanes in parallel (a lane needs ~105 cycles per copy): each waits for
//     the ring slot to be released (empty mbarrier, NC arrivals = the NC tasks that read a chunk), arms the full mbarrier
//     with expect_tx and issues the TMA; when its last chunk is issued the warp joins the consumers;
//   * the CONSUMER warps (K3_MAX_NW = 11) pull tasks from a shared-memory counter (balances the four SM
//     sub-partitions), wait on the full barriers of their NC chunks, sum, release the chunks, solve.
//     No __syncthreads after set-up.  Which warp runs a task does not change its arithmetic, so the
//     result stays bit-reproducible (H8);
//   * per lane (2 adjacent columns x K3_SEG rows): (K3_SEG+2R) LDS.64 per field feed K3_SEG*(2R+1) FFMA2 (packed
//     fp32 pair FMA, scalar weight); then the damped 2x2 solve on the pair (D14), clamp (D15),
//     update, validity byte.
// Direct (2R+1)-tap sums, fixed order, no atomics on data: no cancellation (H2).
#pragma once
#include "of_common.cuh"
#include "of_async.cuh"
#include <type_traits>

#ifndef K3_SEG
#define K3_SEG 4                                          // rows per task = rows per TMA chunk (4: finer tasks, better
                                                          // balance and shorter coarse-level passes than 8; measured)
#endif
#define K3_CHUNK_BYTES (64 * K3_SEG * 5 * 4)
#ifndef K3_MAX_NW
#define K3_MAX_NW 11                                      // consumer warps (+1 producer warp)
#endif
#ifndef K3_RING
#define K3_RING (176 / K3_SEG)                            // chunks in the ring (220 KB)
#endif
#define K3_BATCH (K3_RING > 32 ? 32 : 16)                 // lanes of the producer warp that issue copies; must be < K3_RING (see the producer)

template <int R> struct K3Geom {
    static constexpr int NIN = K3_SEG + 2 * R;           // input rows per task
    static constexpr int NC = (NIN + K3_SEG - 1) / K3_SEG;   // chunks spanned by one task
    static constexpr int SMEM = K3_RING * K3_CHUNK_BYTES + 2 * K3_RING * 8 + 16;
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
    int zero_uv;                     // 1 = the incoming field is identically zero and is not read (see of_k2.cuh)
    int dbg;                         // -DOF_PROFILE builds only: 1 = no TMA/no waits, 2 = no window sum, 4 = no solve
    MaskDesc md;                     // obstacle mask and compacted task lists of the level (all zero: none)
    float *G;                        // of_set_hoist: three planes (stride `gplane`, pitch `pitch`) holding the window sums a, b, c
    size_t gplane;                   //   of IxIx, IxIy, IyIy of the level (written by an HM = 1 pass, read by HM = 2 passes)
};

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
    float2 inv;                                                 // MUFU.RCP, <= 1 ulp; D > 0 wherever tr > 0
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(inv.x) : "f"(D.x));
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(inv.y) : "f"(D.y));
    du = __fmul2_rn(nu, inv);
    dv = __fmul2_rn(nv, inv);
    const float ms = sp.max_step;
    du.x = tr.x > 0.f ? fminf(fmaxf(du.x, -ms), ms) : 0.f;
    du.y = tr.y > 0.f ? fminf(fmaxf(du.y, -ms), ms) : 0.f;
    dv.x = tr.x > 0.f ? fminf(fmaxf(dv.x, -ms), ms) : 0.f;
    dv.y = tr.y > 0.f ? fminf(fmaxf(dv.y, -ms), ms) : 0.f;
}

// Damped 2x2 solve, clamp, update and stores of one task (K3_SEG rows x 2 columns per lane) from its five window sums.  Shared by
// the K3 pass and the fused coarse-level pass (of_fused.cuh), so both form every value with the same instructions.
template <bool MK, int SEG = K3_SEG>
__device__ __forceinline__ void k3_solve_store(const K3Params &p, const float2 (&acc)[5][SEG], const float2 (&uu)[SEG], const float2 (&vv)[SEG],
                                               const unsigned (&mk)[SEG], int gx, int gy0, int nrows)
{
    const int W = p.W, pitch = p.pitch;
    // ---- solve + update for K3_SEG rows x 2 columns
    const bool pair_ok = gx + 1 < W;
    const bool vec_out = (p.out_pitch & 1) == 0 && pair_ok;
    float *uo = p.u_out + (size_t)gy0 * p.out_pitch + gx, *vo = p.v_out + (size_t)gy0 * p.out_pitch + gx;
    float2 trs[SEG], dets[SEG];
#pragma unroll
    for (int j = 0; j < SEG; ++j) {
        float2 du, dv;
        k3_solve_pair(acc[0][j], acc[1][j], acc[2][j], acc[3][j], acc[4][j], uu[j], vv[j], p.sp, du, dv, trs[j], dets[j]);
        float2 un = __fadd2_rn(uu[j], du), vn = __fadd2_rn(vv[j], dv);
        if (MK) {                                    // M3: no vector over an obstacle
            if (!(mk[j] & 0xffu)) { un.x = 0.f; vn.x = 0.f; trs[j].x = 0.f; dets[j].x = 0.f; }
            if (!(mk[j] >> 8)) { un.y = 0.f; vn.y = 0.f; trs[j].y = 0.f; dets[j].y = 0.f; }
        }
        if (j < nrows) {
            if (vec_out) {
                *reinterpret_cast<float2 *>(uo + j * p.out_pitch) = un;
                *reinterpret_cast<float2 *>(vo + j * p.out_pitch) = vn;
            } else {
                uo[j * p.out_pitch] = un.x; vo[j * p.out_pitch] = vn.x;
                if (pair_ok) { uo[j * p.out_pitch + 1] = un.y; vo[j * p.out_pitch + 1] = vn.y; }
            }
        }
    }
    if (p.valid) {                                   // last iteration of level 0 only
        uint8_t *m = p.valid + (size_t)gy0 * W + gx;
        float *d = p.det + (size_t)gy0 * pitch + gx;
#pragma unroll
        for (int j = 0; j < SEG; ++j) {
            if (j < nrows) {
                m[j * W] = trs[j].x > 0.f ? 1 : 0;
                d[j * pitch] = dets[j].x;
                if (pair_ok) { m[j * W + 1] = trs[j].y > 0.f ? 1 : 0; d[j * pitch + 1] = dets[j].y; }
            }
        }
    }
}

// Shared-memory carve-up of the K3 ring: chunks | full barriers | empty barriers | task counter.
struct K3Smem {
    unsigned char *base;
    uint32_t ring0, full0, empty0;
    int *counter;
    __device__ __forceinline__ explicit K3Smem(unsigned char *b)
        : base(b), ring0(smem_u32(b)), full0(ring0 + K3_RING * K3_CHUNK_BYTES), empty0(full0 + 8 * K3_RING),
          counter(reinterpret_cast<int *>(b + K3_RING * K3_CHUNK_BYTES + 16 * K3_RING)) {}
};

// Thread 0 of the CTA, once per kernel, followed by __syncthreads.
template <int R> __device__ __forceinline__ void k3_init_barriers(const K3Smem &sm)
{
    for (int j = 0; j < K3_RING; ++j) {
        mbar_init(sm.full0 + 8 * j, 1);
        mbar_init(sm.empty0 + 8 * j, K3Geom<R>::NC);
    }
    sm.counter[0] = 0;
    sm.counter[1] = 0;                     // tile counter of the K2 pass in the persistent kernel
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

// Number of ring chunks a CTA that owns tasks [t_begin, t_end) consumes in one K3 pass (advances the chunk base).
template <int R> __device__ __forceinline__ int k3_cta_chunks(int t_begin, int t_end, int nrb)
{
    if (t_end <= t_begin) return 0;
    return (t_end - t_begin) + ((t_end - 1) / nrb - t_begin / nrb + 1) * (K3Geom<R>::NC - 1);
}

// One K3 pass over a level by the CTA that owns tasks [t_begin, t_end) (cta_range).  Warp `nwc` (the last one) is the producer, warps
// 0..nwc-1 consume.  `gc0` = number of ring chunks this CTA has consumed in earlier passes of the same
// kernel (keeps slot / parity bookkeeping continuous); *sm.counter must be 0 on entry (CTA-synchronised).
// All reads of u, v go through L2 (ld.global.cg): see of_k2.cuh.
// MK = an obstacle mask is set (p.md is valid): a separate instantiation (cf. of_k2.cuh).
// HM = hoisting mode (of_set_hoist; a, b, c are the same in every iteration of a level, reading D9):
//   0: five planes in, nothing kept (default);  1: five planes in, a, b, c also stored to p.G (first iteration of a level);
//   2: tmS is the two-plane map (box 64 x K3_SEG x 2) read at field 3: only IxIt, IyIt are fetched and summed, a, b, c come from p.G.
// The value of every sum is formed by the same instructions in the same order in all three modes.
template <int R, bool MK, int HM, bool BX>
__device__ __forceinline__ void k3_phase(const CUtensorMap *tmS, const K3Params &p, const K3Smem &sm, int warp, int lane, int nwc,
                                         int t_begin, int t_end, uint32_t gc0)
{
    typedef K3Geom<R> G;
    constexpr int NC = G::NC;
    constexpr int F0 = HM == 2 ? 3 : 0;                  // first field fetched and summed
    constexpr uint32_t CHUNK_TX = 64 * K3_SEG * (5 - F0) * 4;
    unsigned char *const k3_smem = sm.base;
    const uint32_t ring0 = sm.ring0, full0 = sm.full0, empty0 = sm.empty0;
    int *const counter = sm.counter;
    const int NWC = nwc;
    const int W = p.W, H = p.H, pitch = p.pitch, nrb = p.nrb;
    const int s_first = t_begin / nrb;
    // Task i of this CTA (global task t_begin+i in strip s) reads ring chunks gc0 + i + (s-s_first)*(NC-1) + k.

    if (warp == NWC) {
        // ===================== producer: the 32 lanes share the chunks of every run (lane k issues chunks k, k + 32, ...).
        // One lane needs ~105 cycles per bulk tensor copy (expect_tx + issue; measured, profiles/r2_notes.md, section 4), so a single
        // lane delivered the ~40 chunks of a level-0 pass only after ~6700 cycles; 32 lanes have them in flight after ~2300.
        // Consumers wait on the full barrier of each chunk, so the order of issue does not matter.
        if (!OF_DBG(p.dbg, 1)) {
            // one run = `ntask` consecutive tasks of strip s from row block rb0; its chunks start at ring chunk gbase
            auto produce_run = [&](int s, int rb0, int ntask, int gbase) {
                const int total = ntask + NC - 1;
                const int x0 = 64 * s, yc0 = K3_SEG * rb0 - R;          // chunk c holds rows yc0 + K3_SEG*c ...
                // batches of K3_BATCH chunks with a warp barrier in between: two uses of one ring slot are K3_RING > K3_BATCH chunks
                // apart, so no lane can wait for a slot's release two uses ahead (an mbarrier only tells the parity of its phase)
                static_assert(K3_RING > K3_BATCH && K3_RING >= NC + 2, "ring too small");
                for (int c0 = 0; c0 < total; c0 += K3_BATCH) {
                    const int c = c0 + lane;
                    if (lane < K3_BATCH && c < total) {
                        const int gc = gbase + c, slot = gc % K3_RING, use = gc / K3_RING;
                        if (use > 0) mbar_wait(empty0 + 8 * slot, (use - 1) & 1);
                        const int readers = min(ntask - 1, c) - max(0, c - NC + 1) + 1;
                        if (readers < NC) mbar_arrive(empty0 + 8 * slot, NC - readers);   // stand-ins for tasks that do not exist
                        mbar_expect_tx(full0 + 8 * slot, CHUNK_TX);
                        tma_load_3d(ring0 + slot * K3_CHUNK_BYTES, tmS, x0, yc0 + K3_SEG * c, F0, full0 + 8 * slot);
                    }
                    __syncwarp();
                }
            };
            if (MK) {                                                   // compacted lists: the host has cut the runs
                const K3Cta cd = p.md.k3_cta[blockIdx.x];
                for (int r = cd.run_b; r < cd.run_e; ++r) {
                    const K3Run rd = p.md.k3_runs[r];
                    const int s = rd.t0 / nrb;
                    produce_run(s, rd.t0 - s * nrb, rd.ntask, (int)gc0 + rd.chunk_off);
                }
            } else {
                for (int t = t_begin; t < t_end;) {
                    const int s = t / nrb, rb0 = t - s * nrb;
                    const int ntask = min(nrb - rb0, t_end - t);
                    produce_run(s, rb0, ntask, (int)gc0 + (t - t_begin) + (s - s_first) * (NC - 1));
                    t += ntask;
                }
            }
        }
        __syncwarp();                                   // production done (or nothing to produce): join the consumers
    }

    // ========================= consumers
    for (;;) {
        int i = 0;
        if (lane == 0) i = atomicAdd(counter, 1);
        i = __shfl_sync(0xffffffffu, i, 0);
        if (i >= t_end - t_begin) break;
        int gt = t_begin + i, gbase;
        if (MK) {
            const int2 e = __ldg(p.md.k3_ent + gt);
            gt = e.x;
            gbase = (int)gc0 + e.y;
        } else {
            gbase = (int)gc0 + i + (gt / nrb - s_first) * (NC - 1);
        }
        const int s = gt / nrb, rb = gt - s * nrb;
        const int gx = 64 * s + 2 * lane, gy0 = K3_SEG * rb;
        const bool active = gx < W;
        // this lane's field values, issued before the waits (rows past the image re-read the last row)
        const int nrows = min(K3_SEG, H - gy0);
        const float *ui = p.u_in + (size_t)gy0 * pitch + gx, *vi = p.v_in + (size_t)gy0 * pitch + gx;
        float2 uu[K3_SEG], vv[K3_SEG];
        unsigned mk[K3_SEG];                             // mask bytes of the lane's two columns, row by row (MK only)
#pragma unroll
        for (int j = 0; j < K3_SEG; ++j) {
            const int jj = min(j, nrows - 1) * pitch;
            mk[j] = 0x0101u;
            if (MK) mk[j] = active ? __ldg(reinterpret_cast<const unsigned short *>(p.md.mask + (size_t)gy0 * pitch + gx + jj)) : 0u;
            uu[j] = (active && !p.zero_uv) ? __ldcg(reinterpret_cast<const float2 *>(ui + jj)) : make_float2(0.f, 0.f);
            vv[j] = (active && !p.zero_uv) ? __ldcg(reinterpret_cast<const float2 *>(vi + jj)) : make_float2(0.f, 0.f);
        }
        float2 ga[K3_SEG], gb[K3_SEG], gcc[K3_SEG];      // HM = 2: the level's a, b, c (L2 reads: written by another pass of this launch)
        if (HM == 2) {
            const float *gp = p.G + (size_t)gy0 * pitch + gx;
#pragma unroll
            for (int j = 0; j < K3_SEG; ++j) {
                const int jj = min(j, nrows - 1) * pitch;
                ga[j] = active ? __ldcg(reinterpret_cast<const float2 *>(gp + jj)) : make_float2(0.f, 0.f);
                gb[j] = active ? __ldcg(reinterpret_cast<const float2 *>(gp + p.gplane + jj)) : make_float2(0.f, 0.f);
                gcc[j] = active ? __ldcg(reinterpret_cast<const float2 *>(gp + 2 * p.gplane + jj)) : make_float2(0.f, 0.f);
            }
        }
        const unsigned char *cb[NC];
        uint32_t eb[NC], fb[NC], fpar[NC];
#pragma unroll
        for (int k = 0; k < NC; ++k) {
            const int gc = gbase + k, slot = gc % K3_RING;
            cb[k] = k3_smem + slot * K3_CHUNK_BYTES + lane * 8;
            eb[k] = empty0 + 8 * slot;
            fb[k] = full0 + 8 * slot;
            fpar[k] = (gc / K3_RING) & 1;
        }
        float2 acc[5][K3_SEG], core[5];
#pragma unroll
        for (int f = 0; f < 5; ++f) {
            core[f] = make_float2(0.f, 0.f);
#pragma unroll
            for (int j = 0; j < K3_SEG; ++j) acc[f][j] = make_float2(0.f, 0.f);
        }
        auto sum_rows = [&](auto box) {
            constexpr bool BOX = decltype(box)::value;
#pragma unroll
            for (int r = 0; r < G::NIN; ++r) {
                if ((r % K3_SEG) == 0 && !OF_DBG(p.dbg, 1)) mbar_wait(fb[r / K3_SEG], fpar[r / K3_SEG]);   // chunk by chunk, as the TMA delivers them
#pragma unroll
                for (int f = F0; f < 5; ++f)
                    win_vrow<R, K3_SEG, BOX>(p.ww, r, *reinterpret_cast<const float2 *>(cb[r / K3_SEG] + (f - F0) * (K3_SEG * 256) + (r % K3_SEG) * 256),
                                             acc[f], core[f]);
            }
#pragma unroll
            for (int f = F0; f < 5; ++f) win_vfinish<K3_SEG, BOX>(acc[f], core[f]);
        };
        if (!OF_DBG(p.dbg, 2)) {
            sum_rows(std::integral_constant<bool, BX>());
        }
        __syncwarp();
        if (lane == 0 && !OF_DBG(p.dbg, 1)) {
#pragma unroll
            for (int k = 0; k < NC; ++k) mbar_arrive(eb[k], 1);
        }
        if (!active || OF_DBG(p.dbg, 4)) continue;
        if (HM == 1) {                                   // keep a, b, c for the later iterations of the level
            float *gp = p.G + (size_t)gy0 * pitch + gx;
#pragma unroll
            for (int j = 0; j < K3_SEG; ++j)
                if (j < nrows) {
                    *reinterpret_cast<float2 *>(gp + j * pitch) = acc[0][j];
                    *reinterpret_cast<float2 *>(gp + p.gplane + j * pitch) = acc[1][j];
                    *reinterpret_cast<float2 *>(gp + 2 * p.gplane + j * pitch) = acc[2][j];
                }
        }
        if (HM == 2) {
#pragma unroll
            for (int j = 0; j < K3_SEG; ++j) { acc[0][j] = ga[j]; acc[1][j] = gb[j]; acc[2][j] = gcc[j]; }
        }
        k3_solve_store<MK>(p, acc, uu, vv, mk, gx, gy0, nrows);
    }
}

template <int R, bool MK, bool BX>
__global__ void __launch_bounds__(32 * (K3_MAX_NW + 1), 1) k3_vsum_solve(const __grid_constant__ CUtensorMap tmS, const K3Params p)
{
    extern __shared__ __align__(1024) unsigned char k3_smem_[];
    const K3Smem sm(k3_smem_);
    if (threadIdx.x == 0) k3_init_barriers<R>(sm);
    __syncthreads();
    int t_begin, t_end;
    cta_range(p.ntasks, blockIdx.x, gridDim.x, t_begin, t_end);
    if (MK) { t_begin = p.md.k3_cta[blockIdx.x].ent_b; t_end = p.md.k3_cta[blockIdx.x].ent_e; }
    k3_phase<R, MK, 0, BX>(&tmS, p, sm, threadIdx.x >> 5, threadIdx.x & 31, (blockDim.x >> 5) - 1, t_begin, t_end, 0u);
}
