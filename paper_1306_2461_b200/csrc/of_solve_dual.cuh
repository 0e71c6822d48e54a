// of_solve_dual.cuh -- the persistent solve kernel for TWO independent frame pairs in one cooperative launch (throughput mode of
// rows a3-a10 of the scope table; "the computation of a velocity field is independent of all other computations").
//
// Why: in of_solve_pair every pass ends in a grid barrier (one L2 atomic + an acquire spin, 1.1-1.6 us), 62 of them per pair at config 3
// = 60 of 488 us, and on top of that every CTA waits there for the slowest one (profiles/r2_solve.md: 27 % of all warp samples sit in front
// of barriers).  The barrier cannot be made much cheaper -- it is two dependent L2 round trips -- but it can be taken off the critical
// path: with two pairs A and B in flight the passes alternate, A's pass, then B's pass, and the barrier is SPLIT: a CTA ARRIVES on A's
// counter when it has finished its part of A's pass, runs its part of B's pass, and only at the end of that checks A's counter, which by
// then has long been complete.  No CTA ever spins unless another CTA is a whole pass behind, and there is ONE CTA barrier per pass.
//
// Each pair has its own handle, hence its own planes, fields, pyramids and barrier counter; the arithmetic of every value, the tile
// and task plans and the order of the passes of one pair are those of of_solve_pair (the same k2_phase / k3_phase / fused_iteration /
// upsample_phase are called), so both results are bit-identical to two single solves (tests/test_gpu_parity.py).  The price is
// latency: a pair's field is ready when both are.  Unmasked, un-hoisted form only; of_compute_dual falls back to two launches otherwise.
#pragma once
#include "of_solve.cuh"

// Split grid barrier.  Each pair has a counter that is 0 at launch; at the end of each of its passes every CTA adds 1 to it (release:
// the CTA barrier in front orders the CTA's stores of the pass before it), so "pass r of that pair is complete everywhere" reads
// counter >= r * ncta.  The WAIT for a pair's counter is not placed in front of that pair's next pass but at the end of the OTHER pair's
// pass that runs in between: thread 0 polls (acquire) when it has run out of work, in front of the CTA barrier that ends the pass, so the
// poll -- one L2 round trip in the steady state, the counter being long complete -- is covered by the warps still working, and the one
// CTA barrier per pass both ends the pass and hands the acquired state to all warps.  After it thread 0 alone pays for the release
// (fence + atomic); the other warps are already in the next pass, where work is handed out by counters.
//   reset: shared-memory work counter of the pass that ended (next used two passes later), or NULL.
__device__ __forceinline__ void dual_end_pass(unsigned *bar_self, const unsigned *bar_other, unsigned other_target, int *reset)
{
    if (threadIdx.x == 0 && other_target != 0)
        while (ld_acquire_u32(bar_other) < other_target) { }
    __syncthreads();
    if (threadIdx.x == 0) {
        if (reset != nullptr) *reset = 0;
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar_self) : "memory");
    }
}

template <int R, bool BX>
__global__ void __launch_bounds__(32 * SOLVE_WARPS, 1) of_solve_dual(const __grid_constant__ SolveArgs a0, const __grid_constant__ SolveArgs a1)
{
    extern __shared__ __align__(1024) unsigned char solve_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int cta = blockIdx.x, ncta = gridDim.x;
    const K3Smem sm(solve_smem);
    if (threadIdx.x == 0) {
        k3_init_barriers<R>(sm);
        sm.counter[2] = 0;                                       // work counters: K3 tasks of pair q in counter[2q], K2 tiles in counter[2q + 1]
        sm.counter[3] = 0;
    }
    __syncthreads();

    uint32_t gc0 = 0;                                            // ring chunks consumed so far by this CTA (both pairs)
    unsigned n = 0;                                              // rounds completed = arrivals made on each counter before this round
    int pi = 0;
    prof_stamp(a0, pi);
    const int top = a0.levels - 1, iterations = a0.iterations;   // same geometry for both pairs (checked by of_compute_dual)
    // Everything that is the same for both pairs (window weights, conditioning, sizes, plans) is read from a0, i.e. from fixed
    // offsets of the constant bank: the window weights are the broadcast operand of every FFMA2 of the sums, and through the
    // run-time choice `q ? a1 : a0` they would become generic loads into registers (measured: passes 25-30 % slower).
    // counter value the OTHER pair must have reached before its next pass may start, polled at the end of pair q's pass of round n
    // (pair 0's next pass belongs to round n + 1; nothing follows the last pass of the launch)
#define DUAL_OTHER_TARGET(q, final_round) ((q) == 0 ? n * ncta : ((final_round) ? 0u : (n + 1) * ncta))
    for (int l = top; l >= 0; --l) {
        const bool fused = a0.lv[l].f_ntiles > 0;
        if (l < top) {
#pragma unroll 1
            for (int q = 0; q < 2; ++q) {
                const SolveArgs &a = q ? a1 : a0;
                const SolveArgs &o = q ? a0 : a1;
                LevelDesc Lw = a.lv[l];
                if (fused && (iterations & 1)) { Lw.u = Lw.u2; Lw.v = Lw.v2; }
                upsample_phase<false>(Lw, a.lv[l + 1], nullptr, cta * blockDim.x + threadIdx.x, ncta * blockDim.x);
                dual_end_pass(a.gbar, o.gbar, DUAL_OTHER_TARGET(q, false), nullptr);
            }
            ++n;
            prof_stamp(a0, pi);
            prof_stamp(a0, pi);
        }
        if (fused) {
            for (int it = 0; it < iterations; ++it) {
                const bool last = (l == 0 && it == iterations - 1);
#pragma unroll 1
                for (int q = 0; q < 2; ++q) {
                    const SolveArgs &a = q ? a1 : a0;
                    const SolveArgs &o = q ? a0 : a1;
                    const LevelDesc L = a.lv[l];
                    // the field alternates between (u, v) and (u2, v2) and ends in (u, v): iteration `it` reads (u, v) iff iterations - it is even
                    const bool from_uv = ((iterations - it) & 1) == 0;
                    float *ui = from_uv ? L.u : L.u2, *vi = from_uv ? L.v : L.v2, *uo = from_uv ? L.u2 : L.u, *vo = from_uv ? L.v2 : L.v;
                    const FusedParams fp = {L.pyr[a.s1], L.pyr[a.s2], ui, vi, last ? a.u_out : uo, last ? a.v_out : vo, last ? a.valid : nullptr,
                                            last ? a.det : nullptr, L.W, L.H, L.pitch, last ? a.out_pitch : L.pitch, L.f_tw, L.f_th, L.f_tiles_x, L.f_ntiles,
                                            a0.ww, a0.sp, (l == top && it == 0) ? 1 : 0, nullptr};
                    fused_iteration<R, BX>(fp, solve_smem, cta, ncta);
                    dual_end_pass(a.gbar, o.gbar, DUAL_OTHER_TARGET(q, last), nullptr);
                }
                ++n;
                prof_stamp(a0, pi);                              // (four stamps per iteration, as in of_solve_pair)
                prof_stamp(a0, pi);
                prof_stamp(a0, pi);
                prof_stamp(a0, pi);
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the tile buffers were written by generic stores; a K3 pass copies into them
            continue;
        }
        int k2_b, k2_e, k3_b, k3_e;                              // this CTA's share of the level's tiles and tasks
        cta_range(a0.lv[l].k2_ntiles, cta, ncta, k2_b, k2_e);
        cta_range(a0.lv[l].k3_ntasks, cta, ncta, k3_b, k3_e);
        const uint32_t k3_chunks = (uint32_t)k3_cta_chunks<R>(k3_b, k3_e, a0.lv[l].k3_nrb);
        for (int it = 0; it < iterations; ++it) {
            const int zero_uv = (l == top && it == 0) ? 1 : 0;   // zero initial guess at the coarsest level
            const bool last = (l == 0 && it == iterations - 1);
            // ---- K2 pass of A, then of B: warp + gradients + products + horizontal sums -> five planes
#pragma unroll 1
            for (int q = 0; q < 2; ++q) {
                const SolveArgs &a = q ? a1 : a0;
                const SolveArgs &o = q ? a0 : a1;
                const LevelDesc L = a.lv[l];
                const K2Params p2 = {L.pyr[a.s1], L.pyr[a.s2], L.u, L.v, a.S, a.plane, L.W, L.H, L.pitch,
                                     L.k2_nseg, L.k2_nrp, L.k2_tiles_y, L.k2_ntiles, a0.ww, zero_uv, a0.dbg, nullptr, nullptr, 0};
                k2_phase<R, false, false, BX>(p2, solve_smem, sm.counter + 2 * q + 1, warp, lane, k2_b, k2_e);
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                dual_end_pass(a.gbar, o.gbar, DUAL_OTHER_TARGET(q, false), sm.counter + 2 * q + 1);
            }
            ++n;
            prof_stamp(a0, pi);
            prof_stamp(a0, pi);
            // ---- K3 pass of A, then of B: vertical sums + solve + update
#pragma unroll 1
            for (int q = 0; q < 2; ++q) {
                const SolveArgs &a = q ? a1 : a0;
                const SolveArgs &o = q ? a0 : a1;
                const LevelDesc L = a.lv[l];
                const K3Params p3 = {L.u, L.v, last ? a.u_out : L.u, last ? a.v_out : L.v, last ? a.valid : nullptr, last ? a.det : nullptr,
                                     L.W, L.H, L.pitch, last ? a.out_pitch : L.pitch, L.k3_nrb, L.k3_ntasks, a0.ww, a0.sp, zero_uv, a0.dbg, MaskDesc{}, nullptr, a.plane};
                K3Smem smq = sm;
                smq.counter = sm.counter + 2 * q;
                if (warp == SOLVE_WARPS - 1 && lane == 0) asm volatile("fence.proxy.async.global;" ::: "memory");
                k3_phase<R, false, 0, BX>(&a.tm[l], p3, smq, warp, lane, SOLVE_WARPS - 1, k3_b, k3_e, gc0);
                gc0 += k3_chunks;
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the ring was read by generic loads; the next K2 pass stores into it
                dual_end_pass(a.gbar, o.gbar, DUAL_OTHER_TARGET(q, last), smq.counter);
            }
            ++n;
            prof_stamp(a0, pi);
            prof_stamp(a0, pi);
        }
    }
#undef DUAL_OTHER_TARGET
    grid_barrier_exit(a0.gbar, ncta);
    grid_barrier_exit(a1.gbar, ncta);
}
