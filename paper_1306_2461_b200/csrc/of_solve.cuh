// of_solve.cuh -- the persistent solve kernel: every level, every iteration of one frame pair in ONE
// cooperative launch (rows a3-a10 of the scope table).
//
// Why: at 1280x1024 an iteration kernel runs 10-15 us and at the coarse levels 1-3 us, while a
// kernel boundary costs 2-4 us on B200 (measured: an empty K2/K3 launch, back to back in a stream,
// takes 4.1 us; profiles/r2_notes.md, section 2).  With ~65 launches per pair the boundaries were half
// of the time.  Here one CTA per SM stays resident and the K2 pass (of_k2.cuh), the K3 pass
// (of_k3.cuh) and the flow hand-down alternate, separated by a grid-wide barrier (one L2 atomic +
// one acquire spin, < 1 us).  The decomposition of the method is unchanged: K2 still writes the five
// horizontally summed planes, K3 still reads them back (through TMA) -- 72 B per pixel-iteration.
//
// Memory-model notes
//   * u, v are rewritten by the K3 pass and read by the next K2 pass on other SMs: both sides use
//     L2-only accesses (ld.global.cg) and the barrier carries __threadfence + acquire/release.
//   * the five planes are written with ordinary stores and read by the TMA unit (async proxy): the
//     producer lane issues fence.proxy.async.global after the barrier and before its first TMA.
//   * shared memory is a union of the K2 warp slices and the K3 ring: fence.proxy.async.shared::cta
//     after the K2 pass orders its generic-proxy stores before the TMA writes of the K3 pass.
#pragma once
#include "of_k2.cuh"
#include "of_k2s.cuh"
#include "of_k3.cuh"
#include "of_fused.cuh"

// K2 variant of the unmasked kernels: 0 (default) = warp tiles with global gathers (of_k2.cuh), 1 (-DOF_K2_STREAMING) = the
// task-queue form with the TMA-staged I2 window (of_k2s.cuh).  Both are kept bit-identical; profiles/r2_k2_streaming.md has the
// measurements that decided the default.
#ifdef OF_K2_STREAMING
#define SOLVE_K2S 1
#else
#define SOLVE_K2S 0
#endif

#define SOLVE_TIMELINE_MAX 4096
#ifndef SOLVE_WARPS
#define SOLVE_WARPS 12                       // 11 K3 consumers + 1 producer; all 12 work in the K2 pass
#endif
#ifndef SOLVE_CTAS_PER_SM
#define SOLVE_CTAS_PER_SM 1
#endif

struct LevelDesc {
    const float *pyr[2];                     // pyramid slots (I1 / I2 chosen per job)
    float *u, *v;
    int W, H, pitch;
    int k2_nseg, k2_nrp, k2_tiles_y, k2_ntiles;   // warp tiles of of_k2.cuh (masked instantiations)
    int k3_nrb, k3_ntasks;
    int k2s_nuy, k2s_nunits;                 // units of of_k2s.cuh: per strip, per level
    unsigned long long k2s_magic;            // ceil(2^40 / k2s_nuy)
    float *u2, *v2;                          // second field buffer of a fused level (of_fused.cuh)
    int f_tw, f_th, f_tiles_x, f_ntiles;     // fused coarse-level iteration: tile size and count, f_ntiles = 0: two-pass form
};

// Dynamic shared memory of the solve kernel: [0, 225280) data (K3 ring / K2 product buffers, A slots and I2 ring), then the K3
// barriers and counters (720 B), then the K2 barriers, descriptors and ticket counter.
#define SOLVE_K2S_BAR_OFF (K3_RING * K3_CHUNK_BYTES + 768)
template <int R> struct SolveSmem {
#if SOLVE_K2S
    static constexpr int BYTES = SOLVE_K2S_BAR_OFF + K2S<R>::BAR_BYTES;
    static_assert(K3Geom<R>::SMEM <= SOLVE_K2S_BAR_OFF && K2S<R>::DATA_BYTES <= K3_RING * K3_CHUNK_BYTES && K2S<R>::DATA_MAX == K3_RING * K3_CHUNK_BYTES,
                  "shared-memory map of the solve kernel");
#else
    static constexpr int BYTES = K3Geom<R>::SMEM;
#endif
};

#define SOLVE_MAX_LEVELS 12
struct SolveArgs {
    alignas(64) CUtensorMap tm[SOLVE_MAX_LEVELS];   // per level: the five planes as an (x, y, field) tensor; lives in
                                                    // the kernel's parameter space (__grid_constant__), no global fetch
    const LevelDesc *lv;                     // device array [levels]
    unsigned *gbar;                          // {arrival count, generation}, zero-initialised once
    float *S;
    size_t plane;
    float *u_out, *v_out;                    // dense level-0 result
    uint8_t *valid;
    float *det;
    int levels, iterations, s1, s2, out_pitch, dbg;
    unsigned long long *prof;                // optional timelines [ncta][SOLVE_TIMELINE_MAX] (SM clock at every phase boundary) or NULL
    WinWeights ww;
    SolveParams sp;
    const K2SMaps *k2maps;                   // device array [levels]: tensor maps of the K2 inputs (of_k2s.cuh)
    const MaskDesc *md;                      // device array [levels]: obstacle masks and work lists (read by the MK kernel only;
                                             // last, so that every other field keeps its place in the parameter bank)
    // of_set_hoist (HO instantiation only): the planes IxIt, IyIt of a level as an (x, y, field) tensor with a two-field
    // box, and the three planes that keep the level's window sums a, b, c
    float *G;
    alignas(64) CUtensorMap tm2[SOLVE_MAX_LEVELS];
};

__device__ __forceinline__ unsigned ld_acquire_u32(const unsigned *p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// Grid barrier k (k = 0, 1, ... within one launch) on a counter that is 0 at launch: every CTA adds 1
// with release semantics and spins (acquire) until the counter reaches (k+1)*ncta.  One L2 atomic and
// one or two L2 polls; no generation word, no reset between barriers.  grid_barrier_exit() returns the
// counter to 0 when the last CTA leaves the kernel, so a captured graph can replay the launch.
__device__ __forceinline__ void grid_barrier(unsigned *bar, unsigned ncta, unsigned &k)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned target = (k + 1) * ncta;
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");
#ifdef OF_WATCHDOG
        const long long t0 = clock64();
        while (ld_acquire_u32(bar) < target)
            if (clock64() - t0 > 2000000000ll) { printf("[optflow watchdog] block %d: grid barrier %u never completed\n", blockIdx.x, k); __trap(); }
#else
        while (ld_acquire_u32(bar) < target) { }
#endif
    }
    ++k;
    __syncthreads();
}

__device__ __forceinline__ void grid_barrier_exit(unsigned *bar, unsigned ncta)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned old = atomicInc(bar + 1, ncta - 1);      // wraps to 0 with the last CTA
        if (old == ncta - 1) atomicExch(bar, 0u);                // every CTA has passed the last barrier
    }
}

__device__ __forceinline__ void prof_stamp(const SolveArgs &a, int &idx)
{
    if (a.prof != nullptr) {
        // stamp when the whole CTA is done, not just warp 0: the clock read consumes the barrier's reduction result, so it cannot
        // be issued before the barrier has released (a plain bar.sync lets the warp run ahead to the clock read)
        const int n = __syncthreads_count(1);
        if (threadIdx.x == 0) {
            // SM cycle counter: %globaltimer is refreshed too coarsely (several us) to time a pass
            unsigned long long t;
            asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.s32 p, %1, 0;\n\t@p mov.u64 %0, %%clock64;\n\t@!p mov.u64 %0, 0;\n\t}" : "=l"(t) : "r"(n) : "memory");
            a.prof[(size_t)blockIdx.x * SOLVE_TIMELINE_MAX + idx] = t;
        }
    }
    ++idx;
}

// M3 for the level-0 tasks no K3 pass visits: u = v = 0, valid = 0, det = 0.  One warp per task (64 x K3_SEG pixels).
__device__ __forceinline__ void mask_zero_tasks(const int *zl, int n, int nrb, int W, int H, int pitch, float *u_out, float *v_out,
                                                int out_pitch, uint8_t *valid, float *det, int gwarp, int nwarps, int lane)
{
    for (int i = gwarp; i < n; i += nwarps) {
        const int t = __ldg(zl + i), s = t / nrb, rb = t - s * nrb;
        for (int j = 0; j < K3_SEG; ++j) {
            const int y = K3_SEG * rb + j;
            for (int k = 0; k < 2; ++k) {
                const int x = 64 * s + 32 * k + lane;
                if (x < W && y < H) {
                    u_out[(size_t)y * out_pitch + x] = 0.f;
                    v_out[(size_t)y * out_pitch + x] = 0.f;
                    valid[(size_t)y * W + x] = 0;
                    det[(size_t)y * pitch + x] = 0.f;
                }
            }
        }
    }
}

static __global__ void __launch_bounds__(256) k_mask_zero(const int *zl, int n, int nrb, int W, int H, int pitch, float *u_out, float *v_out,
                                                   int out_pitch, uint8_t *valid, float *det)
{
    mask_zero_tasks(zl, n, nrb, W, H, pitch, u_out, v_out, out_pitch, valid, det, (blockIdx.x * blockDim.x + threadIdx.x) >> 5,
                    (gridDim.x * blockDim.x) >> 5, threadIdx.x & 31);
}

// Flow hand-down (row a10, D6): u_l = 2*bilinear(u_{l+1}; x/2, y/2), grid-stride over the fine level.
template <bool MK>
__device__ __forceinline__ void upsample_phase(const LevelDesc &F, const LevelDesc &C, const uint8_t *fmask, int gtid, int nthreads)
{
    const int W = F.W, H = F.H, Wc = C.W, Hc = C.H, cp = C.pitch, qw = (W + 3) >> 2;
    for (int i = gtid; i < qw * H; i += nthreads) {              // four adjacent fine pixels per thread
        const int y = i / qw, x = 4 * (i - y * qw);
        const int x0 = x >> 1, x1 = min(x0 + 1, Wc - 1), x2 = min(x0 + 2, Wc - 1), y0 = y >> 1, y1 = min(y0 + 1, Hc - 1);
        const float fy = (y & 1) * 0.5f, gy = 1.0f - fy;
        const float *ur0 = C.u + y0 * cp, *ur1 = C.u + y1 * cp, *vr0 = C.v + y0 * cp, *vr1 = C.v + y1 * cp;
        uchar4 m = make_uchar4(1, 1, 1, 1);
        if (MK) m = __ldg(reinterpret_cast<const uchar4 *>(fmask + y * F.pitch + x));   // issued with the field loads
        const float a00 = __ldcg(ur0 + x0), a01 = __ldcg(ur0 + x1), a02 = __ldcg(ur0 + x2);
        const float a10 = __ldcg(ur1 + x0), a11 = __ldcg(ur1 + x1), a12 = __ldcg(ur1 + x2);
        const float b00 = __ldcg(vr0 + x0), b01 = __ldcg(vr0 + x1), b02 = __ldcg(vr0 + x2);
        const float b10 = __ldcg(vr1 + x0), b11 = __ldcg(vr1 + x1), b12 = __ldcg(vr1 + x2);
        // even fine x: fx = 0; odd fine x: fx = 1/2 (same expression tree as k4_upsample_flow)
        float uo[4], vo[4];
        uo[0] = 2.0f * (gy * (1.0f * a00 + 0.0f * a01) + fy * (1.0f * a10 + 0.0f * a11));
        uo[1] = 2.0f * (gy * (0.5f * a00 + 0.5f * a01) + fy * (0.5f * a10 + 0.5f * a11));
        uo[2] = 2.0f * (gy * (1.0f * a01 + 0.0f * a02) + fy * (1.0f * a11 + 0.0f * a12));
        uo[3] = 2.0f * (gy * (0.5f * a01 + 0.5f * a02) + fy * (0.5f * a11 + 0.5f * a12));
        vo[0] = 2.0f * (gy * (1.0f * b00 + 0.0f * b01) + fy * (1.0f * b10 + 0.0f * b11));
        vo[1] = 2.0f * (gy * (0.5f * b00 + 0.5f * b01) + fy * (0.5f * b10 + 0.5f * b11));
        vo[2] = 2.0f * (gy * (1.0f * b01 + 0.0f * b02) + fy * (1.0f * b11 + 0.0f * b12));
        vo[3] = 2.0f * (gy * (0.5f * b01 + 0.5f * b02) + fy * (0.5f * b11 + 0.5f * b12));
        if (MK) {                                                 // M3: the field stays zero over an obstacle
            if (!m.x) { uo[0] = 0.f; vo[0] = 0.f; }
            if (!m.y) { uo[1] = 0.f; vo[1] = 0.f; }
            if (!m.z) { uo[2] = 0.f; vo[2] = 0.f; }
            if (!m.w) { uo[3] = 0.f; vo[3] = 0.f; }
        }
        float *pu = F.u + y * F.pitch + x, *pv = F.v + y * F.pitch + x;
        if (x + 3 < W) {
            *reinterpret_cast<float4 *>(pu) = make_float4(uo[0], uo[1], uo[2], uo[3]);
            *reinterpret_cast<float4 *>(pv) = make_float4(vo[0], vo[1], vo[2], vo[3]);
        } else {
            for (int k = 0; x + k < W; ++k) { pu[k] = uo[k]; pv[k] = vo[k]; }
        }
    }
}

// MK = an obstacle mask is set (of_set_mask): compacted work lists, masked products / outputs.
// HO = of_set_hoist: IxIx, IxIy, IyIy and their window sums a, b, c are formed in the first iteration of a level only
// (they depend on I1 alone, reading D9): later iterations write, fetch and sum the two It planes (60 B per pixel-iteration
// instead of 72).  A separate instantiation: the default kernel carries none of it.
// BX = box window: the sums take the add-only form (of_common.cuh).
template <int R, bool MK, bool HO, bool BX>
__global__ void __launch_bounds__(32 * SOLVE_WARPS, SOLVE_CTAS_PER_SM) of_solve_pair(const __grid_constant__ SolveArgs a)
{
    extern __shared__ __align__(1024) unsigned char solve_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int cta = blockIdx.x, ncta = gridDim.x;
    const K3Smem sm(solve_smem);
    const K2SSmem<R> sm2(solve_smem, solve_smem + SOLVE_K2S_BAR_OFF);
    if (threadIdx.x == 0) {
        if (SOLVE_K2S && !MK) k2s_init_barriers<R>(sm2);
        k3_init_barriers<R>(sm);
    }
    __syncthreads();

    uint32_t gc0 = 0;                                            // ring chunks consumed so far by this CTA
    uint32_t uk0 = 0;                                            // K2 units processed so far by this CTA
    unsigned nbar = 0;                                           // grid barriers passed so far
    int pi = 0;
    prof_stamp(a, pi);
    const int top = a.levels - 1;
    if (MK && a.md[0].zero_n > 0)                                // disjoint from everything the passes write: no barrier needed
        mask_zero_tasks(a.md[0].zero_list, a.md[0].zero_n, a.lv[0].k3_nrb, a.lv[0].W, a.lv[0].H, a.lv[0].pitch, a.u_out, a.v_out, a.out_pitch,
                        a.valid, a.det, cta * SOLVE_WARPS + warp, ncta * SOLVE_WARPS, lane);
    for (int l = top; l >= 0; --l) {
        const LevelDesc L = a.lv[l];
        MaskDesc M = {};
        if (MK) M = a.md[l];
        // fused coarse level (of_fused.cuh): the field alternates between (u, v) and (u2, v2); start so that the last iteration ends in (u, v)
        const bool fused = L.f_ntiles > 0;
        LevelDesc Lw = L;
        if (fused && (a.iterations & 1)) { Lw.u = L.u2; Lw.v = L.v2; }
        if (l < top) {
            upsample_phase<MK>(Lw, a.lv[l + 1], M.mask, cta * blockDim.x + threadIdx.x, ncta * blockDim.x);
            prof_stamp(a, pi);
            if (!OF_DBG(a.dbg, 8)) grid_barrier(a.gbar, ncta, nbar); else __syncthreads();
            prof_stamp(a, pi);
        }
        if (fused) {
            float *ui = Lw.u, *vi = Lw.v, *uo = (ui == L.u) ? L.u2 : L.u, *vo = (vi == L.v) ? L.v2 : L.v;
            for (int it = 0; it < a.iterations; ++it) {
                const bool last = (l == 0 && it == a.iterations - 1);
                const FusedParams fp = {L.pyr[a.s1], L.pyr[a.s2], ui, vi, last ? a.u_out : uo, last ? a.v_out : vo, last ? a.valid : nullptr,
                                        last ? a.det : nullptr, L.W, L.H, L.pitch, last ? a.out_pitch : L.pitch, L.f_tw, L.f_th, L.f_tiles_x, L.f_ntiles,
                                        a.ww, a.sp, (l == top && it == 0) ? 1 : 0, M.mask};
                fused_iteration<R, BX, MK>(fp, solve_smem, cta, ncta);
                prof_stamp(a, pi);                               // (four stamps per iteration, as in the two-pass form)
                prof_stamp(a, pi);
                prof_stamp(a, pi);
                if (!last) { if (!OF_DBG(a.dbg, 8)) grid_barrier(a.gbar, ncta, nbar); else __syncthreads(); }
                prof_stamp(a, pi);
                float *tu = ui, *tv = vi;
                ui = uo; vi = vo; uo = tu; vo = tv;
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the tile buffers were written by generic stores; a K3 pass copies into them
            continue;
        }
        int k2_b, k2_e, k3_b, k3_e;                              // this CTA's share of the level's tiles and tasks
        cta_range(MK ? M.k2_n : (SOLVE_K2S ? L.k2s_nunits : L.k2_ntiles), cta, ncta, k2_b, k2_e);
        cta_range(L.k3_ntasks, cta, ncta, k3_b, k3_e);
        uint32_t k3_chunks = (uint32_t)k3_cta_chunks<R>(k3_b, k3_e, L.k3_nrb);
        if (MK) {                                                // mask set: the host has cut the compacted task list per CTA
            const K3Cta cd = M.k3_cta[cta];
            k3_b = cd.ent_b; k3_e = cd.ent_e; k3_chunks = (uint32_t)cd.nchunks;
        }
        K2Params p2 = {L.pyr[a.s1], L.pyr[a.s2], L.u, L.v, a.S, a.plane, L.W, L.H, L.pitch,
                       L.k2_nseg, L.k2_nrp, L.k2_tiles_y, L.k2_ntiles, a.ww, 0, a.dbg, M.mask, M.k2_list, 0};
        K2SParams q2 = {a.k2maps + l, a.s2, L.pyr[a.s1], L.pyr[a.s2], L.u, L.v, a.S, a.plane, L.W, L.H, L.pitch, L.k2s_nuy, L.k2s_nunits, L.k2s_magic, a.ww, 0, 0};
        for (int it = 0; it < a.iterations; ++it) {
            // ---- K2 pass: warp + gradients + products + horizontal sums -> five planes
            p2.zero_uv = (l == top && it == 0) ? 1 : 0;            // zero initial guess at the coarsest level
            p2.f_first = (HO && it > 0) ? 3 : 0;
            if constexpr (MK || !SOLVE_K2S) {
                k2_phase<R, MK, HO, BX>(p2, solve_smem, sm.counter + 1, warp, lane, k2_b, k2_e);
            } else {
                q2.zero_uv = p2.zero_uv; q2.f_first = p2.f_first;
                k2s_phase<R, HO, BX>(q2, sm2, warp, lane, k2_b, k2_e, uk0);
                uk0 += (uint32_t)(k2_e - k2_b);
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            prof_stamp(a, pi);
            if (!OF_DBG(a.dbg, 8)) grid_barrier(a.gbar, ncta, nbar); else __syncthreads();
            prof_stamp(a, pi);
            // ---- K3 pass: vertical sums + solve + update
            const bool last = (l == 0 && it == a.iterations - 1);
            K3Params p3 = {L.u, L.v, last ? a.u_out : L.u, last ? a.v_out : L.v, last ? a.valid : nullptr, last ? a.det : nullptr,
                           L.W, L.H, L.pitch, last ? a.out_pitch : L.pitch, L.k3_nrb, L.k3_ntasks, a.ww, a.sp, p2.zero_uv, a.dbg, M, HO ? a.G : nullptr, a.plane};
            if (warp == SOLVE_WARPS - 1 && lane == 0) asm volatile("fence.proxy.async.global;" ::: "memory");
            if (!HO) k3_phase<R, MK, 0, BX>(&a.tm[l], p3, sm, warp, lane, SOLVE_WARPS - 1, k3_b, k3_e, gc0);
            else if (it == 0) k3_phase<R, MK, 1, BX>(&a.tm[l], p3, sm, warp, lane, SOLVE_WARPS - 1, k3_b, k3_e, gc0);
            else k3_phase<R, MK, 2, BX>(&a.tm2[l], p3, sm, warp, lane, SOLVE_WARPS - 1, k3_b, k3_e, gc0);
            gc0 += k3_chunks;
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the ring was read by generic loads; the next K2 pass copies into it
            __syncthreads();
            if (threadIdx.x == 0) { sm.counter[0] = 0; sm.counter[1] = 0; }
            prof_stamp(a, pi);
            if (!last) { if (!OF_DBG(a.dbg, 8)) grid_barrier(a.gbar, ncta, nbar); else __syncthreads(); }
            prof_stamp(a, pi);
        }
    }
    grid_barrier_exit(a.gbar, ncta);
}
