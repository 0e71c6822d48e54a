// of_common.cuh -- small shared definitions of the sm_100a kernels (no arithmetic of the method).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define OFK_MAX_R 16

// Profiling switches of the kernels (phases switched off one by one, profiles/r2_notes.md, section 2) exist in -DOF_PROFILE builds
// only: in the shipped build OF_DBG() is a compile-time 0 and the switches cost neither instructions nor registers.
#ifdef OF_PROFILE
#define OF_DBG(flags, bit) ((flags) & (bit))
#else
#define OF_DBG(flags, bit) 0
#endif

struct WinWeights {                                  // passed by value (param bank)
    float w[2 * OFK_MAX_R + 1];                      // w[t + R], t = -R..R
    int box;                                         // 1 = all weights are 1 (OF_WINDOW_BOX): the sums take the add-only path below
};

__device__ __forceinline__ int clampi(int i, int lo, int hi) { return max(lo, min(i, hi)); }

// Equal, contiguous share of n work items for CTA `cta` of `ncta` (n * ncta < 2^32).
__host__ __device__ __forceinline__ void cta_range(int n, int cta, int ncta, int &begin, int &end)
{
    begin = (int)((unsigned)n * (unsigned)cta / (unsigned)ncta);
    end = (int)((unsigned)n * (unsigned)(cta + 1) / (unsigned)ncta);
}

// packed fp32 pair FMA with a scalar weight (FFMA2 on sm_100a: half the issue slots of two FFMA)
__device__ __forceinline__ float2 fma2s(float w, float2 x, float2 acc) { return __ffma2_rn(x, make_float2(w, w), acc); }

// ---- window sums (D11, D12).  Two forms, chosen at COMPILE time (template parameter BX of the kernels: a kernel that
// carried both forms was 9500 instructions long and lost 3-7 % to instruction fetches), shared by K2, K3 and the fused coarse-level
// pass so that every caller forms a sum with the same instructions:
//   * weighted (Gaussian, and boxes of radius < 4): direct (2R+1)-tap sums, taps in ascending order, one FFMA2 per tap;
//   * box, R >= 4: the outputs of a lane share most of their taps, so the shared CORE is summed once and every output adds its few
//     private taps: add-only (no "add the entering value, subtract the leaving one"), hence no cancellation, a sum of non-negative
//     terms is positive iff one of them is (the validity decision tr > 0 stays exact) and zero stays zero; 2R+19 instead of 16R+8
//     packed instructions per 8 horizontal outputs, 2R+14 instead of 8R+4 per 4 vertical ones.
__host__ __device__ constexpr bool win_box_path(int R) { return R >= 4; }

// Horizontal: 8 adjacent outputs (x 2 rows, packed) of one field from NIN inputs; output j sums in[j+OFF .. j+OFF+2R].
template <int R, int OFF, int NIN, bool BX>
__device__ __forceinline__ void win_hsum8(const WinWeights &ww, const float2 (&in)[NIN], float2 (&acc)[8])
{
    static_assert(!BX || win_box_path(R), "the add-only path needs R >= 4");
    if (BX) {
        float2 core = in[7 + OFF];                                       // taps 7+OFF .. OFF+2R belong to all eight outputs
#pragma unroll
        for (int k = 8 + OFF; k <= OFF + 2 * R; ++k) core = __fadd2_rn(core, in[k]);
        float2 ls[7], rs[8];                                             // ls[j] = in[j+OFF] + .. + in[6+OFF]; rs[j] = in[OFF+2R+1] + .. + in[OFF+2R+j]
        ls[6] = in[6 + OFF];
#pragma unroll
        for (int j = 5; j >= 0; --j) ls[j] = __fadd2_rn(in[j + OFF], ls[j + 1]);
        rs[1] = in[OFF + 2 * R + 1];
#pragma unroll
        for (int j = 2; j < 8; ++j) rs[j] = __fadd2_rn(rs[j - 1], in[OFF + 2 * R + j]);
        acc[0] = __fadd2_rn(ls[0], core);
        acc[7] = __fadd2_rn(rs[7], core);
#pragma unroll
        for (int j = 1; j < 7; ++j) acc[j] = __fadd2_rn(__fadd2_rn(ls[j], rs[j]), core);
    } else {
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[j] = make_float2(0.f, 0.f);
        // input-major: one input pair feeds up to eight independent accumulators; the taps of an output are added left to right
#pragma unroll
        for (int i = 0; i < NIN; ++i)
#pragma unroll
            for (int j = 0; j < 8; ++j)
                if (i - j - OFF >= 0 && i - j - OFF <= 2 * R) acc[j] = fma2s(ww.w[i - j - OFF], in[i], acc[j]);
    }
}

// Vertical: input row r (0 .. SEG+2R-1, a compile-time constant in the unrolled caller) of a task of SEG output rows; output j sums
// rows j .. j+2R.  BOX = the add-only path: rows SEG-1 .. 2R go to `core`, which win_vfinish adds to every output at the end.
template <int R, int SEG, bool BOX>
__device__ __forceinline__ void win_vrow(const WinWeights &ww, int r, float2 val, float2 (&acc)[SEG], float2 &core)
{
    if (BOX) {
        if (r < SEG - 1) {
#pragma unroll
            for (int j = 0; j < SEG; ++j)
                if (j <= r) acc[j] = __fadd2_rn(acc[j], val);
        } else if (r <= 2 * R) {
            core = __fadd2_rn(core, val);
        } else {
#pragma unroll
            for (int j = 0; j < SEG; ++j)
                if (j >= r - 2 * R) acc[j] = __fadd2_rn(acc[j], val);
        }
    } else {
#pragma unroll
        for (int j = 0; j < SEG; ++j)
            if (r - j >= 0 && r - j <= 2 * R) acc[j] = fma2s(ww.w[r - j], val, acc[j]);
    }
}
template <int SEG, bool BOX>
__device__ __forceinline__ void win_vfinish(float2 (&acc)[SEG], float2 core)
{
    if (BOX) {
#pragma unroll
        for (int j = 0; j < SEG; ++j) acc[j] = __fadd2_rn(acc[j], core);
    }
}

// ---- obstacle masks (NEXT item f4; readings M1-M5 of DESIGN.md).  Built by the host in
// of_set_mask: per level a byte plane (pitch = the level's float pitch, 0 in the padding, 1 = fluid) and
// compacted work lists, so that a pass only visits tiles / tasks that hold or feed a fluid pixel and the
// remaining work is still split evenly over the CTAs.
struct K3Run { int t0, ntask, chunk_off, pad; };          // consecutive active tasks of one strip owned by one CTA;
                                                          // chunk_off = its first ring chunk, relative to the CTA's pass
struct K3Cta { int ent_b, ent_e, run_b, run_e, nchunks, pad0, pad1, pad2; };   // one CTA's share of a level
struct MaskDesc {                                         // all zero when no mask is set
    const uint8_t *mask;
    const int *k2_list;                                   // active K2 tiles, ascending
    const int2 *k3_ent;                                   // active K3 tasks, ascending: {task, first ring chunk rel. to the CTA's pass}
    const K3Run *k3_runs;
    const K3Cta *k3_cta;                                  // [number of CTAs]
    int k2_n, k3_n;
    const int *zero_list;                                 // level 0 only: K3 tasks without a fluid pixel (their outputs are zero-filled)
    int zero_n, pad;
};
