// of_k2.cuh -- K2: bilinear warp of I2 + central differences of I1 + It + five products + horizontal
// window sum (rows a4-a7 of the scope table; BASELINE.json:5 "(2) Per-iteration warp+gradient+product
// kernel"; readings D8-D12 of DESIGN.md).
//
// Warp-autonomous design for sm_100a: every WARP owns a tile of (8*nseg) x (2*nrp) outputs
// (nseg*nrp <= 32) and a private slice of shared memory; there is no block-level barrier, so the
// LSU-heavy product phase of one warp overlaps the FMA-heavy sum phase of the others on the same SM.
//
//   phase 1 (products): lane task = 2 columns x 2 rows.  All loads of I1/u/v are 8-byte vectors, I2
//       is gathered with 4 scalar loads per pixel (L1/L2 hits: the field is smooth).  The products of
//       a ROW PAIR are stored interleaved, {row y, row y+1} per column, so that phase 2 reads
//       register pairs that feed the packed fp32 FMA (FFMA2) directly.
//   phase 2 (horizontal sum): lane task = 8 adjacent outputs x 2 rows x 5 fields: (8+2RL)/2
//       LDS.128 and 8*(2R+1) FFMA2 per field; the window weight is the scalar (broadcast) operand.
//       Direct (2R+1)-tap sums: no running sums, no cancellation (H2), zero stays zero (D14 mask).
//
// Shared-memory layout per (field, row pair): column c at byte 8*c + 16*(c>>3) (16 B of padding per
// 8 columns -> the LDS.128 of phase 2, 64 B apart between lanes, are bank-conflict free).
#pragma once
#include "of_common.cuh"

#ifndef K2_AHEAD_MIN_ROUNDS
#define K2_AHEAD_MIN_ROUNDS 2                      // tiles with more product rounds than this request u, v of all rounds up front
#endif
#ifndef K2_AHEAD_MAX_ROUNDS
#define K2_AHEAD_MAX_ROUNDS 5                      // ... and at most this many (32 segments of 8 columns + halo = 140 tasks)
#endif
#ifndef K2_MAX_WARPS
#define K2_MAX_WARPS 12                            // warps per CTA (independent of each other); runtime blockDim
#endif

template <int R> struct K2Geom {
    static constexpr int RL = (R + 3) / 4 * 4;     // left/right halo rounded up: aligned vector loads
    static constexpr int OFF = RL - R;             // first tap sits OFF columns into the halo
    static constexpr int NIN = 8 + 2 * RL;         // input columns per phase-2 lane
    __host__ __device__ static constexpr int pw(int nseg) { return 8 * nseg + 2 * RL; }
    __host__ __device__ static constexpr int block_bytes(int nseg) { return pw(nseg) * 10; }
    __host__ __device__ static constexpr int warp_bytes(int nseg, int nrp) { return 5 * nrp * block_bytes(nseg); }
};

struct K2Params {
    const float *I1, *I2, *u, *v;
    float *S;
    size_t plane;
    int W, H, pitch;
    int nseg, nrp;                                 // lane layout of a warp tile
    int tiles_y, ntiles;                           // tile t -> (tx = t / tiles_y, ty = t % tiles_y)
    WinWeights ww;
    int zero_uv;                                   // 1 = the field is identically zero (first iteration at the coarsest level,
                                                   // PAPER.md:61 "initial guess of zero displacement"): u, v are not read
    int dbg;                                       // -DOF_PROFILE builds only: 1 = no product phase, 2 = no sum phase, 32 = no plane stores
    const uint8_t *mask;                           // obstacle mask of the level (pitch = `pitch`) or NULL (M2: zero weight)
    const int *list;                               // compacted tile list (then ntiles = its length) or NULL
    int f_first;                                   // first plane this pass forms: 0 = all five; 3 = IxIt, IyIt only (of_set_hoist:
                                                   // IxIx, IxIy, IyIy depend on I1 alone and keep their values of the level's first
                                                   // pass); read by the HO instantiation only
};

// Inputs of one phase-1 task (2 columns x 2 rows): I1 rows y-1..y+2 at columns x, x+1, the left and
// right neighbours of both rows, and the current field.  Loaded one round ahead (software prefetch).
// u, v are read through L2 only (ld.global.cg): the persistent solve kernel rewrites them between phases,
// so the non-coherent L1 path must not be used for them; I1 / I2 are read-only for a whole solve.
struct K2In {
    float2 cm, c0, c1, c2, u0, u1, v0, v1;
    float l0, q0, l1, q1;
    unsigned m0, m1;                               // mask bytes of (x, x+1) in rows y, y+1 (only read when a mask is set)
};

// base + 4*idx as ONE IMAD.WIDE (FMA pipe).  The integer/compare pipe (16 lanes per clock per SM sub-partition)
// is what bounds the product phase, so address arithmetic is kept off it.
__device__ __forceinline__ const float *ptr_at(const float *base, int idx)
{
    const float *r;
    asm("mad.wide.s32 %0, %1, 4, %2;" : "=l"(r) : "r"(idx), "l"(base));
    return r;
}

template <bool MK, bool LOADUV = true> __device__ __forceinline__ K2In k2_load(const K2Params &p, int x, int y)
{
    K2In in;
    const int W = p.W, H = p.H, pitch = p.pitch;
    const int i0 = y * pitch + x;                                  // one index, rows by +-pitch
    const int dm = y > 0 ? -pitch : 0, d1 = y + 1 < H ? pitch : 0, d2 = (y + 2 < H ? pitch : 0) + d1;
    const float *c = ptr_at(p.I1, i0), *c1p = ptr_at(c, d1);
    in.cm = __ldg(reinterpret_cast<const float2 *>(ptr_at(c, dm)));
    in.c0 = __ldg(reinterpret_cast<const float2 *>(c));
    in.c1 = __ldg(reinterpret_cast<const float2 *>(c1p));
    in.c2 = __ldg(reinterpret_cast<const float2 *>(ptr_at(c, d2)));
    if (p.zero_uv || !LOADUV) {
        in.u0 = in.u1 = in.v0 = in.v1 = make_float2(0.f, 0.f);
    } else {
        const float *pu = ptr_at(p.u, i0), *pv = ptr_at(p.v, i0);
        in.u0 = __ldcg(reinterpret_cast<const float2 *>(pu));
        in.u1 = __ldcg(reinterpret_cast<const float2 *>(ptr_at(pu, d1)));
        in.v0 = __ldcg(reinterpret_cast<const float2 *>(pv));
        in.v1 = __ldcg(reinterpret_cast<const float2 *>(ptr_at(pv, d1)));
    }
    in.m0 = in.m1 = 0x0101u;
    if (MK) {
        const uint8_t *pm = p.mask + i0;           // x is even and the pitch a multiple of 32: 2-byte aligned
        in.m0 = __ldg(reinterpret_cast<const unsigned short *>(pm));
        in.m1 = __ldg(reinterpret_cast<const unsigned short *>(pm + d1));
    }
    // left / right neighbours with clamp-to-edge: x-1 -> x at the left border, x+2 -> W-1 at the right
    const int ol = x > 0 ? -1 : 0, orr = x + 2 < W ? 2 : (x + 1 < W ? 1 : 0);
    in.l0 = __ldg(ptr_at(c, ol));
    in.q0 = __ldg(ptr_at(c, orr));
    in.l1 = __ldg(ptr_at(c1p, ol));
    in.q1 = __ldg(ptr_at(c1p, orr));
    return in;
}

// Bilinear sample of I2 at (x+u, y+v) (D8: the integer part of the displacement is added to the
// pixel index; x+u is never formed in fp32).  Clamp-to-edge is applied as: clamp the cell origin to
// [0, W-2] x [0, H-2] and force the fraction to 0 / 1 outside, which selects the same pixels as
// clamping both taps (and is exact at the borders), with two row pointers + immediate offsets
// instead of four separate addresses.  Split in two so that a lane can issue the gathers of all its
// pixels before it consumes the first one.
struct K2Tap { float i00, i01, i10, i11, ax, ay; };

// xf, yf = the pixel's coordinates as floats.  x + floor(u) is formed in fp32, which is exact (two integers
// below 2^24); x + u never is (D8).  Clamping is done on that float: Xc = clamp(X, 0, W-2), and the
// fraction becomes saturate(ax + (X - Xc)): unchanged inside, 0 left of the image, 1 right of it -- no
// compare / select instructions.
__device__ __forceinline__ K2Tap k2_gather(const float *__restrict__ I2, float xf, float yf, float Wm2f, float Hm2f, int pitch, float uu, float vv)
{
    K2Tap t;
    const float fu = floorf(uu), fv = floorf(vv);
    const float Xf = xf + fu, Yf = yf + fv;
    const float Xc = fminf(fmaxf(Xf, 0.f), Wm2f), Yc = fminf(fmaxf(Yf, 0.f), Hm2f);
    t.ax = __saturatef((uu - fu) + (Xf - Xc));
    t.ay = __saturatef((vv - fv) + (Yf - Yc));
    const float *p0 = ptr_at(I2, __float2int_rn(Yc) * pitch + __float2int_rn(Xc));
    const float *p1 = ptr_at(p0, pitch);
    t.i00 = __ldg(p0); t.i01 = __ldg(p0 + 1); t.i10 = __ldg(p1); t.i11 = __ldg(p1 + 1);
    return t;
}

// The four pixels of one phase-1 task: gathers first (k2_task_gather), products later (k2_task_products).
__device__ __forceinline__ void k2_task_gather(const K2Params &p, const K2In &in, int x, int y, K2Tap (&t)[4])
{
    const float Wm2f = (float)(p.W - 2), Hm2f = (float)(p.H - 2), xf = (float)x, yf = (float)y;
    t[0] = k2_gather(p.I2, xf, yf, Wm2f, Hm2f, p.pitch, in.u0.x, in.v0.x);
    t[1] = k2_gather(p.I2, xf, yf + 1.0f, Wm2f, Hm2f, p.pitch, in.u1.x, in.v1.x);
    t[2] = k2_gather(p.I2, xf + 1.0f, yf, Wm2f, Hm2f, p.pitch, in.u0.y, in.v0.y);
    t[3] = k2_gather(p.I2, xf + 1.0f, yf + 1.0f, Wm2f, Hm2f, p.pitch, in.u1.y, in.v1.y);
}

// It = I2w - I1 - Ix*u - Iy*v (D10) and the five products of the four pixels of a task, two pixels (rows y, y+1 of one column) per
// packed fp32 instruction (FADD2 / FMUL2 / FFMA2: every component is rounded exactly like the scalar instruction, so the values do
// not depend on the packing).  gx, gy are already multiplied by the validity mask (0 outside the image -> all five products are
// zero, D12).
__device__ __forceinline__ float2 k2_lerp2(const K2Tap &a, const K2Tap &b)
{
    const float2 one = make_float2(1.0f, 1.0f);
    const float2 ax = make_float2(a.ax, b.ax), ay = make_float2(a.ay, b.ay);
    const float2 bx = __fadd2_rn(one, make_float2(-a.ax, -b.ax)), by = __fadd2_rn(one, make_float2(-a.ay, -b.ay));
    const float2 top = __ffma2_rn(ax, make_float2(a.i01, b.i01), __fmul2_rn(bx, make_float2(a.i00, b.i00)));
    const float2 bot = __ffma2_rn(ax, make_float2(a.i11, b.i11), __fmul2_rn(bx, make_float2(a.i10, b.i10)));
    return __ffma2_rn(ay, bot, __fmul2_rn(by, top));
}

// one column of a task: pixels (x, y) and (x, y+1)
__device__ __forceinline__ void k2_products2(float2 I2w, float2 uu, float2 vv, float2 c, float2 gx, float2 gy,
                                             float2 &xx, float2 &xy, float2 &yy, float2 &xt, float2 &yt)
{
    const float2 ngx = make_float2(-gx.x, -gx.y), ngy = make_float2(-gy.x, -gy.y);
    const float2 It = __ffma2_rn(ngy, vv, __ffma2_rn(ngx, uu, __fadd2_rn(I2w, make_float2(-c.x, -c.y))));
    xx = __fmul2_rn(gx, gx); xy = __fmul2_rn(gx, gy); yy = __fmul2_rn(gy, gy); xt = __fmul2_rn(gx, It); yt = __fmul2_rn(gy, It);
}

template <bool MK> __device__ __forceinline__ void k2_task_products(const K2Params &p, const K2In &cur, int x, int y, const K2Tap (&t)[4], float4 (&o)[5])
{
    const bool in1 = x + 1 < p.W, row1 = y + 1 < p.H;
    float m00 = 0.5f, m01 = in1 ? 0.5f : 0.f, m10 = row1 ? 0.5f : 0.f, m11 = (in1 && row1) ? 0.5f : 0.f;
    if (MK) {                                      // M2: an obstacle pixel gets zero gradients, hence five zero products
        m00 = (cur.m0 & 0xffu) ? m00 : 0.f; m01 = (cur.m0 >> 8) ? m01 : 0.f;
        m10 = (cur.m1 & 0xffu) ? m10 : 0.f; m11 = (cur.m1 >> 8) ? m11 : 0.f;
    }
    // column x (rows y, y+1), then column x+1
    const float2 ma = make_float2(m00, m10), mb = make_float2(m01, m11);
    const float2 rgt_a = make_float2(in1 ? cur.c0.y : cur.c0.x, in1 ? cur.c1.y : cur.c1.x);
    const float2 gxa = __fmul2_rn(ma, __fadd2_rn(rgt_a, make_float2(-cur.l0, -cur.l1)));
    const float2 gya = __fmul2_rn(ma, __fadd2_rn(make_float2(cur.c1.x, cur.c2.x), make_float2(-cur.cm.x, -cur.c0.x)));
    const float2 gxb = __fmul2_rn(mb, __fadd2_rn(make_float2(cur.q0, cur.q1), make_float2(-cur.c0.x, -cur.c1.x)));
    const float2 gyb = __fmul2_rn(mb, __fadd2_rn(make_float2(cur.c1.y, cur.c2.y), make_float2(-cur.cm.y, -cur.c0.y)));
    float2 xx, xy, yy, xt, yt;
    k2_products2(k2_lerp2(t[0], t[1]), make_float2(cur.u0.x, cur.u1.x), make_float2(cur.v0.x, cur.v1.x), make_float2(cur.c0.x, cur.c1.x), gxa, gya,
                 xx, xy, yy, xt, yt);
    o[0].x = xx.x; o[0].y = xx.y; o[1].x = xy.x; o[1].y = xy.y; o[2].x = yy.x; o[2].y = yy.y; o[3].x = xt.x; o[3].y = xt.y; o[4].x = yt.x; o[4].y = yt.y;
    k2_products2(k2_lerp2(t[2], t[3]), make_float2(cur.u0.y, cur.u1.y), make_float2(cur.v0.y, cur.v1.y), make_float2(cur.c0.y, cur.c1.y), gxb, gyb,
                 xx, xy, yy, xt, yt);
    o[0].z = xx.x; o[0].w = xx.y; o[1].z = xy.x; o[1].w = xy.y; o[2].z = yy.x; o[2].w = yy.y; o[3].z = xt.x; o[3].w = xt.y; o[4].z = yt.x; o[4].w = yt.y;
}

// One K2 pass over a level by one CTA: it owns the contiguous range [t_begin, t_end) of warp tiles
// (cta_range) and its warps pull tiles from `tile_counter` (shared memory, 0 on entry, CTA-synchronised), so
// fast warps take more tiles.  Which warp computes a tile does not change its arithmetic.  `smem_cta`
// is the CTA's dynamic shared memory, of which this warp uses slice `warp`.  Called by the stand-alone
// kernel below and by the persistent solve kernel (of_solve.cuh).
// MK = an obstacle mask is set (p.mask and p.list are valid): a separate instantiation, so that the unmasked
// path carries none of the mask's instructions or registers.
// HO = of_set_hoist: p.f_first selects the planes formed (0 otherwise, at compile time).
template <int R, bool MK, bool HO, bool BX>
__device__ __forceinline__ void k2_phase(const K2Params &p, unsigned char *smem_cta, int *tile_counter, int warp, int lane, int t_begin, int t_end)
{
    typedef K2Geom<R> G;
    const int nseg = p.nseg, nrp = p.nrp;
    const int f_first = HO ? p.f_first : 0;
    const int PW = G::pw(nseg), half = PW >> 1, BB = G::block_bytes(nseg);
    char *const sm = reinterpret_cast<char *>(smem_cta) + warp * G::warp_bytes(nseg, nrp);
    const int W = p.W, H = p.H, pitch = p.pitch;
    const int ntasks = half * nrp;
    const int TW = 8 * nseg, TH = 2 * nrp;
    // phase-2 role of this lane: (field group, row pair, segment).  Narrow tiles leave lanes free, so
    // up to five fields are summed side by side, which shortens the serial chain of a coarse-level pass.
    const int nf_par = max(1, min(5, 32 / (nseg * nrp)));
    const int h_seg = lane % nseg, h_rp = (lane / nseg) % nrp, h_f0 = lane / (nseg * nrp);

    for (;;) {
        int t = 0;
        if (lane == 0) t = atomicAdd(tile_counter, 1);
        t = __shfl_sync(0xffffffffu, t, 0) + t_begin;
        if (t >= t_end) break;
        if (MK) t = __ldg(p.list + t);
        const int tx = t / p.tiles_y, ty = t - tx * p.tiles_y;
        const int x0 = tx * TW, y0 = ty * TH, xs = x0 - G::RL;

        // ---------------- phase 1: products of (PW x TH) pixels -> shared memory
        // task k -> (row pair rp, column pair cp): input loads, then the 16 gathers of its four pixels,
        // then the arithmetic (other warps of the SM cover the two memory latencies)
        if (ntasks > 32 * K2_AHEAD_MIN_ROUNDS && ntasks <= 32 * K2_AHEAD_MAX_ROUNDS) {
        // wide tiles (three or more product rounds): the field values of ALL rounds of the tile are requested first, so that a
        // round's gathers wait for one L2 round trip (I1 / I2) instead of two (u, v, then I2).  Measured (profiles/r2_notes.md, section 3):
        // level-0 K2 pass 16.0 -> 15.1 us at 1280x1024, 57.2 -> 50.1 us at 2048x2048; one-round tiles of the coarse levels lose
        // 0.4 us with it (unrolled guards), so they keep the rolled loop below.
        constexpr int MAXR = K2_AHEAD_MAX_ROUNDS;          // (wider tiles take the rolled loop below.  Every unrolled round is ~350 instructions
                                                           // and the kernel is sensitive to its code size: 6 -> 5 rounds gave the hoisted kernel 7 %.
                                                           // One rolled loop with the requested values moved down a place per round was slower.)
        float2 pu0[MAXR], pu1[MAXR], pv0[MAXR], pv1[MAXR];
#pragma unroll
        for (int r = 0; r < MAXR; ++r) {
            pu0[r] = pu1[r] = pv0[r] = pv1[r] = make_float2(0.f, 0.f);
            const int k = lane + 32 * r;
            int rp = 0, cp = k;
            while (cp >= half) { cp -= half; ++rp; }
            const int x = xs + 2 * cp, y = y0 + 2 * rp;
            if (k < ntasks && !p.zero_uv && x >= 0 && x < W && y < H) {
                const int i0 = y * pitch + x, d1 = y + 1 < H ? pitch : 0;
                const float *qu = ptr_at(p.u, i0), *qv = ptr_at(p.v, i0);
                pu0[r] = __ldcg(reinterpret_cast<const float2 *>(qu));
                pu1[r] = __ldcg(reinterpret_cast<const float2 *>(ptr_at(qu, d1)));
                pv0[r] = __ldcg(reinterpret_cast<const float2 *>(qv));
                pv1[r] = __ldcg(reinterpret_cast<const float2 *>(ptr_at(qv, d1)));
            }
        }
#pragma unroll
        for (int r = 0; r < MAXR; ++r) {
            const int k = lane + 32 * r;
            if (32 * r >= ntasks || k >= ntasks || OF_DBG(p.dbg, 1)) continue;
            int rp = 0, cp = k;
            while (cp >= half) { cp -= half; ++rp; }
            const int x = xs + 2 * cp, y = y0 + 2 * rp;
            float4 o[5];
            if (x >= 0 && x < W && y < H) {
                K2In in = k2_load<MK, false>(p, x, y);
                in.u0 = pu0[r]; in.u1 = pu1[r]; in.v0 = pv0[r]; in.v1 = pv1[r];
                K2Tap t[4];
                k2_task_gather(p, in, x, y, t);
                k2_task_products<MK>(p, in, x, y, t, o);
            } else {
#pragma unroll
                for (int f = 0; f < 5; ++f) o[f] = make_float4(0.f, 0.f, 0.f, 0.f);
            }
            char *d = sm + rp * BB + cp * 16 + (cp >> 2) * 16;
#pragma unroll
            for (int f = 0; f < 5; ++f)
                if (f >= f_first) *reinterpret_cast<float4 *>(d + f * nrp * BB) = o[f];
        }
        } else
#pragma unroll 1
        for (int k = lane; k < ntasks && !OF_DBG(p.dbg, 1); k += 32) {
            int rp = 0, cp = k;
            while (cp >= half) { cp -= half; ++rp; }
            const int x = xs + 2 * cp, y = y0 + 2 * rp;
            float4 o[5];
            if (x >= 0 && x < W && y < H) {
                const K2In in = k2_load<MK>(p, x, y);
                K2Tap t[4];
                k2_task_gather(p, in, x, y, t);
                k2_task_products<MK>(p, in, x, y, t, o);
            } else {
#pragma unroll
                for (int f = 0; f < 5; ++f) o[f] = make_float4(0.f, 0.f, 0.f, 0.f);
            }
            char *d = sm + rp * BB + cp * 16 + (cp >> 2) * 16;
#pragma unroll
            for (int f = 0; f < 5; ++f)
                if (f >= f_first) *reinterpret_cast<float4 *>(d + f * nrp * BB) = o[f];
        }
        __syncwarp();

        // ---------------- phase 2: horizontal window sum, 8 outputs x 2 rows per lane
        if (h_f0 < nf_par && !OF_DBG(p.dbg, 2)) {
            const int gx = x0 + 8 * h_seg, gy = y0 + 2 * h_rp;
            const char *src = sm + h_rp * BB + h_seg * 80;
#pragma unroll 1
            for (int f = f_first + h_f0; f < 5; f += nf_par) {
                float2 in[G::NIN];
#pragma unroll
                for (int k = 0; k < G::NIN / 2; ++k) {
                    const float4 q = *reinterpret_cast<const float4 *>(src + f * nrp * BB + 16 * k + 16 * (k >> 2));
                    in[2 * k] = make_float2(q.x, q.y);
                    in[2 * k + 1] = make_float2(q.z, q.w);
                }
                float2 acc[8];
                win_hsum8<R, G::OFF, G::NIN, BX>(p.ww, in, acc);
                if (gx < pitch && !OF_DBG(p.dbg, 32)) {
                    float *d0 = p.S + f * p.plane + (size_t)gy * pitch + gx;
                    if (gy < H) {
                        *reinterpret_cast<float4 *>(d0) = make_float4(acc[0].x, acc[1].x, acc[2].x, acc[3].x);
                        *reinterpret_cast<float4 *>(d0 + 4) = make_float4(acc[4].x, acc[5].x, acc[6].x, acc[7].x);
                    }
                    if (gy + 1 < H) {
                        *reinterpret_cast<float4 *>(d0 + pitch) = make_float4(acc[0].y, acc[1].y, acc[2].y, acc[3].y);
                        *reinterpret_cast<float4 *>(d0 + pitch + 4) = make_float4(acc[4].y, acc[5].y, acc[6].y, acc[7].y);
                    }
                }
            }
        }
        __syncwarp();
    }
}

template <int R, bool MK, bool BX>
__global__ void __launch_bounds__(32 * K2_MAX_WARPS, 1) k2_products_hsum(const K2Params p)
{
    extern __shared__ float4 smem4[];                          // warp slices, then 16 bytes for the tile counter
    int *tile_counter = reinterpret_cast<int *>(reinterpret_cast<unsigned char *>(smem4) +
                                                (blockDim.x >> 5) * K2Geom<R>::warp_bytes(p.nseg, p.nrp));
    if (threadIdx.x == 0) *tile_counter = 0;
    __syncthreads();
    int t_begin, t_end;
    cta_range(p.ntiles, blockIdx.x, gridDim.x, t_begin, t_end);
    k2_phase<R, MK, false, BX>(p, reinterpret_cast<unsigned char *>(smem4), tile_counter, threadIdx.x >> 5, threadIdx.x & 31, t_begin, t_end);
}
