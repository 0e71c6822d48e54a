// optflow.cu -- host orchestration and C-ABI (include/optflow.h) of the dense optical-flow solve.
//
// Level loop / iteration loop / stream + event wiring / CUDA-graph replay; all arithmetic of the
// method runs in the kernels of of_kernels.cuh.  No CPU fallback anywhere: every path that cannot
// reach the GPU returns an error.
#include "../../include/optflow.h"
#include "of_kernels.cuh"
#include "of_solve.cuh"
#include "of_dispatch.cuh"
#include "of_equalise.cuh"
#include "of_post.cuh"

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

static_assert(OFK_MAX_R == OF_MAX_WINDOW_RADIUS, "radius limits out of sync");

namespace {

thread_local std::string g_err;

int fail(int code, const char *fmt, ...) __attribute__((format(printf, 2, 3)));
int fail(int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return code;
}

#define CU_TRY(expr)                                                                              \
    do {                                                                                          \
        cudaError_t e_ = (expr);                                                                  \
        if (e_ != cudaSuccess)                                                                    \
            return fail(OF_ERR_CUDA, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

struct Level { int W, H, pitch; };

// Launch geometry of the two iteration kernels at one level (chosen once in of_create).
struct K2Plan { int nseg, nrp, tiles_y, ntiles, grid, warps, smem; };
struct K3Plan { int nrb, ntasks, grid, warps, smem; };
constexpr int SMEM_MAX = 227 * 1024;

// One enqueue of the whole path.  Also the key of the graph cache.
struct Job {
    int dtype;                 // of_dtype of rawA/rawB
    const void *rawA, *rawB;   // frames to convert into pyramid slots cvtA / cvtB (rawB may be NULL)
    int cvtA, cvtB;            // pyramid slots to (re)build, -1 = none
    int s1, s2;                // pyramid slots used as I1 / I2
    float *u_out, *v_out;      // level-0 result, dense
    uint8_t *valid_out;        // validity bytes of the result (the handle's own plane, or a slot of the streaming result ring)
    bool operator==(const Job &o) const { return memcmp(this, &o, sizeof(Job)) == 0; }
};

struct GraphEntry { Job job; cudaGraphExec_t exec; unsigned long long stamp; int launches; };

constexpr int N_PYR = 2;       // pyramid slots
constexpr int N_PIN = 4;       // pinned upload slots (the paper's double buffering, two deeper: up to N_RES - 2 = 3 fields may be in flight)
constexpr int N_RES = 5;       // result ring: a returned field stays valid until the second-next of_stream_result call

struct Pipeline {
    bool open = false;
    int dtype = 0, mode = 0, host_result = 0;
    size_t frame_bytes = 0, slot_bytes = 0, field_bytes = 0;
    cudaStream_t s_copy = nullptr, s_comp = nullptr, s_down = nullptr;
    void *pin[N_PIN] = {};
    void *raw[N_PIN] = {};
    float *res_dev[N_RES] = {};            // per slot: u, v (2 x field_bytes), then the validity bytes (W*H)
    float *res_host[N_RES] = {};
    cudaEvent_t h2d_done[N_PIN] = {}, cvt_done[N_PIN] = {}, solve_done[N_RES] = {}, d2h_done[N_RES] = {};
    bool cvt_rec[N_PIN] = {}, d2h_rec[N_RES] = {};
    long long acquired = 0, submitted = 0, produced = 0, collected = 0;
    int cur_slot = -1;
    const uint8_t *last_valid = nullptr;   // validity bytes of the field of_stream_result returned last
};

}  // namespace

struct of_context {
    int W, H, levels, R, iterations, window_type;
    int device;
    float eps_rel, max_step;
    int eq_radius;                      // 0 = frames are converted as they are; > 0 = eq. 2 pre-filter of that radius
    Level lv[OF_MAX_LEVELS];
    float *pyr[N_PYR][OF_MAX_LEVELS];
    float *u[OF_MAX_LEVELS], *v[OF_MAX_LEVELS];
    float *u2[OF_MAX_LEVELS], *v2[OF_MAX_LEVELS];      // second field buffer of the levels iterated in fused form (of_fused.cuh)
    int f_tw[OF_MAX_LEVELS], f_th[OF_MAX_LEVELS], f_tiles_x[OF_MAX_LEVELS], f_ntiles[OF_MAX_LEVELS];
    bool fuse_coarse;                   // of_set_fused: coarse levels iterate inside the CTA (default on)
    float *S;
    size_t plane;
    float *det;
    uint8_t *valid;
    WinWeights ww;
    int sms, dbg;
    K2Plan k2[OF_MAX_LEVELS];
    K3Plan k3[OF_MAX_LEVELS];
    CUtensorMap tmS[OF_MAX_LEVELS];     // the five summed planes of a level as one (x, y, field) tensor
    K2SMaps *d_k2maps;                  // tensor maps of the K2 inputs per level (of_k2s.cuh), device array
    int k2s_nuy[OF_MAX_LEVELS], k2s_nunits[OF_MAX_LEVELS];
    LevelDesc *d_lv;                    // device copies for the persistent solve kernel
    MaskDesc *d_md;
    CUtensorMap *d_tm;
    unsigned *d_gbar;
    unsigned *d_post;                   // scratch of the post-processing reductions (min/max words)
    unsigned long long *d_prof;         // timeline buffer of the persistent kernel (of_solve_timeline)
    bool prof_on;
    bool persistent;                    // whole solve in one cooperative launch (default) vs one launch per kernel
    bool hoist;                         // of_set_hoist: IxIx, IxIy, IyIy planes and their sums formed once per level (default off)
    float *G;                           // three planes for the level's window sums a, b, c (allocated by of_set_hoist)
    CUtensorMap tmS2[OF_MAX_LEVELS];    // planes 3, 4 (IxIt, IyIt) of a level as an (x, y, field) tensor with a two-field box
    bool use_graph;
    std::vector<GraphEntry> graphs;
    unsigned long long stamp;
    int last_launches;
    std::string launch_err;            // first failing launch of the last enqueue ("" if none)
    std::vector<void *> allocs;
    MaskDesc md[OF_MAX_LEVELS];         // obstacle mask + compacted work lists per level (of_set_mask); all zero = none
    int *d_zero;                        // level-0 K3 tasks without a fluid pixel
    int zero_n;
    std::vector<void *> mask_allocs;
    Pipeline pipe;
    cudaEvent_t last_done;             // recorded after every submit (one solve in flight per handle)
    cudaStream_t last_stream;
    bool have_last;
    float *bench_out;                  // of_run_solve: a dense u, v pair of its own for the discarded result
};

namespace {

inline int round_up(int a, int b) { return (a + b - 1) / b * b; }
inline unsigned long long k2s_magic(int nuy) { return ((1ull << 40) + (unsigned long long)nuy - 1) / (unsigned long long)nuy; }

template <int R, bool BX> int setup_attrs()
{
#if SOLVE_K2S
    CU_TRY(cudaFuncSetAttribute(k2s_products_hsum<R, BX>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_MAX));
#else
    CU_TRY(cudaFuncSetAttribute(k2_products_hsum<R, false, BX>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_MAX));
#endif
    CU_TRY(cudaFuncSetAttribute(k3_vsum_solve<R, false, BX>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_MAX));
    CU_TRY(cudaFuncSetAttribute(of_solve_pair<R, false, false, BX>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_MAX));
    return OF_OK;
}

// K2: warp tiles of (8*nseg) x (2*nrp) outputs; every CTA owns an equal range of tiles and its
// SOLVE_WARPS warps pull from it.  The model only ranks candidates by the serial latency of a CTA's pass
// (coarse levels: one-round tiles with field-parallel sums; fine levels: fewer, wider tiles).
template <int R> K2Plan plan_k2(int W, int H, int sms, double active = 1.0)   // active = share of the tiles a mask leaves
{
    typedef K2Geom<R> G;
    K2Plan best = {};
    double best_cost = 1e30;
    int f_nseg = 0, f_nrp = 0;                     // (-DOF_PROFILE builds: tile shape forced through the environment, for sweeps)
#ifdef OF_PROFILE
    if (const char *e = getenv("OF_K2_GEOM")) sscanf(e, "%d,%d", &f_nseg, &f_nrp);
#endif
    const int segs = (W + 7) / 8;
    for (int nrp = 1; nrp <= 4; nrp *= 2) {
        const int nsegmax = 32 / nrp, tx_min = (segs + nsegmax - 1) / nsegmax;
        int last_nseg = 0;
        for (int tx = tx_min; tx <= segs; ++tx) {
            int nseg = (segs + tx - 1) / tx;
            if (f_nseg) { if (nrp != f_nrp) break; nseg = std::min(f_nseg, nsegmax); }
            if (nseg == last_nseg) continue;
            last_nseg = nseg;
            const int txr = (segs + nseg - 1) / nseg;
            const int tasks = G::pw(nseg) / 2 * nrp, rounds = (tasks + 31) / 32;
            const int ty = (H + 2 * nrp - 1) / (2 * nrp), ntiles = txr * ty;
            const int wb = G::warp_bytes(nseg, nrp);
            if (SOLVE_WARPS * wb > K3_RING * K3_CHUNK_BYTES) { if (f_nseg) break; continue; }   // must fit under the K3 barriers
            const int nf_par = std::max(1, std::min(5, 32 / (nseg * nrp)));
            const int hs = (5 + nf_par - 1) / nf_par;                      // serial field sums per lane
            // Serial latency of a CTA's pass, in SM cycles, fitted to the in-kernel timeline (profiles/
            // r2_notes.md, section 3): a tile costs 1850 + 1300 per product round + (550 + 400 x warps sharing a
            // sub-partition's FMA pipe) per serial field sum; a CTA runs its tiles in waves of SOLVE_WARPS.
            const int tiles_cta = ((int)std::ceil(ntiles * active) + sms - 1) / sms;
            double cost = 0.0;
            for (int left = tiles_cta; left > 0; left -= SOLVE_WARPS) {
                const int conc = std::min(left, SOLVE_WARPS);
                cost += 1850.0 + rounds * 1300.0 + hs * (550.0 + 400.0 * ((conc + 3) / 4));
            }
            if (cost < best_cost) {
                best_cost = cost;
                best = {nseg, nrp, ty, ntiles, sms, SOLVE_WARPS, SOLVE_WARPS * wb};
            }
            if (f_nseg) break;
        }
    }
    return best;
}

// K3: tasks of 64 columns x K3_SEG rows, equal contiguous share per CTA, one CTA per SM.
template <int R> K3Plan plan_k3(int W, int H, int sms)
{
    K3Plan p = {};
    p.nrb = (H + K3_SEG - 1) / K3_SEG;
    p.ntasks = ((W + 63) / 64) * p.nrb;
    p.grid = sms;
    p.warps = SOLVE_WARPS - 1;                                  // consumer warps; one producer warp is added at launch
    p.smem = K3Geom<R>::SMEM;
    return p;
}

// Fused coarse-level iteration (of_fused.cuh): one tile per CTA, tile + window halo in shared memory.  Chosen when the level can be
// cut into at most `sms` tiles that fit; among those the tiling with the fewest product pixels (tile + halo) per CTA.
template <int R> void plan_fused(of_context *c, int l)
{
    typedef FusedGeom<R> G;
    const int W = c->lv[l].W, H = c->lv[l].H;
    long best = -1;
    c->f_tw[l] = c->f_th[l] = c->f_tiles_x[l] = c->f_ntiles[l] = 0;
    for (int tw = 8; tw <= 256; tw += 8)
        for (int th = K3_SEG; th <= 256; th += K3_SEG) {
            const int tx = (W + tw - 1) / tw, ty = (H + th - 1) / th;
            if (tx * ty > c->sms || G::smem_bytes(tw, th) > K3_RING * K3_CHUNK_BYTES) continue;
            const long cost = (long)G::pw(tw) * G::ph(th) * 3 + (long)tw * G::ph(th) * 2 + (long)tw * th * 5;   // products, hsum, vsum + solve
            if (best < 0 || cost < best) { best = cost; c->f_tw[l] = tw; c->f_th[l] = th; c->f_tiles_x[l] = tx; c->f_ntiles[l] = tx * ty; }
        }
}

template <int R> void plan_level(of_context *c, int l)
{
    plan_fused<R>(c, l);
    c->k2[l] = plan_k2<R>(c->lv[l].W, c->lv[l].H, c->sms);
    c->k3[l] = plan_k3<R>(c->lv[l].W, c->lv[l].H, c->sms);
    c->k2s_nuy[l] = (c->lv[l].H + K2S<R>::RU - 1) / K2S<R>::RU;
    c->k2s_nunits[l] = ((c->lv[l].W + K2S<R>::TW - 1) / K2S<R>::TW) * c->k2s_nuy[l];
}

template <int R, bool BX>
void launch_k2(const of_context *c, int l, const float *I1, const float *I2, bool zero_uv, cudaStream_t st)
{
    const Level &L = c->lv[l];
    const K2Plan &P = c->k2[l];
    const MaskDesc &M = c->md[l];
    K2Params p = {I1, I2, c->u[l], c->v[l], c->S, c->plane, L.W, L.H, L.pitch, P.nseg, P.nrp, P.tiles_y, M.k2_list ? M.k2_n : P.ntiles,
                  c->ww, zero_uv ? 1 : 0, c->dbg, M.mask, M.k2_list, 0};
    if (M.mask) { of_launch_k2_masked(R, p, P.grid, 32 * P.warps, P.smem + 16, st); return; }    // compiled in optflow_mask.cu
#if !SOLVE_K2S
    k2_products_hsum<R, false, BX><<<P.grid, 32 * P.warps, P.smem + 16, st>>>(p);
#else
    const int s2 = I2 == c->pyr[1][l] ? 1 : 0;
    K2SParams q = {c->d_k2maps + l, s2, I1, I2, c->u[l], c->v[l], c->S, c->plane, L.W, L.H, L.pitch, c->k2s_nuy[l], c->k2s_nunits[l], k2s_magic(c->k2s_nuy[l]), c->ww, zero_uv ? 1 : 0, 0};
    k2s_products_hsum<R, BX><<<c->sms, 32 * (K2S_WORKERS + 1), K2S<R>::DATA_MAX + K2S<R>::BAR_BYTES, st>>>(q);
#endif
}

template <int R, bool BX>
void launch_k3(const of_context *c, int l, float *u_out, float *v_out, int out_pitch, bool last, bool zero_uv, cudaStream_t st, uint8_t *valid_out = nullptr)
{
    const Level &L = c->lv[l];
    const K3Plan &P = c->k3[l];
    K3Params p = {c->u[l], c->v[l], u_out, v_out, last ? (valid_out ? valid_out : c->valid) : nullptr, last ? c->det : nullptr,
                  L.W, L.H, L.pitch, out_pitch, P.nrb, P.ntasks, c->ww, {0.5f * c->eps_rel, c->max_step}, zero_uv ? 1 : 0, c->dbg, c->md[l], nullptr, 0};
    if (c->md[l].mask) of_launch_k3_masked(R, c->tmS[l], p, P.grid, 32 * (P.warps + 1), P.smem, st);
    else k3_vsum_solve<R, false, BX><<<P.grid, 32 * (P.warps + 1), P.smem, st>>>(c->tmS[l], p);
}

// Arguments of the persistent solve kernel for one pair of handle c (of_solve_pair, of_solve_dual).
void fill_solve_args(const of_context *c, int s1, int s2, float *u_out, float *v_out, uint8_t *valid_out, SolveArgs &a)
{
    static_assert(SOLVE_MAX_LEVELS == OF_MAX_LEVELS, "level limits out of sync");
    memcpy(a.tm, c->tmS, sizeof(CUtensorMap) * c->levels);
    a.lv = c->d_lv; a.gbar = c->d_gbar; a.S = c->S; a.plane = c->plane; a.u_out = u_out; a.v_out = v_out;
    a.valid = valid_out ? valid_out : c->valid; a.det = c->det; a.levels = c->levels; a.iterations = c->iterations; a.s1 = s1; a.s2 = s2;
    a.md = c->d_md; a.G = c->G; a.k2maps = c->d_k2maps;
    if (c->hoist && c->G != nullptr) memcpy(a.tm2, c->tmS2, sizeof(CUtensorMap) * c->levels);
    a.out_pitch = c->W; a.dbg = c->dbg; a.prof = c->prof_on ? c->d_prof : nullptr; a.ww = c->ww;
    a.sp.eps_half = 0.5f * c->eps_rel; a.sp.max_step = c->max_step;
}

template <int R, bool BX>
cudaError_t launch_solve(const of_context *c, const float *const *, int s1, int s2, float *u_out, float *v_out, cudaStream_t st, uint8_t *valid_out = nullptr)
{
    SolveArgs a;
    fill_solve_args(c, s1, s2, u_out, v_out, valid_out, a);
    const bool ho = c->hoist && c->G != nullptr;
    void *args[] = {&a};
    if (ho) return of_launch_solve_hoisted(R, c->md[0].mask != nullptr, a, c->sms, st);     // compiled in optflow_hoist.cu
    if (c->md[0].mask) return of_launch_solve_masked(R, a, c->sms, st);                              // compiled in optflow_mask.cu
    return cudaLaunchCooperativeKernel((const void *)of_solve_pair<R, false, false, BX>, dim3(c->sms), dim3(32 * SOLVE_WARPS), args,
                                       (size_t)SolveSmem<R>::BYTES, st);
}

// Tensor maps of the staged K2 input (of_k2s.cuh): per level the two pyramid slots as I2, box = one group of window rows.
template <int R> int encode_k2s_maps(of_context *c, void *fn)
{
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    typedef K2S<R> G;
    std::vector<K2SMaps> maps(c->levels);
    for (int l = 0; l < c->levels; ++l) {
        const Level &L = c->lv[l];
        cuuint64_t dims[2] = {(cuuint64_t)L.pitch, (cuuint64_t)L.H};
        cuuint64_t strides[1] = {(cuuint64_t)L.pitch * sizeof(float)};
        cuuint32_t box[2] = {G::PWB, G::RU};
        cuuint32_t estr[2] = {1, 1};
        for (int s = 0; s < N_PYR; ++s) {
            CUresult r = ((encode_fn)fn)(&maps[l].i2[s], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, c->pyr[s][l], dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                         CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) return fail(OF_ERR_CUDA, "cuTensorMapEncodeTiled(I2 window, level %d) failed: CUresult %d", l, (int)r);
        }
    }
    CU_TRY(cudaMemcpy(c->d_k2maps, maps.data(), sizeof(K2SMaps) * c->levels, cudaMemcpyHostToDevice));
    return OF_OK;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link-time libcuda dependency:
// the library must load on a machine without a driver, cf. tests/test_abi_cpu.py).
int encode_tensor_maps(of_context *c)
{
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    CU_TRY(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
    if (!fn || qres != cudaDriverEntryPointSuccess) return fail(OF_ERR_CUDA, "cuTensorMapEncodeTiled is not available in this driver");
    {
        int rc = OF_OK;
        DISPATCH_R(c->R, rc = encode_k2s_maps<R>(c, fn));
        if (rc != OF_OK) return rc;
    }
    for (int l = 0; l < c->levels; ++l) {
        const Level &L = c->lv[l];
        cuuint64_t dims[3] = {(cuuint64_t)L.pitch, (cuuint64_t)L.H, 5};
        cuuint64_t strides[2] = {(cuuint64_t)L.pitch * sizeof(float), (cuuint64_t)c->plane * sizeof(float)};
        cuuint32_t box[3] = {64, K3_SEG, 5};
        cuuint32_t estr[3] = {1, 1, 1};
        CUresult r = ((encode_fn)fn)(&c->tmS[l], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, c->S, dims, strides, box, estr,
                                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(OF_ERR_CUDA, "cuTensorMapEncodeTiled(level %d) failed: CUresult %d", l, (int)r);
        cuuint32_t box2[3] = {64, K3_SEG, 2};                   // of_set_hoist: the two It planes fetched at field 3
        r = ((encode_fn)fn)(&c->tmS2[l], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, c->S, dims, strides, box2, estr,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return fail(OF_ERR_CUDA, "cuTensorMapEncodeTiled(level %d, two-field box) failed: CUresult %d", l, (int)r);
    }
    return OF_OK;
}


void run_k2(const of_context *c, int l, const float *I1, const float *I2, bool zero_uv, cudaStream_t st)
{
    DISPATCH_RB(c->R, c->ww.box, (launch_k2<R, BX>(c, l, I1, I2, zero_uv, st)));
}
void run_k3(const of_context *c, int l, float *u_out, float *v_out, int out_pitch, bool last, bool zero_uv, cudaStream_t st, uint8_t *valid_out = nullptr)
{
    DISPATCH_RB(c->R, c->ww.box, (launch_k3<R, BX>(c, l, u_out, v_out, out_pitch, last, zero_uv, st, valid_out)));
}

void run_convert(const of_context *c, int dtype, const void *a, const void *b, float *da, float *db, cudaStream_t st)
{
    const Level &L = c->lv[0];
    if (c->eq_radius > 0) {                                            // eq. 2 fused with the conversion
        const int r = c->eq_radius;
        dim3 grid((L.W + EQ_TW - 1) / EQ_TW, (L.H + EQ_TH - 1) / EQ_TH, b ? 2 : 1);
        if (dtype == OF_DTYPE_U8 && r == 5)                               // the paper's radius: unrolled instantiation
            k0_equalise<uint8_t, 5><<<grid, 256, eq_smem_bytes(r, 1), st>>>((const uint8_t *)a, (const uint8_t *)b, da, db, L.W, L.H, L.pitch, r);
        else if (dtype == OF_DTYPE_U16 && r == 5)
            k0_equalise<uint16_t, 5><<<grid, 256, eq_smem_bytes(r, 2), st>>>((const uint16_t *)a, (const uint16_t *)b, da, db, L.W, L.H, L.pitch, r);
        else if (dtype == OF_DTYPE_U8)
            k0_equalise<uint8_t><<<grid, 256, eq_smem_bytes(r, 1), st>>>((const uint8_t *)a, (const uint8_t *)b, da, db, L.W, L.H, L.pitch, r);
        else if (dtype == OF_DTYPE_U16)
            k0_equalise<uint16_t><<<grid, 256, eq_smem_bytes(r, 2), st>>>((const uint16_t *)a, (const uint16_t *)b, da, db, L.W, L.H, L.pitch, r);
        else
            k0_equalise<float><<<grid, 256, eq_smem_bytes(r, 4), st>>>((const float *)a, (const float *)b, da, db, L.W, L.H, L.pitch, r);
        return;
    }
    dim3 grid((L.W + 1023) / 1024, L.H, b ? 2 : 1);
    if (dtype == OF_DTYPE_U8)
        k0_convert<uint8_t><<<grid, 256, 0, st>>>((const uint8_t *)a, (const uint8_t *)b, da, db, L.W, L.H, L.pitch);
    else if (dtype == OF_DTYPE_U16)
        k0_convert<uint16_t><<<grid, 256, 0, st>>>((const uint16_t *)a, (const uint16_t *)b, da, db, L.W, L.H, L.pitch);
    else
        k0_convert<float><<<grid, 256, 0, st>>>((const float *)a, (const float *)b, da, db, L.W, L.H, L.pitch);
}

void run_pyramid(const of_context *c, int l, const float *sa, const float *sb, float *da, float *db, cudaStream_t st)
{
    const Level &S = c->lv[l], &D = c->lv[l + 1];
    dim3 grid((D.W + K1_TW - 1) / K1_TW, (D.H + K1_TH - 1) / K1_TH, sb ? 2 : 1);
    k1_pyramid_down<float><<<grid, 256, 0, st>>>(sa, sb, da, db, S.W, S.H, S.pitch, D.W, D.H, D.pitch, nullptr, nullptr, 0);
}

// First pyramid step fused with the frame conversion: raw frame -> fp32 level 0 AND level 1 in one kernel.
void run_convert_pyramid(const of_context *c, int dtype, const void *a, const void *b, float *a0, float *b0, float *a1, float *b1, cudaStream_t st)
{
    const Level &S = c->lv[0], &D = c->lv[1];
    dim3 grid((D.W + K1_TW - 1) / K1_TW, (D.H + K1_TH - 1) / K1_TH, b ? 2 : 1);
    if (dtype == OF_DTYPE_U8)
        k1_pyramid_down<uint8_t><<<grid, 256, 0, st>>>((const uint8_t *)a, (const uint8_t *)b, a1, b1, S.W, S.H, S.W, D.W, D.H, D.pitch, a0, b0, S.pitch);
    else if (dtype == OF_DTYPE_U16)
        k1_pyramid_down<uint16_t><<<grid, 256, 0, st>>>((const uint16_t *)a, (const uint16_t *)b, a1, b1, S.W, S.H, S.W, D.W, D.H, D.pitch, a0, b0, S.pitch);
    else
        k1_pyramid_down<float><<<grid, 256, 0, st>>>((const float *)a, (const float *)b, a1, b1, S.W, S.H, S.W, D.W, D.H, D.pitch, a0, b0, S.pitch);
}

void run_upsample(const of_context *c, int l, cudaStream_t st)   // level l+1 -> l
{
    const Level &F = c->lv[l], &Cc = c->lv[l + 1];
    dim3 grid((F.W + 63) / 64, (F.H + 3) / 4);
    k4_upsample_flow<<<grid, 256, 0, st>>>(c->u[l + 1], c->v[l + 1], Cc.W, Cc.H, Cc.pitch, c->u[l], c->v[l], F.W, F.H, F.pitch, c->md[l].mask);
}

void note_launch(of_context *c, const char *what, int level)
{
    cudaError_t e = cudaPeekAtLastError();
    if (e != cudaSuccess && c->launch_err.empty()) {
        char buf[160];
        snprintf(buf, sizeof buf, "%s (level %d): %s", what, level, cudaGetErrorString(e));
        c->launch_err = buf;
    }
}

// Frame conversion + pyramid of one Job (rows a1-a2).  Returns the number of kernels launched.
int enqueue_pyramids(of_context *c, const Job &j, cudaStream_t st)
{
    int n = 0;
    c->launch_err.clear();
    if (j.cvtA >= 0) {
        const bool both = j.cvtB >= 0;
        int l0 = 0;
        if (c->levels > 1 && c->eq_radius == 0) {               // conversion fused into the first pyramid step
            run_convert_pyramid(c, j.dtype, j.rawA, both ? j.rawB : nullptr, c->pyr[j.cvtA][0], both ? c->pyr[j.cvtB][0] : nullptr,
                                c->pyr[j.cvtA][1], both ? c->pyr[j.cvtB][1] : nullptr, st);
            note_launch(c, "convert+pyramid", 0);
            ++n;
            l0 = 1;
        } else {
            run_convert(c, j.dtype, j.rawA, both ? j.rawB : nullptr, c->pyr[j.cvtA][0], both ? c->pyr[j.cvtB][0] : nullptr, st);
            note_launch(c, "convert", 0);
            ++n;
        }
        for (int l = l0; l + 1 < c->levels; ++l) {
            run_pyramid(c, l, c->pyr[j.cvtA][l], both ? c->pyr[j.cvtB][l] : nullptr, c->pyr[j.cvtA][l + 1],
                        both ? c->pyr[j.cvtB][l + 1] : nullptr, st);
            note_launch(c, "pyramid", l);
            ++n;
        }
    }
    return n;
}

// Enqueue the whole path of one Job (rows a1-a10).  Returns the number of kernels launched.
int enqueue_job(of_context *c, const Job &j, cudaStream_t st)
{
    int n = enqueue_pyramids(c, j, st);
    const int top = c->levels - 1;     // (no memset of the coarsest field: its first iteration takes u = v = 0 without reading it)
    if (c->persistent) {
        cudaError_t e = cudaSuccess;
        DISPATCH_RB(c->R, c->ww.box, (e = launch_solve<R, BX>(c, nullptr, j.s1, j.s2, j.u_out, j.v_out, st, j.valid_out)));
        if (e != cudaSuccess && c->launch_err.empty()) c->launch_err = std::string("solve (persistent): ") + cudaGetErrorString(e);
        note_launch(c, "solve (persistent)", 0);
        return n + 1;
    }
    if (c->zero_n > 0) {               // mask set: outputs of the level-0 tasks no K3 pass visits (M3)
        k_mask_zero<<<c->sms, 256, 0, st>>>(c->d_zero, c->zero_n, c->k3[0].nrb, c->W, c->H, c->lv[0].pitch, j.u_out, j.v_out, c->W, j.valid_out ? j.valid_out : c->valid, c->det);
        note_launch(c, "mask zero-fill", 0);
        ++n;
    }
    for (int l = top; l >= 0; --l) {
        if (l < top) { run_upsample(c, l, st); note_launch(c, "upsample", l); ++n; }
        for (int it = 0; it < c->iterations; ++it) {
            const bool zero_uv = (l == top && it == 0);
            run_k2(c, l, c->pyr[j.s1][l], c->pyr[j.s2][l], zero_uv, st);
            note_launch(c, "products+hsum", l);
            const bool last = (l == 0 && it == c->iterations - 1);
            if (last) run_k3(c, l, j.u_out, j.v_out, c->W, true, zero_uv, st, j.valid_out);
            else run_k3(c, l, c->u[l], c->v[l], c->lv[l].pitch, false, zero_uv, st);
            note_launch(c, "vsum+solve", l);
            n += 2;
        }
    }
    return n;
}

int submit_job_inner(of_context *c, const Job &j, cudaStream_t st);

// All scratch (pyramids, fields, planes, the grid-barrier word) belongs to the handle, so only one solve of a handle may be in flight:
// a submit on another stream than the previous one is ordered after it with an event.
int submit_job(of_context *c, const Job &j, cudaStream_t st)
{
    CU_TRY(cudaSetDevice(c->device));
    if (c->have_last && st != c->last_stream) CU_TRY(cudaStreamWaitEvent(st, c->last_done, 0));
    int rc = submit_job_inner(c, j, st);
    if (rc == OF_OK) {
        CU_TRY(cudaEventRecord(c->last_done, st));
        c->last_stream = st;
        c->have_last = true;
    }
    return rc;
}

int submit_job_inner(of_context *c, const Job &j, cudaStream_t st)
{
    if (!c->use_graph || st == nullptr) {
        c->last_launches = enqueue_job(c, j, st);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return fail(OF_ERR_CUDA, "launch failed: %s; first failing launch: %s", cudaGetErrorString(e), c->launch_err.c_str());
        return OF_OK;
    }
    ++c->stamp;
    for (auto &g : c->graphs)
        if (g.job == j) {
            g.stamp = c->stamp;
            CU_TRY(cudaGraphLaunch(g.exec, st));
            c->last_launches = g.launches;
            return OF_OK;
        }
    cudaGraph_t graph = nullptr;
    CU_TRY(cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
    int n = enqueue_job(c, j, st);
    cudaError_t e1 = cudaGetLastError();
    cudaError_t e2 = cudaStreamEndCapture(st, &graph);
    if (e1 != cudaSuccess || e2 != cudaSuccess || graph == nullptr) {
        if (graph) cudaGraphDestroy(graph);
        return fail(OF_ERR_CUDA, "graph capture failed: %s / %s; first failing launch: %s", cudaGetErrorString(e1), cudaGetErrorString(e2),
                    c->launch_err.c_str());
    }
    if (c->graphs.size() >= 64) {
        // cache full (a caller that rotates more than 64 pointer sets): re-use the least recently used executable graph by
        // patching the kernel parameters of its nodes in place (cudaGraphExecUpdate: same topology, no instantiation)
        size_t old = 0;
        for (size_t i = 1; i < c->graphs.size(); ++i)
            if (c->graphs[i].stamp < c->graphs[old].stamp) old = i;
        cudaGraphExecUpdateResultInfo info;
        if (cudaGraphExecUpdate(c->graphs[old].exec, graph, &info) == cudaSuccess) {
            cudaGraphDestroy(graph);
            c->graphs[old].job = j; c->graphs[old].stamp = c->stamp; c->graphs[old].launches = n;
            CU_TRY(cudaGraphLaunch(c->graphs[old].exec, st));
            c->last_launches = n;
            return OF_OK;
        }
        (void)cudaGetLastError();
        cudaGraphExecDestroy(c->graphs[old].exec);
        c->graphs.erase(c->graphs.begin() + old);
    }
    cudaGraphExec_t exec = nullptr;
    cudaError_t e3 = cudaGraphInstantiate(&exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e3 != cudaSuccess) return fail(OF_ERR_CUDA, "cudaGraphInstantiate failed: %s", cudaGetErrorString(e3));
    c->graphs.push_back({j, exec, c->stamp, n});
    CU_TRY(cudaGraphLaunch(exec, st));
    c->last_launches = n;
    return OF_OK;
}

// Host-side construction of the mask pyramid (M4) and of the compacted work lists of one handle.
//   K3 task (strip s, row block rb) is active iff its 64 x K3_SEG pixels hold a fluid pixel;
//   K2 tile is active iff an active K3 task reads one of its plane rows (task rows -R .. K3_SEG-1+R);
//   the active K3 tasks are cut into equal shares per CTA, each share into runs of consecutive tasks of
//   one strip (a run shares ring chunks between neighbours exactly like the unmasked strip walk).
int build_mask(of_context *c, const uint8_t *mask, int row_stride)
{
    for (void *p : c->mask_allocs) cudaFree(p);
    c->mask_allocs.clear();
    memset(c->md, 0, sizeof c->md);
    c->d_zero = nullptr;
    c->zero_n = 0;
    if (!mask) {
        for (int l = 0; l < c->levels; ++l) { DISPATCH_R(c->R, c->k2[l] = plan_k2<R>(c->lv[l].W, c->lv[l].H, c->sms)); }
        return OF_OK;
    }
    auto upload = [&](const void *src, size_t bytes, void **dst) -> int {
        cudaError_t e = cudaMalloc(dst, std::max<size_t>(bytes, 16));
        if (e != cudaSuccess) return fail(OF_ERR_ALLOC, "cudaMalloc(%zu) failed: %s", bytes, cudaGetErrorString(e));
        c->mask_allocs.push_back(*dst);
        if (bytes) CU_TRY(cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice));
        return OF_OK;
    };
    const int R = c->R, NC = (K3_SEG + 2 * R + K3_SEG - 1) / K3_SEG, ncta = c->sms;
    std::vector<uint8_t> cur, nxt;
    for (int l = 0; l < c->levels; ++l) {
        const Level &L = c->lv[l];
        nxt.assign((size_t)L.pitch * L.H, 0);
        if (l == 0) {
            for (int y = 0; y < L.H; ++y)
                for (int x = 0; x < L.W; ++x) nxt[(size_t)y * L.pitch + x] = mask[(size_t)y * row_stride + x] ? 1 : 0;
        } else {
            const Level &F = c->lv[l - 1];
            for (int Y = 0; Y < L.H; ++Y)
                for (int X = 0; X < L.W; ++X) {
                    int any = 0;
                    for (int dy = 0; dy < 2; ++dy)
                        for (int dx = 0; dx < 2; ++dx) {
                            const int x = 2 * X + dx, y = 2 * Y + dy;
                            if (x < F.W && y < F.H && cur[(size_t)y * F.pitch + x]) any = 1;
                        }
                    nxt[(size_t)Y * L.pitch + X] = (uint8_t)any;
                }
        }
        cur.swap(nxt);
        MaskDesc &M = c->md[l];
        int rc = upload(cur.data(), cur.size(), (void **)&M.mask);
        if (rc != OF_OK) return rc;
        // ---- K3 tasks
        const K3Plan &P3 = c->k3[l];
        const int nrb = P3.nrb, nstrips = P3.ntasks / nrb;
        std::vector<int> act, idle;
        std::vector<uint8_t> need((size_t)nstrips * L.H, 0);
        for (int s = 0; s < nstrips; ++s)
            for (int rb = 0; rb < nrb; ++rb) {
                bool any = false;
                for (int y = K3_SEG * rb; y < std::min(K3_SEG * rb + K3_SEG, L.H) && !any; ++y)
                    for (int x = 64 * s; x < std::min(64 * s + 64, L.W); ++x)
                        if (cur[(size_t)y * L.pitch + x]) { any = true; break; }
                if (!any) { idle.push_back(s * nrb + rb); continue; }
                act.push_back(s * nrb + rb);
                for (int y = std::max(0, K3_SEG * rb - R); y <= std::min(L.H - 1, K3_SEG * rb + K3_SEG - 1 + R); ++y) need[(size_t)s * L.H + y] = 1;
            }
        std::vector<int2> ent(act.size());
        std::vector<K3Run> runs;
        std::vector<K3Cta> ctas(ncta);
        for (int cta = 0; cta < ncta; ++cta) {
            int b, e;
            cta_range((int)act.size(), cta, ncta, b, e);
            K3Cta cd = {b, e, (int)runs.size(), 0, 0, 0, 0, 0};
            int chunks = 0;
            for (int i = b; i < e;) {
                int n = 1;
                while (i + n < e && act[i + n] == act[i] + n && act[i + n] / nrb == act[i] / nrb) ++n;
                runs.push_back({act[i], n, chunks, 0});
                for (int k = 0; k < n; ++k) ent[i + k] = make_int2(act[i + k], chunks + k);
                chunks += n + NC - 1;
                i += n;
            }
            cd.run_e = (int)runs.size();
            cd.nchunks = chunks;
            ctas[cta] = cd;
        }
        M.k3_n = (int)act.size();
        if ((rc = upload(ent.data(), ent.size() * sizeof(int2), (void **)&M.k3_ent)) != OF_OK) return rc;
        if ((rc = upload(runs.data(), runs.size() * sizeof(K3Run), (void **)&M.k3_runs)) != OF_OK) return rc;
        if ((rc = upload(ctas.data(), ctas.size() * sizeof(K3Cta), (void **)&M.k3_cta)) != OF_OK) return rc;
        if (l == 0) {
            c->zero_n = (int)idle.size();
            if ((rc = upload(idle.data(), idle.size() * sizeof(int), (void **)&c->d_zero)) != OF_OK) return rc;
            M.zero_list = c->d_zero;
            M.zero_n = c->zero_n;
        }
        // ---- K2 tiles (geometry re-planned for the share of the level that is left)
        {
            size_t cnt = 0;
            for (uint8_t b : need) cnt += b;
            const double share = std::max(0.02, (double)cnt / (double)std::max<size_t>(need.size(), 1));
            DISPATCH_R(c->R, c->k2[l] = plan_k2<R>(L.W, L.H, c->sms, share));
        }
        const K2Plan &P2 = c->k2[l];
        const int TW = 8 * P2.nseg, TH = 2 * P2.nrp, tiles_x = P2.ntiles / P2.tiles_y;
        std::vector<int> tiles;
        for (int tx = 0; tx < tiles_x; ++tx)
            for (int ty = 0; ty < P2.tiles_y; ++ty) {
                bool any = false;
                const int s0 = (tx * TW) / 64, s1 = std::min(nstrips - 1, (tx * TW + TW - 1) / 64);
                for (int sidx = s0; sidx <= s1 && !any; ++sidx)
                    for (int y = ty * TH; y < std::min(ty * TH + TH, L.H); ++y)
                        if (need[(size_t)sidx * L.H + y]) { any = true; break; }
                if (any) tiles.push_back(tx * P2.tiles_y + ty);
            }
        M.k2_n = (int)tiles.size();
        if ((rc = upload(tiles.data(), tiles.size() * sizeof(int), (void **)&M.k2_list)) != OF_OK) return rc;
#ifdef OF_PROFILE
        if (getenv("OF_DEBUG"))
            fprintf(stderr, "[optflow] mask level %d: K2 tiles %d of %d, K3 tasks %d of %d (%zu runs)\n", l, M.k2_n, P2.ntiles, M.k3_n, P3.ntasks, runs.size());
#endif
    }
    return OF_OK;
}

int upload_level_descs(of_context *c)
{
    LevelDesc hl[OF_MAX_LEVELS];
    for (int l = 0; l < c->levels; ++l)
        hl[l] = {{c->pyr[0][l], c->pyr[1][l]}, c->u[l], c->v[l], c->lv[l].W, c->lv[l].H, c->lv[l].pitch,
                 c->k2[l].nseg, c->k2[l].nrp, c->k2[l].tiles_y, c->k2[l].ntiles, c->k3[l].nrb, c->k3[l].ntasks,
                 c->k2s_nuy[l], c->k2s_nunits[l], k2s_magic(c->k2s_nuy[l]), c->u2[l], c->v2[l],
                 c->f_tw[l], c->f_th[l], c->f_tiles_x[l], c->fuse_coarse ? c->f_ntiles[l] : 0};
    CU_TRY(cudaMemcpy(c->d_lv, hl, sizeof(LevelDesc) * c->levels, cudaMemcpyHostToDevice));
    CU_TRY(cudaMemcpy(c->d_md, c->md, sizeof(MaskDesc) * c->levels, cudaMemcpyHostToDevice));
    return OF_OK;
}

void drop_graphs(of_context *c)
{
    for (auto &g : c->graphs) cudaGraphExecDestroy(g.exec);
    c->graphs.clear();
}

int dev_alloc(of_context *c, void **p, size_t bytes)
{
    cudaError_t e = cudaMalloc(p, bytes);
    if (e != cudaSuccess) return fail(OF_ERR_ALLOC, "cudaMalloc(%zu) failed: %s", bytes, cudaGetErrorString(e));
    c->allocs.push_back(*p);
    return OF_OK;
}

// Argument checks of one pair and its Job.
int make_pair_job(of_handle h, int dtype, const void *I1, const void *I2, float *u, float *v, Job &j)
{
    if (!h) return fail(OF_ERR_INVALID_ARG, "null handle");
    if (!I1 || !I2 || !u || !v) return fail(OF_ERR_INVALID_ARG, "null image or field pointer");
    if (h->pipe.open) return fail(OF_ERR_STATE, "handle is in streaming mode; call of_stream_close first");
    if ((reinterpret_cast<uintptr_t>(u) | reinterpret_cast<uintptr_t>(v)) & 15)
        return fail(OF_ERR_INVALID_ARG, "u and v must be 16-byte aligned (the last pass stores float2 / float4)");
    if (dtype != OF_DTYPE_F32 && dtype != OF_DTYPE_U8 && dtype != OF_DTYPE_U16) return fail(OF_ERR_INVALID_ARG, "unknown dtype %d", dtype);
    const size_t es = dtype == OF_DTYPE_U8 ? 1 : (dtype == OF_DTYPE_U16 ? 2 : 4);
    if ((reinterpret_cast<uintptr_t>(I1) | reinterpret_cast<uintptr_t>(I2)) & (es - 1))
        return fail(OF_ERR_INVALID_ARG, "I1 and I2 must be aligned to their element size");
    memset(&j, 0, sizeof j);
    j.dtype = dtype; j.rawA = I1; j.rawB = I2; j.cvtA = 0; j.cvtB = 1; j.s1 = 0; j.s2 = 1; j.u_out = u; j.v_out = v;
    return OF_OK;
}

int compute_any(of_handle h, int dtype, const void *I1, const void *I2, float *u, float *v, void *stream)
{
    Job j;
    int rc = make_pair_job(h, dtype, I1, I2, u, v, j);
    if (rc != OF_OK) return rc;
    return submit_job(h, j, (cudaStream_t)stream);
}

// Two handles can share one of_solve_dual launch iff they describe the same problem and neither needs a variant kernel.
bool dual_eligible(const of_context *a, const of_context *b)
{
    return a != b && a->device == b->device && a->W == b->W && a->H == b->H && a->levels == b->levels && a->R == b->R &&
           a->iterations == b->iterations && a->window_type == b->window_type && a->persistent && b->persistent &&
           a->fuse_coarse == b->fuse_coarse && a->eps_rel == b->eps_rel && a->max_step == b->max_step && !a->md[0].mask && !b->md[0].mask && !(a->hoist && a->G) && !(b->hoist && b->G) &&
           a->dbg == 0 && b->dbg == 0;
}

// Both pairs: conversion + pyramids of each, then ONE solve launch for the two (of_solve_dual.cuh).  Both handles are busy until it ends.
int submit_dual(of_context *a, const Job &ja, of_context *b, const Job &jb, cudaStream_t st)
{
    CU_TRY(cudaSetDevice(a->device));
    if (a->have_last && st != a->last_stream) CU_TRY(cudaStreamWaitEvent(st, a->last_done, 0));
    if (b->have_last && st != b->last_stream) CU_TRY(cudaStreamWaitEvent(st, b->last_done, 0));
    int n = enqueue_pyramids(a, ja, st);
    n += enqueue_pyramids(b, jb, st);
    SolveArgs sa, sb;
    fill_solve_args(a, ja.s1, ja.s2, ja.u_out, ja.v_out, ja.valid_out, sa);
    fill_solve_args(b, jb.s1, jb.s2, jb.u_out, jb.v_out, jb.valid_out, sb);
    sb.prof = nullptr;                                     // the timeline of a two-pair launch is kept by the first handle
    cudaError_t e = of_launch_solve_dual(a->R, sa, sb, a->sms, st);
    if (e != cudaSuccess) return fail(OF_ERR_CUDA, "solve (two pairs) launch failed: %s; first failing launch before it: %s", cudaGetErrorString(e),
                                      (a->launch_err + b->launch_err).c_str());
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(OF_ERR_CUDA, "launch failed: %s; first failing launch: %s", cudaGetErrorString(e), (a->launch_err + b->launch_err).c_str());
    a->last_launches = b->last_launches = n + 1;
    CU_TRY(cudaEventRecord(a->last_done, st));
    CU_TRY(cudaEventRecord(b->last_done, st));
    a->last_stream = b->last_stream = st;
    a->have_last = b->have_last = true;
    return OF_OK;
}

int copy_plane_dense(const float *src, int pitch, int W, int H, float *dst, cudaStream_t st)
{
    CU_TRY(cudaMemcpy2DAsync(dst, sizeof(float) * W, src, sizeof(float) * pitch, sizeof(float) * W, H,
                             cudaMemcpyDeviceToDevice, st));
    return OF_OK;
}

void pipe_release(of_context *c)
{
    Pipeline &p = c->pipe;
    if (p.s_copy) cudaStreamSynchronize(p.s_copy);
    if (p.s_comp) cudaStreamSynchronize(p.s_comp);
    if (p.s_down) cudaStreamSynchronize(p.s_down);
    for (int i = 0; i < N_PIN; ++i) {
        if (p.pin[i]) cudaFreeHost(p.pin[i]);
        if (p.raw[i]) cudaFree(p.raw[i]);
        if (p.h2d_done[i]) cudaEventDestroy(p.h2d_done[i]);
        if (p.cvt_done[i]) cudaEventDestroy(p.cvt_done[i]);
    }
    for (int i = 0; i < N_RES; ++i) {
        if (p.res_dev[i]) cudaFree(p.res_dev[i]);
        if (p.res_host[i]) cudaFreeHost(p.res_host[i]);
        if (p.solve_done[i]) cudaEventDestroy(p.solve_done[i]);
        if (p.d2h_done[i]) cudaEventDestroy(p.d2h_done[i]);
    }
    if (p.s_copy) cudaStreamDestroy(p.s_copy);
    if (p.s_comp) cudaStreamDestroy(p.s_comp);
    if (p.s_down) cudaStreamDestroy(p.s_down);
    p = Pipeline();
}

}  // namespace

// error reporting for the other translation units (optflow_static.cu): sets the string of_last_error returns
int of_detail_fail(int code, const char *msg) { return fail(code, "%s", msg); }

// =================================================================================================
// C ABI
// =================================================================================================
extern "C" {

const char *of_last_error(void) { return g_err.c_str(); }

of_handle of_create(int width, int height, int levels, int window_radius, int iterations, int window_type)
{
    g_err.clear();
    if (width < 1 || height < 1 || width > (1 << 15) || height > (1 << 15)) { fail(OF_ERR_INVALID_ARG, "bad image size %dx%d", width, height); return nullptr; }
    if (levels < 1 || levels > OF_MAX_LEVELS) { fail(OF_ERR_INVALID_ARG, "levels must be in [1,%d]", OF_MAX_LEVELS); return nullptr; }
    if (window_radius < 1 || window_radius > OF_MAX_WINDOW_RADIUS) { fail(OF_ERR_INVALID_ARG, "window_radius must be in [1,%d]", OF_MAX_WINDOW_RADIUS); return nullptr; }
    if (iterations < 1) { fail(OF_ERR_INVALID_ARG, "iterations must be >= 1"); return nullptr; }
    if (window_type != OF_WINDOW_BOX && window_type != OF_WINDOW_GAUSSIAN) { fail(OF_ERR_INVALID_ARG, "unknown window_type %d", window_type); return nullptr; }
    Level lv[OF_MAX_LEVELS];
    lv[0] = {width, height, round_up(width, 32)};
    for (int l = 1; l < levels; ++l) {
        lv[l].W = (lv[l - 1].W + 1) / 2;
        lv[l].H = (lv[l - 1].H + 1) / 2;
        lv[l].pitch = round_up(lv[l].W, 32);
    }
    if (lv[levels - 1].W < 2 * window_radius + 1 || lv[levels - 1].H < 2 * window_radius + 1) {
        fail(OF_ERR_INVALID_ARG, "coarsest level %dx%d is smaller than the window (%d)", lv[levels - 1].W, lv[levels - 1].H, 2 * window_radius + 1);
        return nullptr;
    }
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { fail(OF_ERR_CUDA, "no usable CUDA device: %s", cudaGetErrorString(e)); return nullptr; }
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) { fail(OF_ERR_CUDA, "cudaGetDeviceProperties: %s", cudaGetErrorString(e)); return nullptr; }
    if (prop.major != 10) { fail(OF_ERR_CUDA, "device %s is sm_%d%d; this library is built for sm_100a only", prop.name, prop.major, prop.minor); return nullptr; }

    of_context *c = new (std::nothrow) of_context();
    if (!c) { fail(OF_ERR_ALLOC, "out of host memory"); return nullptr; }
    c->W = width; c->H = height; c->levels = levels; c->R = window_radius; c->iterations = iterations;
    c->window_type = window_type; c->device = dev; c->eps_rel = 1e-3f; c->max_step = 3.0f;
    c->use_graph = true; c->stamp = 0; c->last_launches = 0; c->fuse_coarse = true;
    c->last_done = nullptr; c->last_stream = nullptr; c->have_last = false; c->bench_out = nullptr;
    memcpy(c->lv, lv, sizeof lv);
    memset(&c->ww, 0, sizeof c->ww);
    c->ww.box = window_type == OF_WINDOW_BOX ? 1 : 0;
    for (int t = -window_radius; t <= window_radius; ++t) {
        double w = 1.0;
        if (window_type == OF_WINDOW_GAUSSIAN) {
            double sigma = (double)window_radius / 3.0;
            w = std::exp(-(double)(t * t) / (2.0 * sigma * sigma));
        }
        c->ww.w[t + window_radius] = (float)w;
    }
    int rc = OF_OK;
    for (int l = 0; l < levels && rc == OF_OK; ++l) {
        size_t bytes = sizeof(float) * (size_t)lv[l].pitch * lv[l].H;
        for (int s = 0; s < N_PYR && rc == OF_OK; ++s) rc = dev_alloc(c, (void **)&c->pyr[s][l], bytes);
        if (rc == OF_OK) rc = dev_alloc(c, (void **)&c->u[l], 4 * bytes);      // u, v, u2, v2
        if (rc == OF_OK) {
            c->v[l] = c->u[l] + (size_t)lv[l].pitch * lv[l].H;
            c->u2[l] = c->v[l] + (size_t)lv[l].pitch * lv[l].H;
            c->v2[l] = c->u2[l] + (size_t)lv[l].pitch * lv[l].H;
        }
    }
    c->plane = (size_t)lv[0].pitch * lv[0].H;
    if (rc == OF_OK) rc = dev_alloc(c, (void **)&c->S, sizeof(float) * 5 * c->plane);
    if (rc == OF_OK) rc = dev_alloc(c, (void **)&c->det, sizeof(float) * c->plane);
    if (rc == OF_OK) rc = dev_alloc(c, (void **)&c->valid, (size_t)width * height);
    if (rc == OF_OK) {
        // padding columns of every plane must hold finite values (they are read, never used)
        for (void *p : c->allocs) (void)p;
        for (int l = 0; l < levels; ++l) {
            size_t bytes = sizeof(float) * (size_t)lv[l].pitch * lv[l].H;
            for (int s = 0; s < N_PYR; ++s) cudaMemset(c->pyr[s][l], 0, bytes);
            cudaMemset(c->u[l], 0, 4 * bytes);
        }
        cudaMemset(c->S, 0, sizeof(float) * 5 * c->plane);
        cudaMemset(c->det, 0, sizeof(float) * c->plane);
        cudaMemset(c->valid, 0, (size_t)width * height);
        if (cudaDeviceSynchronize() != cudaSuccess) rc = fail(OF_ERR_CUDA, "memset failed: %s", cudaGetErrorString(cudaGetLastError()));
    }
    if (rc == OF_OK && cudaEventCreateWithFlags(&c->last_done, cudaEventDisableTiming) != cudaSuccess)
        rc = fail(OF_ERR_CUDA, "cudaEventCreate failed: %s", cudaGetErrorString(cudaGetLastError()));
    if (rc == OF_OK) { DISPATCH_RB(window_radius, c->ww.box, (rc = setup_attrs<R, BX>())); }
    if (rc == OF_OK) {
        cudaError_t e = of_setup_attrs_hoisted(window_radius, SMEM_MAX);
        if (e == cudaSuccess) e = of_setup_attrs_masked(window_radius, SMEM_MAX);
        if (e == cudaSuccess) e = of_setup_attrs_dual(window_radius, SMEM_MAX);
        if (e != cudaSuccess) rc = fail(OF_ERR_CUDA, "cudaFuncSetAttribute (hoisted / masked / two-pair kernels): %s", cudaGetErrorString(e));
    }
    if (rc == OF_OK) {
        c->sms = prop.multiProcessorCount;
        c->dbg = 0;
#ifdef OF_PROFILE
        c->dbg = getenv("OF_KERNEL_DEBUG") ? atoi(getenv("OF_KERNEL_DEBUG")) : 0;
#endif
        for (int l = 0; l < levels; ++l) { DISPATCH_R(window_radius, plan_level<R>(c, l)); }
        rc = dev_alloc(c, (void **)&c->d_k2maps, sizeof(K2SMaps) * levels);
        if (rc == OF_OK) rc = encode_tensor_maps(c);
        if (rc == OF_OK) rc = dev_alloc(c, (void **)&c->d_lv, sizeof(LevelDesc) * levels);
        if (rc == OF_OK) rc = dev_alloc(c, (void **)&c->d_md, sizeof(MaskDesc) * OF_MAX_LEVELS);
        if (rc == OF_OK) rc = dev_alloc(c, (void **)&c->d_tm, sizeof(CUtensorMap) * levels);
        if (rc == OF_OK) rc = dev_alloc(c, (void **)&c->d_gbar, 256);
        if (rc == OF_OK) rc = dev_alloc(c, (void **)&c->d_post, 256);
        if (rc == OF_OK) rc = dev_alloc(c, (void **)&c->d_prof, sizeof(unsigned long long) * OF_TIMELINE_MAX * c->sms);
        if (rc == OF_OK) {
            rc = upload_level_descs(c);
            cudaMemcpy(c->d_tm, c->tmS, sizeof(CUtensorMap) * levels, cudaMemcpyHostToDevice);
            cudaMemset(c->d_gbar, 0, 256);
            if (cudaDeviceSynchronize() != cudaSuccess) rc = fail(OF_ERR_CUDA, "descriptor upload failed: %s", cudaGetErrorString(cudaGetLastError()));
            int coop = 0;
            cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
            c->persistent = coop != 0;
        }
#ifdef OF_PROFILE
        if (getenv("OF_DEBUG"))
            for (int l = 0; l < levels; ++l)
                fprintf(stderr, "[optflow] level %d %dx%d pitch %d | K2 nseg %d nrp %d tiles %d grid %d warps %d smem %d | K3 tasks %d grid %d warps %d smem %d\n",
                        l, lv[l].W, lv[l].H, lv[l].pitch, c->k2[l].nseg, c->k2[l].nrp, c->k2[l].ntiles, c->k2[l].grid, c->k2[l].warps,
                        c->k2[l].smem, c->k3[l].ntasks, c->k3[l].grid, c->k3[l].warps, c->k3[l].smem);
#endif
    }
    if (rc != OF_OK) { std::string keep = g_err; of_destroy(c); g_err = keep; return nullptr; }
    return c;
}

void of_destroy(of_handle h)
{
    if (!h) return;
    cudaSetDevice(h->device);
    if (h->pipe.open) pipe_release(h);
    cudaDeviceSynchronize();
    drop_graphs(h);
    if (h->last_done) cudaEventDestroy(h->last_done);
    for (void *p : h->allocs) cudaFree(p);
    for (void *p : h->mask_allocs) cudaFree(p);
    delete h;
}

int of_compute(of_handle h, const float *I1, const float *I2, float *u, float *v, void *stream)
{
    return compute_any(h, OF_DTYPE_F32, I1, I2, u, v, stream);
}
int of_compute_u8(of_handle h, const uint8_t *I1, const uint8_t *I2, float *u, float *v, void *stream)
{
    return compute_any(h, OF_DTYPE_U8, I1, I2, u, v, stream);
}
int of_compute_u16(of_handle h, const uint16_t *I1, const uint16_t *I2, float *u, float *v, void *stream)
{
    return compute_any(h, OF_DTYPE_U16, I1, I2, u, v, stream);
}

int of_compute_dual(of_handle ha, of_handle hb, int dtype, const void *I1a, const void *I2a, float *ua, float *va,
                    const void *I1b, const void *I2b, float *ub, float *vb, void *stream)
{
    Job ja, jb;
    int rc = make_pair_job(ha, dtype, I1a, I2a, ua, va, ja);
    if (rc == OF_OK) rc = make_pair_job(hb, dtype, I1b, I2b, ub, vb, jb);
    if (rc != OF_OK) return rc;
    if (ha == hb) return fail(OF_ERR_INVALID_ARG, "of_compute_dual needs two different handles (each pair uses its handle's scratch)");
    if (ha->device != hb->device) return fail(OF_ERR_INVALID_ARG, "the two handles belong to different devices");
    if (!dual_eligible(ha, hb)) {                              // different problems, a mask, of_set_hoist, per-kernel mode: two ordinary solves
        rc = submit_job(ha, ja, (cudaStream_t)stream);
        if (rc == OF_OK) rc = submit_job(hb, jb, (cudaStream_t)stream);
        return rc;
    }
    return submit_dual(ha, ja, hb, jb, (cudaStream_t)stream);
}

int of_set_conditioning(of_handle h, float eps_rel, float max_step_px)
{
    if (!h) return fail(OF_ERR_INVALID_ARG, "null handle");
    if (!(eps_rel >= 0.f) || !(max_step_px > 0.f)) return fail(OF_ERR_INVALID_ARG, "eps_rel must be >= 0 and max_step_px > 0");
    h->eps_rel = eps_rel;
    h->max_step = max_step_px;
    drop_graphs(h);
    return OF_OK;
}

int of_set_equalisation(of_handle h, int radius)
{
    if (!h) return fail(OF_ERR_INVALID_ARG, "null handle");
    if (radius < 0 || radius > OF_MAX_WINDOW_RADIUS) return fail(OF_ERR_INVALID_ARG, "equalisation radius must be in [0,%d]", OF_MAX_WINDOW_RADIUS);
    if (radius > 0) {
        CU_TRY(cudaSetDevice(h->device));
        CU_TRY(cudaFuncSetAttribute(k0_equalise<uint8_t>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)eq_smem_bytes(OF_MAX_WINDOW_RADIUS, 1)));
        CU_TRY(cudaFuncSetAttribute(k0_equalise<uint16_t>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)eq_smem_bytes(OF_MAX_WINDOW_RADIUS, 2)));
        CU_TRY(cudaFuncSetAttribute(k0_equalise<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)eq_smem_bytes(OF_MAX_WINDOW_RADIUS, 4)));
        CU_TRY(cudaFuncSetAttribute(k0_equalise<uint8_t, 5>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)eq_smem_bytes(5, 1)));
        CU_TRY(cudaFuncSetAttribute(k0_equalise<uint16_t, 5>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)eq_smem_bytes(5, 2)));
    }
    h->eq_radius = radius;
    drop_graphs(h);
    return OF_OK;
}

int of_set_mask(of_handle h, const uint8_t *mask_host, int row_stride)
{
    if (!h) return fail(OF_ERR_INVALID_ARG, "null handle");
    if (mask_host && row_stride < h->W) return fail(OF_ERR_INVALID_ARG, "row_stride %d is smaller than the width %d", row_stride, h->W);
    CU_TRY(cudaSetDevice(h->device));
    CU_TRY(cudaDeviceSynchronize());                   // set-up call: nothing of this handle may be in flight
    drop_graphs(h);
    int rc = build_mask(h, mask_host, row_stride);
    if (rc != OF_OK) { std::string keep = g_err; build_mask(h, nullptr, 0); upload_level_descs(h); g_err = keep; return rc; }
    // tasks that no pass visits must read as "no vector" for ever: the level fields start from zero (M3)
    for (int l = 0; l < h->levels; ++l) {
        const size_t bytes = sizeof(float) * (size_t)h->lv[l].pitch * h->lv[l].H;
        CU_TRY(cudaMemset(h->u[l], 0, bytes));
        CU_TRY(cudaMemset(h->v[l], 0, bytes));
    }
    rc = upload_level_descs(h);
    if (rc != OF_OK) return rc;
    CU_TRY(cudaDeviceSynchronize());
    return OF_OK;
}

int of_set_graph(of_handle h, int enable)
{
    if (!h) return fail(OF_ERR_INVALID_ARG, "null handle");
    h->use_graph = enable != 0;
    if (!h->use_graph) drop_graphs(h);
    return OF_OK;
}

int of_set_persistent(of_handle h, int enable)
{
    if (!h) return fail(OF_ERR_INVALID_ARG, "null handle");
    h->persistent = enable != 0;
    drop_graphs(h);
    return OF_OK;
}

int of_set_fused(of_handle h, int enable)
{
    if (!h) return fail(OF_ERR_INVALID_ARG, "null handle");
    h->fuse_coarse = enable != 0;
    drop_graphs(h);
    CU_TRY(cudaSetDevice(h->device));
    CU_TRY(cudaDeviceSynchronize());
    return upload_level_descs(h);
}

int of_set_hoist(of_handle h, int enable)
{
    if (!h) return fail(OF_ERR_INVALID_ARG, "null handle");
    if (enable && !h->G) {
        CU_TRY(cudaSetDevice(h->device));
        int rc = dev_alloc(h, (void **)&h->G, sizeof(float) * 3 * h->plane);
        if (rc != OF_OK) return rc;
    }
    h->hoist = enable != 0;
    drop_graphs(h);
    return OF_OK;
}

int of_solve_timeline(of_handle h, int enable, int cta, unsigned long long *out_host, int max_entries)
{
    static_assert(OF_TIMELINE_MAX == SOLVE_TIMELINE_MAX, "timeline sizes out of sync");
    if (!h) return fail(OF_ERR_INVALID_ARG, "null handle");
    const int n = 1 + 2 * (h->levels - 1) + 4 * h->levels * h->iterations;
    if (n > OF_TIMELINE_MAX) return fail(OF_ERR_INVALID_ARG, "timeline of %d entries exceeds OF_TIMELINE_MAX", n);
    if (cta >= h->sms) return fail(OF_ERR_INVALID_ARG, "cta must be < %d", h->sms);
    int got = 0;
    if (out_host && h->prof_on) {
        CU_TRY(cudaSetDevice(h->device));
        CU_TRY(cudaDeviceSynchronize());
        got = std::min(n, max_entries);
        std::vector<unsigned long long> all((size_t)OF_TIMELINE_MAX * h->sms);
        CU_TRY(cudaMemcpy(all.data(), h->d_prof, sizeof(unsigned long long) * all.size(), cudaMemcpyDeviceToHost));
        // stamps are SM cycle counts: make them relative to each CTA's first stamp (CTAs start within ~1 us)
        for (int i = 0; i < got; ++i) {
            unsigned long long v = 0;
            for (int c = (cta >= 0 ? cta : 0); c < (cta >= 0 ? cta + 1 : h->sms); ++c)
                v = std::max(v, all[(size_t)c * OF_TIMELINE_MAX + i] - all[(size_t)c * OF_TIMELINE_MAX]);
            out_host[i] = v;
        }
    }
    if ((enable != 0) != h->prof_on) { h->prof_on = enable != 0; drop_graphs(h); }
    return got;
}

int of_get_validity(of_handle h, uint8_t *mask_dev, void *stream)
{
    if (!h || !mask_dev) return fail(OF_ERR_INVALID_ARG, "null argument");
    CU_TRY(cudaMemcpyAsync(mask_dev, h->valid, (size_t)h->W * h->H, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return OF_OK;
}

int of_level_size(of_handle h, int level, int *width, int *height)
{
    if (!h || level < 0 || level >= h->levels) return fail(OF_ERR_INVALID_ARG, "bad level");
    if (width) *width = h->lv[level].W;
    if (height) *height = h->lv[level].H;
    return OF_OK;
}

int of_last_launch_count(of_handle h) { return h ? h->last_launches : fail(OF_ERR_INVALID_ARG, "null handle"); }

int of_get_debug_plane(of_handle h, int level, int which, float *out_dev, void *stream)
{
    if (!h || !out_dev || level < 0 || level >= h->levels) return fail(OF_ERR_INVALID_ARG, "bad argument");
    const Level &L = h->lv[level];
    const float *src = nullptr;
    if (which == 0) src = h->pyr[0][level];
    else if (which == 1) src = h->pyr[1][level];
    else if (which == 2) src = h->u[level];
    else if (which == 3) src = h->v[level];
    else if (which >= 4 && which <= 8) src = h->S + (size_t)(which - 4) * h->plane;
    else if (which == 9 && level == 0) src = h->det;
    else return fail(OF_ERR_INVALID_ARG, "bad plane selector %d", which);
    return copy_plane_dense(src, L.pitch, L.W, L.H, out_dev, (cudaStream_t)stream);
}

int of_run_step(of_handle h, int level, int which, int repeat, void *stream)
{
    if (!h || level < 0 || level >= h->levels || which < 0 || which > 1 || repeat < 1) return fail(OF_ERR_INVALID_ARG, "bad argument");
    CU_TRY(cudaSetDevice(h->device));
    for (int i = 0; i < repeat; ++i) {
        if (which == 0) run_k2(h, level, h->pyr[0][level], h->pyr[1][level], false, (cudaStream_t)stream);
        else run_k3(h, level, h->u[level], h->v[level], h->lv[level].pitch, false, false, (cudaStream_t)stream);
    }
    CU_TRY(cudaGetLastError());
    return OF_OK;
}

int of_run_solve(of_handle h, int repeat, void *stream)
{
    if (!h || repeat < 1) return fail(OF_ERR_INVALID_ARG, "bad argument");
    if (!h->persistent) return fail(OF_ERR_STATE, "persistent mode is off");
    CU_TRY(cudaSetDevice(h->device));
    cudaStream_t st = (cudaStream_t)stream;
    if (!h->bench_out) {                                  // the discarded result gets a dense u, v pair of its own (first call only)
        int rc = dev_alloc(h, (void **)&h->bench_out, sizeof(float) * 2 * (size_t)h->W * h->H);
        if (rc != OF_OK) return rc;
    }
    for (int i = 0; i < repeat; ++i) {
        cudaError_t e = cudaSuccess;
        DISPATCH_RB(h->R, h->ww.box, (e = launch_solve<R, BX>(h, nullptr, 0, 1, h->bench_out, h->bench_out + (size_t)h->W * h->H, st)));
        if (e != cudaSuccess) return fail(OF_ERR_CUDA, "solve launch failed: %s", cudaGetErrorString(e));
    }
    return OF_OK;
}

int of_run_solve_dual(of_handle ha, of_handle hb, int repeat, void *stream)
{
    if (!ha || !hb || repeat < 1) return fail(OF_ERR_INVALID_ARG, "bad argument");
    if (!dual_eligible(ha, hb)) return fail(OF_ERR_STATE, "the two handles cannot share a launch (different problems, a mask, of_set_hoist or per-kernel mode)");
    CU_TRY(cudaSetDevice(ha->device));
    cudaStream_t st = (cudaStream_t)stream;
    of_context *hs[2] = {ha, hb};
    SolveArgs sa[2];
    for (int q = 0; q < 2; ++q) {
        of_context *h = hs[q];
        if (!h->bench_out) {                              // the discarded result gets a dense u, v pair of its own (first call only)
            int rc = dev_alloc(h, (void **)&h->bench_out, sizeof(float) * 2 * (size_t)h->W * h->H);
            if (rc != OF_OK) return rc;
        }
        fill_solve_args(h, 0, 1, h->bench_out, h->bench_out + (size_t)h->W * h->H, nullptr, sa[q]);
    }
    sa[1].prof = nullptr;
    for (int i = 0; i < repeat; ++i) {
        cudaError_t e = of_launch_solve_dual(ha->R, sa[0], sa[1], ha->sms, st);
        if (e != cudaSuccess) return fail(OF_ERR_CUDA, "solve (two pairs) launch failed: %s", cudaGetErrorString(e));
    }
    return OF_OK;
}

int of_field_accumulate(of_handle h, float *sum_dev, const float *field_dev, void *stream)
{
    if (!h || !sum_dev || !field_dev) return fail(OF_ERR_INVALID_ARG, "null argument");
    const size_t n = (size_t)h->W * h->H;
    kp_accumulate<<<2 * h->sms, 256, 0, (cudaStream_t)stream>>>(sum_dev, field_dev, n);
    CU_TRY(cudaGetLastError());
    return OF_OK;
}

int of_field_minmax(of_handle h, const float *field_dev, const uint8_t *valid_dev, float *out_dev, void *stream)
{
    if (!h || !field_dev || !out_dev) return fail(OF_ERR_INVALID_ARG, "null argument");
    const size_t n = (size_t)h->W * h->H;
    cudaStream_t st = (cudaStream_t)stream;
    kp_minmax_init<<<1, 1, 0, st>>>(h->d_post);
    kp_minmax<<<2 * h->sms, 256, 0, st>>>(field_dev, valid_dev, n, h->d_post);
    kp_minmax_finish<<<1, 1, 0, st>>>(h->d_post, out_dev);
    CU_TRY(cudaGetLastError());
    return OF_OK;
}

int of_bubble_count(of_handle h, const float *vx_dev, const uint8_t *valid_dev, float threshold, unsigned long long *out_dev, void *stream)
{
    if (!h || !vx_dev || !out_dev) return fail(OF_ERR_INVALID_ARG, "null argument");
    const size_t n = (size_t)h->W * h->H;
    cudaStream_t st = (cudaStream_t)stream;
    CU_TRY(cudaMemsetAsync(out_dev, 0, 2 * sizeof(unsigned long long), st));
    kp_bubble_count<<<2 * h->sms, 256, 0, st>>>(vx_dev, valid_dev, n, threshold, nullptr, out_dev);
    CU_TRY(cudaGetLastError());
    return OF_OK;
}

int of_bubble_threshold(of_handle h, const float *sum_dev, int n_fields, const uint8_t *valid_dev, float *threshold_dev, void *stream)
{
    if (!h || !sum_dev || !threshold_dev || n_fields < 1) return fail(OF_ERR_INVALID_ARG, "bad argument");
    const size_t n = (size_t)h->W * h->H;
    cudaStream_t st = (cudaStream_t)stream;
    kp_minmax_init<<<1, 1, 0, st>>>(h->d_post);
    kp_minmax<<<2 * h->sms, 256, 0, st>>>(sum_dev, valid_dev, n, h->d_post);
    kp_threshold_finish<<<1, 1, 0, st>>>(h->d_post, (float)n_fields, threshold_dev);
    CU_TRY(cudaGetLastError());
    return OF_OK;
}

int of_bubble_count_dev(of_handle h, const float *vx_dev, const uint8_t *valid_dev, const float *threshold_dev, unsigned long long *out_dev, void *stream)
{
    if (!h || !vx_dev || !out_dev || !threshold_dev) return fail(OF_ERR_INVALID_ARG, "null argument");
    const size_t n = (size_t)h->W * h->H;
    cudaStream_t st = (cudaStream_t)stream;
    CU_TRY(cudaMemsetAsync(out_dev, 0, 2 * sizeof(unsigned long long), st));
    kp_bubble_count<<<2 * h->sms, 256, 0, st>>>(vx_dev, valid_dev, n, 0.f, threshold_dev, out_dev);
    CU_TRY(cudaGetLastError());
    return OF_OK;
}

int of_pyramid_down(const float *src, int width, int height, float *dst, void *stream)
{
    if (!src || !dst || width < 1 || height < 1) return fail(OF_ERR_INVALID_ARG, "bad argument");
    int Wd = (width + 1) / 2, Hd = (height + 1) / 2;
    dim3 grid((Wd + K1_TW - 1) / K1_TW, (Hd + K1_TH - 1) / K1_TH, 1);
    k1_pyramid_down<float><<<grid, 256, 0, (cudaStream_t)stream>>>(src, nullptr, dst, nullptr, width, height, width, Wd, Hd, Wd, nullptr, nullptr, 0);
    CU_TRY(cudaGetLastError());
    return OF_OK;
}

int of_upsample_flow(const float *uc, const float *vc, int wc, int hc, float *u, float *v, int width, int height, void *stream)
{
    if (!uc || !vc || !u || !v || wc < 1 || hc < 1 || width < 1 || height < 1) return fail(OF_ERR_INVALID_ARG, "bad argument");
    if (wc != (width + 1) / 2 || hc != (height + 1) / 2) return fail(OF_ERR_INVALID_ARG, "coarse size must be ((W+1)/2,(H+1)/2)");
    dim3 grid((width + 63) / 64, (height + 3) / 4);
    k4_upsample_flow<<<grid, 256, 0, (cudaStream_t)stream>>>(uc, vc, wc, hc, wc, u, v, width, height, width, nullptr);
    CU_TRY(cudaGetLastError());
    return OF_OK;
}

// ------------------------------------------------------------------------------------------------
// frame pipeline (row a11)
// ------------------------------------------------------------------------------------------------
int of_stream_open(of_handle h, int dtype, int mode, int result_on_host)
{
    if (!h) return fail(OF_ERR_INVALID_ARG, "null handle");
    if (h->pipe.open) return fail(OF_ERR_STATE, "pipeline already open");
    if (dtype < OF_DTYPE_F32 || dtype > OF_DTYPE_U16) return fail(OF_ERR_INVALID_ARG, "bad dtype");
    if (mode != OF_STREAM_CONSECUTIVE && mode != OF_STREAM_PAIRS) return fail(OF_ERR_INVALID_ARG, "bad mode");
    CU_TRY(cudaSetDevice(h->device));
    Pipeline &p = h->pipe;
    p = Pipeline();
    p.dtype = dtype; p.mode = mode; p.host_result = result_on_host ? 1 : 0;
    size_t es = dtype == OF_DTYPE_U8 ? 1 : (dtype == OF_DTYPE_U16 ? 2 : 4);
    p.frame_bytes = es * (size_t)h->W * h->H;
    p.slot_bytes = p.frame_bytes * (mode == OF_STREAM_PAIRS ? 2 : 1);
    p.field_bytes = sizeof(float) * (size_t)h->W * h->H;
    cudaError_t e = cudaSuccess;
    auto ok = [&](cudaError_t r) { if (e == cudaSuccess) e = r; return r == cudaSuccess; };
    ok(cudaStreamCreateWithFlags(&p.s_copy, cudaStreamNonBlocking));
    ok(cudaStreamCreateWithFlags(&p.s_comp, cudaStreamNonBlocking));
    ok(cudaStreamCreateWithFlags(&p.s_down, cudaStreamNonBlocking));
    for (int i = 0; i < N_PIN; ++i) {
        ok(cudaHostAlloc(&p.pin[i], p.slot_bytes, cudaHostAllocDefault));
        ok(cudaMalloc(&p.raw[i], p.slot_bytes));
        ok(cudaEventCreateWithFlags(&p.h2d_done[i], cudaEventDisableTiming));
        ok(cudaEventCreateWithFlags(&p.cvt_done[i], cudaEventDisableTiming));
    }
    for (int i = 0; i < N_RES; ++i) {
        ok(cudaMalloc((void **)&p.res_dev[i], 2 * p.field_bytes + (size_t)h->W * h->H));
        if (p.host_result) ok(cudaHostAlloc((void **)&p.res_host[i], 2 * p.field_bytes + (size_t)h->W * h->H, cudaHostAllocDefault));
        ok(cudaEventCreateWithFlags(&p.solve_done[i], cudaEventDisableTiming));
        ok(cudaEventCreateWithFlags(&p.d2h_done[i], cudaEventDisableTiming));
    }
    if (e != cudaSuccess) {
        pipe_release(h);
        return fail(e == cudaErrorMemoryAllocation ? OF_ERR_ALLOC : OF_ERR_CUDA, "of_stream_open: %s", cudaGetErrorString(e));
    }
    p.open = true;
    return OF_OK;
}

void *of_stream_acquire(of_handle h)
{
    if (!h || !h->pipe.open) { fail(OF_ERR_STATE, "pipeline not open"); return nullptr; }
    Pipeline &p = h->pipe;
    if (p.cur_slot >= 0) return p.pin[p.cur_slot];          // acquired but not yet submitted
    int s = (int)(p.acquired % N_PIN);
    if (p.acquired >= N_PIN) {
        cudaError_t e = cudaEventSynchronize(p.h2d_done[s]);
        if (e != cudaSuccess) { fail(OF_ERR_CUDA, "cudaEventSynchronize: %s", cudaGetErrorString(e)); return nullptr; }
    }
    p.cur_slot = s;
    ++p.acquired;
    return p.pin[s];
}

int of_stream_submit(of_handle h)
{
    if (!h || !h->pipe.open) return fail(OF_ERR_STATE, "pipeline not open");
    Pipeline &p = h->pipe;
    if (p.cur_slot < 0) return fail(OF_ERR_STATE, "of_stream_submit without of_stream_acquire");
    const bool yields = (p.mode == OF_STREAM_PAIRS) || p.submitted >= 1;
    if (yields && p.produced - p.collected >= N_RES - 2)
        return fail(OF_ERR_STATE, "%d fields are waiting: call of_stream_result before submitting more", N_RES - 2);
    CU_TRY(cudaSetDevice(h->device));
    const int s = p.cur_slot;
    // upload: the device slot must have been consumed by the conversion of the frame it held before
    if (p.cvt_rec[s]) CU_TRY(cudaStreamWaitEvent(p.s_copy, p.cvt_done[s], 0));
    CU_TRY(cudaMemcpyAsync(p.raw[s], p.pin[s], p.slot_bytes, cudaMemcpyHostToDevice, p.s_copy));
    CU_TRY(cudaEventRecord(p.h2d_done[s], p.s_copy));
    CU_TRY(cudaStreamWaitEvent(p.s_comp, p.h2d_done[s], 0));

    Job j;
    memset(&j, 0, sizeof j);
    j.dtype = p.dtype;
    const int r = (int)(p.produced % N_RES);
    if (p.mode == OF_STREAM_PAIRS) {
        j.rawA = p.raw[s]; j.rawB = (const char *)p.raw[s] + p.frame_bytes; j.cvtA = 0; j.cvtB = 1; j.s1 = 0; j.s2 = 1;
    } else {
        const int ps = (int)(p.submitted % N_PYR);
        j.rawA = p.raw[s]; j.rawB = nullptr; j.cvtA = ps; j.cvtB = -1; j.s1 = 1 - ps; j.s2 = ps;
    }
    if (yields) {
        if (p.d2h_rec[r]) CU_TRY(cudaStreamWaitEvent(p.s_comp, p.d2h_done[r], 0));
        j.u_out = p.res_dev[r];
        j.v_out = p.res_dev[r] + (size_t)h->W * h->H;
        j.valid_out = reinterpret_cast<uint8_t *>(p.res_dev[r] + 2 * (size_t)h->W * h->H);
        int rc = submit_job(h, j, p.s_comp);
        if (rc != OF_OK) return rc;
        CU_TRY(cudaEventRecord(p.cvt_done[s], p.s_comp));   // (recorded after the solve: conservative)
        p.cvt_rec[s] = true;
        CU_TRY(cudaEventRecord(p.solve_done[r], p.s_comp));
        if (p.host_result) {
            CU_TRY(cudaStreamWaitEvent(p.s_down, p.solve_done[r], 0));
            CU_TRY(cudaMemcpyAsync(p.res_host[r], p.res_dev[r], 2 * p.field_bytes + (size_t)h->W * h->H, cudaMemcpyDeviceToHost, p.s_down));
            CU_TRY(cudaEventRecord(p.d2h_done[r], p.s_down));
            p.d2h_rec[r] = true;
        }
        ++p.produced;
    } else {
        // first frame of a consecutive stream: convert + pyramid only
        const int ps = (int)(p.submitted % N_PYR);
        run_convert(h, p.dtype, p.raw[s], nullptr, h->pyr[ps][0], nullptr, p.s_comp);
        for (int l = 0; l + 1 < h->levels; ++l) run_pyramid(h, l, h->pyr[ps][l], nullptr, h->pyr[ps][l + 1], nullptr, p.s_comp);
        CU_TRY(cudaGetLastError());
        CU_TRY(cudaEventRecord(p.cvt_done[s], p.s_comp));
        p.cvt_rec[s] = true;
        h->last_launches = h->levels;
    }
    ++p.submitted;
    p.cur_slot = -1;
    return OF_OK;
}

int of_stream_result(of_handle h, const float **u, const float **v, int *pair_index)
{
    if (!h || !h->pipe.open) return fail(OF_ERR_STATE, "pipeline not open");
    Pipeline &p = h->pipe;
    if (p.collected >= p.produced) return fail(OF_ERR_STATE, "no field pending");
    const int r = (int)(p.collected % N_RES);
    CU_TRY(cudaEventSynchronize(p.host_result ? p.d2h_done[r] : p.solve_done[r]));
    const float *base = p.host_result ? p.res_host[r] : p.res_dev[r];
    if (u) *u = base;
    if (v) *v = base + (size_t)h->W * h->H;
    if (pair_index) *pair_index = (int)p.collected;
    p.last_valid = reinterpret_cast<const uint8_t *>(base + 2 * (size_t)h->W * h->H);
    ++p.collected;
    return OF_OK;
}

int of_stream_result_validity(of_handle h, const uint8_t **valid)
{
    if (!h || !h->pipe.open) return fail(OF_ERR_STATE, "pipeline not open");
    if (!valid) return fail(OF_ERR_INVALID_ARG, "null argument");
    if (!h->pipe.last_valid) return fail(OF_ERR_STATE, "no field has been collected yet");
    *valid = h->pipe.last_valid;
    return OF_OK;
}

int of_stream_close(of_handle h)
{
    if (!h) return fail(OF_ERR_INVALID_ARG, "null handle");
    if (!h->pipe.open) return OF_OK;
    cudaSetDevice(h->device);
    pipe_release(h);
    drop_graphs(h);
    return OF_OK;
}

}  // extern "C"
