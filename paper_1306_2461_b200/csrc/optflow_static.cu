// optflow_static.cu -- of_field_minmax_static: the min / max step of eq. 3 (of_field_minmax in optflow.cu) for
// callers that cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  It takes no
// handle (of_create allocates) and calls no cudaMalloc / cudaFree or allocating library routine.  Its scratch memory -- one
// partial {min, max} per 4096-pixel chunk plus an arrival counter -- is the file-scope __device__ array below, which every GPU
// that loads liboptflow.so holds until the process exits (OF_STATIC_SCRATCH_BYTES = 33 024 bytes).
//
// Host code never passes the array's NAME to a kernel: in host code that name is a host-side stand-in, not a device address.  The
// device address is taken once per device, with that device current, by cudaGetSymbolAddress (static_scratch_ptr below) and handed
// to the kernel as an ordinary pointer argument.
//
// All calls share the one array, and it keeps the contents of the last call: the arrival counter is cleared on the stream before
// every launch (and reset by the kernel's last block), the partials are all rewritten before they are read.  Two calls that
// overlap on the GPU (different streams without an ordering between them, or two host threads) race on it; order them.
#include <cuda_runtime.h>
#include <cstdint>
#include <cstdio>
#include <mutex>
#include "../../include/optflow.h"

int of_detail_fail(int code, const char *msg);        // optflow.cu: sets the string of_last_error returns

// The scratch memory: arrival counter (first 256 bytes), then one {min, max} partial per 4096-pixel chunk.
static __device__ __align__(256) unsigned char g_static_scratch[OF_STATIC_SCRATCH_BYTES];

namespace {

constexpr int ST_CHUNK = 4096;                         // pixels per block = per partial
constexpr int ST_THREADS = 256;
constexpr int ST_HEADER = 256;                         // bytes in front of the partials: the arrival counter
constexpr size_t ST_MAX_CHUNKS = OF_STATIC_MAX_PIXELS / ST_CHUNK;
static_assert(OF_STATIC_MAX_PIXELS % ST_CHUNK == 0, "maximum size is a whole number of chunks");
static_assert(OF_STATIC_SCRATCH_BYTES == ST_HEADER + 8 * ST_MAX_CHUNKS, "optflow.h states the size of the array");

// same order-preserving map float <-> unsigned as of_post.cuh (integer min / max = float min / max)
__device__ __forceinline__ unsigned st_f2ord(float x)
{
    const unsigned u = __float_as_uint(x);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float st_ord2f(unsigned o) { return __uint_as_float((o & 0x80000000u) ? (o & 0x7fffffffu) : ~o); }

__device__ __forceinline__ void st_take(float x, bool ok, unsigned &lo, unsigned &hi)
{
    if (ok && x == x) {
        const unsigned o = st_f2ord(x);
        lo = min(lo, o);
        hi = max(hi, o);
    }
}

// {lo, hi} of the block's 256 threads in thread 0 (8 warps)
__device__ __forceinline__ void st_block_reduce(unsigned &lo, unsigned &hi, unsigned (*sh)[ST_THREADS / 32])
{
    lo = __reduce_min_sync(0xffffffffu, lo);
    hi = __reduce_max_sync(0xffffffffu, hi);
    const int w = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) { sh[0][w] = lo; sh[1][w] = hi; }
    __syncthreads();
    if (threadIdx.x < 32) {
        lo = threadIdx.x < ST_THREADS / 32 ? sh[0][threadIdx.x] : 0xffffffffu;
        hi = threadIdx.x < ST_THREADS / 32 ? sh[1][threadIdx.x] : 0u;
        lo = __reduce_min_sync(0xffffffffu, lo);
        hi = __reduce_max_sync(0xffffffffu, hi);
    }
    __syncthreads();
}

// Block b reduces pixels [b * 4096, min(n, (b + 1) * 4096)) to scratch partial b; the block that arrives last reduces the
// partials in index order to out[0] = min, out[1] = max and resets the counter.  Integer min / max: the result does not depend
// on which block is last.  `scratch` is the device address of g_static_scratch (a kernel argument, see the header comment).
__global__ void __launch_bounds__(ST_THREADS) kp_minmax_static(const float *__restrict__ f, const uint8_t *__restrict__ valid, size_t n,
                                                               unsigned char *scratch, float *__restrict__ out, int vec)
{
    __shared__ unsigned sh[2][ST_THREADS / 32];
    __shared__ unsigned last;
    unsigned *counter = reinterpret_cast<unsigned *>(scratch);
    uint2 *partial = reinterpret_cast<uint2 *>(scratch + ST_HEADER);

    const size_t base = (size_t)blockIdx.x * ST_CHUNK;
    const size_t end = min(n, base + ST_CHUNK);
    unsigned lo = 0xffffffffu, hi = 0u;
    if (vec) {                                         // f 16-byte aligned, valid NULL or 4-byte aligned; base is a multiple of 4
        const size_t end4 = base + ((end - base) & ~(size_t)3);
        for (size_t i = base + 4 * threadIdx.x; i < end4; i += 4 * ST_THREADS) {
            const float4 x = *reinterpret_cast<const float4 *>(f + i);
            uchar4 m = make_uchar4(1, 1, 1, 1);
            if (valid != nullptr) m = *reinterpret_cast<const uchar4 *>(valid + i);
            st_take(x.x, m.x != 0, lo, hi);
            st_take(x.y, m.y != 0, lo, hi);
            st_take(x.z, m.z != 0, lo, hi);
            st_take(x.w, m.w != 0, lo, hi);
        }
        for (size_t i = end4 + threadIdx.x; i < end; i += ST_THREADS) st_take(f[i], valid == nullptr || valid[i] != 0, lo, hi);
    } else {
        for (size_t i = base + threadIdx.x; i < end; i += ST_THREADS) st_take(f[i], valid == nullptr || valid[i] != 0, lo, hi);
    }
    st_block_reduce(lo, hi, sh);
    if (threadIdx.x == 0) {
        partial[blockIdx.x] = make_uint2(lo, hi);
        __threadfence();                               // the partial is visible before the arrival is
        last = atomicAdd(counter, 1u) == gridDim.x - 1 ? 1u : 0u;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    lo = 0xffffffffu, hi = 0u;
    for (unsigned i = threadIdx.x; i < gridDim.x; i += ST_THREADS) {
        const uint2 p = __ldcg(partial + i);
        lo = min(lo, p.x);
        hi = max(hi, p.y);
    }
    st_block_reduce(lo, hi, sh);
    if (threadIdx.x == 0) {
        out[0] = st_ord2f(lo);
        out[1] = st_ord2f(hi);
        *counter = 0u;
    }
}

// Device address of g_static_scratch on the current device: cudaGetSymbolAddress once per device, with that device current.
constexpr int ST_MAX_DEVICES = 64;
std::mutex g_static_mutex;
unsigned char *g_static_ptr[ST_MAX_DEVICES] = {};

int static_scratch_ptr(unsigned char **ptr)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        char msg[256];
        snprintf(msg, sizeof msg, "of_field_minmax_static: cudaGetDevice failed: %s", cudaGetErrorString(e));
        return of_detail_fail(OF_ERR_CUDA, msg);
    }
    if (dev < 0 || dev >= ST_MAX_DEVICES) return of_detail_fail(OF_ERR_INVALID_ARG, "of_field_minmax_static: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (g_static_ptr[dev] == nullptr) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || p == nullptr) {
            char msg[256];
            snprintf(msg, sizeof msg, "of_field_minmax_static: cudaGetSymbolAddress(g_static_scratch) failed on device %d: %s", dev,
                     cudaGetErrorString(e));
            return of_detail_fail(OF_ERR_CUDA, msg);
        }
        g_static_ptr[dev] = static_cast<unsigned char *>(p);
    }
    *ptr = g_static_ptr[dev];
    return OF_OK;
}

}   // namespace

extern "C" int of_field_minmax_static(const float *field_dev, const uint8_t *valid_dev, size_t n, float *out_dev, void *stream)
{
    if (!field_dev || !out_dev) return of_detail_fail(OF_ERR_INVALID_ARG, "of_field_minmax_static: null argument");
    if (n == 0) return of_detail_fail(OF_ERR_INVALID_ARG, "of_field_minmax_static: empty field");
    if (n > (size_t)OF_STATIC_MAX_PIXELS) {
        char msg[256];
        snprintf(msg, sizeof msg,
                 "of_field_minmax_static: %zu pixels exceed the maximum of %zu (OF_STATIC_MAX_PIXELS) that the static scratch array holds; "
                 "use of_field_minmax",
                 n, (size_t)OF_STATIC_MAX_PIXELS);
        return of_detail_fail(OF_ERR_INVALID_ARG, msg);
    }
    if (((uintptr_t)field_dev & 3) || ((uintptr_t)out_dev & 3)) return of_detail_fail(OF_ERR_INVALID_ARG, "of_field_minmax_static: misaligned pointer");
    unsigned char *scratch = nullptr;
    int rc = static_scratch_ptr(&scratch);
    if (rc != OF_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const int vec = (((uintptr_t)field_dev & 15) == 0 && (valid_dev == nullptr || ((uintptr_t)valid_dev & 3) == 0)) ? 1 : 0;
    const unsigned grid = (unsigned)((n + ST_CHUNK - 1) / ST_CHUNK);
    cudaError_t e = cudaMemsetAsync(scratch, 0, ST_HEADER, st);      // the arrival counter starts at zero whatever the last call left
    if (e == cudaSuccess) {
        kp_minmax_static<<<grid, ST_THREADS, 0, st>>>(field_dev, valid_dev, n, scratch, out_dev, vec);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        char msg[256];
        snprintf(msg, sizeof msg, "of_field_minmax_static: launch failed: %s", cudaGetErrorString(e));
        return of_detail_fail(OF_ERR_CUDA, msg);
    }
    return OF_OK;
}
