// kern_static.cu -- mm_average_static: <f> over all cells (the reduction of mm_average) for callers
// that cannot allocate: no context, no cudaMalloc / cudaFree / allocating library call anywhere on this path.
// Product code; shares nothing with oracle/.
//
// The per-block partial sums and the arrival counter live in ONE file-scope device array of fixed size (below).
// Every GPU that loads the library holds that array until the process exits.  All calls share it: two calls that
// overlap on the GPU (different streams, no ordering between them) race on it.  Nothing in it has to survive a call:
// the counter is cleared at the start of every call, every partial sum a call reads was written by that call.
#include <cstdio>
#include <cstring>
#include <cuda_runtime.h>
#include "../../include/mm.h"

namespace {

constexpr int ST_BLOCK = 256;                    // threads per block
constexpr int ST_CHUNK = 8192;                   // cells per block (32 per thread)
constexpr int ST_MAX_BLOCKS = 8192;              // => at most 8192 * 8192 = 67 108 864 cells per call
constexpr int ST_MAX_DEV = 64;

struct __align__(256) StScratch {
    double part[3][ST_MAX_BLOCKS];               // per-block sums of the three components (192 KB)
    unsigned int arrived;                        // blocks that have published their sums
};

// In HOST code this name is a host-side stand-in, not a device address: only cudaGetSymbolAddress (st_scratch_ptr)
// turns it into the pointer a kernel may be given.  Device code below takes that pointer as an argument.
static __device__ __align__(256) StScratch st_scratch;

// Each block sums one chunk of ST_CHUNK cells in fp64 and publishes the three sums; the block that arrives last adds
// the published sums in block order (so the result does not depend on the order the blocks ran in), divides by n and
// writes avg_dev[3].
__global__ void __launch_bounds__(ST_BLOCK)
k_average_static(size_t n, const float* __restrict__ f, StScratch* __restrict__ sc, double* __restrict__ avg_dev)
{
    __shared__ double sh[3][ST_BLOCK / 32];
    __shared__ bool last;
    const int tid = threadIdx.x;
    const size_t i0 = (size_t)blockIdx.x * ST_CHUNK;
    const size_t i1 = i0 + ST_CHUNK < n ? i0 + ST_CHUNK : n;
    double acc[3] = { 0.0, 0.0, 0.0 };
    for (size_t i = i0 + tid; i < i1; i += ST_BLOCK)
        for (int cc = 0; cc < 3; ++cc) acc[cc] += (double)f[i + cc * n];
    for (int cc = 0; cc < 3; ++cc) {
        double v = acc[cc];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if ((tid & 31) == 0) sh[cc][tid >> 5] = v;
    }
    __syncthreads();
    if (tid < 3) {
        double v = 0.0;
        for (int w = 0; w < ST_BLOCK / 32; ++w) v += sh[tid][w];
        sc->part[tid][blockIdx.x] = v;
    }
    __syncthreads();
    if (tid == 0) {
        __threadfence();                         // the three sums are visible before the arrival is counted
        last = atomicAdd(&sc->arrived, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    for (int cc = 0; cc < 3; ++cc) {
        double v = 0.0;
        for (unsigned b = tid; b < gridDim.x; b += ST_BLOCK) v += __ldcg(&sc->part[cc][b]);
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if ((tid & 31) == 0) sh[cc][tid >> 5] = v;
    }
    __syncthreads();
    if (tid < 3) {
        double v = 0.0;
        for (int w = 0; w < ST_BLOCK / 32; ++w) v += sh[tid][w];
        avg_dev[tid] = v / (double)n;
    }
    if (tid == 0) sc->arrived = 0;               // left clean for the next call (which clears it again anyway)
}

mm_status st_fail(mm_status s, char* err, size_t err_len, const char* msg, const char* detail = nullptr)
{
    if (err && err_len) {
        if (detail) snprintf(err, err_len, "mm_average_static: %s: %s", msg, detail);
        else snprintf(err, err_len, "mm_average_static: %s", msg);
    }
    return s;
}

// device address of st_scratch on the CURRENT device, looked up once per device (set-up: the first call on a device)
cudaError_t st_scratch_ptr(StScratch** out)
{
    static StScratch* ptr[ST_MAX_DEV] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= ST_MAX_DEV) return cudaErrorInvalidDevice;
    StScratch* p = __atomic_load_n(&ptr[dev], __ATOMIC_ACQUIRE);
    if (!p) {
        e = cudaGetSymbolAddress((void**)&p, st_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        __atomic_store_n(&ptr[dev], p, __ATOMIC_RELEASE);      // (two threads racing here store the same address)
    }
    *out = p;
    return cudaSuccess;
}

}  // namespace

extern "C" mm_status mm_average_static(const float* field_dev, size_t ncell, double* avg_dev, void* stream, char* err,
                                       size_t err_len)
{
    if (err && err_len) err[0] = '\0';
    if (!field_dev || !avg_dev) return st_fail(MM_EINVAL, err, err_len, "NULL field_dev or avg_dev");
    if (ncell == 0) return st_fail(MM_EINVAL, err, err_len, "ncell must be positive");
    const size_t max_cells = (size_t)ST_MAX_BLOCKS * ST_CHUNK;
    if (ncell > max_cells) {
        char d[160];
        snprintf(d, sizeof d, "%zu cells asked, the static scratch array covers at most %zu (MM_AVERAGE_STATIC_MAX_CELLS); "
                              "use mm_average of a context for larger fields", ncell, max_cells);
        return st_fail(MM_EUNSUPPORTED, err, err_len, "field too large", d);
    }
    StScratch* sc = nullptr;
    cudaError_t e = st_scratch_ptr(&sc);
    if (e != cudaSuccess) return st_fail(MM_ECUDA, err, err_len, "cudaGetSymbolAddress(st_scratch)", cudaGetErrorString(e));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    e = cudaMemsetAsync(&sc->arrived, 0, sizeof(unsigned int), st);          // what must start at zero
    if (e != cudaSuccess) return st_fail(MM_ECUDA, err, err_len, "cudaMemsetAsync", cudaGetErrorString(e));
    const unsigned nblock = (unsigned)((ncell + ST_CHUNK - 1) / ST_CHUNK);
    k_average_static<<<nblock, ST_BLOCK, 0, st>>>(ncell, field_dev, sc, avg_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return st_fail(MM_ECUDA, err, err_len, "kernel launch", cudaGetErrorString(e));
    return MM_OK;
}
