// kern_gen.cu -- the generic shared-memory passes (run-time radices 2, 3, 4, 5, 7) and their launches.
// Product code; shares nothing with oracle/.
#include "mm_kernels.h"
#include "fft_generic.cuh"

namespace mm {

bool gen_set_smem()
{
    const int lim = 224 * 1024;
    return cudaFuncSetAttribute(k_gen_fwd_x, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) == cudaSuccess &&
           cudaFuncSetAttribute(k_gen_y<-1>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) == cudaSuccess &&
           cudaFuncSetAttribute(k_gen_y<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) == cudaSuccess &&
           cudaFuncSetAttribute(k_gen_mid, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) == cudaSuccess &&
           cudaFuncSetAttribute(k_gen_inv_x, cudaFuncAttributeMaxDynamicSharedMemorySize, lim) == cudaSuccess;
}

void gen_fwd_x(const Geom& g, const FftPlan& pl, const float* m, float2* specA, int tx, size_t bytes, cudaStream_t st)
{
    const int npair = 3 * g.Nz * ((g.Ny + 1) / 2);
    k_gen_fwd_x<<<(npair + tx - 1) / tx, 256, bytes, st>>>(g, pl, m, specA, tx);
}

void gen_y(const Geom& g, const FftPlan& pl, int sgn, const float2* src, float2* dst, int tx, size_t bytes,
           cudaStream_t st)
{
    dim3 grid((g.Cx + tx - 1) / tx, 3 * g.Nz);
    if (sgn < 0) k_gen_y<-1><<<grid, 256, bytes, st>>>(g, pl, src, dst, tx);
    else k_gen_y<1><<<grid, 256, bytes, st>>>(g, pl, src, dst, tx);
}

void gen_mid(const Geom& g, const FftPlan& pl, float2* spec, const float* khat, int axis, int tx, size_t bytes,
             cudaStream_t st)
{
    dim3 grid((g.Cx + tx - 1) / tx, axis == 2 ? g.Py : 1);
    k_gen_mid<<<grid, 256, bytes, st>>>(g, pl, spec, khat, axis, tx);
}

void gen_mul1d(const Geom& g, float2* spec, const float* khat, cudaStream_t st)
{
    k_gen_mul1d<<<(g.Cx + 127) / 128, 128, 0, st>>>(g, spec, khat);
}

void gen_inv_x(const Geom& g, const FftPlan& pl, const float2* specA, const EpiParams& ep, int tx, size_t bytes,
               cudaStream_t st)
{
    const int npy = (g.Ny + 1) / 2;
    dim3 grid((npy + tx - 1) / tx, g.Nz);
    k_gen_inv_x<<<grid, 256, bytes, st>>>(g, pl, specA, ep, tx);
}

}  // namespace mm
