// kern_x.cu -- x passes (a1, a5, fused a5-a10): size-specialised kernels, their launches and size dispatch.
// Product code; shares nothing with oracle/.
#include <string>
#include <vector>
#include "mm_kernels.h"
#include "epilogue.cuh"
#include "fft_fast.cuh"

namespace mm {
namespace ff {
template <int T, int E, bool PER>
bool launch_fwd_x(const FastPlan& fp, const Geom& g, cudaStream_t st, const float* m, float2* specA)
{
    const size_t bytes = (size_t)(128 / T) * T * (E + 1) * sizeof(float2);
    static bool once[MM_MAX_DEV] = {};
    if (!ensure_smem_dev(k_fwd_x<T, E, PER>, bytes, once)) return false;
    const int nslot = 128 / T;
    const int npair = 3 * g.Nz * ((g.Ny + 1) / 2);
    const int want = (npair + nslot - 1) / nslot;
    const int grid = want < fp.nsm * 8 ? want : fp.nsm * 8;
    if ((fp.x_pipe & 1) && g.Nx % 4 == 0) {
        static bool oncep[MM_MAX_DEV] = {};
        if (!ensure_smem_dev(k_fwd_x_p<T, E, PER>, bytes, oncep)) return false;
        const int gridp = want < fp.nsm * 4 ? want : fp.nsm * 4;      // resident blocks: the loop is pipelined
        k_fwd_x_p<T, E, PER><<<gridp, 128, bytes, st>>>(g, m, specA, fp.tw[0]);
        return true;
    }
    k_fwd_x<T, E, PER><<<grid, 128, bytes, st>>>(g, m, specA, fp.tw[0]);
    return true;
}

template <int T, int E, bool PER>
bool launch_inv_x(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, const EpiParams& ep)
{
    constexpr int NX = PER ? T * E : T * E / 2;
    const size_t bytes = (size_t)(128 / T) * (T * (E + 1) + 2 * NX) * sizeof(float2);
    static bool once[MM_MAX_DEV] = {};
    if (!ensure_smem_dev(k_inv_x<T, E, PER>, bytes, once)) return false;
    const int nslot = 128 / T;
    const int npair = g.Nz * ((g.Ny + 1) / 2);
    const int want = (npair + nslot - 1) / nslot;
    const int grid = want < fp.nsm * 8 ? want : fp.nsm * 8;
    k_inv_x<T, E, PER><<<grid, 128, bytes, st>>>(g, specA, fp.tw[0], ep);
    return true;
}

template <int T, int E, bool PER>
bool launch_inv_x_h(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, float* out, float scale)
{
    const size_t bytes = (size_t)(128 / T) * T * (E + 1) * sizeof(float2);
    static bool once[MM_MAX_DEV] = {};
    if (!ensure_smem_dev(k_inv_x_h<T, E, PER>, bytes, once)) return false;
    const int nslot = 128 / T;
    const int npair = 3 * g.Nz * ((g.Ny + 1) / 2);
    const int want = (npair + nslot - 1) / nslot;
    const int grid = want < fp.nsm * 8 ? want : fp.nsm * 8;
    if ((fp.x_pipe & 2) && g.CxS % 2 == 0) {      // measured slower than the plain form on B200: off by default
        static bool oncep[MM_MAX_DEV] = {};
        if (!ensure_smem_dev(k_inv_x_h_p<T, E, PER>, bytes, oncep)) return false;
        const int gridp = want < fp.nsm * 4 ? want : fp.nsm * 4;
        k_inv_x_h_p<T, E, PER><<<gridp, 128, bytes, st>>>(g, specA, fp.tw[0], out, scale);
        return true;
    }
    k_inv_x_h<T, E, PER><<<grid, 128, bytes, st>>>(g, specA, fp.tw[0], out, scale);
    return true;
}

template <int T, int E, bool PER>
bool launch_fwd_x_r(const FastPlan& fp, const Geom& g, cudaStream_t st, const float* m, float2* specA)
{
    const size_t bytes = (size_t)(128 / T) * T * (E + 1) * sizeof(float2);
    static bool once[MM_MAX_DEV] = {};
    if (!ensure_smem_dev(k_fwd_x_r<T, E, PER>, bytes, once)) return false;
    const int nslot = 128 / T;
    const int want = (3 * g.Nz * g.Ny + nslot - 1) / nslot;
    const int grid = want < fp.nsm * 8 ? want : fp.nsm * 8;
    k_fwd_x_r<T, E, PER><<<grid, 128, bytes, st>>>(g, m, specA, fp.tw[0], fp.twx);
    return true;
}

template <int T, int E, bool PER>
bool launch_inv_x_h_r(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, float* out,
                      float scale)
{
    const size_t bytes = (size_t)(128 / T) * T * (E + 1) * sizeof(float2);
    static bool once[MM_MAX_DEV] = {};
    if (!ensure_smem_dev(k_inv_x_h_r<T, E, PER>, bytes, once)) return false;
    const int nslot = 128 / T;
    const int want = (3 * g.Nz * g.Ny + nslot - 1) / nslot;
    const int grid = want < fp.nsm * 8 ? want : fp.nsm * 8;
    k_inv_x_h_r<T, E, PER><<<grid, 128, bytes, st>>>(g, specA, fp.tw[0], fp.twx, out, scale);
    return true;
}

#define MM_FF_SIZES(L, CALL)                 \
    switch (L) {                              \
    case 32: { CALL(4, 8); } break;           \
    case 64: { CALL(8, 8); } break;           \
    case 192: { CALL(8, 24); } break;         \
    case 384: { CALL(8, 48); } break;         \
    case 768: { CALL(16, 48); } break;        \
    case 128: { CALL(8, 16); } break;         \
    case 256: { CALL(16, 16); } break;        \
    case 512: { CALL(16, 32); } break;        \
    case 1024: { CALL(32, 32); } break;       \
    default: break;                           \
    }
}  // namespace ff

// ---------------------------------------------------------------------------------------------
// x lines of 4096 (2048 cells, open; 4096 cells, periodic -- PAPER.md:245, the largest 2D grid of Table 1): one
// decimation-in-time level outside the kernels.  The even and the odd samples of a row are two real sequences of
// half the length; each goes through the 2048-point real transform (k_fwd_x_r / k_inv_x_h_r, unchanged), and
//   forward:  X[j] = E[j] + w^j O[j],  X[2048 - j] = conj(E[j] - w^j O[j]),  j <= 1024,  w = exp(-2 pi i / 4096)
//   inverse:  E'[j] = X[j] + conj X[2048 - j],  O'[j] = conj(w^j) (X[j] - conj X[2048 - j])
namespace ff {
__global__ void k_x_deinterleave(const float2* __restrict__ m, float* __restrict__ tmp, size_t nrow, int half)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nrow * half; i += (size_t)gridDim.x * blockDim.x) {
        const size_t row = i / half, n = i - row * half;
        const float2 v = m[i];
        tmp[(2 * row) * half + n] = v.x;
        tmp[(2 * row + 1) * half + n] = v.y;
    }
}
__global__ void k_x_interleave(const float* __restrict__ tmp, float2* __restrict__ out, size_t nrow, int half)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nrow * half; i += (size_t)gridDim.x * blockDim.x) {
        const size_t row = i / half, n = i - row * half;
        out[i] = make_float2(tmp[(2 * row) * half + n], tmp[(2 * row + 1) * half + n]);
    }
}
template <int SGN>
__global__ void k_x_combine(float2* __restrict__ ts, float2* __restrict__ specA, size_t nrow, int CxS,
                            const float2* __restrict__ tw4)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    const size_t row = blockIdx.y;
    if (j > 1024 || row >= nrow) return;
    float2* e = ts + (2 * row) * MM_XS_STRIDE + j;
    float2* o = ts + (2 * row + 1) * MM_XS_STRIDE + j;
    float2* x = specA + row * CxS;
    const float2 w = __ldg(tw4 + j);
    if (SGN < 0) {
        const float2 E = *e, wO = cmul(w, *o);
        x[j] = cadd(E, wO);
        if (j != 1024) x[2048 - j] = cconj(csub(E, wO));
    } else {
        const float2 A = x[j], B = cconj(x[2048 - j]);
        *e = cadd(A, B);
        *o = cmul(cconj(w), csub(A, B));
    }
}
}  // namespace ff

bool fast_fwd_x(const FastPlan& fp, const Geom& g, cudaStream_t st, const float* m, float2* specA)
{
    if (fp.x_split) {
        const size_t nrow = (size_t)3 * g.Nz * g.Ny;
        const Geom h = x_split_geom(g);
        ff::k_x_deinterleave<<<fp.nsm * 8, 256, 0, st>>>(reinterpret_cast<const float2*>(m), fp.xs_real, nrow, g.Nx / 2);
        if (!(g.perx ? ff::launch_fwd_x_r<32, 32, true>(fp, h, st, fp.xs_real, fp.xs_spec)
                     : ff::launch_fwd_x_r<32, 32, false>(fp, h, st, fp.xs_real, fp.xs_spec)))
            return false;
        dim3 cg((1025 + 127) / 128, (unsigned)nrow);
        ff::k_x_combine<-1><<<cg, 128, 0, st>>>(fp.xs_spec, specA, nrow, g.CxS, fp.twx4);
        return true;
    }
    if (fp.ok_xr) {
        if (g.Px == 1536) return g.perx ? ff::launch_fwd_x_r<16, 48, true>(fp, g, st, m, specA)
                                        : ff::launch_fwd_x_r<16, 48, false>(fp, g, st, m, specA);
        if (g.Px == 2048) return g.perx ? ff::launch_fwd_x_r<32, 32, true>(fp, g, st, m, specA)
                                        : ff::launch_fwd_x_r<32, 32, false>(fp, g, st, m, specA);
        return false;
    }
    if (!fp.ok_x) return false;
    bool r = false;
#define CALL(T, E) r = g.perx ? ff::launch_fwd_x<T, E, true>(fp, g, st, m, specA) \
                              : ff::launch_fwd_x<T, E, false>(fp, g, st, m, specA)
    MM_FF_SIZES(g.Px, CALL)
#undef CALL
    return r;
}

// fused inverse x + epilogue (bit 8): power-of-two lengths only; the split pass (bit 16) is the default
bool fast_inv_x(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, const EpiParams& ep)
{
    if (!fp.ok_x) return false;
#define CALL(T, E) return g.perx ? ff::launch_inv_x<T, E, true>(fp, g, st, specA, ep) \
                                 : ff::launch_inv_x<T, E, false>(fp, g, st, specA, ep)
    switch (g.Px) {
    case 64: CALL(8, 8);
    case 128: CALL(8, 16);
    case 256: CALL(16, 16);
    case 512: CALL(16, 32);
    case 1024: CALL(32, 32);
    default: break;
    }
#undef CALL
    return false;
}

// split variant of the last pass, first half: H_ms * scale -> out (a field)
bool fast_inv_x_h(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, float* out,
                         float scale)
{
    if (fp.x_split) {
        const size_t nrow = (size_t)3 * g.Nz * g.Ny;
        const Geom h = x_split_geom(g);
        dim3 cg((1025 + 127) / 128, (unsigned)nrow);
        ff::k_x_combine<1><<<cg, 128, 0, st>>>(fp.xs_spec, const_cast<float2*>(specA), nrow, g.CxS, fp.twx4);
        if (!(g.perx ? ff::launch_inv_x_h_r<32, 32, true>(fp, h, st, fp.xs_spec, fp.xs_real, scale)
                     : ff::launch_inv_x_h_r<32, 32, false>(fp, h, st, fp.xs_spec, fp.xs_real, scale)))
            return false;
        ff::k_x_interleave<<<fp.nsm * 8, 256, 0, st>>>(fp.xs_real, reinterpret_cast<float2*>(out), nrow, g.Nx / 2);
        return true;
    }
    if (fp.ok_xr) {
        if (g.Px == 1536) return g.perx ? ff::launch_inv_x_h_r<16, 48, true>(fp, g, st, specA, out, scale)
                                        : ff::launch_inv_x_h_r<16, 48, false>(fp, g, st, specA, out, scale);
        if (g.Px == 2048) return g.perx ? ff::launch_inv_x_h_r<32, 32, true>(fp, g, st, specA, out, scale)
                                        : ff::launch_inv_x_h_r<32, 32, false>(fp, g, st, specA, out, scale);
        return false;
    }
    if (!fp.ok_x) return false;
    bool r = false;
#define CALL(T, E) r = g.perx ? ff::launch_inv_x_h<T, E, true>(fp, g, st, specA, out, scale) \
                              : ff::launch_inv_x_h<T, E, false>(fp, g, st, specA, out, scale)
    MM_FF_SIZES(g.Px, CALL)
#undef CALL
    return r;
}


}  // namespace mm
