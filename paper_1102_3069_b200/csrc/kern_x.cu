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
        const int gridp = want < fp.nsm * 4 ? want : fp.nsm * 4;      // resident blocks: the loop is pipelined
        if (fp.x_pipe & 4) {                // rows by bulk copies (one mbarrier per slot behind the exchange buffers)
            static bool onceb[MM_MAX_DEV] = {};
            if (!ensure_smem_dev(k_fwd_x_p<T, E, PER, true>, bytes + 64, onceb)) return false;
            k_fwd_x_p<T, E, PER, true><<<gridp, 128, bytes + 64, st>>>(g, m, specA, fp.tw[0]);
            return true;
        }
        static bool oncep[MM_MAX_DEV] = {};
        if (!ensure_smem_dev(k_fwd_x_p<T, E, PER>, bytes, oncep)) return false;
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
// x lines whose length Px has no kernel of its own but factors as Px = R * Ls, R in {2, 3, 4, 5, 7, 9}, Ls a length the
// real-transform kernels take (4096 = 2 * 2048: the 2048^2 grid of the paper's Table 1; 2^n * {5, 7, 9},
// PAPER.md:171): one decimation-in-time level outside the kernels.  The samples R n + q of a row are R real sequences
// of length Ls (zero padded like the row); each goes through the Ls-point real transform, unchanged, and with
// w = exp(-2 pi i / Px) and the half spectra S_q extended by S_q[Ls - j] = conj S_q[j]:
//   forward:  X[k] = sum_q w^(q k) S_q[k mod Ls],  k <= Px / 2
//   inverse:  S'_q[j] = sum_m conj(w^(q (j + Ls m))) X[j + Ls m],  j <= Ls / 2,  X[Px - k] = conj X[k]
// ---------------------------------------------------------------------------------------------
namespace ff {
__global__ void k_x_deinterleave(const float* __restrict__ m, float* __restrict__ tmp, size_t nrow, int Nx, int R)
{
    const int sub = Nx / R;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nrow * Nx; i += (size_t)gridDim.x * blockDim.x) {
        const size_t row = i / Nx;
        const int x = (int)(i - row * Nx), n = x / R, q = x - n * R;
        tmp[(row * R + q) * sub + n] = m[i];
    }
}
__global__ void k_x_interleave(const float* __restrict__ tmp, float* __restrict__ out, size_t nrow, int Nx, int R)
{
    const int sub = Nx / R;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nrow * Nx; i += (size_t)gridDim.x * blockDim.x) {
        const size_t row = i / Nx;
        const int x = (int)(i - row * Nx), n = x / R, q = x - n * R;
        out[i] = tmp[(row * R + q) * sub + n];
    }
}
// forward: one thread per (row, k <= P/2)
template <int R>
__global__ void k_x_combine_fwd(const float2* __restrict__ ts, float2* __restrict__ specA, size_t nrow, int CxS,
                                int Ls, int S, int P, const float2* __restrict__ twl)
{
    const int k = blockIdx.y * blockDim.x + threadIdx.x;
    const size_t row = blockIdx.x;
    if (k > P / 2 || row >= nrow) return;
    const int j = k % Ls;
    const bool mir = 2 * j > Ls;
    const int jj = mir ? Ls - j : j;
    float2 acc = make_float2(0.f, 0.f);
#pragma unroll
    for (int q = 0; q < R; ++q) {
        float2 v = ts[(row * R + q) * S + jj];
        if (mir) v.y = -v.y;
        const float2 w = __ldg(twl + (int)(((long long)q * k) % P));
        acc.x = fmaf(w.x, v.x, fmaf(-w.y, v.y, acc.x));
        acc.y = fmaf(w.x, v.y, fmaf(w.y, v.x, acc.y));
    }
    specA[row * CxS + k] = acc;
}
// inverse: one thread per (row, q, j <= Ls/2)
template <int R>
__global__ void k_x_combine_inv(float2* __restrict__ ts, const float2* __restrict__ specA, size_t nrow, int CxS,
                                int Ls, int S, int P, const float2* __restrict__ twl)
{
    const int j = blockIdx.y * blockDim.x + threadIdx.x;
    const size_t rq = blockIdx.x;                 // row * R + q
    if (j > Ls / 2 || rq >= nrow * R) return;
    const size_t row = rq / R;
    const int q = (int)(rq - row * R);
    const float2* __restrict__ x = specA + row * CxS;
    float2 acc = make_float2(0.f, 0.f);
#pragma unroll
    for (int m = 0; m < R; ++m) {
        const int k = j + m * Ls;
        float2 v = 2 * k > P ? cconj(x[P - k]) : x[k];
        float2 w = __ldg(twl + (int)(((long long)q * k) % P));
        w.y = -w.y;
        acc.x = fmaf(w.x, v.x, fmaf(-w.y, v.y, acc.x));
        acc.y = fmaf(w.x, v.y, fmaf(w.y, v.x, acc.y));
    }
    ts[rq * S + j] = acc;
}
}  // namespace ff

// the Px-point real transform of every row by a kernel that takes Px itself (tables of fp are those of g.Px)
static bool fwd_x_direct(const FastPlan& fp, const Geom& g, cudaStream_t st, const float* m, float2* specA)
{
    int T, E;
    if (!ff::split(g.Px, &T, &E)) {
        if (g.Px == 1536) return g.perx ? ff::launch_fwd_x_r<16, 48, true>(fp, g, st, m, specA)
                                        : ff::launch_fwd_x_r<16, 48, false>(fp, g, st, m, specA);
        if (g.Px == 2048) return g.perx ? ff::launch_fwd_x_r<32, 32, true>(fp, g, st, m, specA)
                                        : ff::launch_fwd_x_r<32, 32, false>(fp, g, st, m, specA);
        return false;
    }
    bool r = false;
#define CALL(T, E) r = g.perx ? ff::launch_fwd_x<T, E, true>(fp, g, st, m, specA) \
                              : ff::launch_fwd_x<T, E, false>(fp, g, st, m, specA)
    MM_FF_SIZES(g.Px, CALL)
#undef CALL
    return r;
}

static bool inv_x_direct(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, float* out, float scale)
{
    int T, E;
    if (!ff::split(g.Px, &T, &E)) {
        if (g.Px == 1536) return g.perx ? ff::launch_inv_x_h_r<16, 48, true>(fp, g, st, specA, out, scale)
                                        : ff::launch_inv_x_h_r<16, 48, false>(fp, g, st, specA, out, scale);
        if (g.Px == 2048) return g.perx ? ff::launch_inv_x_h_r<32, 32, true>(fp, g, st, specA, out, scale)
                                        : ff::launch_inv_x_h_r<32, 32, false>(fp, g, st, specA, out, scale);
        return false;
    }
    bool r = false;
#define CALL(T, E) r = g.perx ? ff::launch_inv_x_h<T, E, true>(fp, g, st, specA, out, scale) \
                              : ff::launch_inv_x_h<T, E, false>(fp, g, st, specA, out, scale)
    MM_FF_SIZES(g.Px, CALL)
#undef CALL
    return r;
}

// geometry of the R sub-rows per row: a field of R Ny rows of Nx / R cells, padded length Ls
static Geom x_sub_geom(const FastPlan& fp, const Geom& g)
{
    Geom h = g;
    h.Nx = g.Nx / fp.x_R; h.Ny = fp.x_R * g.Ny; h.Px = fp.x_Ls; h.Cx = h.Px / 2 + 1; h.CxS = fp.xs_stride;
    return h;
}

bool fast_fwd_x(const FastPlan& fp, const Geom& g, cudaStream_t st, const float* m, float2* specA)
{
    if (fp.x_R > 1) {
        const size_t nrow = (size_t)3 * g.Nz * g.Ny;
        ff::k_x_deinterleave<<<fp.nsm * 8, 256, 0, st>>>(m, fp.xs_real, nrow, g.Nx, fp.x_R);
        if (!fwd_x_direct(fp, x_sub_geom(fp, g), st, fp.xs_real, fp.xs_spec)) return false;
        dim3 cg((unsigned)nrow, (g.Px / 2 + 1 + 127) / 128);
#define XC(RR) case RR: ff::k_x_combine_fwd<RR><<<cg, 128, 0, st>>>(fp.xs_spec, specA, nrow, g.CxS, fp.x_Ls, fp.xs_stride, g.Px, fp.twxl); break
        switch (fp.x_R) { XC(2); XC(3); XC(4); XC(5); XC(7); XC(9); default: return false; }
#undef XC
        return true;
    }
    if (!(fp.ok_x || fp.ok_xr)) return false;
    return fwd_x_direct(fp, g, st, m, specA);
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
bool fast_inv_x_h(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, float* out, float scale)
{
    if (fp.x_R > 1) {
        const size_t nrow = (size_t)3 * g.Nz * g.Ny;
        dim3 cg((unsigned)(nrow * fp.x_R), (fp.x_Ls / 2 + 1 + 127) / 128);
#define XC(RR) case RR: ff::k_x_combine_inv<RR><<<cg, 128, 0, st>>>(fp.xs_spec, specA, nrow, g.CxS, fp.x_Ls, fp.xs_stride, g.Px, fp.twxl); break
        switch (fp.x_R) { XC(2); XC(3); XC(4); XC(5); XC(7); XC(9); default: return false; }
#undef XC
        if (!inv_x_direct(fp, x_sub_geom(fp, g), st, fp.xs_spec, fp.xs_real, scale)) return false;
        ff::k_x_interleave<<<fp.nsm * 8, 256, 0, st>>>(fp.xs_real, out, nrow, g.Nx, fp.x_R);
        return true;
    }
    if (!(fp.ok_x || fp.ok_xr)) return false;
    return inv_x_direct(fp, g, st, specA, out, scale);
}

}  // namespace mm
