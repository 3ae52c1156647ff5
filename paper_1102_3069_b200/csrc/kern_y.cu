// kern_y.cu -- y passes (a2, a4): size-specialised kernel, long lines, launches and size dispatch.
// Product code; shares nothing with oracle/.
#include <string>
#include <vector>
#include "mm_kernels.h"
#include "fft_fast.cuh"

namespace mm {
namespace ff {
template <int T, int E, int SGN, bool PER>
bool launch_y(const FastPlan& fp, const Geom& g, cudaStream_t st, const ColTile& ct, float2* a, float2* b)
{
    const size_t bytes = (size_t)T * (E + 1) * 8 * sizeof(float2);
    static bool oncep[MM_MAX_DEV] = {};
    if (!ensure_smem_dev(k_y_p<T, E, SGN, PER>, bytes, oncep)) return false;
    const int ntile = ((ct.ncol + 7) / 8) * 3 * g.Nz;
    int per_sm = (int)((227 * 1024) / (bytes + 1024));
    const int cap = 2048 / (8 * T) < ((T == 32) ? 2 : 8) ? 2048 / (8 * T) : ((T == 32) ? 2 : 8);
    if (per_sm > cap) per_sm = cap;
    if (per_sm < 1) per_sm = 1;
    const int grid = ntile < fp.nsm * per_sm ? ntile : fp.nsm * per_sm;
    k_y_p<T, E, SGN, PER><<<grid, 8 * T, bytes, st>>>(ct, 3 * g.Nz, a, b, fp.tw[1]);
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
// Long y lines (Py = R * 1024, R = 2 or 4; the paper's Table 1 goes to 1024^2 and 2048^2 cells):
// one decimation-in-time level outside the size-specialised kernel.  Rows n = R r + q form R interleaved
// sequences; each is transformed by the 1024-point kernel with a row stride of R (the ColTile strides carry it,
// the kernel is unchanged: a zero-padded line of Py has zero-padded sub-sequences of 1024), sub-spectrum S_q
// landing in rows q * 1024 + k of the spectrum.  k_y_combine then forms, in place and per (plane, k, column),
//   forward:  X[k + 1024 m] = sum_q w_R^(q m) (w_Py^(q k) S_q[k])
//   inverse:  Y_q[k] = w_Py^(-q k) sum_m w_R^(-q m) X[k + 1024 m]      (before the R inverse transforms)
// ---------------------------------------------------------------------------------------------
namespace ff {
template <int R, int SGN>
__global__ void __launch_bounds__(128)
k_y_combine(ColTile ct, int nplane, int Ls, float2* __restrict__ b, const float2* __restrict__ twl)
{
    const int col = blockIdx.x * blockDim.x + threadIdx.x;
    const int k = blockIdx.y, cz = blockIdx.z;
    if (col >= ct.ncol || cz >= nplane) return;
    float2* p = b + (size_t)cz * ct.b_plane + (size_t)k * ct.b_row + col;
    const size_t rs = (size_t)Ls * ct.b_row;
    float2 v[R];
#pragma unroll
    for (int q = 0; q < R; ++q) v[q] = p[q * rs];
    auto tw = [&](int q) {                       // w_Py^(q k), conjugated for the inverse
        float2 w = __ldg(twl + q * k);
        if (SGN > 0) w.y = -w.y;
        return w;
    };
    if (SGN < 0) {
#pragma unroll
        for (int q = 1; q < R; ++q) v[q] = cmul(v[q], tw(q));
    }
    if constexpr (R == 2) {
        const float2 a0 = cadd(v[0], v[1]), a1 = csub(v[0], v[1]);
        v[0] = a0; v[1] = a1;
    } else {
        const float2 s02 = cadd(v[0], v[2]), d02 = csub(v[0], v[2]);
        const float2 s13 = cadd(v[1], v[3]), d13 = cmuli<SGN>(csub(v[1], v[3]));
        v[0] = cadd(s02, s13); v[2] = csub(s02, s13);
        v[1] = cadd(d02, d13); v[3] = csub(d02, d13);
    }
    if (SGN > 0) {
#pragma unroll
        for (int q = 1; q < R; ++q) v[q] = cmul(v[q], tw(q));
    }
#pragma unroll
    for (int q = 0; q < R; ++q) p[q * rs] = v[q];
}
}  // namespace ff

template <int R>
bool fast_y_long(const FastPlan& fp, const Geom& g, cudaStream_t st, int sgn, const ff::ColTile& ct, float2* a,
                        float2* b)
{
    constexpr int Ls = 1024;
    const int nplane = 3 * g.Nz;
    dim3 cg((ct.ncol + 127) / 128, Ls, nplane);
    if (sgn > 0) ff::k_y_combine<R, 1><<<cg, 128, 0, st>>>(ct, nplane, Ls, b, fp.twl);
    for (int q = 0; q < R; ++q) {
        ff::ColTile cq = ct;
        cq.a_row = ct.a_row * R;
        float2* aq = a + (size_t)q * ct.a_row;
        float2* bq = b + (size_t)q * Ls * ct.b_row;
        const bool ok = sgn < 0 ? (g.pery ? ff::launch_y<32, 32, -1, true>(fp, g, st, cq, aq, bq)
                                          : ff::launch_y<32, 32, -1, false>(fp, g, st, cq, aq, bq))
                                : (g.pery ? ff::launch_y<32, 32, 1, true>(fp, g, st, cq, aq, bq)
                                          : ff::launch_y<32, 32, 1, false>(fp, g, st, cq, aq, bq));
        if (!ok) return false;
    }
    if (sgn < 0) ff::k_y_combine<R, -1><<<cg, 128, 0, st>>>(ct, nplane, Ls, b, fp.twl);
    return true;
}

// sgn < 0: specA rows y < Ny -> specB rows ky < Py; sgn > 0: back.  a, b point at column ct.kx0.
bool fast_y(const FastPlan& fp, const Geom& g, cudaStream_t st, int sgn, const ff::ColTile& ct, float2* a,
                   float2* b)
{
    if (!fp.ok_y) return false;
    if (fp.y_split == 2) return fast_y_long<2>(fp, g, st, sgn, ct, a, b);
    if (fp.y_split == 4) return fast_y_long<4>(fp, g, st, sgn, ct, a, b);
    bool r = false;
#define CALL(T, E)                                                                         \
    r = sgn < 0 ? (g.pery ? ff::launch_y<T, E, -1, true>(fp, g, st, ct, a, b)              \
                          : ff::launch_y<T, E, -1, false>(fp, g, st, ct, a, b))            \
                : (g.pery ? ff::launch_y<T, E, 1, true>(fp, g, st, ct, a, b)               \
                          : ff::launch_y<T, E, 1, false>(fp, g, st, ct, a, b))
    MM_FF_SIZES(g.Py, CALL)
#undef CALL
    return r;
}


}  // namespace mm
