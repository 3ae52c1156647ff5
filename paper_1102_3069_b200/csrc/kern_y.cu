// kern_y.cu -- y passes (a2, a4): size-specialised kernel, long lines, launches and size dispatch.
// Product code; shares nothing with oracle/.
#include <string>
#include <vector>
#include "mm_kernels.h"
#include "fft_fast.cuh"
#include "fft_packed.cuh"

namespace mm {
namespace ff {
// ---------------------------------------------------------------------------------------------
// a2 / a4 with the tile loaded by TMA (whole-array passes with specB in panels): k_y_p with its 16 cp.async
// per thread and tile replaced by ROWS / 256 cp.async.bulk.tensor issued by one thread (box 8 columns x 256 rows,
// landing as [rows][8] float2 exactly where k_y_p stages its tile); completion on an mbarrier.
//   forward: map = specA as (2 Cx floats, Ny, 3 Nz);  inverse: map = specB panels as (32 floats, Py, 3 Nz, panel).
// ---------------------------------------------------------------------------------------------
extern __shared__ __align__(128) unsigned char yt_smem[];

template <int T, int E, int SGN, bool PER, bool TST>
__global__ void __launch_bounds__(8 * T, (T == 32) ? 2 : 1)
k_y_t(const __grid_constant__ CUtensorMap map, const __grid_constant__ CUtensorMap map_o, ColTile ct, int nplane,
      float2* __restrict__ a, float2* __restrict__ b, const float2* __restrict__ tw)
{
    constexpr bool FWD = SGN < 0;
    constexpr int NIN = (FWD && !PER) ? E / 2 : E;
    constexpr int NOUT = (!FWD && !PER) ? E / 2 : E;
    constexpr int ROWS = NIN * T;
    constexpr int BR = ROWS < 256 ? ROWS : 256;         // rows per TMA box
    static_assert(ROWS % BR == 0, "tile rows in whole boxes");
    float2* sm = reinterpret_cast<float2*>(yt_smem);
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(yt_smem + (size_t)T * (E + 1) * 8 * sizeof(float2));
    // TST: results leave through a staging tile of SB rows [SB][8] and TMA tile stores (map_o: the destination array)
    constexpr int SB = 16 * T;                  // 512 rows = the registers j .. j + 15 of every thread
    float2* ob = reinterpret_cast<float2*>(yt_smem + (size_t)T * (E + 1) * 8 * sizeof(float2) + 128);
    const int tid = threadIdx.x, c = tid & 7, t = tid >> 3;
    const int ntx = (ct.ncol + 7) >> 3;
    const int ntile = ntx * nplane;
    const size_t d_row = FWD ? ct.b_row : ct.a_row, d_plane = FWD ? ct.b_plane : ct.a_plane;
    float2* __restrict__ dst = FWD ? b : a;
    auto boff = [&](int bx) -> size_t { return (size_t)(bx >> 1) * ct.b_panel + (size_t)(bx & 1) * 8; };
    if (tid == 0) {
        pk::tma_prefetch_desc(&map);
        pk::mbar_init(bar, 1);
        pk::mbar_fence_init();
    }
    __syncthreads();
    auto issue = [&](int i) {                   // thread 0 only
        const int bx = i % ntx, cz = i / ntx;
        pk::mbar_expect_tx(bar, (unsigned)(ROWS * 8 * sizeof(float2)));
#pragma unroll
        for (int r0 = 0; r0 < ROWS; r0 += BR) {
            if (FWD) pk::tma_load_3d(sm + r0 * 8, &map, bar, 16 * bx, r0, cz);
            else pk::tma_load_4d(sm + r0 * 8, &map, bar, 16 * (bx & 1), r0, cz, bx >> 1);
        }
    };
    int i = blockIdx.x;
    if (tid == 0 && i < ntile) issue(i);
    unsigned par = 0;
    for (; i < ntile; i += gridDim.x) {
        const int bx = i % ntx, cz = i / ntx;
        const int col = bx * 8 + c;
        pk::mbar_wait(bar, par);                // this tile has landed
        par ^= 1u;
        float2 v[E];
#pragma unroll
        for (int j = 0; j < NIN; ++j) v[j] = sm[(t + T * j) * 8 + c];
        __syncthreads();                        // the region now serves as the exchange buffer
        if constexpr (FWD && !PER) fft_reg_half<E, SGN>(v);
        else fft_reg<E, SGN>(v);
        apply_twiddles<T, E, (SGN > 0)>(v, tw, t);
#pragma unroll
        for (int k2 = 0; k2 < E; ++k2) sm[(t * (E + 1) + k2) * 8 + c] = v[k2];
        __syncthreads();
        float2 u[E / T][T];
#pragma unroll
        for (int q = 0; q < E / T; ++q)
#pragma unroll
            for (int n1 = 0; n1 < T; ++n1) u[q][n1] = sm[(n1 * (E + 1) + t + T * q) * 8 + c];
        if (TST && tid == 0) pk::bulk_wait_read0();      // the staging tile has been read (stores of the previous tile)
        __syncthreads();                        // exchange read back: the region is free for the next tile
        if (tid == 0 && i + (int)gridDim.x < ntile) {
            pk::fence_proxy_async_smem();
            issue(i + gridDim.x);
        }
#pragma unroll
        for (int q = 0; q < E / T; ++q) {
            fft_reg<T, SGN>(u[q]);
#pragma unroll
            for (int k1 = 0; k1 < T; ++k1) v[q + (E / T) * k1] = u[q][k1];
        }
        if constexpr (TST) {
            static_assert(NOUT % 16 == 0, "whole staging chunks");
#pragma unroll
            for (int h = 0; h < NOUT / 16; ++h) {
                if (h > 0) {
                    if (tid == 0) pk::bulk_wait_read0();
                    __syncthreads();
                }
#pragma unroll
                for (int j = 0; j < 16; ++j) ob[(t + T * j) * 8 + c] = v[16 * h + j];
                pk::fence_proxy_async_smem();
                __syncthreads();
                if (tid == 0) {
#pragma unroll
                    for (int r0 = 0; r0 < SB; r0 += 256) {
                        if (FWD) pk::tma_store_4d(&map_o, ob + r0 * 8, 16 * (bx & 1), SB * h + r0, cz, bx >> 1);
                        else pk::tma_store_3d(&map_o, ob + r0 * 8, 16 * bx, SB * h + r0, cz);
                    }
                    pk::bulk_commit();
                }
            }
        } else if (col < ct.ncol) {
            float2* __restrict__ dp = dst + (size_t)cz * d_plane + (FWD ? boff(bx) + c : (size_t)col);
#pragma unroll
            for (int j = 0; j < NOUT; ++j) dp[(size_t)(t + T * j) * d_row] = v[j];
        }
    }
    if (TST && tid == 0) pk::bulk_wait_read0();         // shared memory must outlive the last store's read
}

template <int T, int E, int SGN, bool PER, bool TST>
bool launch_lines_t(const FastPlan& fp, cudaStream_t st, const ColTile& ct, int nplane, float2* a, float2* b,
                    const float2* tw)
{
    const size_t bytes = (size_t)T * (E + 1) * 8 * sizeof(float2) + 128 + (TST ? (size_t)16 * T * 8 * sizeof(float2) : 0);
    static bool once[MM_MAX_DEV] = {};
    if (!ensure_smem_dev(k_y_t<T, E, SGN, PER, TST>, bytes, once)) return false;
    const int ntile = ((ct.ncol + 7) / 8) * nplane;
    const int grid = ntile < fp.nsm * 2 ? ntile : fp.nsm * 2;
    k_y_t<T, E, SGN, PER, TST><<<grid, 8 * T, bytes, st>>>(SGN < 0 ? fp.map_ya : fp.map_yb, SGN < 0 ? fp.map_yb : fp.map_ya, ct,
                                                          nplane, a, b, tw);
    return true;
}

// lines along any strided axis: nplane planes, strides in the ColTile, twiddle table tw of the line length
template <int T, int E, int SGN, bool PER>
bool launch_lines(const FastPlan& fp, cudaStream_t st, const ColTile& ct, int nplane, float2* a, float2* b,
                  const float2* tw)
{
    if constexpr (T == 32 && E == 32) {
        // whole-array pass with specB in panels: tile loads by TMA (fp.y_tma; the maps describe exactly that case)
        if (fp.y_tma && fp.ok_ymaps && ct.b_panel && ct.kx0 == 0 && a == fp.y_a && b == fp.y_b)
            return (fp.y_tma >= 3 || (fp.y_tma == 2 && SGN < 0)) ? launch_lines_t<T, E, SGN, PER, true>(fp, st, ct, nplane, a, b, tw)
                                                                  : launch_lines_t<T, E, SGN, PER, false>(fp, st, ct, nplane, a, b, tw);
    }
    const size_t bytes = (size_t)T * (E + 1) * 8 * sizeof(float2);
    static bool oncep[MM_MAX_DEV] = {};
    if (!ensure_smem_dev(k_y_p<T, E, SGN, PER>, bytes, oncep)) return false;
    const int ntile = ((ct.ncol + 7) / 8) * nplane;
    int per_sm = (int)((227 * 1024) / (bytes + 1024));
    const int cap = 2048 / (8 * T) < ((T == 32) ? 2 : 8) ? 2048 / (8 * T) : ((T == 32) ? 2 : 8);
    if (per_sm > cap) per_sm = cap;
    if (per_sm < 1) per_sm = 1;
    const int grid = ntile < fp.nsm * per_sm ? ntile : fp.nsm * per_sm;
    k_y_p<T, E, SGN, PER><<<grid, 8 * T, bytes, st>>>(ct, nplane, a, b, tw);
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
// Lines whose length P has no kernel of its own but factors as P = R * Ls with Ls a size-specialised length and
// R in {2, 3, 4, 5, 7, 9} -- long lines (2048, 4096; the paper's Table 1 goes to 2048^2 cells) and
// the lengths 2^n * {5, 7, 9} of PAPER.md:171: one decimation-in-time level outside the kernel.  Rows n = R r + q form
// R interleaved sequences; each is transformed by the Ls-point kernel with a row stride of R (the ColTile strides
// carry it, the kernel is unchanged: a zero-padded line has zero-padded sub-sequences), sub-spectrum S_q landing in
// rows q * Ls + k.  k_lines_combine then forms, in place and per (plane, k, column), with w = exp(-2 pi i / P):
//   forward:  X[k + Ls m] = sum_q w^(q (k + Ls m)) S_q[k]
//   inverse:  Y_q[k] = sum_m conj(w^(q (k + Ls m))) X[k + Ls m]      (before the R inverse transforms)
// ---------------------------------------------------------------------------------------------
namespace ff {
template <int R, int SGN>
__global__ void __launch_bounds__(128)
k_lines_combine(ColTile ct, int nplane, int Ls, int P, float2* __restrict__ b, const float2* __restrict__ twl)
{
    __shared__ float2 W[R * R];                  // W[q * R + m] = w^(q (k + Ls m)), conjugated for the inverse
    const int k = blockIdx.y, cz = blockIdx.z;
    if ((int)threadIdx.x < R * R) {
        const int q = threadIdx.x / R, m = threadIdx.x - q * R;
        float2 w = __ldg(twl + (int)(((long long)q * (k + (long long)m * Ls)) % P));
        if (SGN > 0) w.y = -w.y;
        W[threadIdx.x] = w;
    }
    __syncthreads();
    const int col = blockIdx.x * blockDim.x + threadIdx.x;
    if (col >= ct.ncol || cz >= nplane) return;
    float2* p = b + (size_t)cz * ct.b_plane + (size_t)k * ct.b_row + col;
    const size_t rs = (size_t)Ls * ct.b_row;
    float2 v[R], o[R];
#pragma unroll
    for (int q = 0; q < R; ++q) v[q] = p[q * rs];
    if constexpr (R == 2 || R == 4) {
        // w^(q (k + Ls m)) = w^(q k) w_R^(q m): twiddle by w^(q k) = W[q * R] (m = 0), then a radix-R butterfly
        if (SGN < 0) {
#pragma unroll
            for (int q = 1; q < R; ++q) v[q] = cmul(v[q], W[q * R]);
        }
        if constexpr (R == 2) {
            o[0] = cadd(v[0], v[1]); o[1] = csub(v[0], v[1]);
        } else {
            const float2 s02 = cadd(v[0], v[2]), d02 = csub(v[0], v[2]);
            const float2 s13 = cadd(v[1], v[3]), d13 = cmuli<SGN>(csub(v[1], v[3]));
            o[0] = cadd(s02, s13); o[2] = csub(s02, s13);
            o[1] = cadd(d02, d13); o[3] = csub(d02, d13);
        }
        if (SGN > 0) {
#pragma unroll
            for (int q = 1; q < R; ++q) o[q] = cmul(o[q], W[q * R]);
        }
    } else {
#pragma unroll
        for (int u = 0; u < R; ++u) {
            float2 acc = make_float2(0.f, 0.f);
#pragma unroll
            for (int q = 0; q < R; ++q) {
                // forward: output m = u sums over q; inverse: output q = u sums over m
                const float2 w = SGN < 0 ? W[q * R + u] : W[u * R + q];
                acc.x = fmaf(w.x, v[q].x, fmaf(-w.y, v[q].y, acc.x));
                acc.y = fmaf(w.x, v[q].y, fmaf(w.y, v[q].x, acc.y));
            }
            o[u] = acc;
        }
    }
#pragma unroll
    for (int q = 0; q < R; ++q) p[q * rs] = o[q];
}

template <int SGN>
inline void launch_lines_combine(cudaStream_t st, dim3 cg, const ColTile& ct, int nplane, int R, int Ls, int P, float2* b,
                                 const float2* twl)
{
    switch (R) {
    case 2: k_lines_combine<2, SGN><<<cg, 128, 0, st>>>(ct, nplane, Ls, P, b, twl); break;
    case 3: k_lines_combine<3, SGN><<<cg, 128, 0, st>>>(ct, nplane, Ls, P, b, twl); break;
    case 4: k_lines_combine<4, SGN><<<cg, 128, 0, st>>>(ct, nplane, Ls, P, b, twl); break;
    case 5: k_lines_combine<5, SGN><<<cg, 128, 0, st>>>(ct, nplane, Ls, P, b, twl); break;
    case 7: k_lines_combine<7, SGN><<<cg, 128, 0, st>>>(ct, nplane, Ls, P, b, twl); break;
    case 9: k_lines_combine<9, SGN><<<cg, 128, 0, st>>>(ct, nplane, Ls, P, b, twl); break;
    default: break;
    }
}
}  // namespace ff

// lines of length P along a strided axis: directly, or as R interleaved transforms of Ls = P / R plus the combine
bool fast_lines(const FastPlan& fp, cudaStream_t st, int sgn, bool per, const ff::ColTile& ct, int nplane, float2* a,
                float2* b, int P, const AxisPlan& ap)
{
    auto sub = [&](int L, const ff::ColTile& c2, float2* a2, float2* b2) {
        bool r = false;
#define CALL(T, E)                                                                                   \
    r = sgn < 0 ? (per ? ff::launch_lines<T, E, -1, true>(fp, st, c2, nplane, a2, b2, ap.tw)          \
                       : ff::launch_lines<T, E, -1, false>(fp, st, c2, nplane, a2, b2, ap.tw))        \
                : (per ? ff::launch_lines<T, E, 1, true>(fp, st, c2, nplane, a2, b2, ap.tw)           \
                       : ff::launch_lines<T, E, 1, false>(fp, st, c2, nplane, a2, b2, ap.tw))
        MM_FF_SIZES(L, CALL)
#undef CALL
        return r;
    };
    if (ap.R <= 1) return sub(P, ct, a, b);
    const int R = ap.R, Ls = ap.Ls;
    dim3 cg((ct.ncol + 127) / 128, Ls, nplane);
    if (sgn > 0) ff::launch_lines_combine<1>(st, cg, ct, nplane, R, Ls, P, b, ap.twl);
    for (int q = 0; q < R; ++q) {
        ff::ColTile cq = ct;
        cq.a_row = ct.a_row * R;
        if (!sub(Ls, cq, a + (size_t)q * ct.a_row, b + (size_t)q * Ls * ct.b_row)) return false;
    }
    if (sgn < 0) ff::launch_lines_combine<-1>(st, cg, ct, nplane, R, Ls, P, b, ap.twl);
    return true;
}

// sgn < 0: specA rows y < Ny -> specB rows ky < Py; sgn > 0: back.  a, b point at column ct.kx0.
bool fast_y(const FastPlan& fp, const Geom& g, cudaStream_t st, int sgn, const ff::ColTile& ct, float2* a, float2* b)
{
    if (!fp.ok_y) return false;
    return fast_lines(fp, st, sgn, g.pery != 0, ct, 3 * g.Nz, a, b, g.Py, fp.ax[1]);
}

// ---------------------------------------------------------------------------------------------
// a3 for z lines that do not fit the fused last-axis kernels (padded z length 384, 512, 768, 1024: a thread cannot hold
// the line of all three components): the z pass unfused -- forward z transform of each component into a z-padded
// buffer [3][Pz][Py][CxS] by the y-pass kernel (a line is a line: the strides sit in the ColTile), the K-hat product
// as an elementwise kernel with the octant's mirror and sign rules, inverse z transform back into the Nz planes.
// More bytes than the fused kernels (the padded spectrum is materialised), but every pass at streaming speed.
// ---------------------------------------------------------------------------------------------
namespace ff {
__global__ void __launch_bounds__(128)
k_mul3d(Geom g, float2* __restrict__ spec, const float* __restrict__ khat)
{
    const int kx = blockIdx.x * blockDim.x + threadIdx.x;
    if (kx >= g.Cx) return;
    const int ky = blockIdx.y, kz = blockIdx.z;
    int qy = ky, qz = kz;
    float sy = 1.f, sz = 1.f;
    if (2 * qy > g.Py) { qy = g.Py - qy; sy = -1.f; }
    if (2 * qz > g.Pz) { qz = g.Pz - qz; sz = -1.f; }
    const size_t nC = (size_t)g.CxK * g.Cy * g.Cz;
    const size_t ko = ((size_t)qz * g.Cy + qy) * g.CxK + kx;
    const float kxx = __ldg(khat + ko), kyy = __ldg(khat + ko + nC), kzz = __ldg(khat + ko + 2 * nC);
    const float kxy = sy * __ldg(khat + ko + 3 * nC), kxz = sz * __ldg(khat + ko + 4 * nC);
    const float kyz = sy * sz * __ldg(khat + ko + 5 * nC);
    const size_t cs = (size_t)g.Pz * g.Py * g.CxS;
    float2* p = spec + ((size_t)kz * g.Py + ky) * g.CxS + kx;
    const float2 mx = p[0], my = p[cs], mz = p[2 * cs];
    p[0] = make_float2(kxx * mx.x + kxy * my.x + kxz * mz.x, kxx * mx.y + kxy * my.y + kxz * mz.y);
    p[cs] = make_float2(kxy * mx.x + kyy * my.x + kyz * mz.x, kxy * mx.y + kyy * my.y + kyz * mz.y);
    p[2 * cs] = make_float2(kxz * mx.x + kyz * my.x + kzz * mz.x, kxz * mx.y + kyz * my.y + kzz * mz.y);
}
}  // namespace ff

bool fast_z_long(const FastPlan& fp, const Geom& g, cudaStream_t st, float2* specB, const float* khat)
{
    if (!fp.z_long || !fp.zbuf) return false;
    ff::ColTile ct;
    ct.kx0 = 0; ct.ncol = g.Cx;
    ct.a_row = (size_t)g.Py * g.CxS; ct.a_plane = g.CxS;        // a "row" is a z plane, a "plane" a ky row
    ct.b_row = (size_t)g.Py * g.CxS; ct.b_plane = g.CxS;
    const size_t ca = (size_t)g.Nz * g.Py * g.CxS, cb = (size_t)g.Pz * g.Py * g.CxS;
    for (int sgn = -1; sgn <= 1; sgn += 2) {
        for (int comp = 0; comp < 3; ++comp)
            if (!fast_lines(fp, st, sgn, g.perz != 0, ct, g.Py, specB + comp * ca, fp.zbuf + comp * cb, g.Pz, fp.ax[2]))
                return false;
        if (sgn < 0) {
            dim3 grid((g.Cx + 127) / 128, g.Py, g.Pz);
            ff::k_mul3d<<<grid, 128, 0, st>>>(g, fp.zbuf, khat);
        }
    }
    return true;
}

}  // namespace mm
