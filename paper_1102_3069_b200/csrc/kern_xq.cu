// kern_xq.cu -- the last pass in one kernel (a5-a10): inverse x transform and per-cell tail of a row pair in one
// block (ff::k_inv_x_q), its launch and instantiations.  Product code; shares nothing with oracle/.
#include <string>
#include <vector>
#include "mm_kernels.h"
#include "epilogue.cuh"
#include "fft_fast.cuh"
#include "fft_packed.cuh"

namespace mm {
namespace ff {
// ---------------------------------------------------------------------------------------------
// a5-a10 in one kernel, second form (lines of T = 32 or 16 threads): a block of four warps owns 32 / T pairs of rows
// (y0, y0+1) of z planes.  Warps 0-2 run the inverse transforms of one component each (one line per T lanes) exactly
// as k_inv_x_h does and leave H_ms in a shared tile [pair][3][2][Nx]; after a block barrier all 128 threads run the
// per-cell tail on the pairs' quads exactly as k_epi4 does (float4 traffic for m, its neighbours and the Runge-Kutta
// buffers), with H_ms read from the tile instead of from HBM: the 2 x 12 N bytes of the two-kernel form's H_ms
// round trip are gone.  Needs Nx % 128 == 0 (a warp's 32 quads lie in one row).  Measured at 512 x 512 x 64:
// 0.264 ms against 0.297 ms for k_inv_x_h + k_epi4; three warps per block (2.67 quads per thread) 0.288 ms; spectrum
// rows staged by cp.async during the tail 0.30-0.32 ms; the idle fourth warp prefetching the tail's rows into L2:
// no difference.
// ---------------------------------------------------------------------------------------------
#ifndef MM_Q_MINB
#define MM_Q_MINB 4
#endif
template <int T, int E, bool PER, bool LEAN, int NA>
__global__ void __launch_bounds__(128, MM_Q_MINB)
k_inv_x_q(Geom g, const float2* __restrict__ specA, const float2* __restrict__ tw, EpiParams ep)
{
    static_assert(T == 32 || T == 16, "whole lines per warp");
    constexpr int L = T * E;
    constexpr int LB = T * (E + 1);
    constexpr int NX = PER ? L : L / 2;        // == g.Nx
    constexpr int NOUT = PER ? E : E / 2;
    constexpr int LPW = 32 / T;                // lines per warp = row pairs per block
    const int t = threadIdx.x % T;
    const int sub = (threadIdx.x & 31) / T;    // which of the block's row pairs this lane group transforms
    const int comp = threadIdx.x >> 5;
    float2* sb = ff_smem + (comp * LPW + sub) * LB;
    const int npy = (g.Ny + 1) >> 1;
    const int npair = g.Nz * npy;
    const int ngroup = (npair + LPW - 1) / LPW;
    float* hb = reinterpret_cast<float*>(ff_smem + 3 * LPW * LB);     // [LPW][3][2][NX]
    // the two spectrum rows of a line arrive in the line's exchange buffer by one bulk copy each (issued by lane t = 0
    // of the line once the exchange of the previous pair has been read back, i.e. during the per-cell tail)
    constexpr int CXP = L / 2 + 2;              // second staged row starts 16-byte aligned
    constexpr unsigned ROWB = ((L / 2 + 1) * 8 + 15) & ~15u;        // bytes of a row, whole 16-byte units
    static_assert(2 * CXP <= LB && CXP * 8 >= ROWB, "staged rows must fit the exchange buffer");
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(hb + LPW * 6 * NX);
    unsigned long long* bar = bars + (comp < 3 ? comp * LPW + sub : 0);
    auto issue = [&](int gq) {                  // lane t == 0 of an FFT line
        const int pq = gq * LPW + sub;
        const int pp = pq < npair ? pq : npair - 1;
        const int zq = pp / npy, yq = 2 * (pp - zq * npy);
        const bool twoq = yq + 1 < g.Ny;
        const float2* a0 = specA + (((size_t)comp * g.Nz + zq) * g.Ny + yq) * g.CxS;
        pk::fence_proxy_async_smem();
        pk::mbar_expect_tx(bar, twoq ? 2 * ROWB : ROWB);
        pk::bulk_load_1d(sb, a0, ROWB, bar);
        if (twoq) pk::bulk_load_1d(sb + CXP, a0 + g.CxS, ROWB, bar);
    };
    const unsigned srcl = (threadIdx.x & 31 & ~(T - 1)) + (T - t) % T;
    unsigned int red = 0u;
    if (threadIdx.x < 3 * LPW) pk::mbar_init(bars + threadIdx.x, 1);
    if (threadIdx.x == 0) pk::mbar_fence_init();
    __syncthreads();
    if (comp < 3 && t == 0 && (int)blockIdx.x < ngroup) issue(blockIdx.x);
    unsigned par = 0;
    for (int gi = blockIdx.x; gi < ngroup; gi += gridDim.x) {
        if (comp < 3) {
            const int pq = gi * LPW + sub;
            const int pp = pq < npair ? pq : npair - 1;         // a ragged last group repeats the last pair (not used)
            const int z = pp / npy, y0 = 2 * (pp - z * npy);
            const bool two = y0 + 1 < g.Ny;
            pk::mbar_wait(bar, par);            // this pair's rows have landed
            par ^= 1u;
            float2 v[E];
#pragma unroll
            for (int j = 0; j < E / 2; ++j) {
                const float2 A = sb[t + T * j];
                const float2 B = two ? sb[CXP + t + T * j] : make_float2(0.f, 0.f);
                v[j] = make_float2(A.x - B.y, A.y + B.x);
                v[E - 1 - j] = make_float2(A.x + B.y, B.x - A.y);
            }
            float2 nyq = make_float2(0.f, 0.f);
            if (t == 0) {
                const float2 A = sb[L / 2];
                const float2 B = two ? sb[CXP + L / 2] : make_float2(0.f, 0.f);
                nyq = make_float2(A.x - B.y, A.y + B.x);
            }
            float2 own[E / 2];
#pragma unroll
            for (int j = 0; j < E / 2; ++j) own[j] = v[E - 1 - j];
#pragma unroll
            for (int j = E / 2; j < E; ++j) {
                float2 p;
                p.x = __shfl_sync(0xffffffffu, v[j].x, srcl);
                p.y = __shfl_sync(0xffffffffu, v[j].y, srcl);
                v[j] = p;
            }
            if (t == 0) {
                v[E / 2] = nyq;
#pragma unroll
                for (int j = E / 2 + 1; j < E; ++j) v[j] = own[E - j];
            }
            __syncwarp();                       // the staged rows are in registers: the region is the exchange buffer
            fft_reg<E, 1>(v);
#pragma unroll
            for (int k2 = 1; k2 < E; ++k2) v[k2] = cmul(v[k2], cconj(__ldg(tw + k2 * T + t)));
#pragma unroll
            for (int k2 = 0; k2 < E; ++k2) sb[t * (E + 1) + k2] = v[k2];
            __syncwarp();
#pragma unroll
            for (int q = 0; q < E / T; ++q) {
                float2 u[T];
#pragma unroll
                for (int n1 = 0; n1 < T; ++n1) u[n1] = sb[n1 * (E + 1) + t + T * q];
                fft_reg<T, 1>(u);
#pragma unroll
                for (int k1 = 0; k1 < T; ++k1) v[q + (E / T) * k1] = u[k1];
            }
            __syncwarp();                       // exchange read back: the next pair's rows may land
            if (t == 0 && gi + (int)gridDim.x < ngroup) issue(gi + gridDim.x);
            float* __restrict__ h0 = hb + (sub * 3 + comp) * 2 * NX;
#pragma unroll
            for (int j = 0; j < NOUT; ++j) {
                h0[t + T * j] = v[j].x;
                h0[NX + t + T * j] = v[j].y;
            }
        }
        __syncthreads();                        // H_ms of the three components is in the tile
        constexpr int NQ = NX / 4;              // quads per row (a multiple of 32: every warp stays in one row)
#pragma unroll 1
        for (int q = threadIdx.x; q < LPW * 2 * NQ; q += 128) {
            const int s = q / (2 * NQ), r = q - s * 2 * NQ;
            const int row = r / NQ, x4 = r - row * NQ;
            const int pq = gi * LPW + s;
            if (pq >= npair) continue;
            const int z = pq / npy, y0 = 2 * (pq - z * npy);
            if (y0 + row >= g.Ny) continue;
            const float* __restrict__ hq = hb + (s * 6 + row) * NX + 4 * x4;
            red = max(red, epilogue_quad<LEAN, NA>(g, ep, x4, y0 + row, z,
                                                   [&](int c, float (&hv)[4]) { ldv<4>(hq + c * 2 * NX, hv); }));
        }
        __syncthreads();                        // the tile is free for the next pairs
    }
    if (ep.do_err) block_max_atomic(red, ep.maxbits);
}

// one-kernel last pass (k_inv_x_q): x lines of T = 32 or 16 threads
template <int T, int E, bool PER, bool LEAN, int NA>
bool launch_inv_x_q(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, const EpiParams& ep)
{
    constexpr int NX = PER ? T * E : T * E / 2;
    constexpr int LPW = 32 / T;
    const size_t bytes = (size_t)3 * LPW * T * (E + 1) * sizeof(float2) + (size_t)LPW * 6 * NX * sizeof(float) + 64;
    static bool once[MM_MAX_DEV] = {};
    if (!ensure_smem_dev(k_inv_x_q<T, E, PER, LEAN, NA>, bytes, once)) return false;
    const int npair = g.Nz * ((g.Ny + 1) / 2);
    const int ngroup = (npair + LPW - 1) / LPW;
    int per_sm = (int)((227 * 1024) / (bytes + 1024));
    if (per_sm > fp.q_blocks) per_sm = fp.q_blocks;
    const int grid = ngroup < fp.nsm * per_sm ? ngroup : fp.nsm * per_sm;
    k_inv_x_q<T, E, PER, LEAN, NA><<<grid, 128, bytes, st>>>(g, specA, fp.tw[0], ep);
    return true;
}

template <bool LEAN, int NA>
bool launch_inv_x_q_size(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, const EpiParams& ep)
{
#define CALLQ(T, E) return g.perx ? launch_inv_x_q<T, E, true, LEAN, NA>(fp, g, st, specA, ep) \
                                  : launch_inv_x_q<T, E, false, LEAN, NA>(fp, g, st, specA, ep)
    switch (g.Px) {
    case 1024: CALLQ(32, 32);
    case 512: CALLQ(16, 32);
    case 256: CALLQ(16, 16);
    default: break;
    }
#undef CALLQ
    return false;
}
}  // namespace ff

// a5-a10 fused, quad form; false: not for this grid / mode (the caller takes the split variant)
bool fast_inv_x_q(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, const EpiParams& ep)
{
    if (!fast_inv_x_q_ok(fp, g, ep)) return false;
    const bool lean = !ep.cubic && !ep.thermal && !ep.stt && !ep.hext_b;
    const int na = (ep.mode == EPI_STAGE && ep.m_out) ? ep.na : 0;
#define CALLQ(LEAN, NA) return ff::launch_inv_x_q_size<LEAN, NA>(fp, g, st, specA, ep)
    // the same instantiations as launch_epi4, so that both variants of the last pass give the same bits
    if (lean && na == 0) CALLQ(true, 0);
    if (lean && na == 1) CALLQ(true, 1);
    if (lean && na == 2) CALLQ(true, 2);
    if (lean && na == 3) CALLQ(true, 3);
    if (lean && na == 4) CALLQ(true, 4);
    if (lean) CALLQ(true, -1);
    CALLQ(false, -1);
#undef CALLQ
}

}  // namespace mm
