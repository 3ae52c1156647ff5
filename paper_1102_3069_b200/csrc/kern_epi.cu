// kern_epi.cu -- the per-cell tail a6-a10 as streaming kernels of their own (split last pass) and their launches.
// Product code; shares nothing with oracle/.
#include "mm_kernels.h"
#include "epilogue.cuh"

namespace mm {

// a6-a10 as a streaming kernel, one thread per cell (any Nx; staircase geometry, reading A15): the per-cell
// tail of the generic path on the H_ms field the inverse x pass has left.
__global__ void __launch_bounds__(256)
k_epi1(Geom g, const float* __restrict__ hms, EpiParams ep)
{
    const size_t n = (size_t)g.Nx * g.Ny * g.Nz;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned int red = 0u;
    if (i < n) {
        const int x = (int)(i % g.Nx);
        const size_t yz = i / g.Nx;
        const int y = (int)(yz % g.Ny), z = (int)(yz / g.Ny);
        red = __float_as_uint(epilogue_cell(g, ep, x, y, z, hms[i], hms[i + n], hms[i + 2 * n])) & 0x7fffffffu;
    }
    if (ep.do_err) block_max_atomic(red, ep.maxbits);
}

// ---------------------------------------------------------------------------------------------
// a6-a10 as a streaming kernel of their own (the "split" variant of the last pass): the inverse x
// pass has left H_ms (units of Ms) in `hms`, laid out like a field; each thread owns 4 consecutive
// cells along x (float4 traffic), takes its x neighbours from the adjacent lanes and the y / z
// neighbours from the rows above and below.  Needs Nx % 4 == 0.  One quad per thread.
// ---------------------------------------------------------------------------------------------
#ifndef MM_EPI4_MINB
#define MM_EPI4_MINB 3
#endif
template <bool LEAN, int NA>
__global__ void __launch_bounds__(256, MM_EPI4_MINB)
k_epi4(Geom g, const float* __restrict__ hms, EpiParams ep)
{
    const int nx4 = g.Nx >> 2;
    const size_t total = (size_t)nx4 * g.Ny * g.Nz;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool active = i < total;
    if (!active) i = total - 1;
    const int x4 = (int)(i % nx4);
    const size_t yz = i / nx4;
    const int y = (int)(yz % g.Ny), z = (int)(yz / g.Ny);
    const int x = x4 << 2;
    const size_t plane = (size_t)g.Ny * g.Nx;
    const size_t n = plane * g.Nz;
    const size_t rowc = (size_t)z * plane + (size_t)y * g.Nx;
    const size_t idx = rowc + x;
    const float* __restrict__ mi = ep.m_in;
    const unsigned lane = threadIdx.x & 31;
    float m[3][4], h[3][4], D[3][4];
#pragma unroll
    for (int c = 0; c < 3; ++c) ldv<4>(mi + idx + c * n, m[c]);
    // x neighbours of the quad's end cells: adjacent lanes hold them unless the lane is at a warp or row end
    float xl[3], xr[3];
    {
        const bool lsh = lane > 0 && x4 > 0, rsh = lane < 31 && x4 + 1 < nx4;
        const int xli = x > 0 ? x - 1 : (g.perx ? g.Nx - 1 : x);
        const int xri = x + 4 < g.Nx ? x + 4 : (g.perx ? 0 : x + 3);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float up = __shfl_up_sync(0xffffffffu, m[c][3], 1);
            const float dn = __shfl_down_sync(0xffffffffu, m[c][0], 1);
            xl[c] = lsh ? up : mi[rowc + xli + c * n];
            xr[c] = rsh ? dn : mi[rowc + xri + c * n];
        }
    }
    unsigned int red = 0u;
    // no neighbour is needed when the exchange rides on the convolution kernel and no current flows
    const bool need_nb = ep.wex[0] != 0.f || ep.wex[1] != 0.f || ep.wex[2] != 0.f || ep.stt;
    if (active && !need_nb) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            ldv<4>(hms + idx + c * n, h[c]);
#pragma unroll
            for (int u = 0; u < 4; ++u) if (!LEAN) D[c][u] = 0.f;
        }
        red = __float_as_uint(epilogue_finish_v<4, LEAN, NA>(ep, idx, n, m, h, D)) & 0x7fffffffu;
    } else if (active) {
        const int ym = y > 0 ? y - 1 : (g.pery ? g.Ny - 1 : y);
        const int yp = y + 1 < g.Ny ? y + 1 : (g.pery ? 0 : y);
        const int zm = z > 0 ? z - 1 : (g.perz ? g.Nz - 1 : z);
        const int zp = z + 1 < g.Nz ? z + 1 : (g.perz ? 0 : z);
        const size_t iym = (size_t)z * plane + (size_t)ym * g.Nx + x, iyp = (size_t)z * plane + (size_t)yp * g.Nx + x;
        const size_t izm = (size_t)zm * plane + (size_t)y * g.Nx + x, izp = (size_t)zp * plane + (size_t)y * g.Nx + x;
        // slab decomposition: the planes below the first and above the last local plane come from the neighbours
        const bool lo_h = ep.zlo != nullptr && z == 0, hi_h = ep.zhi != nullptr && z == g.Nz - 1;
        const float* __restrict__ pzm = lo_h ? ep.zlo + (size_t)y * g.Nx + x : mi + izm;
        const float* __restrict__ pzp = hi_h ? ep.zhi + (size_t)y * g.Nx + x : mi + izp;
        const size_t szm = lo_h ? plane : n, szp = hi_h ? plane : n;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            float a[4], b[4], d[4], e[4];
            ldv<4>(hms + idx + c * n, h[c]);
            ldv<4>(mi + iym + c * n, a);
            ldv<4>(mi + iyp + c * n, b);
            ldv<4>(pzm + c * szm, d);
            ldv<4>(pzp + c * szp, e);
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const float mc = m[c][u];
                const float xm = u > 0 ? m[c][u > 0 ? u - 1 : 0] : xl[c];
                const float xp = u < 3 ? m[c][u < 3 ? u + 1 : 3] : xr[c];
                h[c][u] += ep.wex[0] * ((xp - mc) + (xm - mc));
                h[c][u] += ep.wex[1] * ((b[u] - mc) + (a[u] - mc));
                h[c][u] += ep.wex[2] * ((e[u] - mc) + (d[u] - mc));
                if (!LEAN) D[c][u] = ep.cj[0] * (xp - xm) + ep.cj[1] * (b[u] - a[u]) + ep.cj[2] * (e[u] - d[u]);
            }
        }
        red = __float_as_uint(epilogue_finish_v<4, LEAN, NA>(ep, idx, n, m, h, D)) & 0x7fffffffu;
    }
    if (ep.do_err) block_max_atomic(red, ep.maxbits);
}


void launch_epi4(const Geom& g, const float* hms, const EpiParams& ep, cudaStream_t st)
{
    const size_t quads = (size_t)g.Nx * g.Ny * g.Nz / 4;
    // the common case (no cubic anisotropy, thermal field, current, per-film field) has leaner instantiations, with
    // the number of earlier stage derivatives fixed for the usual stage shapes (RK4: 0, 0, 0, 3; Dormand-Prince: 0 ... 4)
    const unsigned nb = (unsigned)((quads + 255) / 256);
    const bool lean = !ep.cubic && !ep.thermal && !ep.stt && !ep.hext_b;
    const int na = (ep.mode == EPI_STAGE && ep.m_out) ? ep.na : 0;
    if (lean && na == 0) k_epi4<true, 0><<<nb, 256, 0, st>>>(g, hms, ep);
    else if (lean && na == 1) k_epi4<true, 1><<<nb, 256, 0, st>>>(g, hms, ep);
    else if (lean && na == 2) k_epi4<true, 2><<<nb, 256, 0, st>>>(g, hms, ep);
    else if (lean && na == 3) k_epi4<true, 3><<<nb, 256, 0, st>>>(g, hms, ep);
    else if (lean && na == 4) k_epi4<true, 4><<<nb, 256, 0, st>>>(g, hms, ep);
    else if (lean) k_epi4<true, -1><<<nb, 256, 0, st>>>(g, hms, ep);
    else k_epi4<false, -1><<<nb, 256, 0, st>>>(g, hms, ep);
}

void launch_epi1(const Geom& g, const float* hms, const EpiParams& ep, cudaStream_t st)
{
    const size_t n = (size_t)g.Nx * g.Ny * g.Nz;
    k_epi1<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(g, hms, ep);
}

}  // namespace mm
