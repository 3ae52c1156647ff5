// epilogue.cuh -- per-cell tail of one evaluation (steps a6-a10 of DESIGN.md): exchange stencil,
// anisotropy, Zeeman and thermal fields, Landau-Lifshitz torque with the Zhang-Li terms, the
// Runge-Kutta stage combine and the max-norm reduction.  Called by the inverse x pass with the
// magnetostatic field of the cell still in registers.
//
// Product code; shares nothing with oracle/.
#pragma once
#include "mm_common.cuh"

namespace mm {

// ---- Philox4x32-10 (reading A6: key = seed, counter = (cell lo, cell hi, step lo, step hi)) ----
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t out[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
        c0 = h1 ^ c1 ^ k0;
        c1 = l1;
        c2 = h0 ^ c3 ^ k1;
        c3 = l0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// -2 ln u for u = (x+1) 2^-32 without losing the resolution of u near 1 (reading A6)
__device__ __forceinline__ float neg2ln_u(uint32_t x)
{
    if (x >= 0x80000000u) {
        const float d = (float)(0xFFFFFFFFu - x) * 2.3283064365386963e-10f;   // 1 - u, exact scaling
        return -2.0f * log1pf(-d);
    }
    const float u = ((float)x + 1.0f) * 2.3283064365386963e-10f;
    return -2.0f * logf(u);
}

// three N(0,1) numbers of cell `cell` at step (step0, step1): Box-Muller on the four Philox words
__device__ __forceinline__ void thermal_eta(const EpiParams& p, uint64_t cell, float eta[3])
{
    uint32_t w[4];
    uint32_t st0 = p.step0, st1 = p.step1;
    if (p.step_dev) {
        const unsigned long long st = __ldg(p.step_dev);
        st0 = (uint32_t)st; st1 = (uint32_t)(st >> 32);
    }
    philox4x32_10((uint32_t)cell, (uint32_t)(cell >> 32), st0, st1, p.key0, p.key1, w);
    const float r1 = sqrtf(neg2ln_u(w[0]));
    const float r2 = sqrtf(neg2ln_u(w[2]));
    float s1, c1, s2, c2;
    // angle = 2 pi w 2^-32 = pi * (w 2^-31); w -> float keeps 24 bits (error <= 2 pi 2^-25 rad)
    sincospif((float)w[1] * 4.656612873077393e-10f, &s1, &c1);
    sincospif((float)w[3] * 4.656612873077393e-10f, &s2, &c2);
    eta[0] = r1 * c1;
    eta[1] = r1 * s1;
    eta[2] = r2 * c2;
}

__device__ __forceinline__ void cross3(const float a[3], const float b[3], float c[3])
{
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}

// V consecutive floats (V = 1 or 4; the address is 16-byte aligned when V = 4)
template <int V>
__device__ __forceinline__ void ldv(const float* __restrict__ p, float (&v)[V])
{
    if constexpr (V == 4) {
        const float4 t = *reinterpret_cast<const float4*>(p);
        v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
    } else {
#pragma unroll
        for (int u = 0; u < V; ++u) v[u] = p[u];
    }
}
template <int V>
__device__ __forceinline__ void stv(float* __restrict__ p, const float (&v)[V])
{
    if constexpr (V == 4) {
        *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
    } else {
#pragma unroll
        for (int u = 0; u < V; ++u) p[u] = v[u];
    }
}

// Tail of V consecutive cells (along x, first index idx) once their neighbours are known:
// m = the cells, h = H_ms + H_ex (units of Ms), D = (b_j j.grad) m in reduced units, all [3][V].
// Adds anisotropy, Zeeman and thermal fields, forms the torque, does the Runge-Kutta stage combine.
// All loads come before all stores.  Returns the value to be max-reduced (error norm or
// |dm/dtau|), 0 when no reduction is asked for.
// LEAN: no cubic anisotropy, thermal field, current or per-film field (the caller has checked): those branches and
// the gradient array D drop out at compile time, which is worth a dozen registers in the streaming kernel.
// NA >= 0: the number of earlier stage derivatives in the combine is known at compile time (their loads unroll and
// can be issued early); -1: taken from p.na.
template <int V, bool LEAN = false, int NA = -1>
__device__ __forceinline__ float epilogue_finish_v(const EpiParams& p, size_t idx, size_t n, const float (&m)[3][V],
                                                   float (&h)[3][V], const float (&D)[3][V])
{
    // ---- anisotropy (Eq. (4), reading A5), Zeeman ----
#pragma unroll
    for (int u = 0; u < V; ++u) {
        const float mu = m[0][u] * p.u[0] + m[1][u] * p.u[1] + m[2][u] * p.u[2];
        const float s = p.kan * mu;
#pragma unroll
        for (int c = 0; c < 3; ++c) h[c][u] += s * p.u[c] + p.hext[c];
    }
    if (!LEAN && p.hext_b) {      // one applied field per film of a batch (the V cells lie in one row, hence in one plane)
        const float* __restrict__ hb = p.hext_b + 3 * (idx / p.plane_cells);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float d = __ldg(hb + c) - p.hext[c];
#pragma unroll
            for (int u = 0; u < V; ++u) h[c][u] += d;
        }
    }
    // ---- cubic anisotropy (Eq. (5), reading A14): h -= sum_i (dE/da_i) c_i ----
    if (!LEAN && p.cubic) {
#pragma unroll
        for (int u = 0; u < V; ++u) {
            const float a1 = m[0][u] * p.c1[0] + m[1][u] * p.c1[1] + m[2][u] * p.c1[2];
            const float a2 = m[0][u] * p.c2[0] + m[1][u] * p.c2[1] + m[2][u] * p.c2[2];
            const float a3 = m[0][u] * p.c3[0] + m[1][u] * p.c3[1] + m[2][u] * p.c3[2];
            const float q1 = a1 * a1, q2 = a2 * a2, q3 = a3 * a3;
            const float d1 = a1 * (p.k1c * (q2 + q3) + p.k2c * q2 * q3);
            const float d2 = a2 * (p.k1c * (q3 + q1) + p.k2c * q3 * q1);
            const float d3 = a3 * (p.k1c * (q1 + q2) + p.k2c * q1 * q2);
#pragma unroll
            for (int c = 0; c < 3; ++c) h[c][u] -= d1 * p.c1[c] + d2 * p.c2[c] + d3 * p.c3[c];
        }
    }
    // ---- thermal field (Eq. (6), reading A6) ----
    if (!LEAN && p.thermal) {
#pragma unroll
        for (int u = 0; u < V; ++u) {
            float eta[3];
            thermal_eta(p, (uint64_t)(idx + u) + p.cell0, eta);
#pragma unroll
            for (int c = 0; c < 3; ++c) h[c][u] += p.sig_th * eta[c];
        }
    }
    if (p.mode == EPI_HEFF) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            float o[V];
#pragma unroll
            for (int u = 0; u < V; ++u) o[u] = p.out_scale * h[c][u];
            stv<V>(p.out + idx + c * n, o);
        }
        return 0.f;
    }
    // ---- torque, Eq. (1): dm/dtau = -1/(1+alpha^2) [ m x h + alpha m x (m x h) ] ----
    float k[3][V];
#pragma unroll
    for (int u = 0; u < V; ++u) {
        const float mm_[3] = { m[0][u], m[1][u], m[2][u] };
        const float hh[3] = { h[0][u], h[1][u], h[2][u] };
        float mxh[3], mxmxh[3];
        cross3(mm_, hh, mxh);
        cross3(mm_, mxh, mxmxh);
#pragma unroll
        for (int c = 0; c < 3; ++c) k[c][u] = -p.inv1pa2 * (mxh[c] + p.alpha * mxmxh[c]);
        if (!LEAN && p.stt) {   // Eq. (7): - c_ad m x (m x D) - c_nad m x D
            const float DD[3] = { D[0][u], D[1][u], D[2][u] };
            float mxD[3], mxmxD[3];
            cross3(mm_, DD, mxD);
            cross3(mm_, mxD, mxmxD);
#pragma unroll
            for (int c = 0; c < 3; ++c) k[c][u] -= p.c_ad * mxmxD[c] + p.c_nad * mxD[c];
        }
    }
    if (p.mode == EPI_TORQUE) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            float o[V];
#pragma unroll
            for (int u = 0; u < V; ++u) o[u] = p.out_scale * k[c][u];
            stv<V>(p.out + idx + c * n, o);
        }
        return 0.f;
    }
    // ---- Runge-Kutta stage combine ----
    const float ds = p.dt_scale ? __ldg(p.dt_scale) : 1.0f;     // step length kept on the device (a11)
    float r[3][V];
    if (p.m_out) {
        float acc[3][V];
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int u = 0; u < V; ++u) acc[c][u] = ds * p.a_self * k[c][u];
#pragma unroll
        for (int j = 0; j < (NA >= 0 ? NA : p.na); ++j) {
            const float* __restrict__ kj = p.ka[j];
            const float aj = ds * p.a[j];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                float t[V];
                ldv<V>(kj + idx + c * n, t);
#pragma unroll
                for (int u = 0; u < V; ++u) acc[c][u] += aj * t[u];
            }
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            float t[V];
            ldv<V>(p.m_n + idx + c * n, t);
#pragma unroll
            for (int u = 0; u < V; ++u) r[c][u] = t[u] + acc[c][u];
        }
        if (p.normalise) {
#pragma unroll
            for (int u = 0; u < V; ++u) {
                const float q = r[0][u] * r[0][u] + r[1][u] * r[1][u] + r[2][u] * r[2][u];
                const float s = q > 0.f ? rsqrtf(q) : 0.f;        // an empty cell stays empty (reading A15)
                r[0][u] *= s; r[1][u] *= s; r[2][u] *= s;
            }
        }
    }
    float red = 0.f;
    if (p.do_err) {
        float e[3][V];
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int u = 0; u < V; ++u) e[c][u] = ds * p.e_self * k[c][u];
        for (int j = 0; j < p.ne; ++j) {
            const float* __restrict__ kj = p.ke[j];
            const float ej = ds * p.e[j];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                float t[V];
                ldv<V>(kj + idx + c * n, t);
#pragma unroll
                for (int u = 0; u < V; ++u) e[c][u] += ej * t[u];
            }
        }
#pragma unroll
        for (int u = 0; u < V; ++u) {
            const float q = sqrtf(e[0][u] * e[0][u] + e[1][u] * e[1][u] + e[2][u] * e[2][u]);
            // NaN must win the reduction: compare bit patterns of |q|
            red = __uint_as_float(max(__float_as_uint(red), __float_as_uint(q) & 0x7fffffffu));
        }
    }
    if (p.k_out) {
#pragma unroll
        for (int c = 0; c < 3; ++c) stv<V>(p.k_out + idx + c * n, k[c]);
    }
    if (p.m_out) {
#pragma unroll
        for (int c = 0; c < 3; ++c) stv<V>(p.m_out + idx + c * n, r[c]);
    }
    return red;
}

__device__ __forceinline__ float epilogue_finish(const EpiParams& p, size_t idx, size_t n, const float (&m)[3],
                                                 float (&h)[3], const float (&D)[3])
{
    const float m1[3][1] = { { m[0] }, { m[1] }, { m[2] } };
    float h1[3][1] = { { h[0] }, { h[1] }, { h[2] } };
    const float D1[3][1] = { { D[0] }, { D[1] }, { D[2] } };
    return epilogue_finish_v<1>(p, idx, n, m1, h1, D1);
}

// One cell.  hms = magnetostatic field in units of Ms.  Returns the value to be max-reduced.
__device__ __forceinline__ float epilogue_cell(const Geom& g, const EpiParams& p, int x, int y, int z,
                                               float hx, float hy, float hz)
{
    const size_t plane = (size_t)g.Ny * g.Nx;
    const size_t n = plane * g.Nz;
    const size_t idx = (size_t)z * plane + (size_t)y * g.Nx + x;
    const float* __restrict__ mi = p.m_in;
    float m[3] = { mi[idx], mi[idx + n], mi[idx + 2 * n] };
    float h[3] = { hx, hy, hz };
    if (p.mode == EPI_HMS) {
        p.out[idx] = p.out_scale * h[0];
        p.out[idx + n] = p.out_scale * h[1];
        p.out[idx + 2 * n] = p.out_scale * h[2];
        return 0.f;
    }
    // ---- neighbours: exchange (Eq. (3), reading A3) and (j.grad) m (Eq. (7), reading A7) ----
    float D[3] = { 0.f, 0.f, 0.f };
    {
        const int pos[3] = { x, y, z };
        const int ext[3] = { g.Nx, g.Ny, g.Nz };
        const int per[3] = { g.perx, g.pery, g.perz };
        const size_t str[3] = { (size_t)1, (size_t)g.Nx, plane };
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            if (ext[a] == 1) continue;
            const bool need_ex = p.wex[a] != 0.f;
            const bool need_j = p.stt && p.cj[a] != 0.f;
            if (!need_ex && !need_j) continue;
            // index of the +/- neighbours; a missing neighbour is replaced by the cell itself
            size_t ip = idx, im = idx;
            if (pos[a] + 1 < ext[a]) ip = idx + str[a];
            else if (per[a]) ip = idx - (size_t)(ext[a] - 1) * str[a];
            if (pos[a] > 0) im = idx - str[a];
            else if (per[a]) im = idx + (size_t)(ext[a] - 1) * str[a];
            float mp[3] = { mi[ip], mi[ip + n], mi[ip + 2 * n] };
            float mm_[3] = { mi[im], mi[im + n], mi[im + 2 * n] };
            if (p.geometry) {     // reading A15: an empty neighbour is a missing one; an empty cell has no field
                const bool full = m[0] * m[0] + m[1] * m[1] + m[2] * m[2] > 0.f;
                if (!full || !(mp[0] * mp[0] + mp[1] * mp[1] + mp[2] * mp[2] > 0.f)) { mp[0] = m[0]; mp[1] = m[1]; mp[2] = m[2]; }
                if (!full || !(mm_[0] * mm_[0] + mm_[1] * mm_[1] + mm_[2] * mm_[2] > 0.f)) { mm_[0] = m[0]; mm_[1] = m[1]; mm_[2] = m[2]; }
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                h[c] += p.wex[a] * ((mp[c] - m[c]) + (mm_[c] - m[c]));
                D[c] += p.cj[a] * (mp[c] - mm_[c]);
            }
        }
    }
    return epilogue_finish(p, idx, n, m, h, D);
}

// ---- two vertically adjacent cells (x, y0) and (x, y0 + 1) at once: the inverse x pass owns row
// pairs.  PairNbr holds every m value the two cells need (12 positions x 3 components); it is loaded
// one x ahead of its use so that the loads of the next pair are in flight during the arithmetic
// and stores of the current one. ----
struct PairNbr {
    float col[4][3];     // rows y0-1, y0, y0+1, y0+2 at x (missing row -> the cell's own row)
    float xm[2][3], xp[2][3], zm[2][3], zp[2][3];
};

struct PairGeom {        // per row pair, uniform over x
    size_t n;            // cells per component
    size_t row[4];       // start of rows y0-1 .. y0+2 in plane z (clamped / wrapped)
    size_t rzm[2], rzp[2];   // start of rows y0, y0+1 in planes z-1, z+1 (clamped / wrapped)
};

__device__ __forceinline__ PairGeom pair_geom(const Geom& g, int y0, int z, bool two)
{
    PairGeom q;
    const size_t plane = (size_t)g.Ny * g.Nx;
    q.n = plane * g.Nz;
    const int y1 = two ? y0 + 1 : y0;
    const int ym = y0 > 0 ? y0 - 1 : (g.pery ? g.Ny - 1 : y0);
    int yA = y0 + 1, yB = y0 + 2;                 // + neighbours of the two cells
    if (yA >= g.Ny) yA = g.pery ? yA - g.Ny : y0;
    if (yB >= g.Ny) yB = g.pery ? yB - g.Ny : y1;
    const int zm = z > 0 ? z - 1 : (g.perz ? g.Nz - 1 : z);
    const int zp = z + 1 < g.Nz ? z + 1 : (g.perz ? 0 : z);
    const size_t zb = (size_t)z * plane;
    q.row[0] = zb + (size_t)ym * g.Nx;
    q.row[1] = zb + (size_t)y0 * g.Nx;
    q.row[2] = zb + (size_t)yA * g.Nx;            // == row y0+1 when it exists
    q.row[3] = zb + (size_t)yB * g.Nx;
    q.rzm[0] = (size_t)zm * plane + (size_t)y0 * g.Nx;
    q.rzm[1] = (size_t)zm * plane + (size_t)y1 * g.Nx;
    q.rzp[0] = (size_t)zp * plane + (size_t)y0 * g.Nx;
    q.rzp[1] = (size_t)zp * plane + (size_t)y1 * g.Nx;
    return q;
}

__device__ __forceinline__ void pair_load(const Geom& g, const float* __restrict__ mi, const PairGeom& q, int x,
                                          bool two, PairNbr& v)
{
    const int xl = x > 0 ? x - 1 : (g.perx ? g.Nx - 1 : x);
    const int xr = x + 1 < g.Nx ? x + 1 : (g.perx ? 0 : x);
    const size_t r1 = two ? q.row[1] + g.Nx : q.row[1];     // the pair's second row (or the first again)
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float* __restrict__ mc = mi + c * q.n;
        v.col[0][c] = mc[q.row[0] + x];
        v.col[1][c] = mc[q.row[1] + x];
        v.col[2][c] = mc[q.row[2] + x];
        v.col[3][c] = mc[q.row[3] + x];
        v.xm[0][c] = mc[q.row[1] + xl];
        v.xp[0][c] = mc[q.row[1] + xr];
        v.xm[1][c] = mc[r1 + xl];
        v.xp[1][c] = mc[r1 + xr];
        v.zm[0][c] = mc[q.rzm[0] + x];
        v.zm[1][c] = mc[q.rzm[1] + x];
        v.zp[0][c] = mc[q.rzp[0] + x];
        v.zp[1][c] = mc[q.rzp[1] + x];
    }
}

// which = 0: cell (x, y0); which = 1: cell (x, y0 + 1).  hms = magnetostatic field in units of Ms.
__device__ __forceinline__ float pair_cell(const EpiParams& p, const PairGeom& q, const PairNbr& v, int which,
                                           int x, int Nx, float hx, float hy, float hz)
{
    const size_t idx = (which ? q.row[1] + Nx : q.row[1]) + x;
    float h[3] = { hx, hy, hz };
    if (p.mode == EPI_HMS) {
#pragma unroll
        for (int c = 0; c < 3; ++c) p.out[idx + c * q.n] = p.out_scale * h[c];
        return 0.f;
    }
    float m[3], D[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float mc = v.col[1 + which][c];
        m[c] = mc;
        const float xp = v.xp[which][c], xm = v.xm[which][c];
        const float yp = v.col[2 + which][c], ym = v.col[which][c];
        const float zp = v.zp[which][c], zm = v.zm[which][c];
        h[c] += p.wex[0] * ((xp - mc) + (xm - mc));
        h[c] += p.wex[1] * ((yp - mc) + (ym - mc));
        h[c] += p.wex[2] * ((zp - mc) + (zm - mc));
        D[c] = p.cj[0] * (xp - xm) + p.cj[1] * (yp - ym) + p.cj[2] * (zp - zm);
    }
    return epilogue_finish(p, idx, q.n, m, h, D);
}

// Block-wide max of non-negative floats (NaN wins), one atomicMax per block (step a10).
// Order-independent, hence bit-reproducible.
// ---------------------------------------------------------------------------------------------
// The per-cell tail of one quad (4 consecutive cells along x, first cell (4 x4, y, z)) with H_ms read through `hs`
// (hs(c, v): the quad's four values of component c; shared memory in the fused last pass k_inv_x_q).  Same
// arithmetic as k_epi4.  Must be called by all 32 lanes of a warp, whose quads are consecutive along x in one row
// (the x neighbours of a quad's end cells come from the adjacent lanes).  Returns the value to be max-reduced.
// ---------------------------------------------------------------------------------------------
template <bool LEAN, int NA, typename HS>
__device__ __forceinline__ unsigned int epilogue_quad(const Geom& g, const EpiParams& ep, int x4, int y, int z, HS hs)
{
    const int nx4 = g.Nx >> 2;
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
    const bool need_nb = ep.wex[0] != 0.f || ep.wex[1] != 0.f || ep.wex[2] != 0.f || ep.stt;
    if (!need_nb) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            hs(c, h[c]);
#pragma unroll
            for (int u = 0; u < 4; ++u) if (!LEAN) D[c][u] = 0.f;
        }
        return __float_as_uint(epilogue_finish_v<4, LEAN, NA>(ep, idx, n, m, h, D)) & 0x7fffffffu;
    }
    const int ym = y > 0 ? y - 1 : (g.pery ? g.Ny - 1 : y);
    const int yp = y + 1 < g.Ny ? y + 1 : (g.pery ? 0 : y);
    const int zm = z > 0 ? z - 1 : (g.perz ? g.Nz - 1 : z);
    const int zp = z + 1 < g.Nz ? z + 1 : (g.perz ? 0 : z);
    const size_t iym = (size_t)z * plane + (size_t)ym * g.Nx + x, iyp = (size_t)z * plane + (size_t)yp * g.Nx + x;
    const size_t izm = (size_t)zm * plane + (size_t)y * g.Nx + x, izp = (size_t)zp * plane + (size_t)y * g.Nx + x;
    const bool lo_h = ep.zlo != nullptr && z == 0, hi_h = ep.zhi != nullptr && z == g.Nz - 1;
    const float* __restrict__ pzm = lo_h ? ep.zlo + (size_t)y * g.Nx + x : mi + izm;
    const float* __restrict__ pzp = hi_h ? ep.zhi + (size_t)y * g.Nx + x : mi + izp;
    const size_t szm = lo_h ? plane : n, szp = hi_h ? plane : n;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        float a[4], b[4], d[4], e[4];
        hs(c, h[c]);
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
    return __float_as_uint(epilogue_finish_v<4, LEAN, NA>(ep, idx, n, m, h, D)) & 0x7fffffffu;
}

__device__ __forceinline__ void block_max_atomic(unsigned int b, unsigned int* target)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) b = max(b, __shfl_xor_sync(0xffffffffu, b, o));
    __shared__ unsigned int wmax[32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) wmax[w] = b;
    __syncthreads();
    if (w == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        b = lane < nw ? wmax[lane] : 0u;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) b = max(b, __shfl_xor_sync(0xffffffffu, b, o));
        if (lane == 0 && b != 0u) atomicMax(target, b);
    }
}

}  // namespace mm
