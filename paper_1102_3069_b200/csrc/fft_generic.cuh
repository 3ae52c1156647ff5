// fft_generic.cuh -- shared-memory Stockham FFT over a tile of columns, radices 2, 3, 4, 5, any length
// 2^a 3^b 5^c ("1D FFT sets per axis", PAPER.md:171 smooth sizes), and the four generic
// passes built on it.  These kernels accept every supported grid; the size-specialised register
// kernels of fft_fast.cuh replace them where the grid allows (mm_set_fast_path).
//
// A tile is `ncol` independent lines of length L held as s[i * TXP + c] (i = position along the
// transformed axis, c = column).  Zero padding is applied on load and cropping on store, so padded
// arrays never exist in HBM ("zero lines skipped").
//
// Product code; shares nothing with oracle/.
#pragma once
#include "mm_common.cuh"
#include "epilogue.cuh"

namespace mm {


// (struct FftPlan: mm_kernels.h)

template <int SGN>
__device__ __forceinline__ void bfly2(float2* v)
{
    const float2 a = v[0], b = v[1];
    v[0] = cadd(a, b);
    v[1] = csub(a, b);
}

template <int SGN>
__device__ __forceinline__ void bfly4(float2* v)
{
    const float2 a = cadd(v[0], v[2]), b = csub(v[0], v[2]);
    const float2 c = cadd(v[1], v[3]), d = cmuli<SGN>(csub(v[1], v[3]));
    v[0] = cadd(a, c);
    v[1] = cadd(b, d);
    v[2] = csub(a, c);
    v[3] = csub(b, d);
}

template <int SGN>
__device__ __forceinline__ void bfly3(float2* v)
{
    const float S = 0.86602540378443864676f;
    const float2 t = cadd(v[1], v[2]);
    const float2 d = cmuli<SGN>(cscale(csub(v[1], v[2]), S));
    const float2 m = make_float2(v[0].x - 0.5f * t.x, v[0].y - 0.5f * t.y);
    v[0] = cadd(v[0], t);
    v[1] = cadd(m, d);
    v[2] = csub(m, d);
}

template <int SGN>
__device__ __forceinline__ void bfly5(float2* v)
{
    const float C1 = 0.30901699437494742410f, C2 = -0.80901699437494742410f;
    const float S1 = 0.95105651629515357212f, S2 = 0.58778525229247312917f;
    const float2 t1 = cadd(v[1], v[4]), t2 = cadd(v[2], v[3]);
    const float2 d1 = csub(v[1], v[4]), d2 = csub(v[2], v[3]);
    const float2 a1 = make_float2(v[0].x + C1 * t1.x + C2 * t2.x, v[0].y + C1 * t1.y + C2 * t2.y);
    const float2 a2 = make_float2(v[0].x + C2 * t1.x + C1 * t2.x, v[0].y + C2 * t1.y + C1 * t2.y);
    const float2 b1 = cmuli<SGN>(make_float2(S1 * d1.x + S2 * d2.x, S1 * d1.y + S2 * d2.y));
    const float2 b2 = cmuli<SGN>(make_float2(S2 * d1.x - S1 * d2.x, S2 * d1.y - S1 * d2.y));
    v[0] = cadd(v[0], cadd(t1, t2));
    v[1] = cadd(a1, b1);
    v[4] = csub(a1, b1);
    v[2] = cadd(a2, b2);
    v[3] = csub(a2, b2);
}

// radix 7 (PAPER.md:171 lists sizes 2^n x {1, 3, 5, 7}): X_k = v0 + sum_j t_j cos(2 pi j k / 7) + SGN i sum_j d_j sin(...),
// t_j = v_j + v_(7-j), d_j = v_j - v_(7-j), j = 1..3
template <int SGN>
__device__ __forceinline__ void bfly7(float2* v)
{
    const float C[3] = { 0.62348980185873353053f, -0.22252093395631440429f, -0.90096886790241912624f };
    const float S[3] = { 0.78183148246802980871f, 0.97492791218182360702f, 0.43388373911755812048f };
    float2 t[3], d[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) { t[j] = cadd(v[j + 1], v[6 - j]); d[j] = csub(v[j + 1], v[6 - j]); }
    const float2 v0 = v[0];
    v[0] = cadd(v0, cadd(t[0], cadd(t[1], t[2])));
#pragma unroll
    for (int k = 1; k <= 3; ++k) {
        float2 a = v0, b = make_float2(0.f, 0.f);
#pragma unroll
        for (int j = 1; j <= 3; ++j) {
            const int q = (j * k) % 7;                    // cos(2 pi q / 7), sin(2 pi q / 7) from q in 1..3 by symmetry
            const float c = q <= 3 ? C[q - 1] : C[6 - q];
            const float s = q <= 3 ? S[q - 1] : -S[6 - q];
            a.x += c * t[j - 1].x; a.y += c * t[j - 1].y;
            b.x += s * d[j - 1].x; b.y += s * d[j - 1].y;
        }
        const float2 ib = cmuli<SGN>(b);
        v[k] = cadd(a, ib);
        v[7 - k] = csub(a, ib);
    }
}

// One Stockham pass of radix R: in -> out.
template <int R, int SGN>
__device__ __forceinline__ void stockham_pass(const float2* __restrict__ in, float2* __restrict__ out,
                                              int L, int ns, int TXP, int ncol,
                                              const float2* __restrict__ tw)
{
    const int m = L / R;
    const int twstep = L / (ns * R);
    for (int it = threadIdx.x; it < m * ncol; it += blockDim.x) {
        const int c = it % ncol;
        const int j = it / ncol;
        const int k = j % ns;
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            v[r] = in[(j + r * m) * TXP + c];
            if (r > 0 && ns > 1) {
                float2 w = __ldg(&tw[r * k * twstep]);
                if (SGN > 0) w.y = -w.y;
                v[r] = cmul(v[r], w);
            }
        }
        if (R == 2) bfly2<SGN>(v);
        if (R == 3) bfly3<SGN>(v);
        if (R == 4) bfly4<SGN>(v);
        if (R == 5) bfly5<SGN>(v);
        if (R == 7) bfly7<SGN>(v);
        const int j0 = (j / ns) * ns * R + k;
#pragma unroll
        for (int s = 0; s < R; ++s) out[(j0 + s * ns) * TXP + c] = v[s];
    }
}

// Transform every column of the tile; returns the buffer that holds the result (a or b).
// All threads of the block must call it; ends with a __syncthreads().
template <int SGN>
__device__ float2* tile_fft(float2* a, float2* b, const FftPlan& pl, int TXP, int ncol)
{
    int ns = 1;
    __syncthreads();
    for (int q = 0; q < pl.nrad; ++q) {
        const int R = pl.rad[q];
        if (R == 4) stockham_pass<4, SGN>(a, b, pl.L, ns, TXP, ncol, pl.tw);
        else if (R == 2) stockham_pass<2, SGN>(a, b, pl.L, ns, TXP, ncol, pl.tw);
        else if (R == 3) stockham_pass<3, SGN>(a, b, pl.L, ns, TXP, ncol, pl.tw);
        else if (R == 5) stockham_pass<5, SGN>(a, b, pl.L, ns, TXP, ncol, pl.tw);
        else stockham_pass<7, SGN>(a, b, pl.L, ns, TXP, ncol, pl.tw);
        ns *= R;
        float2* t = a; a = b; b = t;
        __syncthreads();
    }
    return a;
}

extern __shared__ float2 mm_smem[];

// ---------------------------------------------------------------------------------------------
// a1: forward x pass, real -> complex.  Two real lines (rows y, y+1 of one (component, z)) are
// packed as the real and imaginary part of one complex line; the two spectra are separated
// afterwards using the Hermitian symmetry of a real signal's transform.
// grid.x = ceil(npair_total / TX), npair_total = 3 Nz ceil(Ny/2).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_gen_fwd_x(Geom g, FftPlan pl, const float* __restrict__ m, float2* __restrict__ specA, int TX)
{
    const int TXP = TX + 1;
    float2* a = mm_smem;
    float2* b = mm_smem + (size_t)pl.L * TXP;
    const int npy = (g.Ny + 1) >> 1;
    const int npair = 3 * g.Nz * npy;
    const int p0 = blockIdx.x * TX;
    const int ncol = min(TX, npair - p0);
    // load (x fastest => coalesced), zero pad on the fly
    for (int it = threadIdx.x; it < pl.L * ncol; it += blockDim.x) {
        const int i = it % pl.L, c = it / pl.L;
        float2 v = make_float2(0.f, 0.f);
        if (i < g.Nx) {
            const int pp = p0 + c;
            const int cz = pp / npy, y0 = 2 * (pp % npy);
            const size_t row = ((size_t)cz * g.Ny + y0) * g.Nx;
            v.x = m[row + i];
            if (y0 + 1 < g.Ny) v.y = m[row + g.Nx + i];
        }
        a[i * TXP + c] = v;
    }
    float2* s = tile_fft<-1>(a, b, pl, TXP, ncol);
    const int P = pl.L;
    for (int it = threadIdx.x; it < g.Cx * ncol; it += blockDim.x) {
        const int k = it % g.Cx, c = it / g.Cx;
        const float2 zk = s[k * TXP + c];
        const float2 zc = cconj(s[((P - k) % P) * TXP + c]);
        const float2 A = cscale(cadd(zk, zc), 0.5f);
        const float2 d = csub(zk, zc);
        const float2 B = make_float2(0.5f * d.y, -0.5f * d.x);
        const int pp = p0 + c;
        const int cz = pp / npy, y0 = 2 * (pp % npy);
        const size_t row = ((size_t)cz * g.Ny + y0) * g.CxS;
        specA[row + k] = A;
        if (y0 + 1 < g.Ny) specA[row + g.CxS + k] = B;
    }
}

// ---------------------------------------------------------------------------------------------
// a2 / a4: y pass, complex, on TX adjacent kx columns of one (component, z) plane.
// forward: specA rows y < Ny -> specB rows ky < Py.  inverse: specB -> specA rows y < Ny.
// grid = (ceil(Cx / TX), 3 Nz)
// ---------------------------------------------------------------------------------------------
template <int SGN>
__global__ void __launch_bounds__(256)
k_gen_y(Geom g, FftPlan pl, const float2* __restrict__ src, float2* __restrict__ dst, int TX)
{
    const int TXP = TX + 1;
    float2* a = mm_smem;
    float2* b = mm_smem + (size_t)pl.L * TXP;
    const int kx0 = blockIdx.x * TX;
    const int ncol = min(TX, g.Cx - kx0);
    const int cz = blockIdx.y;
    const int nin = SGN < 0 ? g.Ny : g.Py;
    const int nout = SGN < 0 ? g.Py : g.Ny;
    const float2* __restrict__ sp = src + (size_t)cz * nin * g.CxS + kx0;
    float2* __restrict__ dp = dst + (size_t)cz * nout * g.CxS + kx0;
    for (int it = threadIdx.x; it < pl.L * ncol; it += blockDim.x) {
        const int c = it % ncol, i = it / ncol;
        a[i * TXP + c] = i < nin ? sp[(size_t)i * g.CxS + c] : make_float2(0.f, 0.f);
    }
    float2* s = tile_fft<SGN>(a, b, pl, TXP, ncol);
    for (int it = threadIdx.x; it < nout * ncol; it += blockDim.x) {
        const int c = it % ncol, i = it / ncol;
        dp[(size_t)i * g.CxS + c] = s[i * TXP + c];
    }
}

// ---------------------------------------------------------------------------------------------
// a3: last-axis pass, fused: forward transform of the three components, multiply by the symmetric
// real kernel K-hat (6 unique real components), inverse transform, crop; in place.
// axis 2 (z, 3D): one block per (kx tile, ky); axis 1 (y, Nz = 1): one block per kx tile.
// Shared memory: 4 tile buffers (three components + one scratch).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_gen_mid(Geom g, FftPlan pl, float2* __restrict__ spec, const float* __restrict__ khat, int axis, int TX)
{
    const int TXP = TX + 1;
    const size_t tile = (size_t)pl.L * TXP;
    float2* buf[4] = { mm_smem, mm_smem + tile, mm_smem + 2 * tile, mm_smem + 3 * tile };
    const int kx0 = blockIdx.x * TX;
    const int ncol = min(TX, g.Cx - kx0);
    const int other = blockIdx.y;                       // ky when axis == 2
    const int nrow = axis == 2 ? g.Nz : g.Ny;           // rows that exist in HBM
    const size_t rstride = axis == 2 ? (size_t)g.Py * g.CxS : (size_t)g.CxS;
    const size_t cstride = (size_t)g.Nz * (axis == 2 ? g.Py : g.Ny) * g.CxS;
    const size_t base = (axis == 2 ? (size_t)other * g.CxS : 0) + kx0;
    for (int comp = 0; comp < 3; ++comp) {
        const float2* __restrict__ sp = spec + comp * cstride + base;
        float2* a = buf[comp];
        for (int it = threadIdx.x; it < pl.L * ncol; it += blockDim.x) {
            const int c = it % ncol, i = it / ncol;
            a[i * TXP + c] = i < nrow ? sp[(size_t)i * rstride + c] : make_float2(0.f, 0.f);
        }
    }
    // forward transforms; the scratch buffer rotates
    float2* scratch = buf[3];
    float2* dat[3];
    for (int comp = 0; comp < 3; ++comp) {
        float2* r = tile_fft<-1>(buf[comp], scratch, pl, TXP, ncol);
        if (r != buf[comp]) { scratch = buf[comp]; }
        dat[comp] = r;
    }
    // h = K m  (the sign and 1/(Px Py Pz) are folded into K-hat)
    {
        const int ky = axis == 2 ? other : 0;
        const size_t nC = (size_t)g.CxK * g.Cy * g.Cz;
        for (int it = threadIdx.x; it < pl.L * ncol; it += blockDim.x) {
            const int c = it % ncol, i = it / ncol;
            int kyy = ky, kzz = 0;
            if (axis == 2) kzz = i; else kyy = i;
            float sy = 1.f, sz = 1.f;
            if (2 * kyy > g.Py) { kyy = g.Py - kyy; sy = -1.f; }
            if (2 * kzz > g.Pz) { kzz = g.Pz - kzz; sz = -1.f; }
            const size_t ko = ((size_t)kzz * g.Cy + kyy) * g.CxK + kx0 + c;
            const float kxx = __ldg(&khat[ko]), kyy_ = __ldg(&khat[ko + nC]), kzz_ = __ldg(&khat[ko + 2 * nC]);
            const float kxy = sy * __ldg(&khat[ko + 3 * nC]);
            const float kxz = sz * __ldg(&khat[ko + 4 * nC]);
            const float kyz = sy * sz * __ldg(&khat[ko + 5 * nC]);
            const float2 mx = dat[0][i * TXP + c], my = dat[1][i * TXP + c], mz = dat[2][i * TXP + c];
            dat[0][i * TXP + c] = make_float2(kxx * mx.x + kxy * my.x + kxz * mz.x,
                                              kxx * mx.y + kxy * my.y + kxz * mz.y);
            dat[1][i * TXP + c] = make_float2(kxy * mx.x + kyy_ * my.x + kyz * mz.x,
                                              kxy * mx.y + kyy_ * my.y + kyz * mz.y);
            dat[2][i * TXP + c] = make_float2(kxz * mx.x + kyz * my.x + kzz_ * mz.x,
                                              kxz * mx.y + kyz * my.y + kzz_ * mz.y);
        }
    }
    for (int comp = 0; comp < 3; ++comp) {
        float2* r = tile_fft<1>(dat[comp], scratch, pl, TXP, ncol);
        if (r != dat[comp]) { scratch = dat[comp]; }
        float2* __restrict__ dp = spec + comp * cstride + base;
        for (int it = threadIdx.x; it < nrow * ncol; it += blockDim.x) {
            const int c = it % ncol, i = it / ncol;
            dp[(size_t)i * rstride + c] = r[i * TXP + c];
        }
    }
}

// k-space multiply on its own (only when neither a y nor a z pass exists: Ny = Nz = 1).
__global__ void k_gen_mul1d(Geom g, float2* __restrict__ spec, const float* __restrict__ khat)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= g.Cx) return;
    const size_t nC = (size_t)g.CxK * g.Cy * g.Cz;
    const float kxx = khat[k], kyy = khat[k + nC], kzz = khat[k + 2 * nC];
    const float kxy = khat[k + 3 * nC], kxz = khat[k + 4 * nC], kyz = khat[k + 5 * nC];
    const float2 mx = spec[k], my = spec[g.CxS + k], mz = spec[2 * (size_t)g.CxS + k];
    spec[k] = make_float2(kxx * mx.x + kxy * my.x + kxz * mz.x, kxx * mx.y + kxy * my.y + kxz * mz.y);
    spec[g.CxS + k] = make_float2(kxy * mx.x + kyy * my.x + kyz * mz.x, kxy * mx.y + kyy * my.y + kyz * mz.y);
    spec[2 * (size_t)g.CxS + k] = make_float2(kxz * mx.x + kyz * my.x + kzz * mz.x,
                                              kxz * mx.y + kyz * my.y + kzz * mz.y);
}

// ---------------------------------------------------------------------------------------------
// a5-a10: inverse x pass, complex -> real, fused with the epilogue.  One block handles TXP2 row
// pairs (y, y+1) of one z plane, all three components (3 * TXP2 columns), so that the three field
// components of a cell meet in one block.  grid = (ceil(npy / TXP2), Nz).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_gen_inv_x(Geom g, FftPlan pl, const float2* __restrict__ specA, EpiParams ep, int TXP2)
{
    const int npy = (g.Ny + 1) >> 1;
    const int pr0 = blockIdx.x * TXP2;
    const int npr = min(TXP2, npy - pr0);
    const int ncol = 3 * npr;
    const int TXP = 3 * TXP2 + 1;
    float2* a = mm_smem;
    float2* b = mm_smem + (size_t)pl.L * TXP;
    const int z = blockIdx.y;
    const int P = pl.L;
    float2* s = a;
    if (ep.demag) {
        // Z[k] = A[k] + i B[k], Z[P-k] = conj(A[k]) + i conj(B[k])
        for (int it = threadIdx.x; it < g.Cx * ncol; it += blockDim.x) {
            const int k = it % g.Cx, c = it / g.Cx;
            const int comp = c / npr, y0 = 2 * (pr0 + c % npr);
            const size_t row = (((size_t)comp * g.Nz + z) * g.Ny + y0) * g.CxS;
            const float2 A = specA[row + k];
            const float2 B = (y0 + 1 < g.Ny) ? specA[row + g.CxS + k] : make_float2(0.f, 0.f);
            a[k * TXP + c] = make_float2(A.x - B.y, A.y + B.x);
            if (k > 0 && 2 * k < P) a[(P - k) * TXP + c] = make_float2(A.x + B.y, -A.y + B.x);
        }
        s = tile_fft<1>(a, b, pl, TXP, ncol);
    }
    unsigned int red = 0u;   // bit pattern of a non-negative float; NaN patterns compare largest
    for (int it = threadIdx.x; it < g.Nx * 2 * npr; it += blockDim.x) {
        const int x = it % g.Nx, r = it / g.Nx;      // r: row within the block's 2*npr rows
        const int pr = r >> 1, odd = r & 1;
        const int y = 2 * (pr0 + pr) + odd;
        if (y >= g.Ny) continue;
        float h[3] = { 0.f, 0.f, 0.f };
        if (ep.demag) {
#pragma unroll
            for (int comp = 0; comp < 3; ++comp) {
                const float2 v = s[x * TXP + comp * npr + pr];
                h[comp] = odd ? v.y : v.x;
            }
        }
        red = max(red, __float_as_uint(epilogue_cell(g, ep, x, y, z, h[0], h[1], h[2])) & 0x7fffffffu);
    }
    if (ep.do_err) block_max_atomic(red, ep.maxbits);
}

}  // namespace mm
