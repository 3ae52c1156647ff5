// fft_fast_kernels.cuh -- the five passes of one evaluation built on ff::fft_line (steps a1-a10).
// Included by fft_fast.cuh.  Product code; shares nothing with oracle/.
#pragma once

namespace mm {
namespace ff {

extern __shared__ float2 ff_smem[];

// ---------------------------------------------------------------------------------------------
// a1: forward x pass, real -> complex.  T threads own one pair of rows (y0, y0+1) packed as
// real/imaginary part of one complex line; the two spectra are separated with the Hermitian
// partner k <-> L-k, which in standard form lives in thread T-t, register E-1-j (shuffle).
// PER = periodic x axis (no zero padding: Nx == L); otherwise Nx == L/2.
// block = 128 threads = 128/T line slots; persistent grid-stride loop over row pairs.
// ---------------------------------------------------------------------------------------------
template <int T, int E, bool PER>
__global__ void __launch_bounds__(128)
k_fwd_x(Geom g, const float* __restrict__ m, float2* __restrict__ specA, const float2* __restrict__ tw)
{
    constexpr int L = T * E;
    constexpr int LB = T * (E + 1);            // exchange buffer of one line, float2
    constexpr int NIN = PER ? E : E / 2;
    const int t = threadIdx.x % T;
    const int slot = threadIdx.x / T;
    const int nslot = 128 / T;
    float2* sb = ff_smem + slot * LB;
    const int npy = (g.Ny + 1) >> 1;
    const int npair = 3 * g.Nz * npy;
    const unsigned lane = threadIdx.x & 31;
    const unsigned lbase = lane - t;           // first lane of this line's thread group
    // the trip count is uniform over the block (full-mask shuffles); an idle slot redoes the last pair
    for (int pb = blockIdx.x * nslot; pb < npair; pb += gridDim.x * nslot) {
        const bool act = pb + slot < npair;
        const int pp = act ? pb + slot : npair - 1;
        const int cz = pp / npy, y0 = 2 * (pp - cz * npy);
        const bool two = y0 + 1 < g.Ny;
        const float* __restrict__ r0 = m + ((size_t)cz * g.Ny + y0) * g.Nx;
        float2 v[E];
#pragma unroll
        for (int j = 0; j < NIN; ++j) {
            v[j].x = r0[t + T * j];
            v[j].y = two ? r0[g.Nx + t + T * j] : 0.f;
        }
        __syncwarp();                           // previous iteration's reads of sb are done
        fft_line<T, E, -1, !PER>(v, sb, 1, t, tw, SyncWarp());
        // separate: A[k] = (Z[k] + conj Z[L-k]) / 2,  B[k] = (Z[k] - conj Z[L-k]) / (2i)
        float2* __restrict__ o0 = specA + ((size_t)cz * g.Ny + y0) * g.CxS;
        float2* __restrict__ o1 = o0 + g.CxS;
        const unsigned src = lbase + ((T - t) % T);
#pragma unroll
        for (int j = 0; j < E / 2; ++j) {
            float2 p;
            p.x = __shfl_sync(0xffffffffu, v[E - 1 - j].x, src);
            p.y = __shfl_sync(0xffffffffu, v[E - 1 - j].y, src);
            if (t == 0) p = v[(E - j) % E];
            const float2 z = v[j];
            if (act) o0[t + T * j] = make_float2(0.5f * (z.x + p.x), 0.5f * (z.y - p.y));
            if (act && two) o1[t + T * j] = make_float2(0.5f * (z.y + p.y), 0.5f * (p.x - z.x));
        }
        if (t == 0 && act) {                    // k = L/2 is its own partner
            o0[L / 2] = make_float2(v[E / 2].x, 0.f);
            if (two) o1[L / 2] = make_float2(v[E / 2].y, 0.f);
        }
    }
}

// ---- cp.async helpers (16-byte copies global -> shared, zero-filled beyond src_bytes) ----
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, int src_bytes)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

// ---------------------------------------------------------------------------------------------
// a1 / a5, software-pipelined forms of k_fwd_x / k_inv_x_h (same arithmetic, same thread layout): the
// rows of the NEXT pair are staged by cp.async into the slot's exchange buffer -- free between the
// read-back of the exchange and the next first register FFT -- while the second register FFT, the
// separation shuffles and the stores of the current pair run.  Needs 16-byte aligned rows (Nx % 4 == 0).
// ---------------------------------------------------------------------------------------------
// BULK: the two rows of a pair are adjacent in m, so they arrive by ONE bulk copy (cp.async.bulk, issued by lane t = 0
// of the slot, completion on the slot's mbarrier) instead of 8 cp.async per thread.
template <int T, int E, bool PER, bool BULK = false>
__global__ void __launch_bounds__(128)
k_fwd_x_p(Geom g, const float* __restrict__ m, float2* __restrict__ specA, const float2* __restrict__ tw)
{
    constexpr int L = T * E;
    constexpr int LB = T * (E + 1);
    constexpr int NIN = PER ? E : E / 2;
    constexpr int NXC = PER ? L : L / 2;       // == g.Nx
    const int t = threadIdx.x % T;
    const int slot = threadIdx.x / T;
    const int nslot = 128 / T;
    float2* sb = ff_smem + slot * LB;
    float* sf = reinterpret_cast<float*>(sb);  // staged rows: [2][NXC] floats
    const int npy = (g.Ny + 1) >> 1;
    const int npair = 3 * g.Nz * npy;
    const unsigned lane = threadIdx.x & 31;
    const unsigned src = lane - t + ((T - t) % T);
    const int stride = gridDim.x * nslot;

    unsigned long long* bar = reinterpret_cast<unsigned long long*>(ff_smem + nslot * LB) + slot;
    if (BULK) {
        if (t == 0) pk::mbar_init(bar, 1);
        if (threadIdx.x == 0) pk::mbar_fence_init();
        __syncthreads();
    }
    unsigned par = 0;
    auto issue = [&](int pb) {
        const int pp = pb + slot < npair ? pb + slot : npair - 1;
        const int cz = pp / npy, y0 = 2 * (pp - cz * npy);
        const bool two = y0 + 1 < g.Ny;
        const float* __restrict__ r0 = m + ((size_t)cz * g.Ny + y0) * g.Nx;
        if (BULK) {
            if (t == 0) {
                const unsigned nb = (two ? 2u : 1u) * NXC * (unsigned)sizeof(float);
                pk::fence_proxy_async_smem();
                pk::mbar_expect_tx(bar, nb);
                pk::bulk_load_1d(sf, r0, nb, bar);
            }
            return;
        }
        for (int u = t; u < NXC / 2; u += T) {
            const int row = u / (NXC / 4), q = u - row * (NXC / 4);
            const bool ok = row == 0 || two;
            cp_async16(sf + row * NXC + 4 * q, ok ? r0 + (size_t)row * g.Nx + 4 * q : m, ok ? 16 : 0);
        }
    };

    int pb = blockIdx.x * nslot;
    if (pb < npair) issue(pb);
    cp_async_commit();
    for (; pb < npair; pb += stride) {
        const bool act = pb + slot < npair;
        const int pp = act ? pb + slot : npair - 1;
        const int cz = pp / npy, y0 = 2 * (pp - cz * npy);
        const bool two = y0 + 1 < g.Ny;
        if (BULK) { pk::mbar_wait(bar, par); par ^= 1u; }
        else { cp_async_wait<0>(); __syncwarp(); }
        float2 v[E];
#pragma unroll
        for (int j = 0; j < NIN; ++j) v[j] = make_float2(sf[t + T * j], (!BULK || two) ? sf[NXC + t + T * j] : 0.f);
        __syncwarp();                           // the region now serves as the exchange buffer
        if constexpr (!PER) fft_reg_half<E, -1>(v);
        else fft_reg<E, -1>(v);
        apply_twiddles<T, E, false>(v, tw, t);
#pragma unroll
        for (int k2 = 0; k2 < E; ++k2) sb[t * (E + 1) + k2] = v[k2];
        __syncwarp();
        float2 u[E / T][T];
#pragma unroll
        for (int q = 0; q < E / T; ++q)
#pragma unroll
            for (int n1 = 0; n1 < T; ++n1) u[q][n1] = sb[n1 * (E + 1) + t + T * q];
        __syncwarp();                           // exchange read back: stage the next pair
        if (pb + stride < npair) issue(pb + stride);
        cp_async_commit();
#pragma unroll
        for (int q = 0; q < E / T; ++q) {
            fft_reg<T, -1>(u[q]);
#pragma unroll
            for (int k1 = 0; k1 < T; ++k1) v[q + (E / T) * k1] = u[q][k1];
        }
        float2* __restrict__ o0 = specA + ((size_t)cz * g.Ny + y0) * g.CxS;
        float2* __restrict__ o1 = o0 + g.CxS;
#pragma unroll
        for (int j = 0; j < E / 2; ++j) {
            float2 p;
            p.x = __shfl_sync(0xffffffffu, v[E - 1 - j].x, src);
            p.y = __shfl_sync(0xffffffffu, v[E - 1 - j].y, src);
            if (t == 0) p = v[(E - j) % E];
            const float2 z = v[j];
            if (act) o0[t + T * j] = make_float2(0.5f * (z.x + p.x), 0.5f * (z.y - p.y));
            if (act && two) o1[t + T * j] = make_float2(0.5f * (z.y + p.y), 0.5f * (p.x - z.x));
        }
        if (t == 0 && act) {
            o0[L / 2] = make_float2(v[E / 2].x, 0.f);
            if (two) o1[L / 2] = make_float2(v[E / 2].y, 0.f);
        }
    }
    cp_async_wait<0>();
}

template <int T, int E, bool PER>
__global__ void __launch_bounds__(128)
k_inv_x_h_p(Geom g, const float2* __restrict__ specA, const float2* __restrict__ tw, float* __restrict__ out,
            float scale)
{
    constexpr int L = T * E;
    constexpr int LB = T * (E + 1);
    constexpr int NOUT = PER ? E : E / 2;
    constexpr int CX = L / 2 + 1;               // == g.Cx
    constexpr int CXP = L / 2 + 2;              // second staged row starts 16-byte aligned
    static_assert(2 * CXP <= LB, "staged rows must fit the exchange buffer");
    const int t = threadIdx.x % T;
    const int slot = threadIdx.x / T;
    const int nslot = 128 / T;
    float2* sb = ff_smem + slot * LB;
    const int npy = (g.Ny + 1) >> 1;
    const int npair = 3 * g.Nz * npy;
    const unsigned lane = threadIdx.x & 31;
    const unsigned srcl = lane - t + ((T - t) % T);
    const int stride = gridDim.x * nslot;

    auto issue = [&](int pb) {
        const int pp = pb + slot < npair ? pb + slot : npair - 1;
        const int cz = pp / npy, y0 = 2 * (pp - cz * npy);
        const bool two = y0 + 1 < g.Ny;
        const float2* __restrict__ a0 = specA + ((size_t)cz * g.Ny + y0) * g.CxS;
        for (int u = t; u < CXP; u += T) {       // CXP / 2 units of two complex values per row
            const int row = u / (CXP / 2), q = u - row * (CXP / 2);
            const bool ok = row == 0 || two;
            const int nb = !ok ? 0 : (2 * q + 2 <= CX ? 16 : 8);
            cp_async16(sb + row * CXP + 2 * q, ok ? a0 + (size_t)row * g.CxS + 2 * q : specA, nb);
        }
    };

    int pb = blockIdx.x * nslot;
    if (pb < npair) issue(pb);
    cp_async_commit();
    for (; pb < npair; pb += stride) {
        const bool act = pb + slot < npair;
        const int pp = act ? pb + slot : npair - 1;
        const int cz = pp / npy, y0 = 2 * (pp - cz * npy);
        const bool two = y0 + 1 < g.Ny;
        cp_async_wait<0>();
        __syncwarp();
        float2 v[E];
#pragma unroll
        for (int j = 0; j < E / 2; ++j) {
            const float2 A = sb[t + T * j], B = sb[CXP + t + T * j];
            v[j] = make_float2(A.x - B.y, A.y + B.x);
            v[E - 1 - j] = make_float2(A.x + B.y, B.x - A.y);
        }
        float2 nyq = make_float2(0.f, 0.f);
        if (t == 0) {
            const float2 A = sb[L / 2], B = sb[CXP + L / 2];
            nyq = make_float2(A.x - B.y, A.y + B.x);
        }
        __syncwarp();                           // the region now serves as the exchange buffer
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
        fft_reg<E, 1>(v);
#pragma unroll
        for (int k2 = 1; k2 < E; ++k2) v[k2] = cmul(v[k2], cconj(__ldg(tw + k2 * T + t)));
#pragma unroll
        for (int k2 = 0; k2 < E; ++k2) sb[t * (E + 1) + k2] = v[k2];
        __syncwarp();
        float2 u[E / T][T];
#pragma unroll
        for (int q = 0; q < E / T; ++q)
#pragma unroll
            for (int n1 = 0; n1 < T; ++n1) u[q][n1] = sb[n1 * (E + 1) + t + T * q];
        __syncwarp();                           // exchange read back: stage the next pair
        if (pb + stride < npair) issue(pb + stride);
        cp_async_commit();
#pragma unroll
        for (int q = 0; q < E / T; ++q) {
            fft_reg<T, 1>(u[q]);
#pragma unroll
            for (int k1 = 0; k1 < T; ++k1) v[q + (E / T) * k1] = u[q][k1];
        }
        float* __restrict__ o0 = out + ((size_t)cz * g.Ny + y0) * g.Nx;
        if (act) {
#pragma unroll
            for (int j = 0; j < NOUT; ++j) {
                o0[t + T * j] = scale * v[j].x;
                if (two) o0[g.Nx + t + T * j] = scale * v[j].y;
            }
        }
    }
    cp_async_wait<0>();
}

// ---------------------------------------------------------------------------------------------
// Where the columns of a y / last-axis pass live.  The whole-array mode uses the layouts of
// mm_common.cuh (row stride CxS); the chunked mode works on `ncol`
// kx columns starting at kx0, with the y-padded spectrum in a compact chunk buffer [3][Nz][Py][W]
// that stays in L2 between the forward y pass, the last-axis pass and the inverse y pass.
// ---------------------------------------------------------------------------------------------
// (struct ColTile: mm_kernels.h)

// ---------------------------------------------------------------------------------------------
// a2 / a4: y pass, persistent and software-pipelined.  A tile is 8 adjacent kx columns (64-byte
// segments) of one (component, z) plane; thread = (column c = tid & 7, t = tid >> 3), block = 8 T.
// forward (SGN = -1): specA rows y < Ny (PER: all) -> specB rows ky < Py; inverse: back, rows y < Ny;
// `a` and `b` point at column kx0.  A block loops over tiles and the NEXT tile's rows arrive by
// cp.async while the second register FFT and the stores of the current tile run.  The staged tile
// [rows][8] and the exchange buffer share one shared-memory region (the tile is consumed into
// registers before the exchange starts, and the copy for the next tile is issued once the exchange
// has been read back).  grid = resident blocks; tile i -> (columns i % ntx, plane i / ntx).
// ---------------------------------------------------------------------------------------------
template <int T, int E, int SGN, bool PER>
__global__ void __launch_bounds__(8 * T, (T == 32) ? 2 : 1)
k_y_p(ColTile ct, int nplane, float2* __restrict__ a, float2* __restrict__ b, const float2* __restrict__ tw)
{
    constexpr bool FWD = SGN < 0;
    constexpr int NIN = (FWD && !PER) ? E / 2 : E;
    constexpr int NOUT = (!FWD && !PER) ? E / 2 : E;
    constexpr int NT = 8 * T;
    constexpr int ROWS = NIN * T;               // rows of the input tile
    float2* sm = ff_smem;
    const int tid = threadIdx.x, c = tid & 7, t = tid >> 3;
    const int ntx = (ct.ncol + 7) >> 3;
    const int ntile = ntx * nplane;
    const size_t s_row = FWD ? ct.a_row : ct.b_row, d_row = FWD ? ct.b_row : ct.a_row;
    const size_t s_plane = FWD ? ct.a_plane : ct.b_plane, d_plane = FWD ? ct.b_plane : ct.a_plane;
    const float2* __restrict__ src = FWD ? a : b;
    float2* __restrict__ dst = FWD ? b : a;

    // column offset of tile bx on the specB side (panels of 16 columns: two tiles per panel)
    auto boff = [&](int bx) -> size_t {
        return ct.b_panel ? (size_t)(bx >> 1) * ct.b_panel + (size_t)(bx & 1) * 8 : (size_t)bx * 8;
    };
    auto issue = [&](int i) {
        const int bx = i % ntx, cz = i / ntx;
        const float2* __restrict__ s0 = src + (size_t)cz * s_plane + (FWD ? (size_t)bx * 8 : boff(bx));
        for (int u = tid; u < ROWS * 4; u += NT) {
            const int cu = u & 3, r = u >> 2;
            const int left = ct.ncol - (bx * 8 + 2 * cu);
            const int nb = left >= 2 ? 16 : (left == 1 ? 8 : 0);
            cp_async16(sm + r * 8 + 2 * cu, nb ? s0 + (size_t)r * s_row + 2 * cu : src, nb);
        }
    };

    int i = blockIdx.x;
    if (i < ntile) issue(i);
    cp_async_commit();
    for (; i < ntile; i += gridDim.x) {
        const int bx = i % ntx, cz = i / ntx;
        const int col = bx * 8 + c;
        cp_async_wait<0>();
        __syncthreads();                        // this tile has landed
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
        __syncthreads();                        // exchange read back: the region is free for the next tile
        if (i + (int)gridDim.x < ntile) issue(i + gridDim.x);
        cp_async_commit();
#pragma unroll
        for (int q = 0; q < E / T; ++q) {
            fft_reg<T, SGN>(u[q]);
#pragma unroll
            for (int k1 = 0; k1 < T; ++k1) v[q + (E / T) * k1] = u[q][k1];
        }
        if (col < ct.ncol) {
            float2* __restrict__ dp = dst + (size_t)cz * d_plane + (FWD ? boff(bx) + c : (size_t)col);
#pragma unroll
            for (int j = 0; j < NOUT; ++j) dp[(size_t)(t + T * j) * d_row] = v[j];
        }
    }
    cp_async_wait<0>();
}

// ---------------------------------------------------------------------------------------------
// a3: last-axis pass: forward transform of the three components, H^ = K^ M^ with the real
// symmetric kernel from its octant, inverse transform, crop; in place.
// Each thread carries one line of all three components (3 E registers), so the 3x3 product
// needs no exchange.  A block handles 16 kx columns of one line set; when PAIR, blockIdx.y = 2 p + h
// and the blocks h = 0, 1 take the lines `other` = p and P_other - p, which share the same K^
// octant entries: they are adjacent in launch order, so the second fetch hits L2.
//   3D: axis z (stride sz = Py CxS), other = ky.     2D (Nz = 1): axis y, PAIR = false.
// thread = (c = tid & 15, t = tid >> 4); block = 16 T.
// ---------------------------------------------------------------------------------------------
template <int T, int E, bool PER, bool PAIR, int MINB>
__global__ void __launch_bounds__(16 * T, MINB)
k_mid(Geom g, ColTile ct, float2* __restrict__ spec, const float* __restrict__ khat,
      const float2* __restrict__ tw, int axis)
{
    constexpr int L = T * E;
    constexpr int LB = T * (E + 1) * 16;       // one component's exchange tile, float2
    constexpr int NIO = PER ? E : E / 2;
    const int c = threadIdx.x & 15, t = threadIdx.x >> 4;
    const int h = PAIR ? (blockIdx.y & 1) : 0;
    const int col = blockIdx.x * 16 + c;
    const bool valid = col < ct.ncol;
    const int kx = ct.kx0 + col;
    // line geometry
    const int Pother = axis == 2 ? g.Py : 1;
    const int oth_oct = PAIR ? (blockIdx.y >> 1) : blockIdx.y;     // 0 .. Pother/2
    int other = oth_oct;
    float so = 1.f;                             // sign of the components odd in `other`
    if (PAIR && h == 1) {
        other = (Pother - oth_oct) % Pother;
        if (other == oth_oct) return;           // self-paired line: done by the h = 0 block
        so = -1.f;
    }
    const bool store = valid;
    // `spec` points at column kx0; along z consecutive elements of a line are one (z) plane apart
    const size_t rstride = axis == 2 ? ct.b_plane : ct.b_row;
    const size_t cstride = (size_t)g.Nz * ct.b_plane;
    float2* __restrict__ base = spec + (axis == 2 ? (size_t)other * ct.b_row : 0) + col;
    float2 v[3][E];
#pragma unroll
    for (int comp = 0; comp < 3; ++comp) {
        if (valid) {
#pragma unroll
            for (int j = 0; j < NIO; ++j) v[comp][j] = base[comp * cstride + (size_t)(t + T * j) * rstride];
        } else {
#pragma unroll
            for (int j = 0; j < NIO; ++j) v[comp][j] = make_float2(0.f, 0.f);
        }
    }
#pragma unroll
    for (int comp = 0; comp < 3; ++comp)
        fft_line<T, E, -1, !PER>(v[comp], ff_smem + comp * LB + c, 16, t, tw, SyncBlock());
    // ---- multiply: the octant index of (k_axis, other) and the signs of the odd components ----
    {
        const size_t nC = (size_t)g.CxK * g.Cy * g.Cz;
        const int kxc = valid ? kx : 0;
#pragma unroll
        for (int j = 0; j < E; ++j) {
            int ka = t + T * j;
            float sa = 1.f;
            if (2 * ka > L) { ka = L - ka; sa = -1.f; }
            const size_t ko = axis == 2 ? ((size_t)ka * g.Cy + oth_oct) * g.CxK + kxc
                                        : ((size_t)ka) * g.CxK + kxc;
            const float sy = axis == 2 ? so : sa;
            const float sz = axis == 2 ? sa : 1.f;
            const float kxx = __ldg(khat + ko), kyy = __ldg(khat + ko + nC), kzz = __ldg(khat + ko + 2 * nC);
            const float kxy = sy * __ldg(khat + ko + 3 * nC);
            const float kxz = sz * __ldg(khat + ko + 4 * nC);
            const float kyz = sy * sz * __ldg(khat + ko + 5 * nC);
            const float2 mx = v[0][j], my = v[1][j], mz = v[2][j];
            v[0][j] = make_float2(kxx * mx.x + kxy * my.x + kxz * mz.x, kxx * mx.y + kxy * my.y + kxz * mz.y);
            v[1][j] = make_float2(kxy * mx.x + kyy * my.x + kyz * mz.x, kxy * mx.y + kyy * my.y + kyz * mz.y);
            v[2][j] = make_float2(kxz * mx.x + kyz * my.x + kzz * mz.x, kxz * mx.y + kyz * my.y + kzz * mz.y);
        }
    }
    __syncthreads();                            // all reads of the forward exchange are done
#pragma unroll
    for (int comp = 0; comp < 3; ++comp)
        fft_line<T, E, 1, false>(v[comp], ff_smem + comp * LB + c, 16, t, tw, SyncBlock());
    if (store) {
#pragma unroll
        for (int comp = 0; comp < 3; ++comp)
#pragma unroll
            for (int j = 0; j < NIO; ++j) base[comp * cstride + (size_t)(t + T * j) * rstride] = v[comp][j];
    }
}

// ---------------------------------------------------------------------------------------------
// a3, persistent and software-pipelined (3D grids, z axis): same arithmetic as k_mid, but a block
// loops over work items (16 kx columns x one ky pair {p, Py - p}) and, while it transforms one
// line set, cp.async already brings in the next one's spectrum tile [3][Nz][16] and, once per pair,
// the K^ octant tile [6][Cz][16], so neither load latency is exposed and the two lines of a pair
// share one K^ fetch.  The three components go through ONE exchange tile in turn (a barrier in
// between), which keeps the footprint at 67 KB and the registers at 168: 3 blocks = 12 warps per SM.
// grid = resident blocks; block = 16 T.
// ---------------------------------------------------------------------------------------------
template <int T, int E, bool PER>
__global__ void __launch_bounds__(16 * T, (T * E <= 128) ? 3 : 1)
k_mid_p(Geom g, ColTile ct, float2* __restrict__ spec, const float* __restrict__ khat,
        const float2* __restrict__ tw)
{
    constexpr int L = T * E;
    constexpr int LB = T * (E + 1) * 16;       // one component's exchange tile, float2
    constexpr int NIO = PER ? E : E / 2;
    constexpr int NZ = PER ? L : L / 2;        // == g.Nz
    constexpr int CZ = L / 2 + 1;              // == g.Cz
    constexpr int NT = 16 * T;
    float2* xb = ff_smem;
    float2* ib = xb + LB;                       // one exchange tile, used by the components in turn
    float* kb = reinterpret_cast<float*>(ib + 3 * NZ * 16);     // [6][CZ][16]
    const int tid = threadIdx.x, c = tid & 15, t = tid >> 4;
    const int ntx = (ct.ncol + 15) >> 4;
    const int nitem = ntx * (g.Py / 2 + 1);
    const size_t rstride = ct.b_plane, cstride = (size_t)g.Nz * ct.b_plane;
    const size_t nCk = (size_t)g.CxK * g.Cy * g.Cz;

    auto issue_in = [&](int bx, int other) {
        const float2* __restrict__ src0 = spec + (size_t)other * ct.b_row + bx * 16;
        for (int u = tid; u < 3 * NZ * 8; u += NT) {
            const int cu = u & 7, r = (u >> 3) % NZ, comp = (u >> 3) / NZ;
            const int left = ct.ncol - (bx * 16 + 2 * cu);
            const int nb = left >= 2 ? 16 : (left == 1 ? 8 : 0);
            const float2* src = nb ? src0 + comp * cstride + (size_t)r * rstride + 2 * cu : spec;
            cp_async16(ib + (comp * NZ + r) * 16 + 2 * cu, src, nb);
        }
    };
    auto issue_k = [&](int bx, int p) {
        const int kxb = ct.kx0 + bx * 16;
        for (int u = tid; u < 6 * CZ * 4; u += NT) {
            const int cu = u & 3, kz = (u >> 2) % CZ, comp = (u >> 2) / CZ;
            const int kx = kxb + 4 * cu;
            const int nb = kx < g.CxK ? 16 : 0;
            const float* src = nb ? khat + comp * nCk + ((size_t)kz * g.Cy + p) * g.CxK + kx : khat;
            cp_async16(kb + (comp * CZ + kz) * 16 + 4 * cu, src, nb);
        }
    };

    int q = blockIdx.x;
    if (q < nitem) { issue_k(q % ntx, q / ntx); issue_in(q % ntx, q / ntx); }
    cp_async_commit();
    cp_async_commit();                          // (empty) keeps "all but the newest group" == everything needed
    for (; q < nitem; q += gridDim.x) {
        const int bx = q % ntx, p = q / ntx;
        const int mir = (g.Py - p) % g.Py;
        const int nh = mir == p ? 1 : 2;
        const int qn = q + gridDim.x;
        const int col = bx * 16 + c;
        const bool valid = col < ct.ncol;
        for (int h = 0; h < nh; ++h) {
            const int other = h ? mir : p;
            const float so = h ? -1.f : 1.f;    // sign of the components odd in ky
            cp_async_wait<1>();
            __syncthreads();                    // this line set's spectrum tile has landed
            float2 v[3][E];
#pragma unroll
            for (int comp = 0; comp < 3; ++comp)
#pragma unroll
                for (int j = 0; j < NIO; ++j) v[comp][j] = ib[(comp * NZ + t + T * j) * 16 + c];
            __syncthreads();
            if (h + 1 < nh) issue_in(bx, mir);
            else if (qn < nitem) issue_in(qn % ntx, qn / ntx);
            cp_async_commit();
#pragma unroll
            for (int comp = 0; comp < 3; ++comp) {
                if (comp) __syncthreads();
                fft_line<T, E, -1, !PER>(v[comp], xb + c, 16, t, tw, SyncBlock());
            }
            cp_async_wait<1>();
            __syncthreads();                    // K^ tile of this pair has landed
#pragma unroll
            for (int j = 0; j < E; ++j) {
                int ka = t + T * j;
                float sz = 1.f;
                if (2 * ka > L) { ka = L - ka; sz = -1.f; }
                const float* kr = kb + ka * 16 + c;
                const float kxx = kr[0], kyy = kr[CZ * 16], kzz = kr[2 * CZ * 16];
                const float kxy = so * kr[3 * CZ * 16];
                const float kxz = sz * kr[4 * CZ * 16];
                const float kyz = so * sz * kr[5 * CZ * 16];
                const float2 mx = v[0][j], my = v[1][j], mz = v[2][j];
                v[0][j] = make_float2(kxx * mx.x + kxy * my.x + kxz * mz.x, kxx * mx.y + kxy * my.y + kxz * mz.y);
                v[1][j] = make_float2(kxy * mx.x + kyy * my.x + kyz * mz.x, kxy * mx.y + kyy * my.y + kyz * mz.y);
                v[2][j] = make_float2(kxz * mx.x + kyz * my.x + kzz * mz.x, kxz * mx.y + kyz * my.y + kzz * mz.y);
            }
            __syncthreads();                    // K^ tile and the forward exchange are free again
            if (h + 1 == nh && qn < nitem) issue_k(qn % ntx, qn / ntx);
            cp_async_commit();
#pragma unroll
            for (int comp = 0; comp < 3; ++comp) {
                if (comp) __syncthreads();
                fft_line<T, E, 1, false>(v[comp], xb + c, 16, t, tw, SyncBlock());
            }
            if (valid) {
                float2* __restrict__ base = spec + (size_t)other * ct.b_row + col;
#pragma unroll
                for (int comp = 0; comp < 3; ++comp)
#pragma unroll
                    for (int j = 0; j < NIO; ++j) base[comp * cstride + (size_t)(t + T * j) * rstride] = v[comp][j];
            }
        }
    }
    cp_async_wait<0>();
}

// ---------------------------------------------------------------------------------------------
// a5-a10: inverse x pass, complex -> real, and the fused epilogue.  T threads own one pair of rows
// (y0, y0+1) of one z plane and run the three components one after the other; the magnetostatic
// field of the pair goes to shared memory as float2 (row y0, row y0+1) per x, and the same threads
// then do the per-cell tail (exchange, anisotropy, Zeeman, thermal, torque, RK combine, max-norm).
// ---------------------------------------------------------------------------------------------
template <int T, int E, bool PER>
__global__ void __launch_bounds__(128)
k_inv_x(Geom g, const float2* __restrict__ specA, const float2* __restrict__ tw, EpiParams ep)
{
    constexpr int L = T * E;
    constexpr int LB = T * (E + 1);
    constexpr int NX = PER ? L : L / 2;        // == g.Nx
    constexpr int NOUT = PER ? E : E / 2;
    const int t = threadIdx.x % T;
    const int slot = threadIdx.x / T;
    const int nslot = 128 / T;
    float2* sb = ff_smem + slot * (LB + 2 * NX);
    float2* hb = sb + LB;                       // [2][NX] float2: components x, y (z reuses sb)
    const int npy = (g.Ny + 1) >> 1;
    const int npair = g.Nz * npy;
    const unsigned lane = threadIdx.x & 31;
    const unsigned lbase = lane - t;
    const unsigned srcl = lbase + ((T - t) % T);
    unsigned int red = 0u;
    for (int pb = blockIdx.x * nslot; pb < npair; pb += gridDim.x * nslot) {
        const bool act = pb + slot < npair;
        const int pp = act ? pb + slot : npair - 1;
        const int z = pp / npy, y0 = 2 * (pp - z * npy);
        const bool two = y0 + 1 < g.Ny;
#pragma unroll 1
        for (int comp = 0; comp < 3; ++comp) {
            const float2* __restrict__ a0 = specA + (((size_t)comp * g.Nz + z) * g.Ny + y0) * g.CxS;
            const float2* __restrict__ a1 = a0 + g.CxS;
            float2 v[E];
            // Z[k] = A[k] + i B[k] (k <= L/2),  Z[L-k] = conj A[k] + i conj B[k]
#pragma unroll
            for (int j = 0; j < E / 2; ++j) {
                const float2 A = a0[t + T * j];
                const float2 B = two ? a1[t + T * j] : make_float2(0.f, 0.f);
                v[j] = make_float2(A.x - B.y, A.y + B.x);
                v[E - 1 - j] = make_float2(A.x + B.y, B.x - A.y);      // belongs to thread T-t
            }
            float2 nyq = make_float2(0.f, 0.f);
            if (t == 0) {
                const float2 A = a0[L / 2];
                const float2 B = two ? a1[L / 2] : make_float2(0.f, 0.f);
                nyq = make_float2(A.x - B.y, A.y + B.x);
            }
            // thread 0 keeps its own mirrored values (k = T j' <-> L - T j' = T (E - j')), shifted by one
            // register; every other thread takes register E-1-j from thread T-t
            float2 own[E / 2];
#pragma unroll
            for (int j = 0; j < E / 2; ++j) own[j] = v[E - 1 - j];    // own[j] = Zrev of register j
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
            __syncwarp();
            fft_line<T, E, 1, false>(v, sb, 1, t, tw, SyncWarp());
            if (comp < 2) {
#pragma unroll
                for (int j = 0; j < NOUT; ++j) hb[comp * NX + t + T * j] = v[j];
            } else {
                __syncwarp();                   // the exchange buffer is free: it takes the z component
#pragma unroll
                for (int j = 0; j < NOUT; ++j) sb[t + T * j] = v[j];
            }
        }
        __syncwarp();
        if (act) {
            // per-cell tail, software-pipelined: the neighbour loads of x + T are issued before the
            // arithmetic and stores of x
            const PairGeom q = pair_geom(g, y0, z, two);
            PairNbr na, nb;
            pair_load(g, ep.m_in, q, t, two, na);
#pragma unroll 1
            for (int j = 0; j < NOUT; j += 2) {
                const int x0 = t + T * j, x1 = x0 + T;
                pair_load(g, ep.m_in, q, x1, two, nb);
                {
                    const float2 hx = hb[x0], hy = hb[NX + x0], hz = sb[x0];
                    red = max(red, __float_as_uint(pair_cell(ep, q, na, 0, x0, g.Nx, hx.x, hy.x, hz.x)) & 0x7fffffffu);
                    if (two)
                        red = max(red, __float_as_uint(pair_cell(ep, q, na, 1, x0, g.Nx, hx.y, hy.y, hz.y)) & 0x7fffffffu);
                }
                if (j + 2 < NOUT) pair_load(g, ep.m_in, q, x1 + T, two, na);
                {
                    const float2 hx = hb[x1], hy = hb[NX + x1], hz = sb[x1];
                    red = max(red, __float_as_uint(pair_cell(ep, q, nb, 0, x1, g.Nx, hx.x, hy.x, hz.x)) & 0x7fffffffu);
                    if (two)
                        red = max(red, __float_as_uint(pair_cell(ep, q, nb, 1, x1, g.Nx, hx.y, hy.y, hz.y)) & 0x7fffffffu);
                }
            }
        }
        __syncwarp();
    }
    if (ep.do_err) block_max_atomic(red, ep.maxbits);
}

// ---------------------------------------------------------------------------------------------
// a5 on its own (the "split" variant of the last pass): inverse x pass, complex -> real, cropped,
// scaled, written as a field [3][Nz][Ny][Nx]; k_epi4 then does the per-cell tail.  Same thread
// layout as k_fwd_x: T threads own one pair of rows of one (component, z).
// ---------------------------------------------------------------------------------------------
template <int T, int E, bool PER>
__global__ void __launch_bounds__(128)
k_inv_x_h(Geom g, const float2* __restrict__ specA, const float2* __restrict__ tw, float* __restrict__ out,
          float scale)
{
    constexpr int L = T * E;
    constexpr int LB = T * (E + 1);
    constexpr int NOUT = PER ? E : E / 2;
    const int t = threadIdx.x % T;
    const int slot = threadIdx.x / T;
    const int nslot = 128 / T;
    float2* sb = ff_smem + slot * LB;
    const int npy = (g.Ny + 1) >> 1;
    const int npair = 3 * g.Nz * npy;
    const unsigned lane = threadIdx.x & 31;
    const unsigned lbase = lane - t;
    const unsigned srcl = lbase + ((T - t) % T);
    for (int pb = blockIdx.x * nslot; pb < npair; pb += gridDim.x * nslot) {
        const bool act = pb + slot < npair;
        const int pp = act ? pb + slot : npair - 1;
        const int cz = pp / npy, y0 = 2 * (pp - cz * npy);
        const bool two = y0 + 1 < g.Ny;
        const float2* __restrict__ a0 = specA + ((size_t)cz * g.Ny + y0) * g.CxS;
        const float2* __restrict__ a1 = a0 + g.CxS;
        float2 v[E];
#pragma unroll
        for (int j = 0; j < E / 2; ++j) {
            const float2 A = a0[t + T * j];
            const float2 B = two ? a1[t + T * j] : make_float2(0.f, 0.f);
            v[j] = make_float2(A.x - B.y, A.y + B.x);
            v[E - 1 - j] = make_float2(A.x + B.y, B.x - A.y);
        }
        float2 nyq = make_float2(0.f, 0.f);
        if (t == 0) {
            const float2 A = a0[L / 2];
            const float2 B = two ? a1[L / 2] : make_float2(0.f, 0.f);
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
        __syncwarp();
        fft_line<T, E, 1, false>(v, sb, 1, t, tw, SyncWarp());
        float* __restrict__ o0 = out + ((size_t)cz * g.Ny + y0) * g.Nx;
        if (act) {
#pragma unroll
            for (int j = 0; j < NOUT; ++j) {
                o0[t + T * j] = scale * v[j].x;
                if (two) o0[g.Nx + t + T * j] = scale * v[j].y;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// a1 / a5 for x lengths Px = 2 Lc whose half Lc = T E has a register plan (1536 = 2 * 768,
// 2048 = 2 * 1024): the real transform of ONE row through a complex transform of half the length,
// z[n] = x[2n] + i x[2n+1] (read straight from the row as float2), then
//   X[k] = E[k] + w^k O[k],  E = (Z[k] + conj Z[Lc-k]) / 2,  O = (Z[k] - conj Z[Lc-k]) / (2i),  w = exp(-i pi / Lc)
// with the partner Z[Lc-k] taken from lane T-t, register E-1-j as in k_fwd_x.  twx[k] = w^k.
// ---------------------------------------------------------------------------------------------
template <int T, int E, bool PER>
__global__ void __launch_bounds__(128)
k_fwd_x_r(Geom g, const float* __restrict__ m, float2* __restrict__ specA, const float2* __restrict__ tw,
          const float2* __restrict__ twx)
{
    constexpr int Lc = T * E;
    constexpr int LB = T * (E + 1);
    constexpr int NIN = PER ? E : E / 2;
    const int t = threadIdx.x % T;
    const int slot = threadIdx.x / T;
    const int nslot = 128 / T;
    float2* sb = ff_smem + slot * LB;
    const int nrow = 3 * g.Nz * g.Ny;
    const unsigned lane = threadIdx.x & 31;
    const unsigned src = lane - t + ((T - t) % T);
    for (int rb = blockIdx.x * nslot; rb < nrow; rb += gridDim.x * nslot) {
        const bool act = rb + slot < nrow;
        const int row = act ? rb + slot : nrow - 1;
        const float2* __restrict__ r0 = reinterpret_cast<const float2*>(m + (size_t)row * g.Nx);
        float2 v[E];
#pragma unroll
        for (int j = 0; j < NIN; ++j) v[j] = r0[t + T * j];
        __syncwarp();
        fft_line<T, E, -1, !PER>(v, sb, 1, t, tw, SyncWarp());
        float2* __restrict__ o = specA + (size_t)row * g.CxS;
#pragma unroll
        for (int j = 0; j < E; ++j) {
            float2 p;
            p.x = __shfl_sync(0xffffffffu, v[E - 1 - j].x, src);
            p.y = __shfl_sync(0xffffffffu, v[E - 1 - j].y, src);
            if (t == 0) p = v[(E - j) % E];
            const float2 z = v[j];
            const float2 ek = make_float2(0.5f * (z.x + p.x), 0.5f * (z.y - p.y));
            const float2 ok = make_float2(0.5f * (z.y + p.y), 0.5f * (p.x - z.x));
            const float2 w = __ldg(twx + t + T * j);
            if (act) o[t + T * j] = cadd(ek, cmul(w, ok));
        }
        if (t == 0 && act) o[Lc] = make_float2(v[0].x - v[0].y, 0.f);
    }
}

template <int T, int E, bool PER>
__global__ void __launch_bounds__(128)
k_inv_x_h_r(Geom g, const float2* __restrict__ specA, const float2* __restrict__ tw,
            const float2* __restrict__ twx, float* __restrict__ out, float scale)
{
    constexpr int Lc = T * E;
    constexpr int LB = T * (E + 1);
    constexpr int NOUT = PER ? E : E / 2;
    const int t = threadIdx.x % T;
    const int slot = threadIdx.x / T;
    const int nslot = 128 / T;
    float2* sb = ff_smem + slot * LB;
    const int nrow = 3 * g.Nz * g.Ny;
    const unsigned lane = threadIdx.x & 31;
    const unsigned src = lane - t + ((T - t) % T);
    for (int rb = blockIdx.x * nslot; rb < nrow; rb += gridDim.x * nslot) {
        const bool act = rb + slot < nrow;
        const int row = act ? rb + slot : nrow - 1;
        const float2* __restrict__ a0 = specA + (size_t)row * g.CxS;
        float2 x[E], v[E];
#pragma unroll
        for (int j = 0; j < E; ++j) x[j] = a0[t + T * j];
        float2 xn = make_float2(0.f, 0.f);
        if (t == 0) xn = a0[Lc];
        // 2 Z[k] = (X[k] + conj X[Lc-k]) + i conj(w^k) (X[k] - conj X[Lc-k])
#pragma unroll
        for (int j = 0; j < E; ++j) {
            float2 p;
            p.x = __shfl_sync(0xffffffffu, x[E - 1 - j].x, src);
            p.y = __shfl_sync(0xffffffffu, x[E - 1 - j].y, src);
            if (t == 0) p = j == 0 ? xn : x[(E - j) % E];
            const float2 z = x[j];
            const float2 e2 = make_float2(z.x + p.x, z.y - p.y);
            const float2 d = make_float2(z.x - p.x, z.y + p.y);
            const float2 w = cconj(__ldg(twx + t + T * j));
            const float2 o2 = cmul(w, d);
            v[j] = make_float2(e2.x - o2.y, e2.y + o2.x);
        }
        __syncwarp();
        fft_line<T, E, 1, false>(v, sb, 1, t, tw, SyncWarp());
        float2* __restrict__ o = reinterpret_cast<float2*>(out + (size_t)row * g.Nx);
        if (act) {
#pragma unroll
            for (int j = 0; j < NOUT; ++j) o[t + T * j] = make_float2(scale * v[j].x, scale * v[j].y);
        }
    }
}

}  // namespace ff
}  // namespace mm

