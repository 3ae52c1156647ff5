// fft_packed.cuh -- "sibling-packed" register FFT codelets and the TMA helpers of the last-axis pass.
//
// Two independent sub-transforms that share their twiddles (siblings a, b) are carried in ONE set of
// registers: a packed complex value is {re = (re_a, re_b), im = (im_a, im_b)}, so that every butterfly is
// a packed f32x2 instruction (FADD2 / FMUL2 / FFMA2 on sm_100: two lanes per issue slot) and a
// multiplication by +-i costs nothing (the re / im registers swap roles).  Where the recursion has to
// combine the two siblings with each other, one level is done on the scalar halves; such a level can
// re-pair its outputs for free, because each half of a pair is an ordinary 32-bit register.
//
// Product code; shares nothing with oracle/.  (the transforms of the convolution.)
#pragma once
#include <cuda.h>            // CUtensorMap (types only; the encoder is fetched through the runtime)
#include <cuda_runtime.h>
#include "ptx_async.cuh"

namespace mm {
namespace pk {

struct P2 { float2 re, im; };      // one complex value of each of the two siblings

__device__ __forceinline__ float2 f2(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ float2 neg(float2 a) { return make_float2(-a.x, -a.y); }       // folds into the operand
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __fadd2_rn(a, neg(b)); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 bc(float s) { return make_float2(s, s); }               // scalar operand, both lanes

__device__ __forceinline__ P2 padd(P2 a, P2 b) { return { add2(a.re, b.re), add2(a.im, b.im) }; }
__device__ __forceinline__ P2 psub(P2 a, P2 b) { return { sub2(a.re, b.re), sub2(a.im, b.im) }; }
// a + SGN i b  and  a - SGN i b
template <int SGN>
__device__ __forceinline__ P2 padd_i(P2 a, P2 b)
{
    return SGN > 0 ? P2{ sub2(a.re, b.im), add2(a.im, b.re) } : P2{ add2(a.re, b.im), sub2(a.im, b.re) };
}
template <int SGN>
__device__ __forceinline__ P2 psub_i(P2 a, P2 b) { return padd_i<-SGN>(a, b); }

// in-place DFT of 4 packed values, natural order; SGN = -1 forward (exp(-i...)), +1 inverse
template <int SGN>
__device__ __forceinline__ void fft4(P2& v0, P2& v1, P2& v2, P2& v3)
{
    const P2 a = padd(v0, v2), b = psub(v0, v2), c = padd(v1, v3), d = psub(v1, v3);
    v0 = padd(a, c);
    v2 = psub(a, c);
    v1 = padd_i<SGN>(b, d);
    v3 = psub_i<SGN>(b, d);
}

// in-place DFT of 8 packed values, natural order (decimation in time): 52 packed instructions
template <int SGN>
__device__ __forceinline__ void fft8(P2 (&v)[8])
{
    constexpr float C = 0.70710678118654752440f;
    fft4<SGN>(v[0], v[2], v[4], v[6]);      // even inputs -> e[0..3] in v[0], v[2], v[4], v[6]
    fft4<SGN>(v[1], v[3], v[5], v[7]);      // odd inputs  -> o[0..3] in v[1], v[3], v[5], v[7]
    const P2 e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6];
    const P2 o0 = v[1], o1 = v[3], o2 = v[5], o3 = v[7];
    // K = 0: w = 1
    v[0] = padd(e0, o0);
    v[4] = psub(e0, o0);
    // K = 2: w = SGN i
    v[2] = padd_i<SGN>(e2, o2);
    v[6] = psub_i<SGN>(e2, o2);
    // K = 1: w = C (1 + SGN i):  w o = C ((x - SGN y) + i (y + SGN x))
    {
        const float2 tr = SGN > 0 ? sub2(o1.re, o1.im) : add2(o1.re, o1.im);
        const float2 ti = SGN > 0 ? add2(o1.im, o1.re) : sub2(o1.im, o1.re);
        v[1] = { fma2(tr, bc(C), e1.re), fma2(ti, bc(C), e1.im) };
        v[5] = { fma2(tr, bc(-C), e1.re), fma2(ti, bc(-C), e1.im) };
    }
    // K = 3: w = C (-1 + SGN i):  w o = -C ((x + SGN y) + i (y - SGN x))
    {
        const float2 tr = SGN > 0 ? add2(o3.re, o3.im) : sub2(o3.re, o3.im);
        const float2 ti = SGN > 0 ? sub2(o3.im, o3.re) : add2(o3.im, o3.re);
        v[3] = { fma2(tr, bc(-C), e3.re), fma2(ti, bc(-C), e3.im) };
        v[7] = { fma2(tr, bc(C), e3.re), fma2(ti, bc(C), e3.im) };
    }
}

// v *= (c + i SGN_S s) per lane: tw = (c_a, c_b, s_a, s_b) of the FORWARD twiddle exp(-i phi) = (cos, -sin)
// stored as (cos phi, sin phi) >= the caller picks the direction: CONJ = false multiplies by (c - i s)
// (forward), CONJ = true by (c + i s) (inverse).
template <bool CONJ>
__device__ __forceinline__ P2 ptwiddle(P2 v, float4 tw)
{
    const float2 c = f2(tw.x, tw.y), s = f2(tw.z, tw.w);
    P2 r;
    if (CONJ) {          // (re + i im)(c + i s) = (re c - im s) + i (im c + re s)
        r.re = fma2(neg(v.im), s, mul2(v.re, c));
        r.im = fma2(v.re, s, mul2(v.im, c));
    } else {             // (re + i im)(c - i s) = (re c + im s) + i (im c - re s)
        r.re = fma2(v.im, s, mul2(v.re, c));
        r.im = fma2(neg(v.re), s, mul2(v.im, c));
    }
    return r;
}

// (mbarrier / TMA helpers: ptx_async.cuh)


// ---------------------------------------------------------------------------------------------
// a3 (3D grids, padded z length 128): z forward -> H^ = K^ M^ -> z inverse, in place, for work items of
// 16 kx columns x one ky pair {p, Py - p} (same items, same octant handling as ff::k_mid_p).
//
// Index split of one line: n = 8 n1 + n2 (thread t = n2 holds rows t + 8 n1: standard form), k = k2 + 16 k1.
//   forward: FFT16 over n1 (rows >= Nz are zero: one decimation-in-frequency level gives the sibling
//            inputs x and x w16^n1, then ONE packed FFT8 whose lanes are k2 = 2k, 2k+1), twiddle
//            w128^(n2 k2), exchange (64-bit, planar re / im pairs, conflict free), packed FFT8 over n2 -> lanes k2 = 2t, 2t+1 of
//            thread t, register k1.
//   multiply: per register k1 the two lanes are kz = 2t + 16 k1 (+1); K^ from the octant tile in shared
//            memory (mirrored index and sign for kz > 64).
//   inverse: packed FFT8 over k1, conjugate twiddle, exchange, packed FFT8 over even / odd k2 (the two
//            lanes), and one scalar level x[n1] = E[n1] + w16^-n1 O[n1] that keeps only rows < Nz.
// The spectrum tile [3][Nz][16] and the K^ tile [2][6][33][16] (even / odd kz) of the NEXT item arrive by TMA
// (cp.async.bulk.tensor, one instruction each, completion on an mbarrier) while the current one is
// transformed.  block = 128 threads (c = tid & 15 column, t = tid >> 4); persistent grid.
// twp[a * 8 + b] = (cos, cos', sin, sin') of the angles 2 pi a (2b) / 128 and 2 pi a (2b + 1) / 128.
// ---------------------------------------------------------------------------------------------
extern __shared__ __align__(1024) unsigned char pk_smem[];

template <bool PER, int C>
struct MidT {
    static constexpr int T = 8, E = 16, L = 128;
    static constexpr int NZ = PER ? L : L / 2;
    static constexpr int CZ = L / 2 + 1;
    static constexpr int NIO = PER ? E : E / 2;
    static constexpr int RS = 8 * C + (C == 8 ? 8 : 0);   // exchange row stride (float2): rows t, t + 1 on different bank halves
    static constexpr int XP = 8 * RS;                     // float2 per exchange plane (re pairs | im pairs)
    static constexpr unsigned XB_BYTES = 2 * XP * 8;
    static constexpr unsigned IB_BYTES = 3 * NZ * C * 8;
    static constexpr int CH = CZ / 2 + 1;          // rows of one kz-parity half of the K^ tile
    static constexpr unsigned KB_BYTES = 2 * 6 * CH * C * 4;
    static constexpr unsigned SMEM_BYTES = XB_BYTES + IB_BYTES + KB_BYTES + 64;
};

template <bool PER, int C, bool PANEL>
__global__ void __launch_bounds__(8 * C, (PER ? 2 : 3) * (16 / C))
k_mid_t(const __grid_constant__ CUtensorMap map_s, const __grid_constant__ CUtensorMap map_k, Geom g,
        float2* __restrict__ spec, const float4* __restrict__ twp)
{
    using M = MidT<PER, C>;
    constexpr int NZ = M::NZ, CH = M::CH, NIO = M::NIO, L = M::L;
    float2* xb = reinterpret_cast<float2*>(pk_smem);         // exchange tile: plane of re pairs, plane of im pairs
    const float2* ib = reinterpret_cast<const float2*>(pk_smem + M::XB_BYTES);
    const float* kb = reinterpret_cast<const float*>(pk_smem + M::XB_BYTES + M::IB_BYTES);
    unsigned long long* bar = reinterpret_cast<unsigned long long*>(pk_smem + M::XB_BYTES + M::IB_BYTES + M::KB_BYTES);
    const int tid = threadIdx.x, c = tid % C, t = tid / C;
    const int ntx = (g.Cx + C - 1) / C;
    const int nitem = ntx * (g.Py / 2 + 1);
    // PANEL: specB is [panel][3][Nz][Py][16] (mm_kernels.h panel_tile) and consecutive items are consecutive ky
    const int npair = g.Py / 2 + 1;
    const size_t rstride = PANEL ? (size_t)g.Py * 16 : (size_t)g.Py * g.CxS;
    const size_t cstride = (size_t)g.Nz * rstride, step8 = 8 * rstride;

    if (tid == 0) {
        tma_prefetch_desc(&map_s);
        tma_prefetch_desc(&map_k);
        mbar_init(bar, 1);
        mbar_init(bar + 1, 1);
        mbar_fence_init();
    }
    __syncthreads();
    auto issue_in = [&](int bx, int other) {
        mbar_expect_tx(bar, M::IB_BYTES);
        if (PANEL) tma_load_5d(const_cast<float2*>(ib), &map_s, bar, 0, other, 0, 0, bx);
        else tma_load_4d(const_cast<float2*>(ib), &map_s, bar, 2 * C * bx, other, 0, 0);
    };
    auto issue_k = [&](int bx, int p) {
        mbar_expect_tx(bar + 1, M::KB_BYTES);
        tma_load_5d(const_cast<float*>(kb), &map_k, bar + 1, C * bx, p, 0, 0, 0);
    };
    // item order.  Plain rows: column tile fastest.  Panels: ky fastest within a PAIR of adjacent panels (bx = 2g, 2g + 1
    // alternate): the spectrum rows of consecutive items are adjacent in each panel, and the two K^ tiles that share
    // 128-byte lines are read one after the other (ky fastest over single panels left half of every K^ line unused
    // until 500 items later: ncu showed 1673 MB read per launch instead of 1255 MB).
    const int npp = 2 * npair * (ntx / 2);       // items of the whole panel pairs; an odd last panel follows alone
    auto item_bx = [&](int i) { return !PANEL ? i % ntx : (i < npp ? 2 * (i / (2 * npair)) + (i & 1) : ntx - 1); };
    auto item_p = [&](int i) { return !PANEL ? i / ntx : (i < npp ? (i % (2 * npair)) >> 1 : i - npp); };
    int q = blockIdx.x;
    if (tid == 0 && q < nitem) { issue_k(item_bx(q), item_p(q)); issue_in(item_bx(q), item_p(q)); }
    unsigned par_in = 0, par_k = 0;
    // per-thread bases of the exchange tile (writer row t / reader column t) and of the K^ tile
    constexpr int XP = M::XP, RS = M::RS;
    float2* xw = xb + t * RS + c;                // + k * C   : entry (row t, column k); + XP: im pair
    float2* xr = xb + t * C + c;                 // + n * RS  : entry (row n, column t)
    // K^ tile [parity of kz][component][kz >> 1][16]: a warp's two thread rows t, t + 1 then read rows 64 bytes
    // apart (no bank conflict); direct rows kz = 2t + 16 k1 (+1), mirrored rows 128 - kz
    const float* kd = kb + c + C * t;
    const float* km = kb + c - C * t;
    const float4* twf = twp + t * 8;             // forward: row t
    const float4* twi = twp + t;                 // inverse: column t (stride 8)

    for (; q < nitem; q += gridDim.x) {
        const int bx = item_bx(q), p = item_p(q);
        const int mir = (g.Py - p) % g.Py;
        const int nh = mir == p ? 1 : 2;
        const int qn = q + gridDim.x;
        const int col = bx * C + c;
        const bool valid = col < g.Cx;
        for (int h = 0; h < nh; ++h) {
            const int other = h ? mir : p;
            const float so = h ? -1.f : 1.f;     // sign of the components odd in ky
            P2 V[3][8];
            mbar_wait(bar, par_in);
            par_in ^= 1u;
            float2 x[3][NIO];
#pragma unroll
            for (int comp = 0; comp < 3; ++comp)
#pragma unroll
                for (int j = 0; j < NIO; ++j) x[comp][j] = ib[(comp * NZ + t + 8 * j) * C + c];
            __syncthreads();                     // the spectrum tile is in registers: refill it
            if (tid == 0) {
                if (h + 1 < nh) issue_in(bx, mir);
                else if (qn < nitem) issue_in(item_bx(qn), item_p(qn));
            }
            // ---------------- forward ----------------
            // Software-pipelined over the components: the read-back of component c is issued, then the first
            // register FFT of component c + 1 runs while it lands, and the second register FFT of component c
            // runs after the next exchange write -- shared-memory and FP phases of one warp interleave.
            auto fwd_first = [&](int comp, P2 (&A)[8]) {
#pragma unroll
                for (int n = 0; n < 8; ++n) {
                    float2 a, d;
                    if (PER) { a = make_float2(x[comp][n].x + x[comp][n + NIO / 2].x, x[comp][n].y + x[comp][n + NIO / 2].y);
                               d = make_float2(x[comp][n].x - x[comp][n + NIO / 2].x, x[comp][n].y - x[comp][n + NIO / 2].y); }
                    else { a = x[comp][n]; d = a; }
                    // b = d * exp(-2 pi i n / 16) = (d.x cs + d.y sn, d.y cs - d.x sn)
                    float2 b;
                    if (n == 0) b = d;
                    else if (n == 4) b = make_float2(d.y, -d.x);
                    else {
                        const float cs = ff::cos32(2 * n), sn = ff::sin32(2 * n);
                        b = make_float2(fmaf(d.y, sn, d.x * cs), fmaf(-d.x, sn, d.y * cs));
                    }
                    A[n].re = make_float2(a.x, b.x);
                    A[n].im = make_float2(a.y, b.y);
                }
                fft8<-1>(A);                     // A[k] lanes: Y[2k], Y[2k+1]
#pragma unroll
                for (int k = 0; k < 8; ++k) A[k] = ptwiddle<false>(A[k], __ldg(twf + k));
            };
            auto put_rows = [&](const P2 (&A)[8]) {      // entry (row t, column k)
#pragma unroll
                for (int k = 0; k < 8; ++k) { xw[k * C] = A[k].re; xw[XP + k * C] = A[k].im; }
            };
            auto get_cols = [&](P2 (&B)[8]) {            // entry (row n, column t)
#pragma unroll
                for (int n = 0; n < 8; ++n) { B[n].re = xr[n * RS]; B[n].im = xr[XP + n * RS]; }
            };
            {
                P2 A[8];
                fwd_first(0, A);
                put_rows(A);
                __syncthreads();
                get_cols(V[0]);
                fwd_first(1, A);
                __syncthreads();                 // component 0 has been read back by every thread
                put_rows(A);
                fft8<-1>(V[0]);                  // V[comp][k1] lanes: kz = 2t + 16 k1, 2t + 1 + 16 k1
                __syncthreads();
                get_cols(V[1]);
                fwd_first(2, A);
                __syncthreads();
                put_rows(A);
                fft8<-1>(V[1]);
                __syncthreads();
                get_cols(V[2]);
                fft8<-1>(V[2]);
            }
            // ---------------- multiply ----------------
            if (h == 0) { mbar_wait(bar + 1, par_k); par_k ^= 1u; }
            {
                const float2 so2 = make_float2(so, so);
#pragma unroll
                for (int k1 = 0; k1 < 8; ++k1) {
                    float2 kk[6];
                    if (k1 < 4) {
#pragma unroll
                        for (int i = 0; i < 6; ++i)
                            kk[i] = make_float2(kd[(i * CH + 8 * k1) * C], kd[((6 + i) * CH + 8 * k1) * C]);
                    } else {
#pragma unroll
                        for (int i = 0; i < 6; ++i)
                            kk[i] = make_float2(km[(i * CH + L / 2 - 8 * k1) * C], km[((6 + i) * CH + L / 2 - 1 - 8 * k1) * C]);
                    }
                    float2 kxy = mul2(kk[3], so2), kxz = kk[4], kyz = mul2(kk[5], so2);
                    if (k1 >= 4) {
                        // kz > 64: mirrored entry, components odd in kz change sign (kz = 64 itself does not)
                        const float2 sz = make_float2((k1 == 4 && t == 0) ? 1.f : -1.f, -1.f);
                        kxz = mul2(kxz, sz);
                        kyz = mul2(kyz, sz);
                    }
                    const P2 mx = V[0][k1], my = V[1][k1], mz = V[2][k1];
                    V[0][k1].re = fma2(kxz, mz.re, fma2(kxy, my.re, mul2(kk[0], mx.re)));
                    V[0][k1].im = fma2(kxz, mz.im, fma2(kxy, my.im, mul2(kk[0], mx.im)));
                    V[1][k1].re = fma2(kyz, mz.re, fma2(kk[1], my.re, mul2(kxy, mx.re)));
                    V[1][k1].im = fma2(kyz, mz.im, fma2(kk[1], my.im, mul2(kxy, mx.im)));
                    V[2][k1].re = fma2(kk[2], mz.re, fma2(kyz, my.re, mul2(kxz, mx.re)));
                    V[2][k1].im = fma2(kk[2], mz.im, fma2(kyz, my.im, mul2(kxz, mx.im)));
                }
            }
            __syncthreads();                     // K^ tile and the forward exchange are free again
            if (tid == 0 && h + 1 == nh && qn < nitem) issue_k(item_bx(qn), item_p(qn));
            // ---------------- inverse ----------------
            // rows t, t + 8, ... of this column: pointer increments instead of 64-bit multiplies per store
            float2* op = PANEL ? spec + (size_t)bx * (3 * cstride) + (size_t)other * 16 + c + (size_t)t * rstride
                                            : spec + (size_t)other * g.CxS + col + (size_t)t * rstride;
            auto inv_first = [&](int comp) {
                fft8<1>(V[comp]);                // V[comp][n2] lanes: k2 = 2t, 2t + 1
#pragma unroll
                for (int n = 0; n < 8; ++n) V[comp][n] = ptwiddle<true>(V[comp][n], __ldg(twi + n * 8));
            };
            auto put_cols = [&](const P2 (&B)[8]) {
#pragma unroll
                for (int n = 0; n < 8; ++n) { xr[n * RS] = B[n].re; xr[XP + n * RS] = B[n].im; }
            };
            auto get_rows = [&](P2 (&R)[8]) {
#pragma unroll
                for (int k = 0; k < 8; ++k) { R[k].re = xw[k * C]; R[k].im = xw[XP + k * C]; }
            };
            auto inv_last = [&](P2 (&R)[8], int comp) {
                fft8<1>(R);                      // R[n1] lanes: E[n1] (even k2), O[n1] (odd k2)
                // x[n1] = E + w O, x[n1 + 8] = E - w O, w = exp(+2 pi i n1 / 16); row = t + 8 n1
                float2 o[NIO];
#pragma unroll
                for (int n = 0; n < 8; ++n) {
                    const float er = R[n].re.x, ei = R[n].im.x, pr = R[n].re.y, pi = R[n].im.y;
                    float wr, wi;                // w O
                    if (n == 0) { wr = pr; wi = pi; }
                    else if (n == 4) { wr = -pi; wi = pr; }
                    else {
                        const float cs = ff::cos32(2 * n), sn = ff::sin32(2 * n);
                        wr = fmaf(-pi, sn, pr * cs);
                        wi = fmaf(pr, sn, pi * cs);
                    }
                    o[n] = make_float2(er + wr, ei + wi);
                    if (PER) o[n + 8] = make_float2(er - wr, ei - wi);
                }
                if (valid) {
                    float2* __restrict__ oc = op + comp * cstride;
#pragma unroll
                    for (int n = 0; n < NIO; ++n) oc[n * step8] = o[n];
                }
            };
            {
                P2 R[8];
                inv_first(0);
                put_cols(V[0]);
                __syncthreads();
                get_rows(R);
                inv_first(1);
                __syncthreads();
                put_cols(V[1]);
                inv_last(R, 0);
                __syncthreads();
                get_rows(R);
                inv_first(2);
                __syncthreads();
                put_cols(V[2]);
                inv_last(R, 1);
                __syncthreads();
                get_rows(R);
                inv_last(R, 2);
            }
        }
    }
}

}  // namespace pk
}  // namespace mm
