// fft_fast.cuh -- size-specialised register FFT passes for padded lengths 64..1024 (powers of two).
//
// Every line transform of length L = T * E is done by T threads that hold E complex values each
// ("standard form": thread t holds elements t + T j in register j), as two register FFTs (length E,
// then length T) with ONE exchange through shared memory in between ("1D FFT sets per
// axis"; the zero-padded half is never loaded and the cropped half never stored).
// Layouts are those of mm_common.cuh, so each fast pass is interchangeable with its generic
// counterpart of fft_generic.cuh (mm_set_fast_path takes a bit mask).
//
// Product code; shares nothing with oracle/.
#pragma once
#include <string>
#include <vector>
#include "mm_common.cuh"
#include "epilogue.cuh"
#include "ptx_async.cuh"

namespace mm {
namespace ff {

// cos(2 pi j / 32) and sin(2 pi j / 32) as compile-time constants
__host__ __device__ constexpr float cos32(int j)
{
    j &= 31;
    if (j > 16) j = 32 - j;
    bool neg = false;
    if (j > 8) { j = 16 - j; neg = true; }
    const float t[9] = { 1.0f, 0.98078528040323044913f, 0.92387953251128675613f, 0.83146961230254523708f,
                         0.70710678118654752440f, 0.55557023301960222474f, 0.38268343236508977173f,
                         0.19509032201612826785f, 0.0f };
    return neg ? -t[j] : t[j];
}
__host__ __device__ constexpr float sin32(int j) { return cos32(j - 8); }

// cos(2 pi j / 48) and sin(2 pi j / 48): the lengths with one factor 3 (24, 48)
__host__ __device__ constexpr float cos48(int j)
{
    j %= 48;
    if (j < 0) j += 48;
    if (j > 24) j = 48 - j;
    bool neg = false;
    if (j > 12) { j = 24 - j; neg = true; }
    const float t[13] = { 1.0f, 0.9914448613738104f, 0.9659258262890683f, 0.9238795325112867f, 0.8660254037844387f, 0.7933533402912352f, 0.7071067811865476f, 0.6087614290087207f, 0.5000000000000001f, 0.38268343236508984f, 0.25881904510252074f, 0.1305261922200517f, 0.0f };
    return neg ? -t[j] : t[j];
}
__host__ __device__ constexpr float sin48(int j) { return cos48(j - 12); }

// real and imaginary part of exp(2 pi i k / N) for N dividing 32 or 48
template <int N>
__host__ __device__ constexpr float cosN(int k) { return 32 % N == 0 ? cos32(k * (32 / (32 % N == 0 ? N : 1))) : cos48(k * (48 / N)); }
template <int N>
__host__ __device__ constexpr float sinN(int k) { return 32 % N == 0 ? sin32(k * (32 / (32 % N == 0 ? N : 1))) : sin48(k * (48 / N)); }

template <int N, int SGN>
__device__ __forceinline__ void fft_reg(float2 (&v)[N]);

// complex add / subtract of two values that already sit in register pairs: one packed f32x2
// instruction each on sm_100 (halves the issue slots of the trivial butterflies)
#ifndef MM_NO_PACKED_F32X2
__device__ __forceinline__ float2 padd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 psub(float2 a, float2 b) { return __ffma2_rn(b, make_float2(-1.f, -1.f), a); }
#else
__device__ __forceinline__ float2 padd(float2 a, float2 b) { return cadd(a, b); }
__device__ __forceinline__ float2 psub(float2 a, float2 b) { return csub(a, b); }
#endif

// last level of the decimation-in-time recursion: v[K] = e[K] + w^K o[K], v[K + N/2] = e[K] - w^K o[K]
template <int N, int SGN, int K>
__device__ __forceinline__ void dit_combine(float2 (&v)[N], const float2 (&e)[N / 2], const float2 (&o)[N / 2])
{
    if constexpr (K < N / 2) {
        if constexpr (K == 0) {
            v[0] = padd(e[0], o[0]);
            v[N / 2] = psub(e[0], o[0]);
        } else if constexpr (4 * K == N) {
            const float2 t = cmuli<SGN>(o[K]);
            v[K] = cadd(e[K], t);
            v[K + N / 2] = csub(e[K], t);
        } else {
            constexpr float c = cos32(K * (32 / N));
            constexpr float s = SGN * sin32(K * (32 / N));      // w^K = (c, s)
            float2 a;
            a.x = fmaf(c, o[K].x, e[K].x);
            a.x = fmaf(-s, o[K].y, a.x);
            a.y = fmaf(c, o[K].y, e[K].y);
            a.y = fmaf(s, o[K].x, a.y);
            v[K] = a;
            v[K + N / 2] = make_float2(fmaf(2.0f, e[K].x, -a.x), fmaf(2.0f, e[K].y, -a.y));
        }
        dit_combine<N, SGN, K + 1>(v, e, o);
    }
}

// top level of a length N = 3 M transform (decimation in time by 3): v[k + M m] = sum_r w3^(r m) w_N^(r k) e_r[k]
template <int N, int SGN, int K>
__device__ __forceinline__ void dit3_combine(float2 (&v)[N], const float2 (&e0)[N / 3], const float2 (&e1)[N / 3],
                                             const float2 (&e2)[N / 3])
{
    constexpr int M = N / 3;
    if constexpr (K < M) {
        float2 b = e1[K], c = e2[K];
        if constexpr (K > 0) {
            constexpr float c1 = cosN<N>(K), s1 = SGN * sinN<N>(K);
            constexpr float c2 = cosN<N>(2 * K), s2 = SGN * sinN<N>(2 * K);
            b = make_float2(fmaf(c1, b.x, -s1 * b.y), fmaf(c1, b.y, s1 * b.x));
            c = make_float2(fmaf(c2, c.x, -s2 * c.y), fmaf(c2, c.y, s2 * c.x));
        }
        const float S = 0.86602540378443864676f;
        const float2 a = e0[K];
        const float2 s = padd(b, c);
        const float2 d = cmuli<SGN>(cscale(psub(b, c), S));
        const float2 m = make_float2(fmaf(-0.5f, s.x, a.x), fmaf(-0.5f, s.y, a.y));
        v[K] = padd(a, s);
        v[K + M] = cadd(m, d);
        v[K + 2 * M] = csub(m, d);
        dit3_combine<N, SGN, K + 1>(v, e0, e1, e2);
    }
}

// in-place DFT of N = 2, 4, 8, 16, 32 or 24, 48 register values, natural order in and out
template <int N, int SGN>
__device__ __forceinline__ void fft_reg(float2 (&v)[N])
{
    static_assert(N == 2 || N == 4 || N == 8 || N == 16 || N == 32 || N == 12 || N == 24 || N == 48, "register FFT size");
    if constexpr (N % 3 == 0) {
        constexpr int M = N / 3;
        float2 e0[M], e1[M], e2[M];
#pragma unroll
        for (int i = 0; i < M; ++i) { e0[i] = v[3 * i]; e1[i] = v[3 * i + 1]; e2[i] = v[3 * i + 2]; }
        fft_reg<M, SGN>(e0);
        fft_reg<M, SGN>(e1);
        fft_reg<M, SGN>(e2);
        dit3_combine<N, SGN, 0>(v, e0, e1, e2);
    } else if constexpr (N == 2) {
        const float2 a = v[0], b = v[1];
        v[0] = padd(a, b);
        v[1] = psub(a, b);
    } else if constexpr (N == 4) {
        const float2 a = padd(v[0], v[2]), b = psub(v[0], v[2]);
        const float2 c = padd(v[1], v[3]), d = cmuli<SGN>(psub(v[1], v[3]));
        v[0] = padd(a, c);
        v[1] = cadd(b, d);
        v[2] = psub(a, c);
        v[3] = csub(b, d);
    } else {
        float2 e[N / 2], o[N / 2];
#pragma unroll
        for (int i = 0; i < N / 2; ++i) { e[i] = v[2 * i]; o[i] = v[2 * i + 1]; }
        fft_reg<N / 2, SGN>(e);
        fft_reg<N / 2, SGN>(o);
        dit_combine<N, SGN, 0>(v, e, o);
    }
}

template <int N, int SGN, int K>
__device__ __forceinline__ void half_twiddle(float2 (&b)[N / 2])
{
    if constexpr (K < N / 2) {
        if constexpr (4 * K == N) {
            b[K] = cmuli<SGN>(b[K]);
        } else if constexpr (K > 0) {
            constexpr float c = cosN<N>(K);
            constexpr float s = SGN * sinN<N>(K);
            const float2 x = b[K];
            b[K] = make_float2(fmaf(c, x.x, -s * x.y), fmaf(c, x.y, s * x.x));
        }
        half_twiddle<N, SGN, K + 1>(b);
    }
}

// DFT of N values of which v[N/2..N-1] are zero (not read): one decimation-in-frequency level,
// X[2k] = FFT_{N/2}(x)[k], X[2k+1] = FFT_{N/2}(x w^n)[k]
template <int N, int SGN>
__device__ __forceinline__ void fft_reg_half(float2 (&v)[N])
{
    float2 a[N / 2], b[N / 2];
#pragma unroll
    for (int i = 0; i < N / 2; ++i) { a[i] = v[i]; b[i] = v[i]; }
    half_twiddle<N, SGN, 0>(b);
    fft_reg<N / 2, SGN>(a);
    fft_reg<N / 2, SGN>(b);
#pragma unroll
    for (int i = 0; i < N / 2; ++i) { v[2 * i] = a[i]; v[2 * i + 1] = b[i]; }
}

// Inter-stage twiddles v[k2] *= w^(t k2), w = exp(SGN' 2 pi i / (T E)), from the table tw[k2 * T + t] (forward
// sign; CONJ takes the conjugate).  For E >= 16 only k2 <= E/4 and k2 = E/2 are loaded; the others follow from
//   w^(t (E/2 + k)) = d w^(t k),  w^(t (E/2 - k)) = d conj(w^(t k)),  w^(t (E - k)) = d^2 conj(w^(t k)),  d = w^(t E/2)
// -- 9 loads instead of 31 for E = 32 at the price of a few dozen FMAs: the passes that wait on these loads
// (long-scoreboard stalls with every register taken by the line) have FP slots to spare (measured: y passes 3 %
// faster, x passes unchanged; -DMM_TW_PLAIN restores one load per element).
template <int T, int E, bool CONJ>
__device__ __forceinline__ void apply_twiddles(float2 (&v)[E], const float2* __restrict__ tw, const int t)
{
#if !defined(MM_TW_PLAIN)
    constexpr bool SYM = E % 4 == 0 && E >= 16;
#else
    constexpr bool SYM = false;
#endif
    if constexpr (SYM) {
        auto ld = [&](int k2) { float2 w = __ldg(tw + k2 * T + t); if (CONJ) w.y = -w.y; return w; };
        const float2 d = ld(E / 2);
        const float2 d2 = cmul(d, d);
        v[E / 2] = cmul(v[E / 2], d);
#pragma unroll
        for (int k = 1; k <= E / 4; ++k) {
            const float2 w = ld(k), wc = cconj(w);
            v[k] = cmul(v[k], w);
            if (k < E / 4) {
                v[E / 2 - k] = cmul(v[E / 2 - k], cmul(d, wc));
                v[E - k] = cmul(v[E - k], cmul(d2, wc));
            }
            v[E / 2 + k] = cmul(v[E / 2 + k], cmul(d, w));
        }
    } else {
#pragma unroll
        for (int k2 = 1; k2 < E; ++k2) {
            float2 w = __ldg(tw + k2 * T + t);
            if (CONJ) w.y = -w.y;
            v[k2] = cmul(v[k2], w);
        }
    }
}

struct SyncWarp { __device__ __forceinline__ void operator()() const { __syncwarp(); } };
struct SyncBlock { __device__ __forceinline__ void operator()() const { __syncthreads(); } };

// Length T*E transform of one line in standard form.  sb: this line's exchange buffer, already
// offset by the column; element `slot` lives at sb[slot * CS], slot = n1 (E + 1) + k2.
// tw[k2 * T + t] = exp(-2 pi i t k2 / (T E)).
template <int T, int E, int SGN, bool IN_HALF, class Sync>
__device__ __forceinline__ void fft_line(float2 (&v)[E], float2* sb, const int CS, const int t,
                                         const float2* __restrict__ tw, Sync sync)
{
    static_assert(E % T == 0, "E must be a multiple of T");
    if constexpr (IN_HALF) fft_reg_half<E, SGN>(v);
    else fft_reg<E, SGN>(v);
#pragma unroll
    for (int k2 = 1; k2 < E; ++k2) {
        float2 w = __ldg(tw + k2 * T + t);
        if (SGN > 0) w.y = -w.y;
        v[k2] = cmul(v[k2], w);
    }
#pragma unroll
    for (int k2 = 0; k2 < E; ++k2) sb[(t * (E + 1) + k2) * CS] = v[k2];
    sync();
#pragma unroll
    for (int q = 0; q < E / T; ++q) {
        float2 u[T];
#pragma unroll
        for (int n1 = 0; n1 < T; ++n1) u[n1] = sb[(n1 * (E + 1) + t + T * q) * CS];
        fft_reg<T, SGN>(u);
#pragma unroll
        for (int k1 = 0; k1 < T; ++k1) v[q + (E / T) * k1] = u[k1];
    }
}

}  // namespace ff
}  // namespace mm

#include "fft_fast_kernels.cuh"
