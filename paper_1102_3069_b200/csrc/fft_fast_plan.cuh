// fft_fast_plan.cuh -- host side of the fast passes: size dispatch, twiddle tables, launches.
// Included by fft_fast_kernels.cuh.  Product code; shares nothing with oracle/.
#pragma once

namespace mm {

enum FastBits { FAST_FWD_X = 1, FAST_Y = 2, FAST_MID = 4, FAST_INV_X = 8, FAST_SPLIT = 16, FAST_ALL = 31 };

struct FastPlan {
    bool ok_x, ok_y, ok_mid3, ok_mul2;   // which passes have a size-specialised kernel for this grid
    float2* tw[3];                       // per axis: tw[k2 * T + t] = exp(-2 pi i t k2 / L)
    int nsm;                             // SM count (persistent grids)
};

namespace ff {

inline bool split(int L, int* T, int* E)
{
    switch (L) {
    case 64: *T = 8; *E = 8; return true;
    case 128: *T = 8; *E = 16; return true;
    case 256: *T = 16; *E = 16; return true;
    case 512: *T = 16; *E = 32; return true;
    case 1024: *T = 32; *E = 32; return true;
    }
    return false;
}

// k-space multiply on its own, 2D grids (Nz = 1): spec[3][Py][CxS] in place, K-hat octant [6][1][Cy][Cx]
__global__ void __launch_bounds__(256)
k_mul2d(Geom g, float2* __restrict__ spec, const float* __restrict__ khat)
{
    const int kx = blockIdx.x * blockDim.x + threadIdx.x;
    const int ky = blockIdx.y;
    if (kx >= g.Cx) return;
    int kyy = ky;
    float sy = 1.f;
    if (2 * kyy > g.Py) { kyy = g.Py - kyy; sy = -1.f; }
    const size_t nC = (size_t)g.Cx * g.Cy * g.Cz;
    const size_t ko = (size_t)kyy * g.Cx + kx;
    const float kxx = __ldg(khat + ko), kyy_ = __ldg(khat + ko + nC), kzz = __ldg(khat + ko + 2 * nC);
    const float kxy = sy * __ldg(khat + ko + 3 * nC), kxz = __ldg(khat + ko + 4 * nC);
    const float kyz = sy * __ldg(khat + ko + 5 * nC);
    const size_t cs = (size_t)g.Py * g.CxS;
    float2* p = spec + (size_t)ky * g.CxS + kx;
    const float2 mx = p[0], my = p[cs], mz = p[2 * cs];
    p[0] = make_float2(kxx * mx.x + kxy * my.x + kxz * mz.x, kxx * mx.y + kxy * my.y + kxz * mz.y);
    p[cs] = make_float2(kxy * mx.x + kyy_ * my.x + kyz * mz.x, kxy * mx.y + kyy_ * my.y + kyz * mz.y);
    p[2 * cs] = make_float2(kxz * mx.x + kyz * my.x + kzz * mz.x, kxz * mx.y + kyz * my.y + kzz * mz.y);
}

template <class K>
inline bool ensure_smem(K kern, size_t bytes)
{
    if (bytes <= 48 * 1024) return true;
    return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) == cudaSuccess;
}

template <int T, int E, bool PER>
bool launch_fwd_x(const FastPlan& fp, const Geom& g, cudaStream_t st, const float* m, float2* specA)
{
    const size_t bytes = (size_t)(128 / T) * T * (E + 1) * sizeof(float2);
    static bool once = ensure_smem(k_fwd_x<T, E, PER>, bytes);
    if (!once) return false;
    const int nslot = 128 / T;
    const int npair = 3 * g.Nz * ((g.Ny + 1) / 2);
    const int want = (npair + nslot - 1) / nslot;
    const int grid = want < fp.nsm * 8 ? want : fp.nsm * 8;
    k_fwd_x<T, E, PER><<<grid, 128, bytes, st>>>(g, m, specA, fp.tw[0]);
    return true;
}

template <int T, int E, bool PER>
bool launch_inv_x(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, const EpiParams& ep)
{
    constexpr int NX = PER ? T * E : T * E / 2;
    const size_t bytes = (size_t)(128 / T) * (T * (E + 1) + 2 * NX) * sizeof(float2);
    static bool once = ensure_smem(k_inv_x<T, E, PER>, bytes);
    if (!once) return false;
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
    static bool once = ensure_smem(k_inv_x_h<T, E, PER>, bytes);
    if (!once) return false;
    const int nslot = 128 / T;
    const int npair = 3 * g.Nz * ((g.Ny + 1) / 2);
    const int want = (npair + nslot - 1) / nslot;
    const int grid = want < fp.nsm * 8 ? want : fp.nsm * 8;
    k_inv_x_h<T, E, PER><<<grid, 128, bytes, st>>>(g, specA, fp.tw[0], out, scale);
    return true;
}

template <int T, int E, int SGN, bool PER>
bool launch_y(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* src, float2* dst)
{
    const size_t bytes = (size_t)T * (E + 1) * 8 * sizeof(float2);
    static bool once = ensure_smem(k_y<T, E, SGN, PER>, bytes);
    if (!once) return false;
    dim3 grid((g.Cx + 7) / 8, 3 * g.Nz);
    k_y<T, E, SGN, PER><<<grid, 8 * T, bytes, st>>>(g, src, dst, fp.tw[1]);
    return true;
}

template <int T, int E, bool PER>
bool launch_mid3(const FastPlan& fp, const Geom& g, cudaStream_t st, float2* specB, const float* khat)
{
    const size_t bytes = (size_t)3 * T * (E + 1) * 16 * sizeof(float2);
    static bool once = ensure_smem(k_mid<T, E, PER, true>, bytes);
    if (!once) return false;
    dim3 grid((g.Cx + 15) / 16, 2 * (g.Py / 2 + 1));
    k_mid<T, E, PER, true><<<grid, 16 * T, bytes, st>>>(g, specB, khat, fp.tw[2], 2);
    return true;
}

#define MM_FF_SIZES(L, CALL)                 \
    switch (L) {                              \
    case 64: { CALL(8, 8); } break;           \
    case 128: { CALL(8, 16); } break;         \
    case 256: { CALL(16, 16); } break;        \
    case 512: { CALL(16, 32); } break;        \
    case 1024: { CALL(32, 32); } break;       \
    default: break;                           \
    }

}  // namespace ff

inline bool fast_fwd_x(const FastPlan& fp, const Geom& g, cudaStream_t st, const float* m, float2* specA)
{
    if (!fp.ok_x) return false;
    bool r = false;
#define CALL(T, E) r = g.perx ? ff::launch_fwd_x<T, E, true>(fp, g, st, m, specA) \
                              : ff::launch_fwd_x<T, E, false>(fp, g, st, m, specA)
    MM_FF_SIZES(g.Px, CALL)
#undef CALL
    return r;
}

inline bool fast_inv_x(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, const EpiParams& ep)
{
    if (!fp.ok_x) return false;
    bool r = false;
#define CALL(T, E) r = g.perx ? ff::launch_inv_x<T, E, true>(fp, g, st, specA, ep) \
                              : ff::launch_inv_x<T, E, false>(fp, g, st, specA, ep)
    MM_FF_SIZES(g.Px, CALL)
#undef CALL
    return r;
}

// split variant of the last pass, first half: H_ms * scale -> out (a field)
inline bool fast_inv_x_h(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, float* out,
                         float scale)
{
    if (!fp.ok_x) return false;
    bool r = false;
#define CALL(T, E) r = g.perx ? ff::launch_inv_x_h<T, E, true>(fp, g, st, specA, out, scale) \
                              : ff::launch_inv_x_h<T, E, false>(fp, g, st, specA, out, scale)
    MM_FF_SIZES(g.Px, CALL)
#undef CALL
    return r;
}

// sgn < 0: specA rows y < Ny -> specB rows ky < Py; sgn > 0: back
inline bool fast_y(const FastPlan& fp, const Geom& g, cudaStream_t st, int sgn, const float2* src, float2* dst)
{
    if (!fp.ok_y) return false;
    bool r = false;
#define CALL(T, E)                                                                              \
    r = sgn < 0 ? (g.pery ? ff::launch_y<T, E, -1, true>(fp, g, st, src, dst)                   \
                          : ff::launch_y<T, E, -1, false>(fp, g, st, src, dst))                 \
                : (g.pery ? ff::launch_y<T, E, 1, true>(fp, g, st, src, dst)                    \
                          : ff::launch_y<T, E, 1, false>(fp, g, st, src, dst))
    MM_FF_SIZES(g.Py, CALL)
#undef CALL
    return r;
}

inline bool fast_mid3(const FastPlan& fp, const Geom& g, cudaStream_t st, float2* specB, const float* khat)
{
    if (!fp.ok_mid3) return false;
#define CALL(T, E) return g.perz ? ff::launch_mid3<T, E, true>(fp, g, st, specB, khat) \
                                 : ff::launch_mid3<T, E, false>(fp, g, st, specB, khat)
    switch (g.Pz) {      // three components of a line live in one thread: E <= 16
    case 64: CALL(8, 8);
    case 128: CALL(8, 16);
    case 256: CALL(16, 16);
    default: break;
    }
#undef CALL
    return false;
}

inline bool fast_mul2(const FastPlan& fp, const Geom& g, cudaStream_t st, float2* specB, const float* khat)
{
    if (!fp.ok_mul2) return false;
    dim3 grid((g.Cx + 255) / 256, g.Py);
    ff::k_mul2d<<<grid, 256, 0, st>>>(g, specB, khat);
    return true;
}

inline bool fast_plan_init(FastPlan& fp, const Geom& g, std::string* err)
{
    int T, E, dev = 0;
    fp.ok_x = ff::split(g.Px, &T, &E);
    fp.ok_y = g.Py > 1 && ff::split(g.Py, &T, &E);
    fp.ok_mid3 = g.Pz > 1 && g.Py > 1 && ff::split(g.Pz, &T, &E) && E <= 16;
    fp.ok_mul2 = g.Pz == 1 && fp.ok_y;
    fp.nsm = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&fp.nsm, cudaDevAttrMultiProcessorCount, dev);
    const int P[3] = { g.Px, g.Py, g.Pz };
    for (int a = 0; a < 3; ++a) {
        fp.tw[a] = nullptr;
        if (!ff::split(P[a], &T, &E)) continue;
        std::vector<float2> tw((size_t)P[a]);
        for (int k2 = 0; k2 < E; ++k2)
            for (int t = 0; t < T; ++t) {
                const long double ang = -2.0L * 3.14159265358979323846264338327950288L * ((long long)t * k2 % P[a]) / P[a];
                tw[(size_t)k2 * T + t] = make_float2((float)cosl(ang), (float)sinl(ang));
            }
        if (cudaMalloc(&fp.tw[a], tw.size() * sizeof(float2)) != cudaSuccess ||
            cudaMemcpy(fp.tw[a], tw.data(), tw.size() * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess) {
            if (err) *err = "fast plan: twiddle table allocation failed";
            return false;
        }
    }
    return true;
}

inline void fast_plan_destroy(FastPlan& fp)
{
    for (int a = 0; a < 3; ++a) { cudaFree(fp.tw[a]); fp.tw[a] = nullptr; }
}

}  // namespace mm
