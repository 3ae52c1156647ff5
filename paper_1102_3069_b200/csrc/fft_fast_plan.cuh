// fft_fast_plan.cuh -- host side of the fast passes: size dispatch, twiddle tables, launches.
// Included by fft_fast_kernels.cuh.  Product code; shares nothing with oracle/.
#pragma once

namespace mm {

enum FastBits { FAST_FWD_X = 1, FAST_Y = 2, FAST_MID = 4, FAST_INV_X = 8, FAST_SPLIT = 16, FAST_CHUNK = 32, FAST_ALL = 63 };

struct FastPlan {
    bool ok_x, ok_y, ok_mid3, ok_mul2;   // which passes have a size-specialised kernel for this grid
    bool ok_xr;                          // x passes through the half-length complex transform (Px = 1536, 2048)
    float2* twx;                         // ok_xr: exp(-i pi k / Lc), k < Lc = Px / 2
    float2* tw[3];                       // per axis: tw[k2 * T + t] = exp(-2 pi i t k2 / L)
    bool x_split;                        // Px = 4096: even / odd samples through the 2048-point real transform + combine
    float* xs_real;                      // x_split: de-interleaved rows [2 nrow][Nx / 2]
    float2* xs_spec;                     // x_split: their half spectra [2 nrow][XS_STRIDE]
    float2* twx4;                        // x_split: exp(-2 pi i j / 4096), j <= 1024
    int y_split;                         // y lines of 2048 / 4096: 2 / 4 interleaved transforms of 1024 (else 0)
    float2* twl;                         // y_split: exp(-2 pi i j / Py), j < Py
    int nsm;                             // SM count (persistent grids)
    int x_pipe;                          // x passes, cp.async-pipelined forms: bit 0 forward (default), bit 1 inverse (option "x_pipe")
    int mid_pipe;                        // last-axis pass: persistent pipelined kernel (option "mid_pipe")
    // last-axis pass through TMA tiles and sibling-packed codelets (pk::k_mid_t; mid_pipe >= 2, Pz = 128)
    bool ok_mid_t, has_kex_map;
    int mid_cols;                        // kx columns per work item of pk::k_mid_t
    CUtensorMap map_spec, map_k, map_kex;  // specB [3][Nz][Py][2 CxS] floats; K-hat / K-hat + exchange [6][Cz][Cy][CxK]
    const float* k_ptr;                  // the K-hat array map_k describes (map_kex: any other)
    float4* twp;                         // pk::k_mid_t twiddles
    int chunk_w, nstream;                // chunked a2-a4: columns per chunk (0 = whole-array passes), streams
    cudaStream_t stream[4];
    cudaEvent_t ev_fork, ev_join[4];
};

namespace ff {

inline bool split(int L, int* T, int* E)
{
    switch (L) {
    case 32: *T = 4; *E = 8; return true;
    case 64: *T = 8; *E = 8; return true;
    case 192: *T = 8; *E = 24; return true;
    case 384: *T = 8; *E = 48; return true;
    case 768: *T = 16; *E = 48; return true;
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
    const size_t nC = (size_t)g.CxK * g.Cy * g.Cz;
    const size_t ko = (size_t)kyy * g.CxK + kx;
    const float kxx = __ldg(khat + ko), kyy_ = __ldg(khat + ko + nC), kzz = __ldg(khat + ko + 2 * nC);
    const float kxy = sy * __ldg(khat + ko + 3 * nC), kxz = __ldg(khat + ko + 4 * nC);
    const float kyz = sy * __ldg(khat + ko + 5 * nC);
    // blockIdx.z = plane: a batch of B independent films is B planes of one array (mm_create_batch); Nz = 1 else
    const size_t cs = (size_t)g.Nz * g.Py * g.CxS;
    float2* p = spec + ((size_t)blockIdx.z * g.Py + ky) * g.CxS + kx;
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

// the dynamic shared-memory limit is a per-device attribute of a kernel: set it once per (kernel, device)
#define MM_MAX_DEV 64
template <class K>
inline bool ensure_smem_dev(K kern, size_t bytes, bool (&done)[MM_MAX_DEV])
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MM_MAX_DEV) return ensure_smem(kern, bytes);
    if (!done[dev]) {
        if (!ensure_smem(kern, bytes)) return false;
        done[dev] = true;
    }
    return true;
}

template <int T, int E, bool PER>
bool launch_fwd_x(const FastPlan& fp, const Geom& g, cudaStream_t st, const float* m, float2* specA)
{
    const size_t bytes = (size_t)(128 / T) * T * (E + 1) * sizeof(float2);
    static bool once[MM_MAX_DEV] = {};
    if (!ensure_smem_dev(k_fwd_x<T, E, PER>, bytes, once)) return false;
    const int nslot = 128 / T;
    const int npair = 3 * g.Nz * ((g.Ny + 1) / 2);
    const int want = (npair + nslot - 1) / nslot;
    const int grid = want < fp.nsm * 8 ? want : fp.nsm * 8;
    if ((fp.x_pipe & 1) && g.Nx % 4 == 0) {
        static bool oncep[MM_MAX_DEV] = {};
        if (!ensure_smem_dev(k_fwd_x_p<T, E, PER>, bytes, oncep)) return false;
        const int gridp = want < fp.nsm * 4 ? want : fp.nsm * 4;      // resident blocks: the loop is pipelined
        k_fwd_x_p<T, E, PER><<<gridp, 128, bytes, st>>>(g, m, specA, fp.tw[0]);
        return true;
    }
    k_fwd_x<T, E, PER><<<grid, 128, bytes, st>>>(g, m, specA, fp.tw[0]);
    return true;
}

template <int T, int E, bool PER>
bool launch_inv_x(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, const EpiParams& ep)
{
    constexpr int NX = PER ? T * E : T * E / 2;
    const size_t bytes = (size_t)(128 / T) * (T * (E + 1) + 2 * NX) * sizeof(float2);
    static bool once[MM_MAX_DEV] = {};
    if (!ensure_smem_dev(k_inv_x<T, E, PER>, bytes, once)) return false;
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
    static bool once[MM_MAX_DEV] = {};
    if (!ensure_smem_dev(k_inv_x_h<T, E, PER>, bytes, once)) return false;
    const int nslot = 128 / T;
    const int npair = 3 * g.Nz * ((g.Ny + 1) / 2);
    const int want = (npair + nslot - 1) / nslot;
    const int grid = want < fp.nsm * 8 ? want : fp.nsm * 8;
    if ((fp.x_pipe & 2) && g.CxS % 2 == 0) {      // measured slower than the plain form on B200: off by default
        static bool oncep[MM_MAX_DEV] = {};
        if (!ensure_smem_dev(k_inv_x_h_p<T, E, PER>, bytes, oncep)) return false;
        const int gridp = want < fp.nsm * 4 ? want : fp.nsm * 4;
        k_inv_x_h_p<T, E, PER><<<gridp, 128, bytes, st>>>(g, specA, fp.tw[0], out, scale);
        return true;
    }
    k_inv_x_h<T, E, PER><<<grid, 128, bytes, st>>>(g, specA, fp.tw[0], out, scale);
    return true;
}

template <int T, int E, bool PER>
bool launch_fwd_x_r(const FastPlan& fp, const Geom& g, cudaStream_t st, const float* m, float2* specA)
{
    const size_t bytes = (size_t)(128 / T) * T * (E + 1) * sizeof(float2);
    static bool once[MM_MAX_DEV] = {};
    if (!ensure_smem_dev(k_fwd_x_r<T, E, PER>, bytes, once)) return false;
    const int nslot = 128 / T;
    const int want = (3 * g.Nz * g.Ny + nslot - 1) / nslot;
    const int grid = want < fp.nsm * 8 ? want : fp.nsm * 8;
    k_fwd_x_r<T, E, PER><<<grid, 128, bytes, st>>>(g, m, specA, fp.tw[0], fp.twx);
    return true;
}

template <int T, int E, bool PER>
bool launch_inv_x_h_r(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, float* out,
                      float scale)
{
    const size_t bytes = (size_t)(128 / T) * T * (E + 1) * sizeof(float2);
    static bool once[MM_MAX_DEV] = {};
    if (!ensure_smem_dev(k_inv_x_h_r<T, E, PER>, bytes, once)) return false;
    const int nslot = 128 / T;
    const int want = (3 * g.Nz * g.Ny + nslot - 1) / nslot;
    const int grid = want < fp.nsm * 8 ? want : fp.nsm * 8;
    k_inv_x_h_r<T, E, PER><<<grid, 128, bytes, st>>>(g, specA, fp.tw[0], fp.twx, out, scale);
    return true;
}

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

template <bool PER, int C>
bool launch_mid_t(const FastPlan& fp, const Geom& g, cudaStream_t st, float2* specB, const float* khat)
{
    using M = pk::MidT<PER, C>;
    static bool once[MM_MAX_DEV] = {};
    if (!ensure_smem_dev(pk::k_mid_t<PER, C>, M::SMEM_BYTES, once)) return false;
    const int nitem = ((g.Cx + C - 1) / C) * (g.Py / 2 + 1);
    const int per_sm = (PER ? 2 : 3) * (16 / C);
    const int grid = nitem < fp.nsm * per_sm ? nitem : fp.nsm * per_sm;
    pk::k_mid_t<PER, C><<<grid, 8 * C, M::SMEM_BYTES, st>>>(fp.map_spec, khat == fp.k_ptr ? fp.map_k : fp.map_kex, g,
                                                             specB, fp.twp);
    return true;
}

template <int T, int E, bool PER>
bool launch_mid3(const FastPlan& fp, const Geom& g, cudaStream_t st, const ColTile& ct, float2* specB,
                 const float* khat)
{
    if constexpr (T * E == 128) {
        // whole-array tiles only: the tensor maps describe specB and K-hat as laid out in mm_common.cuh
        if (fp.mid_pipe >= 2 && fp.ok_mid_t && ct.kx0 == 0 && ct.ncol == g.Cx && ct.b_row == (size_t)g.CxS &&
            (khat == fp.k_ptr || fp.has_kex_map))
            return launch_mid_t<PER, 16>(fp, g, st, specB, khat);
    }
    if (fp.mid_pipe) {
        constexpr int L = T * E;
        constexpr int NZ = PER ? L : L / 2;
        constexpr int NXB = 1;           // one exchange tile, used by the three components in turn
        const size_t pb = (size_t)NXB * T * (E + 1) * 16 * sizeof(float2) + (size_t)3 * NZ * 16 * sizeof(float2) +
                          (size_t)6 * (L / 2 + 1) * 16 * sizeof(float);
        if (pb <= 227 * 1024) {
            const int nitem = ((ct.ncol + 15) / 16) * (g.Py / 2 + 1);
            const int per_sm = (T * E <= 128) ? 3 : 1;
            const int grid = nitem < fp.nsm * per_sm ? nitem : fp.nsm * per_sm;
            static bool oncep[MM_MAX_DEV] = {};
            if (!ensure_smem_dev(k_mid_p<T, E, PER>, pb, oncep)) return false;
            k_mid_p<T, E, PER><<<grid, 16 * T, pb, st>>>(g, ct, specB, khat, fp.tw[2]);
            return true;
        }
    }
    const size_t bytes = (size_t)3 * T * (E + 1) * 16 * sizeof(float2);
    constexpr int MINB = (T * E <= 128) ? 2 : 1;
    dim3 grid((ct.ncol + 15) / 16, 2 * (g.Py / 2 + 1));
    static bool once[MM_MAX_DEV] = {};
    if (!ensure_smem_dev(k_mid<T, E, PER, true, MINB>, bytes, once)) return false;
    k_mid<T, E, PER, true, MINB><<<grid, 16 * T, bytes, st>>>(g, ct, specB, khat, fp.tw[2], 2);
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
// x lines of 4096 (2048 cells, open; 4096 cells, periodic -- PAPER.md:245, the largest 2D grid of Table 1): one
// decimation-in-time level outside the kernels.  The even and the odd samples of a row are two real sequences of
// half the length; each goes through the 2048-point real transform (k_fwd_x_r / k_inv_x_h_r, unchanged), and
//   forward:  X[j] = E[j] + w^j O[j],  X[2048 - j] = conj(E[j] - w^j O[j]),  j <= 1024,  w = exp(-2 pi i / 4096)
//   inverse:  E'[j] = X[j] + conj X[2048 - j],  O'[j] = conj(w^j) (X[j] - conj X[2048 - j])
// ---------------------------------------------------------------------------------------------
#define MM_XS_STRIDE 1032
namespace ff {
__global__ void k_x_deinterleave(const float2* __restrict__ m, float* __restrict__ tmp, size_t nrow, int half)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nrow * half; i += (size_t)gridDim.x * blockDim.x) {
        const size_t row = i / half, n = i - row * half;
        const float2 v = m[i];
        tmp[(2 * row) * half + n] = v.x;
        tmp[(2 * row + 1) * half + n] = v.y;
    }
}
__global__ void k_x_interleave(const float* __restrict__ tmp, float2* __restrict__ out, size_t nrow, int half)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nrow * half; i += (size_t)gridDim.x * blockDim.x) {
        const size_t row = i / half, n = i - row * half;
        out[i] = make_float2(tmp[(2 * row) * half + n], tmp[(2 * row + 1) * half + n]);
    }
}
template <int SGN>
__global__ void k_x_combine(float2* __restrict__ ts, float2* __restrict__ specA, size_t nrow, int CxS,
                            const float2* __restrict__ tw4)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    const size_t row = blockIdx.y;
    if (j > 1024 || row >= nrow) return;
    float2* e = ts + (2 * row) * MM_XS_STRIDE + j;
    float2* o = ts + (2 * row + 1) * MM_XS_STRIDE + j;
    float2* x = specA + row * CxS;
    const float2 w = __ldg(tw4 + j);
    if (SGN < 0) {
        const float2 E = *e, wO = cmul(w, *o);
        x[j] = cadd(E, wO);
        if (j != 1024) x[2048 - j] = cconj(csub(E, wO));
    } else {
        const float2 A = x[j], B = cconj(x[2048 - j]);
        *e = cadd(A, B);
        *o = cmul(cconj(w), csub(A, B));
    }
}
}  // namespace ff

inline Geom x_split_geom(const Geom& g)
{
    Geom h = g;
    h.Nx = g.Nx / 2; h.Ny = 2 * g.Ny; h.Px = g.Px / 2; h.Cx = h.Px / 2 + 1; h.CxS = MM_XS_STRIDE;
    return h;
}

inline bool fast_fwd_x(const FastPlan& fp, const Geom& g, cudaStream_t st, const float* m, float2* specA)
{
    if (fp.x_split) {
        const size_t nrow = (size_t)3 * g.Nz * g.Ny;
        const Geom h = x_split_geom(g);
        ff::k_x_deinterleave<<<fp.nsm * 8, 256, 0, st>>>(reinterpret_cast<const float2*>(m), fp.xs_real, nrow, g.Nx / 2);
        if (!(g.perx ? ff::launch_fwd_x_r<32, 32, true>(fp, h, st, fp.xs_real, fp.xs_spec)
                     : ff::launch_fwd_x_r<32, 32, false>(fp, h, st, fp.xs_real, fp.xs_spec)))
            return false;
        dim3 cg((1025 + 127) / 128, (unsigned)nrow);
        ff::k_x_combine<-1><<<cg, 128, 0, st>>>(fp.xs_spec, specA, nrow, g.CxS, fp.twx4);
        return true;
    }
    if (fp.ok_xr) {
        if (g.Px == 1536) return g.perx ? ff::launch_fwd_x_r<16, 48, true>(fp, g, st, m, specA)
                                        : ff::launch_fwd_x_r<16, 48, false>(fp, g, st, m, specA);
        if (g.Px == 2048) return g.perx ? ff::launch_fwd_x_r<32, 32, true>(fp, g, st, m, specA)
                                        : ff::launch_fwd_x_r<32, 32, false>(fp, g, st, m, specA);
        return false;
    }
    if (!fp.ok_x) return false;
    bool r = false;
#define CALL(T, E) r = g.perx ? ff::launch_fwd_x<T, E, true>(fp, g, st, m, specA) \
                              : ff::launch_fwd_x<T, E, false>(fp, g, st, m, specA)
    MM_FF_SIZES(g.Px, CALL)
#undef CALL
    return r;
}

// fused inverse x + epilogue (bit 8): power-of-two lengths only; the split pass (bit 16) is the default
inline bool fast_inv_x(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, const EpiParams& ep)
{
    if (!fp.ok_x) return false;
#define CALL(T, E) return g.perx ? ff::launch_inv_x<T, E, true>(fp, g, st, specA, ep) \
                                 : ff::launch_inv_x<T, E, false>(fp, g, st, specA, ep)
    switch (g.Px) {
    case 64: CALL(8, 8);
    case 128: CALL(8, 16);
    case 256: CALL(16, 16);
    case 512: CALL(16, 32);
    case 1024: CALL(32, 32);
    default: break;
    }
#undef CALL
    return false;
}

// split variant of the last pass, first half: H_ms * scale -> out (a field)
inline bool fast_inv_x_h(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, float* out,
                         float scale)
{
    if (fp.x_split) {
        const size_t nrow = (size_t)3 * g.Nz * g.Ny;
        const Geom h = x_split_geom(g);
        dim3 cg((1025 + 127) / 128, (unsigned)nrow);
        ff::k_x_combine<1><<<cg, 128, 0, st>>>(fp.xs_spec, const_cast<float2*>(specA), nrow, g.CxS, fp.twx4);
        if (!(g.perx ? ff::launch_inv_x_h_r<32, 32, true>(fp, h, st, fp.xs_spec, fp.xs_real, scale)
                     : ff::launch_inv_x_h_r<32, 32, false>(fp, h, st, fp.xs_spec, fp.xs_real, scale)))
            return false;
        ff::k_x_interleave<<<fp.nsm * 8, 256, 0, st>>>(fp.xs_real, reinterpret_cast<float2*>(out), nrow, g.Nx / 2);
        return true;
    }
    if (fp.ok_xr) {
        if (g.Px == 1536) return g.perx ? ff::launch_inv_x_h_r<16, 48, true>(fp, g, st, specA, out, scale)
                                        : ff::launch_inv_x_h_r<16, 48, false>(fp, g, st, specA, out, scale);
        if (g.Px == 2048) return g.perx ? ff::launch_inv_x_h_r<32, 32, true>(fp, g, st, specA, out, scale)
                                        : ff::launch_inv_x_h_r<32, 32, false>(fp, g, st, specA, out, scale);
        return false;
    }
    if (!fp.ok_x) return false;
    bool r = false;
#define CALL(T, E) r = g.perx ? ff::launch_inv_x_h<T, E, true>(fp, g, st, specA, out, scale) \
                              : ff::launch_inv_x_h<T, E, false>(fp, g, st, specA, out, scale)
    MM_FF_SIZES(g.Px, CALL)
#undef CALL
    return r;
}

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
inline bool fast_y_long(const FastPlan& fp, const Geom& g, cudaStream_t st, int sgn, const ff::ColTile& ct, float2* a,
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
inline bool fast_y(const FastPlan& fp, const Geom& g, cudaStream_t st, int sgn, const ff::ColTile& ct, float2* a,
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

inline bool fast_mid3(const FastPlan& fp, const Geom& g, cudaStream_t st, const ff::ColTile& ct, float2* specB,
                      const float* khat)
{
    if (!fp.ok_mid3) return false;
#define CALL(T, E) return g.perz ? ff::launch_mid3<T, E, true>(fp, g, st, ct, specB, khat) \
                                 : ff::launch_mid3<T, E, false>(fp, g, st, ct, specB, khat)
    switch (g.Pz) {      // three components of a line live in one thread: E <= 16
    case 64: CALL(8, 8);
    case 128: CALL(8, 16);
    case 256: CALL(16, 16);
    default: break;
    }
#undef CALL
    return false;
}

// the whole-array tile: every column, strides of mm_common.cuh
inline ff::ColTile whole_tile(const Geom& g)
{
    ff::ColTile ct;
    ct.kx0 = 0; ct.ncol = g.Cx;
    ct.a_row = g.CxS; ct.a_plane = (size_t)g.Ny * g.CxS;
    ct.b_row = g.CxS; ct.b_plane = (size_t)g.Py * g.CxS;
    return ct;
}

// a2-a4 in chunks of fp.chunk_w kx columns (3D grids): forward y pass into a compact chunk buffer
// (a slot of specB), last-axis pass in place, inverse y pass back into specA.  A chunk is a few tens
// of MB, so between the three kernels it stays in the 126 MB L2 and the y-padded spectrum never
// travels to HBM.  Chunks rotate over fp.nstream streams so that the tail of one kernel overlaps the
// next chunk.  `st` is the context's stream: forked from and joined back to with events.
inline bool fast_yzy_chunked(FastPlan& fp, const Geom& g, cudaStream_t st, float2* specA, float2* specB,
                             const float* khat)
{
    if (!(fp.ok_y && fp.ok_mid3 && fp.chunk_w > 0 && fp.nstream > 0)) return false;
    const int W = fp.chunk_w;
    const size_t slot = (size_t)3 * g.Nz * g.Py * W;
    cudaEventRecord(fp.ev_fork, st);
    for (int s = 0; s < fp.nstream; ++s) cudaStreamWaitEvent(fp.stream[s], fp.ev_fork, 0);
    int i = 0;
    for (int kx0 = 0; kx0 < g.Cx; kx0 += W, ++i) {
        const int s = i % fp.nstream;
        ff::ColTile ct;
        ct.kx0 = kx0; ct.ncol = g.Cx - kx0 < W ? g.Cx - kx0 : W;
        ct.a_row = g.CxS; ct.a_plane = (size_t)g.Ny * g.CxS;
        ct.b_row = W; ct.b_plane = (size_t)g.Py * W;
        float2* buf = specB + (size_t)s * slot;
        if (!fast_y(fp, g, fp.stream[s], -1, ct, specA + kx0, buf)) return false;
        if (!fast_mid3(fp, g, fp.stream[s], ct, buf, khat)) return false;
        if (!fast_y(fp, g, fp.stream[s], 1, ct, specA + kx0, buf)) return false;
    }
    for (int s = 0; s < fp.nstream; ++s) {
        cudaEventRecord(fp.ev_join[s], fp.stream[s]);
        cudaStreamWaitEvent(st, fp.ev_join[s], 0);
    }
    return true;
}

inline bool fast_mul2(const FastPlan& fp, const Geom& g, cudaStream_t st, float2* specB, const float* khat)
{
    if (!fp.ok_mul2) return false;
    dim3 grid((g.Cx + 255) / 256, g.Py, g.Nz);
    ff::k_mul2d<<<grid, 256, 0, st>>>(g, specB, khat);
    return true;
}

inline bool fast_plan_init(FastPlan& fp, const Geom& g, std::string* err)
{
    int T, E, dev = 0;
    fp.ok_x = ff::split(g.Px, &T, &E);
    fp.ok_xr = !fp.ok_x && (g.Px == 1536 || g.Px == 2048) && g.Nx % 2 == 0;
    fp.x_split = g.Px == 4096 && g.Nx % 4 == 0 && (size_t)3 * g.Nz * g.Ny <= 65535;      // (rows: grid.y of the combine)
    fp.xs_real = nullptr; fp.xs_spec = nullptr; fp.twx4 = nullptr;
    fp.twx = nullptr;
    fp.y_split = (g.Py == 2048 || g.Py == 4096) ? g.Py / 1024 : 0;
    fp.twl = nullptr;
    fp.ok_y = g.Py > 1 && (ff::split(g.Py, &T, &E) || fp.y_split);
    fp.ok_mid3 = g.Pz >= 64 && g.Py > 1 && ff::split(g.Pz, &T, &E) && E <= 16;
    fp.ok_mul2 = g.Pz == 1 && fp.ok_y;
    // fp.x_pipe, fp.mid_pipe, fp.chunk_w, fp.nstream come from the context (mm_set_option; defaults set by
    // mm_create).  L2-resident chunks (chunk_w = columns per chunk, multiple of 16) are off by default:
    // measured on B200 at 512x512x64 they give bit-identical results and cut DRAM traffic, but no time,
    // because the y and last-axis passes are bound by instruction issue, not by HBM (profiles/).
    if (fp.chunk_w % 16 != 0 || fp.chunk_w < 0 || !(fp.ok_y && fp.ok_mid3)) fp.chunk_w = 0;
    if (fp.nstream < 1) fp.nstream = 1;
    if (fp.nstream > 4) fp.nstream = 4;
    if ((size_t)fp.chunk_w * fp.nstream > (size_t)g.CxS) fp.chunk_w = 0;      // slots must fit specB
    for (int s = 0; s < 4; ++s) { fp.stream[s] = nullptr; fp.ev_join[s] = nullptr; }
    fp.ev_fork = nullptr;
    if (fp.chunk_w > 0) {
        for (int s = 0; s < fp.nstream; ++s) {
            if (cudaStreamCreateWithFlags(&fp.stream[s], cudaStreamNonBlocking) != cudaSuccess ||
                cudaEventCreateWithFlags(&fp.ev_join[s], cudaEventDisableTiming) != cudaSuccess) {
                if (err) *err = "fast plan: stream / event creation failed";
                return false;
            }
        }
        if (cudaEventCreateWithFlags(&fp.ev_fork, cudaEventDisableTiming) != cudaSuccess) {
            if (err) *err = "fast plan: event creation failed";
            return false;
        }
    }
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&fp.nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || fp.nsm < 1) {
        if (err) *err = "fast plan: cannot read the SM count of the current device";
        return false;
    }
    const int P[3] = { fp.x_split ? 1024 : (fp.ok_xr ? g.Px / 2 : g.Px), fp.y_split ? 1024 : g.Py, g.Pz };
    if (fp.x_split) {
        const size_t nrow = (size_t)3 * g.Nz * g.Ny;
        std::vector<float2> t4(1025);
        for (int j = 0; j <= 1024; ++j) {
            const long double ang = -2.0L * 3.14159265358979323846264338327950288L * j / 4096.0L;
            t4[j] = make_float2((float)cosl(ang), (float)sinl(ang));
        }
        if (cudaMalloc(&fp.xs_real, nrow * g.Nx * sizeof(float)) != cudaSuccess ||
            cudaMalloc(&fp.xs_spec, 2 * nrow * MM_XS_STRIDE * sizeof(float2)) != cudaSuccess ||
            cudaMemset(fp.xs_spec, 0, 2 * nrow * MM_XS_STRIDE * sizeof(float2)) != cudaSuccess ||
            cudaMalloc(&fp.twx4, t4.size() * sizeof(float2)) != cudaSuccess ||
            cudaMemcpy(fp.twx4, t4.data(), t4.size() * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess) {
            if (err) *err = "fast plan: x-split workspace allocation failed";
            return false;
        }
    }
    if (fp.y_split) {
        std::vector<float2> tl((size_t)g.Py);
        for (int j = 0; j < g.Py; ++j) {
            const long double ang = -2.0L * 3.14159265358979323846264338327950288L * j / g.Py;
            tl[j] = make_float2((float)cosl(ang), (float)sinl(ang));
        }
        if (cudaMalloc(&fp.twl, tl.size() * sizeof(float2)) != cudaSuccess ||
            cudaMemcpy(fp.twl, tl.data(), tl.size() * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess) {
            if (err) *err = "fast plan: twiddle table allocation failed";
            return false;
        }
    }
    if (fp.ok_xr || fp.x_split) {
        const int Lc = fp.x_split ? 1024 : g.Px / 2;
        std::vector<float2> tx((size_t)Lc);
        for (int k = 0; k < Lc; ++k) {
            const long double ang = -3.14159265358979323846264338327950288L * k / Lc;
            tx[k] = make_float2((float)cosl(ang), (float)sinl(ang));
        }
        if (cudaMalloc(&fp.twx, tx.size() * sizeof(float2)) != cudaSuccess ||
            cudaMemcpy(fp.twx, tx.data(), tx.size() * sizeof(float2), cudaMemcpyHostToDevice) != cudaSuccess) {
            if (err) *err = "fast plan: twiddle table allocation failed";
            return false;
        }
    }
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

// ---- TMA tensor maps (cuTensorMapEncodeTiled, fetched through the runtime: libcuda is not linked) ----
typedef CUresult (*mm_encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                       const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                       CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline mm_encode_tiled_fn tensor_map_encoder()
{
    static mm_encode_tiled_fn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) == cudaSuccess &&
            qr == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<mm_encode_tiled_fn>(p);
        else
            cudaGetLastError();
    }
    return fn;
}

// 4D float32 map: dims[0] is the contiguous one; stride_bytes[i] = byte stride of dims[i + 1]; out-of-range reads give 0
inline bool make_map4(CUtensorMap* m, const void* base, const cuuint64_t dims[4], const cuuint64_t stride_bytes[3],
                      const cuuint32_t box[4])
{
    mm_encode_tiled_fn enc = tensor_map_encoder();
    if (!enc) return false;
    const cuuint32_t es[4] = { 1, 1, 1, 1 };
    return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, const_cast<void*>(base), dims, stride_bytes, box, es,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// K-hat octant [6][Cz][Cy][CxK] seen as (kx, ky, kz >> 1, component, kz & 1): a box of all kz lands in shared
// memory as [parity][component][kz >> 1][16].  Row kz = Cz (parity 1 of the last pair when Cz is odd) is
// addressed but never used: the K-hat allocations carry one spare plane (mm_api.cu).
inline bool khat_map(CUtensorMap* m, const Geom& g, const float* khat, int cols)
{
    mm_encode_tiled_fn enc = tensor_map_encoder();
    if (!enc) return false;
    const cuuint64_t row = (cuuint64_t)g.CxK * 4, plane = row * g.Cy;
    const cuuint32_t ch = (cuuint32_t)(g.Cz / 2 + 1);
    const cuuint64_t dims[5] = { (cuuint64_t)g.CxK, (cuuint64_t)g.Cy, ch, 6, 2 };
    const cuuint64_t sb[4] = { row, 2 * plane, plane * g.Cz, plane };
    const cuuint32_t box[5] = { (cuuint32_t)cols, 1, ch, 6, 2 };
    const cuuint32_t es[5] = { 1, 1, 1, 1, 1 };
    return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 5, const_cast<float*>(khat), dims, sb, box, es,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// called by mm_demag_init once specB and K-hat exist; failure only switches pk::k_mid_t off
inline void fast_plan_maps(FastPlan& fp, const Geom& g, const float2* specB, const float* khat)
{
    fp.ok_mid_t = false;
    fp.has_kex_map = false;
    fp.k_ptr = khat;
    if (!(fp.ok_mid3 && g.Pz == 128 && specB && khat)) return;
    const cuuint64_t dims[4] = { (cuuint64_t)2 * g.CxS, (cuuint64_t)g.Py, (cuuint64_t)g.Nz, 3 };
    const cuuint64_t sb[3] = { (cuuint64_t)g.CxS * 8, (cuuint64_t)g.CxS * g.Py * 8, (cuuint64_t)g.CxS * g.Py * g.Nz * 8 };
    fp.mid_cols = 16;       // 8-column items (6 blocks per SM) were measured: 0.84 ms against 0.49 ms
    const cuuint32_t box[4] = { (cuuint32_t)(2 * fp.mid_cols), 1, (cuuint32_t)g.Nz, 3 };
    if (!make_map4(&fp.map_spec, specB, dims, sb, box) || !khat_map(&fp.map_k, g, khat, fp.mid_cols)) return;
    std::vector<float4> tw(64);
    for (int a = 0; a < 8; ++a)
        for (int b = 0; b < 8; ++b) {
            const long double w = 2.0L * 3.14159265358979323846264338327950288L / 128.0L;
            const long double p0 = w * (a * 2 * b), p1 = w * (a * (2 * b + 1));
            tw[a * 8 + b] = make_float4((float)cosl(p0), (float)cosl(p1), (float)sinl(p0), (float)sinl(p1));
        }
    if (cudaMalloc(&fp.twp, tw.size() * sizeof(float4)) != cudaSuccess ||
        cudaMemcpy(fp.twp, tw.data(), tw.size() * sizeof(float4), cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError();
        return;
    }
    fp.ok_mid_t = true;
}

inline void fast_plan_destroy(FastPlan& fp)
{
    cudaFree(fp.twp);
    fp.twp = nullptr;
    fp.ok_mid_t = false;
    for (int a = 0; a < 3; ++a) { cudaFree(fp.tw[a]); fp.tw[a] = nullptr; }
    cudaFree(fp.twx);
    fp.twx = nullptr;
    cudaFree(fp.twl);
    fp.twl = nullptr;
    cudaFree(fp.xs_real); cudaFree(fp.xs_spec); cudaFree(fp.twx4);
    fp.xs_real = nullptr; fp.xs_spec = nullptr; fp.twx4 = nullptr;
    for (int s = 0; s < 4; ++s) {
        if (fp.stream[s]) cudaStreamDestroy(fp.stream[s]);
        if (fp.ev_join[s]) cudaEventDestroy(fp.ev_join[s]);
        fp.stream[s] = nullptr; fp.ev_join[s] = nullptr;
    }
    if (fp.ev_fork) cudaEventDestroy(fp.ev_fork);
    fp.ev_fork = nullptr;
}

}  // namespace mm
