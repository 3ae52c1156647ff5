// kern_mid.cu -- last-axis pass (a3): z forward, K-hat multiply, z inverse; 2D multiply.
// Product code; shares nothing with oracle/.
#include <string>
#include <vector>
#include "mm_kernels.h"
#include "fft_fast.cuh"
#include "fft_packed.cuh"

namespace mm {
namespace ff {
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

template <bool PER, int C, bool PANEL>
bool launch_mid_t(const FastPlan& fp, const Geom& g, cudaStream_t st, float2* specB, const float* khat)
{
    using M = pk::MidT<PER, C>;
    static bool once[MM_MAX_DEV] = {};
    if (!ensure_smem_dev(pk::k_mid_t<PER, C, PANEL>, M::SMEM_BYTES, once)) return false;
    const int nitem = ((g.Cx + C - 1) / C) * (g.Py / 2 + 1);
    const int per_sm = (PER ? 2 : 3) * (16 / C);
    const int grid = nitem < fp.nsm * per_sm ? nitem : fp.nsm * per_sm;
    pk::k_mid_t<PER, C, PANEL><<<grid, 8 * C, M::SMEM_BYTES, st>>>(PANEL ? fp.map_spec_p : fp.map_spec,
                                                                    khat == fp.k_ptr ? fp.map_k : fp.map_kex, g, specB,
                                                                    fp.twp);
    return true;
}

template <int T, int E, bool PER>
bool launch_mid3(const FastPlan& fp, const Geom& g, cudaStream_t st, const ColTile& ct, float2* specB,
                 const float* khat)
{
    if constexpr (T * E == 128) {
        // whole-array tiles only: the tensor maps describe specB and K-hat as laid out in mm_common.cuh
        if (fp.mid_pipe >= 2 && fp.ok_mid_t && ct.kx0 == 0 && ct.ncol == g.Cx && (khat == fp.k_ptr || fp.has_kex_map)) {
            if (ct.b_panel) return fp.ok_panel && launch_mid_t<PER, 16, true>(fp, g, st, specB, khat);
            if (ct.b_row == (size_t)g.CxS) return launch_mid_t<PER, 16, false>(fp, g, st, specB, khat);
        }
    }
    if (ct.b_panel) return false;        // only pk::k_mid_t reads the panel layout
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
}  // namespace ff

bool fast_mid3(const FastPlan& fp, const Geom& g, cudaStream_t st, const ff::ColTile& ct, float2* specB,
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


bool fast_mul2(const FastPlan& fp, const Geom& g, cudaStream_t st, float2* specB, const float* khat)
{
    if (!fp.ok_mul2) return false;
    dim3 grid((g.Cx + 255) / 256, g.Py, g.Nz);
    ff::k_mul2d<<<grid, 256, 0, st>>>(g, specB, khat);
    return true;
}


void launch_mul2d(const Geom& g, float2* spec, const float* khat, cudaStream_t st)
{
    dim3 grid((g.Cx + 255) / 256, g.Py, g.Nz);
    ff::k_mul2d<<<grid, 256, 0, st>>>(g, spec, khat);
}

}  // namespace mm
