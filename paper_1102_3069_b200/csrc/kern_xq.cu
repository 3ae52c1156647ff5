// kern_xq.cu -- the last pass in one kernel (a5-a10): inverse x transform and per-cell tail of a row pair in one
// block (ff::k_inv_x_q), its launch and instantiations.  Product code; shares nothing with oracle/.
#include <string>
#include <vector>
#include "mm_kernels.h"
#include "epilogue.cuh"
#include "fft_fast.cuh"

namespace mm {
namespace ff {
// one-kernel last pass (k_inv_x_q): x lines of T = 32 or 16 threads
template <int T, int E, bool PER, bool LEAN, int NA>
bool launch_inv_x_q(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, const EpiParams& ep)
{
    constexpr int NX = PER ? T * E : T * E / 2;
    constexpr int LPW = 32 / T;
    const size_t bytes = (size_t)3 * LPW * T * (E + 1) * sizeof(float2) + (size_t)LPW * 6 * NX * sizeof(float);
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
