// mm_kernels.h -- what the host side (mm_api.cu) and the kernel translation units share: plan structures and the
// launch entry points of every pass.  Each kernel family is compiled in a translation unit of its own (kern_x.cu,
// kern_y.cu, kern_mid.cu, kern_epi.cu, kern_gen.cu), so that a change in one family cannot perturb the code
// generated for another and the library builds in parallel.  Product code; shares nothing with oracle/.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <string>
#include "mm_common.cuh"

namespace mm {

#define MM_MAXRAD 16
struct FftPlan {            // one axis
    int L;                  // transform length
    int nrad;
    int rad[MM_MAXRAD];
    const float2* tw;       // device, tw[q] = exp(-2 pi i q / L), q < L
};

namespace ff {
// ---------------------------------------------------------------------------------------------
// Where the columns of a y / last-axis pass live.  The whole-array mode uses the layouts of
// mm_common.cuh (row stride CxS); the chunked mode and the slab pencils work on
// `ncol` kx columns starting at kx0, with the y-padded spectrum in a compact buffer [3][Nz][Py][W].
// ---------------------------------------------------------------------------------------------
struct ColTile {
    ColTile() : kx0(0), ncol(0), a_row(0), a_plane(0), b_row(0), b_plane(0), b_panel(0) {}
    int kx0, ncol;                 // first global column, number of valid columns
    size_t a_row, a_plane;         // specA side: strides in float2 (row y, plane (component, z))
    size_t b_row, b_plane;         // specB / chunk side
    size_t b_panel;                // specB in panels of 16 columns [panel][3 Nz][Py][16] (stride of a panel), 0: plain rows
};
}  // namespace ff

enum FastBits { FAST_FWD_X = 1, FAST_Y = 2, FAST_MID = 4, FAST_INV_X = 8, FAST_SPLIT = 16, FAST_CHUNK = 32, FAST_ALL = 63 };

// a line length P handled directly (R = 1, Ls = P) or as R interleaved transforms of Ls = P / R plus a combine
struct AxisPlan {
    int R, Ls;
    const float2* tw;                    // twiddles of the Ls-point kernel, tw[k2 * T + t]
    float2* twl;                         // R > 1: exp(-2 pi i j / P), j < P
};

struct FastPlan {
    bool ok_x, ok_y, ok_mid3, ok_mul2;   // which passes have a size-specialised kernel for this grid
    bool ok_xr;                          // x passes through the half-length complex transform (Px = 1536, 2048)
    float2* twx;                         // ok_xr: exp(-i pi k / Lc), k < Lc = Px / 2
    float2* tw[3];                       // per axis: tw[k2 * T + t] = exp(-2 pi i t k2 / L)
    int x_R, x_Ls, xs_stride;            // x lines as x_R interleaved real transforms of x_Ls = Px / x_R (x_R <= 1: direct)
    float* xs_real;                      // x_R > 1: de-interleaved rows [x_R nrow][Nx / x_R]
    float2* xs_spec;                     // x_R > 1: their half spectra [x_R nrow][xs_stride]
    float2* twxl;                        // x_R > 1: exp(-2 pi i j / Px), j < Px
    bool z_long;                         // z lines too long for the fused last-axis kernels: unfused z pass through zbuf
    float2* zbuf;                        // z_long: z-padded spectrum [3][Pz][Py][CxS]
    AxisPlan ax[3];                      // lines along y ([1]) and z ([2]): direct or R interleaved sub-transforms
    int nsm;                             // SM count (persistent grids)
    int x_pipe;                          // x passes, cp.async-pipelined forms: bit 0 forward (default), bit 1 inverse (option "x_pipe")
    int mid_pipe;                        // last-axis pass: persistent pipelined kernel (option "mid_pipe")
    // last-axis pass through TMA tiles and sibling-packed codelets (pk::k_mid_t; mid_pipe >= 2, Pz = 128)
    bool ok_mid_t, has_kex_map;
    bool ok_panel;                       // specB may be kept in 16-column panels between a2, a3 and a4 (option "spec_panel")
    int spec_panel;
    int y_tma;                           // option "y_tma": y-pass tiles of 1024-long lines loaded by TMA (panel mode)
    bool ok_ymaps;
    CUtensorMap map_ya, map_yb;          // specA as (2 Cx floats, Ny, 3 Nz); specB panels as (32 floats, Py, 3 Nz, panel)
    const float2 *y_a, *y_b;             // the arrays those maps describe
    int last_fused;                      // option "last_fused": a5-a10 in one kernel (k_inv_x_q) where it applies
    int q_blocks;                        // option "q_blocks": resident blocks per SM of k_inv_x_q
    CUtensorMap map_spec_p;              // specB in panels: (32 floats, Py, Nz, 3, panel)
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
}  // namespace ff

// the whole-array tile: every column, strides of mm_common.cuh
inline ff::ColTile whole_tile(const Geom& g)
{
    ff::ColTile ct;
    ct.kx0 = 0; ct.ncol = g.Cx;
    ct.a_row = g.CxS; ct.a_plane = (size_t)g.Ny * g.CxS;
    ct.b_row = g.CxS; ct.b_plane = (size_t)g.Py * g.CxS;
    ct.b_panel = 0;
    return ct;
}

// the whole array with specB in panels of 16 kx columns: [panel][3][Nz][Py][16].  A y-pass tile (8 columns, all ky of
// one plane) and its neighbour then fill one contiguous 16 Py float2 block, and the rows of a last-axis work item
// (16 columns, one ky) sit next to those of ky + 1 -- the DRAM-friendly form of the same traffic.
inline ff::ColTile panel_tile(const Geom& g)
{
    ff::ColTile ct = whole_tile(g);
    ct.b_row = 16; ct.b_plane = (size_t)g.Py * 16;
    ct.b_panel = (size_t)3 * g.Nz * g.Py * 16;
    return ct;
}
// columns specB must have room for (the last panel is padded)
inline size_t specb_cols(const Geom& g) { const size_t cp = (size_t)((g.Cx + 15) / 16) * 16; return cp > (size_t)g.CxS ? cp : (size_t)g.CxS; }


// ---- size-specialised passes (return false: no kernel for this size, the caller falls back) ----
bool fast_fwd_x(const FastPlan& fp, const Geom& g, cudaStream_t st, const float* m, float2* specA);
bool fast_inv_x(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, const EpiParams& ep);
bool fast_inv_x_h(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, float* out, float scale);
bool fast_inv_x_q(const FastPlan& fp, const Geom& g, cudaStream_t st, const float2* specA, const EpiParams& ep);
// where the one-kernel last pass applies: x lines of 1024, 512 or 256 with their own kernel, whole warps of quads per row, no
// staircase geometry, an output that needs the per-cell tail
inline bool fast_inv_x_q_ok(const FastPlan& fp, const Geom& g, const EpiParams& ep)
{
    return fp.last_fused && fp.ok_x && fp.x_R <= 1 && (g.Px == 1024 || g.Px == 512 || g.Px == 256) && g.Nx % 128 == 0 &&
           !ep.geometry && ep.mode != EPI_HMS;
}
bool fast_lines(const FastPlan& fp, cudaStream_t st, int sgn, bool per, const ff::ColTile& ct, int nplane, float2* a,
                float2* b, int P, const AxisPlan& ap);
bool fast_y(const FastPlan& fp, const Geom& g, cudaStream_t st, int sgn, const ff::ColTile& ct, float2* a, float2* b);
bool fast_mid3(const FastPlan& fp, const Geom& g, cudaStream_t st, const ff::ColTile& ct, float2* specB,
               const float* khat);
// true: a2, a3, a4 of a whole-array evaluation may run with specB in panels (pk::k_mid_t is the z pass, the y passes
// have a kernel for Py itself)
inline bool fast_panel_ok(const FastPlan& fp, const Geom& g, const float* khat)
{
    return fp.spec_panel && fp.mid_pipe >= 2 && fp.ok_mid_t && fp.ok_panel && fp.ok_y && g.Pz == 128 &&
           (khat == fp.k_ptr || fp.has_kex_map);
}
bool fast_z_long(const FastPlan& fp, const Geom& g, cudaStream_t st, float2* specB, const float* khat);
bool fast_mul2(const FastPlan& fp, const Geom& g, cudaStream_t st, float2* specB, const float* khat);
void launch_mul2d(const Geom& g, float2* spec, const float* khat, cudaStream_t st);      // any size
// ---- per-cell tail of the split last pass ----
void launch_epi4(const Geom& g, const float* hms, const EpiParams& ep, cudaStream_t st);
void launch_epi1(const Geom& g, const float* hms, const EpiParams& ep, cudaStream_t st);
// ---- generic shared-memory passes (any 2^a 3^b 5^c 7^d length that fits the tile) ----
bool gen_set_smem();
void gen_fwd_x(const Geom& g, const FftPlan& pl, const float* m, float2* specA, int tx, size_t bytes, cudaStream_t st);
void gen_y(const Geom& g, const FftPlan& pl, int sgn, const float2* src, float2* dst, int tx, size_t bytes,
           cudaStream_t st);
void gen_mid(const Geom& g, const FftPlan& pl, float2* spec, const float* khat, int axis, int tx, size_t bytes,
             cudaStream_t st);
void gen_mul1d(const Geom& g, float2* spec, const float* khat, cudaStream_t st);
void gen_inv_x(const Geom& g, const FftPlan& pl, const float2* specA, const EpiParams& ep, int tx, size_t bytes,
               cudaStream_t st);

}  // namespace mm
