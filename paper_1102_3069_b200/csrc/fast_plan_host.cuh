// fast_plan_host.cuh -- host side of the size-specialised passes: which sizes have a kernel, twiddle tables, TMA
// tensor maps, the chunked a2-a4 driver.  Included by mm_api.cu.  Product code; shares nothing with oracle/.
#pragma once
#include <vector>
#include "mm_kernels.h"

namespace mm {

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


// P = R * Ls with Ls a length the line kernels take and the smallest R of {2, 3, 4, 5, 7, 9} (largest Ls)
inline bool choose_split(int P, int* R, int* Ls, bool real_x = false)
{
    int T, E;
    for (int r : { 2, 3, 4, 5, 7, 9 }) {
        if (P % r != 0) continue;
        const int ls = P / r;
        if (ff::split(ls, &T, &E) || (real_x && (ls == 1536 || ls == 2048))) { *R = r; *Ls = ls; return true; }
    }
    return false;
}

inline bool upload(float2** dst, const std::vector<float2>& v)
{
    return cudaMalloc(dst, v.size() * sizeof(float2)) == cudaSuccess &&
           cudaMemcpy(*dst, v.data(), v.size() * sizeof(float2), cudaMemcpyHostToDevice) == cudaSuccess;
}

inline std::vector<float2> roots_of_unity(int P)          // exp(-2 pi i j / P), j < P
{
    std::vector<float2> t((size_t)P);
    for (int j = 0; j < P; ++j) {
        const long double ang = -2.0L * 3.14159265358979323846264338327950288L * j / P;
        t[j] = make_float2((float)cosl(ang), (float)sinl(ang));
    }
    return t;
}

inline bool fast_plan_init(FastPlan& fp, const Geom& g, std::string* err)
{
    int T, E, dev = 0;
    // x: a kernel for Px itself (pair-packed rows, or the half-length form for 1536 / 2048), else R interleaved
    // real transforms of Ls = Px / R (cells per sub-row: Nx / R must be a whole number, even for the half-length form)
    fp.ok_x = ff::split(g.Px, &T, &E);
    fp.ok_xr = !fp.ok_x && (g.Px == 1536 || g.Px == 2048) && g.Nx % 2 == 0;
    fp.x_R = 1; fp.x_Ls = g.Px; fp.xs_stride = 0;
    fp.xs_real = nullptr; fp.xs_spec = nullptr; fp.twxl = nullptr;
    fp.twx = nullptr;
    if (!fp.ok_x && !fp.ok_xr) {
        int R, Ls;
        if (choose_split(g.Px, &R, &Ls, true) && g.Nx % R == 0 && (g.Nx / R) % 4 == 0 && g.Nx % 4 == 0) {
            fp.x_R = R; fp.x_Ls = Ls; fp.xs_stride = (Ls / 2 + 1 + 7) & ~7;
        }
    }
    // y and z lines
    for (int a = 1; a < 3; ++a) {
        const int P = a == 1 ? g.Py : g.Pz;
        fp.ax[a].R = 1; fp.ax[a].Ls = P; fp.ax[a].tw = nullptr; fp.ax[a].twl = nullptr;
        if (P > 1 && !ff::split(P, &T, &E)) {
            int R, Ls;
            if (choose_split(P, &R, &Ls)) { fp.ax[a].R = R; fp.ax[a].Ls = Ls; }
            else fp.ax[a].R = 0;                 // no size-specialised path along this axis
        }
    }
    fp.ax[0] = fp.ax[1];
    fp.ok_y = g.Py > 1 && fp.ax[1].R >= 1;
    fp.ok_mid3 = g.Pz >= 64 && g.Py > 1 && ff::split(g.Pz, &T, &E) && E <= 16;
    fp.ok_mul2 = g.Pz == 1 && fp.ok_y;
    fp.z_long = !fp.ok_mid3 && g.Pz >= 32 && g.Py > 1 && fp.ax[2].R >= 1 && g.Pz <= 65535 && g.Py <= 65535;
    fp.zbuf = nullptr;
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
    if (fp.z_long) {
        const size_t nz = (size_t)3 * g.Pz * g.Py * g.CxS;
        if (cudaMalloc(&fp.zbuf, nz * sizeof(float2)) != cudaSuccess || cudaMemset(fp.zbuf, 0, nz * sizeof(float2)) != cudaSuccess) {
            if (err) *err = "fast plan: z-padded spectrum allocation failed";
            return false;
        }
    }
    if (fp.x_R > 1) {
        const size_t nrow = (size_t)3 * g.Nz * g.Ny, ns = nrow * fp.x_R * fp.xs_stride;
        if (cudaMalloc(&fp.xs_real, nrow * g.Nx * sizeof(float)) != cudaSuccess ||
            cudaMalloc(&fp.xs_spec, ns * sizeof(float2)) != cudaSuccess ||
            cudaMemset(fp.xs_spec, 0, ns * sizeof(float2)) != cudaSuccess || !upload(&fp.twxl, roots_of_unity(g.Px))) {
            if (err) *err = "fast plan: x-split workspace allocation failed";
            return false;
        }
    }
    for (int a = 1; a < 3; ++a)
        if (fp.ax[a].R > 1 && !upload(&fp.ax[a].twl, roots_of_unity(a == 1 ? g.Py : g.Pz))) {
            if (err) *err = "fast plan: twiddle table allocation failed";
            return false;
        }
    // the kernels' own tables are those of the length they transform: the sub-length where a line is split
    const int xin = fp.x_R > 1 ? fp.x_Ls : g.Px;                       // length of the real transform the x kernels run
    const bool x_half = !ff::split(xin, &T, &E) && (xin == 1536 || xin == 2048);
    const int P[3] = { x_half ? xin / 2 : xin, fp.ax[1].R >= 1 ? fp.ax[1].Ls : 0, fp.ax[2].R >= 1 ? fp.ax[2].Ls : 0 };
    if (x_half) {
        const int Lc = xin / 2;
        std::vector<float2> tx((size_t)Lc);
        for (int k = 0; k < Lc; ++k) {
            const long double ang = -3.14159265358979323846264338327950288L * k / Lc;
            tx[k] = make_float2((float)cosl(ang), (float)sinl(ang));
        }
        if (!upload(&fp.twx, tx)) {
            if (err) *err = "fast plan: twiddle table allocation failed";
            return false;
        }
    }
    for (int a = 0; a < 3; ++a) {
        fp.tw[a] = nullptr;
        if (P[a] < 2 || !ff::split(P[a], &T, &E)) continue;
        std::vector<float2> tw((size_t)P[a]);
        for (int k2 = 0; k2 < E; ++k2)
            for (int t = 0; t < T; ++t) {
                const long double ang = -2.0L * 3.14159265358979323846264338327950288L * ((long long)t * k2 % P[a]) / P[a];
                tw[(size_t)k2 * T + t] = make_float2((float)cosl(ang), (float)sinl(ang));
            }
        if (!upload(&fp.tw[a], tw)) {
            if (err) *err = "fast plan: twiddle table allocation failed";
            return false;
        }
        if (a > 0) fp.ax[a].tw = fp.tw[a];
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
inline void fast_plan_maps(FastPlan& fp, const Geom& g, const float2* specA, const float2* specB, const float* khat)
{
    fp.ok_ymaps = false;
    fp.y_a = specA; fp.y_b = specB;
    fp.ok_mid_t = false;
    fp.ok_panel = false;
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
    // the same array seen in panels of 16 columns (panel_tile): 5D (32 floats, Py, Nz, 3, panel)
    {
        mm_encode_tiled_fn enc = tensor_map_encoder();
        const cuuint64_t rowb = 128, d5[5] = { 32, (cuuint64_t)g.Py, (cuuint64_t)g.Nz, 3, (cuuint64_t)((g.Cx + 15) / 16) };
        const cuuint64_t s5[4] = { rowb, rowb * g.Py, rowb * g.Py * g.Nz, rowb * g.Py * g.Nz * 3 };
        const cuuint32_t b5[5] = { 32, 1, (cuuint32_t)g.Nz, 3, 1 }, es[5] = { 1, 1, 1, 1, 1 };
        auto mk = [&](CUtensorMap* m, const cuuint32_t* bx) {
            return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 5, const_cast<float2*>(specB), d5, s5, bx, es,
                       CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                       CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
        };
        fp.ok_panel = enc && fp.ok_y && fp.ax[1].R == 1 && mk(&fp.map_spec_p, b5);
        if (fp.ok_panel && specA && g.Py == 1024) {
            // y-pass tiles: 8 columns x 256 rows
            const cuuint32_t by[4] = { 16, 256, 1, 1 };
            const cuuint64_t d4[4] = { 32, (cuuint64_t)g.Py, (cuuint64_t)3 * g.Nz, (cuuint64_t)((g.Cx + 15) / 16) };
            const cuuint64_t s4[3] = { rowb, rowb * g.Py, rowb * g.Py * g.Nz * 3 };
            const cuuint64_t d3[3] = { (cuuint64_t)2 * g.Cx, (cuuint64_t)g.Ny, (cuuint64_t)3 * g.Nz };
            const cuuint64_t s3[2] = { (cuuint64_t)g.CxS * 8, (cuuint64_t)g.CxS * 8 * g.Ny };
            const cuuint32_t es4[4] = { 1, 1, 1, 1 };
            fp.ok_ymaps =
                enc(&fp.map_yb, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, const_cast<float2*>(specB), d4, s4, by, es4,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS &&
                enc(&fp.map_ya, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float2*>(specA), d3, s3, by, es4,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
        }
    }
}

inline void fast_plan_destroy(FastPlan& fp)
{
    cudaFree(fp.twp);
    fp.twp = nullptr;
    fp.ok_mid_t = false;
    for (int a = 0; a < 3; ++a) { cudaFree(fp.tw[a]); fp.tw[a] = nullptr; }
    cudaFree(fp.twx);
    fp.twx = nullptr;
    for (int a = 1; a < 3; ++a) { cudaFree(fp.ax[a].twl); fp.ax[a].twl = nullptr; fp.ax[a].tw = nullptr; }
    cudaFree(fp.zbuf);
    fp.zbuf = nullptr;
    cudaFree(fp.xs_real); cudaFree(fp.xs_spec); cudaFree(fp.twxl);
    fp.xs_real = nullptr; fp.xs_spec = nullptr; fp.twxl = nullptr;
    for (int s = 0; s < 4; ++s) {
        if (fp.stream[s]) cudaStreamDestroy(fp.stream[s]);
        if (fp.ev_join[s]) cudaEventDestroy(fp.ev_join[s]);
        fp.stream[s] = nullptr; fp.ev_join[s] = nullptr;
    }
    if (fp.ev_fork) cudaEventDestroy(fp.ev_fork);
    fp.ev_fork = nullptr;
}


}  // namespace mm
