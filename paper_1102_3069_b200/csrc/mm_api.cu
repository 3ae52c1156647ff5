// mm_api.cu -- the C ABI of include/mm.h: context, plans, launches.
//
// Product code; shares nothing with oracle/.  No CPU fallback: without a CUDA device mm_create fails.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "../../include/mm.h"
#include "demag_host.h"
#include "mm_kernels.h"
#include "fast_plan_host.cuh"

using namespace mm;

namespace {

const double MU0 = 4e-7 * M_PI;
const double KB = 1.380649e-23;
const double MUB = 9.2740100783e-24;
const double QE = 1.602176634e-19;
const double GAMMA0_DEFAULT = 2.211e5;

thread_local std::string g_create_error;

// ---- Runge-Kutta tableaux ----
struct Tableau {
    int S;
    double A[7][7];
    double b[7];
    double bs[7];
    bool embedded;
    bool fsal;      // last row of A equals b: the last stage is f(new state) and is reused
};

Tableau make_tableau(mm_method m)
{
    Tableau t;
    std::memset(&t, 0, sizeof(t));
    switch (m) {
    case MM_RK1:
        t.S = 1; t.b[0] = 1.0;
        break;
    case MM_RK2:    // Heun
        t.S = 2; t.A[1][0] = 1.0; t.b[0] = 0.5; t.b[1] = 0.5;
        break;
    case MM_RK12:   // Heun-Euler 2(1)
        t.S = 2; t.A[1][0] = 1.0; t.b[0] = 0.5; t.b[1] = 0.5; t.bs[0] = 1.0; t.embedded = true;
        break;
    case MM_RK4:
        t.S = 4; t.A[1][0] = 0.5; t.A[2][1] = 0.5; t.A[3][2] = 1.0;
        t.b[0] = 1.0 / 6; t.b[1] = 1.0 / 3; t.b[2] = 1.0 / 3; t.b[3] = 1.0 / 6;
        break;
    case MM_RK23:   // Bogacki-Shampine 3(2)
        t.S = 4; t.A[1][0] = 0.5; t.A[2][1] = 0.75;
        t.A[3][0] = 2.0 / 9; t.A[3][1] = 1.0 / 3; t.A[3][2] = 4.0 / 9;
        t.b[0] = 2.0 / 9; t.b[1] = 1.0 / 3; t.b[2] = 4.0 / 9; t.b[3] = 0.0;
        t.bs[0] = 7.0 / 24; t.bs[1] = 0.25; t.bs[2] = 1.0 / 3; t.bs[3] = 0.125;
        t.embedded = true; t.fsal = true;
        break;
    case MM_RK3:    // Kutta's third-order method
        t.S = 3; t.A[1][0] = 0.5; t.A[2][0] = -1.0; t.A[2][1] = 2.0;
        t.b[0] = 1.0 / 6; t.b[1] = 2.0 / 3; t.b[2] = 1.0 / 6;
        break;
    case MM_RKCK: {  // Cash-Karp 5(4)
        t.S = 6;
        const double A[7][7] = {
            { 0 },
            { 1.0 / 5 },
            { 3.0 / 40, 9.0 / 40 },
            { 3.0 / 10, -9.0 / 10, 6.0 / 5 },
            { -11.0 / 54, 5.0 / 2, -70.0 / 27, 35.0 / 27 },
            { 1631.0 / 55296, 175.0 / 512, 575.0 / 13824, 44275.0 / 110592, 253.0 / 4096 } };
        std::memcpy(t.A, A, sizeof(A));
        const double b[7] = { 37.0 / 378, 0, 250.0 / 621, 125.0 / 594, 0, 512.0 / 1771, 0 };
        const double bs[7] = { 2825.0 / 27648, 0, 18575.0 / 48384, 13525.0 / 55296, 277.0 / 14336, 1.0 / 4, 0 };
        std::memcpy(t.b, b, sizeof(b));
        std::memcpy(t.bs, bs, sizeof(bs));
        t.embedded = true;
        break;
    }
    case MM_RKDP: {  // Dormand-Prince 5(4)
        t.S = 7;
        const double A[7][7] = {
            { 0 },
            { 1.0 / 5 },
            { 3.0 / 40, 9.0 / 40 },
            { 44.0 / 45, -56.0 / 15, 32.0 / 9 },
            { 19372.0 / 6561, -25360.0 / 2187, 64448.0 / 6561, -212.0 / 729 },
            { 9017.0 / 3168, -355.0 / 33, 46732.0 / 5247, 49.0 / 176, -5103.0 / 18656 },
            { 35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84 } };
        std::memcpy(t.A, A, sizeof(A));
        const double b[7] = { 35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84, 0 };
        const double bs[7] = { 5179.0 / 57600, 0, 7571.0 / 16695, 393.0 / 640, -92097.0 / 339200,
                               187.0 / 2100, 1.0 / 40 };
        std::memcpy(t.b, b, sizeof(b));
        std::memcpy(t.bs, bs, sizeof(bs));
        t.embedded = true; t.fsal = true;
        break;
    }
    default:
        t.S = 0;
    }
    return t;
}

bool smooth235(int n)
{
    for (int p : { 2, 3, 5, 7 })
        while (n % p == 0) n /= p;
    return n == 1;
}

}  // namespace

struct mm_ctx {
    Geom g;
    double cell[3];
    int pbc[3];
    cudaStream_t stream;
    bool has_mat, has_demag;
    mm_material mat;
    std::string err;
    KTimer kt;
    int fast;
    cudaStream_t gstream;   // the context's own stream for graph capture / replay (created on first use)
    cudaEvent_t gev[2];
    cudaGraphExec_t gexec;  // instantiated graph of one fixed step, reused while its key below holds
    int g_method; double g_dt; float* g_m; uint64_t g_epoch, g_per;
    uint64_t epoch;   // bumped by mm_set_material / mm_set_option / mm_set_fast_path
    int use_graph;    // mm_steps_fixed may replay a captured step (option "graph" = 0 switches it off)
    // device
    float* khat;      // demag kernel octant
    float* khat_ex;   // khat + exchange stencil on the diagonal (exchange_in_kernel), built at mm_set_material
    float2 *specA, *specB;
    float2* tw[3];
    FftPlan plan[3];
    float* kb[7];
    float* ms[2];
    float* mtmp;
    float* hfield;    // H_ms in units of Ms between the two halves of the split last pass
    float* mhost;     // device copy of a caller's host state (mm_steps_fixed_host)
    unsigned int* maxbits;
    StepCtl* ctl;     // device-side step controller state (a11)
    double* ctl_scratch;   // 4 doubles of device scratch (mm_average)
    unsigned long long* step_dev;   // device copy of step_index, advanced on the device during graph replay
    bool step_on_device;
    // stepper state
    uint64_t step_index;
    bool k0_valid;
    int k0_method;
    FastPlan fp;
    // batch of independent films (mm_create_batch): g.Nz = number of films, Pz = 1, no coupling along z
    int batch;
    float* hext_b;    // per-film applied field [batch][3], reduced units (mm_batch_set_field), or NULL
    // slab decomposition (mm_dist.cuh): g holds the LOCAL planes, gmid the geometry of the z pass on the pencil
    bool dist;
    mm_slab slab;
    std::vector<mm_slab> peers;
    int gNz;
    Geom gmid;
    float2 *slab_buf, *pencil_buf;
    size_t slab_elems, pencil_elems;
};

namespace {

mm_status fail(mm_ctx* c, mm_status s, const std::string& msg)
{
    if (c) c->err = msg;
    else g_create_error = msg;
    return s;
}

#define CUDA_TRY(c, call)                                                                         \
    do {                                                                                          \
        cudaError_t e_ = (call);                                                                  \
        if (e_ != cudaSuccess)                                                                    \
            return fail((c), e_ == cudaErrorMemoryAllocation ? MM_ENOMEM : MM_ECUDA,             \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                      \
    } while (0)

size_t ncell(const Geom& g) { return (size_t)g.Nx * g.Ny * g.Nz; }

void make_plan(FftPlan& pl, int L)
{
    pl.L = L;
    pl.nrad = 0;
    int m = L;
    while (m % 4 == 0) { pl.rad[pl.nrad++] = 4; m /= 4; }
    while (m % 2 == 0) { pl.rad[pl.nrad++] = 2; m /= 2; }
    while (m % 3 == 0) { pl.rad[pl.nrad++] = 3; m /= 3; }
    while (m % 5 == 0) { pl.rad[pl.nrad++] = 5; m /= 5; }
    while (m % 7 == 0) { pl.rad[pl.nrad++] = 7; m /= 7; }
}

// largest column count from {16, 8, 4, 2, 1} (times `mult`, plus one pad column) whose tile fits
int pick_tx(int L, int nbuf, int mult, size_t* bytes)
{
    const size_t soft = 110 * 1024, hard = 220 * 1024;
    for (size_t lim : { soft, hard })
        for (int tx : { 16, 8, 4, 2, 1 }) {
            const size_t b = (size_t)nbuf * L * (mult * tx + 1) * sizeof(float2);
            if (b <= lim) { *bytes = b; return tx; }
        }
    *bytes = 0;
    return 0;
}

// fill the material-dependent part of the epilogue parameters
void fill_material(const mm_ctx* c, EpiParams& p, uint64_t step, double dt_thermal)
{
    const mm_material& M = c->mat;
    const Geom& g = c->g;
    const double Ms = M.Ms;
    const double g0 = M.gamma0 > 0 ? M.gamma0 : GAMMA0_DEFAULT;
    // a slab has z neighbours even with one local plane; the films of a batch are not coupled
    const int ext[3] = { g.Nx, g.Ny, c->dist ? c->gNz : (c->batch ? 1 : g.Nz) };
    p.demag = M.demag ? 1 : 0;
    const bool ex_in_k = M.exchange_in_kernel && M.demag;      // then the convolution carries the exchange field
    for (int a = 0; a < 3; ++a)
        p.wex[a] = (ext[a] > 1 && !ex_in_k) ? (float)(2.0 * M.Aex / (MU0 * Ms * Ms * c->cell[a] * c->cell[a])) : 0.f;
    double u[3] = { M.anis_u[0], M.anis_u[1], M.anis_u[2] };
    const double un = std::sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
    p.kan = (M.Ku != 0.0 && un > 0) ? (float)(2.0 * M.Ku / (MU0 * Ms * Ms)) : 0.f;
    for (int a = 0; a < 3; ++a) {
        p.u[a] = un > 0 ? (float)(u[a] / un) : 0.f;
        p.hext[a] = (float)(M.Bext[a] / (MU0 * Ms));
    }
    p.hext_b = c->batch ? c->hext_b : nullptr;
    p.plane_cells = (unsigned)(g.Nx * g.Ny);
    p.geometry = M.geometry ? 1 : 0;
    p.cubic = (M.K1 != 0.0 || M.K2 != 0.0) ? 1 : 0;
    if (p.cubic) {
        // reading A14: c1 normalised, c2 orthogonalised against c1, c3 = c1 x c2
        double a[3] = { M.anis_c1[0], M.anis_c1[1], M.anis_c1[2] }, b[3] = { M.anis_c2[0], M.anis_c2[1], M.anis_c2[2] };
        const double na = std::sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
        for (int i = 0; i < 3; ++i) a[i] /= na;
        const double ab = a[0] * b[0] + a[1] * b[1] + a[2] * b[2];
        for (int i = 0; i < 3; ++i) b[i] -= ab * a[i];
        const double nb = std::sqrt(b[0] * b[0] + b[1] * b[1] + b[2] * b[2]);
        for (int i = 0; i < 3; ++i) b[i] /= nb;
        const double cc[3] = { a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0] };
        for (int i = 0; i < 3; ++i) { p.c1[i] = (float)a[i]; p.c2[i] = (float)b[i]; p.c3[i] = (float)cc[i]; }
        p.k1c = (float)(2.0 * M.K1 / (MU0 * Ms * Ms));
        p.k2c = (float)(2.0 * M.K2 / (MU0 * Ms * Ms));
    }
    p.thermal = (M.T > 0.0 && dt_thermal > 0.0) ? 1 : 0;
    p.sig_th = 0.f;
    if (p.thermal) {
        const double V = c->cell[0] * c->cell[1] * c->cell[2];
        p.sig_th = (float)(std::sqrt(2.0 * M.alpha * KB * M.T / (g0 * MU0 * Ms * V * dt_thermal)) / Ms);
    }
    p.key0 = (uint32_t)(M.seed & 0xffffffffu);
    p.key1 = (uint32_t)(M.seed >> 32);
    p.step0 = (uint32_t)(step & 0xffffffffu);
    p.step1 = (uint32_t)(step >> 32);
    p.step_dev = c->step_on_device ? c->step_dev : nullptr;
    p.alpha = (float)M.alpha;
    p.inv1pa2 = (float)(1.0 / (1.0 + M.alpha * M.alpha));
    p.stt = (M.j[0] != 0.0 || M.j[1] != 0.0 || M.j[2] != 0.0) ? 1 : 0;
    const double bj = M.P * MUB / (QE * Ms * (1.0 + M.xi * M.xi));
    for (int a = 0; a < 3; ++a)
        p.cj[a] = (p.stt && ext[a] > 1) ? (float)(bj * M.j[a] / (2.0 * c->cell[a] * g0 * Ms)) : 0.f;
    const double cad = M.stt_literal_eq7 ? 1.0 : 1.0 + M.alpha * M.xi;
    p.c_ad = (float)(cad / (1.0 + M.alpha * M.alpha));
    p.c_nad = (float)((M.xi - M.alpha) / (1.0 + M.alpha * M.alpha));
}


// ---- one evaluation: the five passes, the last one carrying the epilogue `ep`.  Each pass runs its
// size-specialised kernel (fft_fast*.cuh) when one exists for the grid and the bit of c->fast is set,
// else the generic shared-memory kernel; both use the same layouts. ----
mm_status launch_eval(mm_ctx* c, const EpiParams& ep)
{
    if (c->dist) return fail(c, MM_ESTATE, "a slab context evaluates through mm_dist_forward / _mid / _backward");
    const Geom& g = c->g;
    cudaStream_t st = c->stream;
    const FastPlan& fp = c->fp;
    size_t bytes;
    // mm_demag_field (EPI_HMS) always uses the pure magnetostatic kernel
    const float* kh = (ep.mode != EPI_HMS && c->mat.exchange_in_kernel && c->mat.demag && c->khat_ex) ? c->khat_ex
                                                                                                       : c->khat;
    if (ep.demag) {
        {   // a1
            c->kt.begin(KT_FWD_X);
            if (!((c->fast & FAST_FWD_X) && fast_fwd_x(fp, g, st, ep.m_in, c->specA))) {
                const int tx = pick_tx(g.Px, 2, 1, &bytes);
                if (!tx) return fail(c, MM_EUNSUPPORTED, "x line too long for the shared-memory tile");
                gen_fwd_x(g, c->plan[0], ep.m_in, c->specA, tx, bytes, st);
            }
            c->kt.end(KT_FWD_X);
        }
        if (g.Pz > 1 && (c->fast & FAST_CHUNK) && (c->fast & FAST_Y) && (c->fast & FAST_MID) && fp.chunk_w > 0) {
            // a2-a4 chunked over kx so that the y-padded spectrum stays in L2 (timed as one category)
            c->kt.begin(KT_MID);
            if (!fast_yzy_chunked(c->fp, g, st, c->specA, c->specB, kh))
                return fail(c, MM_ECUDA, "chunked y-z-y launch failed");
            c->kt.end(KT_MID);
            c->kt.launches += 3 * ((g.Cx + fp.chunk_w - 1) / fp.chunk_w) - 1;
        } else if (g.Pz > 1) {
            const bool panel = (c->fast & FAST_Y) && (c->fast & FAST_MID) && fast_panel_ok(fp, g, kh);
            const ff::ColTile wt = panel ? panel_tile(g) : whole_tile(g);
            {   // a2
                c->kt.begin(KT_FWD_Y);
                if (!((c->fast & FAST_Y) && fast_y(fp, g, st, -1, wt, c->specA, c->specB))) {
                    const int tx = pick_tx(g.Py, 2, 1, &bytes);
                    if (!tx) return fail(c, MM_EUNSUPPORTED, "y line too long for the shared-memory tile");
                    gen_y(g, c->plan[1], -1, c->specA, c->specB, tx, bytes, st);
                }
                c->kt.end(KT_FWD_Y);
            }
            {   // a3
                c->kt.begin(KT_MID);
                if (!((c->fast & FAST_MID) && (fast_mid3(fp, g, st, wt, c->specB, kh) || fast_z_long(fp, g, st, c->specB, kh)))) {
                    const int tx = pick_tx(g.Pz, 4, 1, &bytes);
                    if (!tx) return fail(c, MM_EUNSUPPORTED, "z line too long for the shared-memory tile");
                    gen_mid(g, c->plan[2], c->specB, kh, 2, tx, bytes, st);
                }
                c->kt.end(KT_MID);
            }
            {   // a4
                c->kt.begin(KT_INV_Y);
                if (!((c->fast & FAST_Y) && fast_y(fp, g, st, 1, wt, c->specA, c->specB))) {
                    const int tx = pick_tx(g.Py, 2, 1, &bytes);
                    gen_y(g, c->plan[1], 1, c->specB, c->specA, tx, bytes, st);
                }
                c->kt.end(KT_INV_Y);
            }
        } else if (g.Py > 1) {
            if ((c->fast & FAST_MID) && fp.ok_mul2) {
                // 2D: y forward, k-space multiply, y inverse as three launches (the spectra of a 2D grid
                // are L2-resident, so the extra round trip does not reach HBM)
                const ff::ColTile wt = whole_tile(g);
                c->kt.begin(KT_FWD_Y);
                fast_y(fp, g, st, -1, wt, c->specA, c->specB);
                c->kt.end(KT_FWD_Y);
                c->kt.begin(KT_MID);
                fast_mul2(fp, g, st, c->specB, kh);
                c->kt.end(KT_MID);
                c->kt.begin(KT_INV_Y);
                fast_y(fp, g, st, 1, wt, c->specA, c->specB);
                c->kt.end(KT_INV_Y);
            } else if (const int tx = pick_tx(g.Py, 4, 1, &bytes)) {
                // generic: y forward, multiply, y inverse in one kernel
                c->kt.begin(KT_MID);
                gen_mid(g, c->plan[1], c->specA, kh, 1, tx, bytes, st);
                c->kt.end(KT_MID);
            } else {
                // very long y lines (four tile buffers do not fit): three launches through specB
                const int ty = pick_tx(g.Py, 2, 1, &bytes);
                if (!ty) return fail(c, MM_EUNSUPPORTED, "y line too long for the shared-memory tile");
                c->kt.begin(KT_FWD_Y);
                gen_y(g, c->plan[1], -1, c->specA, c->specB, ty, bytes, st);
                c->kt.end(KT_FWD_Y);
                c->kt.begin(KT_MID);
                launch_mul2d(g, c->specB, kh, st);
                c->kt.end(KT_MID);
                c->kt.begin(KT_INV_Y);
                gen_y(g, c->plan[1], 1, c->specB, c->specA, ty, bytes, st);
                c->kt.end(KT_INV_Y);
            }
        } else {
            c->kt.begin(KT_MID);
            gen_mul1d(g, c->specA, kh, st);
            c->kt.end(KT_MID);
        }
    }
    // a5-a10
    bool done = false;
    if (ep.demag && (c->fast & FAST_SPLIT) && fast_inv_x_q_ok(fp, g, ep)) {
        c->kt.begin(KT_INV_X);
        done = fast_inv_x_q(fp, g, st, c->specA, ep);
        c->kt.end(KT_INV_X);
    }
    if (!done && ep.demag && (c->fast & FAST_SPLIT) && (fp.ok_x || fp.ok_xr || fp.x_R > 1) && (g.Nx % 4 == 0 || ep.geometry)) {
        // split variant: inverse x pass -> H_ms field, then the streaming per-cell tail
        c->kt.begin(KT_INV_X);
        if (ep.mode == EPI_HMS) {
            done = fast_inv_x_h(fp, g, st, c->specA, ep.out, ep.out_scale);
            c->kt.end(KT_INV_X);
        } else {
            done = fast_inv_x_h(fp, g, st, c->specA, c->hfield, 1.0f);
            c->kt.end(KT_INV_X);
            if (done) {
                c->kt.begin(KT_EPI);
                if (ep.geometry) launch_epi1(g, c->hfield, ep, st);
                else launch_epi4(g, c->hfield, ep, st);
                c->kt.end(KT_EPI);
            }
        }
    }
    if (!done) {
        c->kt.begin(KT_INV_X);
        if (!(ep.demag && !ep.geometry && (c->fast & FAST_INV_X) && fast_inv_x(fp, g, st, c->specA, ep))) {
            const int tx = pick_tx(g.Px, 2, 3, &bytes);
            if (!tx) return fail(c, MM_EUNSUPPORTED, "x line too long for the shared-memory tile");
            gen_inv_x(g, c->plan[0], c->specA, ep, tx, bytes, st);
        }
        c->kt.end(KT_INV_X);
    }
    CUDA_TRY(c, cudaGetLastError());
    return MM_OK;
}

__global__ void k_khat_exchange(Geom g, const float* __restrict__ khat, float* __restrict__ out, float wx, float wy,
                                float wz);

// (re)build khat_ex = khat + exchange stencil when the material asks for the paper's variant
mm_status refresh_khat_ex(mm_ctx* c)
{
    if (!(c->has_mat && c->has_demag && c->mat.exchange_in_kernel && c->mat.demag)) return MM_OK;
    const Geom& g = c->g;
    const size_t nK = (size_t)6 * g.Cz * g.Cy * g.CxK;
    if (!c->khat_ex) {
        CUDA_TRY(c, cudaMalloc(&c->khat_ex, (nK + (size_t)g.Cy * g.CxK) * sizeof(float)));
        CUDA_TRY(c, cudaMemsetAsync(c->khat_ex + nK, 0, (size_t)g.Cy * g.CxK * sizeof(float), c->stream));
        c->fp.has_kex_map = c->fp.ok_mid_t && khat_map(&c->fp.map_kex, g, c->khat_ex, c->fp.mid_cols);
    }
    const double Ms = c->mat.Ms;
    const int ext[3] = { g.Nx, g.Ny, g.Nz };
    float w[3];
    for (int a = 0; a < 3; ++a)
        w[a] = ext[a] > 1 ? (float)(2.0 * c->mat.Aex / (MU0 * Ms * Ms * c->cell[a] * c->cell[a])) : 0.f;
    k_khat_exchange<<<c->fp.nsm * 8, 256, 0, c->stream>>>(g, c->khat, c->khat_ex, w[0], w[1], w[2]);
    CUDA_TRY(c, cudaGetLastError());
    return MM_OK;
}

mm_status check_ready(mm_ctx* c)
{
    if (!c) return MM_EINVAL;
    if (c->dist && (c->mat.exchange_in_kernel || c->mat.geometry))
        return fail(c, MM_EUNSUPPORTED, "slab decomposition: exchange_in_kernel and geometry are not supported");
    if (!c->has_mat) return fail(c, MM_ESTATE, "mm_set_material has not been called");
    if (!c->has_demag) return fail(c, MM_ESTATE, "mm_demag_init has not been called");
    return MM_OK;
}

double gamma0_of(const mm_ctx* c) { return c->mat.gamma0 > 0 ? c->mat.gamma0 : GAMMA0_DEFAULT; }

// m_out = [normalise](m_n + sum_j a_j k_j): used when an evaluation is skipped (FSAL reuse).
__global__ void k_combine(size_t n, const float* __restrict__ m_n, float* __restrict__ m_out, int na,
                          float a0, float a1, const float* __restrict__ k0, const float* __restrict__ k1,
                          const float* __restrict__ dt_scale)
{
    if (dt_scale) { a0 *= *dt_scale; a1 *= *dt_scale; }
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < 3 * n;
         i += (size_t)gridDim.x * blockDim.x) {
        float v = m_n[i] + a0 * k0[i];
        if (na > 1) v += a1 * k1[i];
        m_out[i] = v;
    }
}

__global__ void k_normalise(size_t n, const float* __restrict__ src, float* __restrict__ dst)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float x = src[i], y = src[i + n], z = src[i + 2 * n];
        const float q = x * x + y * y + z * z;
        const float s = q > 0.f ? rsqrtf(q) : 0.f;
        dst[i] = x * s; dst[i + n] = y * s; dst[i + 2 * n] = z * s;
    }
}

// K-hat with the exchange stencil added to its diagonal: in k space the 6-neighbour stencil
// is sum_a w_a (2 cos(2 pi k_a / P_a) - 2); the convolution carries the factor 1/(Px Py Pz) of K-hat.
__global__ void k_khat_exchange(Geom g, const float* __restrict__ khat, float* __restrict__ out, float wx, float wy,
                                float wz)
{
    const size_t nC = (size_t)g.CxK * g.Cy * g.Cz;
    const float norm = 1.0f / ((float)g.Px * (float)g.Py * (float)g.Pz);
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < 6 * nC; i += (size_t)gridDim.x * blockDim.x) {
        const size_t r = i % nC;
        const int comp = (int)(i / nC);
        float v = khat[i];
        if (comp < 3) {
            const int kx = (int)(r % g.CxK), ky = (int)((r / g.CxK) % g.Cy), kz = (int)(r / ((size_t)g.CxK * g.Cy));
            if (kx < g.Cx) {
                const float ex = wx * (2.0f * cospif(2.0f * kx / (float)g.Px) - 2.0f) +
                                 wy * (2.0f * cospif(2.0f * ky / (float)g.Py) - 2.0f) +
                                 wz * (2.0f * cospif(2.0f * kz / (float)g.Pz) - 2.0f);
                v += norm * ex;
            }
        }
        out[i] = v;
    }
}

__global__ void k_copy4(const float4* __restrict__ src, float4* __restrict__ dst, size_t n4)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x)
        dst[i] = src[i];
}

// One stage of `tab` (0-based s).  Enqueues only.
EpiParams stage_params(mm_ctx* c, float* m_dev, const Tableau& tab, int s, double dt, uint64_t step,
                       bool adaptive_target, bool dev_dt)
{
    const int S = tab.S;
    // dev_dt: the step length lives on the device (StepCtl::dtr); the tableau goes in unscaled
    const double dtr = dev_dt ? 1.0 : dt * gamma0_of(c) * c->mat.Ms;
    EpiParams ep;
    std::memset(&ep, 0, sizeof(ep));
    if (dev_dt) ep.dt_scale = &c->ctl->dtr;
    fill_material(c, ep, step, dt);
    ep.mode = EPI_STAGE;
    ep.m_in = s == 0 ? m_dev : c->ms[(s - 1) & 1];
    ep.m_n = m_dev;
    ep.maxbits = c->maxbits;
    const bool last = s == S - 1;
    // k_s must be stored if a later stage row, the final combination or the FSAL hand-over reads it
    bool store_k = false;
    for (int r = s + 2; r < S; ++r) store_k |= tab.A[r][s] != 0.0;
    if (!last) {
        if (!tab.fsal) store_k |= tab.b[s] != 0.0;                       // read by the final combine
        if (tab.embedded) store_k |= (tab.b[s] - tab.bs[s]) != 0.0;      // read by the error estimate
    }
    if (tab.fsal && last) store_k = true;                                // handed to the next step
    ep.k_out = store_k ? c->kb[s] : nullptr;
    const double* row = nullptr;     // coefficients of the state this stage produces
    if (!last) row = tab.A[s + 1];
    else if (!tab.fsal) row = tab.b;
    if (row) {
        ep.a_self = (float)(dtr * row[s]);
        for (int j = 0; j < s; ++j)
            if (row[j] != 0.0) {
                ep.a[ep.na] = (float)(dtr * row[j]);
                ep.ka[ep.na] = c->kb[j];
                ep.na++;
            }
        const bool is_new_state = last || (tab.fsal && s == S - 2);
        ep.normalise = is_new_state ? 1 : 0;
        if (last) ep.m_out = (S > 1 && !adaptive_target) ? m_dev : c->mtmp;
        else ep.m_out = c->ms[s & 1];
    }
    if (last) {
        ep.do_err = 1;
        if (tab.embedded) {
            ep.e_self = (float)(dtr * (tab.b[s] - tab.bs[s]));
            for (int j = 0; j < s; ++j) {
                const double d = tab.b[j] - tab.bs[j];
                if (d != 0.0) {
                    ep.e[ep.ne] = (float)(dtr * d);
                    ep.ke[ep.ne] = c->kb[j];
                    ep.ne++;
                }
            }
        } else {
            ep.e_self = (float)dtr;   // max |dm| of the last stage: NaN sentinel and diagnostics
        }
    }
    return ep;
}

mm_status run_stage(mm_ctx* c, float* m_dev, const Tableau& tab, int s, double dt, uint64_t step,
                    bool adaptive_target, bool dev_dt = false)
{
    return launch_eval(c, stage_params(c, m_dev, tab, s, dt, step, adaptive_target, dev_dt));
}

// One trial step; enqueues everything, no synchronisation.  After it, maxbits holds the error
// estimate and the new state is in *newstate (m_dev itself when written in place).
mm_status enqueue_step(mm_ctx* c, float* m_dev, mm_method method, const Tableau& tab, double dt,
                       bool adaptive_target, float** newstate, bool dev_dt = false)
{
    const int S = tab.S;
    const size_t n = ncell(c->g);
    CUDA_TRY(c, cudaMemsetAsync(c->maxbits, 0, sizeof(unsigned int), c->stream));
    const uint64_t step = c->step_index;
    int s0 = 0;
    // a method without the FSAL property overwrites kb[0] with its own first stage: the saved one is gone
    if (!tab.fsal) c->k0_valid = false;
    // with a thermal field the saved stage carries the previous step's draw (reading A6: one draw per
    // step, held over that step's own stages): evaluate k_1 afresh
    if (tab.fsal && c->k0_valid && c->k0_method == (int)method && !(c->mat.T > 0)) {
        // k_1 of this step is the last stage of the previous accepted step: skip the evaluation
        const double dtr = dev_dt ? 1.0 : dt * gamma0_of(c) * c->mat.Ms;
        c->kt.begin(KT_OTHER);
        k_combine<<<c->fp.nsm * 8, 256, 0, c->stream>>>(n, m_dev, c->ms[0], 1, (float)(dtr * tab.A[1][0]), 0.f,
                                                  c->kb[0], c->kb[0], dev_dt ? &c->ctl->dtr : nullptr);
        c->kt.end(KT_OTHER);
        s0 = 1;
    }
    for (int s = s0; s < S; ++s) {
        mm_status st = run_stage(c, m_dev, tab, s, dt, step, adaptive_target, dev_dt);
        if (st != MM_OK) return st;
    }
    if (tab.fsal) *newstate = c->ms[(S - 2) & 1];
    else *newstate = (S > 1 && !adaptive_target) ? m_dev : c->mtmp;
    return MM_OK;
}

mm_status commit_step(mm_ctx* c, float* m_dev, mm_method method, const Tableau& tab, float* newstate)
{
    const size_t n = ncell(c->g);
    if (newstate != m_dev)
        CUDA_TRY(c, cudaMemcpyAsync(m_dev, newstate, 3 * n * sizeof(float), cudaMemcpyDeviceToDevice, c->stream));
    if (tab.fsal) {
        std::swap(c->kb[0], c->kb[tab.S - 1]);
        c->k0_valid = true;
        c->k0_method = (int)method;
    }
    c->step_index++;
    return MM_OK;
}

}  // namespace

// ==================================================================================================
extern "C" {

mm_status mm_create(mm_ctx** out, const int grid[3], const double cellsize[3], const int pbc[3],
                    void* cuda_stream)
{
    if (!out || !grid || !cellsize || !pbc) return fail(nullptr, MM_EINVAL, "NULL argument");
    *out = nullptr;
    for (int a = 0; a < 3; ++a) {
        if (grid[a] < 1) return fail(nullptr, MM_EINVAL, "grid sizes must be >= 1");
        if (!(cellsize[a] > 0)) return fail(nullptr, MM_EINVAL, "cell sizes must be > 0");
        if (pbc[a] < 0) return fail(nullptr, MM_EINVAL, "pbc must be >= 0");
    }
    int P[3];
    if (mm_padded_size_of(grid, pbc, P, nullptr) != MM_OK)
        return fail(nullptr, MM_EUNSUPPORTED, "padded size has a prime factor other than 2, 3, 5, 7");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(nullptr, MM_ECUDA, "no CUDA device: this library has no CPU fallback");
    }
    mm_ctx* c = new (std::nothrow) mm_ctx();
    if (!c) return fail(nullptr, MM_ENOMEM, "host allocation failed");
    Geom& g = c->g;
    g.Nx = grid[0]; g.Ny = grid[1]; g.Nz = grid[2];
    g.Px = P[0]; g.Py = P[1]; g.Pz = P[2];
    g.Cx = P[0] / 2 + 1; g.Cy = P[1] / 2 + 1; g.Cz = P[2] / 2 + 1;
    g.CxS = (g.Cx + 7) & ~7;     // rows start on 64-byte boundaries
    // K-hat rows: 16-byte multiples; whole 128-byte lines where the TMA tiles of pk::k_mid_t read 64-byte pieces of them
    // (a piece that straddles lines made the pass read 1.3 - 1.5 times its K-hat bytes)
    g.CxK = g.Cx >= 128 ? (g.Cx + 31) & ~31 : (g.Cx + 3) & ~3;
    g.perx = pbc[0] > 0; g.pery = pbc[1] > 0; g.perz = pbc[2] > 0;
    for (int a = 0; a < 3; ++a) { c->cell[a] = cellsize[a]; c->pbc[a] = pbc[a]; }
    c->stream = (cudaStream_t)cuda_stream;
    c->has_mat = c->has_demag = false;
    std::memset(&c->kt, 0, sizeof(c->kt));
    c->kt.stream = c->stream;
    c->mhost = nullptr;
    c->hfield = nullptr;
    c->fast = FAST_ALL;
    c->gstream = nullptr;
    c->gev[0] = c->gev[1] = nullptr;
    c->use_graph = 1;
    c->batch = 0; c->hext_b = nullptr;
    c->dist = false; c->gNz = grid[2]; c->slab_buf = c->pencil_buf = nullptr; c->slab_elems = c->pencil_elems = 0;
    c->gexec = nullptr; c->g_method = -1; c->g_dt = 0.0; c->g_m = nullptr; c->g_epoch = 0; c->g_per = 0;
    c->epoch = 1;
    c->khat = nullptr; c->khat_ex = nullptr; c->specA = c->specB = nullptr;
    for (int a = 0; a < 3; ++a) c->tw[a] = nullptr;
    for (int i = 0; i < 7; ++i) c->kb[i] = nullptr;
    c->ms[0] = c->ms[1] = c->mtmp = nullptr;
    c->maxbits = nullptr;
    c->ctl = nullptr;
    c->ctl_scratch = nullptr;
    c->step_dev = nullptr;
    c->step_on_device = false;
    c->step_index = 0;
    c->k0_valid = false;
    c->k0_method = -1;
    std::memset(&c->fp, 0, sizeof(c->fp));
    {
        int dev = 0;
        c->fp.nsm = 0;
        if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&c->fp.nsm, cudaDevAttrMultiProcessorCount, dev);
        if (c->fp.nsm < 1) c->fp.nsm = 1;
    }
    c->fp.x_pipe = 1; c->fp.spec_panel = 1; c->fp.y_tma = 2; c->fp.last_fused = 1; c->fp.q_blocks = 4; c->fp.mid_pipe = 2; c->fp.mid_cols = 16; c->fp.chunk_w = 0; c->fp.nstream = 3;     // mm_set_option defaults
    *out = c;
    return MM_OK;
}

mm_status mm_set_material(mm_ctx* c, const mm_material* mat)
{
    if (!c || !mat) return MM_EINVAL;
    if (!(mat->Ms > 0)) return fail(c, MM_EINVAL, "Ms must be > 0");
    if (mat->Aex < 0 || mat->alpha < 0 || mat->T < 0) return fail(c, MM_EINVAL, "Aex, alpha, T must be >= 0");
    if (mat->Ku != 0.0 && mat->anis_u[0] == 0.0 && mat->anis_u[1] == 0.0 && mat->anis_u[2] == 0.0)
        return fail(c, MM_EINVAL, "anisotropy axis is zero");
    if (mat->K1 != 0.0 || mat->K2 != 0.0) {
        const double* a = mat->anis_c1;
        const double* b = mat->anis_c2;
        const double cx = a[1] * b[2] - a[2] * b[1], cy = a[2] * b[0] - a[0] * b[2], cz = a[0] * b[1] - a[1] * b[0];
        if (cx * cx + cy * cy + cz * cz == 0.0) return fail(c, MM_EINVAL, "cubic anisotropy axes are zero or parallel");
    }
    c->mat = *mat;
    c->has_mat = true;
    c->epoch++;
    c->k0_valid = false;
    return refresh_khat_ex(c);
}

// everything mm_demag_init allocates; pointers are reset so that the call can be repeated after a failure
static void free_workspaces(mm_ctx* c)
{
    auto fr = [](auto*& p) { if (p) cudaFree(p); p = nullptr; };
    fr(c->khat); fr(c->khat_ex); fr(c->specA); fr(c->specB);
    for (int a = 0; a < 3; ++a) fr(c->tw[a]);
    for (int i = 0; i < 7; ++i) fr(c->kb[i]);
    fr(c->ms[0]); fr(c->ms[1]); fr(c->mtmp); fr(c->mhost); fr(c->hfield);
    fr(c->hext_b);
    fr(c->maxbits); fr(c->ctl); fr(c->ctl_scratch); fr(c->step_dev); fr(c->slab_buf); fr(c->pencil_buf);
    fast_plan_destroy(c->fp);
}

static mm_status demag_init_impl(mm_ctx* c);

mm_status mm_demag_init(mm_ctx* c)
{
    if (!c) return MM_EINVAL;
    if (c->has_demag) return MM_OK;
    mm_status s = demag_init_impl(c);
    // the set-up copies and memsets run on the legacy default stream, the kernels of this context on the
    // caller's stream (possibly non-blocking): order everything before returning (the call is blocking)
    if (s == MM_OK && cudaDeviceSynchronize() != cudaSuccess) s = fail(c, MM_ECUDA, "mm_demag_init: device synchronisation failed");
    if (s != MM_OK) {
        c->has_demag = false;
        free_workspaces(c);
        cudaGetLastError();
    }
    return s;
}

static mm_status demag_init_impl(mm_ctx* c)
{
    const Geom& g = c->g;
    // the kernel is that of the whole grid (slab ranks) / of one film (batch)
    const int grid[3] = { g.Nx, g.Ny, c->dist ? c->gNz : (c->batch ? 1 : g.Nz) };
    const size_t nC = (size_t)g.Cx * g.Cy * g.Cz;
    std::vector<float> kh;
    try {
        kh.resize(6 * nC);
    } catch (const std::bad_alloc&) {
        return fail(c, MM_ENOMEM, "host allocation of K-hat failed");
    }
    std::string err;
    const int rc = mmh::build_khat(c->cell, grid, c->pbc, kh.data(), &err);
    if (rc != 0) return fail(c, (mm_status)rc, err);
    const size_t nrow = (size_t)6 * g.Cz * g.Cy;         // device rows are padded to CxK floats (zeros)
    // a rank of a slab decomposition keeps only the columns it transforms along z
    const int k0 = c->dist ? c->slab.kx0 : 0, kw = c->dist ? c->slab.kx1 - c->slab.kx0 : g.Cx;
    const size_t kstride = c->dist ? (size_t)c->gmid.CxK : (size_t)g.CxK;
    // one spare kz plane at the end: the even / odd kz view of the TMA map addresses row kz = Cz (never used)
    CUDA_TRY(c, cudaMalloc(&c->khat, (nrow + g.Cy) * kstride * sizeof(float)));
    CUDA_TRY(c, cudaMemset(c->khat, 0, (nrow + g.Cy) * kstride * sizeof(float)));
    CUDA_TRY(c, cudaMemcpy2D(c->khat, kstride * sizeof(float), kh.data() + k0, g.Cx * sizeof(float), kw * sizeof(float),
                             nrow, cudaMemcpyHostToDevice));
    if (c->dist) {
        size_t wsum = 0;
        for (const mm_slab& q : c->peers) wsum += (size_t)((q.kx1 - q.kx0 + 7) & ~7);
        c->slab_elems = (size_t)3 * g.Nz * g.Py * wsum;
        c->pencil_elems = (size_t)3 * c->gNz * g.Py * (size_t)((kw + 7) & ~7);
        CUDA_TRY(c, cudaMalloc(&c->slab_buf, c->slab_elems * sizeof(float2)));
        CUDA_TRY(c, cudaMalloc(&c->pencil_buf, c->pencil_elems * sizeof(float2)));
        CUDA_TRY(c, cudaMemset(c->slab_buf, 0, c->slab_elems * sizeof(float2)));
        CUDA_TRY(c, cudaMemset(c->pencil_buf, 0, c->pencil_elems * sizeof(float2)));
    }
    const size_t nA = (size_t)3 * g.Nz * g.Ny * g.CxS;
    CUDA_TRY(c, cudaMalloc(&c->specA, nA * sizeof(float2)));
    CUDA_TRY(c, cudaMemset(c->specA, 0, nA * sizeof(float2)));
    if (g.Py > 1 && !c->dist) {      // (a slab rank's y passes write into / read from slab_buf)
        const size_t nB = (size_t)3 * g.Nz * g.Py * specb_cols(g);     // room for the 16-column panel form
        CUDA_TRY(c, cudaMalloc(&c->specB, nB * sizeof(float2)));
        CUDA_TRY(c, cudaMemset(c->specB, 0, nB * sizeof(float2)));
    }
    const int P[3] = { g.Px, g.Py, g.Pz };
    for (int a = 0; a < 3; ++a) {
        make_plan(c->plan[a], P[a]);
        std::vector<float2> tw(P[a]);
        for (int q = 0; q < P[a]; ++q) {
            const long double ang = -2.0L * 3.14159265358979323846264338327950288L * q / P[a];
            tw[q] = make_float2((float)cosl(ang), (float)sinl(ang));
        }
        CUDA_TRY(c, cudaMalloc(&c->tw[a], P[a] * sizeof(float2)));
        CUDA_TRY(c, cudaMemcpy(c->tw[a], tw.data(), P[a] * sizeof(float2), cudaMemcpyHostToDevice));
        c->plan[a].tw = c->tw[a];
    }
    const size_t fb = 3 * ncell(g) * sizeof(float);
    for (int i = 0; i < 7; ++i) CUDA_TRY(c, cudaMalloc(&c->kb[i], fb));
    for (int i = 0; i < 2; ++i) CUDA_TRY(c, cudaMalloc(&c->ms[i], fb));
    CUDA_TRY(c, cudaMalloc(&c->mtmp, fb));
    CUDA_TRY(c, cudaMalloc(&c->mhost, fb));
    CUDA_TRY(c, cudaMalloc(&c->hfield, fb));
    CUDA_TRY(c, cudaMalloc(&c->maxbits, 2 * sizeof(unsigned int)));     // [0] per step, [1] running maximum
    CUDA_TRY(c, cudaMemset(c->maxbits, 0, 2 * sizeof(unsigned int)));
    CUDA_TRY(c, cudaMalloc(&c->ctl, sizeof(StepCtl)));
    CUDA_TRY(c, cudaMemset(c->ctl, 0, sizeof(StepCtl)));
    CUDA_TRY(c, cudaMalloc(&c->ctl_scratch, 4 * sizeof(double)));
    CUDA_TRY(c, cudaMalloc(&c->step_dev, sizeof(unsigned long long)));
    // (status of the set-up steps below)
    if (!gen_set_smem()) return fail(c, MM_ECUDA, "cannot raise the shared-memory limit of the generic kernels");
    std::string ferr;
    if (!fast_plan_init(c->fp, g, &ferr)) return fail(c, MM_ECUDA, ferr);
    if (c->batch && !((c->fp.ok_x || c->fp.ok_xr) && c->fp.ok_mul2 && g.Nx % 4 == 0))
        return fail(c, MM_EUNSUPPORTED, "mm_create_batch needs padded x and y lengths with size-specialised kernels (32 ... 1024) and Nx % 4 == 0");
    if (c->dist) {
        if (!(c->fp.ok_x && c->fp.ok_y && c->fp.ok_mid3))
            return fail(c, MM_EUNSUPPORTED, "mm_create_dist needs size-specialised kernels for all three padded lengths");
    } else {
        fast_plan_maps(c->fp, g, c->specA, c->specB, c->khat);
    }
    c->has_demag = true;
    return refresh_khat_ex(c);
}

static mm_status eval_to(mm_ctx* c, const float* m_dev, float* out, int mode, uint64_t step, double dt_th)
{
    mm_status s = check_ready(c);
    if (s != MM_OK) return s;
    if (c->dist) return fail(c, MM_ESTATE, "a slab context evaluates through mm_dist_forward / _mid / _backward");
    if (!m_dev || !out) return fail(c, MM_EINVAL, "NULL device pointer");
    EpiParams ep;
    std::memset(&ep, 0, sizeof(ep));
    fill_material(c, ep, step, dt_th);
    ep.mode = mode;
    ep.m_in = m_dev;
    ep.out = out;
    ep.out_scale = mode == EPI_TORQUE ? (float)(gamma0_of(c) * c->mat.Ms) : (float)c->mat.Ms;
    if (mode == EPI_HMS) ep.demag = 1;
    return launch_eval(c, ep);
}

mm_status mm_heff(mm_ctx* c, const float* m_dev, float* H_dev, double t, uint64_t step, double dt_th)
{
    (void)t;
    return eval_to(c, m_dev, H_dev, EPI_HEFF, step, dt_th);
}

mm_status mm_torque(mm_ctx* c, const float* m_dev, float* dmdt_dev, double t, uint64_t step, double dt_th)
{
    (void)t;
    return eval_to(c, m_dev, dmdt_dev, EPI_TORQUE, step, dt_th);
}

mm_status mm_demag_field(mm_ctx* c, const float* m_dev, float* H_dev)
{
    return eval_to(c, m_dev, H_dev, EPI_HMS, 0, 0.0);
}

mm_status mm_step(mm_ctx* c, float* m_dev, mm_method method, double* dt_inout, double tol, double* t_inout,
                  double* err_out, int* accepted_out)
{
    mm_status s = check_ready(c);
    if (s != MM_OK) return s;
    if (!m_dev || !dt_inout || !(*dt_inout > 0)) return fail(c, MM_EINVAL, "bad m_dev / dt");
    const Tableau tab = make_tableau(method);
    if (tab.S == 0) return fail(c, MM_EINVAL, "unknown method");
    if (tab.embedded && c->mat.T > 0)
        return fail(c, MM_EUNSUPPORTED, "thermal field needs a fixed-step method (reading A6)");
    if (tab.embedded && !(tol > 0)) return fail(c, MM_EINVAL, "tol must be > 0");
    const double dt = *dt_inout;
    float* newstate = nullptr;
    s = enqueue_step(c, m_dev, method, tab, dt, tab.embedded, &newstate);
    if (s != MM_OK) return s;
    unsigned int bits = 0;
    CUDA_TRY(c, cudaMemcpyAsync(&bits, c->maxbits, sizeof(bits), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    float errf;
    std::memcpy(&errf, &bits, sizeof(errf));
    if (!std::isfinite(errf)) {
        c->k0_valid = false;
        return fail(c, MM_ENUMERIC, "non-finite value met by the max-norm reduction");
    }
    int accept = 1;
    double err = 0.0;
    if (tab.embedded) {
        // reading A10: accept iff err <= tol; dt <- dt clamp(0.8 (tol/err)^(1/order), 0.2, 2)
        err = (double)errf;
        accept = err <= tol;
        const double order = (method == MM_RKDP || method == MM_RKCK) ? 5.0 : (method == MM_RK23 ? 3.0 : 2.0);
        const double fac = err == 0.0 ? 2.0 : std::fmin(2.0, std::fmax(0.2, 0.8 * std::pow(tol / err, 1.0 / order)));
        *dt_inout = dt * fac;
    }
    if (accept) {
        s = commit_step(c, m_dev, method, tab, newstate);
        if (s != MM_OK) return s;
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
        if (t_inout) *t_inout += dt;
    }
    // on a rejected FSAL step k_1 = f(m_n) in kb[0] is still valid: keep it
    if (tab.fsal && !accept && !c->k0_valid) {
        c->k0_valid = true;
        c->k0_method = (int)method;
    }
    if (err_out) *err_out = err;
    if (accepted_out) *accepted_out = accept;
    return MM_OK;
}

// running maximum over the steps of one mm_steps_fixed call (bit patterns: NaN / Inf compare largest)
__global__ void k_track_max(const unsigned int* __restrict__ maxbits, unsigned int* __restrict__ run,
                            unsigned long long* __restrict__ step_dev)
{
    atomicMax(run, *maxbits);
    if (step_dev) *step_dev += 1ull;          // the step index of the next thermal draw (reading A6)
}

static mm_status steps_fixed_impl(mm_ctx* c, float* m_dev, mm_method method, const Tableau& tab, double dt, int n,
                                  bool graph_ok, double* t_inout, double* max_err_out)
{
    mm_status s = MM_OK;
    unsigned int* run = c->maxbits + 1;
    CUDA_TRY(c, cudaMemsetAsync(run, 0, sizeof(unsigned int), c->stream));
    auto one_step = [&]() -> mm_status {
        float* newstate = nullptr;
        mm_status st = enqueue_step(c, m_dev, method, tab, dt, false, &newstate);
        if (st == MM_OK) st = commit_step(c, m_dev, method, tab, newstate);
        if (st != MM_OK) return st;
        k_track_max<<<1, 1, 0, c->stream>>>(c->maxbits, run, c->step_on_device ? c->step_dev : nullptr);
        c->kt.launches++;
        return MM_OK;
    };
    int done = 0;
    if (graph_ok) {
        // with a thermal field the step index that selects the draw lives on the device during the replay
        c->step_on_device = c->mat.T > 0;
        if (c->step_on_device) {
            const unsigned long long si = c->step_index;
            cudaMemcpyAsync(c->step_dev, &si, sizeof(si), cudaMemcpyHostToDevice, c->stream);
            cudaStreamSynchronize(c->stream);              // `si` is a stack variable
        }
        // the instantiated graph of one step is kept in the context and reused while everything baked into
        // its kernel arguments is unchanged: method, dt, the state pointer, material / options (epoch)
        const bool hit = c->gexec && c->g_method == (int)method && c->g_dt == dt && c->g_m == m_dev &&
                         c->g_epoch == c->epoch;
        if (!hit) {
            if (c->gexec) { cudaGraphExecDestroy(c->gexec); c->gexec = nullptr; }
            if ((s = one_step()) != MM_OK) { c->step_on_device = false; return s; }   // also sets kernel attributes outside the capture
            done = 1;
            cudaGraph_t graph = nullptr;
            const uint64_t l0 = c->kt.launches;
            if (n > 1 && cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
                const mm_status sc = one_step();
                const cudaError_t ec = cudaStreamEndCapture(c->stream, &graph);
                if (sc == MM_OK && ec == cudaSuccess && graph &&
                    cudaGraphInstantiate(&c->gexec, graph, 0) == cudaSuccess) {
                    c->g_method = (int)method; c->g_dt = dt; c->g_m = m_dev; c->g_epoch = c->epoch;
                    c->g_per = c->kt.launches - l0;
                } else {
                    c->gexec = nullptr;
                }
                c->kt.launches = l0;
                c->step_index--;                           // the captured step has not run
                if (graph) cudaGraphDestroy(graph);
            }
        }
        if (c->gexec) {
            for (; done < n; ++done) {
                if (cudaGraphLaunch(c->gexec, c->stream) != cudaSuccess) break;
                c->kt.launches += c->g_per;
                c->step_index++;
            }
        }
        cudaGetLastError();                                // a refused capture must not surface later
        if (c->step_on_device) {
            // the remaining plain steps (if any) take the index from the host again
            cudaStreamSynchronize(c->stream);
            c->step_on_device = false;
        }
    }
    for (; done < n; ++done)
        if ((s = one_step()) != MM_OK) return s;
    unsigned int bits = 0;
    if (n > 0) {
        CUDA_TRY(c, cudaMemcpyAsync(&bits, run, sizeof(unsigned int), cudaMemcpyDeviceToHost, c->stream));
        CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    }
    float f;
    std::memcpy(&f, &bits, sizeof(f));
    if (!std::isfinite(f)) {
        c->k0_valid = false;
        return fail(c, MM_ENUMERIC, "non-finite value met by the max-norm reduction");
    }
    if (t_inout) *t_inout += dt * n;
    if (max_err_out) *max_err_out = tab.embedded ? (double)f : 0.0;
    return MM_OK;
}

mm_status mm_steps_fixed(mm_ctx* c, float* m_dev, mm_method method, double dt, int n, double* t_inout,
                         double* max_err_out)
{
    mm_status s = check_ready(c);
    if (s != MM_OK) return s;
    if (!m_dev || !(dt > 0) || n < 0) return fail(c, MM_EINVAL, "bad m_dev / dt / n");
    const Tableau tab = make_tableau(method);
    if (tab.S == 0) return fail(c, MM_EINVAL, "unknown method");
    // Every step of a fixed-step, non-FSAL method without thermal field enqueues the same launches with
    // the same arguments: capture the second step into a CUDA graph and replay it (launch-bound grids).
    // The caller's stream may be the legacy default stream, which cannot be captured: the sequence runs
    // on a stream of the context's own, ordered after and before the caller's stream with events.
    const bool chunked = (c->fast & FAST_CHUNK) && c->fp.chunk_w > 0 && c->g.Pz > 1;
    bool graph_ok = c->use_graph && n >= 4 && !tab.fsal && !c->kt.on && !chunked;
    if (graph_ok && !c->gstream) {
        if (cudaStreamCreateWithFlags(&c->gstream, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->gev[0], cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->gev[1], cudaEventDisableTiming) != cudaSuccess) {
            cudaGetLastError();
            graph_ok = false;
        }
    }
    if (!graph_ok) return steps_fixed_impl(c, m_dev, method, tab, dt, n, false, t_inout, max_err_out);
    cudaStream_t user = c->stream;
    CUDA_TRY(c, cudaEventRecord(c->gev[0], user));
    CUDA_TRY(c, cudaStreamWaitEvent(c->gstream, c->gev[0], 0));
    c->stream = c->gstream;
    s = steps_fixed_impl(c, m_dev, method, tab, dt, n, true, t_inout, max_err_out);
    c->stream = user;
    cudaEventRecord(c->gev[1], c->gstream);
    cudaStreamWaitEvent(user, c->gev[1], 0);
    return s;
}

// ---- a11 on the device: accept / reject and the next step length (reading A10), one thread ----
__global__ void k_step_control(StepCtl* __restrict__ ctl, const unsigned int* __restrict__ maxbits)
{
    const float ef = __uint_as_float(*maxbits);
    const double err = (double)ef;
    ctl->ntrial++;
    ctl->last_err = err;
    if (!isfinite(ef)) { ctl->nonfinite = 1; ctl->last_accept = 0; return; }
    const int accept = err <= ctl->tol;
    const double fac = err == 0.0 ? 2.0 : fmin(2.0, fmax(0.2, 0.8 * pow(ctl->tol / err, 1.0 / ctl->order)));
    if (accept) { ctl->t += ctl->dt; ctl->naccept++; }
    ctl->dt *= fac;
    ctl->dtr = (float)(ctl->dt * ctl->g0Ms);
    ctl->last_accept = accept;
}

// commit of a trial step decided on the device: new state -> m, last stage -> first stage (FSAL)
__global__ void k_step_commit(size_t n4, const float4* __restrict__ newstate, float4* __restrict__ m,
                              const float4* __restrict__ klast, float4* __restrict__ kfirst,
                              const StepCtl* __restrict__ ctl)
{
    if (!ctl->last_accept) return;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
        m[i] = newstate[i];
        if (kfirst) kfirst[i] = klast[i];
    }
}

mm_status mm_steps_adaptive(mm_ctx* c, float* m_dev, mm_method method, int ntrials, double* dt_inout, double tol,
                            double* t_inout, int* naccepted_out, double* last_err_out)
{
    mm_status s = check_ready(c);
    if (s != MM_OK) return s;
    if (!m_dev || !dt_inout || !(*dt_inout > 0) || ntrials < 0 || !(tol > 0))
        return fail(c, MM_EINVAL, "bad m_dev / dt / ntrials / tol");
    const Tableau tab = make_tableau(method);
    if (tab.S == 0 || !tab.embedded) return fail(c, MM_EINVAL, "mm_steps_adaptive needs an embedded method");
    if (c->mat.T > 0) return fail(c, MM_EUNSUPPORTED, "thermal field needs a fixed-step method (reading A6)");
    if (ncell(c->g) % 4 != 0) return fail(c, MM_EUNSUPPORTED, "mm_steps_adaptive needs a cell count divisible by 4");
    StepCtl h;
    std::memset(&h, 0, sizeof(h));
    h.t = t_inout ? *t_inout : 0.0;
    h.dt = *dt_inout;
    h.tol = tol;
    h.g0Ms = gamma0_of(c) * c->mat.Ms;
    h.order = (method == MM_RKDP || method == MM_RKCK) ? 5.0 : (method == MM_RK23 ? 3.0 : 2.0);
    h.dtr = (float)(h.dt * h.g0Ms);
    CUDA_TRY(c, cudaMemcpyAsync(c->ctl, &h, sizeof(h), cudaMemcpyHostToDevice, c->stream));
    const size_t n4 = 3 * ncell(c->g) / 4;
    for (int i = 0; i < ntrials; ++i) {
        float* newstate = nullptr;
        s = enqueue_step(c, m_dev, method, tab, 0.0, true, &newstate, true);
        if (s != MM_OK) return s;
        k_step_control<<<1, 1, 0, c->stream>>>(c->ctl, c->maxbits);
        const bool fs = tab.fsal;
        k_step_commit<<<c->fp.nsm * 8, 256, 0, c->stream>>>(n4, (const float4*)newstate, (float4*)m_dev,
                                                       fs ? (const float4*)c->kb[tab.S - 1] : nullptr,
                                                       fs ? (float4*)c->kb[0] : nullptr, c->ctl);
        c->kt.launches += 2;
        if (fs) {
            // accepted: k_1 <- k_S; rejected: k_1 = f(m_n) is still in place -- valid either way
            c->k0_valid = true;
            c->k0_method = (int)method;
        }
    }
    CUDA_TRY(c, cudaMemcpyAsync(&h, c->ctl, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    c->step_index += (uint64_t)h.naccept;
    *dt_inout = h.dt;
    if (t_inout) *t_inout = h.t;
    if (naccepted_out) *naccepted_out = h.naccept;
    if (last_err_out) *last_err_out = h.last_err;
    if (h.nonfinite) {
        c->k0_valid = false;
        return fail(c, MM_ENUMERIC, "non-finite value met by the max-norm reduction");
    }
    return MM_OK;
}

// ---- "fixed maximum variation of m per step": dt = max_dm / max |dm/dtau|, on the device ----
__global__ void k_maxdm_dt(StepCtl* __restrict__ ctl, const unsigned int* __restrict__ maxbits, double max_dm)
{
    const float kmax = __uint_as_float(*maxbits);        // max_i |dm/dtau(i)|, reduced time
    if (!isfinite(kmax) || !(kmax > 0.f)) { ctl->nonfinite = 1; ctl->dtr = 0.f; return; }
    const double dtr = max_dm / (double)kmax;
    ctl->dtr = (float)dtr;
    ctl->dt = dtr / ctl->g0Ms;
    ctl->t += ctl->dt;
    ctl->ntrial++;
}

mm_status mm_steps_maxdm(mm_ctx* c, float* m_dev, mm_method method, double max_dm, int n, double* t_inout,
                         double* last_dt_out)
{
    mm_status s = check_ready(c);
    if (s != MM_OK) return s;
    if (!m_dev || !(max_dm > 0) || n < 0) return fail(c, MM_EINVAL, "bad m_dev / max_dm / n");
    const Tableau tab = make_tableau(method);
    if (tab.S == 0 || tab.embedded) return fail(c, MM_EINVAL, "mm_steps_maxdm needs a fixed-step method");
    if (c->mat.T > 0) return fail(c, MM_EUNSUPPORTED, "thermal field needs a step length known in advance (reading A6)");
    StepCtl h;
    std::memset(&h, 0, sizeof(h));
    h.t = t_inout ? *t_inout : 0.0;
    h.g0Ms = gamma0_of(c) * c->mat.Ms;
    CUDA_TRY(c, cudaMemcpyAsync(c->ctl, &h, sizeof(h), cudaMemcpyHostToDevice, c->stream));
    const size_t ncl = ncell(c->g);
    for (int i = 0; i < n; ++i) {
        // stage 1 on its own: k_1 -> kb[0] and max |k_1|, then dt, then m_2 = m + dt a_21 k_1 (or the Euler update)
        CUDA_TRY(c, cudaMemsetAsync(c->maxbits, 0, sizeof(unsigned int), c->stream));
        EpiParams ep;
        std::memset(&ep, 0, sizeof(ep));
        fill_material(c, ep, c->step_index, 0.0);
        ep.mode = EPI_STAGE;
        ep.m_in = m_dev;
        ep.m_n = m_dev;
        ep.k_out = c->kb[0];
        ep.do_err = 1;
        ep.e_self = 1.0f;
        ep.maxbits = c->maxbits;
        if ((s = launch_eval(c, ep)) != MM_OK) return s;
        k_maxdm_dt<<<1, 1, 0, c->stream>>>(c->ctl, c->maxbits, max_dm);
        c->kt.launches++;
        if (tab.S == 1) {
            k_combine<<<c->fp.nsm * 8, 256, 0, c->stream>>>(ncl, m_dev, c->mtmp, 1, (float)tab.b[0], 0.f, c->kb[0], c->kb[0],
                                                      &c->ctl->dtr);
            k_normalise<<<c->fp.nsm * 8, 256, 0, c->stream>>>(ncl, c->mtmp, m_dev);
            c->kt.launches += 2;
        } else {
            k_combine<<<c->fp.nsm * 8, 256, 0, c->stream>>>(ncl, m_dev, c->ms[0], 1, (float)tab.A[1][0], 0.f, c->kb[0],
                                                      c->kb[0], &c->ctl->dtr);
            c->kt.launches++;
            for (int st = 1; st < tab.S; ++st)
                if ((s = run_stage(c, m_dev, tab, st, 0.0, c->step_index, false, true)) != MM_OK) return s;
        }
        c->step_index++;
    }
    c->k0_valid = false;
    CUDA_TRY(c, cudaMemcpyAsync(&h, c->ctl, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    if (t_inout) *t_inout = h.t;
    if (last_dt_out) *last_dt_out = h.dt;
    if (h.nonfinite) return fail(c, MM_ENUMERIC, "non-finite or zero torque norm in the maximum-variation step");
    return MM_OK;
}

// ---- <f> over all cells, fp64 accumulation ----
__global__ void k_average(size_t n, const float* __restrict__ f, double* __restrict__ out)
{
    double acc[3] = { 0.0, 0.0, 0.0 };
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        for (int cc = 0; cc < 3; ++cc) acc[cc] += (double)f[i + cc * n];
    __shared__ double sh[3][8];
    for (int cc = 0; cc < 3; ++cc) {
        double v = acc[cc];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0) sh[cc][threadIdx.x >> 5] = v;
    }
    __syncthreads();
    if (threadIdx.x < 3) {
        double v = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) v += sh[threadIdx.x][w];
        atomicAdd(out + threadIdx.x, v);
    }
}

mm_status mm_average(mm_ctx* c, const float* field_dev, double avg_host[3])
{
    if (!c || !field_dev || !avg_host) return MM_EINVAL;
    if (!c->has_demag) return fail(c, MM_ESTATE, "mm_demag_init has not been called");
    double* acc = reinterpret_cast<double*>(c->ctl_scratch);
    CUDA_TRY(c, cudaMemsetAsync(acc, 0, 3 * sizeof(double), c->stream));
    const size_t n = ncell(c->g);
    k_average<<<c->fp.nsm * 4, 256, 0, c->stream>>>(n, field_dev, acc);
    c->kt.launches++;
    double h[3];
    CUDA_TRY(c, cudaMemcpyAsync(h, acc, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    for (int i = 0; i < 3; ++i) avg_host[i] = h[i] / (double)n;
    return MM_OK;
}

mm_status mm_steps_fixed_host(mm_ctx* c, float* m_host, mm_method method, double dt, int n, double* t_inout,
                              double* max_err_out)
{
    mm_status s = check_ready(c);
    if (s != MM_OK) return s;
    if (!m_host) return fail(c, MM_EINVAL, "NULL host pointer");
    const size_t fb = 3 * ncell(c->g) * sizeof(float);
    CUDA_TRY(c, cudaMemcpyAsync(c->mhost, m_host, fb, cudaMemcpyHostToDevice, c->stream));
    c->k0_valid = false;
    s = mm_steps_fixed(c, c->mhost, method, dt, n, t_inout, max_err_out);
    if (s != MM_OK) return s;
    CUDA_TRY(c, cudaMemcpyAsync(m_host, c->mhost, fb, cudaMemcpyDeviceToHost, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    return MM_OK;
}

mm_status mm_kernel_timing(mm_ctx* c, int enable)
{
    if (!c) return MM_EINVAL;
    cudaStreamSynchronize(c->stream);
    c->kt.on = enable != 0;
    for (int k = 0; k < KT_N; ++k) c->kt.nev[k] = 0;
    return MM_OK;
}

mm_status mm_kernel_times(mm_ctx* c, double sec_out[7], uint64_t count_out[7])
{
    if (!c || !sec_out || !count_out) return MM_EINVAL;
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));
    for (int k = 0; k < KT_N; ++k) {
        double tot = 0.0;
        for (int i = 0; i + 1 < c->kt.nev[k]; i += 2) {
            float ms = 0.f;
            CUDA_TRY(c, cudaEventElapsedTime(&ms, c->kt.ev[k][i], c->kt.ev[k][i + 1]));
            tot += ms * 1e-3;
        }
        sec_out[k] = tot;
        count_out[k] = (uint64_t)(c->kt.nev[k] / 2);
        c->kt.nev[k] = 0;
    }
    return MM_OK;
}

mm_status mm_fused_eval(mm_ctx* c, float* m_dev, mm_method method, int stage, double dt, uint64_t step)
{
    mm_status s = check_ready(c);
    if (s != MM_OK) return s;
    const Tableau tab = make_tableau(method);
    if (tab.S == 0 || stage < 0 || stage >= tab.S || !m_dev || !(dt > 0))
        return fail(c, MM_EINVAL, "bad method / stage / dt");
    c->k0_valid = false;
    return run_stage(c, m_dev, tab, stage, dt, step, false);
}

mm_status mm_reset_stepper(mm_ctx* c, uint64_t step_index)
{
    if (!c) return MM_EINVAL;
    c->step_index = step_index;
    c->k0_valid = false;
    return MM_OK;
}

mm_status mm_get_demag_kernel(mm_ctx* c, int comp, float* host_out, size_t n)
{
    if (!c || !host_out || comp < 0 || comp > 5) return MM_EINVAL;
    if (!c->has_demag) return fail(c, MM_ESTATE, "mm_demag_init has not been called");
    if (c->dist) return fail(c, MM_EUNSUPPORTED, "a slab context holds only its own K-hat columns");
    const size_t nC = (size_t)c->g.Cx * c->g.Cy * c->g.Cz;
    if (n < nC) return fail(c, MM_EINVAL, "host_out too small");
    const Geom& g = c->g;
    CUDA_TRY(c, cudaMemcpy2D(host_out, g.Cx * sizeof(float), c->khat + (size_t)comp * g.Cz * g.Cy * g.CxK,
                             g.CxK * sizeof(float), g.Cx * sizeof(float), (size_t)g.Cz * g.Cy,
                             cudaMemcpyDeviceToHost));
    return MM_OK;
}

mm_status mm_demag_tensor_host(const double cellsize[3], const int grid[3], const int pbc[3], size_t n,
                               const long* off_host, double* out_host)
{
    if (!cellsize || !grid || !pbc || (n && (!off_host || !out_host))) return MM_EINVAL;
    mmh::tensor_at(cellsize, grid, pbc, n, off_host, out_host);
    return MM_OK;
}

mm_status mm_demag_khat_host(const double cellsize[3], const int grid[3], const int pbc[3], float* out_host,
                             size_t n)
{
    if (!cellsize || !grid || !pbc || !out_host) return MM_EINVAL;
    int Cs[3];
    const mm_status ps = mm_padded_size_of(grid, pbc, nullptr, Cs);
    if (ps != MM_OK) return ps;
    const size_t nC = (size_t)Cs[0] * Cs[1] * Cs[2];
    if (n < 6 * nC) return MM_EINVAL;
    std::string err;
    return (mm_status)mmh::build_khat(cellsize, grid, pbc, out_host, &err);
}

mm_status mm_padded_size(const mm_ctx* c, int P_out[3], int C_out[3])
{
    if (!c) return MM_EINVAL;
    if (P_out) { P_out[0] = c->g.Px; P_out[1] = c->g.Py; P_out[2] = c->g.Pz; }
    if (C_out) { C_out[0] = c->g.Cx; C_out[1] = c->g.Cy; C_out[2] = c->g.Cz; }
    return MM_OK;
}

mm_status mm_create_batch(mm_ctx** out, const int grid[3], const double cellsize[3], const int pbc[3],
                          void* cuda_stream, int nfilms)
{
    if (!out) return MM_EINVAL;
    *out = nullptr;
    if (!grid || nfilms < 1) return fail(nullptr, MM_EINVAL, "mm_create_batch: nfilms must be >= 1");
    if (grid[2] != 1) return fail(nullptr, MM_EUNSUPPORTED, "mm_create_batch: the members are films (Nz = 1)");
    mm_ctx* c = nullptr;
    const mm_status s = mm_create(&c, grid, cellsize, pbc, cuda_stream);
    if (s != MM_OK) return s;
    c->batch = nfilms;
    c->g.Nz = nfilms;            // planes of every field and spectrum; Pz = Cz = 1: no transform along z
    *out = c;
    return MM_OK;
}

mm_status mm_batch_set_field(mm_ctx* c, const double* B_host)
{
    if (!c || !c->batch) return MM_EINVAL;
    mm_status s = check_ready(c);
    if (s != MM_OK) return s;
    c->epoch++;
    if (!B_host) {               // back to the material's uniform field
        if (c->hext_b) { cudaFree(c->hext_b); c->hext_b = nullptr; }
        return MM_OK;
    }
    std::vector<float> h((size_t)3 * c->batch);
    for (size_t i = 0; i < h.size(); ++i) h[i] = (float)(B_host[i] / (MU0 * c->mat.Ms));
    if (!c->hext_b) CUDA_TRY(c, cudaMalloc(&c->hext_b, h.size() * sizeof(float)));
    CUDA_TRY(c, cudaMemcpyAsync(c->hext_b, h.data(), h.size() * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(c, cudaStreamSynchronize(c->stream));       // `h` is a local
    return MM_OK;
}

mm_status mm_padded_size_of(const int grid[3], const int pbc[3], int P_out[3], int C_out[3])
{
    if (!grid || !pbc) return MM_EINVAL;
    for (int a = 0; a < 3; ++a) {
        if (grid[a] < 1 || pbc[a] < 0) return MM_EINVAL;
        const int P = pbc[a] > 0 ? grid[a] : (grid[a] > 1 ? 2 * grid[a] : 1);
        if (!smooth235(P)) return MM_EUNSUPPORTED;
        if (P_out) P_out[a] = P;
        if (C_out) C_out[a] = P / 2 + 1;
    }
    return MM_OK;
}

mm_status mm_set_option(mm_ctx* c, const char* key, int value)
{
    if (!c || !key) return MM_EINVAL;
    const std::string k(key);
    c->epoch++;
    if (k == "graph") { c->use_graph = value != 0; return MM_OK; }
    if (k == "x_pipe") { c->fp.x_pipe = value & 7; return MM_OK; }
    if (k == "mid_pipe") { c->fp.mid_pipe = value; return MM_OK; }
    if (k == "spec_panel") { c->fp.spec_panel = value; return MM_OK; }
    if (k == "y_tma") { c->fp.y_tma = value; return MM_OK; }
    if (k == "last_fused") { c->fp.last_fused = value; return MM_OK; }
    if (k == "q_blocks") { c->fp.q_blocks = value < 1 ? 1 : value; return MM_OK; }
    if (k == "chunk_w" || k == "chunk_streams") {
        // the chunk streams and the slot layout are fixed when the workspaces are made
        if (c->has_demag) return fail(c, MM_ESTATE, "option " + k + " must be set before mm_demag_init");
        if (value < 0) return fail(c, MM_EINVAL, "option " + k + " must be >= 0");
        if (k == "chunk_w") c->fp.chunk_w = value;
        else c->fp.nstream = value;
        return MM_OK;
    }
    return fail(c, MM_EINVAL, "unknown option '" + k + "'");
}

uint64_t mm_launch_count(const mm_ctx* c) { return c ? c->kt.launches : 0; }

mm_status mm_set_fast_path(mm_ctx* c, int enable)
{
    if (!c) return MM_EINVAL;
    if ((c->batch || c->dist) && enable >= 0 && (enable & FAST_ALL) != FAST_ALL)
        return fail(c, MM_EUNSUPPORTED, "batch and slab contexts run the size-specialised kernels only");
    c->fast = enable < 0 ? FAST_ALL : (enable & FAST_ALL);
    c->epoch++;
    return MM_OK;
}

mm_status mm_copy_bandwidth(mm_ctx* c, const void* src_dev, void* dst_dev, size_t nbytes, int reps,
                            double* sec_out)
{
    if (!c || !src_dev || !dst_dev || nbytes < 16 || reps < 1 || !sec_out) return MM_EINVAL;
    cudaEvent_t e0, e1;
    CUDA_TRY(c, cudaEventCreate(&e0));
    CUDA_TRY(c, cudaEventCreate(&e1));
    const size_t n4 = nbytes / 16;
    k_copy4<<<c->fp.nsm * 16, 512, 0, c->stream>>>((const float4*)src_dev, (float4*)dst_dev, n4);
    CUDA_TRY(c, cudaEventRecord(e0, c->stream));
    for (int i = 0; i < reps; ++i)
        k_copy4<<<c->fp.nsm * 16, 512, 0, c->stream>>>((const float4*)src_dev, (float4*)dst_dev, n4);
    CUDA_TRY(c, cudaEventRecord(e1, c->stream));
    CUDA_TRY(c, cudaEventSynchronize(e1));
    float ms = 0.f;
    CUDA_TRY(c, cudaEventElapsedTime(&ms, e0, e1));
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    c->kt.launches += reps + 1;
    *sec_out = (double)ms * 1e-3 / reps;
    return MM_OK;
}

const char* mm_last_error(const mm_ctx* c) { return c ? c->err.c_str() : g_create_error.c_str(); }

void mm_destroy(mm_ctx* c)
{
    if (!c) return;
    free_workspaces(c);
    for (int k = 0; k < KT_N; ++k) {
        for (int i = 0; i < c->kt.cap[k]; ++i) cudaEventDestroy(c->kt.ev[k][i]);
        delete[] c->kt.ev[k];
    }
    if (c->gexec) cudaGraphExecDestroy(c->gexec);
    if (c->gstream) cudaStreamDestroy(c->gstream);
    for (int i = 0; i < 2; ++i)
        if (c->gev[i]) cudaEventDestroy(c->gev[i]);
    delete c;
}

}  // extern "C"

#include "mm_dist.cuh"
