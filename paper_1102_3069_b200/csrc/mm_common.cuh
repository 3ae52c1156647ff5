// mm_common.cuh -- shared device-side types of the hot path.
//
// Product code.  Nothing here is shared with oracle/.
//
// Layouts (x fastest everywhere):
//   field      float  [3][Nz][Ny][Nx]                      m, H, k_s, caller or context owned
//   specA      float2 [3][Nz][Ny][CxS]                     after the x pass   (CxS >= Cx = Px/2+1)
//   specB      float2 [3][Nz][Py][CxS]                     after the y pass   (3D only)
//   khat       float  [6][Cz][Cy][CxK] (xx,yy,zz,xy,xz,yz) one octant, includes -1/(Px Py Pz)
// Units on the device (section 3.3): fields in units of Ms, time in 1/(gamma0 Ms).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mm {

struct Geom {
    int Nx, Ny, Nz;      // cells
    int Px, Py, Pz;      // padded transform sizes (reading A9)
    int Cx, Cy, Cz;      // P/2 + 1
    int CxS;             // row stride of the spectra, in complex elements
    int CxK;             // row stride of K-hat, in floats (Cx rounded up to 4: 16-byte rows; to 32 from Cx = 128 on)
    int perx, pery, perz;
};

enum EpiMode { EPI_HMS = 0, EPI_HEFF = 1, EPI_TORQUE = 2, EPI_STAGE = 3 };

#define MM_MAXK 8

// Everything the fused epilogue needs (steps a6-a10), passed by value.
struct EpiParams {
    const float* m_in;   // state this evaluation acts on
    float* out;          // EPI_HMS / EPI_HEFF / EPI_TORQUE: output field
    int mode;
    int demag;           // 0: H_ms taken as zero
    float out_scale;     // Ms (A/m) for fields, gamma0 Ms (1/s) for the torque
    // local field terms, reduced units
    float wex[3];        // 2A/(mu0 Ms^2 d_a^2); 0 for a one-cell axis           Eq. (3)
    float kan, u[3];     // 2Ku/(mu0 Ms^2), axis                                  Eq. (4)
    float hext[3];       // B/(mu0 Ms)
    const float* hext_b; // batch of films (mm_create_batch): per-plane applied field [Nz][3], overrides hext; or NULL
    unsigned plane_cells; // Ny * Nx (plane index of a cell = idx / plane_cells), used with hext_b
    int geometry;        // cells with m = 0 are empty (reading A15)
    int cubic;           // Eq. (5)
    float k1c, k2c;      // 2 K1/(mu0 Ms^2), 2 K2/(mu0 Ms^2)
    float c1[3], c2[3], c3[3];   // orthonormal cubic axes (reading A14)
    int thermal;         // Eq. (6)
    float sig_th;        // sqrt(2 alpha kB T/(gamma0 mu0 Ms V dt)) / Ms
    uint32_t key0, key1, step0, step1;
    const unsigned long long* step_dev;   // if set, the step index of the thermal draw is read here (graph replay)
    // torque
    float alpha, inv1pa2;   // Eq. (1)
    int stt;                // Eq. (7)-(8)
    float cj[3];            // b_j j_a / (2 d_a gamma0 Ms)
    float c_ad, c_nad;      // (1 + alpha xi | 1)/(1+alpha^2), (xi - alpha)/(1+alpha^2)
    // Runge-Kutta stage combine (EPI_STAGE)
    const float* m_n;    // state at the start of the step
    float* m_out;        // next stage input / new state (may be NULL)
    float* k_out;        // where k_s is stored (may be NULL)
    int normalise;
    float a_self;        // dt * a_{s+1,s}
    int na;
    float a[MM_MAXK];
    const float* ka[MM_MAXK];
    int do_err;          // error / max-norm reduction
    float e_self;
    int ne;
    float e[MM_MAXK];
    const float* ke[MM_MAXK];
    unsigned int* maxbits;   // atomicMax target (bit pattern of a non-negative float)
    // slab decomposition (mm_dist_*): planes z = -1 and z = Nz of m_in held by the neighbouring ranks, [3][Ny][Nx]
    // each; NULL: the slab ends at an open boundary of the global grid (or the grid is not split)
    const float* zlo;
    const float* zhi;
    unsigned long long cell0;   // global index of the slab's first cell (thermal counter, reading A6)
    const float* dt_scale;   // device scalar dt gamma0 Ms multiplying a_self, a[], e_self, e[] (NULL: already folded in)
};

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b)
{
    return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ float2 cconj(float2 a) { return make_float2(a.x, -a.y); }
__device__ __forceinline__ float2 cscale(float2 a, float s) { return make_float2(a.x * s, a.y * s); }
// multiply by SGN * i  (SGN = -1: forward transform convention exp(-i ...))
template <int SGN>
__device__ __forceinline__ float2 cmuli(float2 a)
{
    return SGN < 0 ? make_float2(a.y, -a.x) : make_float2(-a.y, a.x);
}

// ---- optional per-pass timing with CUDA events on the launching stream (bench.py "roofline") ----
enum KernelCat { KT_FWD_X = 0, KT_FWD_Y = 1, KT_MID = 2, KT_INV_Y = 3, KT_INV_X = 4, KT_OTHER = 5, KT_EPI = 6, KT_N = 7 };

struct KTimer {
    bool on;
    cudaStream_t stream;
    uint64_t launches;
    cudaEvent_t* ev[KT_N];      // start/stop pairs
    int nev[KT_N], cap[KT_N];
    void begin(int cat) { if (on) rec(cat); }
    void end(int cat) { launches++; if (on) rec(cat); }
    void rec(int cat)
    {
        if (nev[cat] == cap[cat]) {
            const int ncap = cap[cat] ? 2 * cap[cat] : 256;
            cudaEvent_t* e = new cudaEvent_t[ncap];
            for (int i = 0; i < nev[cat]; ++i) e[i] = ev[cat][i];
            for (int i = nev[cat]; i < ncap; ++i) cudaEventCreate(&e[i]);
            delete[] ev[cat];
            ev[cat] = e;
            cap[cat] = ncap;
        }
        cudaEventRecord(ev[cat][nev[cat]++], stream);
    }
};

// device-side state of the step controller (reading A10; step a11): lives in the context
struct StepCtl {
    double t, dt, tol;       // seconds
    double g0Ms;             // gamma0 Ms: reduced time step = dt * g0Ms
    double order;            // exponent 1/order in the step-size rule
    double last_err;
    float dtr;               // (float)(dt * g0Ms), what the kernels multiply the tableau by
    int last_accept;
    int naccept, ntrial;
    int nonfinite;
};

}  // namespace mm
