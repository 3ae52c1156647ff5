// demag_host.cpp -- host-side set-up of the transformed demagnetisation kernel K-hat
// (step a0 of DESIGN.md; Eq. (2), "only large data transfers occur at
// initialization", "completely symmetrical ... purely real").
//
// Product code; shares nothing with oracle/ (which evaluates the same tensor in __float128).
//
// The paper prints no closed form for the kernel (reading A1).  The cell-averaged tensor of two equal
// cuboids is evaluated here in two regimes:
//   near field (R < R_NEAR cell diagonals): second differences (weights 1,-2,1 per axis) of the two
//       classical auxiliary functions, written with logarithms and evaluated in 80-bit long double
//       on a lattice table;
//   far field: multipole series  N_ij = -(V/4pi) sum_alpha mu_alpha/alpha! d^(alpha+e_i+e_j) (1/R),
//       alpha running over even multi-indices up to order 6, mu the moments of the triangular
//       distribution that the double cell average produces.  The derivative polynomials are built
//       once by the recursion  d_a [P/R^(2n+1)] = [R^2 d_a P - (2n+1) x_a P] / R^(2n+3).
//       It has no cancellation, so fp64 is enough (the closed form loses ~R^6 eps, PAPER.md:169
//       "avoid subtracting nearly equal numbers").
// Periodic images are summed in real space (reading A8), then every axis is transformed
// with the even / odd symmetry of the component (cosine / sine series through a complex FFT of the
// mirrored line, fp64), and one octant is kept.
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <map>
#include <vector>
#include <array>
#include <algorithm>

#include "demag_host.h"

namespace mmh {

typedef long double ld;
static const ld PI_L = 3.14159265358979323846264338327950288L;
static const double R_NEAR = 40.0;   // switch radius in units of the longest cell edge

// ---------------------------------------------------------------------------------------------
// near field: auxiliary functions (diagonal "F", off-diagonal "G"), non-negative arguments only
// ---------------------------------------------------------------------------------------------
static inline ld lg_ratio(ld a, ld R, ld b2)   // asinh(a / sqrt(b2)) = log((a + R)/sqrt(b2)), R^2 = a^2 + b2
{
    return logl((a + R) / sqrtl(b2));
}

static ld auxF(ld x, ld y, ld z)
{
    x = fabsl(x); y = fabsl(y); z = fabsl(z);
    const ld xx = x * x, yy = y * y, zz = z * z;
    const ld R = sqrtl(xx + yy + zz);
    ld s = (2 * xx - yy - zz) * R / 6;
    if (R == 0) return 0;
    if (y > 0 && xx + zz > 0) s += 0.5L * y * (zz - xx) * lg_ratio(y, R, xx + zz);
    if (z > 0 && xx + yy > 0) s += 0.5L * z * (yy - xx) * lg_ratio(z, R, xx + yy);
    if (x > 0 && y > 0 && z > 0) s -= x * y * z * atanl(y * z / (x * R));
    return s;
}

static ld auxG(ld x, ld y, ld z)
{
    ld sign = 1;
    if (x < 0) { x = -x; sign = -sign; }
    if (y < 0) { y = -y; sign = -sign; }
    z = fabsl(z);
    if (x == 0 || y == 0) return 0;
    const ld xx = x * x, yy = y * y, zz = z * z;
    const ld R = sqrtl(xx + yy + zz);
    ld s = -x * y * R / 3;
    s += (y / 6) * (3 * zz - yy) * lg_ratio(x, R, yy + zz);
    s += (x / 6) * (3 * zz - xx) * lg_ratio(y, R, xx + zz);
    if (z > 0) {
        s += x * y * z * lg_ratio(z, R, xx + yy);
        s -= (z * zz / 6) * atanl(x * y / (z * R));
        s -= (z * yy / 2) * atanl(x * z / (y * R));
        s -= (z * xx / 2) * atanl(y * z / (x * R));
    }
    return sign * s;
}

// component q = xx,yy,zz,xy,xz,yz of the generator at point (x,y,z)
static inline ld generator(int q, ld x, ld y, ld z)
{
    switch (q) {
    case 0: return auxF(x, y, z);
    case 1: return auxF(y, x, z);
    case 2: return auxF(z, y, x);
    case 3: return auxG(x, y, z);
    case 4: return auxG(x, z, y);
    default: return auxG(y, z, x);
    }
}

// parity of component q under reflection of axis a
static const int PAR[6][3] = { {1, 1, 1}, {1, 1, 1}, {1, 1, 1}, {-1, -1, 1}, {-1, 1, -1}, {1, -1, -1} };

// ---------------------------------------------------------------------------------------------
// far field: derivative polynomials of 1/R
// ---------------------------------------------------------------------------------------------
static const int PD = 9;                        // degrees 0..8 per variable
struct Poly {
    double c[PD][PD][PD];
    Poly() { std::memset(c, 0, sizeof(c)); }
};

static Poly poly_deriv_step(const Poly& P, int n /* |beta| */, int a)
{
    // Q = R^2 d_a P - (2n+1) x_a P
    Poly Q;
    for (int i = 0; i < PD; ++i)
        for (int j = 0; j < PD; ++j)
            for (int k = 0; k < PD; ++k) {
                const double c = P.c[i][j][k];
                if (c == 0.0) continue;
                int e[3] = { i, j, k };
                // -(2n+1) x_a P
                {
                    int f[3] = { i, j, k };
                    f[a] += 1;
                    if (f[a] < PD) Q.c[f[0]][f[1]][f[2]] -= (2 * n + 1) * c;
                }
                // R^2 d_a P
                if (e[a] > 0) {
                    const double dc = c * e[a];
                    int f[3] = { i, j, k };
                    f[a] -= 1;
                    for (int b = 0; b < 3; ++b) {
                        int g[3] = { f[0], f[1], f[2] };
                        g[b] += 2;
                        if (g[b] < PD) Q.c[g[0]][g[1]][g[2]] += dc;
                    }
                }
            }
    return Q;
}

struct Term { int i, j, k; double c; };

struct FarField {
    // terms[q][n]: homogeneous polynomial of degree 2+2n, to be divided by R^(5+4n)
    std::vector<Term> terms[6][4];
    double pref;          // -V/(4 pi), scaled units
    double scale;         // 1/L
    void build(const double cell[3])
    {
        const double L = std::max(cell[0], std::max(cell[1], cell[2]));
        scale = 1.0 / L;
        const double d[3] = { cell[0] / L, cell[1] / L, cell[2] / L };
        pref = -(d[0] * d[1] * d[2]) / (4.0 * M_PI);
        std::map<std::array<int, 3>, Poly> memo;
        Poly one;
        one.c[0][0][0] = 1.0;
        memo[{0, 0, 0}] = one;
        // all beta with |beta| <= 8 in graded order
        for (int n = 1; n <= 8; ++n)
            for (int i = 0; i <= n; ++i)
                for (int j = 0; i + j <= n; ++j) {
                    int k = n - i - j;
                    std::array<int, 3> b = { i, j, k };
                    int a = (i > 0) ? 0 : (j > 0 ? 1 : 2);
                    std::array<int, 3> pb = b;
                    pb[a] -= 1;
                    memo[b] = poly_deriv_step(memo[pb], n - 1, a);
                }
        // even moments of the triangular density on [-D, D]: <u^(2k)> = 2 D^(2k) / ((2k+1)(2k+2))
        auto mom = [&](int a, int two_k) {
            return two_k == 0 ? 1.0 : 2.0 * std::pow(d[a], two_k) / ((two_k + 1.0) * (two_k + 2.0));
        };
        auto fact = [](int n) { double f = 1; for (int i = 2; i <= n; ++i) f *= i; return f; };
        const int ei[6] = { 0, 1, 2, 0, 0, 1 }, ej[6] = { 0, 1, 2, 1, 2, 2 };
        for (int q = 0; q < 6; ++q)
            for (int n = 0; n < 4; ++n) {
                Poly S;
                for (int a0 = 0; a0 <= 2 * n; a0 += 2)
                    for (int a1 = 0; a0 + a1 <= 2 * n; a1 += 2) {
                        int a2 = 2 * n - a0 - a1;
                        double w = mom(0, a0) * mom(1, a1) * mom(2, a2) / (fact(a0) * fact(a1) * fact(a2));
                        std::array<int, 3> b = { a0, a1, a2 };
                        b[ei[q]] += 1;
                        b[ej[q]] += 1;
                        const Poly& P = memo[b];
                        for (int i = 0; i < PD; ++i)
                            for (int j = 0; j < PD; ++j)
                                for (int k = 0; k < PD; ++k)
                                    S.c[i][j][k] += w * P.c[i][j][k];
                    }
                terms[q][n].clear();
                for (int i = 0; i < PD; ++i)
                    for (int j = 0; j < PD; ++j)
                        for (int k = 0; k < PD; ++k)
                            if (S.c[i][j][k] != 0.0) terms[q][n].push_back({ i, j, k, S.c[i][j][k] });
            }
    }
    // N(xx..yz) at (X,Y,Z) in metres
    void eval(double X, double Y, double Z, double out[6]) const
    {
        const double x = X * scale, y = Y * scale, z = Z * scale;
        double px[PD], py[PD], pz[PD];
        px[0] = py[0] = pz[0] = 1.0;
        for (int i = 1; i < PD; ++i) { px[i] = px[i - 1] * x; py[i] = py[i - 1] * y; pz[i] = pz[i - 1] * z; }
        const double r2 = x * x + y * y + z * z;
        const double ir2 = 1.0 / r2;
        const double ir = std::sqrt(ir2);
        const double ir4 = ir2 * ir2;
        double inv[4];
        inv[0] = ir4 * ir;            // R^-5
        inv[1] = inv[0] * ir4;        // R^-9
        inv[2] = inv[1] * ir4;        // R^-13
        inv[3] = inv[2] * ir4;        // R^-17
        for (int q = 0; q < 6; ++q) {
            double s = 0.0;
            for (int n = 3; n >= 0; --n) {
                double p = 0.0;
                for (const Term& t : terms[q][n]) p += t.c * px[t.i] * py[t.j] * pz[t.k];
                s += p * inv[n];
            }
            out[q] = pref * s;
        }
    }
};

// ---------------------------------------------------------------------------------------------
// near-field lattice table
// ---------------------------------------------------------------------------------------------
struct NearTable {
    int B[3];                  // offsets 0..B[a] available
    std::vector<double> N[6];  // [ (B2+1) (B1+1) (B0+1) ]
    double cell[3];
    bool has(long i, long j, long k) const
    {
        return std::labs(i) <= B[0] && std::labs(j) <= B[1] && std::labs(k) <= B[2];
    }
    void get(long i, long j, long k, double out[6]) const
    {
        const long ai = std::labs(i), aj = std::labs(j), ak = std::labs(k);
        const size_t idx = ((size_t)ak * (B[1] + 1) + aj) * (B[0] + 1) + ai;
        const int neg[3] = { i < 0, j < 0, k < 0 };
        for (int q = 0; q < 6; ++q) {
            double s = 1.0;
            for (int a = 0; a < 3; ++a)
                if (neg[a] && PAR[q][a] < 0) s = -s;
            out[q] = s * N[q][idx];
        }
    }
    void build(const double c[3], const int maxoff[3])
    {
        const double L = std::max(c[0], std::max(c[1], c[2]));
        for (int a = 0; a < 3; ++a) {
            cell[a] = c[a];
            long b = (long)std::ceil(R_NEAR * L / c[a]);
            B[a] = (int)std::min<long>(b, maxoff[a]);
        }
        const long l0 = B[0] + 3, l1 = B[1] + 3, l2 = B[2] + 3;   // lattice -1 .. B+1
        const size_t npts = (size_t)l0 * l1 * l2;
        std::vector<ld> tab(npts);
        const ld vol4pi = 4 * PI_L * (ld)c[0] * (ld)c[1] * (ld)c[2];
        // scale lengths by L so that intermediate magnitudes stay O(R^3)
        const ld d0 = c[0], d1 = c[1], d2 = c[2];
        for (int q = 0; q < 6; ++q) {
            N[q].assign((size_t)(B[0] + 1) * (B[1] + 1) * (B[2] + 1), 0.0);
#pragma omp parallel for schedule(dynamic, 1)
            for (long k = 0; k < l2; ++k)
                for (long j = 0; j < l1; ++j)
                    for (long i = 0; i < l0; ++i)
                        tab[((size_t)k * l1 + j) * l0 + i] = generator(q, (i - 1) * d0, (j - 1) * d1, (k - 1) * d2);
            static const ld w3[3] = { 1, -2, 1 };
#pragma omp parallel for schedule(static)
            for (long k = 0; k <= B[2]; ++k)
                for (long j = 0; j <= B[1]; ++j)
                    for (long i = 0; i <= B[0]; ++i) {
                        ld s = 0;
                        for (int c2 = 0; c2 < 3; ++c2)
                            for (int c1 = 0; c1 < 3; ++c1) {
                                const ld* row = &tab[((size_t)(k + c2) * l1 + (j + c1)) * l0 + i];
                                s += w3[c2] * w3[c1] * (row[0] - 2 * row[1] + row[2]);
                            }
                        N[q][((size_t)k * (B[1] + 1) + j) * (B[0] + 1) + i] = (double)(-s / vol4pi);
                    }
        }
    }
};

// ---------------------------------------------------------------------------------------------
// tensor with images
// ---------------------------------------------------------------------------------------------
struct TensorEval {
    FarField far;
    NearTable near;
    double cell[3];
    int grid[3], nimg[3];
    double rnear2;
    void init(const double c[3], const int g[3], const int pbc[3])
    {
        int maxoff[3];
        for (int a = 0; a < 3; ++a) {
            cell[a] = c[a];
            grid[a] = g[a];
            nimg[a] = pbc[a] > 0 ? pbc[a] : 0;
            maxoff[a] = pbc[a] > 0 ? (pbc[a] + 1) * g[a] : g[a] - 1;
        }
        far.build(c);
        near.build(c, maxoff);
        const double L = std::max(c[0], std::max(c[1], c[2]));
        rnear2 = (R_NEAR * L) * (R_NEAR * L);
    }
    inline void single(long i, long j, long k, double out[6]) const
    {
        const double X = i * cell[0], Y = j * cell[1], Z = k * cell[2];
        if (X * X + Y * Y + Z * Z < rnear2 && near.has(i, j, k)) near.get(i, j, k, out);
        else far.eval(X, Y, Z, out);
    }
    // sum over images of the offset (i,j,k)
    void at(long i, long j, long k, double out[6]) const
    {
        double acc[6] = { 0, 0, 0, 0, 0, 0 };
        // far images first (small terms), accumulation order fixed
        for (long a = -nimg[0]; a <= nimg[0]; ++a)
            for (long b = -nimg[1]; b <= nimg[1]; ++b)
                for (long c = -nimg[2]; c <= nimg[2]; ++c) {
                    if (a == 0 && b == 0 && c == 0) continue;
                    double t[6];
                    single(i + a * grid[0], j + b * grid[1], k + c * grid[2], t);
                    for (int q = 0; q < 6; ++q) acc[q] += t[q];
                }
        double t[6];
        single(i, j, k, t);
        for (int q = 0; q < 6; ++q) out[q] = acc[q] + t[q];
    }
};

void tensor_at(const double cell[3], const int grid[3], const int pbc[3], size_t n, const long* off,
               double* out)
{
    TensorEval te;
    te.init(cell, grid, pbc);
#pragma omp parallel for schedule(dynamic, 64)
    for (long p = 0; p < (long)n; ++p) te.at(off[3 * p], off[3 * p + 1], off[3 * p + 2], out + 6 * p);
}

// ---------------------------------------------------------------------------------------------
// host FFT (fp64, Stockham, any mix of radices 2, 3, 5, 7)
// ---------------------------------------------------------------------------------------------
typedef std::complex<double> cd;

struct HostFFT {
    int n;
    std::vector<int> radices;
    std::vector<cd> tw;      // exp(-2 pi i q / n)
    explicit HostFFT(int n_) : n(n_)
    {
        int m = n;
        for (int p : { 7, 5, 3, 2 })
            while (m % p == 0) { radices.push_back(p); m /= p; }
        tw.resize(n);
        for (int q = 0; q < n; ++q) {
            const long double a = -2.0L * PI_L * q / n;
            tw[q] = cd((double)cosl(a), (double)sinl(a));
        }
    }
    bool ok() const
    {
        int m = 1;
        for (int r : radices) m *= r;
        return m == n;
    }
    // forward transform of x (length n), scratch y; result returned in x
    void forward(std::vector<cd>& x, std::vector<cd>& y) const
    {
        int ns = 1;
        cd* in = x.data();
        cd* outp = y.data();
        for (int R : radices) {
            const int m = n / R;
            for (int j = 0; j < m; ++j) {
                const int k = j % ns;
                cd v[7];
                for (int r = 0; r < R; ++r) v[r] = in[j + r * m] * tw[(size_t)r * k * (n / (ns * R)) % n];
                const int j0 = (j / ns) * ns * R + k;
                for (int s = 0; s < R; ++s) {
                    cd acc = 0;
                    for (int r = 0; r < R; ++r) acc += v[r] * tw[(size_t)(r * s % R) * (n / R)];
                    outp[j0 + s * ns] = acc;
                }
            }
            ns *= R;
            std::swap(in, outp);
        }
        if (in != x.data()) std::copy(in, in + n, x.data());
    }
};

static bool smooth235(int n)
{
    for (int p : { 2, 3, 5, 7 })
        while (n % p == 0) n /= p;
    return n == 1;
}

// extents of the stored real-space octant along one axis and its mirror rule
static inline int octant_extent(int N, int periodic) { return periodic ? N / 2 + 1 : N; }

// transform one axis: in [outer][E][inner] -> out [outer][C][inner], C = P/2+1
static void axis_transform(const std::vector<double>& in, std::vector<double>& out, size_t outer, int E,
                           size_t inner, int N, int P, int periodic, int parity)
{
    const int C = P / 2 + 1;
    out.assign(outer * (size_t)C * inner, 0.0);
    if (P == 1) {   // single cell: identity
        for (size_t o = 0; o < outer; ++o)
            for (size_t i = 0; i < inner; ++i) out[o * inner + i] = (parity > 0) ? in[o * E * inner + i] : 0.0;
        return;
    }
    HostFFT fft(P);
#pragma omp parallel
    {
        std::vector<cd> x(P), y(P);
#pragma omp for schedule(static) collapse(2)
        for (long o = 0; o < (long)outer; ++o)
            for (long i = 0; i < (long)inner; ++i) {
                for (int s = 0; s < P; ++s) x[s] = 0.0;
                for (int d = 0; d < E; ++d) {
                    const double v = in[((size_t)o * E + d) * inner + i];
                    if (d == 0) { x[0] = (parity > 0) ? v : 0.0; continue; }
                    const int mirror = P - d;
                    if (mirror == d) {        // periodic even N, d = N/2: its own mirror image
                        x[d] = (parity > 0) ? v : 0.0;
                    } else {
                        x[d] = v;
                        x[mirror] = parity * v;
                    }
                }
                (void)N; (void)periodic;
                fft.forward(x, y);
                for (int k = 0; k < C; ++k)
                    out[((size_t)o * C + k) * inner + i] = (parity > 0) ? x[k].real() : x[k].imag();
            }
    }
}

int build_khat(const double cell[3], const int grid[3], const int pbc[3], float* khat_out, std::string* err)
{
    int P[3], E[3], C[3], per[3];
    for (int a = 0; a < 3; ++a) {
        per[a] = pbc[a] > 0;
        P[a] = per[a] ? grid[a] : (grid[a] > 1 ? 2 * grid[a] : 1);
        if (!smooth235(P[a])) {
            if (err) *err = "padded size has a prime factor other than 2, 3, 5, 7";
            return 5;
        }
        E[a] = octant_extent(grid[a], per[a]);
        C[a] = P[a] / 2 + 1;
    }
    TensorEval te;
    te.init(cell, grid, pbc);
    const size_t nE = (size_t)E[0] * E[1] * E[2];
    const size_t nC = (size_t)C[0] * C[1] * C[2];
    std::vector<double> oct[6];
    try {
        for (int q = 0; q < 6; ++q) oct[q].assign(nE, 0.0);
    } catch (const std::bad_alloc&) {
        if (err) *err = "host allocation of the tensor octant failed";
        return 2;
    }
#pragma omp parallel for schedule(dynamic, 1) collapse(2)
    for (long k = 0; k < E[2]; ++k)
        for (long j = 0; j < E[1]; ++j)
            for (long i = 0; i < E[0]; ++i) {
                double t[6];
                te.at(i, j, k, t);
                // reading A8: on an even periodic axis the offset N/2 is its own mirror image; the
                // components odd along that axis vanish there (symmetrisation of the image sum)
                const long ijk[3] = { i, j, k };
                for (int q = 0; q < 6; ++q) {
                    double v = t[q];
                    for (int a = 0; a < 3; ++a)
                        if (per[a] && grid[a] % 2 == 0 && ijk[a] == grid[a] / 2 && PAR[q][a] < 0) v = 0.0;
                    oct[q][((size_t)k * E[1] + j) * E[0] + i] = v;
                }
            }
    const double norm = -1.0 / ((double)P[0] * P[1] * P[2]);
    std::vector<double> t1, t2, t3;
    for (int q = 0; q < 6; ++q) {
        // x: [E2*E1][E0][1] -> [E2*E1][C0][1]
        axis_transform(oct[q], t1, (size_t)E[2] * E[1], E[0], 1, grid[0], P[0], per[0], PAR[q][0]);
        std::vector<double>().swap(oct[q]);
        // y: [E2][E1][C0] -> [E2][C1][C0]
        axis_transform(t1, t2, (size_t)E[2], E[1], (size_t)C[0], grid[1], P[1], per[1], PAR[q][1]);
        // z: [1][E2][C1*C0] -> [1][C2][C1*C0]
        axis_transform(t2, t3, 1, E[2], (size_t)C[1] * C[0], grid[2], P[2], per[2], PAR[q][2]);
        // an odd axis contributes a factor i (its transform is i * Im); off-diagonal components have
        // exactly two odd axes -> factor i*i = -1
        const double sgn = (q >= 3) ? -1.0 : 1.0;
        float* dst = khat_out + (size_t)q * nC;
        for (size_t p = 0; p < nC; ++p) dst[p] = (float)(sgn * norm * t3[p]);
    }
    return 0;
}

}  // namespace mmh
