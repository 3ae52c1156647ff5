/*
 * mm.h -- C ABI of the B200-native micromagnetic hot path (after MuMax, arXiv 1102.3069).
 *
 * One effective-field evaluation plus Landau-Lifshitz torque per Runge-Kutta stage on a
 * regular finite-difference grid.  Citations are lines of /root/reference/PAPER.md ("PAPER.md:n")
 * and readings A1..A13 of DESIGN.md where the paper is silent.
 *
 * Conventions that hold for every call
 * ------------------------------------
 *  - No C++ types, no exceptions and no torch types cross this boundary.  Every call returns an
 *    mm_status; mm_last_error(ctx) gives a human-readable message for the last failure.
 *  - Fields are structure-of-arrays float32 [3][Nz][Ny][Nx], x fastest, contiguous, 16-byte aligned,
 *    component order (x, y, z).  "m" holds unit vectors, M = Ms * m.
 *  - Pointers named *_dev are DEVICE pointers owned by the caller (e.g. a torch CUDA tensor's
 *    data_ptr()); pointers named *_host are HOST pointers.  The library never frees, reallocates or
 *    keeps caller memory beyond the call (asynchronous calls keep it until the stream reaches them).
 *  - The context owns the transformed kernel K-hat, FFT workspaces, twiddle tables, Runge-Kutta
 *    buffers and device scalars.  Nothing is allocated on the device after mm_demag_init, with one
 *    exception: the first mm_set_material that asks for exchange_in_kernel allocates a second copy of
 *    K-hat (kept until mm_destroy).
 *  - All device work is enqueued on the CUDA stream given to mm_create.  mm_heff / mm_torque /
 *    mm_demag_field / mm_fused_eval are asynchronous with respect to the host; mm_step synchronises the stream once, at its
 *    end, to return dt / err / accepted.
 *  - A context belongs to the CUDA device that is current when mm_create is called; that device must be
 *    current for every later call on the context (one process per GPU is the intended use).
 *  - A context has no hidden global state: the library reads no environment variable; tuning switches are
 *    per-context options (mm_set_option).
 *  - There is no CPU fallback, no cuFFT and no tensor-core path inside the library: every hot-path
 *    step runs in hand-written sm_100a kernels.  Without a CUDA device mm_create fails with MM_ECUDA.
 */
#ifndef MM_H_
#define MM_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mm_ctx mm_ctx; /* opaque */

typedef enum {
    MM_OK = 0,
    MM_EINVAL = 1,       /* bad argument (NULL, non-positive size, ...)                          */
    MM_ENOMEM = 2,       /* host or device allocation failed                                      */
    MM_ECUDA = 3,        /* CUDA runtime error (message in mm_last_error)                         */
    MM_ESTATE = 4,       /* call order: material / demag kernel not set                           */
    MM_EUNSUPPORTED = 5, /* padded size not 2^a 3^b 5^c 7^d, thermal field with adaptive stepping */
    MM_ENUMERIC = 6      /* non-finite value met by the max-norm reduction                        */
} mm_status;

/* Runge-Kutta family of PAPER.md:123-139 (section 2.2).  RK4 and RKDP are the two the hot path is
 * graded on; the others share the same stage kernel with another tableau. */
typedef enum {
    MM_RK1 = 0,  /* Euler -- the step the paper times              */
    MM_RK2 = 1,  /* Heun                                                           */
    MM_RK4 = 2,  /* classical 4th order                                            */
    MM_RKDP = 3, /* Dormand-Prince 5(4), adaptive; controller: reading A10         */
    MM_RK12 = 4, /* Heun-Euler 2(1), adaptive                                      */
    MM_RK23 = 5, /* Bogacki-Shampine 3(2), adaptive                                */
    MM_RK3 = 6,  /* Kutta's third-order method                                     */
    MM_RKCK = 7  /* Cash-Karp 5(4), adaptive                                       */
} mm_method;

/* Material and drive, SI units in; converted once to the internal reduced units mu0 = gamma0 = Ms = 1
 * of PAPER.md:169 (section 3.3).  Plain data, copied by mm_set_material. */
typedef struct {
    double Ms;        /* saturation magnetisation, A/m, > 0                                       */
    double Aex;       /* exchange stiffness, J/m, >= 0            Eq. (3)            */
    double alpha;     /* damping, >= 0                            Eq. (1)            */
    double gamma0;    /* m/(A s); 0 selects 2.211e5               reading A2                      */
    double Ku;        /* uniaxial anisotropy constant, J/m^3      Eq. (4)            */
    double anis_u[3]; /* anisotropy axis, normalised by the library (ignored if Ku == 0)          */
    double Bext[3];   /* applied field, tesla; H = B / mu0                     */
    double T;         /* temperature, kelvin                      Eq. (6)           */
    uint64_t seed;    /* Philox4x32-10 key                        reading A6                      */
    double j[3];      /* current density, A/m^2                   Eq. (7)           */
    double P;         /* spin polarisation                        Eq. (8)           */
    double xi;        /* degree of non-adiabaticity               Eq. (7)                         */
    int stt_literal_eq7; /* 0: (1 + alpha xi) on the adiabatic term; 1: Eq. (7) as printed (A7)   */
    int demag;        /* 1: magnetostatic field on (default use); 0: off (tests of local terms)   */
    double K1, K2;    /* cubic anisotropy constants, J/m^3         Eq. (5)            */
    int exchange_in_kernel; /* 1: the paper's variant (reading A3'): the exchange stencil is added
                       * to the convolution kernel, so a missing neighbour at an open face counts as m = 0;
                       * 0 (default): stencil in the epilogue, free boundary (reading A3).  Needs demag = 1. */
    int geometry;     /* 1: cells whose m is the zero vector are empty (staircase shapes; reading
                       * A15): no exchange / current coupling to them, they stay empty.  0 (default).      */
    double anis_c1[3], anis_c2[3]; /* first two cubic axes; c2 is made orthogonal to c1, c3 = c1 x c2
                       * (reading A14); ignored if K1 == K2 == 0                                 */
} mm_material;

/* mm_create -- set up a context for a grid of equal cuboid cells.
 *   out          receives the context (host pointer).
 *   grid[3]      cells along x, y, z (each >= 1).
 *   cellsize[3]  cell edge lengths in metres (each > 0).
 *   pbc[3]       0 = open boundary, zero padded to 2 N_a (reading A9);
 *                p > 0 = periodic with images -p..p summed into the kernel and no padding
 *                (reading A8).
 *   cuda_stream  a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream) or NULL for the
 *                default stream.  Every kernel of this context is launched on it.
 * Errors: MM_EINVAL; MM_EUNSUPPORTED if a padded size has a prime factor other than 2, 3, 5, 7
 * (PAPER.md:169-171 restricts sizes to smooth numbers); MM_ECUDA if no device; MM_ENOMEM. */
mm_status mm_create(mm_ctx** out, const int grid[3], const double cellsize[3], const int pbc[3],
                    void* cuda_stream);

/* mm_set_material -- copy material / drive parameters; may be called again between steps.
 * Errors: MM_EINVAL (Ms <= 0, negative Aex / alpha, zero axis with Ku != 0). */
mm_status mm_set_material(mm_ctx* ctx, const mm_material* mat);

/* mm_demag_init -- build the transformed demagnetisation kernel:
 * cell-averaged tensor on the padded offset lattice evaluated on the HOST in extended precision
 * (long double near field, multipole series far field; reading A1), periodic images summed, each
 * axis transformed in fp64, real part kept (the kernel is symmetric), the sign and the
 * 1/(Px Py Pz) normalisation folded in, one octant stored as float32 and copied to the device once
 * (PAPER.md:151).  Also allocates every device workspace.  Blocking.  Independent of the material.
 * Errors: MM_ENOMEM, MM_ECUDA. */
mm_status mm_demag_init(mm_ctx* ctx);

/* mm_heff -- one effective-field evaluation:
 * H_eff = H_ms + H_exch + H_anis + H_ext + H_therm, in A/m, written to H_dev.
 *   m_dev   in,  device, float32 [3][Nz][Ny][Nx]
 *   H_dev   out, device, same layout
 *   step, dt_for_thermal   index of the time step and its length in seconds: the thermal field is one
 *           draw per cell per step with amplitude ~ 1/sqrt(dt) (Eq. (6); reading A6).  Ignored if T = 0.
 * Asynchronous.  Errors: MM_ESTATE before mm_set_material / mm_demag_init; MM_EINVAL. */
mm_status mm_heff(mm_ctx* ctx, const float* m_dev, float* H_dev, double t, uint64_t step,
                  double dt_for_thermal);

/* mm_torque -- dm/dt in 1/s: Eq. (1) for m = M/Ms plus the Zhang-Li terms of
 * Eq. (7)-(8) when j != 0.  Same arguments as mm_heff.  Asynchronous. */
mm_status mm_torque(mm_ctx* ctx, const float* m_dev, float* dmdt_dev, double t, uint64_t step,
                    double dt_for_thermal);

/* mm_step -- one trial step of a Runge-Kutta method, m updated in place.
 *   m_dev       in/out, device.  On an accepted step m <- normalise(m + dt sum b_s k_s); on a
 *               rejected step (adaptive methods only) m is left unchanged.
 *   dt_inout    host: in = step to try (s); out = step proposed for the next call (adaptive methods;
 *               unchanged for fixed-step methods).
 *   tol         maximum tolerable error per step (reading A10); ignored by RK1/RK2/RK4.
 *   t_inout     host: time, advanced by dt when the step is accepted.
 *   err_out     host, may be NULL: error estimate of the embedded pair (0 for fixed-step methods).
 *   accepted_out host, may be NULL: 1 / 0.
 * The thermal field is redrawn once per accepted step and requires a fixed-step method (A6):
 * MM_EUNSUPPORTED otherwise.  Synchronises the stream once at the end.
 * Errors: MM_ESTATE, MM_EINVAL, MM_EUNSUPPORTED, MM_ENUMERIC (NaN/Inf met), MM_ECUDA. */
mm_status mm_step(mm_ctx* ctx, float* m_dev, mm_method method, double* dt_inout, double tol,
                  double* t_inout, double* err_out, int* accepted_out);

/* mm_steps_fixed -- n consecutive steps of fixed length dt with no host synchronisation in between
 * (the whole sequence is enqueued; stage launches are replayed from a CUDA graph when possible).
 * With an adaptive method the embedded error is still reduced on the device but every step is
 * accepted: this is the "replay" mode reading A10 uses for parity of adaptive runs.
 *   max_err_out  host, may be NULL: largest per-step error estimate seen.
 * Synchronises once at the end. */
mm_status mm_steps_fixed(mm_ctx* ctx, float* m_dev, mm_method method, double dt, int n,
                         double* t_inout, double* max_err_out);

/* mm_steps_adaptive -- ntrials trial steps of an embedded method (MM_RKDP, MM_RK23, MM_RK12) with the
 * step controller of reading A10 running ON THE DEVICE (step a11 of DESIGN.md):
 * the error norm, the accept / reject decision, the new step length, the time and the commit of an
 * accepted state never leave the GPU, so the whole sequence is enqueued without a host synchronisation
 * per step (mm_step synchronises once per step).  Synchronises once at the end to return the scalars.
 *   dt_inout       host: first trial step length in, next proposed step length out (seconds)
 *   t_inout        host, may be NULL: time in, time after the accepted steps out
 *   naccepted_out  host, may be NULL: how many of the ntrials steps were accepted
 *   last_err_out   host, may be NULL: error estimate of the last trial step
 * The cell count must be divisible by 4.  Thermal field: MM_EUNSUPPORTED (reading A6). */
mm_status mm_steps_adaptive(mm_ctx* ctx, float* m_dev, mm_method method, int ntrials, double* dt_inout,
                            double tol, double* t_inout, int* naccepted_out, double* last_err_out);

/* mm_steps_maxdm -- n steps of a fixed-step method (MM_RK1, MM_RK2, MM_RK3, MM_RK4) with "a fixed
 * maximum variation of m per step": every step takes dt = max_dm / max_i |dm/dt(i)|
 * evaluated on the state at the start of the step.  The norm, dt and t stay on the device (no host
 * synchronisation per step); synchronises once at the end.
 *   max_dm        largest change of a unit vector per step (dimensionless, > 0)
 *   t_inout       host, may be NULL: time in, time after the n steps out
 *   last_dt_out   host, may be NULL: length of the last step (seconds) */
mm_status mm_steps_maxdm(mm_ctx* ctx, float* m_dev, mm_method method, double max_dm, int n,
                         double* t_inout, double* last_dt_out);

/* mm_average -- <f> over all cells of a field f [3][Nz][Ny][Nx] (e.g. the average magnetisation the
 * paper's output tables list): fp64 accumulation on the device, avg_host[3] out.
 * Synchronises the stream. */
mm_status mm_average(mm_ctx* ctx, const float* field_dev, double avg_host[3]);

/* mm_average_static -- the same reduction (<f> over all cells of f [3][ncell]; fp64 accumulation) for
 * callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops): it needs no
 * context and calls no cudaMalloc / cudaFree / allocating library routine.  Its scratch -- per-block partial sums
 * and an arrival counter, 192 KB -- is a fixed file-scope device array that every GPU loading the library holds
 * until the process exits.
 *   field_dev   device, float [3][ncell], read only
 *   ncell       cells per component, 1 .. MM_AVERAGE_STATIC_MAX_CELLS (larger: MM_EUNSUPPORTED, nothing launched)
 *   avg_dev     DEVICE, double [3], written by the kernel (no host synchronisation; read it after the stream)
 *   stream      cudaStream_t as void* (NULL: the default stream); runs on the device current at the call
 *   err,err_len host, may be NULL / 0: receives a message for a non-OK status
 * All calls share the one scratch array: calls that overlap on the GPU (different streams without an ordering
 * between them, or two host threads) race on it -- order them.  The counter is cleared at the start of every call
 * and every partial sum a call reads is written by that call, so nothing depends on an earlier call.  The first
 * call on a device looks the array's address up (cudaGetSymbolAddress; make that call outside graph capture).
 * The result is the sum in block order: reproducible bit for bit, and equal to mm_average's to fp64 rounding.
 * Errors: MM_EINVAL (NULL pointer, ncell = 0), MM_EUNSUPPORTED (ncell beyond the maximum), MM_ECUDA. */
#define MM_AVERAGE_STATIC_MAX_CELLS ((size_t)67108864)
mm_status mm_average_static(const float* field_dev, size_t ncell, double* avg_dev, void* stream, char* err,
                            size_t err_len);

/* mm_steps_fixed_host -- the same as mm_steps_fixed for a state held in HOST memory (pinned memory
 * gives the full PCIe rate): m_host is copied to the device, advanced n steps and copied back, all on
 * the context's stream; returns after the copy back.  This is the end-to-end call bench.py times. */
mm_status mm_steps_fixed_host(mm_ctx* ctx, float* m_host, mm_method method, double dt, int n,
                              double* t_inout, double* max_err_out);

/* mm_fused_eval -- the unit the throughput metric counts: ONE fused evaluation = demag convolution +
 * local field terms + torque + an RK4-shaped stage combine + max-norm reduction, i.e. stage `stage`
 * (0-based) of `method` applied to m_dev with step dt, writing the stage derivative and the next stage
 * input into the context's Runge-Kutta buffers.  m_dev is not modified unless it is the last stage.
 * Asynchronous; used by bench.py and by the step functions above. */
mm_status mm_fused_eval(mm_ctx* ctx, float* m_dev, mm_method method, int stage, double dt,
                        uint64_t step);

/* mm_reset_stepper -- set the index of the next time step (it selects the thermal draw, reading A6;
 * mm_step / mm_steps_fixed advance it by one per accepted step) and forget the saved first stage of
 * the FSAL methods.  Call it after writing into m_dev from outside between two steps. */
mm_status mm_reset_stepper(mm_ctx* ctx, uint64_t step_index);

/* mm_demag_field -- magnetostatic field only (A/m), H_ms = -Ms sum_j N(r_i - r_j) m_j
 * (discrete Eq. (2)): test and diagnostic entry (reading A12).  Asynchronous. */
mm_status mm_demag_field(mm_ctx* ctx, const float* m_dev, float* H_dev);

/* mm_get_demag_kernel -- test hook: copy component comp (0..5 = xx,yy,zz,xy,xz,yz) of the stored
 * octant K-hat[(Pz/2+1)][(Py/2+1)][(Px/2+1)] (float32, includes the factor -1/(Px Py Pz)) to host_out.
 *   n  capacity of host_out in floats; MM_EINVAL if too small. */
mm_status mm_get_demag_kernel(mm_ctx* ctx, int comp, float* host_out, size_t n);

/* mm_demag_tensor_host -- test hook, HOST only, needs no device and no context state beyond the grid:
 * the library's own real-space tensor N (xx,yy,zz,xy,xz,yz) at n integer cell offsets off[3*i..],
 * periodic images included as mm_create's pbc says.  out_host[6*i..], double. */
mm_status mm_demag_tensor_host(const double cellsize[3], const int grid[3], const int pbc[3],
                               size_t n, const long* off_host, double* out_host);

/* mm_demag_khat_host -- test hook, HOST only, needs no device: the transformed kernel exactly as
 * mm_demag_init would upload it, out_host[6][Cz][Cy][Cx] float32 (n = capacity in floats). */
mm_status mm_demag_khat_host(const double cellsize[3], const int grid[3], const int pbc[3],
                             float* out_host, size_t n);

/* mm_padded_size -- padded FFT sizes P[3] and the octant extents C[3] = P/2 + 1 of this context. */
mm_status mm_padded_size(const mm_ctx* ctx, int P_out[3], int C_out[3]);

/* mm_padded_size_of -- the same rule (reading A9: 2 N open, N periodic, 1 for a one-cell axis) for a grid
 * without a context; HOST only, needs no device.  MM_EUNSUPPORTED if a padded size is not 2^a 3^b 5^c 7^d. */
mm_status mm_padded_size_of(const int grid[3], const int pbc[3], int P_out[3], int C_out[3]);

/* mm_create_batch -- nfilms INDEPENDENT films of the same grid (Nz = 1), cell size, boundary conditions and
 * material in one context (many small simulations, the shape of the paper's 200-run sweep,
 * PAPER.md:181, where one small grid is launch-bound).  Every field is float32 [3][nfilms][Ny][Nx]: film b is plane
 * b.  Each pass is ONE launch over all films (they share K-hat; nothing couples two planes), and every entry point
 * of a plain context works unchanged: the steppers advance all films with the same dt, the max-norm (error
 * estimate, step control) is taken over the whole batch, the thermal draw differs from film to film.
 * Needs padded x and y lengths 32 ... 1024 with a size-specialised kernel and Nx % 4 == 0 (MM_EUNSUPPORTED at
 * mm_demag_init otherwise). */
mm_status mm_create_batch(mm_ctx** out, const int grid[3], const double cellsize[3], const int pbc[3],
                          void* cuda_stream, int nfilms);

/* mm_batch_set_field -- one applied field per film (a hysteresis sweep in one context): B_host[nfilms][3] in
 * tesla replaces mm_material.Bext; NULL returns to the material's uniform field.  Needs mm_set_material and
 * mm_demag_init first.  Blocking. */
mm_status mm_batch_set_field(mm_ctx* ctx, const double* B_host);

/* mm_set_option -- per-context tuning switches (integers; defaults are the measured best on B200):
 *   "graph"          1 (default): mm_steps_fixed replays a captured CUDA graph of one step; 0: plain launches
 *   "x_pipe"         bit 0: forward x pass in its cp.async-pipelined form (default 1); bit 1: inverse x pass too (the
 *                    two-kernel last pass only); bit 2: the forward pass stages its rows by one bulk copy per row pair
 *                    instead of cp.async (measured equal: off)
 *   "mid_pipe"       last-axis pass: 2 (default) persistent, TMA tile loads, packed f32x2 codelets (padded z
 *                    length 128; other lengths take 1); 1: persistent, cp.async-pipelined; 0: one block per line set
 *   "spec_panel"     1 (default): when the "mid_pipe" 2 kernel runs, the y-transformed spectrum is kept in panels of
 *                    16 kx columns between a2, a3 and a4 (same arithmetic, DRAM-friendlier rows); 0: plain rows
 *   "y_tma"          in that panel form, y lines of 1024: 0: tiles by cp.async (16 per thread and tile); 1: by TMA
 *                    (cp.async.bulk.tensor, one thread issues); 2 (default): and the forward pass also stores its
 *                    results through a staging tile and TMA tile stores; 3: both directions do
 *   "last_fused"     1 (default): where it applies (padded x length 1024, 512 or 256, Nx a multiple of 128, no staircase geometry) the
 *                    inverse x pass and the per-cell tail are ONE kernel, H_ms passing through shared memory;
 *                    0: two kernels with H_ms written to and read from device memory (every other grid does that)
 *   "chunk_w"        > 0: run the y / last-axis passes in L2-resident chunks of that many kx columns (multiple
 *                    of 16; default 0 = whole-array passes); "chunk_streams" 1..4 streams for them (default 3).
 *                    These two must be set BEFORE mm_demag_init (MM_ESTATE afterwards).
 * Results do not depend on any option (tested bit for bit).  Errors: MM_EINVAL (unknown key, bad value). */
mm_status mm_set_option(mm_ctx* ctx, const char* key, int value);

/* mm_launch_count -- number of kernels this context has launched so far (bench.py "gpu_launches"). */
uint64_t mm_launch_count(const mm_ctx* ctx);

/* mm_kernel_timing / mm_kernel_times -- optional per-pass timing with CUDA events recorded on the
 * context's stream around every launch (bench.py "roofline").  mm_kernel_timing(ctx, 1) switches it on
 * and clears the counters; mm_kernel_times synchronises the stream and returns, per pass category
 * (0 forward x, 1 forward y, 2 last axis + K-hat multiply, 3 inverse y, 4 inverse x (+ epilogue when
 * fused), 5 other, 6 the per-cell epilogue kernel of the split last pass), the summed device seconds
 * and the number of launches since the last call. */
mm_status mm_kernel_timing(mm_ctx* ctx, int enable);
mm_status mm_kernel_times(mm_ctx* ctx, double sec_out[7], uint64_t count_out[7]);

/* mm_set_fast_path -- bit mask of the passes that may use the size-specialised register FFT kernels
 * when the grid allows (1 forward x, 2 the y passes, 4 last axis + K-hat multiply, 8 inverse x +
 * fused epilogue, 16 the split last pass: inverse x to an H_ms field, then a streaming per-cell
 * kernel; 16 wins over 8; 32 allows the L2-resident kx chunks of the y / last-axis passes when the
 * option "chunk_w" asks for them); a negative value (and the default) enables all, 0
 * forces the generic shared-memory
 * radix-2/3/4/5 kernels.  Both families use the same layouts, so tests compare them pass by pass. */
mm_status mm_set_fast_path(mm_ctx* ctx, int enable);

/* mm_copy_bandwidth -- the library's own float4 grid-stride copy kernel, used by bench.py as the
 * HBM roofline cross-check: copies nbytes from src_dev to dst_dev `reps` times and
 * returns the mean seconds per copy in *sec_out (device-timed with CUDA events).  Blocking. */
mm_status mm_copy_bandwidth(mm_ctx* ctx, const void* src_dev, void* dst_dev, size_t nbytes,
                            int reps, double* sec_out);


/* ---- multi-GPU slab decomposition ("multi-GPU ... efficient communication") ----
 * One process per GPU.  Rank r owns the planes z0 <= z < z1 of every field (all x, y) and, for the transform
 * along z, the columns kx0 <= kx < kx1 of the half spectrum (all ky, all z).  One evaluation is
 *   mm_dist_forward   a1, a2 on the slab; the y pass writes straight into the exchange layout
 *   all-to-all #1     slab buffer -> pencil buffer   (done by the CALLER: NCCL, or copies in a test)
 *   mm_dist_mid       a3 on the pencil (full z lines, this rank's K-hat columns)
 *   all-to-all #2     pencil buffer -> slab buffer
 *   halo exchange     plane z0 to rank r-1, plane z1-1 to rank r+1 (m only, one plane each way)
 *   mm_dist_backward  a4, a5 and the per-cell tail a6-a8 on the slab
 * The library does no communication itself: it exposes the two device buffers and, per (peer, component), the
 * contiguous segment that travels, so that each all-to-all is a list of contiguous sends and receives with no
 * pack or unpack kernel.  DESIGN.md section 10 has the layouts and the byte counts. */
typedef struct {
    int rank, nranks;
    int z0, z1;   /* planes owned                                                                  */
    int kx0, kx1; /* columns of the half spectrum (0 .. Px/2) owned for the z pass; multiples of 16 */
} mm_slab;

/* mm_slab_partition -- the partition rule, HOST only (no device, no context): planes in contiguous balanced
 * ranges, columns in contiguous ranges of whole 16-column tiles.  Errors: MM_EINVAL (nranks < 1, rank out of range,
 * more ranks than planes or than column tiles), MM_EUNSUPPORTED (padded size not 2^a 3^b 5^c 7^d). */
mm_status mm_slab_partition(const int grid[3], const int pbc[3], int nranks, int rank, mm_slab* out);

/* mm_create_dist -- context of one rank: `grid` is the GLOBAL grid; fields passed to the mm_dist_* calls are the
 * local slab, float32 [3][z1-z0][Ny][Nx].  Needs a 3D grid whose passes all have size-specialised kernels and
 * Nx % 4 == 0 (MM_EUNSUPPORTED otherwise).  mm_set_material and mm_demag_init follow as for mm_create
 * (mm_demag_init builds the whole K-hat octant on the host and uploads this rank's columns). */
mm_status mm_create_dist(mm_ctx** out, const int grid[3], const double cellsize[3], const int pbc[3],
                         void* cuda_stream, int rank, int nranks);

/* mm_dist_buffers -- the two exchange buffers (device, float2 elements, owned by the context):
 *   slab_buf    [peer][3][z1-z0][Py][W(peer)]   W(peer) = kx1(peer) - kx0(peer) rounded up to a multiple of 8
 *   pencil_buf  [3][Nz][Py][W(rank)]
 * and their sizes in float2 elements. */
mm_status mm_dist_buffers(mm_ctx* ctx, void** slab_buf_dev, size_t* slab_elems, void** pencil_buf_dev,
                          size_t* pencil_elems);

/* mm_dist_segment -- the contiguous segment exchanged with `peer` for component comp (0..2), in float2
 * elements: all-to-all #1 sends slab_buf[slab_off .. +slab_count) to the peer and receives the peer's planes
 * into pencil_buf[pencil_off .. +pencil_count); all-to-all #2 is the reverse. */
mm_status mm_dist_segment(const mm_ctx* ctx, int peer, int comp, size_t* slab_off, size_t* slab_count,
                          size_t* pencil_off, size_t* pencil_count);

/* mm_slab_segment -- the same bookkeeping without a context, HOST only (the CPU tests drive a two-process
 * all-to-all over gloo with it). */
mm_status mm_slab_segment(const int grid[3], const int pbc[3], int nranks, int rank, int peer, int comp,
                          size_t* slab_off, size_t* slab_count, size_t* pencil_off, size_t* pencil_count);

mm_status mm_dist_forward(mm_ctx* ctx, const float* m_slab_dev);
mm_status mm_dist_mid(mm_ctx* ctx);
/* mm_dist_backward -- what = 0: H_ms (A/m), 1: H_eff (A/m), 2: dm/dt (1/s) into out_slab_dev.
 *   halo_lo_dev / halo_hi_dev   float32 [3][Ny][Nx]: the plane z0-1 / z1 of m from the neighbouring rank (for a
 *   periodic z axis the ring neighbour); NULL at an open boundary of the global grid.  Ignored for what = 0. */
mm_status mm_dist_backward(mm_ctx* ctx, const float* m_slab_dev, const float* halo_lo_dev,
                           const float* halo_hi_dev, float* out_slab_dev, int what, uint64_t step,
                           double dt_for_thermal);

/* Time stepping on slabs: stage `stage` (0-based) of a fixed-step method (MM_RK1, MM_RK2, MM_RK3, MM_RK4) runs like an
 * evaluation -- mm_dist_forward on the stage's input state, the two all-to-alls around mm_dist_mid, the halo exchange of
 * that same state -- and ends with mm_dist_backward_stage instead of mm_dist_backward: a4, a5 and the per-cell tail with
 * the Runge-Kutta stage combine (a9), which writes the next stage's input into a buffer of the context, or, at the last
 * stage, the new normalised state into m_slab_dev.
 *   mm_dist_stage_input   *in_dev_out = the device field stage `stage` acts on (m_slab_dev for stage 0): the caller
 *                         passes it to mm_dist_forward and takes the halo planes from it.
 * The thermal draw is per global cell and step (reading A6).  Step control (embedded methods) is not offered on
 * slabs: its max-norm would need a reduction over the ranks.  Errors: MM_EINVAL for any other method. */
mm_status mm_dist_stage_input(mm_ctx* ctx, mm_method method, int stage, const float* m_slab_dev,
                              const float** in_dev_out);
mm_status mm_dist_backward_stage(mm_ctx* ctx, float* m_slab_dev, mm_method method, int stage, double dt,
                                 uint64_t step, const float* halo_lo_dev, const float* halo_hi_dev);

/* mm_last_error -- message for the last non-OK status of this context ("" if none); for a NULL ctx
 * the message of the last failed mm_create on this thread. */
const char* mm_last_error(const mm_ctx* ctx);

/* mm_destroy -- free everything the context owns (NULL is a no-op). */
void mm_destroy(mm_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* MM_H_ */
