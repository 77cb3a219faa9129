/*
 * steps_cyl.h -- C ABI of libsteps_cyl.so: the data-parallel hot path of the StePS
 * cylindrical (S^1 x R^2, periodic along z, open in x-y) N-body method of
 * arXiv 2602.20787 ("PAPER.md" below = /root/reference/PAPER.md), on one NVIDIA B200
 * (sm_100a).
 *
 * What the library computes
 *   steps_cyl_accel    g_i = sum_{j != i} m_j F_{S1xR2}(x_i - x_j, h_i + h_j)
 *                      Eq. 1 with the one-axis-periodic pair law of Eq. 8
 *                      (PAPER.md:85-90): the truncated z-image sum of the R^3 law Eq. 4
 *                       through the cubic-spline softening Eq. 3
 *                      (PAPER.md:56-61).  g includes G; it EXCLUDES 1/a^3, the Hubble drag
 *                      and the background term of Eq. 11 -- those are applied in kdk_step.
 *   steps_cyl_background
 *                      b_i = -F_h(rho_i; R_sim, N_cut L_z) e_rho: the homogeneous-cylinder
 *                      term of Eq. 11, F_h from Eq. 9 or
 *                      its N_cut -> infinity limit Eq. 10.
 *   steps_cyl_kdk_step one kick-drift-kick leapfrog step of Eq. 11 in cosmic time t
 *                      (PAPER.md:128-133), comoving coordinates.
 *   steps_cyl_friedmann_step
 *                      one RK4 step of the Friedmann equation Eq. 18,
 *                      host scalars.
 *
 * Conventions common to all calls
 *   - Every function returns STEPS_OK (0) or a negative steps_cyl_status.  Nothing throws,
 *     aborts or prints.  steps_cyl_strerror(code) gives a static string; for STEPS_ECUDA the
 *     text of the last CUDA error seen by that context is available through
 *     steps_cyl_last_cuda_error(ctx).
 *   - "device pointer" = CUDA global memory on params.device; "host pointer" = ordinary (or
 *     pinned) host memory.  All arrays are contiguous double precision, length n, SoA (one
 *     array per coordinate).  The caller owns every particle array; the context owns only its
 *     scratch and tables.  No pointer is retained after a call returns.
 *   - Device-pointer calls are ASYNCHRONOUS: work is enqueued on `cuda_stream` (a cudaStream_t
 *     passed as void*; NULL = the legacy default stream) and the call returns without
 *     synchronising.  Host-pointer calls (…_host) copy in, compute, copy out and synchronise
 *     the context's own stream before returning.
 *   - One context serves one stream at a time: calls on one context must be serialised by the
 *     caller.  Different contexts are independent.
 *   - z may lie outside [0, Lz): it is reduced to [0, Lz) first (periodicity).
 *     NaN / Inf inputs are not checked (garbage in, garbage out).
 *   - There is NO CPU fallback: without a CUDA device steps_cyl_init returns STEPS_ECUDA.
 *   - Every call that takes a context makes params.device current while it runs and restores the
 *     caller's current device before it returns.
 */
#ifndef STEPS_CYL_H
#define STEPS_CYL_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    STEPS_OK           =  0,
    STEPS_EINVAL       = -1,  /* bad argument: n < 1, Lz <= 0, n_cut < 1, NULL pointer, unknown enum   */
    STEPS_ESOFT        = -2,  /* softening precondition violated: some h_i <= 0 (or NaN)                   */
    STEPS_ECUDA        = -3,  /* a CUDA runtime call failed (or no device present)                     */
    STEPS_ENOMEM       = -4,  /* host or device allocation failed                                      */
    STEPS_EUNSUPPORTED = -5,  /* a combination this build does not contain (EWALD_TABLE with
                                 STEPS_FLAG_ORDERED_PAIRS, or a float table too large for shared memory) */
    STEPS_ETOOBIG      = -6   /* steps_cyl_accel_noalloc only: n > STEPS_CYL_NOALLOC_MAX_N               */
} steps_cyl_status;

enum { STEPS_PERIODIC_IMAGES = 0,      /* Eq. 8, truncated image sum                                  */
       STEPS_PERIODIC_EWALD_TABLE = 1  /* Eq. 12-17: softened nearest image + interpolated table D
                                          (mixed precision implies tab_fp32 = 1)                       */ };
enum { STEPS_PREC_FP64 = 0,            /* every pair term and the accumulation in double               */
       STEPS_PREC_MIXED = 1            /* pair terms in float (cancellation-safe separations),
                                          accumulation over sources in double                          */ };
enum { STEPS_INTERP_CIC = 0,           /* cloud-in-cell: bilinear in (rho, z)                          */
       STEPS_INTERP_TSC = 1            /* triangular-shaped cloud: quadratic B-spline on 3 x 3 nodes   */ };
enum { STEPS_BG_FINITE = 0,            /* Eq. 9 with L = n_cut * Lz                                    */
       STEPS_BG_INFINITE = 1           /* Eq. 10                                                       */ };

enum { STEPS_FLAG_DETERMINISTIC = 1,   /* bit-reproducible results.  The default kernels evaluate every
                                          unordered pair once and add it to both particles with
                                          floating-point atomics (same terms, summation order varies from
                                          run to run, ~1e-16).  With this flag the fp64 image mode up to
                                          N = 131072 writes every sum to a slot with one writer and adds the
                                          slots in fixed order (~4 % slower, 24 B x N x (N/256 + ~20) of
                                          scratch); larger N and the other modes schedule the evaluation in
                                          conflict-free rounds with plain stores (~3 % slower at N = 1M)     */
       STEPS_FLAG_FAR_ORDER2 = 2,      /* fp64 images mode, default kernel only: the rsqrt refinement of
                                          the FAR images (n != 0) drops its second-order term: 8 % faster,
                                          per-particle error <~ 2e-12 instead of ~1e-14 (bar: 1e-10)  */
       STEPS_FLAG_ORDERED_PAIRS = 4,   /* fp64 / mixed images mode: the literal form of Eq. 1 -- every target
                                          sums over all its sources (ordered pairs, fixed-order reduction,
                                          bit-reproducible, ~1.9x slower than the default)             */
       STEPS_FLAG_GRAPH = 8            /* steps_cyl_accel / steps_cyl_kdk_step replay a CUDA graph captured on the
                                          first call with a given set of array pointers (one launch per call
                                          instead of three: small-N step latency); same kernels, same results.
                                          steps_cyl_last_pair_kernel_ms is not available in this mode  */ };

/* Largest particle number one context takes: the symmetric kernels put chunks of <= 64 source tiles of 128
 * particles on gridDim.y (<= 65535).  (At 40 B/particle in and ~250 B/particle of scratch this is also
 * about what 180 GB hold.) */
#define STEPS_CYL_MAX_N ((int64_t)64 * 65535 * 128)

typedef struct steps_cyl_ctx steps_cyl_ctx;   /* opaque; created by init, freed by destroy */

/* Plain-old-data parameter block (the quantities the problem statement
 * names).  Zero-initialise, then fill. */
typedef struct {
    int64_t n;              /* number of particles, 1 <= n <= STEPS_CYL_MAX_N (else EINVAL at init)   */
    double  Lz;             /* period along z, > 0                                      */
    double  G;              /* gravitational constant, any sign (G < 0: glass making)   */
    int32_t periodic_mode;  /* STEPS_PERIODIC_*                                                       */
    int32_t n_cut;          /* N_cut of Eq. 8, >= 1: 2*N_cut images per pair.  Any value is accepted and gives
                               the same sum; 1..8 run fully unrolled kernel instances, 9..64 a run-time image loop
                               with tabulated per-image constants, larger values a loop that forms them          */
    int32_t precision;      /* STEPS_PREC_*                                                           */
    int32_t background;     /* STEPS_BG_*                                                             */
    double  R_sim;          /* radius R of the simulation volume in Eq. 9; needed if rho0 != 0 and
                               background == STEPS_BG_FINITE                                          */
    double  rho0;           /* comoving mean density of Eq. 9/10; 0 disables the background term      */
    int32_t device;         /* CUDA device ordinal                                                    */
    int32_t flags;          /* bitwise OR of STEPS_FLAG_*; 0 = defaults                               */
    /* STEPS_PERIODIC_EWALD_TABLE only; zeros select the defaults in brackets   */
    int32_t ew_nmax;        /* real-space images n = -nmax..nmax of Eq. 13        [5]                 */
    int32_t ew_mmax;        /* Fourier modes m = 1..mmax of Eq. 14                [12]                */
    double  ew_alpha;       /* Ewald split parameter alpha, 1/length              [2/Lz]              */
    int32_t tab_nrho;       /* radial nodes of the table D(rho, z)                [144]               */
    int32_t tab_nz;         /* axial nodes, z in [0, Lz/2]                        [128]               */
    double  tab_rho_max;    /* radial extent of the table; beyond it the pair force is the line-mass
                               term -2 G m/(Lz rho) e_rho (reading T2)            [5 Lz]              */
    int32_t interp;         /* STEPS_INTERP_CIC or STEPS_INTERP_TSC                    */
    int32_t tab_fp32;       /* precision tier of the table (with precision = STEPS_PREC_FP64; MIXED implies 1):
                               0: nodes in double, interpolated in double -- the fp64 contract (<= 1e-10 per particle
                                  against the same table interpolated by the definition);
                               1: "fp64 pairs, fp32 table": nodes rounded to float, held in shared memory, their
                                  weighted sum taken in fp32, everything else double.  Contract: max <= 2e-6, median
                                  <= 5e-8 per particle against the same float nodes interpolated in double (<= 4 float
                                  roundings of each pair's D; the paper's (5,12) Ewald sum behind the nodes is itself
                                  single-precision accurate).  Needs nrho*nz*8 B + 56 KB of shared
                                  memory per SM (144 x 128 fits), else STEPS_EUNSUPPORTED                     */
} steps_cyl_params;

/* Validate `p`, select the device, allocate scratch for n particles and build the constant
 * tables (image offsets, quadrature nodes of Eq. 9).  Host-synchronous.
 * Errors: EINVAL, EUNSUPPORTED, ECUDA, ENOMEM. */
int steps_cyl_init(const steps_cyl_params *p, steps_cyl_ctx **out);

/* Free everything the context owns.  NULL is allowed. */
void steps_cyl_destroy(steps_cyl_ctx *ctx);

/* g_i = sum_{j != i} m_j F_{S1xR2}(x_i - x_j, h_i + h_j)            (Eq. 1 + Eq. 8 + Eq. 3/4)
 * in : x y z m h   device pointers, length n, read only
 * out: gx gy gz    device pointers, length n, overwritten
 * Asynchronous on cuda_stream.  The softening precondition (every h_i > 0) is checked on the
 * device; its violation is reported by the next call to steps_cyl_check(ctx, stream) (which
 * synchronises), and the outputs are then unspecified.  When 2*max(h) <= Lz/2 only the nearest
 * image of a pair can lie inside the spline support and the fast kernel runs; otherwise
 * (reading S7) a general kernel sends every image through Eq. 3 -- same result, slower; the
 * choice is made on the device, with no host synchronisation. */
int steps_cyl_accel(steps_cyl_ctx *ctx,
                    const double *x, const double *y, const double *z,
                    const double *m, const double *h,
                    double *gx, double *gy, double *gz, void *cuda_stream);

/* Same, with HOST pointers: copies the five inputs to the device, runs the same kernels,
 * copies the three outputs back, synchronises, and reports ESOFT directly. */
int steps_cyl_accel_host(steps_cyl_ctx *ctx,
                         const double *x, const double *y, const double *z,
                         const double *m, const double *h,
                         double *gx, double *gy, double *gz);

/* The same force evaluation as steps_cyl_accel -- g_i = sum_{j != i} m_j F_{S1xR2}(x_i - x_j, h_i + h_j), Eq. 1 +
 * Eq. 8 + Eq. 3/4, fp64, truncated image sum with n_cut, the default symmetric kernel -- for callers that CANNOT
 * ALLOCATE (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  It needs no
 * context: it calls no cudaMalloc, cudaFree or other allocating routine, ever.  Its scratch (packed sources,
 * accumulators, flags) is one static device array of STEPS_CYL_NOALLOC_MAX_N particle slots, 2.25 MiB, which every
 * GPU that loads the library holds until the process exits.
 * in : n, Lz, G, n_cut   as in steps_cyl_params;  x y z m h   device pointers on the CURRENT device, length n
 * out: gx gy gz          device pointers, length n, overwritten.   Asynchronous on cuda_stream.
 * Errors: EINVAL (NULL pointer, n < 1, Lz <= 0, n_cut < 1), ETOOBIG (n > STEPS_CYL_NOALLOC_MAX_N; nothing is
 * launched), ECUDA.  h_i <= 0 is NOT reported by this call (there is no context to ask): the outputs are then
 * unspecified.  2*max(h) > Lz/2 is handled as in steps_cyl_accel (general pair law, chosen on the device).
 * - The first call on a device does the one-time set-up (address of the static array, SM count); make it outside
 *   stream capture.  Later calls enqueue one 48-byte memset and three kernels, nothing else.
 * - Every call on a device shares the one array, which keeps the last call's contents (what must start at zero
 *   is cleared at the start of each call).  Two calls that OVERLAP on the GPU -- different streams, or graphs
 *   replayed concurrently -- race on it: serialise them. */
#define STEPS_CYL_NOALLOC_MAX_N ((int64_t)32768)
int steps_cyl_accel_noalloc(int64_t n, double Lz, double G, int32_t n_cut,
                            const double *x, const double *y, const double *z,
                            const double *m, const double *h,
                            double *gx, double *gy, double *gz, void *cuda_stream);

/* Synchronise `cuda_stream` and return the deferred status of the calls enqueued so far on
 * this context (STEPS_OK, STEPS_ESOFT or STEPS_ECUDA); clears it. */
int steps_cyl_check(steps_cyl_ctx *ctx, void *cuda_stream);

/* b_i = -F_h(rho_i) (x_i, y_i)/rho_i, rho_i = sqrt(x_i^2 + y_i^2)   (Eq. 9 / Eq. 10, Eq. 11)
 * in : x y   device pointers, length n;   out: bx by  device pointers, length n.
 * rho0 == 0 writes zeros.  Asynchronous on cuda_stream. */
int steps_cyl_background(steps_cyl_ctx *ctx, const double *x, const double *y,
                         double *bx, double *by, void *cuda_stream);

/* One KDK leapfrog step of Eq. 11 in cosmic time (readings S4, G5):
 *   kick1 : v <- v + (dt/2) [ (g + b)/a_n^3 - 2 H_n v ]
 *   drift : x <- x + v dt ;  z reduced to [0, Lz)
 *   force : g <- steps_cyl_accel(x) ;  b <- steps_cyl_background(x)
 *   kick2 : v <- [ v + (dt/2) (g + b)/a_np1^3 ] / (1 + H_np1 dt)
 * in/out: x y z vx vy vz   device pointers, length n, updated in place
 * in    : m h              device pointers, length n
 * in/out: gx gy gz         on entry g(x_n) (from steps_cyl_accel or the previous step), on
 *                          return g(x_{n+1})
 * a_n, H_n, a_np1, H_np1   scale factor and Hubble parameter at t_n and t_n + dt (from the
 *                          caller, e.g. steps_cyl_friedmann_step); dt the step in cosmic time.
 * Asynchronous on cuda_stream. */
int steps_cyl_kdk_step(steps_cyl_ctx *ctx,
                       double *x, double *y, double *z,
                       double *vx, double *vy, double *vz,
                       const double *m, const double *h,
                       double *gx, double *gy, double *gz,
                       double a_n, double H_n, double a_np1, double H_np1, double dt,
                       void *cuda_stream);

/* Same step with HOST pointers: copies the eleven arrays to the device (88 B/particle), runs the
 * same kernels, copies x y z vx vy vz gx gy gz back (72 B/particle), synchronises, and reports
 * ESOFT directly.  This is the end-to-end form bench.py times. */
int steps_cyl_kdk_step_host(steps_cyl_ctx *ctx,
                            double *x, double *y, double *z,
                            double *vx, double *vy, double *vz,
                            const double *m, const double *h,
                            double *gx, double *gy, double *gz,
                            double a_n, double H_n, double a_np1, double H_np1, double dt);

/* Friedmann equation Eq. 18 with a cosmological constant:
 * H(a) = H0 sqrt(Or a^-4 + Om a^-3 + Ok a^-2 + OL); one classical RK4 step of da/dt = a H(a)
 * with the N-body step dt.  Host only, no context.  EINVAL on NULL / a <= 0. */
int steps_cyl_friedmann_step(double a, double dt, double H0, double Om, double Or, double Ok,
                             double OL, double *a_next, double *H_next);

/* The same step for a Chevallier-Polarski-Linder dark energy, Eq. 18-20:
 * O_DE(a) = ODE exp[-3 int_1^a (1 + w(a'))/a' da'], w(a) = w0 + wa (1 - a), i.e.
 * O_DE(a) = ODE a^(-3 (1 + w0 + wa)) exp(3 wa (a - 1)).  w0 = -1, wa = 0 is steps_cyl_friedmann_step with
 * OL = ODE; wa = 0 is wCDM.  Host only, no context.  EINVAL on NULL / a <= 0. */
int steps_cyl_friedmann_step_cpl(double a, double dt, double H0, double Om, double Or, double Ok,
                                 double ODE, double w0, double wa, double *a_next, double *H_next);

/* The correction lookup table of Eq. 17, D = F_{S1xR2} - F_{R3} per unit G m_i m_j (Ewald sum of
 * Eq. 12-16 with the Fourier kernel of DESIGN.md reading G4, minus the unsoftened nearest-image
 * force), on the grid rho_i = i rho_max/(nrho-1), z_j = j (Lz/2)/(nz-1).
 * out: HOST pointer, nrho*nz*2 doubles, D[(i*nz + j)*2 + c], c = 0 radial, 1 axial.
 * Host only, no context, no device.  EINVAL on NULL, Lz <= 0, alpha <= 0, nrho < 2, nz < 2,
 * nmax < 0, mmax < 0, rho_max <= 0. */
int steps_cyl_ewald_table(double Lz, double alpha, int32_t nmax, int32_t mmax, int32_t nrho,
                          int32_t nz, double rho_max, double *out);

/* Measured ceiling of the FP64 pipe: runs an unrolled chain of independent DFMAs on every SM
 * of the context's device for about `ms` milliseconds and returns DFMA instructions per
 * second (thread-level) in *dfma_per_s.  Used by bench.py for the roofline denominator.
 * Host-synchronous. */
int steps_cyl_fp64_peak(steps_cyl_ctx *ctx, double ms, double *dfma_per_s);

/* Milliseconds the device spent in the most recent all-pairs kernel launch of this context
 * (CUDA events recorded around that launch on its stream); synchronises on the end event. */
int steps_cyl_last_pair_kernel_ms(steps_cyl_ctx *ctx, float *ms);

/* Name of the all-pairs kernel this context launches for its parameters, as the SASS tally
 * (paper_2602_20787_b200/sassmix.py) spells it, e.g. "pair_fp64_sym_kernel<5,false>".  Static per context. */
const char *steps_cyl_pair_kernel_name(steps_cyl_ctx *ctx);

/* Mixed-precision image kernel only: how many of its two-way ring passes (32 sources x 64 targets of a warp) since
 * init took the SIMPLE form (plain float separations, one nearest-image shift, no spline test; possible where the
 * Morton-ordered groups are far apart) out of all such passes.  Synchronises cuda_stream.  Both 0 for other kernels.
 * bench.py weights the two loops' instruction tallies with this ratio. */
int steps_cyl_pass_stats(steps_cyl_ctx *ctx, void *cuda_stream, uint64_t *simple, uint64_t *total);

const char *steps_cyl_strerror(int code);
const char *steps_cyl_last_cuda_error(steps_cyl_ctx *ctx);

/* Number of kernels this context has launched since init (bench.py's gpu_launches). */
int64_t steps_cyl_launch_count(steps_cyl_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* STEPS_CYL_H */
