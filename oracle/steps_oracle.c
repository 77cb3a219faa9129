/*
 * steps_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision CPU restatement of the hot path of the StePS
 * cylindrical (S^1 x R^2) method, written from the paper's definitions
 * (/root/reference/PAPER.md, arXiv 2602.20787).  It shares no code, header,
 * table or constant with the CUDA path under paper_2602_20787_b200/csrc/ and
 * is never imported, linked or executed by it.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call it.
 *
 * Everything is evaluated term by term in the order of the paper's formulas;
 * there is no blocking, no fast rsqrt, no symmetry trick.  Each pair term is
 * computed in double; the sum over sources is carried in long double (x87
 * 80-bit) so that the summation order does not matter at the 1e-10 parity bar.
 *
 * Pins (tests/test_oracle_pins.py): spline continuity / enclosed-mass form,
 * two-particle values recomputed with 50-digit arithmetic, trigamma on-axis
 * closed form, Bessel-series infinite sum, rod / line-mass limit, periodicity,
 * rotation, momentum conservation, literal Eq. 8 transcription, background
 * force vs 2-D quadrature and Eq. 10, free-streaming and EdS closed forms.
 *
 * Parity unpinned: the default N_cut (the paper
 * states none), and the exact discretisation of the Hubble-drag term inside
 * StePS's KDK (pinned only to O(dt^2)).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------ Eq. 3
 * Cubic-spline softened force magnitude F(r,h), PAPER.md:56-61 (Sect. 2.1,
 * Eq. 3).  DESIGN.md reading G1: the second term of the first branch is
 * 38.4 r^3/h^5 (printed h^3 is dimensionally wrong and discontinuous). */
double oracle_spline_F(double r, double h)
{
    if (r < 0.5 * h) {
        return 32.0 * pow(r, 4) / pow(h, 6) - 38.4 * pow(r, 3) / pow(h, 5)
             + 32.0 * r / (3.0 * pow(h, 3));
    } else if (r < h) {
        return -32.0 * pow(r, 4) / (3.0 * pow(h, 6)) + 38.4 * pow(r, 3) / pow(h, 5)
             - 48.0 * r * r / pow(h, 4) + 64.0 * r / (3.0 * pow(h, 3))
             - 1.0 / (15.0 * r * r);
    }
    return 1.0 / (r * r);
}

/* ------------------------------------------------------------------ Eq. 8
 * One source of unit mass at separation r = x_i - x_j (target minus source);
 * returns the acceleration on the target, PAPER.md:85-90 (Eq. 8) with the
 * R^3 law of Eq. 4 for each image.
 *   1. r_z is reduced to the nearest image, r_z in [-L/2, L/2]   (reading S1)
 *   2. image set: n = -N_cut+1 .. N_cut-1, plus n = +N_cut if r_z > 0,
 *      plus n = -N_cut if r_z < 0  == the literal constraint
 *      |r_z - n L| < N_cut L of Eq. 8 (reading G2)
 *   3. every image goes through the spline with h = h_i + h_j (Eq. 1)
 *   4. an image at zero distance contributes nothing (s -> 0 limit of Eq. 3)
 * acc[] is long double and is ADDED to. */
static void pair_images(double rx, double ry, double rz, double hh, double L,
                        double G, double mj, int ncut, long double acc[3])
{
    rz = rz - L * rint(rz / L);
    int nlo = -ncut + 1, nhi = ncut - 1;
    if (rz > 0.0) nhi = ncut;
    if (rz < 0.0) nlo = -ncut;
    for (int n = nlo; n <= nhi; ++n) {
        double d = rz - (double)n * L;
        double s = sqrt(rx * rx + ry * ry + d * d);
        if (s == 0.0) continue;
        double w = oracle_spline_F(s, hh) / s;      /* F(s,h) * (r/|r|) = w * r */
        acc[0] += (long double)(-G * mj * w * rx);
        acc[1] += (long double)(-G * mj * w * ry);
        acc[2] += (long double)(-G * mj * w * d);
    }
}

void oracle_pair_accel(double rx, double ry, double rz, double hh, double L,
                       double G, int ncut, double g[3])
{
    long double acc[3] = {0.0L, 0.0L, 0.0L};
    pair_images(rx, ry, rz, hh, L, G, 1.0, ncut, acc);
    g[0] = (double)acc[0]; g[1] = (double)acc[1]; g[2] = (double)acc[2];
}

/* ------------------------------------------------------------ Eq. 1 / 11
 * g_i = sum_{j != i} m_j F_{S1xR2}(x_i - x_j, h_i + h_j)
 * (Eq. 1) and PAPER.md:128-131 (Eq. 11) -- the pair sum only: no 1/a^3, no
 * drag, no background term.  targets == NULL means all particles; otherwise
 * nt indices into the particle arrays.  z is first reduced to [0, L)
 * (periodicity).  Returns 0, or -1 on bad arguments. */
int oracle_accel(int64_t n, const double *x, const double *y, const double *z,
                 const double *m, const double *h, double L, double G, int ncut,
                 int64_t nt, const int64_t *targets,
                 double *gx, double *gy, double *gz, int nthreads)
{
    if (n < 1 || L <= 0.0 || ncut < 1 || !x || !y || !z || !m || !h || !gx || !gy || !gz)
        return -1;
    if (!targets) nt = n;
    double *zw = (double *)malloc((size_t)n * sizeof(double));
    if (!zw) return -1;
    for (int64_t j = 0; j < n; ++j) {
        zw[j] = z[j] - L * floor(z[j] / L);
        if (zw[j] >= L) zw[j] -= L;          /* floor() round-off guard: keep [0,L) */
    }
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#endif
    #pragma omp parallel for schedule(dynamic, 4)
    for (int64_t t = 0; t < nt; ++t) {
        int64_t i = targets ? targets[t] : t;
        long double acc[3] = {0.0L, 0.0L, 0.0L};
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            pair_images(x[i] - x[j], y[i] - y[j], zw[i] - zw[j], h[i] + h[j],
                        L, G, m[j], ncut, acc);
        }
        gx[t] = (double)acc[0]; gy[t] = (double)acc[1]; gz[t] = (double)acc[2];
    }
    free(zw);
    return 0;
}

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------ Eq. 9
 * Radial field of the homogeneous cylinder of radius R and height 2L
 * (L = N_cut L_z) in its central plane, PAPER.md:92-96 (Eq. 9, Chang 1988),
 * DESIGN.md reading G3 (signs / square roots of the printed form corrected so
 * that it is the actual field and tends to Eq. 10):
 *   F_h = 2 G rho0 [ +2 int_0^R ln((w+ + L)/(w- + L)) dY - int_0^R ln(a+/a-) dY ]
 *   a+- = R^2 + rho^2 +- 2 rho sqrt(R^2 - Y^2),   w+- = sqrt(L^2 + a+-).
 * Negative = pointing to the axis.  Both integrals are done numerically in Y,
 * as printed, by tanh-sinh quadrature (handles the sqrt end-point at Y = R and
 * the logarithmic one at rho = R). */
/* e = R - Y is passed separately so that sqrt(R^2 - Y^2) = sqrt(e (R + Y)) has no
 * cancellation at the quadrature nodes that crowd the end point Y = R. */
static double fh_integrand(double Y, double e, double rho, double R, double L)
{
    double X = sqrt(fmax(e * (R + Y), 0.0));
    /* a+- = R^2 + rho^2 +- 2 rho X with R^2 = X^2 + Y^2, written as (rho +- X)^2 + Y^2: the same
     * number, but free of the cancellation that a- suffers for rho ~ R near Y = 0 */
    double ap = (rho + X) * (rho + X) + Y * Y;
    double am = (rho - X) * (rho - X) + Y * Y;
    double wp = sqrt(L * L + ap), wm = sqrt(L * L + am);
    if (am <= 0.0) return 0.0;               /* single point rho = R, Y = 0: integrable */
    return 2.0 * log((wp + L) / (wm + L)) - (log(ap) - log(am));   /* ap/am may overflow at rho = R */
}

static double fh_integrand_inf(double Y, double e, double rho, double R)
{
    double X = sqrt(fmax(e * (R + Y), 0.0));
    double ap = (rho + X) * (rho + X) + Y * Y;
    double am = (rho - X) * (rho - X) + Y * Y;
    if (am <= 0.0) return 0.0;
    return -(log(ap) - log(am));
}

/* tanh-sinh on [0,R]; doubles the node count until two levels agree to 1e-14. */
static double tanh_sinh(double rho, double R, double L, int inf_limit)
{
    const double half = 0.5 * R;
    double hstep = 1.0, prev = 0.0, sum = 0.0;
    const double pi2 = 1.5707963267948966192;
    /* level 0: t = 0 and t = +-k h */
    for (int level = 0; level < 12; ++level) {
        double part = 0.0;
        int first = (level == 0);
        for (int k = first ? 0 : 1; ; k += first ? 1 : 2) {
            double t = k * hstep;
            double u = pi2 * sinh(t);
            double ch = cosh(u);
            double wgt = pi2 * cosh(t) / (ch * ch);
            /* distance of the node from the end point, computed without cancellation */
            double delta = exp(-u) / ch * half;      /* = half*(1 - tanh u) */
            if (wgt * half < 1e-300 || delta <= 0.0) break;
            double Yr = R - delta, Yl = delta;
            double fr = inf_limit ? fh_integrand_inf(Yr, delta, rho, R) : fh_integrand(Yr, delta, rho, R, L);
            double fl = inf_limit ? fh_integrand_inf(Yl, R - Yl, rho, R) : fh_integrand(Yl, R - Yl, rho, R, L);
            if (k == 0) part += wgt * (inf_limit ? fh_integrand_inf(half, half, rho, R)
                                                 : fh_integrand(half, half, rho, R, L));
            else        part += wgt * (fr + fl);
            if (t > 7.0) break;
        }
        sum = (level == 0) ? part : sum + part;      /* nodes of earlier levels are reused */
        double val = sum * hstep * half;
        if (level > 3 && fabs(val - prev) <= 1e-14 * fabs(val)) return val;
        prev = val;
        hstep *= 0.5;
    }
    return prev;
}

double oracle_Fh(double rho, double R, double L, double G, double rho0)
{
    return 2.0 * G * rho0 * tanh_sinh(rho, R, L, 0);
}

/* Eq. 10: the N_cut -> infinity limit, closed form. */
double oracle_Fh_inf(double rho, double G, double rho0)
{
    return -2.0 * 3.14159265358979323846 * G * rho0 * rho;
}

/* Same limit obtained by dropping the L-dependent integral of Eq. 9 and
 * integrating numerically (used only to pin the quadrature against Eq. 10). */
double oracle_Fh_inf_quad(double rho, double R, double G, double rho0)
{
    return 2.0 * G * rho0 * tanh_sinh(rho, R, 0.0, 1);
}

/* ---------------------------------------------------------------- Eq. 18
 * Friedmann equation, with a cosmological constant
 * (w0 = -1, wa = 0 in Eq. 19-20): H(a) and one classical RK4 step of
 * da/dt = a H(a) with the N-body time step. */
double oracle_hubble(double a, double H0, double Om, double Or, double Ok, double OL)
{
    return H0 * sqrt(Or / (a * a * a * a) + Om / (a * a * a) + Ok / (a * a) + OL);
}

void oracle_friedmann_rk4(double a, double dt, double H0, double Om, double Or,
                          double Ok, double OL, double *a_next, double *H_next)
{
    double k1 = a * oracle_hubble(a, H0, Om, Or, Ok, OL);
    double a2 = a + 0.5 * dt * k1;
    double k2 = a2 * oracle_hubble(a2, H0, Om, Or, Ok, OL);
    double a3 = a + 0.5 * dt * k2;
    double k3 = a3 * oracle_hubble(a3, H0, Om, Or, Ok, OL);
    double a4 = a + dt * k3;
    double k4 = a4 * oracle_hubble(a4, H0, Om, Or, Ok, OL);
    double an = a + dt * (k1 + 2.0 * k2 + 2.0 * k3 + k4) / 6.0;
    *a_next = an;
    *H_next = oracle_hubble(an, H0, Om, Or, Ok, OL);
}

/* --------------------------------------------------------------- Eq. 11
 * Comoving background acceleration on one particle: -F_h(rho) along the outward
 * radial unit vector (Eq. 11 subtracts m_i F_h; F_h < 0).
 * background: 0 = Eq. 9 with L = N_cut L_z, 1 = Eq. 10; rho0 == 0 disables. */
static void background_acc(double x, double y, double R, double Lhalf, double G,
                           double rho0, int background, double *bx, double *by)
{
    *bx = 0.0; *by = 0.0;
    if (rho0 == 0.0) return;
    double rho = sqrt(x * x + y * y);
    if (rho == 0.0) return;
    double Fh = background ? oracle_Fh_inf(rho, G, rho0) : oracle_Fh(rho, R, Lhalf, G, rho0);
    *bx = -Fh * x / rho;
    *by = -Fh * y / rho;
}

void oracle_background(int64_t n, const double *x, const double *y, double R, double Lhalf,
                       double G, double rho0, int background, double *bx, double *by)
{
    #pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i)
        background_acc(x[i], y[i], R, Lhalf, G, rho0, background, &bx[i], &by[i]);
}

/* One KDK leapfrog step of Eq. 11 in cosmic time t, DESIGN.md
 * reading S4 / G5:
 *   kick1 : v <- v + (dt/2) [ (g + b)/a_n^3 - 2 H_n v ]
 *   drift : x <- x + v dt ;  z reduced to [0, L)
 *   force : g', b' at the new positions
 *   kick2 : v <- [ v + (dt/2) (g' + b')/a_{n+1}^3 ] / (1 + H_{n+1} dt)
 * g[] holds g(x_n) on entry and g(x_{n+1}) on return (pair sum of Eq. 8 only). */
int oracle_kdk_step(int64_t n, double *x, double *y, double *z,
                    double *vx, double *vy, double *vz,
                    const double *m, const double *h,
                    double *gx, double *gy, double *gz,
                    double L, double G, int ncut,
                    double R, double rho0, int background,
                    double a_n, double H_n, double a_np1, double H_np1, double dt,
                    int nthreads)
{
    double Lhalf = (double)ncut * L;
    double ia3 = 1.0 / (a_n * a_n * a_n);
    for (int64_t i = 0; i < n; ++i) {
        double bx, by;
        background_acc(x[i], y[i], R, Lhalf, G, rho0, background, &bx, &by);
        vx[i] = vx[i] + 0.5 * dt * ((gx[i] + bx) * ia3 - 2.0 * H_n * vx[i]);
        vy[i] = vy[i] + 0.5 * dt * ((gy[i] + by) * ia3 - 2.0 * H_n * vy[i]);
        vz[i] = vz[i] + 0.5 * dt * (gz[i] * ia3 - 2.0 * H_n * vz[i]);
        x[i] = x[i] + vx[i] * dt;
        y[i] = y[i] + vy[i] * dt;
        z[i] = z[i] + vz[i] * dt;
        z[i] = z[i] - L * floor(z[i] / L);
        if (z[i] >= L) z[i] -= L;
    }
    int rc = oracle_accel(n, x, y, z, m, h, L, G, ncut, n, NULL, gx, gy, gz, nthreads);
    if (rc) return rc;
    ia3 = 1.0 / (a_np1 * a_np1 * a_np1);
    for (int64_t i = 0; i < n; ++i) {
        double bx, by;
        background_acc(x[i], y[i], R, Lhalf, G, rho0, background, &bx, &by);
        vx[i] = (vx[i] + 0.5 * dt * (gx[i] + bx) * ia3) / (1.0 + H_np1 * dt);
        vy[i] = (vy[i] + 0.5 * dt * (gy[i] + by) * ia3) / (1.0 + H_np1 * dt);
        vz[i] = (vz[i] + 0.5 * dt * gz[i] * ia3) / (1.0 + H_np1 * dt);
    }
    return 0;
}
