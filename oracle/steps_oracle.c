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

/* ================================================================== Sect. 2.2
 * Ewald summation in S^1 x R^2 and the correction lookup table (Eq. 12-17).
 * Unit source at the origin, target at radial separation rho >= 0 and axial separation z;
 * returns the force per unit (G m_i m_j): F[0] radial (negative = towards the axis of the
 * source), F[1] axial.
 *
 *   Eq. 13 (real space, as printed):
 *     F_real = - sum_{n=-nmax}^{nmax} r_n/|r_n|^3 [ erfc(alpha |r_n|) + (2 alpha/sqrt(pi)) |r_n| exp(-alpha^2 |r_n|^2) ],
 *     r_n = r + n L e_z
 *   Eq. 14-15 (Fourier space) -- DESIGN.md reading G4: the printed kernel B is that of the
 *   two-axis-periodic slab problem and does not reproduce the image sum.  For one periodic axis
 *   the two-dimensional Fourier integral of the Gaussian-filtered Green function is
 *     E(k, rho) = int_{1/(4 alpha^2)}^{inf} t^-1 exp(-rho^2/(4t) - k^2 t) dt   (-> 2 K_0(k rho), alpha -> inf)
 *     F_Fourier = + (2/L) sum_{m=1}^{mmax} grad[ cos(k_m z) E(k_m, rho) ],   k_m = 2 pi m / L
 *   Eq. 16 (m = 0 mode, as printed):  F_rho = -(2/(L rho)) (1 - exp(-alpha^2 rho^2)).
 * The integrals over t are done numerically (composite 20-point Gauss-Legendre in u = ln(k^2 t)). */

static const double GL20_X[10] = {
    0.0765265211334973337546404, 0.2277858511416450780804962, 0.3737060887154195606725482,
    0.5108670019508270980043641, 0.6360536807265150254528367, 0.7463319064601507926143051,
    0.8391169718222188233945291, 0.9122344282513259058677524, 0.9639719272779137912676661,
    0.9931285991850949247861224};
static const double GL20_W[10] = {
    0.1527533871307258506980843, 0.1491729864726037467878287, 0.1420961093183820513292983,
    0.1316886384491766268984945, 0.1181945319615184173123774, 0.1019301198172404350367501,
    0.0832767415767047487247581, 0.0626720483341090635695065, 0.0406014298003869413310400,
    0.0176140071391521183118620};

/* I_p(a, s0) = int_{s0}^{inf} s^-p exp(-a/s - s) ds,  p = 1 or 2  (s = k^2 t, a = k^2 rho^2 / 4) */
static double ewald_Ip(int p, double a, double s0)
{
    /* in u = ln s:  int exp(-a e^-u - e^u) e^{(1-p) u} du; the integrand is < 1e-300 beyond
     * s = 700; panels of width 0.25 in u */
    double u0 = log(s0), u1 = log(s0 + 700.0 + 2.0 * sqrt(a));
    int np = (int)ceil((u1 - u0) / 0.25);
    double hp = (u1 - u0) / np, sum = 0.0;
    for (int i = 0; i < np; ++i) {
        double c = u0 + (i + 0.5) * hp, hw = 0.5 * hp;
        for (int q = 0; q < 10; ++q) {
            for (int sg = -1; sg <= 1; sg += 2) {
                double u = c + sg * hw * GL20_X[q];
                double s = exp(u);
                sum += hw * GL20_W[q] * exp(-a / s - s + (1.0 - p) * u);
            }
        }
    }
    return sum;
}

void oracle_ewald_force(double rho, double z, double L, double alpha, int nmax, int mmax,
                        double F[2])
{
    const double pi = 3.14159265358979323846, two_over_sqrtpi = 1.12837916709551257390;
    double Fr = 0.0, Fz = 0.0;
    /* Eq. 13 */
    for (int n = -nmax; n <= nmax; ++n) {
        double dz = z + (double)n * L;
        double r = sqrt(rho * rho + dz * dz);
        if (r == 0.0) continue;
        double br = erfc(alpha * r) + two_over_sqrtpi * alpha * r * exp(-alpha * alpha * r * r);
        Fr += -rho / (r * r * r) * br;
        Fz += -dz / (r * r * r) * br;
    }
    /* Eq. 14-15 (reading G4) */
    for (int m = 1; m <= mmax; ++m) {
        double k = 2.0 * pi * (double)m / L;
        double s0 = k * k / (4.0 * alpha * alpha), a = 0.25 * k * k * rho * rho;
        double E = ewald_Ip(1, a, s0);
        double dE = -0.5 * k * k * rho * ewald_Ip(2, a, s0);        /* dE/drho */
        Fr += 2.0 / L * cos(k * z) * dE;
        Fz += -2.0 / L * k * sin(k * z) * E;
    }
    /* Eq. 16 */
    if (rho > 0.0) Fr += -2.0 / (L * rho) * (1.0 - exp(-alpha * alpha * rho * rho));
    F[0] = Fr; F[1] = Fz;
}

/* Eq. 17: D(rho, z) = F_{S1xR2}(rho, z) - F_{R3}(rho, z) on an equally spaced grid,
 * rho_i = i rho_max/(nrho-1), z_j = j (L/2)/(nz-1)  (reading T1: the paper gives the
 * grid size 144 x 128, not its extent or which axis is which).  F_R3 is the unsoftened
 * nearest-image Newtonian force -r/|r|^3.  The n = 0 term of Eq. 13 and F_R3 are combined
 * analytically, -r/r^3 [erfc(x) + 2x/sqrt(pi) e^{-x^2} - 1] = + r/r^3 [erf(x) - 2x/sqrt(pi) e^{-x^2}],
 * x = alpha r, with its Taylor series for small x, so that D is finite at r = 0.
 * Layout: D[(i*nz + j)*2 + c], c = 0 radial, 1 axial. */
static double ewald_near_factor(double alpha, double r)
{
    /* [erf(x) - (2/sqrt(pi)) x exp(-x^2)] / r^3 */
    const double two_over_sqrtpi = 1.12837916709551257390;
    double x = alpha * r;
    if (x < 0.2) {
        /* (2/sqrt(pi)) alpha^3 sum_{k>=1} (-1)^{k+1} 2k/((2k+1) k!) x^{2k-2} */
        double x2 = x * x, term = 1.0, sum = 0.0, fact = 1.0;
        for (int k = 1; k <= 12; ++k) {
            fact *= (double)k;
            double ck = 2.0 * k / ((2.0 * k + 1.0) * fact);
            sum += ((k & 1) ? 1.0 : -1.0) * ck * term;
            term *= x2;
        }
        return two_over_sqrtpi * alpha * alpha * alpha * sum;
    }
    return (erf(x) - two_over_sqrtpi * x * exp(-x * x)) / (r * r * r);
}

void oracle_ewald_D(double rho, double z, double L, double alpha, int nmax, int mmax, double D[2])
{
    /* full Ewald force minus nearest image, with the n = 0 real-space term replaced by the
     * combined form above; z must lie in [-L/2, L/2] */
    const double pi = 3.14159265358979323846, two_over_sqrtpi = 1.12837916709551257390;
    double Fr = 0.0, Fz = 0.0;
    double r0 = sqrt(rho * rho + z * z);
    double nf = ewald_near_factor(alpha, r0);
    Fr += rho * nf;
    Fz += z * nf;
    for (int n = -nmax; n <= nmax; ++n) {
        if (n == 0) continue;
        double dz = z + (double)n * L;
        double r = sqrt(rho * rho + dz * dz);
        double br = erfc(alpha * r) + two_over_sqrtpi * alpha * r * exp(-alpha * alpha * r * r);
        Fr += -rho / (r * r * r) * br;
        Fz += -dz / (r * r * r) * br;
    }
    for (int m = 1; m <= mmax; ++m) {
        double k = 2.0 * pi * (double)m / L;
        double s0 = k * k / (4.0 * alpha * alpha), a = 0.25 * k * k * rho * rho;
        Fr += 2.0 / L * cos(k * z) * (-0.5 * k * k * rho * ewald_Ip(2, a, s0));
        Fz += -2.0 / L * k * sin(k * z) * ewald_Ip(1, a, s0);
    }
    if (rho > 0.0) {
        double x = alpha * rho;
        /* (1 - exp(-x^2))/rho, series-safe */
        Fr += -2.0 / L * (x < 1e-4 ? alpha * alpha * rho : -expm1(-x * x) / rho);
    }
    D[0] = Fr; D[1] = Fz;
}

void oracle_ewald_table(double L, double alpha, int nmax, int mmax, int nrho, int nz,
                        double rho_max, double *D)
{
    #pragma omp parallel for schedule(dynamic, 1)
    for (int i = 0; i < nrho; ++i) {
        double rho = rho_max * (double)i / (double)(nrho - 1);
        for (int j = 0; j < nz; ++j) {
            double z = 0.5 * L * (double)j / (double)(nz - 1);
            oracle_ewald_D(rho, z, L, alpha, nmax, mmax, &D[((size_t)i * nz + j) * 2]);
        }
    }
}

/* Table value with the symmetries of D used as boundary rules (reading T3):
 * D_rho is odd in rho and even in z, D_z is even in rho and odd in z; both are periodic in z,
 * so about z = L/2 D_rho is even and D_z odd.  Beyond the last radial node the last node is
 * used.  c = 0 radial, 1 axial. */
static double table_get(const double *D, int nrho, int nz, int i, int j, int c)
{
    double sgn = 1.0;
    if (i < 0) { i = -i; if (c == 0) sgn = -sgn; }
    if (i > nrho - 1) i = nrho - 1;
    if (j < 0) { j = -j; if (c == 1) sgn = -sgn; }
    if (j > nz - 1) { j = 2 * (nz - 1) - j; if (c == 1) sgn = -sgn; }
    return sgn * D[((size_t)i * nz + j) * 2 + c];
}

/* Interpolated D at (rho, az), az = |z| in [0, L/2]: interp 0 = cloud-in-cell (bilinear),
 * 1 = triangular-shaped-cloud (quadratic B-spline weights on the 3x3 nearest nodes),
 * PAPER.md:164. */
void oracle_table_interp(const double *D, int nrho, int nz, double rho_max, double L,
                         int interp, double rho, double az, double out[2])
{
    double xr = rho / (rho_max / (double)(nrho - 1));
    double xz = az / (0.5 * L / (double)(nz - 1));
    out[0] = out[1] = 0.0;
    if (interp == 0) {
        int i0 = (int)floor(xr), j0 = (int)floor(xz);
        double fr = xr - i0, fz = xz - j0;
        double wr[2] = {1.0 - fr, fr}, wz[2] = {1.0 - fz, fz};
        for (int a = 0; a < 2; ++a)
            for (int b = 0; b < 2; ++b)
                for (int c = 0; c < 2; ++c)
                    out[c] += wr[a] * wz[b] * table_get(D, nrho, nz, i0 + a, j0 + b, c);
    } else {
        int ic = (int)floor(xr + 0.5), jc = (int)floor(xz + 0.5);
        double dr = xr - ic, dz = xz - jc;
        double wr[3] = {0.5 * (0.5 - dr) * (0.5 - dr), 0.75 - dr * dr, 0.5 * (0.5 + dr) * (0.5 + dr)};
        double wz[3] = {0.5 * (0.5 - dz) * (0.5 - dz), 0.75 - dz * dz, 0.5 * (0.5 + dz) * (0.5 + dz)};
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b)
                for (int c = 0; c < 2; ++c)
                    out[c] += wr[a] * wz[b] * table_get(D, nrho, nz, ic - 1 + a, jc - 1 + b, c);
    }
}

/* Pair sum in EWALD_TABLE mode (Eq. 7-style use of the table):
 *   F(r, h) = F_R3(nearest image, spline-softened, Eq. 3/4) + D(rho, z)        rho < rho_max
 *           = -2 G/(L rho) e_rho  (the line-mass term, Eq. 16 with alpha -> inf) rho >= rho_max
 * (reading T2: the paper does not say what happens beyond the table).
 * D is the table built with G = 1.  Same conventions as oracle_accel. */
int oracle_accel_table(int64_t n, const double *x, const double *y, const double *z,
                       const double *m, const double *h, double L, double G,
                       const double *D, int nrho, int nz, double rho_max, int interp,
                       int64_t nt, const int64_t *targets,
                       double *gx, double *gy, double *gz, int nthreads)
{
    if (n < 1 || L <= 0.0 || !D || nrho < 2 || nz < 2 || rho_max <= 0.0) return -1;
    if (!targets) nt = n;
    double *zw = (double *)malloc((size_t)n * sizeof(double));
    if (!zw) return -1;
    for (int64_t j = 0; j < n; ++j) {
        zw[j] = z[j] - L * floor(z[j] / L);
        if (zw[j] >= L) zw[j] -= L;
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
            double rx = x[i] - x[j], ry = y[i] - y[j], rz = zw[i] - zw[j];
            rz = rz - L * rint(rz / L);
            double rho = sqrt(rx * rx + ry * ry);
            double f[3];
            if (rho < rho_max) {
                double s = sqrt(rx * rx + ry * ry + rz * rz);
                double w = (s == 0.0) ? 0.0 : oracle_spline_F(s, h[i] + h[j]) / s;
                double Dv[2];
                oracle_table_interp(D, nrho, nz, rho_max, L, interp, rho, fabs(rz), Dv);
                double dr = (rho == 0.0) ? 0.0 : Dv[0] / rho;
                f[0] = -w * rx + dr * rx;
                f[1] = -w * ry + dr * ry;
                f[2] = -w * rz + (rz < 0.0 ? -Dv[1] : Dv[1]);
            } else {
                double c = -2.0 / (L * rho * rho);
                f[0] = c * rx; f[1] = c * ry; f[2] = 0.0;
            }
            acc[0] += (long double)(G * m[j] * f[0]);
            acc[1] += (long double)(G * m[j] * f[1]);
            acc[2] += (long double)(G * m[j] * f[2]);
        }
        gx[t] = (double)acc[0]; gy[t] = (double)acc[1]; gz[t] = (double)acc[2];
    }
    free(zw);
    return 0;
}

/* ------------------------------------------------------------- Eq. 18-20
 * Friedmann equation with CPL dark energy, PAPER.md:168-183:
 *   H^2 = H0^2 [ Or a^-4 + Om a^-3 + Ok a^-2 + O_DE(a) ],
 *   O_DE(a) = O_DE0 exp[ -3 int_1^a (1 + w(a'))/a' da' ]   (Eq. 19),   w(a) = w0 + wa (1 - a)   (Eq. 20).
 * The integral of Eq. 19 is done numerically as printed (composite 20-point Gauss-Legendre in
 * ln a'); tests pin it to the closed form and to the constant-w power law. */
double oracle_omega_de(double a, double ODE, double w0, double wa)
{
    double u1 = log(a);                       /* int_1^a (1+w)/a' da' = int_0^{ln a} (1 + w(e^u)) du */
    int np = 8;
    double hp = u1 / np, sum = 0.0;
    for (int i = 0; i < np; ++i) {
        double c = (i + 0.5) * hp, hw = 0.5 * hp;
        for (int q = 0; q < 10; ++q)
            for (int sg = -1; sg <= 1; sg += 2) {
                double u = c + sg * hw * GL20_X[q];
                sum += hw * GL20_W[q] * (1.0 + w0 + wa * (1.0 - exp(u)));
            }
    }
    return ODE * exp(-3.0 * sum);
}

double oracle_hubble_cpl(double a, double H0, double Om, double Or, double Ok, double ODE,
                         double w0, double wa)
{
    return H0 * sqrt(Or / (a * a * a * a) + Om / (a * a * a) + Ok / (a * a)
                     + oracle_omega_de(a, ODE, w0, wa));
}

void oracle_friedmann_rk4_cpl(double a, double dt, double H0, double Om, double Or, double Ok,
                              double ODE, double w0, double wa, double *a_next, double *H_next)
{
    double k1 = a * oracle_hubble_cpl(a, H0, Om, Or, Ok, ODE, w0, wa);
    double a2 = a + 0.5 * dt * k1;
    double k2 = a2 * oracle_hubble_cpl(a2, H0, Om, Or, Ok, ODE, w0, wa);
    double a3 = a + 0.5 * dt * k2;
    double k3 = a3 * oracle_hubble_cpl(a3, H0, Om, Or, Ok, ODE, w0, wa);
    double a4 = a + dt * k3;
    double k4 = a4 * oracle_hubble_cpl(a4, H0, Om, Or, Ok, ODE, w0, wa);
    double an = a + dt * (k1 + 2.0 * k2 + 2.0 * k3 + k4) / 6.0;
    *a_next = an;
    *H_next = oracle_hubble_cpl(an, H0, Om, Or, Ok, ODE, w0, wa);
}
