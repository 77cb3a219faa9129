// ewald_table.h -- host-side builder of the correction lookup table D(rho, z) of the
// EWALD_TABLE mode (Eq. 12-17).  Runs once per steps_cyl_init, O(nrho nz)
// work, no device code.
//
// D = F_{S1xR2} - F_{R3}: Ewald sum of the one-axis-periodic unit point mass minus the unsoftened
// nearest-image Newtonian force, per unit G m_i m_j, on the grid rho_i = i rho_max/(nrho-1),
// z_j = j (L/2)/(nz-1); stored interleaved {D_rho, D_z} (one 16-byte load per node).
//   real space   Eq. 13 as printed, images n = -nmax..nmax, the n = 0 image merged analytically
//                with -F_R3 so that nothing singular is left at r = 0;
//   Fourier      Eq. 14 with the kernel of DESIGN.md reading G4,
//                E(k, rho) = int_{1/(4 alpha^2)}^inf t^-1 exp(-rho^2/(4t) - k^2 t) dt,
//                F_z = -(2/L) sum_m k_m sin(k_m z) E,   F_rho = (2/L) sum_m cos(k_m z) dE/drho;
//                E and dE/drho depend on (m, rho) only and are integrated once per radial node by a
//                double-exponential rule for the half line;
//   m = 0        Eq. 16 as printed.
#pragma once
#include <cmath>
#include <vector>

namespace steps {

// J_p = int_{s0}^{inf} s^-p exp(-a/s - s) ds  (s = k^2 t, a = k^2 rho^2/4), p = 1, 2.
// Substitution s = s0 + exp(t - exp(-t)) (double-exponential rule for exponentially decaying
// integrands on a half line), trapezoid in t.
inline void ewald_J(double a, double s0, double &J1, double &J2)
{
    const double ht = 1.0 / 32.0;
    double j1 = 0.0, j2 = 0.0;
    for (int i = -160; i <= 224; ++i) {            // t in [-5, 7]: s - s0 from 1e-66 to ~1100
        const double t = i * ht, em = std::exp(-t);
        const double x = std::exp(t - em);
        const double s = s0 + x;
        const double wgt = ht * (1.0 + em) * x;
        const double f = std::exp(-a / s - s) / s;
        j1 += wgt * f;
        j2 += wgt * f / s;
    }
    J1 = j1;
    J2 = j2;
}

// [erf(x) - (2/sqrt(pi)) x exp(-x^2)] / r^3 with x = alpha r: what is left of the n = 0 image of
// Eq. 13 after the bare 1/r^2 force has been taken out.
inline double ewald_core(double alpha, double r)
{
    const double c = 1.1283791670955125739;        // 2/sqrt(pi)
    const double x = alpha * r;
    if (x < 0.25) {
        // c alpha^3 (2/3 - 2/5 x^2 + 1/7 x^4 - 1/27 x^6 + ...), coefficient 2k / ((2k+1) k!)
        const double x2 = x * x;
        double sum = 0.0, pw = 1.0, fact = 1.0;
        for (int k = 1; k <= 14; ++k) {
            fact *= k;
            const double ck = 2.0 * k / ((2.0 * k + 1.0) * fact);
            sum += (k % 2 ? ck : -ck) * pw;
            pw *= x2;
        }
        return c * alpha * alpha * alpha * sum;
    }
    return (std::erf(x) - c * x * std::exp(-x * x)) / (r * r * r);
}

inline void build_ewald_table(double L, double alpha, int nmax, int mmax, int nrho, int nz,
                              double rho_max, double *D /* [nrho*nz*2] */)
{
    const double pi = 3.14159265358979323846, c = 1.1283791670955125739;
    std::vector<double> E(mmax + 1), dE(mmax + 1);
    for (int i = 0; i < nrho; ++i) {
        const double rho = rho_max * i / (nrho - 1);
        for (int m = 1; m <= mmax; ++m) {
            const double k = 2.0 * pi * m / L;
            double J1, J2;
            ewald_J(0.25 * k * k * rho * rho, k * k / (4.0 * alpha * alpha), J1, J2);
            E[m] = J1;
            dE[m] = -0.5 * k * k * rho * J2;
        }
        const double ar = alpha * rho;
        const double line = (rho > 0.0) ? (ar < 1e-4 ? alpha * alpha * rho : -std::expm1(-ar * ar) / rho) : 0.0;
        for (int j = 0; j < nz; ++j) {
            const double z = 0.5 * L * j / (nz - 1);
            const double core = ewald_core(alpha, std::sqrt(rho * rho + z * z));
            double Fr = rho * core, Fz = z * core;
            for (int n = 1; n <= nmax; ++n) {
                for (int sg = -1; sg <= 1; sg += 2) {
                    const double dz = z + sg * n * L;
                    const double r2 = rho * rho + dz * dz, r = std::sqrt(r2);
                    const double br = (std::erfc(alpha * r) + c * alpha * r * std::exp(-alpha * alpha * r2)) / (r2 * r);
                    Fr -= rho * br;
                    Fz -= dz * br;
                }
            }
            for (int m = 1; m <= mmax; ++m) {
                const double k = 2.0 * pi * m / L;
                Fr += 2.0 / L * std::cos(k * z) * dE[m];
                Fz -= 2.0 / L * k * std::sin(k * z) * E[m];
            }
            Fr -= 2.0 / L * line;
            D[((size_t)i * nz + j) * 2 + 0] = Fr;
            D[((size_t)i * nz + j) * 2 + 1] = Fz;
        }
    }
}

}  // namespace steps
