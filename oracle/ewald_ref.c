/*
 * ewald_ref.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.  Validation-only companions of
 * rbe_oracle.c: the full (deterministic) Ewald sum of the paper and a brute-force periodic
 * image sum.  They exist to pin rbe_oracle.c to something other than itself; the RBE hot path
 * never needs them.  "P:nnn" = /root/reference/PAPER.md line nnn.  fp64 throughout, positions
 * and charges are double arrays (small N only: everything here is O(N^2 * cells)).
 *
 * Pins (tests/test_oracle_ewald.py): the rock-salt Madelung constant 1.7475645946 for several
 * alpha (Eq. 2.8 constants and the alpha-independence of the total), central finite
 * differences (forces = -grad of Eq. 2.8), and oracle_direct_image_sum + dipole term.
 */
#include <math.h>
#include <stdint.h>

#define PI 3.14159265358979323846264338327950288

/* ---------------------------------------------------------------------------------------
 * Full Ewald sum, Eq. (2.8) P:112 and its forces Eqs. (2.10)-(2.11) P:122-125.
 *
 *   U_real = 1/2 sum_{i,j} sum'_n q_i q_j erfc(sqrt(alpha) |r_ij + nL|) / |r_ij + nL|
 *   U_k    = (2 pi / V) sum_{k != 0} |rho(k)|^2 exp(-k^2/4alpha) / k^2,  k = 2 pi m / L
 *   U_self = - sqrt(alpha/pi) sum_i q_i^2
 *   F_i^short = - q_i sum'_{j,n} q_j ( erfc(sqrt(alpha) r)/r^2
 *                 + 2 sqrt(alpha) exp(-alpha r^2)/(sqrt(pi) r) ) (r_ij + nL)/|r_ij + nL|
 *   F_i^long  = - sum_{k != 0} (4 pi q_i k / (V k^2)) exp(-k^2/4alpha) Im(e^{-i k.r_i} rho(k))
 *
 * r_ij = r_j - r_i (the reading under which Eq. 2.10's leading minus sign makes like charges
 * repel; pinned by the finite-difference test).  The prime drops n = 0 when i = j.
 * Real-space images: all n with |n_d| <= nreal.  k grid: all m != 0 with |m_d| <= mmax.
 * Outputs: U[0..2] = {U_real, U_k, U_self}; Fs[3N] short-range force; Fl[3N] long-range.
 * ------------------------------------------------------------------------------------- */
void oracle_ewald_full(int32_t N, const double *r, const double *q, double L, double alpha,
                       int32_t nreal, int32_t mmax, double *U, double *Fs, double *Fl) {
    const double V = L * L * L;
    const double sa = sqrt(alpha);
    double Ureal = 0.0, Uk = 0.0, Uself = 0.0;
    for (int32_t i = 0; i < 3 * N; ++i) {
        Fs[i] = 0.0;
        Fl[i] = 0.0;
    }
    /* real space */
    for (int32_t i = 0; i < N; ++i)
        for (int32_t j = 0; j < N; ++j)
            for (int32_t a = -nreal; a <= nreal; ++a)
                for (int32_t b = -nreal; b <= nreal; ++b)
                    for (int32_t c = -nreal; c <= nreal; ++c) {
                        if (i == j && a == 0 && b == 0 && c == 0) continue;
                        double dx = r[3 * j + 0] - r[3 * i + 0] + a * L;
                        double dy = r[3 * j + 1] - r[3 * i + 1] + b * L;
                        double dz = r[3 * j + 2] - r[3 * i + 2] + c * L;
                        double d2 = dx * dx + dy * dy + dz * dz;
                        double d = sqrt(d2);
                        Ureal += 0.5 * q[i] * q[j] * erfc(sa * d) / d;
                        double g = erfc(sa * d) / d2 + 2.0 * sa * exp(-alpha * d2) / (sqrt(PI) * d);
                        Fs[3 * i + 0] += -q[i] * q[j] * g * dx / d;
                        Fs[3 * i + 1] += -q[i] * q[j] * g * dy / d;
                        Fs[3 * i + 2] += -q[i] * q[j] * g * dz / d;
                    }
    /* Fourier space */
    for (int32_t a = -mmax; a <= mmax; ++a)
        for (int32_t b = -mmax; b <= mmax; ++b)
            for (int32_t c = -mmax; c <= mmax; ++c) {
                if (a == 0 && b == 0 && c == 0) continue;
                double kx = 2.0 * PI * a / L, ky = 2.0 * PI * b / L, kz = 2.0 * PI * c / L;
                double k2 = kx * kx + ky * ky + kz * kz;
                double g = exp(-k2 / (4.0 * alpha));
                double re = 0.0, im = 0.0;
                for (int32_t j = 0; j < N; ++j) {
                    double ph = kx * r[3 * j] + ky * r[3 * j + 1] + kz * r[3 * j + 2];
                    re += q[j] * cos(ph);
                    im += q[j] * sin(ph);
                }
                Uk += 2.0 * PI / V * (re * re + im * im) * g / k2;
                for (int32_t i = 0; i < N; ++i) {
                    double ph = kx * r[3 * i] + ky * r[3 * i + 1] + kz * r[3 * i + 2];
                    double imag = cos(ph) * im - sin(ph) * re; /* Im(e^{-i ph} rho) */
                    double p = -4.0 * PI * q[i] / (V * k2) * g * imag;
                    Fl[3 * i + 0] += p * kx;
                    Fl[3 * i + 1] += p * ky;
                    Fl[3 * i + 2] += p * kz;
                }
            }
    for (int32_t i = 0; i < N; ++i) Uself += -sqrt(alpha / PI) * q[i] * q[i];
    U[0] = Ureal;
    U[1] = Uk;
    U[2] = Uself;
}

/* ---------------------------------------------------------------------------------------
 * Brute-force image sum of Eq. (2.5), truncated to the SPHERE of cells |n| <= R:
 *   U   = 1/2 sum_{i,j} sum'_{|n|<=R} q_i q_j / |r_ij + nL|
 *   F_i = q_i sum'_{j,|n|<=R} q_j (r_i - r_j - nL) / |r_i - r_j - nL|^3      (-grad_i U)
 * The series is conditionally convergent; summed over spheres it converges to the
 * vacuum-boundary value, which differs from Ewald's (tin-foil) by the dipole term
 * (2 pi / 3V)|M|^2, M = sum q_j r_j.  The test adds that term; it is not in the paper.
 * ------------------------------------------------------------------------------------- */
void oracle_direct_image_sum(int32_t N, const double *r, const double *q, double L, int32_t R,
                             double *U, double *F) {
    double u = 0.0;
    for (int32_t i = 0; i < 3 * N; ++i) F[i] = 0.0;
    for (int32_t a = -R; a <= R; ++a)
        for (int32_t b = -R; b <= R; ++b)
            for (int32_t c = -R; c <= R; ++c) {
                if (a * a + b * b + c * c > R * R) continue;
                for (int32_t i = 0; i < N; ++i)
                    for (int32_t j = 0; j < N; ++j) {
                        if (i == j && a == 0 && b == 0 && c == 0) continue;
                        double dx = r[3 * i + 0] - r[3 * j + 0] - a * L;
                        double dy = r[3 * i + 1] - r[3 * j + 1] - b * L;
                        double dz = r[3 * i + 2] - r[3 * j + 2] - c * L;
                        double d2 = dx * dx + dy * dy + dz * dz;
                        double d = sqrt(d2);
                        u += 0.5 * q[i] * q[j] / d;
                        double g = q[i] * q[j] / (d2 * d);
                        F[3 * i + 0] += g * dx;
                        F[3 * i + 1] += g * dy;
                        F[3 * i + 2] += g * dz;
                    }
            }
    *U = u;
}
