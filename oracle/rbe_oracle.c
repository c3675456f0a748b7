/*
 * rbe_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of what the random batch Ewald (RBE) k-space path
 * computes, written from /root/reference/PAPER.md (arxiv 2407.09315) so that a reader can
 * check it against the paper by eye.  "P:nnn" = PAPER.md line nnn.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call this file.  It shares no code with the CUDA path
 * (paper_2407_09315_b200/csrc) and neither includes the other.
 *
 * Parity pins (tests/test_oracle_*.py):
 *   oracle_ewald_full        -- NaCl Madelung constant (alpha-independent), finite differences
 *   oracle_direct_image_sum  -- used only as the independent side of the Ewald-force pin
 *   oracle_rho/force/energy  -- sum F = 0, two-charge closed form, pair form by brute force,
 *                               symmetries, unbiasedness towards oracle_ewald_full's k-space
 *                               force, closed-form 1/P variance
 *   oracle_S                 -- 3-D grid sum and Poisson-resummed closed form
 * Parity unpinned: nothing in this file.  (The paper's RDF/MSD-vs-LAMMPS curves, P:246-250,
 * are out of scope and therefore unpinned.)
 *
 * Units: Gaussian (Eq. 2.5, has no 1/4 pi eps0): charges e, lengths A, energy e^2/A,
 * force e^2/A^2.  alpha in A^-2 (erfc(sqrt(alpha) r)).
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC (no -ffast-math).  OpenMP only splits independent
 * outputs (one k or one atom per iteration); every sum runs in index order, so results do
 * not depend on the thread count.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

#define PI 3.14159265358979323846264338327950288

int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---------------------------------------------------------------------------------------
 * Normaliser  S = sum_{m in Z^3, m != 0} exp(-|k_m|^2 / 4 alpha),  k_m = 2 pi m / L.
 * P:129 ("Q is the normalization constant"), P:115 (k = 2 pi m / L).  The summand
 * factorises over the three components, so S = H^3 - 1 with
 * H = sum_{m in Z} exp(-pi^2 m^2 / (alpha L^2)); terms are added until they underflow.
 * ------------------------------------------------------------------------------------- */
double oracle_S(double L, double alpha) {
    double c = PI * PI / (alpha * L * L);
    double H = 1.0;
    for (int64_t m = 1;; ++m) {
        double t = exp(-c * (double)m * (double)m);
        if (t == 0.0 || t < 1e-300) break;
        H += 2.0 * t;
    }
    return H * H * H - 1.0;
}

/* Same S by the literal triple sum over |m_d| <= mmax (for the pin; O(mmax^3)). */
double oracle_S_grid(double L, double alpha, int mmax) {
    double c = PI * PI / (alpha * L * L);
    double s = 0.0;
    for (int a = -mmax; a <= mmax; ++a)
        for (int b = -mmax; b <= mmax; ++b)
            for (int d = -mmax; d <= mmax; ++d) {
                if (a == 0 && b == 0 && d == 0) continue;
                s += exp(-c * (double)(a * a + b * b + d * d));
            }
    return s;
}

/* ---------------------------------------------------------------------------------------
 * Structure factor, Eq. (2.9):   rho(k_l) = sum_j q_j exp(i k_l . r_j),
 * k_l = 2 pi m_l / L.  Inputs are the fp32 {x,y,z,q} records the GPU sees, widened
 * exactly to fp64; the phase is k.r in radians from the un-wrapped position.
 * rho[2l] = Re, rho[2l+1] = Im.
 * ------------------------------------------------------------------------------------- */
void oracle_rho(int64_t N, const float *xyzq, double L, int32_t P, const int32_t *m,
                double *rho) {
#pragma omp parallel for schedule(dynamic, 1)
    for (int32_t l = 0; l < P; ++l) {
        double kx = 2.0 * PI * (double)m[3 * l + 0] / L;
        double ky = 2.0 * PI * (double)m[3 * l + 1] / L;
        double kz = 2.0 * PI * (double)m[3 * l + 2] / L;
        double re = 0.0, im = 0.0;
        for (int64_t j = 0; j < N; ++j) {
            double x = (double)xyzq[4 * j + 0], y = (double)xyzq[4 * j + 1];
            double z = (double)xyzq[4 * j + 2], q = (double)xyzq[4 * j + 3];
            double ph = kx * x + ky * y + kz * z;
            re += q * cos(ph);
            im += q * sin(ph);
        }
        rho[2 * l + 0] = re;
        rho[2 * l + 1] = im;
    }
}

/* ---------------------------------------------------------------------------------------
 * RBE force, Eq. (2.12), P:131:
 *   F_i ~= - sum_{l=1..P} (Q/P) (4 pi q_i k_l / (V k_l^2)) Im( exp(-i k_l . r_i) rho(k_l) ),
 * Q == S, V = L^3.  Im(e^{-i phi} rho) = cos(phi) Im(rho) - sin(phi) Re(rho).
 * w == NULL: every sample carries Q/P = S/P (duplicates in the batch count separately,
 * DESIGN.md reading Q9).  w != NULL: w[l] replaces Q/P; with w[l] = exp(-k_l^2/4alpha) and
 * the k-set = every grid vector this is the exact long-range force of Eq. (2.11).
 *
 * Per-atom energy (reading Q7; the importance-sampled second term of Eq. (2.8),
 * P:112):  e_i = (2 pi q_i / V) sum_l w_l Re( exp(-i k_l . r_i) rho(k_l) ) / k_l^2,
 * so that sum_i e_i = U of oracle_energy.
 *
 * sel == NULL: atoms 0..nsel-1 (nsel == N for all); else the listed atom indices.
 * F[3 a + d], e[a] (e may be NULL) for the a-th selected atom.
 * ------------------------------------------------------------------------------------- */
void oracle_force(int64_t N, const float *xyzq, double L, int32_t P, const int32_t *m,
                  const double *w, double S, const double *rho, int64_t nsel,
                  const int64_t *sel, double *F, double *e) {
    const double V = L * L * L;
    (void)N;
#pragma omp parallel for schedule(static)
    for (int64_t a = 0; a < nsel; ++a) {
        int64_t i = sel ? sel[a] : a;
        double x = (double)xyzq[4 * i + 0], y = (double)xyzq[4 * i + 1];
        double z = (double)xyzq[4 * i + 2], q = (double)xyzq[4 * i + 3];
        double fx = 0.0, fy = 0.0, fz = 0.0, en = 0.0;
        for (int32_t l = 0; l < P; ++l) {
            double kx = 2.0 * PI * (double)m[3 * l + 0] / L;
            double ky = 2.0 * PI * (double)m[3 * l + 1] / L;
            double kz = 2.0 * PI * (double)m[3 * l + 2] / L;
            double k2 = kx * kx + ky * ky + kz * kz;
            double wl = w ? w[l] : S / (double)P;
            double ph = kx * x + ky * y + kz * z;
            double c = cos(ph), s = sin(ph);
            double im = c * rho[2 * l + 1] - s * rho[2 * l + 0]; /* Im(e^{-i ph} rho) */
            double re = c * rho[2 * l + 0] + s * rho[2 * l + 1]; /* Re(e^{-i ph} rho) */
            double pref = -wl * 4.0 * PI * q / (V * k2);
            fx += pref * kx * im;
            fy += pref * ky * im;
            fz += pref * kz * im;
            en += wl * 2.0 * PI * q / (V * k2) * re;
        }
        F[3 * a + 0] = fx;
        F[3 * a + 1] = fy;
        F[3 * a + 2] = fz;
        if (e) e[a] = en;
    }
}

/* ---------------------------------------------------------------------------------------
 * k-space energy estimate: second term of Eq. (2.8), P:112,
 *   (2 pi / V) sum_{k != 0} |rho(k)|^2 exp(-k^2/4alpha) / k^2,
 * importance-sampled with the same weights as the force (reading Q7):
 *   U = (2 pi / V) sum_l w_l |rho(k_l)|^2 / k_l^2,   w_l = S/P unless given.
 * ------------------------------------------------------------------------------------- */
double oracle_energy(double L, int32_t P, const int32_t *m, const double *w, double S,
                     const double *rho) {
    const double V = L * L * L;
    double U = 0.0;
    for (int32_t l = 0; l < P; ++l) {
        double kx = 2.0 * PI * (double)m[3 * l + 0] / L;
        double ky = 2.0 * PI * (double)m[3 * l + 1] / L;
        double kz = 2.0 * PI * (double)m[3 * l + 2] / L;
        double k2 = kx * kx + ky * ky + kz * kz;
        double wl = w ? w[l] : S / (double)P;
        double r2 = rho[2 * l] * rho[2 * l] + rho[2 * l + 1] * rho[2 * l + 1];
        U += wl * r2 / k2;
    }
    return 2.0 * PI / V * U;
}
