/*
 * short_range.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.  fp64 CPU oracle of the real-space
 * partner of the RBE force: the short-range part of the Ewald-split Coulomb force, Eq. (2.10)
 * P:122, truncated at the cutoff radius r_s as the paper prescribes ("determining a cutoff
 * radius and calculating the forces exerted by particles in the sphere of radius r_s centered on
 * particle i"), and the matching first term of Eq. (2.8) P:112.  "P:nnn" =
 * /root/reference/PAPER.md line nnn.
 *
 *   F_i = - q_i sum_{j != i, r < r_s} q_j ( erfc(sqrt(alpha) r)/r^2
 *            + 2 sqrt(alpha) exp(-alpha r^2)/(sqrt(pi) r) ) d / r
 *   e_i = 1/2 q_i sum_{j != i, r < r_s} q_j erfc(sqrt(alpha) r)/r          (sum_i e_i = U_short)
 *
 * with d = r_j - r_i folded to the nearest periodic image per component (reading Q5
 * for the direction of r_ij; reading Q18: r_s <= L/2, so at most one image of j lies inside
 * the sphere and the nearest-image fold finds it), r = |d|.  Coincident atoms (r = 0) are
 * skipped (the term is singular; the synthetic inputs do not contain any at r < r_s with both
 * charges non-zero except by construction in tests).
 *
 * Plain double loops over all pairs: O(nsel * N).  Inputs are the fp32 {x,y,z,q} records the
 * GPU sees, widened exactly.  OpenMP over the selected atoms only (each thread owns whole
 * atoms: the sum over j runs in index order, so the result does not depend on the thread count).
 * Shares no code with the CUDA path.  Pins: tests/test_oracle_short_range.py (against
 * oracle_ewald_full, itself pinned by the Madelung constant; the two-charge closed form;
 * Newton's third law; the cutoff rule by brute force).
 */
#include <math.h>
#include <stdint.h>

#define PI 3.14159265358979323846264338327950288

void oracle_short_range(int64_t N, const float *xyzq, double L, double alpha, double rs,
                        int64_t nsel, const int64_t *sel, double *F, double *e) {
    const double sa = sqrt(alpha);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t s = 0; s < nsel; ++s) {
        const int64_t i = sel ? sel[s] : s;
        const double xi = xyzq[4 * i], yi = xyzq[4 * i + 1], zi = xyzq[4 * i + 2], qi = xyzq[4 * i + 3];
        double fx = 0.0, fy = 0.0, fz = 0.0, en = 0.0;
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            double dx = (double)xyzq[4 * j] - xi, dy = (double)xyzq[4 * j + 1] - yi, dz = (double)xyzq[4 * j + 2] - zi;
            dx -= L * nearbyint(dx / L);   /* nearest image */
            dy -= L * nearbyint(dy / L);
            dz -= L * nearbyint(dz / L);
            const double r2 = dx * dx + dy * dy + dz * dz;
            if (!(r2 < rs * rs) || r2 == 0.0) continue;
            const double r = sqrt(r2), qj = xyzq[4 * j + 3];
            const double ec = erfc(sa * r);
            const double g = ec / r2 + 2.0 * sa * exp(-alpha * r2) / (sqrt(PI) * r);
            fx += -qi * qj * g * dx / r;
            fy += -qi * qj * g * dy / r;
            fz += -qi * qj * g * dz / r;
            en += 0.5 * qi * qj * ec / r;
        }
        F[3 * s] = fx; F[3 * s + 1] = fy; F[3 * s + 2] = fz;
        if (e) e[s] = en;
    }
}
