// sr_pair_kernels.cuh -- the force kernel of the real-space partner (Eq. 2.10 P:122 truncated at r_s,
// P:127), second design: every unordered pair is evaluated ONCE (Newton's third law) and whole
// 32 x 32 blocks of pairs are skipped by a bounding-box test, yet the result stays bitwise
// reproducible.  (First design, sr_kernels.cuh::sr_force_kernel: a thread per atom against all 27
// neighbour cells, every ordered pair tested: 2 900 cutoff tests per atom at r_s = 10 A.)
//
// Work unit.  The atoms are sorted by cell and, inside a cell, by a Morton code of sub-cells
// (sr_sort_kernel), so a GROUP = 32 consecutive atoms of one cell is spatially compact; its bounding
// box comes from sr_gbox_kernel.  A warp owns one group I of cell c (a lane = an atom, coordinates in
// fp32 Angstrom relative to the centre of c, nearest image implicit in the wrapped integer
// difference) and meets the groups J of the 13 "forward" neighbour cells, and of its own cell with
// J >= I, so that every unordered pair of groups is met exactly once.  Blocks whose boxes are
// farther apart than r_s are skipped (about half of them).  For a surviving block the J atoms and
// their accumulators sit in shared memory; in step t lane l handles the pair (l, (l + t) mod 32):
// all lanes touch different J atoms, so both sides of a pair are accumulated without atomics and in
// a fixed order.
//
// Combining contributions that come from different warps.  A group receives partial forces from
// ~20 other warps.  They are added in 64-bit FIXED POINT with integer atomics: integer addition is
// associative, so the sum does not depend on the order in which the warps arrive -- no
// floating-point atomics anywhere.  Scale 2^40 per e/A^2 of F_i / q_i (resolution 9e-13, range +-8.4e6:
// two unit charges closer than 3.5e-4 A would overflow; contributions below the resolution are lost).
// sr_finalize_kernel converts back to fp32, applies -q_i and scatters to the caller's atom order.
#pragma once
#include "sr_kernels.cuh"

namespace rbe {

constexpr int SR_GMAX = 8;                       // groups per cell that carry a bounding box (more: never skipped)
constexpr double SR_FIXED_SCALE = 1099511627776.0; // 2^40

struct SrPairParams {
    const uint4* sorted;      // [N] {Sx, Sy, Sz, q} in cell order
    const uint32_t* start;    // [ncell + 1]
    const float* gbox;        // [ncell][SR_GMAX][6] {lo xyz, hi xyz} of a group, A, relative to its cell's centre
    long long* acc;           // [N][4] fixed-point {A_x, A_y, A_z, E}, sorted order, zeroed before the launch
    int32_t nc;
    float len_unit;           // L / 2^32 [A]
    float cell_len;           // L / nc [A]
    float rs2;                // r_s^2 [A^2]
    float sqrt_alpha;
    float nalpha_log2e;       // -alpha log2(e)
    float tab_umin;           // below this r^2 the analytic branch is taken [A^2]
    const float4* tab_f;      // [ntab] cubic coefficients of T_f per interval (sr_table_kernel)
    const float4* tab_e;      // [ntab] ... of T_e
    int32_t ntab;
};

__device__ __forceinline__ uint32_t sr_cell_centre(int cd, int nc) {
    return (uint32_t)((((unsigned long long)(2 * cd + 1)) << 31) / (unsigned)nc);   // (2 c + 1) / (2 nc) of a turn
}

// Bounding boxes of the first SR_GMAX groups of every cell.  One warp per cell.
__global__ void __launch_bounds__(256) sr_gbox_kernel(const uint4* __restrict__ sorted, const uint32_t* __restrict__ start,
                                                       int ncell, int nc, float len_unit, float* __restrict__ gbox) {
    const int c = (int)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (c >= ncell) return;
    const uint32_t s0 = start[c], n = start[c + 1] - s0;
    const uint32_t ox = sr_cell_centre(c % nc, nc), oy = sr_cell_centre((c / nc) % nc, nc), oz = sr_cell_centre(c / (nc * nc), nc);
    for (int g = 0; g < SR_GMAX && (uint32_t)(32 * g) < n; ++g) {
        const uint32_t e = 32u * g + lane;
        float lo[3] = {3.0e38f, 3.0e38f, 3.0e38f}, hi[3] = {-3.0e38f, -3.0e38f, -3.0e38f};
        if (e < n) {
            const float4 a = sr_relative(sorted[s0 + e], ox, oy, oz, len_unit);
            lo[0] = hi[0] = a.x; lo[1] = hi[1] = a.y; lo[2] = hi[2] = a.z;
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1)
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                lo[k] = fminf(lo[k], __shfl_xor_sync(FULL_MASK, lo[k], d));
                hi[k] = fmaxf(hi[k], __shfl_xor_sync(FULL_MASK, hi[k], d));
            }
        if (lane < 6) gbox[((int64_t)c * SR_GMAX + g) * 6 + lane] = lane < 3 ? lo[lane] : hi[lane - 3];
    }
}

__device__ __forceinline__ void sr_atomic_add_fixed(long long* p, float v) {
    atomicAdd(reinterpret_cast<unsigned long long*>(p), (unsigned long long)__double2ll_rn((double)v * SR_FIXED_SCALE));
}

// ---------------------------------------------------------------------------------------
// The pair-term table (PAPER.md: tabulated erfc / exp with interpolation above a small radius, the series
// below it).  Tabulated over u = r^2, so no square root is needed:
//   T_f(u) = e^{alpha u} g(r) / r = [erfcx(sqrt(alpha u)) / sqrt(u) + 2 sqrt(alpha / pi)] / u      (force, Eq. 2.10)
//   T_e(u) = e^{alpha u} erfc(sqrt(alpha) r) / r = erfcx(sqrt(alpha u)) / sqrt(u)                  (energy, Eq. 2.8)
// The Gaussian is factored out (one MUFU.EX2 per pair) so that what is tabulated behaves like a power of u at any
// alpha r_s^2, and intervals of constant RELATIVE width keep a constant relative error: interval i covers
// u in 2^e (1 + m / 32) + [0, 2^e / 32), e = SR_TAB_EMIN + i / 32, m = i % 32 -- the index is the top bits of the fp32
// pattern of u, the interval origin is u with the low mantissa bits cleared.  Per interval a cubic in (u - origin)
// through the four Chebyshev nodes (fp64, erfcx(x) = e^{x^2} erfc(x)); its interpolation error is
// <= 2e-7 relative.  Pairs closer than 2^(EMIN / 2) = 0.125 A take the analytic branch.
// ---------------------------------------------------------------------------------------
constexpr int SR_TAB_EMIN = -6;          // the table starts at u = 2^-6 A^2 (r = 0.125 A)
constexpr int SR_TAB_BITS = 5;           // 32 intervals per octave of u
constexpr int SR_TAB_MAX = 1024;         // entries per table the workspace holds (32 octaves)

// Interval i of the table: its cubic coefficients for T_f (tf) and T_e (te).  Host and device run the same code
// (rbe_pair_table_host returns the host's copy, which the CPU tests check against the closed forms).
__host__ __device__ inline void sr_table_entry(int i, double alpha, float4& tf, float4& te) {
    const double base = ldexp(1.0, SR_TAB_EMIN + (i >> SR_TAB_BITS));
    const double h = base / (1 << SR_TAB_BITS), u0 = base + h * (i & ((1 << SR_TAB_BITS) - 1));
    const double sa = sqrt(alpha), c = 2.0 * sa / sqrt(PI_D);
    double tau[4], ff[4], fe[4];
    for (int k = 0; k < 4; ++k) {
        tau[k] = 0.5 * (1.0 - cos((2 * k + 1) * PI_D / 8.0));      // Chebyshev nodes of [0, 1]
        const double u = u0 + h * tau[k], r = sqrt(u), x = sa * r;
        const double x2 = x * x;                                    // erfcx(x) = e^{x^2} erfc(x); its asymptotic series where e^{x^2} would overflow
        const double ecx = x2 < 600.0 ? exp(x2) * erfc(x) : (1.0 - 0.5 / x2 + 0.75 / (x2 * x2)) / (x * sqrt(PI_D));
        const double ex = ecx / r;
        fe[k] = ex;
        ff[k] = (ex + c) / u;
    }
    for (int which = 0; which < 2; ++which) {
        const double* f = which ? fe : ff;
        // Newton divided differences
        double d[4] = {f[0], f[1], f[2], f[3]};
        for (int lev = 1; lev < 4; ++lev)
            for (int k = 3; k >= lev; --k) d[k] = (d[k] - d[k - 1]) / (tau[k] - tau[k - lev]);
        // Newton form d0 + d1 (t - t0) + d2 (t - t0)(t - t1) + d3 (t - t0)(t - t1)(t - t2), expanded to monomials in tau
        const double t0 = tau[0], t1 = tau[1], t2 = tau[2];
        const double b0 = d[0] - d[1] * t0 + d[2] * t0 * t1 - d[3] * t0 * t1 * t2;
        const double b1 = d[1] - d[2] * (t0 + t1) + d[3] * (t0 * t1 + t0 * t2 + t1 * t2);
        const double b2 = d[2] - d[3] * (t0 + t1 + t2);
        const double b3 = d[3];
        const float4 o = make_float4((float)b0, (float)(b1 / h), (float)(b2 / (h * h)), (float)(b3 / (h * h * h)));
        if (which) te = o; else tf = o;
    }
}

__global__ void __launch_bounds__(128) sr_table_kernel(float4* __restrict__ tf, float4* __restrict__ te, int n, double alpha) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float4 f, e;
    sr_table_entry(i, alpha, f, e);
    tf[i] = f;
    te[i] = e;
}

// dynamic shared memory of the pair kernel: the table(s), when that variant runs (rbe_set_pair_table)
__host__ __device__ constexpr size_t sr_pair_smem_bytes(int ntab, bool table, bool energy) {
    return table ? (size_t)ntab * sizeof(float4) * (energy ? 2 : 1) : 0;
}

constexpr int SR_PAIR_WARPS = 4;   // warps per CTA
constexpr int SR_PAIR_CTAS = 9;    // resident CTAs per SM asked of the compiler

// the own cell, then the 13 forward neighbours: (dz > 0) or (dz == 0 and dy > 0) or (dz == dy == 0 and dx > 0)
__constant__ int8_t SR_HALF_STENCIL[14][3] = {
    {0, 0, 0},  {1, 0, 0},  {-1, 1, 0}, {0, 1, 0},  {1, 1, 0},  {-1, -1, 1}, {0, -1, 1},
    {1, -1, 1}, {-1, 0, 1}, {0, 0, 1},  {1, 0, 1},  {-1, 1, 1}, {0, 1, 1},   {1, 1, 1}};

// TABLE: pair terms from the table (the paper's method); else erfc by the polynomial (sr_erfc_from_exp)
template <bool ENERGY, bool TABLE>
__global__ void __launch_bounds__(32 * SR_PAIR_WARPS, SR_PAIR_CTAS) sr_pair_kernel(const SrPairParams p) {
    __shared__ float4 vpos[SR_PAIR_WARPS][32];   // the visiting group: positions relative to THIS cell's centre, charge
    __shared__ float4 vacc[SR_PAIR_WARPS][32];   // ... and what this warp adds to its atoms
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int nc = p.nc, c = blockIdx.x;
    const int cx = c % nc, cy = (c / nc) % nc, cz = c / (nc * nc);
    const uint32_t ox = sr_cell_centre(cx, nc), oy = sr_cell_centre(cy, nc), oz = sr_cell_centre(cz, nc);
    const uint32_t s0 = p.start[c], n_own = p.start[c + 1] - s0;
    const int ng_own = (int)((n_own + 31) >> 5);
    const float two_sa_over_sqrtpi = 1.1283791670955126f * p.sqrt_alpha;
    const float FAR = 1.0e18f;   // position of an empty lane: its pairs always fail the cutoff test (and FAR - FAR = 0 is skipped)
    extern __shared__ __align__(16) unsigned char sr_dyn_smem[];          // the pair-term table(s), one copy per CTA
    const float4* tab_f = reinterpret_cast<const float4*>(sr_dyn_smem);
    const float4* tab_e = tab_f + p.ntab;
    if (TABLE) {
        float4* dst = reinterpret_cast<float4*>(sr_dyn_smem);
        for (int i = threadIdx.x; i < p.ntab; i += 32 * SR_PAIR_WARPS) dst[i] = p.tab_f[i];
        if (ENERGY) for (int i = threadIdx.x; i < p.ntab; i += 32 * SR_PAIR_WARPS) dst[p.ntab + i] = p.tab_e[i];
        __syncthreads();
    }

    for (int g = w; g < ng_own; g += SR_PAIR_WARPS) {
        const uint32_t ei = 32u * g + lane;
        const bool have = ei < n_own;
        const float4 me = have ? sr_relative(p.sorted[s0 + ei], ox, oy, oz, p.len_unit) : make_float4(FAR, FAR, FAR, 0.f);
        float ilo[3] = {-3.0e38f, -3.0e38f, -3.0e38f}, ihi[3] = {3.0e38f, 3.0e38f, 3.0e38f};
        if (g < SR_GMAX) {
            const float* b = p.gbox + ((int64_t)c * SR_GMAX + g) * 6;
#pragma unroll
            for (int k = 0; k < 3; ++k) { ilo[k] = b[k]; ihi[k] = b[3 + k]; }
        }
        float fx = 0.f, fy = 0.f, fz = 0.f, en = 0.f;

        for (int nb = 0; nb < 14; ++nb) {
            const int dxc = SR_HALF_STENCIL[nb][0], dyc = SR_HALF_STENCIL[nb][1], dzc = SR_HALF_STENCIL[nb][2];
            const int cn = (((cz + dzc + nc) % nc) * nc + (cy + dyc + nc) % nc) * nc + (cx + dxc + nc) % nc;
            const uint32_t n0 = p.start[cn], nn = p.start[cn + 1] - n0;
            const int ngn = (int)((nn + 31) >> 5);
            const float shift[3] = {dxc * p.cell_len, dyc * p.cell_len, dzc * p.cell_len};
            for (int h = nb == 0 ? g : 0; h < ngn; ++h) {
                const bool self_block = nb == 0 && h == g;
                if (g < SR_GMAX && h < SR_GMAX && !self_block) {
                    // squared distance between the two bounding boxes: skip the 32 x 32 block when beyond the cutoff
                    const float* b = p.gbox + ((int64_t)cn * SR_GMAX + h) * 6;
                    float d2 = 0.f;
#pragma unroll
                    for (int k = 0; k < 3; ++k) {
                        const float gap = fmaxf(0.f, fmaxf(b[k] + shift[k] - ihi[k], ilo[k] - (b[3 + k] + shift[k])));
                        d2 = fmaf(gap, gap, d2);
                    }
                    if (d2 >= p.rs2) continue;
                }
                const uint32_t ej = 32u * h + lane;
                const bool jvalid = ej < nn;
                __syncwarp();
                vpos[w][lane] = jvalid ? sr_relative(p.sorted[n0 + ej], ox, oy, oz, p.len_unit) : make_float4(FAR, FAR, FAR, 0.f);
                vacc[w][lane] = make_float4(0.f, 0.f, 0.f, 0.f);
                __syncwarp();
#pragma unroll 4
                for (int t = 0; t < 32; ++t) {
                    const int v = (lane + t) & 31;                 // every lane meets a different visitor in every step
                    const float4 o = vpos[w][v];
                    const float dx = o.x - me.x, dy = o.y - me.y, dz = o.z - me.z;
                    const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                    if (r2 < p.rs2 && r2 > 0.f) {
                        float s, u = 0.f;                            // g / r of Eq. (2.10), erfc / r of Eq. (2.8)
                        if (TABLE && r2 >= p.tab_umin) {
                            const uint32_t bits = __float_as_uint(r2);
                            const int idx = (int)(bits >> (23 - SR_TAB_BITS)) - ((127 + SR_TAB_EMIN) << SR_TAB_BITS);
                            const float dl = r2 - __uint_as_float(bits & ~((1u << (23 - SR_TAB_BITS)) - 1u));
                            const float E = sr_ex2(p.nalpha_log2e * r2);
                            const float4 cf = tab_f[idx];
                            s = fmaf(fmaf(fmaf(cf.w, dl, cf.z), dl, cf.y), dl, cf.x) * E;
                            if (ENERGY) {
                                const float4 ce = tab_e[idx];
                                u = fmaf(fmaf(fmaf(ce.w, dl, ce.z), dl, ce.y), dl, ce.x) * E;
                            }
                        } else {                                     // polynomial erfc; with TABLE: the closest pairs ("below r_0")
                            const float inv_r = sr_rsqrt(r2);
                            const float x = p.sqrt_alpha * (r2 * inv_r);
                            const float E = sr_ex2(-1.4426950408889634f * x * x);
                            const float ec = sr_erfc_from_exp(x, E);
                            s = fmaf(ec, inv_r, two_sa_over_sqrtpi * E) * inv_r * inv_r;
                            u = ec * inv_r;
                        }
                        const float sj = o.w * s;
                        fx = fmaf(sj, dx, fx); fy = fmaf(sj, dy, fy); fz = fmaf(sj, dz, fz);
                        if (ENERGY) en = fmaf(o.w, u, en);
                        if (!self_block) {                          // the same pair term, seen from the visitor (d -> -d)
                            const float si = me.w * s;
                            float4 a = vacc[w][v];
                            a.x = fmaf(-si, dx, a.x); a.y = fmaf(-si, dy, a.y); a.z = fmaf(-si, dz, a.z);
                            if (ENERGY) a.w = fmaf(me.w, u, a.w);
                            vacc[w][v] = a;
                        }
                    }
                    __syncwarp();
                }
                if (!self_block && jvalid) {
                    const float4 a = vacc[w][lane];
                    long long* dst = p.acc + 4 * (int64_t)(n0 + ej);
                    if (a.x != 0.f) sr_atomic_add_fixed(dst + 0, a.x);
                    if (a.y != 0.f) sr_atomic_add_fixed(dst + 1, a.y);
                    if (a.z != 0.f) sr_atomic_add_fixed(dst + 2, a.z);
                    if (ENERGY && a.w != 0.f) sr_atomic_add_fixed(dst + 3, a.w);
                }
            }
        }
        if (have) {
            long long* dst = p.acc + 4 * (int64_t)(s0 + ei);
            sr_atomic_add_fixed(dst + 0, fx);
            sr_atomic_add_fixed(dst + 1, fy);
            sr_atomic_add_fixed(dst + 2, fz);
            if (ENERGY) sr_atomic_add_fixed(dst + 3, en);
        }
    }
}

// Fixed point -> fp32, F_i = -q_i A_i, e_i = q_i E_i / 2, scattered to the caller's atom order.
__global__ void __launch_bounds__(256) sr_finalize_kernel(const long long* __restrict__ acc, const uint4* __restrict__ sorted,
                                                           const uint32_t* __restrict__ sidx, int64_t N, float4* __restrict__ force,
                                                           int accumulate, int with_energy) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const double inv = 1.0 / SR_FIXED_SCALE;
    const float q = __uint_as_float(sorted[k].w);
    const longlong2 a01 = reinterpret_cast<const longlong2*>(acc)[2 * k], a23 = reinterpret_cast<const longlong2*>(acc)[2 * k + 1];
    float4 o = make_float4(-q * (float)((double)a01.x * inv), -q * (float)((double)a01.y * inv), -q * (float)((double)a23.x * inv),
                           with_energy ? 0.5f * q * (float)((double)a23.y * inv) : 0.f);
    const uint32_t i = sidx[k];
    if (accumulate) {
        const float4 prev = force[i];
        o.x += prev.x; o.y += prev.y; o.z += prev.z; o.w += prev.w;
    }
    force[i] = o;
}


}  // namespace rbe
