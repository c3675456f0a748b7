// sr_cell_kernels.cuh -- a second force kernel for the real-space partner (Eq. 2.10 P:122 truncated at r_s),
// selected with rbe_set_pair_kernel(ctx, 1): one CTA per cell of a FINE cell list, the cutoff TEST on the tensor
// cores, every ORDERED pair evaluated by one lane.  (The default, sr_pair_kernels.cuh, walks 32 x 32 blocks of an
// r_s-sided cell list with a warp ring, Newton's third law and fixed-point integer atomics.)
//
// Cells of side >= r_s / 2: the (2R+1)^3 = 125 cells around a cell hold ~1 560 candidates per atom at water density,
// 27 % of them inside the sphere (2 700 and 15 % for 27 cells of side r_s).  Per cell (CTA of SR_W warps):
//   candidates  (2R+1)^2 rows of consecutive cells, each a contiguous run of the cell-sorted array (two runs where a
//               row wraps around the box), taken in opposite pairs so that any stretch of the list lies on both sides
//               of the cell; their sorted positions are listed once in shared memory;
//   per M-TILE of 16 own atoms every WARP walks its own quarter of the candidates, 128 at a time, with no CTA-wide
//   barrier:
//   stage     lane = candidate: fp32 coordinates relative to the cell centre (nearest image implicit in the wrapped
//             integer difference) and the TF32 features of the test, into the warp's own shared memory;
//   test      r_ij^2 = |x_i|^2 + |x_j|^2 - 2 x_i . x_j as a K = 8 product:
//               A_i = (a, a, 1, 1),  a = -2 x_i' (x_i' = x_i rounded to TF32, 3 components),
//               B_j = (x_j^hi, x_j^lo, n_j^hi, n_j^lo),  x_j = x^hi + x^lo, n_j = |x_j|^2, split into TF32 halves,
//               C_i = |x_i'|^2 - (r_s^2 + margin),
//             so D_ij < 0 <=> |x_i' - x_j|^2 < r_s^2 + margin up to 1e-3 A^2: 16 mma.m16n8k8 (TF32, fp32 accumulate)
//             decide 16 x 128 pairs; the sign bits are shifted into two 32-bit words per lane (rows g, g + 8 of the
//             fragment x this lane's 32 columns).  x_i' is at most 2^-12 cell sides from x_i per component and the
//             margin covers it: NO false negatives, ~0.2 % false positives;
//   evaluate  the lane pops its two words: candidate position from shared memory, the EXACT fp32 test
//             0 < r^2 < r_s^2 (what the default kernel tests), the pair term from the table or the
//             polynomial, added to the lane's partial force of that own atom.  A word's 32 candidates are every 16th
//             of a 512-candidate stretch, so every lane sees the same mix of near and far cells;
//   finally the four lanes of a quad, then the warps, are added in a fixed order and F_i = -q_i sum goes straight to
//   the caller's array: no scatter to the partner, no atomics, no fixed point, no zero-fill, no finalise pass.
// Bitwise reproducible.  r_s may reach 0.4 L (five cells per dimension) instead of L / 3.
#pragma once
#include "sr_pair_kernels.cuh"

namespace rbe {

struct SrCellParams {
    const uint4* sorted;      // [N] {Sx, Sy, Sz, q} in cell order
    const uint32_t* sidx;     // [N] caller's index of the atom in slot k
    const uint32_t* start;    // [ncell + 1]
    float4* force;            // [N] out, caller's order: {F_x, F_y, F_z, e_i}
    int32_t nc;
    int32_t R;                // cells the cutoff reaches beyond the own one: ceil(r_s / cell side), 1 or 2
    int32_t accumulate;       // add to what `force` holds
    int32_t cap;              // candidates whose sorted position is listed in shared memory (the rest: searched)
    float len_unit;           // L / 2^32 [A]
    float rs2;                // r_s^2 [A^2]
    float thr;                // r_s^2 + margin of the TF32 test [A^2]
    float sqrt_alpha;
    float nalpha_log2e;       // -alpha log2(e)
    float tab_umin;           // below this r^2 the analytic branch is taken [A^2]
    const float4* tab_f;      // [ntab] cubic coefficients of T_f per interval (sr_table_kernel)
    const float4* tab_e;      // [ntab] ... of T_e
    int32_t ntab;
};

constexpr int SR_W = 4;                 // warps per CTA
constexpr int SR_SLICE = 128;           // candidates a warp stages and tests at a time: 16 mma steps of 8 columns
constexpr int SR_TC = SR_SLICE * SR_W;  // the stretch of the candidate list the warps of a CTA share per round
constexpr int SR_SEGMAX = 2 * 25;       // candidate runs: (2R+1)^2 rows (R <= 2), each split in two where it wraps around the box
constexpr int SR_CAP_MAX = 8192;

__host__ __device__ constexpr size_t sr_cell_smem_bytes(int ntab, bool table, bool energy, int cap) {
    return (table ? (size_t)ntab * sizeof(float4) * (energy ? 2 : 1) : 0) + (size_t)cap * sizeof(uint32_t);
}

__device__ __forceinline__ float sr_tf32(float x) {   // x rounded to TF32 (10 explicit mantissa bits), as an fp32 value
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return __uint_as_float(r);
}
// D (16 x 8, fp32) = A (16 x 8, TF32, row) x B (8 x 8, TF32, col) + C; fragment layouts as in the PTX ISA (g = lane / 4,
// c = lane % 4): a0 (g, c) a1 (g + 8, c) a2 (g, c + 4) a3 (g + 8, c + 4); b0 (k = c, n = g) b1 (k = c + 4, n = g);
// d0 (g, 2c) d1 (g, 2c + 1) d2 (g + 8, 2c) d3 (g + 8, 2c + 1).  C = {c_lo, c_lo, c_hi, c_hi}: one value per row.
__device__ __forceinline__ void sr_mma_tf32(uint32_t (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1, float c_lo, float c_hi) {
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0, %1, %2, %3}, {%4, %5, %6, %7}, {%8, %9}, {%10, %10, %11, %11};"
                 : "=r"(d[0]), "=r"(d[1]), "=r"(d[2]), "=r"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1), "f"(c_lo), "f"(c_hi));
}
__device__ __forceinline__ int sr_top_bit(uint32_t x) {   // index of the highest set bit (x != 0): one FLO
    int r;
    asm("bfind.u32 %0, %1;" : "=r"(r) : "r"(x));
    return r;
}

// One pair: the candidate at o against the own atom at me; adds q_j g(r)/r d (and q_j erfc/r) to acc.
template <bool ENERGY, bool TABLE>
__device__ __forceinline__ void sr_cell_pair(const SrCellParams& p, const float4* tab_f, const float4* tab_e, float two_sa_over_sqrtpi,
                                             const float4 me, const float4 o, float4& acc) {
    const float dx = o.x - me.x, dy = o.y - me.y, dz = o.z - me.z;
    const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
    float s, u = 0.f;
    if (TABLE && r2 >= p.tab_umin) {
        const uint32_t bits = __float_as_uint(r2);
        const int idx = min((int)(bits >> (23 - SR_TAB_BITS)) - ((127 + SR_TAB_EMIN) << SR_TAB_BITS), p.ntab - 1);
        const float dl = r2 - __uint_as_float(bits & ~((1u << (23 - SR_TAB_BITS)) - 1u));
        const float E = sr_ex2(p.nalpha_log2e * r2);
        const float4 cf = tab_f[idx];
        s = fmaf(fmaf(fmaf(cf.w, dl, cf.z), dl, cf.y), dl, cf.x) * E;
        if (ENERGY) {
            const float4 ce = tab_e[idx];
            u = fmaf(fmaf(fmaf(ce.w, dl, ce.z), dl, ce.y), dl, ce.x) * E;
        }
    } else {                                                 // polynomial erfc; with TABLE: the closest pairs ("below r_0")
        const float inv_r = sr_rsqrt(r2);
        const float x = p.sqrt_alpha * (r2 * inv_r);
        const float E = sr_ex2(p.nalpha_log2e * r2);           // x^2 = alpha r^2: off the rsqrt chain
        const float ec = sr_erfc_from_exp(x, E);
        s = fmaf(ec, inv_r, two_sa_over_sqrtpi * E) * (inv_r * inv_r);
        u = ec * inv_r;
    }
    const bool inside = r2 < p.rs2 && r2 > 0.f;            // the exact cutoff test; the atom itself and coincident atoms are skipped (Q18)
    s = inside ? s : 0.f;
    if (ENERGY) u = inside ? u : 0.f;
    const float sj = o.w * s;
    acc.x = fmaf(sj, dx, acc.x); acc.y = fmaf(sj, dy, acc.y); acc.z = fmaf(sj, dz, acc.z);
    if (ENERGY) acc.w = fmaf(o.w, u, acc.w);
}

constexpr int SR_CELL_CTAS = 6;   // resident CTAs per SM asked of the compiler (80 registers); sweep: profiles/r02_sr_designs.md

template <bool ENERGY, bool TABLE>
__global__ void __launch_bounds__(32 * SR_W, SR_CELL_CTAS) sr_cell_kernel(const SrCellParams p) {
    extern __shared__ __align__(16) unsigned char sr_dyn_smem[];      // the pair-term table(s), then the candidate list
    __shared__ float4 cposw[SR_W][4 * 33];                 // per warp: its slice's candidates, word-major [word][bit], one slot of padding per word
    __shared__ __align__(16) float fa[SR_W][SR_SLICE * 4]; // candidate nl: {x^hi, y^hi, z^hi, x^lo}
    __shared__ __align__(16) float fb[SR_W][SR_SLICE * 4]; //               {y^lo, z^lo, n^hi, n^lo}
    __shared__ float4 red[SR_W][16];
    __shared__ uint32_t seg_beg[SR_SEGMAX], seg_pre[SR_SEGMAX + 1], seg_cnt[SR_SEGMAX];

    const int nc = p.nc, c = blockIdx.x, tid = threadIdx.x, lane = tid & 31, w = tid >> 5, g8 = lane >> 2, c4 = lane & 3;
    const uint32_t s0 = p.start[c], n_own = p.start[c + 1] - s0;
    if (n_own == 0u) return;
    const int cx = c % nc, cy = (c / nc) % nc, cz = c / (nc * nc);
    const uint32_t ox = sr_cell_centre(cx, nc), oy = sr_cell_centre(cy, nc), oz = sr_cell_centre(cz, nc);
    const float two_sa_over_sqrtpi = 1.1283791670955126f * p.sqrt_alpha;
    const float FAR = 1.0e15f;   // an empty slot: never inside the cutoff, no overflow in the test
    const size_t tab_bytes = TABLE ? (size_t)p.ntab * sizeof(float4) * (ENERGY ? 2 : 1) : 0;
    const float4* tab_f = reinterpret_cast<const float4*>(sr_dyn_smem);
    const float4* tab_e = tab_f + p.ntab;
    uint32_t* cand = reinterpret_cast<uint32_t*>(sr_dyn_smem + tab_bytes);          // [cap] sorted position of candidate f
    if (TABLE) {
        float4* dst = reinterpret_cast<float4*>(sr_dyn_smem);
        for (int i = tid; i < p.ntab; i += 32 * SR_W) dst[i] = p.tab_f[i];
        if (ENERGY) for (int i = tid; i < p.ntab; i += 32 * SR_W) dst[p.ntab + i] = p.tab_e[i];
    }

    // ---- candidate runs: one row of 2R+1 consecutive cells per (dz, dy), a second part where it wraps around the box.
    // The rows come in opposite pairs (the own row first).
    const int R = p.R, side = 2 * R + 1, nrows = side * side, nseg = 2 * nrows;
    for (int rr = tid; rr < nrows; rr += 32 * SR_W) {
        const int t = (rr - 1) >> 1;
        const int k = rr == 0 ? (nrows - 1) / 2 : (rr & 1) ? t : nrows - 1 - t;
        const int dz = k / side - R, dy = k % side - R;
        const int zz = (cz + dz + nc) % nc, yy = (cy + dy + nc) % nc;
        const int row = (zz * nc + yy) * nc;
        const int x0 = cx - R, x1 = cx + R;                            // inclusive; 2R + 1 <= nc: at most one end wraps
        const int a0 = x0 < 0 ? 0 : x0, a1 = x1 >= nc ? nc - 1 : x1;
        const uint32_t mb = p.start[row + a0], me_ = p.start[row + a1 + 1];
        uint32_t wb = 0u, we = 0u;
        if (x0 < 0) { wb = p.start[row + x0 + nc]; we = p.start[row + nc]; }
        else if (x1 >= nc) { wb = p.start[row]; we = p.start[row + x1 - nc + 1]; }
        seg_beg[2 * rr] = mb; seg_cnt[2 * rr] = me_ - mb;
        seg_beg[2 * rr + 1] = wb; seg_cnt[2 * rr + 1] = we - wb;
    }
    __syncthreads();
    if (w == 0) {     // exclusive prefix over the <= 50 counts: two per lane
        const uint32_t c0 = 2 * lane < nseg ? seg_cnt[2 * lane] : 0u, c1 = 2 * lane + 1 < nseg ? seg_cnt[2 * lane + 1] : 0u;
        uint32_t incl = c0 + c1;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t n = __shfl_up_sync(FULL_MASK, incl, d);
            if (lane >= d) incl += n;
        }
        const uint32_t ex = incl - c0 - c1;
        if (2 * lane < nseg) seg_pre[2 * lane] = ex;
        if (2 * lane + 1 < nseg) seg_pre[2 * lane + 1] = ex + c0;
        if (lane == 31) seg_pre[nseg] = incl;
    }
    __syncthreads();
    const int total = (int)seg_pre[nseg];
    for (int sg = w; sg < nseg; sg += SR_W) {                        // the list: a warp per run
        const int f0 = (int)seg_pre[sg], n = (int)seg_pre[sg + 1] - f0;
        const uint32_t g0 = seg_beg[sg];
        for (int k = lane; k < n && f0 + k < p.cap; k += 32) cand[f0 + k] = g0 + (uint32_t)k;
    }
    __syncthreads();
    // sorted position of candidate f (f < total): from the list, or -- a cell more crowded than the list -- by search
    auto position = [&](int f) -> uint32_t {
        if (f < p.cap) return cand[f];
        int lo = 0, hi = nseg - 1;                 // last run with seg_pre <= f
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if ((int)seg_pre[mid] <= f) lo = mid; else hi = mid - 1;
        }
        return seg_beg[lo] + (uint32_t)(f - (int)seg_pre[lo]);
    };

    const int nround = (total + SR_TC - 1) / SR_TC;
    // column g8 of mma step m is slot 8 m + bcol of the warp's slice; slot nl = word nl % 4, bit nl / 4
    const int bcol = 4 * (g8 & 1) + (g8 >> 1);
    const float4* cw = cposw[w] + c4 * 33;             // the 32 candidates of this lane's two mask words, by bit
    float* wfa = fa[w];
    float* wfb = fb[w];

    for (uint32_t m0 = 0; m0 < n_own; m0 += 16) {
        // ---- the M-tile's own atoms: this lane's rows g8 and g8 + 8 of the fragments
        const bool have_lo = m0 + g8 < n_own, have_hi = m0 + g8 + 8 < n_own;
        const float4 me_lo = have_lo ? sr_relative(p.sorted[s0 + m0 + g8], ox, oy, oz, p.len_unit) : make_float4(FAR, FAR, FAR, 0.f);
        const float4 me_hi = have_hi ? sr_relative(p.sorted[s0 + m0 + g8 + 8], ox, oy, oz, p.len_unit) : make_float4(FAR, FAR, FAR, 0.f);
        uint32_t afr[4];
        float c_lo, c_hi;
        {
            const float xl = sr_tf32(me_lo.x), yl = sr_tf32(me_lo.y), zl = sr_tf32(me_lo.z);
            const float xh = sr_tf32(me_hi.x), yh = sr_tf32(me_hi.y), zh = sr_tf32(me_hi.z);
            afr[0] = __float_as_uint(-2.f * (c4 == 0 ? xl : c4 == 1 ? yl : c4 == 2 ? zl : xl));    // k = c4:     (ax, ay, az, ax)
            afr[1] = __float_as_uint(-2.f * (c4 == 0 ? xh : c4 == 1 ? yh : c4 == 2 ? zh : xh));
            afr[2] = __float_as_uint(c4 == 0 ? -2.f * yl : c4 == 1 ? -2.f * zl : 1.0f);            // k = c4 + 4: (ay, az, 1, 1)
            afr[3] = __float_as_uint(c4 == 0 ? -2.f * yh : c4 == 1 ? -2.f * zh : 1.0f);
            c_lo = fmaf(xl, xl, fmaf(yl, yl, zl * zl)) - p.thr;
            c_hi = fmaf(xh, xh, fmaf(yh, yh, zh * zh)) - p.thr;
        }
        float4 acc_lo = make_float4(0.f, 0.f, 0.f, 0.f), acc_hi = make_float4(0.f, 0.f, 0.f, 0.f);

        for (int t = 0; t < nround; ++t) {
            // this warp's slice of round t: candidates f = T0 + 4 nl + w, nl = 0 .. 127 (every fourth of the stretch)
            const int T0 = t * SR_TC;
            const int left = total - T0 - w;                         // > 0: candidates f = T0 + w, T0 + w + 4, ... < total
            const int nslot = left > 0 ? min(SR_SLICE, (left + 3) >> 2) : 0;
            const int msteps = (nslot + 7) >> 3;
            if (msteps == 0) continue;
            __syncwarp();                                            // the previous slice has been evaluated
            // ---- stage
#pragma unroll
            for (int i = 0; i < SR_SLICE / 32; ++i) {
                const int nl = lane + 32 * i;
                if (nl < 8 * msteps) {
                    float4 v = make_float4(FAR, FAR, FAR, 0.f), va = make_float4(FAR, FAR, FAR, 0.f), vb = make_float4(0.f, 0.f, 1.0e31f, 0.f);
                    if (nl < nslot) {
                        v = sr_relative(p.sorted[position(T0 + 4 * nl + w)], ox, oy, oz, p.len_unit);
                        const float xh = sr_tf32(v.x), yh = sr_tf32(v.y), zh = sr_tf32(v.z);
                        const float nn = fmaf(v.x, v.x, fmaf(v.y, v.y, v.z * v.z)), nh = sr_tf32(nn);
                        va = make_float4(xh, yh, zh, v.x - xh);
                        vb = make_float4(v.y - yh, v.z - zh, nh, nn - nh);
                    }
                    cposw[w][(nl & 3) * 33 + (nl >> 2)] = v;
                    *reinterpret_cast<float4*>(&wfa[4 * nl]) = va;
                    *reinterpret_cast<float4*>(&wfb[4 * nl]) = vb;
                }
            }
            __syncwarp();
            // ---- test: D = C + A B; the sign bit of every element goes into the word of its row; bit 2 m + e <->
            // column 2 c4 + e of step m
            uint32_t w_lo = 0u, w_hi = 0u;
            auto mma_step = [&](int m) {
                const uint32_t b0 = __float_as_uint(wfa[4 * (8 * m + bcol) + c4]), b1 = __float_as_uint(wfb[4 * (8 * m + bcol) + c4]);
                uint32_t d[4];
                sr_mma_tf32(d, afr, b0, b1, c_lo, c_hi);
                w_lo = __funnelshift_l(d[1], w_lo, 1);          // (w << 1) | sign(d)
                w_lo = __funnelshift_l(d[0], w_lo, 1);
                w_hi = __funnelshift_l(d[3], w_hi, 1);
                w_hi = __funnelshift_l(d[2], w_hi, 1);
            };
            if (msteps == 16) {
#pragma unroll
                for (int m = 15; m >= 0; --m) mma_step(m);
            } else {
                for (int m = msteps - 1; m >= 0; --m) mma_step(m);
            }
            // ---- evaluate: the lane's hits of row g8, then of row g8 + 8
            while (__any_sync(FULL_MASK, w_lo != 0u)) {
                if (w_lo != 0u) {
                    const int b = sr_top_bit(w_lo);
                    w_lo &= ~(1u << b);
                    sr_cell_pair<ENERGY, TABLE>(p, tab_f, tab_e, two_sa_over_sqrtpi, me_lo, cw[b], acc_lo);
                }
            }
            while (__any_sync(FULL_MASK, w_hi != 0u)) {
                if (w_hi != 0u) {
                    const int b = sr_top_bit(w_hi);
                    w_hi &= ~(1u << b);
                    sr_cell_pair<ENERGY, TABLE>(p, tab_f, tab_e, two_sa_over_sqrtpi, me_hi, cw[b], acc_hi);
                }
            }
        }

        // ---- the quad, then the warps, in a fixed order; F_i = -q_i sum, e_i = q_i sum / 2
#pragma unroll
        for (int d = 1; d <= 2; d <<= 1) {
            acc_lo.x += __shfl_xor_sync(FULL_MASK, acc_lo.x, d); acc_lo.y += __shfl_xor_sync(FULL_MASK, acc_lo.y, d);
            acc_lo.z += __shfl_xor_sync(FULL_MASK, acc_lo.z, d);
            acc_hi.x += __shfl_xor_sync(FULL_MASK, acc_hi.x, d); acc_hi.y += __shfl_xor_sync(FULL_MASK, acc_hi.y, d);
            acc_hi.z += __shfl_xor_sync(FULL_MASK, acc_hi.z, d);
            if (ENERGY) { acc_lo.w += __shfl_xor_sync(FULL_MASK, acc_lo.w, d); acc_hi.w += __shfl_xor_sync(FULL_MASK, acc_hi.w, d); }
        }
        __syncthreads();                                 // the previous M-tile's partial sums have been read
        if (c4 == 0) { red[w][g8] = acc_lo; red[w][g8 + 8] = acc_hi; }
        __syncthreads();
        if (tid < 16 && m0 + tid < n_own) {
            float4 a = red[0][tid];
#pragma unroll
            for (int ww = 1; ww < SR_W; ++ww) { a.x += red[ww][tid].x; a.y += red[ww][tid].y; a.z += red[ww][tid].z; a.w += red[ww][tid].w; }
            const float q = __uint_as_float(p.sorted[s0 + m0 + tid].w);
            const uint32_t i = p.sidx[s0 + m0 + tid];
            float4 o = make_float4(-q * a.x, -q * a.y, -q * a.z, ENERGY ? 0.5f * q * a.w : 0.f);
            if (p.accumulate) {
                const float4 prev = p.force[i];
                o.x += prev.x; o.y += prev.y; o.z += prev.z; o.w += prev.w;
            }
            p.force[i] = o;
        }
    }
}

}  // namespace rbe
