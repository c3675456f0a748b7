// rbl_kernels.cuh -- the random batch list (RBL) estimator of the short-range force, section 2.3,
// Eqs. (2.13)-(2.16) P:145-166, Algorithm 2, for the electrostatic pair force of Eq. (2.10):
//   F_i = sum_{j in C(i)} F_ij + (N_s / p) sum_{j in B(i)} F_ij + F^corr,   F^corr = -(1/N) sum_i (...)
// C(i): r < r_c (direct sum); S(i): r_c <= r < r_s, N_s = |S(i)|; B(i): the min(p, N_s) members of S(i)
// with the smallest keys u_ij = fmix32((i A + s0) xor (j B + s1)), (s0, s1) a per-step Philox salt
// (reading Q20): a uniformly random p-subset that does not depend on the order in which the
// neighbours are met, so it is bit-for-bit the oracle's.
//
// Design (second; the first walked 27 cells of side r_s with one thread per atom and one Philox call per
// shell pair, and was 8 x slower than the sum it estimates).  The cell list has cells of side >= r_c, as
// Algorithm 2 says; the candidates of an atom are the (2R+1)^3 cells around its own,
// R = ceil(r_s / cell side) (5^3 for r_s = 2 r_c).  One CTA per cell:
//   1. the candidates of the cell (25 rows of 2R+1 consecutive cells: contiguous in the cell-sorted array)
//      are converted ONCE to fp32 coordinates relative to the cell centre and parked in shared memory;
//   2. a WARP owns one atom of the cell at a time.  Lanes = candidates: every step tests 32 consecutive
//      candidates against the atom (full lanes whatever the cell occupancy); a lane notes its hits in its
//      own column of a shared-memory list, branch-free (the write position advances only on a hit; one bit
//      marks core hits) -- no ballots, no atomics;
//   3. N_s = warp sum of the shell counts.  One lock-step pass over the columns evaluates the core entries
//      and computes the keys of the shell entries; a lane keeps those below a threshold chosen from N_s
//      (expected p + 2 sqrt(p) + 3 of them in the warp) in registers;
//   4. the threshold is bisected over the kept keys until exactly p are below it (the keys of one atom are
//      distinct, so it exists; about log2(p) + 2 warp-wide counts);
//   5. the batch is evaluated, core + (N_s / p) batch reduced over the lanes in a fixed butterfly.
// A cell whose candidates do not fit the tile, an atom with more hits in one lane's column than the column
// holds, takes a slower list-free path (exact bisection on the key threshold over rescans), so any
// density is handled.  sum_i F_i for the correction is accumulated in 64-bit fixed point (integer atomics:
// order-independent), rbl_correct_kernel adds F^corr.  Bitwise reproducible.
#pragma once
#include "sr_pair_kernels.cuh"

namespace rbe {

constexpr int RBL_WARPS = 8;
constexpr int RBL_THREADS = 32 * RBL_WARPS;
constexpr int RBL_TC_MAX = 8192;  // most candidates a CTA parks in shared memory (the launch sizes the tile from the mean density)
constexpr int RBL_EMAX = 40;      // hits (r < r_s) a lane can note per atom (13 expected)
constexpr int RBL_PMAX = 32;
constexpr int RBL_SEGMAX = 2 * 81; // candidate segments: (2R+1)^2 rows, each split in two where it wraps around the box (R <= 4)

struct RblParams {
    const uint4* sorted;      // [N] {Sx, Sy, Sz, q} in cell order
    const uint32_t* sidx;     // [N] original atom index
    const uint32_t* start;    // [ncell + 1]
    float4* force;            // [N] original order
    long long* fsum;          // [3] fixed-point sum of all F_i (zeroed before the launch)
    int32_t nc, R, p, accumulate;
    int32_t tc;               // tile capacity [candidates]: 1.3 x the mean candidate count, <= RBL_TC_MAX
    float len_unit, rc2, rs2, sqrt_alpha;
    uint32_t salt0, salt1;    // reading Q20: first two words of Philox4x32-10(counter (step, 0, 0), key seed), from the host
};

// q_j g(r) / r for one pair (Eq. 2.10): multiply by d and by -q_i to get F_ij
__device__ __forceinline__ float rbl_pair(float r2, float qj, float sqrt_alpha, float two_sa_over_sqrtpi) {
    const float inv_r = sr_rsqrt(r2);
    const float x = sqrt_alpha * (r2 * inv_r);
    const float E = sr_ex2(-1.4426950408889634f * x * x);
    const float ec = sr_erfc_from_exp(x, E);
    return qj * fmaf(ec, inv_r, two_sa_over_sqrtpi * E) * inv_r * inv_r;
}

__device__ __forceinline__ uint32_t rbl_fmix32(uint32_t h) {
    h ^= h >> 16; h *= 0x85EBCA6Bu; h ^= h >> 13; h *= 0xC2B2AE35u; h ^= h >> 16;
    return h;
}
// u_ij given a_i = i * 0x9E3779B1 + s0
__device__ __forceinline__ uint32_t rbl_key(uint32_t a_i, uint32_t j, uint32_t s1) { return rbl_fmix32(a_i ^ (j * 0x85EBCA77u + s1)); }

__device__ __forceinline__ float rbl_warp_sum(float v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(FULL_MASK, v, d);
    return v;
}
__device__ __forceinline__ int rbl_warp_sum(int v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(FULL_MASK, v, d);
    return v;
}
__device__ __forceinline__ int rbl_warp_max(int v) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v = max(v, __shfl_xor_sync(FULL_MASK, v, d));
    return v;
}

// The candidate set of a cell: segments of the cell-sorted array (shared memory), optionally parked in the tile.
struct RblCand {
    const uint32_t* seg_beg;   // [nseg] first atom (sorted position) of the segment
    const uint32_t* seg_pre;   // [nseg + 1] candidates before the segment
    int nseg, total;
    const float4* tile;        // [total] cell-relative coordinates + charge, or nullptr (does not fit)
    const uint32_t* tidx;      // [total] original atom indices (with the tile)
    const uint4* sorted;
    const uint32_t* sidx;
    uint32_t ox, oy, oz;
    float len_unit;
    // candidate f: coordinates relative to the cell centre, charge in .w; j = its original atom index
    __device__ __forceinline__ float4 get(int f, uint32_t& j) const {
        if (tile) { j = tidx[f]; return tile[f]; }
        int lo = 0, hi = nseg - 1;                 // last segment with seg_pre <= f
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (seg_pre[mid] <= (uint32_t)f) lo = mid; else hi = mid - 1;
        }
        const uint32_t g = seg_beg[lo] + ((uint32_t)f - seg_pre[lo]);
        j = sidx[g];
        return sr_relative(sorted[g], ox, oy, oz, len_unit);
    }
};

// List-free path for one atom (whole warp): exact, any density.  Returns core + scale * batch partial sums per lane.
__device__ __forceinline__ void rbl_atom_slow(const RblParams& p, const RblCand& cd, float4 me, uint32_t a_i, int lane,
                                              float two_sa, float& tx, float& ty, float& tz) {
    float fx = 0.f, fy = 0.f, fz = 0.f;
    int nsh = 0;
    for (int f = lane; f < cd.total; f += 32) {
        uint32_t j;
        const float4 o = cd.get(f, j);
        const float dx = o.x - me.x, dy = o.y - me.y, dz = o.z - me.z;
        const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
        if (r2 < p.rs2 && r2 > 0.f) {
            if (r2 < p.rc2) {
                const float s = rbl_pair(r2, o.w, p.sqrt_alpha, two_sa);
                fx = fmaf(s, dx, fx); fy = fmaf(s, dy, fy); fz = fmaf(s, dz, fz);
            } else ++nsh;
        }
    }
    const int Ns = rbl_warp_sum(nsh);
    // the threshold T with exactly min(p, Ns) shell keys <= T: bisection on the 32-bit key space
    uint32_t T = 0xffffffffu;
    if (Ns > p.p) {
        uint32_t lo = 0u, hi = 0xffffffffu;       // count(<= hi) >= p always; find the smallest T with count(<= T) >= p
        while (lo < hi) {
            const uint32_t mid = lo + ((hi - lo) >> 1);
            int cnt = 0;
            for (int f = lane; f < cd.total; f += 32) {
                uint32_t j;
                const float4 o = cd.get(f, j);
                const float dx = o.x - me.x, dy = o.y - me.y, dz = o.z - me.z;
                const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                if (r2 < p.rs2 && r2 >= p.rc2 && rbl_key(a_i, j, p.salt1) <= mid) ++cnt;
            }
            if (rbl_warp_sum(cnt) >= p.p) hi = mid; else lo = mid + 1u;
        }
        T = lo;                                   // keys are distinct: exactly p of them are <= T
    }
    float bx = 0.f, by = 0.f, bz = 0.f;
    for (int f = lane; f < cd.total; f += 32) {
        uint32_t j;
        const float4 o = cd.get(f, j);
        const float dx = o.x - me.x, dy = o.y - me.y, dz = o.z - me.z;
        const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
        if (r2 < p.rs2 && r2 >= p.rc2 && rbl_key(a_i, j, p.salt1) <= T) {
            const float s = rbl_pair(r2, o.w, p.sqrt_alpha, two_sa);
            bx = fmaf(s, dx, bx); by = fmaf(s, dy, by); bz = fmaf(s, dz, bz);
        }
    }
    const float scale = Ns > p.p ? (float)Ns / (float)p.p : 1.0f;
    tx = fmaf(scale, bx, fx); ty = fmaf(scale, by, fy); tz = fmaf(scale, bz, fz);
}

__global__ void __launch_bounds__(RBL_THREADS) rbl_kernel(const RblParams p) {
    extern __shared__ __align__(16) unsigned char rbl_smem[];
    float4* tile = reinterpret_cast<float4*>(rbl_smem);                                   // [tc]
    uint32_t* tidx = reinterpret_cast<uint32_t*>(tile + p.tc);                            // [tc]
    uint16_t* hits_all = reinterpret_cast<uint16_t*>(tidx + p.tc);                        // [RBL_WARPS][RBL_EMAX + 1][32]
    __shared__ uint32_t seg_beg[RBL_SEGMAX], seg_pre[RBL_SEGMAX + 1], seg_cnt[RBL_SEGMAX];
    __shared__ int s_nseg;

    const int nc = p.nc, c = blockIdx.x, tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const uint32_t s0 = p.start[c], n_own = p.start[c + 1] - s0;
    if (n_own == 0u) return;
    const int cx = c % nc, cy = (c / nc) % nc, cz = c / (nc * nc);
    const uint32_t ox = sr_cell_centre(cx, nc), oy = sr_cell_centre(cy, nc), oz = sr_cell_centre(cz, nc);
    const float two_sa = 1.1283791670955126f * p.sqrt_alpha;

    // ---- 1. candidate segments: one row of 2R+1 cells per (dz, dy); where it wraps around the box it has a
    // second part.  Two slots per row (main part, wrapped part; either may be empty), filled in parallel.
    const int R = p.R, side = 2 * R + 1, nrows = side * side;
    for (int r = tid; r < nrows; r += RBL_THREADS) {
        const int dz = r / side - R, dy = r % side - R;
        const int zz = (cz + dz + nc) % nc, yy = (cy + dy + nc) % nc;
        const int row = (zz * nc + yy) * nc;
        const int x0 = cx - R, x1 = cx + R;                            // inclusive; 2R + 1 <= nc: at most one end wraps
        const int a0 = x0 < 0 ? 0 : x0, a1 = x1 >= nc ? nc - 1 : x1;
        const uint32_t mb = p.start[row + a0], me_ = p.start[row + a1 + 1];
        uint32_t wb = 0u, we = 0u;
        if (x0 < 0) { wb = p.start[row + x0 + nc]; we = p.start[row + nc]; }
        else if (x1 >= nc) { wb = p.start[row]; we = p.start[row + x1 - nc + 1]; }
        seg_beg[2 * r] = mb; seg_cnt[2 * r] = me_ - mb;
        seg_beg[2 * r + 1] = wb; seg_cnt[2 * r + 1] = we - wb;
    }
    __syncthreads();
    if (w == 0) {     // exclusive prefix over the 2 * nrows <= 162 counts: a blocked scan by one warp
        const int nseg = 2 * nrows, per = (nseg + 31) / 32;
        uint32_t run = 0;
        for (int e = lane * per; e < min(nseg, (lane + 1) * per); ++e) run += seg_cnt[e];
        uint32_t incl = run;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t n = __shfl_up_sync(FULL_MASK, incl, d);
            if (lane >= d) incl += n;
        }
        uint32_t ex = incl - run;
        for (int e = lane * per; e < min(nseg, (lane + 1) * per); ++e) { seg_pre[e] = ex; ex += seg_cnt[e]; }
        if (lane == 31) { seg_pre[nseg] = incl; s_nseg = nseg; }
    }
    __syncthreads();
    RblCand cd;
    cd.seg_beg = seg_beg; cd.seg_pre = seg_pre; cd.nseg = s_nseg; cd.total = (int)seg_pre[s_nseg];
    cd.tile = nullptr; cd.tidx = nullptr; cd.sorted = p.sorted; cd.sidx = p.sidx;
    cd.ox = ox; cd.oy = oy; cd.oz = oz; cd.len_unit = p.len_unit;
    const bool fits = cd.total <= p.tc;
    if (fits) {
        // a warp per segment: coalesced reads of a run of the cell-sorted array, no search
        for (int sg = w; sg < cd.nseg; sg += RBL_WARPS) {
            const uint32_t g0 = seg_beg[sg], f0 = seg_pre[sg], n = seg_pre[sg + 1] - f0;
            for (uint32_t k = lane; k < n; k += 32) {
                tile[f0 + k] = sr_relative(p.sorted[g0 + k], ox, oy, oz, p.len_unit);
                tidx[f0 + k] = p.sidx[g0 + k];
            }
        }
        __syncthreads();
        cd.tile = tile; cd.tidx = tidx;
    }

    uint16_t* hits = hits_all + w * (RBL_EMAX + 1) * 32 + lane;   // this lane's column: entry e at hits[e * 32] (+ one scratch slot)
    long long sx = 0, sy = 0, sz = 0;     // lane 0: this warp's fixed-point sum of forces
    constexpr int KSEL = 6;               // shell members below the key threshold a lane keeps in registers (1.4 expected)

    // ---- 2. a warp per atom
    for (uint32_t a = w; a < n_own; a += RBL_WARPS) {
        const float4 me = sr_relative(p.sorted[s0 + a], ox, oy, oz, p.len_unit);
        const uint32_t i_orig = p.sidx[s0 + a];
        const uint32_t a_i = i_orig * 0x9E3779B1u + p.salt0;
        float tx, ty, tz;
        bool slow = !fits;
        if (!slow) {
            // scan, branch-free: every step stores its candidate index into the lane's column -- at the shell
            // write position (counting up from slot 0) or, for a core hit, at the core write position (counting
            // down from slot RBL_EMAX) -- and a position moves only on a hit of its kind.  r = 0 (the atom itself,
            // coincident atoms) lands in the core list and is skipped when that is evaluated.
            int nsh = 0, nco = 0;
#pragma unroll 4
            for (int f = lane; f < cd.total; f += 32) {
                const float4 o = tile[f];
                const float dx = o.x - me.x, dy = o.y - me.y, dz = o.z - me.z;
                const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                const bool co = r2 < p.rc2, sh = !co && r2 < p.rs2;
                const int pos = co ? RBL_EMAX - nco : nsh;
                hits[max(0, min(pos, RBL_EMAX)) * 32] = (uint16_t)f;
                nsh += sh ? 1 : 0;
                nco += co ? 1 : 0;
            }
            const int nh = nsh + nco;
            const int max_h = rbl_warp_max(nh);
            slow = max_h > RBL_EMAX;           // shell and core lists of some lane met: the column is too short
            if (!slow) {
                const int Ns = rbl_warp_sum(nsh);
                const int max_sh = rbl_warp_max(nsh), max_co = rbl_warp_max(nco);
                const bool all = Ns <= p.p;                 // the whole shell is the batch (scale 1)
                // threshold for the keys: expect p + 2 sqrt(p) + 3 of the Ns below it
                double want = (double)p.p + 2.0 * sqrt((double)p.p) + 3.0;
                float fx = 0.f, fy = 0.f, fz = 0.f, bx = 0.f, by = 0.f, bz = 0.f, scale = 1.0f;
                uint32_t sk[KSEL];
                uint16_t sc[KSEL];
                for (int attempt = 0;; ++attempt) {
                    uint32_t T = 0xffffffffu;
                    if (!all && want < (double)Ns) T = (uint32_t)(want / (double)Ns * 4294967296.0);
                    // ---- 3. lock-step over the shell entries: their keys; those with key <= T are kept in registers,
                    // at most KSEL per lane (or, with the whole shell in the batch, they are evaluated right away)
                    int nsel = 0;
#pragma unroll
                    for (int t = 0; t < KSEL; ++t) { sk[t] = 0xffffffffu; sc[t] = 0; }
                    for (int e = 0; e < max_sh; ++e) {
                        if (e < nsh) {
                            const int f = hits[e * 32];
                            if (all) {
                                const float4 o = tile[f];
                                const float dx = o.x - me.x, dy = o.y - me.y, dz = o.z - me.z;
                                const float s = rbl_pair(fmaf(dx, dx, fmaf(dy, dy, dz * dz)), o.w, p.sqrt_alpha, two_sa);
                                bx = fmaf(s, dx, bx); by = fmaf(s, dy, by); bz = fmaf(s, dz, bz);
                            } else {
                                const uint32_t key = rbl_key(a_i, tidx[f], p.salt1);
                                if (key <= T) {
#pragma unroll
                                    for (int t = 0; t < KSEL; ++t)
                                        if (t == nsel) { sk[t] = key; sc[t] = (uint16_t)f; }
                                    ++nsel;
                                }
                            }
                        }
                    }
                    // ... and, once, over the core entries (a few per lane)
                    if (attempt == 0)
                        for (int e = 0; e < max_co; ++e)
                            if (e < nco) {
                                const float4 o = tile[hits[(RBL_EMAX - e) * 32]];
                                const float dx = o.x - me.x, dy = o.y - me.y, dz = o.z - me.z;
                                const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                                if (r2 > 0.f) {
                                    const float s = rbl_pair(r2, o.w, p.sqrt_alpha, two_sa);
                                    fx = fmaf(s, dx, fx); fy = fmaf(s, dy, fy); fz = fmaf(s, dz, fz);
                                }
                            }
                    if (all) break;
                    scale = (float)Ns / (float)p.p;
                    // ---- 4. the p smallest keys: bisect the threshold over the kept keys until exactly p are below it
                    // (the keys of one atom are distinct).  Fewer than p kept in all (~1 % of the atoms), or more than
                    // KSEL in one lane: the guess was unlucky -- adjust it and make the pass again.
                    const int tot_sel = rbl_warp_sum(nsel);
                    const bool crowded = rbl_warp_max(nsel) > KSEL;
                    if (crowded || tot_sel < p.p) {
                        if (attempt >= 6) { slow = true; break; }
                        want = crowded ? fmax((double)p.p + 1.0, 0.8 * want) : 1.5 * want + 4.0;
                        continue;
                    }
                    uint32_t lo = 0u, hi = T, Tp = T;
                    int cnt = tot_sel;
                    while (cnt != p.p) {
                        Tp = lo + ((hi - lo) >> 1);
                        int mine = 0;
#pragma unroll
                        for (int t = 0; t < KSEL; ++t) mine += sk[t] <= Tp ? 1 : 0;
                        cnt = rbl_warp_sum(mine);
                        if (cnt > p.p) hi = Tp - 1u; else if (cnt < p.p) lo = Tp + 1u;
                    }
                    // ---- 5. the batch
#pragma unroll
                    for (int t = 0; t < KSEL; ++t)
                        if (sk[t] <= Tp && t < nsel) {
                            const float4 o = tile[sc[t]];
                            const float dx = o.x - me.x, dy = o.y - me.y, dz = o.z - me.z;
                            const float s = rbl_pair(fmaf(dx, dx, fmaf(dy, dy, dz * dz)), o.w, p.sqrt_alpha, two_sa);
                            bx = fmaf(s, dx, bx); by = fmaf(s, dy, by); bz = fmaf(s, dz, bz);
                        }
                    break;
                }
                tx = fmaf(scale, bx, fx); ty = fmaf(scale, by, fy); tz = fmaf(scale, bz, fz);
            }
        }
        if (slow) rbl_atom_slow(p, cd, me, a_i, lane, two_sa, tx, ty, tz);
        tx = rbl_warp_sum(tx); ty = rbl_warp_sum(ty); tz = rbl_warp_sum(tz);
        if (lane == 0) {
            float4 out = make_float4(-me.w * tx, -me.w * ty, -me.w * tz, 0.f);
            sx += __double2ll_rn((double)out.x * SR_FIXED_SCALE);
            sy += __double2ll_rn((double)out.y * SR_FIXED_SCALE);
            sz += __double2ll_rn((double)out.z * SR_FIXED_SCALE);
            if (p.accumulate) {
                const float4 prev = p.force[i_orig];
                out.x += prev.x; out.y += prev.y; out.z += prev.z; out.w += prev.w;
            }
            p.force[i_orig] = out;
        }
    }
    // sum of this warp's forces, integers: any order gives the same bits
    if (lane == 0 && (sx | sy | sz) != 0) {
        atomicAdd(reinterpret_cast<unsigned long long*>(p.fsum + 0), (unsigned long long)sx);
        atomicAdd(reinterpret_cast<unsigned long long*>(p.fsum + 1), (unsigned long long)sy);
        atomicAdd(reinterpret_cast<unsigned long long*>(p.fsum + 2), (unsigned long long)sz);
    }
}

constexpr size_t rbl_smem_bytes(int tc) {
    return (size_t)tc * (sizeof(float4) + sizeof(uint32_t)) + (size_t)RBL_WARPS * (RBL_EMAX + 1) * 32 * sizeof(uint16_t);
}

// F_i += F^corr = -(1/N) sum_i F_i  (Eq. 2.16)
__global__ void __launch_bounds__(256) rbl_correct_kernel(const long long* __restrict__ fsum, int64_t N, float4* __restrict__ force) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double inv = -1.0 / (SR_FIXED_SCALE * (double)N);
    float4 f = force[i];
    f.x += (float)((double)fsum[0] * inv);
    f.y += (float)((double)fsum[1] * inv);
    f.z += (float)((double)fsum[2] * inv);
    force[i] = f;
}

}  // namespace rbe
