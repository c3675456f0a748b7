// rbl_kernels.cuh -- the random batch list (RBL) estimator of the short-range force, section 2.3,
// Eqs. (2.13)-(2.16) P:145-166, Algorithm 2, for the electrostatic pair force of Eq. (2.10):
//   F_i = sum_{j in C(i)} F_ij + (N_s / p) sum_{j in B(i)} F_ij + F^corr,   F^corr = -(1/N) sum_i (...)
// C(i): r < r_c (direct sum); S(i): r_c <= r < r_s, N_s = |S(i)|; B(i): the min(p, N_s) members of S(i)
// with the smallest (u_ij, j), u_ij = first word of Philox4x32-10(counter (i, j, step), key seed)
// (reading Q20): a uniformly random p-subset that does not depend on the order in which the
// neighbours are met, so it is bit-for-bit the oracle's.
//
// First implementation, written for parity and as the measurement behind DESIGN.md section 11 (on B200
// the random selection costs more than evaluating the shell it replaces): a thread owns an atom and
// walks the 27 cells of the linked-cell list built by sr_kernels.cuh; core pairs are summed on the fly,
// every shell pair costs one Philox call and a compare against the thread's current p-th smallest key,
// kept with its neighbour slots in shared memory ("replace the maximum, rescan"); the batch is evaluated
// afterwards from the stored slots.  sum_i F_i for the correction is accumulated in 64-bit fixed point
// (integer atomics: order-independent), rbl_correct_kernel adds F^corr.
#pragma once
#include "sr_pair_kernels.cuh"

namespace rbe {

constexpr int RBL_THREADS = 64;
constexpr int RBL_TILE = 128;
constexpr int RBL_PMAX = 32;

struct RblParams {
    const uint4* sorted;      // [N] {Sx, Sy, Sz, q} in cell order
    const uint32_t* sidx;     // [N] original atom index
    const uint32_t* start;    // [ncell + 1]
    float4* force;            // [N] original order
    long long* fsum;          // [3] fixed-point sum of all F_i (zeroed before the launch)
    int32_t nc, p, accumulate;
    float len_unit, rc2, rs2, sqrt_alpha;
    unsigned long long seed, step;
};

// q_j g(r) / r for one pair (Eq. 2.10): multiply by d and by -q_i to get F_ij
__device__ __forceinline__ float rbl_pair(float r2, float qj, float sqrt_alpha, float two_sa_over_sqrtpi) {
    const float inv_r = sr_rsqrt(r2);
    const float x = sqrt_alpha * (r2 * inv_r);
    const float E = sr_ex2(-1.4426950408889634f * x * x);
    const float ec = sr_erfc_from_exp(x, E);
    return qj * fmaf(ec, inv_r, two_sa_over_sqrtpi * E) * inv_r * inv_r;
}

__global__ void __launch_bounds__(RBL_THREADS) rbl_kernel(const RblParams p) {
    __shared__ float4 tile[RBL_TILE];
    __shared__ uint32_t tile_idx[RBL_TILE];
    __shared__ unsigned long long bkey[RBL_PMAX][RBL_THREADS];   // the thread's batch candidates: (u_ij << 32) | j
    __shared__ uint32_t bslot[RBL_PMAX][RBL_THREADS];            // ... and where j sits in the sorted array
    const int nc = p.nc, c = blockIdx.x, tid = threadIdx.x;
    const int cx = c % nc, cy = (c / nc) % nc, cz = c / (nc * nc);
    const uint32_t ox = sr_cell_centre(cx, nc), oy = sr_cell_centre(cy, nc), oz = sr_cell_centre(cz, nc);
    const uint32_t s0 = p.start[c], n_own = p.start[c + 1] - s0;
    const float two_sa_over_sqrtpi = 1.1283791670955126f * p.sqrt_alpha;
    const uint2 key = make_uint2((uint32_t)p.seed, (uint32_t)(p.seed >> 32));
    long long sx = 0, sy = 0, sz = 0;

    for (uint32_t pass = 0; pass < n_own; pass += RBL_THREADS) {
        const bool have = pass + tid < n_own;
        const float4 me = have ? sr_relative(p.sorted[s0 + pass + tid], ox, oy, oz, p.len_unit) : make_float4(1.0e18f, 1.0e18f, 1.0e18f, 0.f);
        const uint32_t i_orig = have ? p.sidx[s0 + pass + tid] : 0u;
        float fx = 0.f, fy = 0.f, fz = 0.f;
        int cnt = 0, Ns = 0, maxpos = 0;
        unsigned long long maxkey = 0ull;
        for (int nb = 0; nb < 27; ++nb) {
            const int dxc = nb % 3 - 1, dyc = (nb / 3) % 3 - 1, dzc = nb / 9 - 1;
            const int cn = (((cz + dzc + nc) % nc) * nc + (cy + dyc + nc) % nc) * nc + (cx + dxc + nc) % nc;
            const uint32_t n0 = p.start[cn], n1 = p.start[cn + 1];
            for (uint32_t t0 = n0; t0 < n1; t0 += RBL_TILE) {
                const int tcnt = (int)min((uint32_t)RBL_TILE, n1 - t0);
                __syncthreads();
                for (int k = tid; k < tcnt; k += RBL_THREADS) {
                    tile[k] = sr_relative(p.sorted[t0 + k], ox, oy, oz, p.len_unit);
                    tile_idx[k] = p.sidx[t0 + k];
                }
                __syncthreads();
                if (!have) continue;
                for (int k = 0; k < tcnt; ++k) {
                    const float4 o = tile[k];
                    const float dx = o.x - me.x, dy = o.y - me.y, dz = o.z - me.z;
                    const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                    if (!(r2 < p.rs2) || !(r2 > 0.f)) continue;
                    if (r2 < p.rc2) {                                     // core: direct sum
                        const float s = rbl_pair(r2, o.w, p.sqrt_alpha, two_sa_over_sqrtpi);
                        fx = fmaf(s, dx, fx); fy = fmaf(s, dy, fy); fz = fmaf(s, dz, fz);
                        continue;
                    }
                    // shell: count it; keep it if its key is among the p smallest so far
                    ++Ns;
                    const uint32_t j_orig = tile_idx[k];
                    const uint32_t u = philox4x32_10(make_uint4(i_orig, j_orig, (uint32_t)p.step, (uint32_t)(p.step >> 32)), key).x;
                    const unsigned long long kk = ((unsigned long long)u << 32) | j_orig;
                    int pos = -1;
                    if (cnt < p.p) pos = cnt++;
                    else if (kk < maxkey) pos = maxpos;
                    if (pos >= 0) {
                        bkey[pos][tid] = kk;
                        bslot[pos][tid] = t0 + k;
                        if (cnt == p.p) {                                 // full: find the largest kept key again
                            maxkey = 0ull;
                            for (int e = 0; e < p.p; ++e) {
                                const unsigned long long v = bkey[e][tid];
                                if (v >= maxkey) { maxkey = v; maxpos = e; }
                            }
                        }
                    }
                }
            }
        }
        if (have) {
            // the batch, in the order it was stored (fixed by the layout: reproducible)
            float bx = 0.f, by = 0.f, bz = 0.f;
            for (int e = 0; e < cnt; ++e) {
                const float4 o = sr_relative(p.sorted[bslot[e][tid]], ox, oy, oz, p.len_unit);
                const float dx = o.x - me.x, dy = o.y - me.y, dz = o.z - me.z;
                const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
                const float s = rbl_pair(r2, o.w, p.sqrt_alpha, two_sa_over_sqrtpi);
                bx = fmaf(s, dx, bx); by = fmaf(s, dy, by); bz = fmaf(s, dz, bz);
            }
            const float scale = Ns > p.p ? (float)Ns / (float)p.p : 1.0f;
            float4 out = make_float4(-me.w * fmaf(scale, bx, fx), -me.w * fmaf(scale, by, fy), -me.w * fmaf(scale, bz, fz), 0.f);
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
    // sum of this CTA's forces, integers: any order gives the same bits
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        sx += __shfl_xor_sync(FULL_MASK, sx, d);
        sy += __shfl_xor_sync(FULL_MASK, sy, d);
        sz += __shfl_xor_sync(FULL_MASK, sz, d);
    }
    if ((tid & 31) == 0 && (sx | sy | sz) != 0) {
        atomicAdd(reinterpret_cast<unsigned long long*>(p.fsum + 0), (unsigned long long)sx);
        atomicAdd(reinterpret_cast<unsigned long long*>(p.fsum + 1), (unsigned long long)sy);
        atomicAdd(reinterpret_cast<unsigned long long*>(p.fsum + 2), (unsigned long long)sz);
    }
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
