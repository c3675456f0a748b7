// sr_kernels.cuh -- sm_100a kernels of the real-space partner of the RBE force: the short-range part
// of the Ewald-split Coulomb force, Eq. (2.10), truncated at the cutoff radius r_s
// (P:127), and the matching first term of Eq. (2.8) P:112.  SURVEY.md s8(f) row 2, first stage: the
// deterministic truncated sum over a linked-cell list (cubic cells of side >= r_s, as Algorithm 2's
// cell list); the random-batch core/shell estimator of Eqs. (2.13)-(2.16) is the stage
// after this one.  Device code only; the C ABI is in rbe_api.cu.
//
// Positions are the same 32-bit fixed-point turns as in the k-space kernels (to_turns): the cell of
// an atom is floor(S * nc / 2^32) = umulhi(S, nc) per dimension (exact, consistent, periodic wrap for
// free), and the wrapped integer difference S_j - S_i IS the nearest-image separation (in units of
// L / 2^32, i.e. 1e-7 A at L = 464 A): no fp32 cancellation at large L, no image search.
//
// Pipeline per call (all on the caller's stream, no host synchronisation):
//   sr_bin      cell index per atom, per-cell counts (integer atomics: the counts are deterministic)
//   sr_scan     exclusive prefix sum of the counts (one CTA)
//   sr_scatter  atom indices into their cell's segment (slot by integer atomic: arbitrary order)
//   sr_sort     one warp per cell: rank-sort the segment by (sub-cell Morton code, atom index), gather
//               {S, q} in that order -> the layout and every sum below are bitwise reproducible
//   sr_gbox, sr_pair, sr_finalize   (sr_pair_kernels.cuh) the force kernel proper
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "rbe_kernels.cuh"

namespace rbe {


__device__ __forceinline__ int sr_cell_of(uint32_t Sx, uint32_t Sy, uint32_t Sz, int nc) {
    return ((int)__umulhi(Sz, (uint32_t)nc) * nc + (int)__umulhi(Sy, (uint32_t)nc)) * nc + (int)__umulhi(Sx, (uint32_t)nc);
}

__global__ void __launch_bounds__(256) sr_bin_kernel(const float4* __restrict__ xyzq, int64_t N, double two32_over_L, int nc,
                                                      uint4* __restrict__ turns, int32_t* __restrict__ cell_of,
                                                      uint32_t* __restrict__ count) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const float4 a = __ldg(&xyzq[i]);
    const uint32_t Sx = to_turns(a.x, two32_over_L), Sy = to_turns(a.y, two32_over_L), Sz = to_turns(a.z, two32_over_L);
    const int c = sr_cell_of(Sx, Sy, Sz, nc);
    turns[i] = make_uint4(Sx, Sy, Sz, __float_as_uint(a.w));
    cell_of[i] = c;
    atomicAdd(&count[c], 1u);
}

// start[c] = sum_{c' < c} count[c'], start[ncell] = N; cursor[c] = 0.  One CTA of 1024 threads.  A warp owns a contiguous
// stretch of cells and walks it 32 cells at a time (coalesced), carrying its running sum; the 32 stretch totals are then
// added in order and a second coalesced pass adds each warp's offset.  (Looping over ALL cells 1024 at a time with two barriers
// per round took 125 us for the 8e4 cells of a fine list; a contiguous run per THREAD is uncoalesced and no faster.)
__global__ void __launch_bounds__(1024) sr_scan_kernel(const uint32_t* __restrict__ count, int ncell, uint32_t* __restrict__ start,
                                                        uint32_t* __restrict__ cursor) {
    __shared__ uint32_t wsum[32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int per = ((ncell + 1023) / 1024) * 32;               // cells per warp: a multiple of 32
    const int c0 = min(ncell, warp * per), c1 = min(ncell, c0 + per);
    uint32_t carry = 0;
    for (int base = c0; base < c1; base += 32) {
        const int c = base + lane;
        const uint32_t v = c < c1 ? count[c] : 0u;
        uint32_t incl = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t n = __shfl_up_sync(FULL_MASK, incl, d);
            if (lane >= d) incl += n;
        }
        if (c < c1) { start[c] = carry + incl - v; cursor[c] = 0u; }
        carry += __shfl_sync(FULL_MASK, incl, 31);
    }
    if (lane == 0) wsum[warp] = carry;
    __syncthreads();
    uint32_t before = 0, total = 0;
#pragma unroll
    for (int w = 0; w < 32; ++w) {
        const uint32_t v = wsum[w];
        before += w < warp ? v : 0u;
        total += v;
    }
    if (before != 0u)
        for (int c = c0 + lane; c < c1; c += 32) start[c] += before;
    if (tid == 0) start[ncell] = total;
}

__global__ void __launch_bounds__(256) sr_scatter_kernel(const int32_t* __restrict__ cell_of, int64_t N,
                                                          const uint32_t* __restrict__ start, uint32_t* __restrict__ cursor,
                                                          uint32_t* __restrict__ order) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int c = cell_of[i];
    order[start[c] + atomicAdd(&cursor[c], 1u)] = (uint32_t)i;
}

// Position of an atom inside its cell as a 6-bit Morton code of 4 x 4 x 4 sub-cells: sorting a cell by
// it makes every run of 32 consecutive atoms (a warp of the force kernel) spatially compact, so that
// for many far neighbours ALL lanes of the warp fail the cutoff test together and the expensive
// branch is skipped (measured: 5 % on the force kernel; the cutoff tests themselves dominate).
__device__ __forceinline__ uint32_t sr_subcell(const uint4 t, int nc) {
    const uint32_t fx = (t.x * (uint32_t)nc) >> 30, fy = (t.y * (uint32_t)nc) >> 30, fz = (t.z * (uint32_t)nc) >> 30;  // 2 bits each
    return ((fz & 2u) << 4) | ((fy & 2u) << 3) | ((fx & 2u) << 2) | ((fz & 1u) << 2) | ((fy & 1u) << 1) | (fx & 1u);
}

// One warp per cell: the segment arrives in arbitrary order (atomic slots); rank-sort it by
// (sub-cell Morton code, atom index) -- a total order, so the layout is deterministic -- in
// O(n^2 / 32) per lane (n ~ 100), and gather the atom records in that order.
constexpr int SR_SORT_CAP = 256;   // keys of a cell kept in shared memory by its warp (larger cells: keys recomputed from global)

__global__ void __launch_bounds__(256) sr_sort_kernel(const uint32_t* __restrict__ order, const uint32_t* __restrict__ start,
                                                       int ncell, int nc, const uint4* __restrict__ turns, uint4* __restrict__ sorted,
                                                       uint32_t* __restrict__ sidx) {
    __shared__ unsigned long long keys[8][SR_SORT_CAP];
    const int c = (int)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (c >= ncell) return;
    const uint32_t s0 = start[c], n = start[c + 1] - s0;
    if (n <= (uint32_t)SR_SORT_CAP) {
        for (uint32_t e = lane; e < n; e += 32) {
            const uint32_t o = order[s0 + e];
            keys[w][e] = ((unsigned long long)sr_subcell(turns[o], nc) << 32) | o;
        }
        __syncwarp();
        for (uint32_t e = lane; e < n; e += 32) {
            const unsigned long long mkey = keys[w][e];
            uint32_t rank = 0;
            for (uint32_t j = 0; j < n; ++j) rank += keys[w][j] < mkey ? 1u : 0u;     // broadcast reads
            const uint32_t me = (uint32_t)mkey;
            sorted[s0 + rank] = turns[me];
            sidx[s0 + rank] = me;
        }
        return;
    }
    for (uint32_t e = lane; e < n; e += 32) {
        const uint32_t me = order[s0 + e];
        const uint4 mt = turns[me];
        const unsigned long long mkey = ((unsigned long long)sr_subcell(mt, nc) << 32) | me;
        uint32_t rank = 0;
        for (uint32_t j = 0; j < n; ++j) {
            const uint32_t o = order[s0 + j];
            const unsigned long long okey = ((unsigned long long)sr_subcell(turns[o], nc) << 32) | o;
            rank += okey < mkey ? 1u : 0u;
        }
        sorted[s0 + rank] = mt;
        sidx[s0 + rank] = me;
    }
}


// E = exp(-x^2) is shared between erfc and the Gaussian term of Eq. (2.10).
__device__ __forceinline__ float sr_rsqrt(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float sr_rcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float sr_ex2(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

__device__ __forceinline__ float sr_erfc_from_exp(float x, float E) {
    // erfc(x) = t c(t) exp(-x^2), t = 1 / (1 + x / 2): degree-8 fit for RELATIVE error over 0 <= x <= 10
    // (csrc/fit_erfcx.py; 3.4e-7 in fp32), so that far pairs, where erfc is tiny, are as accurate as near
    // ones.  (Abramowitz-Stegun 7.1.26 is only absolutely accurate: 1 % relative error already at x = 3.)
    const float t = sr_rcp(fmaf(0.5f, x, 1.0f));
    float p = fmaf(t, -6.010870773e-02f, 2.894461006e-01f);
    p = fmaf(t, p, -4.968295764e-01f);
    p = fmaf(t, p, 2.885151458e-01f);
    p = fmaf(t, p, -3.339901992e-02f);
    p = fmaf(t, p, 2.053604290e-01f);
    p = fmaf(t, p, 2.424793787e-01f);
    p = fmaf(t, p, 2.824538421e-01f);
    p = fmaf(t, p, 2.820823575e-01f);
    return t * p * E;
}

// Coordinates inside the kernel are fp32 Angstrom RELATIVE TO THE CENTRE OF THE CTA's CELL, computed from the
// wrapped integer difference of the fixed-point turns (so the nearest image is implicit): own atoms lie within
// half a cell side, the staged neighbours within 1.5 cell sides, and a separation d = t_j - t_i carries an
// absolute error <= 2^-24 * 1.5 cell sides (1e-6 A at a 10 A cell) -- instead of three integer subtractions
// and three conversions per candidate pair the conversion is paid once per staged atom.
__device__ __forceinline__ float4 sr_relative(const uint4 a, uint32_t ox, uint32_t oy, uint32_t oz, float len_unit) {
    return make_float4((float)(int32_t)(a.x - ox) * len_unit, (float)(int32_t)(a.y - oy) * len_unit,
                       (float)(int32_t)(a.z - oz) * len_unit, __uint_as_float(a.w));
}

}  // namespace rbe
