// rbe_kernels.cuh -- sm_100a kernels of the RBE k-space path (Eq. 2.9, Eq. 2.12,
// Algorithm 1 steps 2-4).  Device code only; the C ABI lives in rbe_api.cu.
//
// Phase arithmetic shared by both hot kernels
// -------------------------------------------
// phi_il = k_l . r_i = 2 pi (m_l . s_i),  s_i = r_i / L.  Each coordinate is converted ONCE per
// atom to 32-bit fixed-point turns  S = round(x * 2^32 / L) mod 2^32  (fp64 FMA + magic number,
// so the fp32 input is used exactly).  Then  m . S  in wrapping 32-bit integer arithmetic IS
// "m . s mod 1" exactly: no range reduction, no growth of the fp32 error with |m| or L, and
// out-of-box atoms wrap for free.  The signed result in [-2^31, 2^31) is converted to fp32 and
// scaled so that the FMUL by fl(1/2pi) inside sin.approx/cos.approx lands on turns; MUFU.SIN /
// MUFU.COS then evaluate sin/cos(2 pi t), |t| <= 1/2.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace rbe {

// ---------------------------------------------------------------------------------------
// tunables (compile time)
// ---------------------------------------------------------------------------------------
constexpr int SF_KPT = 4;       // wavevectors owned by one thread of the structure-factor kernel
constexpr int SF_TMAX = 512;    // max threads per CTA (structure-factor kernel)
constexpr int SF_AI = 64;       // max atoms one atom-group accumulates in fp32 before the fp64 flush
constexpr int F_THREADS = 256;  // threads per CTA (force kernel)
constexpr int F_KCHUNK = 2048;  // wavevectors staged in shared memory at a time (force kernel)
constexpr int FIN_KB = 32;      // wavevectors per CTA (finalise kernel)
constexpr int FIN_SL = 32;      // row slices per wavevector (finalise kernel)

constexpr double TWO32 = 4294967296.0;
constexpr double MAGIC = 6755399441055744.0;  // 2^52 + 2^51: low word of (d + MAGIC) = rint(d) mod 2^32
constexpr double PI_D = 3.14159265358979323846264338327950288;

// fl(2^-32 / fl(1/2pi)): sin.approx multiplies its argument by fl(1/2pi) = 0.15915493667125701904
// (FMUL.RZ) before MUFU; this constant makes that product equal 2^-32 * phase to within 2^-25.
__device__ __forceinline__ float phase_scale() { return (float)(1.0 / (TWO32 * 0.15915493667125701904)); }

__device__ __forceinline__ uint32_t to_turns(float x, double two32_over_L) {
    // round(x * 2^32 / L) mod 2^32, exact for |x / L| < 2^19
    return (uint32_t)__double2loint(fma((double)x, two32_over_L, MAGIC));
}

__device__ __forceinline__ float fast_sin(float x) {
    float r;
    asm("sin.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float fast_cos(float x) {
    float r;
    asm("cos.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// ---------------------------------------------------------------------------------------
// SF kernel -- Algorithm 1 steps 2+3 fused, Eq. (2.9) P:117.
//
// Mapping: a thread OWNS SF_KPT wavevectors (their m in registers) and one of `ng` atom
// groups; the CTA streams its contiguous atom range through shared memory in tiles of
// ng * ai atoms (already converted to fixed-point turns), group g reading atoms g, g+ng, ...
// as a shared-memory broadcast.  The N x P array of Fourier modes the paper materialises
// before its Reduce-by-Key never exists; neither does any cross-lane reduction:
// each thread sums its own (cos, sin) in fp32 over at most SF_AI atoms, then in fp64.
// The `ng` groups are combined through shared memory in group order and one fp64 row of P
// complex partials per CTA goes to global memory.  No atomics anywhere.
// ---------------------------------------------------------------------------------------
struct SfParams {
    const float4* xyzq;
    int64_t N;
    const int4* kvec;  // [P] {mx, my, mz, 0}
    double2* part;     // [gridDim.x][P]
    double two32_over_L;
    int32_t P;
    int32_t gs;    // threads per atom group in this CTA = k-slots / SF_KPT
    int32_t ng;    // atom groups per CTA
    int32_t ai;    // atoms per group per tile (<= SF_AI); tile = ng * ai atoms <= 2 * blockDim.x
};

__device__ __forceinline__ uint4 convert_atom(float4 a, double s) {
    uint4 r;
    r.x = to_turns(a.x, s);
    r.y = to_turns(a.y, s);
    r.z = to_turns(a.z, s);
    r.w = __float_as_uint(a.w);
    return r;
}

__global__ void __launch_bounds__(SF_TMAX, 1) sf_kernel(const SfParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint4* tile = reinterpret_cast<uint4*>(smem_raw);
    const int tid = threadIdx.x, T = blockDim.x;
    const int tile_atoms = p.ng * p.ai;
    const bool active = tid < p.gs * p.ng;
    const int g = active ? tid / p.gs : 0;
    const int j = active ? tid - g * p.gs : 0;
    const int kbase = (blockIdx.y * p.gs + j) * SF_KPT;

    int mx[SF_KPT], my[SF_KPT], mz[SF_KPT];
#pragma unroll
    for (int r = 0; r < SF_KPT; ++r) {
        int4 m = make_int4(0, 0, 0, 0);
        if (kbase + r < p.P) m = __ldg(&p.kvec[kbase + r]);
        mx[r] = m.x; my[r] = m.y; mz[r] = m.z;
    }
    float c[SF_KPT], s[SF_KPT];
    double cd[SF_KPT], sd[SF_KPT];
#pragma unroll
    for (int r = 0; r < SF_KPT; ++r) { c[r] = s[r] = 0.f; cd[r] = sd[r] = 0.0; }

    const int64_t lo = (p.N * (int64_t)blockIdx.x) / gridDim.x;
    const int64_t hi = (p.N * (int64_t)(blockIdx.x + 1)) / gridDim.x;
    const float K = phase_scale();
    const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);

    // prologue: first tile -> buffer 0
    {
        int64_t i0 = lo + tid, i1 = i0 + T;
        float4 a0 = (tid < tile_atoms && i0 < hi) ? __ldg(&p.xyzq[i0]) : zero4;
        float4 a1 = (tid + T < tile_atoms && i1 < hi) ? __ldg(&p.xyzq[i1]) : zero4;
        if (tid < tile_atoms) tile[tid] = convert_atom(a0, p.two32_over_L);
        if (tid + T < tile_atoms) tile[tid + T] = convert_atom(a1, p.two32_over_L);
    }
    __syncthreads();

    int cur = 0;
    for (int64_t t0 = lo; t0 < hi; t0 += tile_atoms) {
        // prefetch the next tile into registers (zero charge beyond the range: contributes 0)
        const int64_t n0 = t0 + tile_atoms + tid, n1 = n0 + T;
        float4 a0 = (tid < tile_atoms && n0 < hi) ? __ldg(&p.xyzq[n0]) : zero4;
        float4 a1 = (tid + T < tile_atoms && n1 < hi) ? __ldg(&p.xyzq[n1]) : zero4;

        const int64_t cnt = (hi - t0 < tile_atoms) ? (hi - t0) : tile_atoms;
        const int n_ai = (int)((cnt + p.ng - 1) / p.ng);  // <= p.ai; uniform over the CTA
        const uint4* src = tile + cur * tile_atoms + g;
#pragma unroll 2
        for (int a = 0; a < n_ai; ++a) {
            const uint4 at = src[a * p.ng];
            const float q = __uint_as_float(at.w);
#pragma unroll
            for (int r = 0; r < SF_KPT; ++r) {
                const uint32_t ph = (uint32_t)mx[r] * at.x + (uint32_t)my[r] * at.y + (uint32_t)mz[r] * at.z;
                const float x = (float)(int32_t)ph * K;
                c[r] = fmaf(q, fast_cos(x), c[r]);
                s[r] = fmaf(q, fast_sin(x), s[r]);
            }
        }
#pragma unroll
        for (int r = 0; r < SF_KPT; ++r) {
            cd[r] += (double)c[r]; sd[r] += (double)s[r];
            c[r] = 0.f; s[r] = 0.f;
        }
        // stage the prefetched tile into the other buffer
        uint4* dst = tile + (cur ^ 1) * tile_atoms;
        if (tid < tile_atoms) dst[tid] = convert_atom(a0, p.two32_over_L);
        if (tid + T < tile_atoms) dst[tid + T] = convert_atom(a1, p.two32_over_L);
        __syncthreads();
        cur ^= 1;
    }

    // combine the atom groups in group order, one fp64 row per CTA
    double2* red = reinterpret_cast<double2*>(smem_raw);
    const int kslots = p.gs * SF_KPT;
    __syncthreads();
    if (active) {
#pragma unroll
        for (int r = 0; r < SF_KPT; ++r) red[g * kslots + j * SF_KPT + r] = make_double2(cd[r], sd[r]);
    }
    __syncthreads();
    for (int idx = tid; idx < kslots; idx += T) {
        const int k = blockIdx.y * kslots + idx;
        if (k < p.P) {
            double re = 0.0, im = 0.0;
            for (int gg = 0; gg < p.ng; ++gg) {
                const double2 v = red[gg * kslots + idx];
                re += v.x; im += v.y;
            }
            p.part[(int64_t)blockIdx.x * p.P + k] = make_double2(re, im);
        }
    }
}

// ---------------------------------------------------------------------------------------
// FIN kernel -- second pass of the reduction and the per-k force coefficients.
//
// rho_l = sum over the SF kernel's per-CTA rows in a FIXED order (row slices sl, sl+32, ...
// summed sequentially, then the 32 slice sums sequentially), so rho is bitwise reproducible.
// Then, with w_l the sample weight (S/P of Eq. 2.12 unless the caller gave weights):
//   Im(e^{-i phi} rho) = |rho| sin(theta - phi),  theta = arg rho,
// so Eq. (2.12) becomes  F_i = q_i sum_l G_l sin(2 pi (theta_l - m_l . s_i))  with
//   G_l = -(4 pi w_l / V) (k_l / k_l^2) |rho_l| = -(2 w_l / L^2) (m_l / |m_l|^2) |rho_l|
// and the force kernel needs ONE special-function evaluation per (atom, k) instead of two.
// Energy weights (2nd term of Eq. 2.8): e_l = (2 pi w_l / V) / k_l^2 = w_l / (2 pi L |m_l|^2).
// ---------------------------------------------------------------------------------------
struct FinParams {
    const double2* part;  // [nrows][P] (nrows = 1 and part = caller's rho for rbe_set_rho)
    int32_t nrows;
    int32_t P;
    const int4* kvec;     // [P]
    const double* w;      // [P] or nullptr -> w_uniform
    double w_uniform;     // S / P
    double L;
    double2* rho;         // [P] out
    double2* rho_user;    // [P] out, or nullptr
    int4* ka;             // [P] out {-mx, -my, -mz, theta in 2^-32 turns}
    float4* kb;           // [P] out {Gx, Gy, Gz, E = e_l |rho_l|}
    double* uk;           // [P] out e_l |rho_l|^2
};

__global__ void __launch_bounds__(FIN_KB * FIN_SL) fin_kernel(const FinParams p) {
    __shared__ double2 sl_sum[FIN_SL][FIN_KB];
    const int kk = threadIdx.x % FIN_KB, sl = threadIdx.x / FIN_KB;
    const int k = blockIdx.x * FIN_KB + kk;
    double re = 0.0, im = 0.0;
    if (k < p.P) {
        for (int row = sl; row < p.nrows; row += FIN_SL) {
            const double2 v = p.part[(int64_t)row * p.P + k];
            re += v.x; im += v.y;
        }
    }
    sl_sum[sl][kk] = make_double2(re, im);
    __syncthreads();
    if (sl != 0 || k >= p.P) return;
    re = 0.0; im = 0.0;
#pragma unroll 1
    for (int t = 0; t < FIN_SL; ++t) { re += sl_sum[t][kk].x; im += sl_sum[t][kk].y; }

    const int4 m = p.kvec[k];
    const double w = p.w ? p.w[k] : p.w_uniform;
    const double m2 = (double)m.x * m.x + (double)m.y * m.y + (double)m.z * m.z;
    const double mag = sqrt(re * re + im * im);
    const double theta = atan2(im, re) * (1.0 / (2.0 * PI_D));        // turns, [-1/2, 1/2]
    const double gs = -2.0 * w / (p.L * p.L * m2) * mag;
    const double el = w / (2.0 * PI_D * p.L * m2);
    p.rho[k] = make_double2(re, im);
    if (p.rho_user) p.rho_user[k] = make_double2(re, im);
    p.ka[k] = make_int4(-m.x, -m.y, -m.z, __double2loint(fma(theta, TWO32, MAGIC)));
    p.kb[k] = make_float4((float)(gs * m.x), (float)(gs * m.y), (float)(gs * m.z), (float)(el * mag));
    p.uk[k] = el * mag * mag;
}

// U = sum_l uk[l] in a fixed order (thread-strided partials, then a fixed tree).
__global__ void __launch_bounds__(256) energy_kernel(const double* uk, int32_t P, double* U) {
    __shared__ double sh[256];
    double a = 0.0;
    for (int k = threadIdx.x; k < P; k += 256) a += uk[k];
    sh[threadIdx.x] = a;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) *U = sh[0];
}

// ---------------------------------------------------------------------------------------
// F kernel -- Algorithm 1 step 4, Eq. (2.12) P:131.
//
// Mapping: a thread owns R atoms (coordinates as fixed-point turns in registers) and loops
// over the wavevectors, whose {-m, theta} and {G, E} records are broadcast from shared memory.
// Work is dealt to WARPS in units of 32 atoms, balanced over the whole grid, so that every
// SM sub-partition gets the same number of (atom, k) pairs to within one unit.
// Per pair: 3 IMAD (phase), I2F, 2 FMUL, 1 MUFU.SIN, 3 FFMA (+ MUFU.COS, FFMA with energy).
// ---------------------------------------------------------------------------------------
struct FParams {
    const float4* xyzq;
    float4* force;
    int64_t N;
    const int4* ka;
    const float4* kb;
    double two32_over_L;
    int32_t P;
};

template <int R, bool ENERGY, bool ACCUM>
__device__ __forceinline__ void f_units(const FParams& p, const int4* s_ka, const float4* s_kb,
                                        int nk, int64_t unit0, int lane) {
    uint32_t sx[R], sy[R], sz[R];
    float q[R], fx[R], fy[R], fz[R], en[R];
    const float K = phase_scale();
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int64_t i = (unit0 + r) * 32 + lane;
        float4 a = make_float4(0.f, 0.f, 0.f, 0.f);
        if (i < p.N) a = __ldg(&p.xyzq[i]);
        sx[r] = to_turns(a.x, p.two32_over_L);
        sy[r] = to_turns(a.y, p.two32_over_L);
        sz[r] = to_turns(a.z, p.two32_over_L);
        q[r] = a.w;
        fx[r] = fy[r] = fz[r] = en[r] = 0.f;
    }
#pragma unroll 2
    for (int k = 0; k < nk; ++k) {
        const int4 a = s_ka[k];
        const float4 b = s_kb[k];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const uint32_t ph = (uint32_t)a.x * sx[r] + ((uint32_t)a.y * sy[r] + ((uint32_t)a.z * sz[r] + (uint32_t)a.w));
            const float x = (float)(int32_t)ph * K;
            const float sn = fast_sin(x);
            fx[r] = fmaf(sn, b.x, fx[r]);
            fy[r] = fmaf(sn, b.y, fy[r]);
            fz[r] = fmaf(sn, b.z, fz[r]);
            if (ENERGY) en[r] = fmaf(fast_cos(x), b.w, en[r]);
        }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int64_t i = (unit0 + r) * 32 + lane;
        if (i < p.N) {
            float4 o = make_float4(q[r] * fx[r], q[r] * fy[r], q[r] * fz[r], ENERGY ? q[r] * en[r] : 0.f);
            if (ACCUM) {
                const float4 prev = p.force[i];
                o.x += prev.x; o.y += prev.y; o.z += prev.z; o.w += prev.w;
            }
            p.force[i] = o;
        }
    }
}

template <int R, bool ENERGY>
__global__ void __launch_bounds__(F_THREADS) f_kernel(const FParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nkmax = p.P < F_KCHUNK ? p.P : F_KCHUNK;
    int4* s_ka = reinterpret_cast<int4*>(smem_raw);
    float4* s_kb = reinterpret_cast<float4*>(smem_raw + (size_t)nkmax * sizeof(int4));
    const int lane = threadIdx.x & 31;
    const int64_t nwarps = (int64_t)gridDim.x * (F_THREADS / 32);
    const int64_t gw = (int64_t)blockIdx.x * (F_THREADS / 32) + (threadIdx.x >> 5);
    const int64_t units = (p.N + 31) / 32;
    const int64_t u0 = units * gw / nwarps, u1 = units * (gw + 1) / nwarps;

    for (int k0 = 0; k0 < p.P; k0 += F_KCHUNK) {
        const int nk = (p.P - k0 < F_KCHUNK) ? (p.P - k0) : F_KCHUNK;
        if (k0 > 0) __syncthreads();
        for (int t = threadIdx.x; t < nk; t += F_THREADS) {
            s_ka[t] = p.ka[k0 + t];
            s_kb[t] = p.kb[k0 + t];
        }
        __syncthreads();
        int64_t u = u0;
        if (k0 == 0) {
            for (; u + R <= u1; u += R) f_units<R, ENERGY, false>(p, s_ka, s_kb, nk, u, lane);
            for (; u < u1; ++u) f_units<1, ENERGY, false>(p, s_ka, s_kb, nk, u, lane);
        } else {
            for (; u + R <= u1; u += R) f_units<R, ENERGY, true>(p, s_ka, s_kb, nk, u, lane);
            for (; u < u1; ++u) f_units<1, ENERGY, true>(p, s_ka, s_kb, nk, u, lane);
        }
    }
}

}  // namespace rbe
