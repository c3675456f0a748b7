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
//
// Measured on B200 (csrc/pipe_probe.cu, profiles/): MUFU 16 lanes/SM/clk, IMAD and I2FP 64,
// FFMA 128; a MUFU also costs ~3 issue slots.  Both hot kernels are bound by MUFU + issue.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace rbe {

// ---------------------------------------------------------------------------------------
// tunables (compile time)
// ---------------------------------------------------------------------------------------
// (each may be overridden with -DRBE_<NAME>=value when sweeping; the defaults are the tuned ones)
#ifndef RBE_SF_TMAX
#define RBE_SF_TMAX 1024
#endif
#ifndef RBE_SF_CTAS_PER_SM
#define RBE_SF_CTAS_PER_SM 1
#endif
#ifndef RBE_SF_TILE_MAX
#define RBE_SF_TILE_MAX 4096
#endif
#ifndef RBE_F_THREADS
#define RBE_F_THREADS 512
#endif
#ifndef RBE_F_CTAS_PER_SM
#define RBE_F_CTAS_PER_SM 2
#endif
#ifndef RBE_SF_KPT
#define RBE_SF_KPT 4
#endif
constexpr int SF_KPT = RBE_SF_KPT;   // wavevectors owned by one thread of the structure-factor kernel
constexpr int SF_TMAX = RBE_SF_TMAX;    // max threads per CTA (structure-factor kernel): <= 64 registers
constexpr int SF_CTAS_PER_SM = RBE_SF_CTAS_PER_SM;
constexpr int SF_TILE_MAX = RBE_SF_TILE_MAX; // max atoms staged in shared memory at a time (structure-factor kernel)
#ifndef RBE_SF_STAGE_UNROLL
#define RBE_SF_STAGE_UNROLL 4
#endif
constexpr int SF_STAGE_UNROLL = RBE_SF_STAGE_UNROLL;   // unroll factor of the two staging loops over 32-atom windows
constexpr int SF_DEPTH = 64;     // max atoms a thread accumulates in fp32 before the fp64 flush
constexpr int F_THREADS = RBE_F_THREADS;   // threads per CTA (force kernel)
constexpr int F_CTAS_PER_SM = RBE_F_CTAS_PER_SM;
constexpr int F_RMAX = 4;        // max atoms per thread per pass (force kernel)
constexpr int F_KCHUNK = 2048;   // wavevectors staged in shared memory at a time (force kernel)
#ifndef RBE_SF_RED_GROUP
#define RBE_SF_RED_GROUP 16
#endif
constexpr int SF_RED_GROUP = RBE_SF_RED_GROUP; // CTAs per group in the two-level reduction of the per-CTA rows

constexpr double TWO32 = 4294967296.0;
constexpr double MAGIC = 6755399441055744.0;  // 2^52 + 2^51: low word of (d + MAGIC) = rint(d) mod 2^32
constexpr double PI_D = 3.14159265358979323846264338327950288;
constexpr uint32_t QUARTER_TURN = 0x40000000u;
constexpr unsigned FULL_MASK = 0xffffffffu;

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
__device__ __forceinline__ float phase_to_arg(uint32_t ph, float K) { return (float)(int32_t)ph * K; }

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gmem_src) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// Programmatic dependent launch (PDL): the force kernel may start while the structure-factor
// kernel drains; it waits here before touching anything that kernel writes.
__device__ __forceinline__ void grid_dependency_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void grid_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// ---------------------------------------------------------------------------------------
// Per-k force coefficients, computed in fp64 from the reduced rho.
//
// With w_l the sample weight (S/P of Eq. 2.12 unless the caller gave weights):
//   Im(e^{-i phi} rho) = |rho| sin(theta - phi),  theta = arg rho,
// so Eq. (2.12) becomes  F_i = q_i sum_l G_l sin(2 pi (theta_l - m_l . s_i))  with
//   G_l = -(4 pi w_l / V) (k_l / k_l^2) |rho_l| = -(2 w_l / L^2) (m_l / |m_l|^2) |rho_l|
// and the force kernel needs ONE special-function evaluation per (atom, k) instead of two.
// Energy weights (2nd term of Eq. 2.8): e_l = (2 pi w_l / V) / k_l^2 = w_l / (2 pi L |m_l|^2).
// Every force CTA builds the records for its shared-memory tile itself (a few hundred fp64
// operations per k, in parallel over the CTAs), so the serial tail of the structure-factor
// kernel is only the reduction.
// ---------------------------------------------------------------------------------------
constexpr int MAX_WORLD = 16;   // ranks (GPUs) one fused exchange can span

// Fused multi-GPU exchange of the structure factors.  Every rank
// owns an exchange buffer that its peers can write (NVLink peer mapping):
//   slots [2][world][P] double2   -- slot (parity, r) = rank r's partial rho of a step with that parity
//   flags [2][world]    uint32    -- epoch of the step whose partial is complete in that slot
// The structure-factor kernel of rank r PUSHES its partial into slot (parity, r) of every rank and
// then releases the flag; the consumers (force / energy kernels) of every rank WAIT for all `world`
// flags of the step and add the slots in rank order, so every rank gets the bitwise identical
// global rho without a collective call or an extra launch.  Two parities: a rank can run at most
// one step ahead of a peer that is still reading (it cannot finish step n+1 before that peer has
// pushed step n+1, which the peer does only after its own step-n force kernel).
struct XchPush {                  // writer side (structure-factor kernel)
    int32_t world;                // 0: no exchange
    uint32_t epoch;
    double2* slot[MAX_WORLD];     // slot (parity, my rank) in rank r's buffer
    uint32_t* flag[MAX_WORLD];    // flag (parity, my rank) in rank r's buffer
};
struct XchPull {                  // reader side (force / energy kernels): this rank's own buffer
    int32_t world;
    uint32_t epoch;
    const double2* slots;         // [world][P] of this step's parity
    const uint32_t* flags;        // [world]
    int32_t* error;               // set to 1 if a flag did not arrive within XCH_TIMEOUT_NS
};
constexpr unsigned long long XCH_TIMEOUT_NS = 10ull * 1000 * 1000 * 1000;

__device__ __forceinline__ uint32_t ld_acquire_sys(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_sys(uint32_t* p, uint32_t v) {
    asm volatile("st.release.sys.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ unsigned long long global_timer_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// All threads of the CTA call this; returns when every rank's partial of this step has arrived.
__device__ __forceinline__ void xch_wait(const XchPull& x) {
    if (x.world < 1) return;
    if ((int)threadIdx.x < x.world) {
        const unsigned long long t0 = global_timer_ns();
        while ((int32_t)(ld_acquire_sys(&x.flags[threadIdx.x]) - x.epoch) < 0) {
            if (global_timer_ns() - t0 > XCH_TIMEOUT_NS) { *x.error = 1; break; }   // never hang the GPU
            __nanosleep(100);
        }
    }
    __syncthreads();
}

struct KTable {
    const int4* kvec;     // [P] {mx, my, mz, 0}
    const double* w;      // [P] or nullptr -> w_uniform
    const double2* rho;   // [P] (this rank's atoms only when an exchange is configured)
    double w_uniform;     // S / P
    double L;
    int32_t P;
    XchPull xch;          // world > 0: rho(k) = sum over ranks, in rank order, of the exchange slots
};

__device__ __forceinline__ double2 k_rho(const KTable& t, int k) {
    if (t.xch.world < 1) return t.rho[k];
    double re = 0.0, im = 0.0;
    for (int r = 0; r < t.xch.world; ++r) {
        const double2 v = __ldcg(&t.xch.slots[(int64_t)r * t.P + k]);   // written by a peer: not through L1
        re += v.x; im += v.y;
    }
    return make_double2(re, im);
}

__device__ __forceinline__ void k_record(const KTable& t, int k, int4& ka, float4& kb) {
    const int4 m = t.kvec[k];
    const double2 r = k_rho(t, k);
    const double w = t.w ? t.w[k] : t.w_uniform;
    const double m2 = (double)m.x * m.x + (double)m.y * m.y + (double)m.z * m.z;
    const double mag = sqrt(r.x * r.x + r.y * r.y);
    const double theta = atan2(r.y, r.x) * (1.0 / (2.0 * PI_D));      // turns, [-1/2, 1/2]
    const double gs = -2.0 * w / (t.L * t.L * m2) * mag;
    const double el = w / (2.0 * PI_D * t.L * m2);
    ka = make_int4(-m.x, -m.y, -m.z, __double2loint(fma(theta, TWO32, MAGIC)));   // {-m, theta in 2^-32 turns}
    kb = make_float4((float)(gs * m.x), (float)(gs * m.y), (float)(gs * m.z), (float)(el * mag));  // {G, e_l |rho_l|}
}

// U = sum_l e_l |rho_l|^2 in a fixed order (thread-strided partials, then a fixed tree).
__global__ void __launch_bounds__(256) energy_kernel(const KTable t, int32_t P, double* U) {
    __shared__ double sh[256];
    xch_wait(t.xch);
    double a = 0.0;
    for (int k = threadIdx.x; k < P; k += 256) {
        const int4 m = t.kvec[k];
        const double2 r = k_rho(t, k);
        const double w = t.w ? t.w[k] : t.w_uniform;
        const double m2 = (double)m.x * m.x + (double)m.y * m.y + (double)m.z * m.z;
        a += w / (2.0 * PI_D * t.L * m2) * (r.x * r.x + r.y * r.y);
    }
    sh[threadIdx.x] = a;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x == 0) *U = sh[0];
}

// k-space virial (reading Q19): W_ab = sum_l e_l |rho_l|^2 [delta_ab - 2 m_a m_b / |m|^2 (1 + pi^2 |m|^2 / (alpha L^2))],
// the strain derivative of the second term of Eq. (2.8) with the weights of Eq. (2.12); k_a k_b / k^2 =
// m_a m_b / |m|^2 and k^2 / 4 alpha = pi^2 |m|^2 / (alpha L^2).  W[0..5] = xx, yy, zz, xy, xz, yz.  Fixed order.
__global__ void __launch_bounds__(256) virial_kernel(const KTable t, int32_t P, double alpha, double* W) {
    __shared__ double sh[6][256];
    xch_wait(t.xch);
    double a[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    for (int k = threadIdx.x; k < P; k += 256) {
        const int4 m = t.kvec[k];
        const double2 r = k_rho(t, k);
        const double w = t.w ? t.w[k] : t.w_uniform;
        const double mx = m.x, my = m.y, mz = m.z;
        const double m2 = mx * mx + my * my + mz * mz;
        const double u = w / (2.0 * PI_D * t.L * m2) * (r.x * r.x + r.y * r.y);       // e_l |rho_l|^2
        const double f = 2.0 / m2 * (1.0 + PI_D * PI_D * m2 / (alpha * t.L * t.L));
        a[0] += u * (1.0 - f * mx * mx); a[1] += u * (1.0 - f * my * my); a[2] += u * (1.0 - f * mz * mz);
        a[3] += u * (-f * mx * my);      a[4] += u * (-f * mx * mz);      a[5] += u * (-f * my * mz);
    }
#pragma unroll
    for (int c = 0; c < 6; ++c) sh[c][threadIdx.x] = a[c];
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if ((int)threadIdx.x < s)
#pragma unroll
            for (int c = 0; c < 6; ++c) sh[c][threadIdx.x] += sh[c][threadIdx.x + s];
        __syncthreads();
    }
    if (threadIdx.x < 6) W[threadIdx.x] = sh[threadIdx.x][0];
}

// ---------------------------------------------------------------------------------------
// Second pass of the structure-factor reduction, inside the SF kernel (no extra launch).
//
// The per-CTA rows are summed in a FIXED order by a two-level tree: CTAs form groups of
// `group_size` consecutive blockIdx.x; the last CTA of a group to finish (atomicInc ticket)
// sums that group's rows into one group row, and the last group to finish sums the group
// rows into rho.  Which CTA does the summing depends on timing; the order of the additions
// does not, so rho is bitwise reproducible.  Tickets wrap to zero by themselves.
// ---------------------------------------------------------------------------------------
struct RedParams {
    double2* part;        // [gridDim.x][P] per-CTA rows
    double2* grow;        // [ngroups][P] group rows
    double2* rho;         // [P] out
    double2* rho_user;    // [P] out, or nullptr
    unsigned int* tickets;  // [ngroups + 1], zero-initialised
    int32_t group_size, ngroups;
    XchPush xch;          // world > 0: push rho to every rank's exchange buffer after the second pass
};

// dst[k] = sum_{row} src[row][k]: row slices sl, sl+nsl, ... sequentially, then the slices in order
__device__ __forceinline__ void reduce_rows(const double2* src, int nrows, int P, double2* dst, double2* dst2,
                                            double2* scratch, int tid, int nt) {
    const int kc = P < nt ? P : nt;       // wavevectors per chunk
    const int nsl = nt / kc;              // row slices per wavevector (>= 1)
    const int kk = tid % kc, sl = tid / kc;
    for (int k0 = 0; k0 < P; k0 += kc) {
        const int k = k0 + kk;
        double re = 0.0, im = 0.0;
        if (sl < nsl && k < P) {
#pragma unroll 8
            for (int row = sl; row < nrows; row += nsl) {
                const double2 v = __ldcg(&src[(int64_t)row * P + k]);
                re += v.x; im += v.y;
            }
        }
        if (sl < nsl) scratch[sl * kc + kk] = make_double2(re, im);
        __syncthreads();
        if (sl == 0 && k < P) {
            re = 0.0; im = 0.0;
#pragma unroll 1
            for (int t = 0; t < nsl; ++t) { re += scratch[t * kc + kk].x; im += scratch[t * kc + kk].y; }
            dst[k] = make_double2(re, im);
            if (dst2) dst2[k] = make_double2(re, im);
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------
// SF kernel -- Algorithm 1 steps 2+3 fused, Eq. (2.9) P:117.
//
// Mapping: a thread OWNS SF_KPT wavevectors (their m in registers) and one of `ng` atom
// groups.  The CTA streams its contiguous atom range through shared memory in tiles of
// blockDim.x atoms (cp.async prefetch of the raw float4 records); the N x P array of Fourier
// modes the paper materialises before its Reduce-by-Key never exists, and there is no
// cross-lane reduction: each thread sums its own (cos, sin) in fp32 over at most ~SF_DEPTH
// atoms, then in fp64 (shared-memory accumulators).  Groups are combined in group order and
// one fp64 row of P complex partials per CTA goes to global memory.  No atomics on data.
//
// Equal-|q| pairing (what makes this kernel 3 MUFU per TWO pairs instead of 4).  For two atoms
// with q_2 = +-q_1 and turns S_1, S_2 let S_d = (S_1 - S_2)/2, S_a = S_2 + S_d.  Then exactly
//   q_1 e^{i phi_1} + q_2 e^{i phi_2} = 2 q_1 cos(2 pi m.S_d - o) e^{i (2 pi m.S_a + o)},
// o = 0 for equal charges, a quarter turn for opposite ones (2i sin d = 2 cos(d - pi/2) e^{i pi/2}).
// While staging a tile each warp matches the 32 atoms of its window by |q| bit pattern
// (MATCH.ANY) and emits pair records {S_a, o}{S_d, 2 q_1} and single records {S, q} for the
// leftovers, so ANY charge assignment is handled (all-distinct charges fall back to 2 MUFU per
// pair).  MD systems have a handful of distinct charge magnitudes, so nearly all atoms pair up.
// Compaction of the records is by warp counts + a prefix scan: deterministic order.
//
// The last CTAs to finish (atomicInc tickets; data order never depends on them) run the second
// pass: the fixed-order two-level sum of the per-CTA rows into rho (reduce_rows), and, with a
// multi-GPU exchange configured, the push of rho into every rank's exchange buffer.
// ---------------------------------------------------------------------------------------
struct SfParams {
    const float4* xyzq;
    int64_t N;
    const int4* kvec;  // [P] {mx, my, mz, 0}
    double2* part;     // [gridDim.x][P]
    double two32_over_L;
    int32_t P;
    int32_t gs;        // threads per atom group in this CTA = k-slots / SF_KPT
    int32_t ng;        // atom groups per CTA
    int32_t tile_atoms;   // atoms staged per tile: a multiple of 32, <= SF_TILE_MAX
    int32_t flush_every;  // tiles between fp64 flushes (keeps the fp32 depth <= ~SF_DEPTH atoms)
    int32_t pairing;      // bit 0: pair equal charges, bit 1: pair opposite charges (3 = both)
    int32_t accumulate;   // add this launch's per-CTA rows to what `part` holds (chunked host step: one launch per chunk)
    int32_t finalise;     // run the second pass (rows -> rho) at the end of this launch
    RedParams red;
#ifdef RBE_SF_PROFILE
    long long* prof;      // [gridDim.x][64] globaltimer stamps of thread 0 (sweep builds only)
#endif
};

#ifdef RBE_SF_PROFILE
#define RBE_STAMP() do { if (tid == 0 && prof_n < 64) { long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); p.prof[blockIdx.x * 64 + prof_n++] = t_; } } while (0)
#else
#define RBE_STAMP() do { } while (0)
#endif

// acc points at this thread's slot of component 0; component r lives `stride` entries further
// (layout [SF_KPT][blockDim.x]: conflict-free).
__device__ __forceinline__ void sf_flush(double2* acc, int stride, float (&c)[SF_KPT], float (&s)[SF_KPT]) {
#pragma unroll
    for (int r = 0; r < SF_KPT; ++r) {
        double2 v = acc[r * stride];
        v.x += (double)c[r]; v.y += (double)s[r];
        acc[r * stride] = v;
        c[r] = 0.f; s[r] = 0.f;
    }
}

// Classification of one 32-atom window (lane = atom) by charge: `leader` lanes own a pair record
// (with the next lane of equal |q|, `partner`), `single` lanes a single record.
struct SfWindow {
    uint32_t lmask, smask;
    int partner;
    bool leader, single;
};
__device__ __forceinline__ SfWindow sf_classify(uint32_t qbits, bool in_range, int pairing, int lane) {
    SfWindow w;
    const uint32_t key = qbits & ((pairing & 3) == 3 ? 0x7fffffffu : 0xffffffffu);
    const bool valid = in_range && (qbits & 0x7fffffffu) != 0u;   // zero charges contribute nothing: dropped
    const uint32_t vmask = __ballot_sync(FULL_MASK, valid);
    const uint32_t peers = (pairing & 3) ? (__match_any_sync(FULL_MASK, key) & vmask) : (valid ? 1u << lane : 0u);
    const int rank = __popc(peers & ((1u << lane) - 1u));
    const uint32_t higher = (peers >> lane) >> 1;                  // peers above this lane
    w.leader = valid && !(rank & 1) && higher != 0u;
    w.single = valid && !(rank & 1) && higher == 0u;
    w.lmask = __ballot_sync(FULL_MASK, w.leader);
    w.smask = __ballot_sync(FULL_MASK, w.single);
    w.partner = w.leader ? lane + __ffs(higher) : lane;
    return w;
}

template <bool DEEP>
__global__ void __launch_bounds__(SF_TMAX, SF_CTAS_PER_SM) sf_kernel(const SfParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = T >> 5;
    const int TA = p.tile_atoms;                                      // multiple of 32, <= SF_TILE_MAX
    float4* raw = reinterpret_cast<float4*>(smem_raw);               // [TA] raw atom records of the tile
    uint4* arena = reinterpret_cast<uint4*>(smem_raw) + TA;          // [TA] pair records from the front, singles from the back
    double2* acc_all = reinterpret_cast<double2*>(arena + TA);       // [SF_KPT][T] fp64 accumulators
    constexpr int WIN_MAX = 128;   // the one-warp scan below covers 4 windows per lane
    static_assert(SF_TILE_MAX / 32 <= WIN_MAX, "tile too large for the window scan");
    __shared__ uint32_t wcount[WIN_MAX], wbase[WIN_MAX + 1];
    __shared__ uint16_t roles[SF_TILE_MAX];
    __shared__ uint32_t s_last;

    const bool active = tid < p.gs * p.ng;
    const int g = active ? tid / p.gs : (1 << 28);  // inactive threads: group index past every list -> empty loops
    const int j = active ? tid % p.gs : 0;
    const int kbase = (blockIdx.y * p.gs + j) * SF_KPT;
    double2* acc = acc_all + tid;

    int mx[SF_KPT], my[SF_KPT], mz[SF_KPT];
    float c[SF_KPT], s[SF_KPT];
#pragma unroll
    for (int r = 0; r < SF_KPT; ++r) {
        int4 m = make_int4(0, 0, 0, 0);
        if (active && kbase + r < p.P) m = __ldg(&p.kvec[kbase + r]);
        mx[r] = m.x; my[r] = m.y; mz[r] = m.z;
        c[r] = s[r] = 0.f;
        acc[r * T] = make_double2(0.0, 0.0);
    }

    // this CTA's atom range, aligned to 32-atom windows
    const int64_t units = (p.N + 31) >> 5;
    const int64_t lo = (units * blockIdx.x / gridDim.x) << 5;
    int64_t hi = (units * (blockIdx.x + 1) / gridDim.x) << 5;
    if (hi > p.N) hi = p.N;
    const float K = phase_scale();
    const uint32_t lt_mask = (1u << lane) - 1u;

    // a short first tile gets the MUFU-bound loop going early; later tiles are full size
    int tl = (TA >> 7) << 5;
    if (tl < 32) tl = 32;
    for (int i = tid; i < tl && lo + i < hi; i += T) cp_async16(&raw[i], &p.xyzq[lo + i]);
    int since_flush = 0;
#ifdef RBE_SF_PROFILE
    int prof_n = 0;
#endif
    RBE_STAMP();

    for (int64_t t0 = lo; t0 < hi; t0 += tl, tl = TA) {
        const int cnt = (int)((hi - t0 < tl) ? (hi - t0) : tl);
        const int nwin = (cnt + 31) >> 5;
        cp_async_wait_all();
        __syncthreads();  // raw holds the tile; everyone is done with the previous arena
        RBE_STAMP();

        // ---- stage 1: per window (one warp each), classify by charge and count the records
#pragma unroll SF_STAGE_UNROLL
        for (int w = warp; w < nwin; w += nwarps) {
            const int idx = (w << 5) + lane;
            const uint32_t qb = idx < cnt ? __float_as_uint(raw[idx].w) : 0u;
            const SfWindow cw = sf_classify(qb, idx < cnt, p.pairing, lane);
            // role word: bits 0-4 partner lane, bit 5 leader, bit 6 single, bits 8.. index in the window's list
            roles[idx] = (uint16_t)(cw.partner | (cw.leader ? 32 : 0) | (cw.single ? 64 : 0) |
                                    (__popc((cw.leader ? cw.lmask : cw.smask) & lt_mask) << 8));
            if (lane == 0) wcount[w] = (uint32_t)__popc(cw.lmask) | ((uint32_t)__popc(cw.smask) << 16);
        }
        __syncthreads();
        // exclusive scan of the window counts (<= SF_TILE_MAX/32 = 128 of them) by one warp: record positions
        if (warp == 0) {
            uint32_t v[4], run = 0;
#pragma unroll
            for (int i = 0; i < 4; ++i) { v[i] = (4 * lane + i < nwin) ? wcount[4 * lane + i] : 0u; run += v[i]; }
            uint32_t incl = run;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t n = __shfl_up_sync(FULL_MASK, incl, d);
                if (lane >= d) incl += n;
            }
            uint32_t ex = incl - run;
#pragma unroll
            for (int i = 0; i < 4; ++i) { wbase[4 * lane + i] = ex; ex += v[i]; }
            if (lane == 31) wbase[WIN_MAX] = incl;
        }
        __syncthreads();
        const uint32_t total = wbase[WIN_MAX];
        const int np = (int)(total & 0xffffu), ns = (int)(total >> 16);

        // ---- stage 2: convert to turns and write the records at their scanned positions
#pragma unroll SF_STAGE_UNROLL
        for (int w = warp; w < nwin; w += nwarps) {
            const int idx = (w << 5) + lane;
            const uint32_t base = wbase[w];
            const float4 a = idx < cnt ? raw[idx] : make_float4(0.f, 0.f, 0.f, 0.f);
            const uint32_t role = roles[idx];
            const int partner = role & 31, e_in = role >> 8;
            const uint32_t Sx = to_turns(a.x, p.two32_over_L);
            const uint32_t Sy = to_turns(a.y, p.two32_over_L);
            const uint32_t Sz = to_turns(a.z, p.two32_over_L);
            const uint32_t Px = __shfl_sync(FULL_MASK, Sx, partner);
            const uint32_t Py = __shfl_sync(FULL_MASK, Sy, partner);
            const uint32_t Pz = __shfl_sync(FULL_MASK, Sz, partner);
            const uint32_t Pq = __shfl_sync(FULL_MASK, __float_as_uint(a.w), partner);
            if (role & 32) {
                // S_d = (S_1 - S_2) / 2 (arithmetic shift of the wrapped difference), S_a = S_2 + S_d
                const int e = (int)(base & 0xffffu) + e_in;
                const uint32_t dx = (uint32_t)((int32_t)(Sx - Px) >> 1);
                const uint32_t dy = (uint32_t)((int32_t)(Sy - Py) >> 1);
                const uint32_t dz = (uint32_t)((int32_t)(Sz - Pz) >> 1);
                // o: a quarter turn for opposite charges; plus half a turn on every other pair, which leaves
                // cos(d - o) e^{i(a + o)} unchanged but alternates the sign of the evaluated amplitude, so
                // the +1.7e-8 mean error of MUFU.COS (measured) cannot add up coherently over the pairs
                // (for single atoms it cancels by neutrality; the sum of pair amplitudes is not neutral)
                const uint32_t off = (((__float_as_uint(a.w) ^ Pq) >> 31) ? QUARTER_TURN : 0u) + ((uint32_t)e << 31);
                arena[2 * e] = make_uint4(Px + dx, Py + dy, Pz + dz, off);
                arena[2 * e + 1] = make_uint4(dx, dy, dz, __float_as_uint(2.0f * a.w));
            } else if (role & 64) {
                const int e = (int)(base >> 16) + e_in;
                arena[TA - 1 - e] = make_uint4(Sx, Sy, Sz, __float_as_uint(a.w));
            }
        }
        __syncthreads();  // records visible; raw fully consumed
        RBE_STAMP();

        // prefetch the next tile while this one is processed
        for (int i = tid; i < TA && t0 + tl + i < hi; i += T) cp_async16(&raw[i], &p.xyzq[t0 + tl + i]);

        // ---- accumulate: pair records g, g+ng, ... then single records g, g+ng, ...
        int depth = 0;
#pragma unroll 1
        for (int e = g; e < np; e += p.ng) {
            const uint4 ra = arena[2 * e];
            const uint4 rd = arena[2 * e + 1];
            const float w2 = __uint_as_float(rd.w);
#pragma unroll
            for (int r = 0; r < SF_KPT; ++r) {
                const uint32_t pa = (uint32_t)mx[r] * ra.x + ((uint32_t)my[r] * ra.y + ((uint32_t)mz[r] * ra.z + ra.w));
                const uint32_t pd = (uint32_t)mx[r] * rd.x + ((uint32_t)my[r] * rd.y + ((uint32_t)mz[r] * rd.z - ra.w));
                const float xa = phase_to_arg(pa, K);
                const float amp = w2 * fast_cos(phase_to_arg(pd, K));
                c[r] = fmaf(amp, fast_cos(xa), c[r]);
                s[r] = fmaf(amp, fast_sin(xa), s[r]);
            }
            if (DEEP) { depth += 2; if (depth >= SF_DEPTH) { sf_flush(acc, T, c, s); depth = 0; } }
        }
#pragma unroll 1
        for (int e = g; e < ns; e += p.ng) {
            const uint4 at = arena[TA - 1 - e];
            const float q = __uint_as_float(at.w);
#pragma unroll
            for (int r = 0; r < SF_KPT; ++r) {
                const uint32_t ph = (uint32_t)mx[r] * at.x + ((uint32_t)my[r] * at.y + (uint32_t)mz[r] * at.z);
                const float x = phase_to_arg(ph, K);
                c[r] = fmaf(q, fast_cos(x), c[r]);
                s[r] = fmaf(q, fast_sin(x), s[r]);
            }
            if (DEEP) { depth += 1; if (depth >= SF_DEPTH) { sf_flush(acc, T, c, s); depth = 0; } }
        }
        if (++since_flush >= p.flush_every) { sf_flush(acc, T, c, s); since_flush = 0; }
    }
    sf_flush(acc, T, c, s);
    RBE_STAMP();

    // let the dependent (force) kernel start launching; it waits for this grid's completion
    grid_launch_dependents();

    // combine the atom groups in group order, one fp64 row per CTA
    const int kslots = p.gs * SF_KPT;
    __syncthreads();
    for (int idx = tid; idx < kslots; idx += T) {
        const int k = blockIdx.y * kslots + idx;
        if (k < p.P) {
            double re = 0.0, im = 0.0;
            for (int gg = 0; gg < p.ng; ++gg) {
                const double2 v = acc_all[(idx % SF_KPT) * T + gg * p.gs + idx / SF_KPT];
                re += v.x; im += v.y;
            }
            double2* row = &p.part[(int64_t)blockIdx.x * p.P + k];
            if (p.accumulate) { const double2 old = *row; re += old.x; im += old.y; }   // chunks arrive in stream order
            *row = make_double2(re, im);
        }
    }
    if (!p.finalise) return;

    // ---- second pass: the last CTA of each group sums the group, the last group sums the groups
    const RedParams& rp = p.red;
    const int grp = blockIdx.x / rp.group_size, first = grp * rp.group_size;
    const int members = ((int)gridDim.x - first < rp.group_size) ? (int)gridDim.x - first : rp.group_size;
    // (the barrier orders the CTA's row before thread 0's fence; the fence is cumulative)
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        s_last = (atomicInc(&rp.tickets[grp], members * gridDim.y - 1) == members * gridDim.y - 1);
        __threadfence();
    }
    __syncthreads();
    RBE_STAMP();
    if (!s_last) return;
    reduce_rows(rp.part + (int64_t)first * p.P, members, p.P, rp.grow + (int64_t)grp * p.P, nullptr, acc_all, tid, T);
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        s_last = (atomicInc(&rp.tickets[rp.ngroups], rp.ngroups - 1) == (unsigned)rp.ngroups - 1);
        __threadfence();
    }
    __syncthreads();
    if (!s_last) return;
    RBE_STAMP();
    reduce_rows(rp.grow, rp.ngroups, p.P, rp.rho, rp.rho_user, acc_all, tid, T);
    RBE_STAMP();
    if (rp.xch.world > 0) {
        // fused exchange: this CTA (the last one of the grid) writes the partial rho into its slot on
        // every rank over NVLink, then releases the per-rank flags (stores, fence, flag)
        __syncthreads();
        for (int r = 0; r < rp.xch.world; ++r)
            for (int k = tid; k < p.P; k += T) rp.xch.slot[r][k] = __ldcg(&rp.rho[k]);
        __threadfence_system();
        __syncthreads();
        if (tid < rp.xch.world) st_release_sys(rp.xch.flag[tid], rp.xch.epoch);
    }
}

// ---------------------------------------------------------------------------------------
// F kernel -- Algorithm 1 step 4, Eq. (2.12) P:131.
//
// Mapping: a thread owns R atoms (coordinates as fixed-point turns in registers) and loops
// over the wavevectors, whose {-m, theta} and {G, E} records are broadcast from shared memory.
// Work is dealt to WARPS in units of 32 atoms, balanced over the whole grid, and every warp
// splits its run into equal passes of R <= 4 units, so that every SM sub-partition gets the
// same number of (atom, k) pairs to within one unit.
// Per pair: 3 IMAD (phase), I2FP, 2 FMUL, 1 MUFU.SIN, 3 FFMA (+ MUFU.COS, FFMA with energy).
// ---------------------------------------------------------------------------------------
struct FParams {
    const float4* xyzq;
    float4* force;
    int64_t N;
    KTable kt;     // rho and the k-set: every CTA builds its {-m, theta}, {G, E} records from these
    double two32_over_L;
    int32_t P;
    int32_t pdl;   // launched with programmatic stream serialisation: wait before reading rho
};

__device__ __forceinline__ float4 f_fetch(const FParams& p, int64_t unit, int lane) {
    const int64_t i = unit * 32 + lane;
    return i < p.N ? __ldg(&p.xyzq[i]) : make_float4(0.f, 0.f, 0.f, 0.f);
}

// One pass: R units (R atoms per thread) against the nk wavevector records in shared memory.
// `pre` != nullptr: the atom records were fetched earlier (prologue overlap), else fetch here.
template <int R, bool ENERGY, bool ACCUM>
__device__ __forceinline__ void f_pass(const FParams& p, const int4* s_ka, const float4* s_kb, int nk, int64_t unit0,
                                       int lane, const float4* pre) {
    uint32_t sx[R], sy[R], sz[R];
    float q[R], fx[R], fy[R], fz[R], en[R];
    const float K = phase_scale();
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const float4 a = pre ? pre[r] : f_fetch(p, unit0 + r, lane);
        sx[r] = to_turns(a.x, p.two32_over_L);
        sy[r] = to_turns(a.y, p.two32_over_L);
        sz[r] = to_turns(a.z, p.two32_over_L);
        q[r] = a.w;
        fx[r] = fy[r] = fz[r] = en[r] = 0.f;
    }
#pragma unroll 4
    for (int k = 0; k < nk; ++k) {
        const int4 a = s_ka[k];
        const float4 b = s_kb[k];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const uint32_t ph = (uint32_t)a.x * sx[r] + ((uint32_t)a.y * sy[r] + ((uint32_t)a.z * sz[r] + (uint32_t)a.w));
            const float x = phase_to_arg(ph, K);
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

// n units in ceil(n / F_RMAX) passes of nearly equal size (e.g. 9 -> 3+3+3, not 4+4+1)
__device__ __forceinline__ int f_first_pass(int n) {
    const int passes = (n + F_RMAX - 1) / F_RMAX;
    return passes ? (n + passes - 1) / passes : 0;
}

template <bool ENERGY, bool ACCUM>
__device__ __forceinline__ void f_run(const FParams& p, const int4* s_ka, const float4* s_kb, int nk, int64_t u, int n,
                                      int lane, const float4* pre) {
    int passes = (n + F_RMAX - 1) / F_RMAX;
    while (n > 0) {
        const int r = (n + passes - 1) / passes;
        switch (r) {
            case 4: f_pass<4, ENERGY, ACCUM>(p, s_ka, s_kb, nk, u, lane, pre); break;
            case 3: f_pass<3, ENERGY, ACCUM>(p, s_ka, s_kb, nk, u, lane, pre); break;
            case 2: f_pass<2, ENERGY, ACCUM>(p, s_ka, s_kb, nk, u, lane, pre); break;
            default: f_pass<1, ENERGY, ACCUM>(p, s_ka, s_kb, nk, u, lane, pre); break;
        }
        u += r; n -= r; --passes;
        pre = nullptr;
    }
}

template <bool ENERGY>
__global__ void __launch_bounds__(F_THREADS, F_CTAS_PER_SM) f_kernel(const FParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nkmax = p.P < F_KCHUNK ? p.P : F_KCHUNK;
    int4* s_ka = reinterpret_cast<int4*>(smem_raw);
    float4* s_kb = reinterpret_cast<float4*>(smem_raw + (size_t)nkmax * sizeof(int4));
    const int lane = threadIdx.x & 31;
    const int64_t nwarps = (int64_t)gridDim.x * (F_THREADS / 32);
    const int64_t gw = (int64_t)blockIdx.x * (F_THREADS / 32) + (threadIdx.x >> 5);
    const int64_t units = (p.N + 31) / 32;
    const int64_t u0 = units * gw / nwarps, u1 = units * (gw + 1) / nwarps;
    const int n = (int)(u1 - u0);

    // fetch the first pass's atoms before waiting for the structure factors: the loads (and, with
    // PDL, this grid's launch) overlap the tail of the preceding grid
    float4 pre[F_RMAX];
    const int r0 = f_first_pass(n);
#pragma unroll
    for (int r = 0; r < F_RMAX; ++r) pre[r] = r < r0 ? f_fetch(p, u0 + r, lane) : make_float4(0.f, 0.f, 0.f, 0.f);

    if (p.pdl) grid_dependency_wait();   // rho comes from the preceding grid
    xch_wait(p.kt.xch);                  // ... and, with a multi-GPU exchange, from the peers' grids

    for (int k0 = 0; k0 < p.P; k0 += F_KCHUNK) {
        const int nk = (p.P - k0 < F_KCHUNK) ? (p.P - k0) : F_KCHUNK;
        if (k0 > 0) __syncthreads();
        for (int t = threadIdx.x; t < nk; t += F_THREADS) k_record(p.kt, k0 + t, s_ka[t], s_kb[t]);
        __syncthreads();
        if (k0 == 0) f_run<ENERGY, false>(p, s_ka, s_kb, nk, u0, n, lane, pre);
        else f_run<ENERGY, true>(p, s_ka, s_kb, nk, u0, n, lane, nullptr);
    }
}

// ---------------------------------------------------------------------------------------
// Sampler kernel -- Algorithm 1 step 1 on the device: P iid draws of m != 0 with
// probability ~ exp(-|2 pi m / L|^2 / 4 alpha).  DESIGN.md readings Q2 (exact iid draws by
// per-dimension inverse CDF, the zero triple rejected) and Q17 (the random numbers):
//   candidate j of step t = first three words of Philox4x32-10, counter (j, t), key = seed;
//   m_d = #{ i : T_i <= word_d } - M with the host-built integer thresholds T (rbe_api.cu);
//   the batch = the first P non-zero candidates in order of j.
// One CTA; candidates are taken 1024 at a time and compacted by ballot + prefix sums, so the
// result is exactly the sequential definition.  If `state` is given, (seed, step) are read
// from it and the step is advanced after the draw (graph replay: no host involvement).
// ---------------------------------------------------------------------------------------
struct SampleParams {
    const uint32_t* T;             // [2M] thresholds
    int32_t M, P;
    int4* kvec;                    // [P] out
    unsigned long long* state;     // {seed, step} on the device, or nullptr
    unsigned long long seed, step; // used when state == nullptr
};

__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
        c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
        k.x += 0x9E3779B9u; k.y += 0xBB67AE85u;
    }
    return c;
}

__device__ __forceinline__ int sample_dim(const uint32_t* T, int M, uint32_t x) {
    int lo = 0, hi = 2 * M;      // #{ i in [0, 2M) : T_i <= x }
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (__ldg(&T[mid]) <= x) lo = mid + 1; else hi = mid;
    }
    return lo - M;
}

__global__ void __launch_bounds__(1024) sample_kernel(const SampleParams p) {
    __shared__ uint32_t wsum[32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned long long seed = p.state ? p.state[0] : p.seed;
    const unsigned long long step = p.state ? p.state[1] : p.step;
    const uint2 key = make_uint2((uint32_t)seed, (uint32_t)(seed >> 32));
    int accepted = 0;
    for (unsigned long long j0 = 0; accepted < p.P; j0 += 1024) {
        const unsigned long long j = j0 + tid;
        const uint4 w = philox4x32_10(make_uint4((uint32_t)j, (uint32_t)(j >> 32), (uint32_t)step, (uint32_t)(step >> 32)), key);
        const int mx = sample_dim(p.T, p.M, w.x), my = sample_dim(p.T, p.M, w.y), mz = sample_dim(p.T, p.M, w.z);
        const bool nz = (mx | my | mz) != 0;
        const uint32_t bal = __ballot_sync(FULL_MASK, nz);
        if (lane == 0) wsum[warp] = __popc(bal);
        __syncthreads();
        int before = 0, total = 0;
#pragma unroll
        for (int i = 0; i < 32; ++i) {
            const int v = (int)wsum[i];
            before += i < warp ? v : 0;
            total += v;
        }
        const int pos = accepted + before + __popc(bal & ((1u << lane) - 1u));
        if (nz && pos < p.P) p.kvec[pos] = make_int4(mx, my, mz, 0);
        accepted += total;
        __syncthreads();
    }
    if (p.state && tid == 0) p.state[1] = step + 1;
}

// ---------------------------------------------------------------------------------------
// Compact host step (rbe_step_host_xyz): only positions travel to the device and only force
// vectors travel back (12 B per atom each way instead of 16); the charges stay on the device.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) pack_xyzq_kernel(const float* __restrict__ xyz, const float* __restrict__ q, int64_t n,
                                                         float4* __restrict__ xyzq) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) xyzq[i] = make_float4(xyz[3 * i], xyz[3 * i + 1], xyz[3 * i + 2], q[i]);
}
__global__ void __launch_bounds__(256) unpack_force_kernel(const float4* __restrict__ f4, int64_t n, float* __restrict__ f3) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        const float4 f = f4[i];
        f3[3 * i] = f.x; f3[3 * i + 1] = f.y; f3[3 * i + 2] = f.z;
    }
}

}  // namespace rbe
