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
// Measured on B200 (rbe_probe_pipe_rates, profiles/): MUFU 16 lanes/SM/clk, IMAD and I2FP 64,
// FFMA 128; a MUFU also costs ~3 issue slots.  Both hot kernels are bound by MUFU + issue.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace rbe {

// ---------------------------------------------------------------------------------------
// tunables (compile time; the values are the measured optima, see profiles/)
// ---------------------------------------------------------------------------------------
constexpr int SF_KPT = 4;        // wavevectors owned by one thread of the structure-factor phase
constexpr int SF_TMAX = 1024;    // max threads per CTA (structure-factor / step kernels): <= 64 registers
constexpr int SF_WPT = 2;        // 32-atom windows a warp stages per tile
constexpr int SF_TILE_MAX = (SF_TMAX / 32) * SF_WPT * 32;   // atoms per tile (one record arena): 2048
constexpr int SF_DEPTH = 128;    // max atoms a thread accumulates in fp32 before the fp64 flush
constexpr int STEP_PMAX = SF_TMAX * SF_KPT;   // largest batch the one-launch step kernel takes (one k-chunk)
constexpr int STEP_KPARAM_MAX = 512;          // largest batch whose wavevectors ride in the kernel parameters
constexpr int F_THREADS = 512;   // threads per CTA (force kernel)
constexpr int F_CTAS_PER_SM = 2;
constexpr int F_RMAX = 4;        // max atoms per thread per pass (force kernel)
constexpr int F_KCHUNK = 2048;   // wavevectors staged in shared memory at a time (force kernel)
constexpr int F_KSPLIT = 8;      // step kernel, small systems: most slices a unit's wavevectors are cut into (one slice per warp)
constexpr int SF_RED_GROUP = 16; // CTAs per group in the two-level reduction of the per-CTA rows (two-launch path)

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
    if (*reinterpret_cast<volatile const int32_t*>(t.xch.error)) {   // a peer never arrived: poison, do not pass silently
        const double nan = __longlong_as_double(0x7ff8000000000000ll);
        return make_double2(nan, nan);
    }
    double re = 0.0, im = 0.0;
    for (int r = 0; r < t.xch.world; ++r) {
        const double2 v = __ldcg(&t.xch.slots[(int64_t)r * t.P + k]);   // written by a peer: not through L1
        re += v.x; im += v.y;
    }
    return make_double2(re, im);
}

__device__ __forceinline__ void k_record_from(int4 m, double2 r, double w, double L, int4& ka, float4& kb) {
    const double m2 = (double)m.x * m.x + (double)m.y * m.y + (double)m.z * m.z;
    const double mag = sqrt(r.x * r.x + r.y * r.y);
    const double theta = atan2(r.y, r.x) * (1.0 / (2.0 * PI_D));      // turns, [-1/2, 1/2]
    const double gs = -2.0 * w / (L * L * m2) * mag;
    const double el = w / (2.0 * PI_D * L * m2);
    ka = make_int4(-m.x, -m.y, -m.z, __double2loint(fma(theta, TWO32, MAGIC)));   // {-m, theta in 2^-32 turns}
    kb = make_float4((float)(gs * m.x), (float)(gs * m.y), (float)(gs * m.z), (float)(el * mag));  // {G, e_l |rho_l|}
}
// The same record with |rho| and arg rho taken in fp32 (sqrtf, atan2f: ~1e-7 relative, far inside the 2e-5
// force tolerance; the products around them stay fp64).  The step kernel builds every record on its critical
// path between two grid barriers, where the fp64 atan2 chain alone costs over a microsecond.
__device__ __forceinline__ void k_record_fast(int4 m, double2 r, double w, double L, int4& ka, float4& kb) {
    const double m2 = (double)m.x * m.x + (double)m.y * m.y + (double)m.z * m.z;
    // scale first: |rho|^2 of a large system overflows nothing in fp32, but tiny ones would underflow
    const double big = fmax(fabs(r.x), fabs(r.y));
    const double inv = big > 0.0 ? 1.0 / big : 0.0;
    const float xr = (float)(r.x * inv), yr = (float)(r.y * inv);
    const double mag = big * (double)sqrtf(fmaf(xr, xr, yr * yr));
    const double theta = (double)atan2f(yr, xr) * (1.0 / (2.0 * PI_D));   // turns, [-1/2, 1/2]
    const double gs = -2.0 * w / (L * L * m2) * mag;
    const double el = w / (2.0 * PI_D * L * m2);
    ka = make_int4(-m.x, -m.y, -m.z, __double2loint(fma(theta, TWO32, MAGIC)));
    kb = make_float4((float)(gs * m.x), (float)(gs * m.y), (float)(gs * m.z), (float)(el * mag));
}
__device__ __forceinline__ void k_record(const KTable& t, int k, int4& ka, float4& kb) {
    k_record_from(t.kvec[k], k_rho(t, k), t.w ? t.w[k] : t.w_uniform, t.L, ka, kb);
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
// SF phase -- Algorithm 1 steps 2+3 fused, Eq. (2.9) P:117.  Shared by the two-launch
// structure-factor kernel (sf_kernel) and the one-launch step kernel (step_kernel).
//
// Mapping: a thread OWNS SF_KPT wavevectors (their m in registers) and one of `ng` atom
// groups.  The CTA walks its contiguous atom range in tiles of nwarps * SF_WPT windows of 32 atoms;
// the N x P array of Fourier modes the paper materialises before its Reduce-by-Key never
// exists, and there is no cross-lane reduction: each thread sums its own (cos, sin) in fp32 over at
// most ~SF_DEPTH atoms, then in fp64 (shared-memory accumulators).  Groups are combined in group
// order and one fp64 row of P complex partials per CTA goes to global memory.  No atomics on data.
//
// Equal-|q| pairing (what makes this phase 3 MUFU per TWO pairs instead of 4).  For two atoms
// with q_2 = +-q_1 and turns S_1, S_2 let S_d = (S_1 - S_2)/2, S_a = S_2 + S_d.  Then exactly
//   q_1 e^{i phi_1} + q_2 e^{i phi_2} = 2 q_1 cos(2 pi m.S_d - o) e^{i (2 pi m.S_a + o)},
// o = 0 for equal charges, a quarter turn for opposite ones (2i sin d = 2 cos(d - pi/2) e^{i pi/2}).
// Staging a tile, each warp matches the 32 atoms of a window by |q| bit pattern (MATCH.ANY) and
// emits pair records {S_a, o}{S_d, 2 q_1} and single records {S, q} for the leftovers, so ANY charge
// assignment is handled (all-distinct charges fall back to 2 MUFU per pair).  MD systems have a
// handful of distinct charge magnitudes, so nearly all atoms pair up.
//
// Staging is warp-local and overlapped.  A warp loads its SF_WPT windows of the NEXT tile straight
// from global memory into registers (lane = atom: one coalesced 512-byte request per window; no raw
// tile in shared memory, no cp.async), classifies and converts them and writes the records into the
// other half of a double-buffered record arena.  It does so in the middle of its accumulation loop
// over the CURRENT tile, at a point that depends on the warp index, so that at any moment about one
// warp per SM is staging (and waiting on HBM) while the other 31 keep the MUFU pipe busy.  Record
// positions are the exclusive prefix over the warps' counts (published through shared-memory flags;
// a warp only ever waits for warps that staged earlier), so the record order -- and with it every
// floating-point sum -- is deterministic.  One __syncthreads per tile.
// ---------------------------------------------------------------------------------------
struct SfArgs {
    const float4* xyzq;
    int64_t N;
    double2* part;     // [gridDim.x][P] per-CTA rows
    double two32_over_L;
    int32_t P;
    int32_t gs;        // threads per atom group in this CTA = k-slots / SF_KPT
    int32_t ng;        // atom groups per CTA
    int32_t pairing;   // bit 0: pair equal charges, bit 1: pair opposite charges (3 = both)
    int32_t accumulate;   // add this launch's per-CTA rows to what `part` holds (chunked host step: one launch per chunk)
};

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

// Shared-memory control words of the staging protocol (one set per CTA).
struct SfCtl {
    volatile uint32_t cnt[32];    // per warp: pair records | single records << 16 of the tile being staged
    volatile uint32_t flag[32];   // per warp: sequence number (tile index + 1) of the tile whose counts are published
    uint32_t tot[2];              // per arena half: total pair | single << 16 records of the tile
};

// Stage this warp's SF_WPT windows of one tile: atoms [a0, a0 + 32 * SF_WPT) clipped to `hi`.  All 32 lanes.
// FIRST: the tile every warp stages at once when the kernel starts -- the counts meet at a __syncthreads
// (called by ALL threads of the CTA); otherwise through the per-warp flags (a warp stages tile t + 1 in the
// middle of its loop over tile t and waits only for warps whose turn came earlier).
// This warp's SF_WPT windows of one tile, lane = atom: atoms [a0, a0 + 32 * SF_WPT) clipped to `hi`.
__device__ __forceinline__ void sf_load(const SfArgs& p, int64_t a0, int64_t hi, int lane, float4 (&a)[SF_WPT]) {
#pragma unroll
    for (int j = 0; j < SF_WPT; ++j) {
        const int64_t i = a0 + j * 32 + lane;
        a[j] = i < hi ? __ldg(&p.xyzq[i]) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
}
// The atom range [lo, hi) of CTA bx of gx, aligned to 32-atom windows.
__device__ __forceinline__ void sf_range(const SfArgs& p, int bx, int gx, int64_t& lo, int64_t& hi) {
    const int64_t units = (p.N + 31) >> 5;
    lo = (units * bx / gx) << 5;
    hi = (units * (bx + 1) / gx) << 5;
    if (hi > p.N) hi = p.N;
}
// The loads of tile 0, for a kernel to issue as its very first instructions (their latency then hides behind its prologue).
__device__ __forceinline__ void sf_load_first(const SfArgs& p, int bx, int gx, float4 (&a)[SF_WPT]) {
    int64_t lo, hi;
    sf_range(p, bx, gx, lo, hi);
    sf_load(p, lo + (int64_t)(threadIdx.x >> 5) * (SF_WPT * 32), hi, threadIdx.x & 31, a);
}

template <bool FIRST>
__device__ __forceinline__ void sf_stage(const SfArgs& p, const float4 (&a)[SF_WPT], int64_t a0, int64_t hi, int warp, int lane, int nwarps,
                                         uint4* A, SfCtl& ctl, uint32_t* tot, uint32_t seq) {
    const uint32_t lt_mask = (1u << lane) - 1u;
    SfWindow cw[SF_WPT];
    uint32_t mine = 0;    // this warp's pair | single << 16 counts
#pragma unroll
    for (int j = 0; j < SF_WPT; ++j) {
        cw[j] = sf_classify(__float_as_uint(a[j].w), a0 + j * 32 + lane < hi, p.pairing, lane);
        mine += (uint32_t)__popc(cw[j].lmask) | ((uint32_t)__popc(cw[j].smask) << 16);
    }
    // publish the counts, then take the exclusive prefix over the warps before this one
    uint32_t base = 0;
    if (FIRST) {
        if (lane == 0) ctl.cnt[warp] = mine;
        __syncthreads();
        if (lane < warp) base = ctl.cnt[lane];
    } else {
        if (lane == 0) {
            ctl.cnt[warp] = mine;
            __threadfence_block();
            ctl.flag[warp] = seq;
        }
        if (lane < warp) {
            while (ctl.flag[lane] != seq) __nanosleep(40);
            __threadfence_block();
            base = ctl.cnt[lane];
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) base += __shfl_xor_sync(FULL_MASK, base, d);   // fields cannot carry: <= 2048 each
    if (warp == nwarps - 1 && lane == 0) *tot = base + mine;
    uint32_t bp = base & 0xffffu, bs = base >> 16;
#pragma unroll
    for (int j = 0; j < SF_WPT; ++j) {
        const uint32_t Sx = to_turns(a[j].x, p.two32_over_L);
        const uint32_t Sy = to_turns(a[j].y, p.two32_over_L);
        const uint32_t Sz = to_turns(a[j].z, p.two32_over_L);
        const uint32_t Px = __shfl_sync(FULL_MASK, Sx, cw[j].partner);
        const uint32_t Py = __shfl_sync(FULL_MASK, Sy, cw[j].partner);
        const uint32_t Pz = __shfl_sync(FULL_MASK, Sz, cw[j].partner);
        const uint32_t Pq = __shfl_sync(FULL_MASK, __float_as_uint(a[j].w), cw[j].partner);
        if (cw[j].leader) {
            // S_d = (S_1 - S_2) / 2 (arithmetic shift of the wrapped difference), S_a = S_2 + S_d
            const uint32_t e = bp + (uint32_t)__popc(cw[j].lmask & lt_mask);
            const uint32_t dx = (uint32_t)((int32_t)(Sx - Px) >> 1);
            const uint32_t dy = (uint32_t)((int32_t)(Sy - Py) >> 1);
            const uint32_t dz = (uint32_t)((int32_t)(Sz - Pz) >> 1);
            // o: a quarter turn for opposite charges; plus half a turn on every other pair, which leaves
            // cos(d - o) e^{i(a + o)} unchanged but alternates the sign of the evaluated amplitude, so
            // the +1.7e-8 mean error of MUFU.COS (measured) cannot add up coherently over the pairs
            // (for single atoms it cancels by neutrality; the sum of pair amplitudes is not neutral)
            const uint32_t off = (((__float_as_uint(a[j].w) ^ Pq) >> 31) ? QUARTER_TURN : 0u) + (e << 31);
            A[2 * e] = make_uint4(Px + dx, Py + dy, Pz + dz, off);
            A[2 * e + 1] = make_uint4(dx, dy, dz, __float_as_uint(2.0f * a[j].w));
        } else if (cw[j].single) {
            const uint32_t e = bs + (uint32_t)__popc(cw[j].smask & lt_mask);
            A[SF_TILE_MAX - 1 - e] = make_uint4(Sx, Sy, Sz, __float_as_uint(a[j].w));   // singles from the back
        }
        bp += (uint32_t)__popc(cw[j].lmask);
        bs += (uint32_t)__popc(cw[j].smask);
    }
}

// Shared-memory footprint of the SF phase: two record arenas + the fp64 accumulators [SF_KPT][threads].
__host__ __device__ constexpr size_t sf_smem_bytes(int threads) {
    return (size_t)2 * SF_TILE_MAX * sizeof(uint4) + (size_t)threads * SF_KPT * sizeof(double2);
}

// The accumulation over this CTA's atoms.  On return the fp64 accumulators in shared memory hold every
// thread's sums (call sf_write_row next).  bx / gx: this CTA's index among the CTAs that share the atoms.
template <bool DEEP>
__device__ __forceinline__ void sf_accumulate(const SfArgs& p, const float4 (&first)[SF_WPT], const int (&mx)[SF_KPT], const int (&my)[SF_KPT],
                                              const int (&mz)[SF_KPT], unsigned char* smem_raw, SfCtl& ctl, int bx, int gx) {
    const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = T >> 5;
    uint4* arena = reinterpret_cast<uint4*>(smem_raw);                           // [2][SF_TILE_MAX] records
    double2* acc_all = reinterpret_cast<double2*>(arena + 2 * SF_TILE_MAX);      // [SF_KPT][T] fp64 accumulators
    // this CTA's atom range, aligned to 32-atom windows, in tiles of nwarps * SF_WPT windows
    int64_t lo, hi;
    sf_range(p, bx, gx, lo, hi);
    const int tile_atoms = nwarps * SF_WPT * 32;
    const int ntiles = hi > lo ? (int)((hi - lo + tile_atoms - 1) / tile_atoms) : 0;
    // tile 0 first, from the atoms the caller loaded when the kernel started (every thread calls: it has a barrier inside)
    sf_stage<true>(p, first, lo + (int64_t)warp * (SF_WPT * 32), hi, warp, lane, nwarps, arena, ctl, &ctl.tot[0], 1u);

    const bool active = tid < p.gs * p.ng;
    const int g = active ? tid / p.gs : (1 << 28);  // inactive threads: cursor past every list -> empty loops
    double2* acc = acc_all + tid;
    float c[SF_KPT], s[SF_KPT];
#pragma unroll
    for (int r = 0; r < SF_KPT; ++r) {
        c[r] = s[r] = 0.f;
        acc[r * T] = make_double2(0.0, 0.0);
    }
    if (tid < 32) ctl.flag[tid] = 0u;
    const float K = phase_scale();
    __syncthreads();   // records of tile 0, tot[0], zeroed flags and accumulators                           // @stamp

    int ep = g, es = g;    // round-robin cursors into the pair / single lists, carried across tiles
    int depth = 0;
#pragma unroll 1
    for (int t = 0; t < ntiles; ++t) {
        const int buf = t & 1;
        const uint4* A = arena + buf * SF_TILE_MAX;
        const uint32_t total = ctl.tot[buf];
        const int np = (int)(total & 0xffffu), ns = (int)(total >> 16);
        const bool more = t + 1 < ntiles;
        // this warp stages its windows of tile t + 1 after the first `split` pair records of tile t: the
        // warps take turns over the first three quarters of the tile
        const int split = more ? (np * 3 * warp) / (4 * nwarps) : np;
#pragma unroll 1
        for (int part = 0; part < 2; ++part) {
            const int end = part == 0 ? split : np;
#pragma unroll 1
            for (; ep < end; ep += p.ng) {
                const uint4 ra = A[2 * ep];
                const uint4 rd = A[2 * ep + 1];
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
            if (part == 0 && more) {
                float4 nxt[SF_WPT];
                const int64_t a0 = lo + (int64_t)(t + 1) * tile_atoms + (int64_t)warp * (SF_WPT * 32);
                sf_load(p, a0, hi, lane, nxt);
                sf_stage<false>(p, nxt, a0, hi, warp, lane, nwarps, arena + (buf ^ 1) * SF_TILE_MAX, ctl, &ctl.tot[buf ^ 1], (uint32_t)t + 2u);
            }
        }
        ep -= np;
#pragma unroll 1
        for (; es < ns; es += p.ng) {
            const uint4 at = A[SF_TILE_MAX - 1 - es];
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
        es -= ns;
        if (!DEEP) sf_flush(acc, T, c, s);   // a thread takes at most SF_DEPTH atoms from one tile
        __syncthreads();   // tile t is consumed (its arena half may be overwritten), tile t + 1 is staged   // @stamp
    }
    if (DEEP) sf_flush(acc, T, c, s);
    __syncthreads();
}

// Combine the atom groups in group order: one fp64 row of this CTA's k-slots.  by: k-chunk index.
__device__ __forceinline__ void sf_write_row(const SfArgs& p, unsigned char* smem_raw, int bx, int by) {
    const int tid = threadIdx.x, T = blockDim.x;
    const double2* acc_all = reinterpret_cast<const double2*>(reinterpret_cast<uint4*>(smem_raw) + 2 * SF_TILE_MAX);
    const int kslots = p.gs * SF_KPT;
    for (int idx = tid; idx < kslots; idx += T) {
        const int k = by * kslots + idx;
        if (k < p.P) {
            double re = 0.0, im = 0.0;
            for (int gg = 0; gg < p.ng; ++gg) {
                const double2 v = acc_all[(idx % SF_KPT) * T + gg * p.gs + idx / SF_KPT];
                re += v.x; im += v.y;
            }
            double2* row = &p.part[(int64_t)bx * p.P + k];
            if (p.accumulate) { const double2 old = *row; re += old.x; im += old.y; }   // chunks arrive in stream order
            *row = make_double2(re, im);
        }
    }
}

// ---------------------------------------------------------------------------------------
// sf_kernel -- the structure factors as their own launch (rbe_structure_factor; the chunked host
// step; the multi-GPU exchange).  The last CTAs to finish (atomicInc tickets; data order never
// depends on them) run the second pass: the fixed-order two-level sum of the per-CTA rows into rho
// (reduce_rows), and, with a multi-GPU exchange configured, the push of rho into every rank's buffer.
// ---------------------------------------------------------------------------------------
struct SfParams {
    SfArgs a;
    const int4* kvec;  // [P] {mx, my, mz, 0}
    int32_t finalise;  // run the second pass (rows -> rho) at the end of this launch
    RedParams red;
};

template <bool DEEP>
__global__ void __launch_bounds__(SF_TMAX, 1) sf_kernel(const SfParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ SfCtl ctl;
    __shared__ uint32_t s_last;
    const int tid = threadIdx.x, T = blockDim.x;
    float4 tile0[SF_WPT];
    sf_load_first(p.a, blockIdx.x, gridDim.x, tile0);
    const bool active = tid < p.a.gs * p.a.ng;
    const int kbase = (blockIdx.y * p.a.gs + (active ? tid % p.a.gs : 0)) * SF_KPT;
    int mx[SF_KPT], my[SF_KPT], mz[SF_KPT];
#pragma unroll
    for (int r = 0; r < SF_KPT; ++r) {
        int4 m = make_int4(0, 0, 0, 0);
        if (active && kbase + r < p.a.P) m = __ldg(&p.kvec[kbase + r]);
        mx[r] = m.x; my[r] = m.y; mz[r] = m.z;
    }
    sf_accumulate<DEEP>(p.a, tile0, mx, my, mz, smem_raw, ctl, blockIdx.x, gridDim.x);

    // let the dependent (force) kernel start launching; it waits for this grid's completion
    grid_launch_dependents();
    sf_write_row(p.a, smem_raw, blockIdx.x, blockIdx.y);
    if (!p.finalise) return;

    // ---- second pass: the last CTA of each group sums the group, the last group sums the groups
    double2* scratch = reinterpret_cast<double2*>(reinterpret_cast<uint4*>(smem_raw) + 2 * SF_TILE_MAX);
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
    if (!s_last) return;
    reduce_rows(rp.part + (int64_t)first * p.a.P, members, p.a.P, rp.grow + (int64_t)grp * p.a.P, nullptr, scratch, tid, T);
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        s_last = (atomicInc(&rp.tickets[rp.ngroups], rp.ngroups - 1) == (unsigned)rp.ngroups - 1);
        __threadfence();
    }
    __syncthreads();
    if (!s_last) return;
    reduce_rows(rp.grow, rp.ngroups, p.a.P, rp.rho, rp.rho_user, scratch, tid, T);
    if (rp.xch.world > 0) {
        // fused exchange: this CTA (the last one of the grid) writes the partial rho into its slot on
        // every rank over NVLink, then releases the per-rank flags (stores, fence, flag)
        __syncthreads();
        for (int idx = tid; idx < rp.xch.world * p.a.P; idx += T) {       // all (rank, k) stores in flight together
            const int r = idx / p.a.P, k = idx - r * p.a.P;
            rp.xch.slot[r][k] = __ldcg(&rp.rho[k]);
        }
        __threadfence_system();
        __syncthreads();
        if (tid < rp.xch.world) st_release_sys(rp.xch.flag[tid], rp.xch.epoch);
    }
}

// ---------------------------------------------------------------------------------------
// F phase -- Algorithm 1 step 4, Eq. (2.12) P:131.  Shared by f_kernel and step_kernel.
//
// Mapping: a thread owns R atoms (coordinates as fixed-point turns in registers) and loops
// over the wavevectors, whose {-m, theta} and {G, E} records are broadcast from shared memory.
// Work is dealt to WARPS in units of 32 atoms, balanced over the whole grid, and every warp
// splits its run into equal passes of R <= 4 units, so that every SM sub-partition gets the
// same number of (atom, k) pairs to within one unit.
// Per pair: 3 IMAD (phase), I2FP, 2 FMUL, 1 MUFU.SIN, 3 FFMA (+ MUFU.COS, FFMA with energy).
// ---------------------------------------------------------------------------------------
struct FArgs {
    const float4* xyzq;
    float4* force;
    int64_t N;
    double two32_over_L;
};

__device__ __forceinline__ float4 f_fetch(const FArgs& p, int64_t unit, int lane) {
    const int64_t i = unit * 32 + lane;
    return i < p.N ? __ldg(&p.xyzq[i]) : make_float4(0.f, 0.f, 0.f, 0.f);
}

// One pass: R units (R atoms per thread) against the nk wavevector records in shared memory.
// (Tried: starting the record loop at a different k in every warp of a sub-partition, so that the warps do not
// march in lock-step.  A stand-alone copy of this loop gained 6 % from it; inside the kernels it lost 1 %.)
// s_out != nullptr (R = 1 only): the q-scaled sums go to s_out[lane] in shared memory instead of the force array
// (the k-split force phase of small systems adds such partial sums in a fixed order).
template <int R, bool ENERGY, bool ACCUM>
__device__ __forceinline__ void f_pass(const FArgs& p, const int4* s_ka, const float4* s_kb, int nk, int64_t unit0, int lane,
                                       float4* s_out = nullptr) {
    uint32_t sx[R], sy[R], sz[R];
    float q[R], fx[R], fy[R], fz[R], en[R];
    const float K = phase_scale();
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const float4 a = f_fetch(p, unit0 + r, lane);
        sx[r] = to_turns(a.x, p.two32_over_L);
        sy[r] = to_turns(a.y, p.two32_over_L);
        sz[r] = to_turns(a.z, p.two32_over_L);
        q[r] = a.w;
        fx[r] = fy[r] = fz[r] = en[r] = 0.f;
    }
    // 8 (atom, k) pairs in flight whatever R is: a thread with one atom is otherwise bound by the latency of its
    // IMAD -> I2FP -> FMUL -> MUFU -> FFMA chain (small systems: 45 cycles per wavevector instead of ~10)
#pragma unroll(R >= 3 ? 2 : R == 2 ? 4 : 8)
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
        if (R == 1 && s_out != nullptr) {
            s_out[lane] = make_float4(q[r] * fx[r], q[r] * fy[r], q[r] * fz[r], ENERGY ? q[r] * en[r] : 0.f);
        } else if (i < p.N) {
            float4 o = make_float4(q[r] * fx[r], q[r] * fy[r], q[r] * fz[r], ENERGY ? q[r] * en[r] : 0.f);
            if (ACCUM) {
                const float4 prev = p.force[i];
                o.x += prev.x; o.y += prev.y; o.z += prev.z; o.w += prev.w;
            }
            p.force[i] = o;
        }
    }
}

// The units [c0, c1) of a CTA dealt to its warps so that the four SM sub-partitions (warp index mod 4) get the
// same number of units to within one: the warps of a sub-partition take CONSECUTIVE shares of the even split.
// (With the plain split by warp index, 212 units over 32 warps give the pattern 7,6,7,7,6,7,6,7 of period 8, and
// one sub-partition gets 56 units against 53 on average: measured 6 % on the CTAs that have 212 units.)
__device__ __forceinline__ void f_warp_share(int64_t c0, int64_t c1, int warp, int nwarps, int64_t& u0, int& n) {
    int pos = warp;
    if ((nwarps & 3) == 0) pos = (warp & 3) * (nwarps >> 2) + (warp >> 2);
    u0 = c0 + (c1 - c0) * pos / nwarps;
    n = (int)(c0 + (c1 - c0) * (pos + 1) / nwarps - u0);
}

template <bool ENERGY, bool ACCUM>
__device__ __forceinline__ void f_run(const FArgs& p, const int4* s_ka, const float4* s_kb, int nk, int64_t u, int n, int lane) {
    int passes = (n + F_RMAX - 1) / F_RMAX;   // n units in passes of nearly equal size (e.g. 9 -> 3+3+3, not 4+4+1)
    while (n > 0) {
        const int r = (n + passes - 1) / passes;
        switch (r) {
            case 4: f_pass<4, ENERGY, ACCUM>(p, s_ka, s_kb, nk, u, lane); break;
            case 3: f_pass<3, ENERGY, ACCUM>(p, s_ka, s_kb, nk, u, lane); break;
            case 2: f_pass<2, ENERGY, ACCUM>(p, s_ka, s_kb, nk, u, lane); break;
            default: f_pass<1, ENERGY, ACCUM>(p, s_ka, s_kb, nk, u, lane); break;
        }
        u += r; n -= r; --passes;
    }
}

// ---------------------------------------------------------------------------------------
// f_kernel -- the forces as their own launch (rbe_forces; the chunked host step; the multi-GPU
// exchange).  Every CTA builds the per-k records for its shared-memory tile from rho (k_record).
// ---------------------------------------------------------------------------------------
struct FParams {
    FArgs a;
    KTable kt;     // rho and the k-set: every CTA builds its {-m, theta}, {G, E} records from these
    int32_t P;
    int32_t pdl;   // launched with programmatic stream serialisation: wait before reading rho
};

template <bool ENERGY>
__global__ void __launch_bounds__(F_THREADS, F_CTAS_PER_SM) f_kernel(const FParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nkmax = p.P < F_KCHUNK ? p.P : F_KCHUNK;
    int4* s_ka = reinterpret_cast<int4*>(smem_raw);
    float4* s_kb = reinterpret_cast<float4*>(smem_raw + (size_t)nkmax * sizeof(int4));
    const int lane = threadIdx.x & 31;
    const int64_t units = (p.a.N + 31) / 32;
    int64_t u0;
    int n;
    f_warp_share(units * blockIdx.x / gridDim.x, units * (blockIdx.x + 1) / gridDim.x, threadIdx.x >> 5, F_THREADS / 32, u0, n);

    // pull this warp's atoms into L2 before waiting for the structure factors: the requests (and, with PDL,
    // this grid's launch) overlap the tail of the preceding grid, and hold no registers across the wait
    for (int r = 0; r < n && r < 2 * F_RMAX; ++r) {
        const int64_t i = (u0 + r) * 32 + lane;
        if (i < p.a.N) asm volatile("prefetch.global.L2 [%0];" ::"l"(p.a.xyzq + i));
    }

    if (p.pdl) grid_dependency_wait();   // rho comes from the preceding grid
    xch_wait(p.kt.xch);                  // ... and, with a multi-GPU exchange, from the peers' grids

    for (int k0 = 0; k0 < p.P; k0 += F_KCHUNK) {
        const int nk = (p.P - k0 < F_KCHUNK) ? (p.P - k0) : F_KCHUNK;
        if (k0 > 0) __syncthreads();
        for (int t = threadIdx.x; t < nk; t += F_THREADS) k_record(p.kt, k0 + t, s_ka[t], s_kb[t]);
        __syncthreads();
        if (k0 == 0) f_run<ENERGY, false>(p.a, s_ka, s_kb, nk, u0, n, lane);
        else f_run<ENERGY, true>(p.a, s_ka, s_kb, nk, u0, n, lane);
    }
}

// ---------------------------------------------------------------------------------------
// step_kernel -- Algorithm 1 steps 2-4 in ONE cooperative launch (rbe_step), one CTA per
// SM, all CTAs co-resident:
//   1. SF phase over the CTA's atoms -> one fp64 row of P partial sums per CTA (global memory);
//   2. grid barrier;
//   3. distributed fixed-order reduction: the P wavevectors are dealt to the CTAs; one warp per
//      wavevector sums the gridDim.x rows (lane l takes rows l, l+32, ... in order, then a fixed
//      butterfly over the lanes), writes rho(k) and builds that wavevector's force record ONCE
//      (k_record_from: fp64 atan2 / sqrt) -- no serial tail, no ticket, no per-CTA rebuild;
//   4. grid barrier;
//   5. F phase over the same atoms with the P records in shared memory.
// Which CTA does what is fixed by blockIdx, so the result is bitwise reproducible.  The grid barrier
// is a 64-bit arrival counter in the workspace that only ever grows (a launch adds 2 * gridDim.x).
// For small batches without weights the wavevectors ride in the kernel parameters (int16 triples), so
// a step is one launch and nothing else: no host-to-device copy.
// ---------------------------------------------------------------------------------------
struct StepParams {
    SfArgs sf;
    FArgs f;
    const int4* kvec;          // [P] wavevectors in the workspace (read unless kparam, written if kparam)
    const double* w;           // [P] weights or nullptr
    double w_uniform, L;
    double2* rho;              // [P] out
    double2* rho_user;         // [P] out or nullptr
    int4* ka;                  // [P] force records, built in step 3
    float4* kb;
    unsigned long long* bar;   // grid-barrier arrival counter
    int32_t kparam;            // wavevectors are in km (P <= STEP_KPARAM_MAX), else in kvec
    int16_t km[STEP_KPARAM_MAX * 3];
};

__device__ __forceinline__ unsigned long long ld_acquire_gpu_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

// Grid barrier of a cooperative launch: a 64-bit arrival counter in the workspace that only ever grows (a launch
// adds 2 * gridDim.x; zeroed by rbe_set_workspace, one grid size per context).  Thread 0 of every CTA reads it when
// the kernel starts -- long before anybody can arrive at the first barrier, so off the critical path -- and rounds
// down to a multiple of gridDim.x: the count before this launch, whatever early arrivals it saw.  The barriers then
// wait for base + gridDim.x and base + 2 gridDim.x.  Arriving is a one-way red.release (no value comes back), so a
// barrier costs one fence, one reduction on its way and the polling load -- not an atomic round trip plus the poll.
__device__ __forceinline__ unsigned long long grid_barrier_base(const unsigned long long* ctr) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(ctr) : "memory");
    return v - v % gridDim.x;
}
// All threads of all CTAs.  Release: barrier + red.release by thread 0; acquire: its polling load before the barrier
// that lets the CTA continue.  No timeout on the wait: the CTAs of a cooperative launch are co-resident by construction, a
// kernel that faults leaves a sticky error that ends the process's use of the device anyway, and the one way to put the
// counter out of step from outside -- two contexts on one workspace -- is refused by rbe_set_workspace.
// (The base stays in thread 0's registers on purpose: parked in shared memory it frees two registers and removes 8 of
// the 28 spilled bytes, and the step gets 7 us SLOWER at N = 1e6 -- 176.9 against 170.0 us, measured in round 3; the same
// happened when the CTA's atom range was parked there, which brings the stack frame to 0 bytes: 176.5 us.  The spills
// sit at tile boundaries, outside the special-function loops, and the allocation ptxas finds with them is the faster one.)
__device__ __forceinline__ void grid_barrier(unsigned long long* ctr, unsigned long long target) {
    __syncthreads();
    if (threadIdx.x == 0) {
        asm volatile("red.release.gpu.global.add.u64 [%0], %1;" ::"l"(ctr), "l"(1ull) : "memory");
        while (ld_acquire_gpu_u64(ctr) < target) { }
    }
    __syncthreads();
}

__device__ __forceinline__ int4 step_kvec(const StepParams& p, const int16_t* s_km, int k) {
    if (p.kparam) return make_int4(s_km[3 * k], s_km[3 * k + 1], s_km[3 * k + 2], 0);
    return __ldg(&p.kvec[k]);
}

template <bool DEEP, bool ENERGY>
__global__ void __launch_bounds__(SF_TMAX, 1) step_kernel(const __grid_constant__ StepParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ SfCtl ctl;
    const int tid = threadIdx.x, T = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = T >> 5;
    const int bx = blockIdx.x, G = gridDim.x, P = p.sf.P;
    float4 first[SF_WPT];
    sf_load_first(p.sf, bx, G, first);                  // the longest latency of the prologue: issued before anything else
    unsigned long long bar_base = 0ull;
    if (tid == 0) bar_base = grid_barrier_base(p.bar);

    // ---- 1. SF phase                                                                   // @stamp
    // wavevectors from the kernel parameters: the constant bank serves one address per request, so every warp
    // reads a run of consecutive words with all its lanes on the SAME word (a broadcast) and parks them in
    // shared memory; per-thread indexing of the parameter array would serialise 32 ways (measured: 11 us)
    __shared__ int16_t s_km[STEP_KPARAM_MAX * 3];
    if (p.kparam) {
        const int n3 = 3 * P, per = (n3 + nwarps - 1) / nwarps;
        const int i1 = (warp + 1) * per < n3 ? (warp + 1) * per : n3;
        for (int i = warp * per; i < i1; ++i) {
            const int16_t v = p.km[i];
            if (lane == 0) s_km[i] = v;
        }
        __syncthreads();
    }
    {
        const bool active = tid < p.sf.gs * p.sf.ng;
        const int kbase = (active ? tid % p.sf.gs : 0) * SF_KPT;
        int mx[SF_KPT], my[SF_KPT], mz[SF_KPT];
#pragma unroll
        for (int r = 0; r < SF_KPT; ++r) {
            int4 m = make_int4(0, 0, 0, 0);
            if (active && kbase + r < P) m = step_kvec(p, s_km, kbase + r);
            mx[r] = m.x; my[r] = m.y; mz[r] = m.z;
        }
        if (p.kparam && bx == 0)   // keep the workspace copy current for the energy / virial / read-back calls
            for (int k = tid; k < P; k += T) const_cast<int4*>(p.kvec)[k] = step_kvec(p, s_km, k);
        sf_accumulate<DEEP>(p.sf, first, mx, my, mz, smem_raw, ctl, bx, G);                    // @stamp
        sf_write_row(p.sf, smem_raw, bx, 0);                                              // @stamp
    }
    grid_barrier(p.bar, bar_base + (unsigned long long)G);                                // @stamp

    // ---- 3. distributed fixed-order reduction + the per-k force records
    {
        const int k_lo = (int)((int64_t)P * bx / G), k_hi = (int)((int64_t)P * (bx + 1) / G);
        for (int k = k_lo + warp; k < k_hi; k += nwarps) {
            double re = 0.0, im = 0.0;
#pragma unroll 5
            for (int row = lane; row < G; row += 32) {     // (148 rows: five independent loads per lane in flight)
                const double2 v = __ldcg(&p.sf.part[(int64_t)row * P + k]);
                re += v.x; im += v.y;
            }
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) {
                re += __shfl_xor_sync(FULL_MASK, re, d);
                im += __shfl_xor_sync(FULL_MASK, im, d);
            }
            if (lane == 0) {
                const double2 r = make_double2(re, im);
                p.rho[k] = r;
                if (p.rho_user) p.rho_user[k] = r;
                int4 a; float4 b;
                k_record_fast(step_kvec(p, s_km, k), r, p.w ? p.w[k] : p.w_uniform, p.L, a, b);
                p.ka[k] = a; p.kb[k] = b;
            }
        }
    }
                                                                                          // @stamp
    grid_barrier(p.bar, bar_base + 2ull * (unsigned long long)G);                         // @stamp

    // ---- 5. F phase: this CTA's warps take the same atom range the CTA had in the SF phase
    if (p.f.force == nullptr) return;
    int4* s_ka = reinterpret_cast<int4*>(smem_raw);
    float4* s_kb = reinterpret_cast<float4*>(smem_raw + (size_t)P * sizeof(int4));
    for (int t = tid; t < P; t += T) { s_ka[t] = __ldcg(&p.ka[t]); s_kb[t] = __ldcg(&p.kb[t]); }
    __syncthreads();
    const int64_t units = (p.f.N + 31) / 32;
    const int64_t c0 = units * bx / G, c1 = units * (bx + 1) / G;              // the CTA's units (as in the SF phase)
    const int nu = (int)(c1 - c0);
    uint32_t dyn_smem;
    asm("mov.u32 %0, %%dynamic_smem_size;" : "=r"(dyn_smem));
    int ksplit = nu > 0 ? nwarps / nu : 0;                 // slices per unit: as many (unit, slice) items as warps, at most F_KSPLIT
    if (ksplit > F_KSPLIT) ksplit = F_KSPLIT;
    if (ksplit >= 2 && P >= 8 * ksplit &&
        (size_t)P * (sizeof(int4) + sizeof(float4)) + (size_t)nu * ksplit * 32 * sizeof(float4) <= (size_t)dyn_smem) {
        // Small system: at most half as many units as warps.  Every unit's wavevectors are cut into ksplit slices, the
        // (unit, slice) items go one to a warp (one atom per thread, 8 wavevectors in flight), and the slices of a unit are
        // added in order.
        float4* parts = reinterpret_cast<float4*>(smem_raw + (size_t)P * (sizeof(int4) + sizeof(float4)));   // [nu * ksplit][32]
        if (warp < nu * ksplit) {
            const int unit = warp / ksplit, part = warp % ksplit;
            const int k0 = P * part / ksplit, k1 = P * (part + 1) / ksplit;
            f_pass<1, ENERGY, false>(p.f, s_ka + k0, s_kb + k0, k1 - k0, c0 + unit, lane, parts + (size_t)warp * 32);
        }
        __syncthreads();
        for (int idx = tid; idx < nu * 32; idx += T) {
            const int unit = idx >> 5, l = idx & 31;
            float4 a = parts[(size_t)(unit * ksplit) * 32 + l];
            for (int q = 1; q < ksplit; ++q) {
                const float4 v = parts[(size_t)(unit * ksplit + q) * 32 + l];
                a.x += v.x; a.y += v.y; a.z += v.z; a.w += v.w;
            }
            const int64_t i = (c0 + unit) * 32 + l;
            if (i < p.f.N) p.f.force[i] = a;
        }
        return;                                                                       // @stamp @stamp_sync
    }
    int64_t u0;
    int n;
    f_warp_share(c0, c1, warp, nwarps, u0, n);
    f_run<ENERGY, false>(p.f, s_ka, s_kb, P, u0, n, lane);                            // @stamp @stamp_sync
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

// ---------------------------------------------------------------------------------------
// Pipe-rate probe (rbe_probe_pipe_rates): the roofline of this path is set by the FP32-FMA, IMAD,
// I2FP and MUFU issue rates, which MEASURED_PEAKS.json does not hold (SURVEY.md s7 stage 6).  One CTA
// of 1024 threads per SM runs 8 dependent-free chains per thread of one instruction kind; thread 0 of
// every CTA reports the SM cycles (clock64) its CTA took, so the rates are per clock, whatever the clock.
// MODE 0: FFMA, 1: IMAD, 2: I2FP.F32.S32, 3: FMUL.RZ + MUFU.SIN (sin.approx).
// ---------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(1024, 1) probe_kernel(long long* cycles, int iters, float fa, float fb, int ia, int ib) {
    constexpr int C = 8;
    float v[C];
    int w[C];
#pragma unroll
    for (int c = 0; c < C; ++c) { v[c] = threadIdx.x * 0.001f + c; w[c] = threadIdx.x + c; }
    __syncthreads();
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int c = 0; c < C; ++c) {
            if (MODE == 0) v[c] = fmaf(v[c], fa, fb);
            if (MODE == 1) w[c] = w[c] * ia + ib;
            if (MODE == 2) w[c] = __float_as_int((float)w[c]);
            if (MODE == 3) v[c] = fast_sin(v[c]);
        }
    }
    float s = 0.f;
    int t = 0;
#pragma unroll
    for (int c = 0; c < C; ++c) { s += v[c]; t += w[c]; }
    __syncthreads();
    const long long t1 = clock64();
    if (threadIdx.x == 0) cycles[blockIdx.x] = (s + (float)t == 123.456f) ? 0 : t1 - t0;
}

}  // namespace rbe
