// rbe_api.cu -- the C ABI of librbe (include/rbe.h): context, workspace carving, k-vector
// upload and kernel launches.  No torch types, no device allocation, no CPU fallback.
#include "rbe.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "rbe_kernels.cuh"
#include "sr_kernels.cuh"
#include "sr_pair_kernels.cuh"
#include "sr_cell_kernels.cuh"
#include "rbl_kernels.cuh"
#include "nve_kernels.cuh"

namespace {

constexpr int NSTAGE = 8;  // pinned staging slots for k-vector uploads in flight
// rbe_step_host: at most this many chunks in the copy/compute pipeline, each of at least this many
// atoms (measured on B200, N = 1e6: 885 / 715 / 693 / 707 / 767 us per step with 1 / 2 / 4 / 8 / 16 chunks)
constexpr int HOST_MAX_CHUNKS = 4;
constexpr int64_t HOST_MIN_CHUNK = 65536;

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

}  // namespace

struct rbe_ctx {
    int64_t N = 0;
    double L = 0, alpha = 0, S = 0;
    int32_t P = 0;

    // device / launch geometry (filled by init_device)
    bool dev_ready = false;
    int device = -1;
    rbe_launch_info li{};
    int sf_gs = 0, sf_ng = 0;
    int sf_pairing = 3;
    int sr_table = 0;          // rbe_set_pair_table
    int sr_kernel = 0;         // rbe_set_pair_kernel: 0 ring kernel (cells of side r_s), 1 cell kernel (cells of side r_s / 2, tensor-core test)
    int sf_ngroups = 1;
    size_t ws_bytes = 0;
    size_t off_kvec = 0, off_w = 0, off_part = 0, off_rho = 0, off_grow = 0, off_U = 0, off_ticket = 0;
    size_t off_ka = 0, off_kb = 0, off_bar = 0, off_nve = 0;
    bool sf_deep = false;       // a thread takes more than SF_DEPTH atoms from one tile: flush inside the loops
    bool step_fused = false;    // the one-launch cooperative step kernel is usable for this context
    size_t step_smem = 0;

    // workspace
    unsigned char* ws = nullptr;
    bool have_k = false, have_w = false, have_rho = false;

    // pinned staging ring
    void* stage[NSTAGE] = {};
    cudaEvent_t stage_ev[NSTAGE] = {};
    bool stage_used[NSTAGE] = {};
    size_t stage_bytes = 0;
    int stage_next = 0;
    double* h_U_pinned = nullptr;

    // chunked host step (rbe_step_host): two copy streams and the events that order the chunks
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
    cudaEvent_t ev_start = nullptr, ev_done = nullptr;
    cudaEvent_t ev_in[HOST_MAX_CHUNKS] = {}, ev_f[HOST_MAX_CHUNKS] = {};

    // device sampler (Algorithm 1 step 1 on the GPU): integer inverse-CDF thresholds, built on the host
    std::vector<uint32_t> sampler_T;
    int32_t sampler_M = 0;
    size_t off_T = 0, off_state = 0;

    // one whole step (sampler + structure factor + force) as an instantiated CUDA graph
    cudaStream_t s_cap = nullptr;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t graph_exec = nullptr;
    bool graph_have_w = false;   // whether the captured step reads the weight table (a replay leaves the context in that state)

    // fused multi-GPU exchange of rho (rbe_set_exchange): peers' buffers, this rank, step epoch
    int32_t xch_world = 0, xch_rank = 0;
    uint32_t xch_epoch = 0;
    unsigned char* xch_buf[rbe::MAX_WORLD] = {};
    size_t off_xch_err = 0;

    const float* d_q = nullptr;   // charges on the device (rbe_set_charges), for the compact host step

    std::string err;
};

namespace {

rbe_status fail(rbe_ctx* c, rbe_status s, const std::string& msg) {
    if (c) c->err = msg;
    return s;
}

rbe_status cuda_fail(rbe_ctx* c, const char* what, cudaError_t e) {
    return fail(c, RBE_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define RBE_CUDA(ctx, call)                                   \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return cuda_fail(ctx, #call, e__); \
    } while (0)

// Which live context owns which workspace buffer.  A workspace carries state from launch to launch (the k-set, rho, the
// sampler's step counter, the arrival counter of step_kernel's grid barrier, which must stay a multiple of ONE grid size):
// two contexts on one buffer corrupt each other silently or leave a grid barrier waiting for arrivals that never come.
// No sanitizer run can vouch for the callers on this pool, so rbe_set_workspace refuses the overlap instead.
struct WsClaim { const rbe_ctx* owner; int device; uintptr_t lo, hi; };
std::mutex g_ws_mu;
std::vector<WsClaim> g_ws_claims;

void ws_release(const rbe_ctx* c) {
    std::lock_guard<std::mutex> lock(g_ws_mu);
    for (size_t i = 0; i < g_ws_claims.size();)
        if (g_ws_claims[i].owner == c) { g_ws_claims[i] = g_ws_claims.back(); g_ws_claims.pop_back(); } else ++i;
}

// true if [lo, hi) on `device` is free of every other context's claim; then it becomes c's (replacing c's previous one)
bool ws_claim(const rbe_ctx* c, int device, uintptr_t lo, uintptr_t hi) {
    std::lock_guard<std::mutex> lock(g_ws_mu);
    for (const WsClaim& w : g_ws_claims)
        if (w.owner != c && w.device == device && lo < w.hi && w.lo < hi) return false;
    for (size_t i = 0; i < g_ws_claims.size();)
        if (g_ws_claims[i].owner == c) { g_ws_claims[i] = g_ws_claims.back(); g_ws_claims.pop_back(); } else ++i;
    g_ws_claims.push_back({c, device, lo, hi});
    return true;
}

// Philox4x32-10 (Salmon et al., SC'11) on the host, for the one call per step that salts the RBL pair keys
void philox4x32_10_host(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1, uint32_t out[4]) {
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1, n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

double normaliser_S(double L, double alpha) {
    // S = H^3 - 1, H = sum_{m in Z} exp(-pi^2 m^2 / (alpha L^2))   (k = 2 pi m / L P:115)
    const double c = rbe::PI_D * rbe::PI_D / (alpha * L * L);
    double H = 1.0;
    for (int64_t m = 1; m < (int64_t)1 << 40; ++m) {
        const double t = std::exp(-c * (double)m * (double)m);
        if (!(t > 1e-300)) break;
        H += 2.0 * t;
    }
    return H * H * H - 1.0;
}

// Thresholds of the 1-D discrete Gaussian exp(-c m^2), c = pi^2 / (alpha L^2), on m = -M .. M
// (reading Q17): M = ceil(sqrt(40 ln 2 / c)); p_i summed in ascending i in fp64;
// T_i = min(2^32 - 1, floor(2^32 * CDF_i)) for i = 0 .. 2M - 1 (the last bin takes the rest).  Returns false
// when the table would be unreasonably large (the device sampler is then unavailable).
constexpr int32_t SAMPLER_M_MAX = 1 << 20;
bool build_sampler_table(double L, double alpha, std::vector<uint32_t>& T, int32_t& M) {
    const double c = rbe::PI_D * rbe::PI_D / (alpha * L * L);
    const double m = std::ceil(std::sqrt(40.0 * std::log(2.0) / c));
    if (!(m >= 1.0) || m > (double)SAMPLER_M_MAX) return false;
    M = (int32_t)m;
    std::vector<double> cum((size_t)2 * M + 1);
    double run = 0.0;
    for (int32_t i = 0; i <= 2 * M; ++i) {
        const double d = (double)(i - M);
        run += std::exp(-c * (d * d));
        cum[i] = run;
    }
    T.resize((size_t)2 * M);
    for (int32_t i = 0; i < 2 * M; ++i) {
        const double t = std::floor(4294967296.0 * (cum[i] / run));
        T[i] = t >= 4294967295.0 ? 4294967295u : (uint32_t)t;   // CDF_i can round to 1 in the far tail
    }
    return true;
}

// Choose the launch geometry for this context on the current device.
rbe_status init_device(rbe_ctx* c) {
    if (c->dev_ready) return RBE_OK;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(c, RBE_ERR_NO_DEVICE, "no CUDA device (librbe has no CPU fallback)");
    }
    RBE_CUDA(c, cudaGetDevice(&c->device));
    cudaDeviceProp prop;
    RBE_CUDA(c, cudaGetDeviceProperties(&prop, c->device));
    if (prop.major != 10)
        return fail(c, RBE_ERR_NO_DEVICE, "librbe is built for sm_100a only; device is sm_" +
                                              std::to_string(prop.major) + std::to_string(prop.minor));
    rbe_launch_info& li = c->li;
    li.num_sms = prop.multiProcessorCount;

    // ---- SF phase: a thread owns SF_KPT wavevectors; gs threads cover one k-chunk, ng atom
    // groups share a CTA of up to SF_TMAX threads (one CTA per SM).
    const int slots = (c->P + rbe::SF_KPT - 1) / rbe::SF_KPT;
    int gy = (slots + rbe::SF_TMAX - 1) / rbe::SF_TMAX;
    int gs = (slots + gy - 1) / gy;
    int ng = rbe::SF_TMAX / gs;
    if (ng < 1) ng = 1;
    int threads = (int)align_up((size_t)gs * ng, 32);
    int gx = li.num_sms / gy;
    if (gx < 1) gx = 1;
    // never more CTAs than 32-atom windows to feed them
    const int64_t max_gx = c->N > 0 ? (c->N + 31) / 32 : 1;
    if ((int64_t)gx > max_gx) gx = (int)max_gx;
    c->sf_gs = gs; c->sf_ng = ng;
    li.sf_threads = threads; li.sf_grid_x = gx;
    const int tile = (threads / 32) * rbe::SF_WPT * 32;     // atoms per tile: SF_WPT windows per warp
    c->sf_deep = (tile + ng - 1) / ng + 2 > rbe::SF_DEPTH;
    li.sf_grid_y = gy;
    li.sf_k_per_thread = rbe::SF_KPT; li.sf_atom_groups = ng; li.sf_tile_atoms = tile;
    // two record arenas (16 B per atom each) + fp64 accumulators [SF_KPT][threads]
    li.sf_smem_bytes = (int32_t)rbe::sf_smem_bytes(threads);

    c->sf_ngroups = (gx + rbe::SF_RED_GROUP - 1) / rbe::SF_RED_GROUP;
    li.sf_red_group = rbe::SF_RED_GROUP;
    li.sf_red_groups = c->sf_ngroups;

    // ---- F kernel: warps take balanced runs of 32-atom units; one wave of CTAs.
    li.f_threads = rbe::F_THREADS;
    li.f_atoms_per_thread = rbe::F_RMAX;
    const int nk = c->P < rbe::F_KCHUNK ? c->P : rbe::F_KCHUNK;
    li.f_smem_bytes = (int32_t)((size_t)nk * (sizeof(int4) + sizeof(float4)));
    // The attribute belongs to the FUNCTION, not to this context: contexts of different sizes live in one
    // process, so it is always raised to the most any context can ask for, never set to this context's need.
    const int f_smem_max = rbe::F_KCHUNK * (int)(sizeof(int4) + sizeof(float4));
    RBE_CUDA(c, cudaFuncSetAttribute(rbe::f_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, f_smem_max));
    RBE_CUDA(c, cudaFuncSetAttribute(rbe::f_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, f_smem_max));
    int occ0 = 0, occ1 = 0;  // resident CTAs per SM: the grid is exactly one wave
    RBE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ0, rbe::f_kernel<false>, rbe::F_THREADS, li.f_smem_bytes));
    RBE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ1, rbe::f_kernel<true>, rbe::F_THREADS, li.f_smem_bytes));
    int f_ctas_per_sm = occ0 < occ1 ? occ0 : occ1;
    if (f_ctas_per_sm < 1) f_ctas_per_sm = 1;
    if (f_ctas_per_sm > rbe::F_CTAS_PER_SM) f_ctas_per_sm = rbe::F_CTAS_PER_SM;
    int64_t f_grid = (int64_t)li.num_sms * f_ctas_per_sm;
    const int64_t units = (c->N + 31) / 32;
    const int64_t max_f = units > 0 ? (units + (rbe::F_THREADS / 32) - 1) / (rbe::F_THREADS / 32) : 1;
    if (f_grid > max_f) f_grid = max_f;
    li.f_grid = (int32_t)f_grid;

    const int sf_smem_max = (int)prop.sharedMemPerBlockOptin - 4 * 1024;   // (static shared memory of the kernels: < 4 KB)
    if (li.sf_smem_bytes > sf_smem_max) return fail(c, RBE_ERR_CUDA, "structure-factor kernel needs more shared memory than the device offers");
    RBE_CUDA(c, cudaFuncSetAttribute(rbe::sf_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, sf_smem_max));
    RBE_CUDA(c, cudaFuncSetAttribute(rbe::sf_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, sf_smem_max));

    // ---- one-launch step kernel (cooperative: one CTA per SM, all co-resident): one k-chunk only
    c->step_smem = (size_t)li.sf_smem_bytes;
    if ((size_t)c->P * (sizeof(int4) + sizeof(float4)) > c->step_smem) c->step_smem = (size_t)c->P * (sizeof(int4) + sizeof(float4));
    int coop = 0;
    RBE_CUDA(c, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, c->device));
    c->step_fused = coop && gy == 1 && c->P <= rbe::STEP_PMAX && c->step_smem <= (size_t)sf_smem_max && gx <= li.num_sms;
    // Beyond ~4e6 (atom, k) pairs per SM the fixed costs the single launch removes (~8 us) are under 0.5 % of the
    // step, while the two-launch force kernel (2 CTAs x 512 threads per SM) runs its loop 4 % faster than the force
    // phase of the 1024-thread step kernel (measured, N = 1e7, P = 200: 1540 against 1592 us per step).
    if ((double)c->N * (double)c->P > 4.0e6 * (double)li.num_sms) c->step_fused = false;
    if (c->step_fused) {
        RBE_CUDA(c, cudaFuncSetAttribute(rbe::step_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, sf_smem_max));
        RBE_CUDA(c, cudaFuncSetAttribute(rbe::step_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, sf_smem_max));
        RBE_CUDA(c, cudaFuncSetAttribute(rbe::step_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, sf_smem_max));
        RBE_CUDA(c, cudaFuncSetAttribute(rbe::step_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, sf_smem_max));
        int occ = 0;
        RBE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, rbe::step_kernel<true, true>, threads, c->step_smem));
        if (occ < 1) c->step_fused = false;
    }
    li.step_fused = c->step_fused ? 1 : 0;
    li.step_smem_bytes = (int32_t)c->step_smem;

    // ---- workspace layout
    size_t off = 0;
    const size_t P = (size_t)c->P;
    c->off_kvec = off; off = align_up(off + P * sizeof(int4), 256);
    c->off_w = off;    off = align_up(off + P * sizeof(double), 256);
    c->off_part = off; off = align_up(off + (size_t)gx * P * sizeof(double2), 256);
    c->off_rho = off;  off = align_up(off + P * sizeof(double2), 256);
    c->off_grow = off; off = align_up(off + (size_t)c->sf_ngroups * P * sizeof(double2), 256);
    c->off_U = off;    off = align_up(off + 8 * sizeof(double), 256);   // U, then the 6 virial components
    c->off_ticket = off; off = align_up(off + (size_t)(c->sf_ngroups + 1) * sizeof(unsigned int), 256);
    c->off_T = off;    off = align_up(off + c->sampler_T.size() * sizeof(uint32_t) + 4, 256);
    c->off_state = off; off = align_up(off + 2 * sizeof(unsigned long long), 256);
    c->off_xch_err = off; off = align_up(off + sizeof(int32_t), 256);
    c->off_ka = off;   off = align_up(off + P * sizeof(int4), 256);      // per-k force records of the step kernel
    c->off_kb = off;   off = align_up(off + P * sizeof(float4), 256);
    c->off_bar = off;  off = align_up(off + sizeof(unsigned long long), 256);   // grid-barrier arrival counter
    c->off_nve = off;  off = align_up(off + (size_t)(rbe::NVE_RED_CTAS + 1) * sizeof(double2), 256);   // partials + result of the NVE sums
    c->ws_bytes = off;

    c->stage_bytes = P * (sizeof(int4) + sizeof(double));
    c->dev_ready = true;
    return RBE_OK;
}

template <typename T>
T* ws_ptr(rbe_ctx* c, size_t off) { return reinterpret_cast<T*>(c->ws + off); }

// exchange buffer layout: slots [2][world][P] double2, then flags [2][world] uint32
size_t xch_flags_offset(int32_t world, int32_t P) { return align_up((size_t)2 * world * P * sizeof(double2), 256); }

rbe::KTable k_table(rbe_ctx* c) {
    rbe::KTable t;
    t.kvec = ws_ptr<int4>(c, c->off_kvec);
    t.w = c->have_w ? ws_ptr<double>(c, c->off_w) : nullptr;
    t.rho = ws_ptr<double2>(c, c->off_rho);
    t.w_uniform = c->S / (double)c->P;
    t.L = c->L;
    t.P = c->P;
    t.xch.world = c->xch_world;
    t.xch.epoch = c->xch_epoch;
    t.xch.slots = nullptr; t.xch.flags = nullptr;
    t.xch.error = ws_ptr<int32_t>(c, c->off_xch_err);
    if (c->xch_world > 0) {
        const size_t parity = c->xch_epoch & 1u;
        unsigned char* own = c->xch_buf[c->xch_rank];
        t.xch.slots = reinterpret_cast<const double2*>(own) + parity * (size_t)c->xch_world * (size_t)c->P;
        t.xch.flags = reinterpret_cast<const uint32_t*>(own + xch_flags_offset(c->xch_world, c->P)) + parity * (size_t)c->xch_world;
    }
    return t;
}

// Algorithm 1 step 1 on the device.  from_state: (seed, step) come from the workspace and the
// step is advanced by the kernel (graph replay); else they are the arguments.
rbe_status launch_sampler(rbe_ctx* c, bool from_state, uint64_t seed, uint64_t step, cudaStream_t st) {
    rbe::SampleParams p;
    p.T = ws_ptr<uint32_t>(c, c->off_T);
    p.M = c->sampler_M;
    p.P = c->P;
    p.kvec = ws_ptr<int4>(c, c->off_kvec);
    p.state = from_state ? ws_ptr<unsigned long long>(c, c->off_state) : nullptr;
    p.seed = seed; p.step = step;
    rbe::sample_kernel<<<1, 1024, 0, st>>>(p);
    RBE_CUDA(c, cudaGetLastError());
    return RBE_OK;
}

rbe::SfArgs sf_args(rbe_ctx* c, const void* d_xyzq, int64_t n, int accumulate) {
    rbe::SfArgs a;
    a.xyzq = static_cast<const float4*>(d_xyzq);
    a.N = n;
    a.part = ws_ptr<double2>(c, c->off_part);
    a.two32_over_L = rbe::TWO32 / c->L;
    a.P = c->P; a.gs = c->sf_gs; a.ng = c->sf_ng;
    a.pairing = c->sf_pairing;
    a.accumulate = accumulate;
    return a;
}

// One launch of the structure-factor kernel over n atoms.  accumulate: add to the per-CTA rows
// already in the workspace; finalise: run the fixed-order second pass (rows -> rho) in this launch.
rbe_status launch_sf(rbe_ctx* c, const void* d_xyzq, int64_t n, int accumulate, int finalise, void* d_rho,
                     cudaStream_t st) {
    rbe::SfParams sp;
    sp.a = sf_args(c, d_xyzq, n, accumulate);
    sp.kvec = ws_ptr<int4>(c, c->off_kvec);
    sp.finalise = finalise;
    sp.red.part = sp.a.part;
    sp.red.grow = ws_ptr<double2>(c, c->off_grow);
    sp.red.rho = ws_ptr<double2>(c, c->off_rho);
    sp.red.rho_user = static_cast<double2*>(d_rho);
    sp.red.tickets = ws_ptr<unsigned int>(c, c->off_ticket);
    sp.red.group_size = rbe::SF_RED_GROUP;
    sp.red.ngroups = c->sf_ngroups;
    sp.red.xch.world = 0;
    if (c->xch_world > 0 && finalise) {
        // one epoch per structure factor; the consumers of this step (k_table) read the same epoch
        const uint32_t epoch = ++c->xch_epoch;
        const size_t parity = epoch & 1u, fo = xch_flags_offset(c->xch_world, c->P);
        sp.red.xch.world = c->xch_world;
        sp.red.xch.epoch = epoch;
        for (int r = 0; r < c->xch_world; ++r) {
            sp.red.xch.slot[r] = reinterpret_cast<double2*>(c->xch_buf[r]) + (parity * c->xch_world + c->xch_rank) * (size_t)c->P;
            sp.red.xch.flag[r] = reinterpret_cast<uint32_t*>(c->xch_buf[r] + fo) + parity * c->xch_world + c->xch_rank;
        }
    }
    const size_t smem = (size_t)c->li.sf_smem_bytes;
    dim3 grid(c->li.sf_grid_x, c->li.sf_grid_y);
    if (c->sf_deep) rbe::sf_kernel<true><<<grid, c->li.sf_threads, smem, st>>>(sp);
    else rbe::sf_kernel<false><<<grid, c->li.sf_threads, smem, st>>>(sp);
    RBE_CUDA(c, cudaGetLastError());
    return RBE_OK;
}

// One launch of the force kernel over n atoms (programmatic dependent launch: the grid may be
// scheduled while the preceding grid drains; the kernel waits, griddepcontrol.wait, before it
// reads anything that grid wrote).
rbe_status launch_f(rbe_ctx* c, const void* d_xyzq, void* d_force, int64_t n, int with_energy, cudaStream_t st) {
    rbe::FParams fp;
    fp.a.xyzq = static_cast<const float4*>(d_xyzq);
    fp.a.force = static_cast<float4*>(d_force);
    fp.a.N = n;
    fp.a.two32_over_L = rbe::TWO32 / c->L;
    fp.kt = k_table(c);
    fp.P = c->P;
    fp.pdl = 1;
    const int64_t units = (n + 31) / 32, wpc = rbe::F_THREADS / 32;
    int64_t grid = (units + wpc - 1) / wpc;
    if (grid > c->li.f_grid) grid = c->li.f_grid;
    if (grid < 1) grid = 1;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3(c->li.f_threads);
    cfg.dynamicSmemBytes = (size_t)c->li.f_smem_bytes;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (with_energy) RBE_CUDA(c, cudaLaunchKernelEx(&cfg, rbe::f_kernel<true>, fp));
    else RBE_CUDA(c, cudaLaunchKernelEx(&cfg, rbe::f_kernel<false>, fp));
    RBE_CUDA(c, cudaGetLastError());
    return RBE_OK;
}

// The whole k-space step as ONE cooperative launch (step_kernel).  h_m != nullptr: the wavevectors ride in
// the kernel parameters (P <= STEP_KPARAM_MAX, uniform weights); else they are read from the workspace.
rbe_status launch_step(rbe_ctx* c, const int32_t* h_m, const void* d_xyzq, void* d_force, int with_energy, void* d_rho,
                       cudaStream_t st) {
    rbe::StepParams sp;
    sp.sf = sf_args(c, d_xyzq, c->N, 0);
    sp.f.xyzq = static_cast<const float4*>(d_xyzq);
    sp.f.force = static_cast<float4*>(d_force);
    sp.f.N = c->N;
    sp.f.two32_over_L = rbe::TWO32 / c->L;
    sp.kvec = ws_ptr<int4>(c, c->off_kvec);
    sp.w = c->have_w ? ws_ptr<double>(c, c->off_w) : nullptr;
    sp.w_uniform = c->S / (double)c->P;
    sp.L = c->L;
    sp.rho = ws_ptr<double2>(c, c->off_rho);
    sp.rho_user = static_cast<double2*>(d_rho);
    sp.ka = ws_ptr<int4>(c, c->off_ka);
    sp.kb = ws_ptr<float4>(c, c->off_kb);
    sp.bar = ws_ptr<unsigned long long>(c, c->off_bar);
    sp.kparam = h_m ? 1 : 0;
    if (h_m)
        for (int32_t i = 0; i < 3 * c->P; ++i) sp.km[i] = (int16_t)h_m[i];   // validated: |m_d| < 2^15
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)c->li.sf_grid_x);
    cfg.blockDim = dim3((unsigned)c->li.sf_threads);
    cfg.dynamicSmemBytes = c->step_smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;
    attr[0].val.cooperative = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (c->sf_deep) {
        if (with_energy) RBE_CUDA(c, cudaLaunchKernelEx(&cfg, rbe::step_kernel<true, true>, sp));
        else RBE_CUDA(c, cudaLaunchKernelEx(&cfg, rbe::step_kernel<true, false>, sp));
    } else {
        if (with_energy) RBE_CUDA(c, cudaLaunchKernelEx(&cfg, rbe::step_kernel<false, true>, sp));
        else RBE_CUDA(c, cudaLaunchKernelEx(&cfg, rbe::step_kernel<false, false>, sp));
    }
    return RBE_OK;
}

// Algorithm 1 steps 2-4 on the k-set in the workspace: the one-launch step kernel where it applies, else two launches
rbe_status launch_kspace(rbe_ctx* c, const void* d_xyzq, void* d_force, int with_energy, cudaStream_t st) {
    if (c->step_fused && c->xch_world == 0) return launch_step(c, nullptr, d_xyzq, d_force, with_energy, nullptr, st);
    rbe_status s = launch_sf(c, d_xyzq, c->N, 0, 1, nullptr, st);
    if (s == RBE_OK && c->N > 0) s = launch_f(c, d_xyzq, d_force, c->N, with_energy, st);
    return s;
}

rbe_status check_kvectors(rbe_ctx* c, const int32_t* h_m, const double* h_w) {
    for (int32_t l = 0; l < c->P; ++l) {
        const int32_t a = h_m[3 * l], b = h_m[3 * l + 1], d = h_m[3 * l + 2];
        if ((a == 0 && b == 0 && d == 0) || a <= -32768 || a >= 32768 || b <= -32768 || b >= 32768 ||
            d <= -32768 || d >= 32768)
            return fail(c, RBE_ERR_BAD_KVECTOR, "k-vector " + std::to_string(l) + " is zero or out of range (|m_d| < 2^15)");
        if (h_w && !std::isfinite(h_w[l]))
            return fail(c, RBE_ERR_BAD_KVECTOR, "weight " + std::to_string(l) + " is not finite");
    }
    return RBE_OK;
}

}  // namespace

extern "C" {

rbe_status rbe_create(rbe_ctx** out, int64_t N, double L, double alpha, int32_t P) {
    if (!out) return RBE_ERR_INVALID_ARG;
    *out = nullptr;
    if (N < 0 || !(L > 0.0) || !(alpha > 0.0) || P < 1 || !std::isfinite(L) || !std::isfinite(alpha) ||
        P > (1 << 20))
        return RBE_ERR_INVALID_ARG;
    rbe_ctx* c = new (std::nothrow) rbe_ctx();
    if (!c) return RBE_ERR_INVALID_ARG;
    c->N = N; c->L = L; c->alpha = alpha; c->P = P;
    c->S = normaliser_S(L, alpha);
    if (!build_sampler_table(L, alpha, c->sampler_T, c->sampler_M)) { c->sampler_T.clear(); c->sampler_M = 0; }
    *out = c;
    return RBE_OK;
}

rbe_status rbe_destroy(rbe_ctx* c) {
    if (!c) return RBE_OK;
    ws_release(c);
    for (int i = 0; i < NSTAGE; ++i) {
        if (c->stage_ev[i]) cudaEventDestroy(c->stage_ev[i]);
        if (c->stage[i]) cudaFreeHost(c->stage[i]);
    }
    if (c->h_U_pinned) cudaFreeHost(c->h_U_pinned);
    for (int i = 0; i < HOST_MAX_CHUNKS; ++i) {
        if (c->ev_in[i]) cudaEventDestroy(c->ev_in[i]);
        if (c->ev_f[i]) cudaEventDestroy(c->ev_f[i]);
    }
    if (c->ev_start) cudaEventDestroy(c->ev_start);
    if (c->ev_done) cudaEventDestroy(c->ev_done);
    if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
    if (c->graph) cudaGraphDestroy(c->graph);
    if (c->s_cap) cudaStreamDestroy(c->s_cap);
    if (c->s_h2d) cudaStreamDestroy(c->s_h2d);
    if (c->s_d2h) cudaStreamDestroy(c->s_d2h);
    delete c;
    return RBE_OK;
}

double rbe_normaliser_S(const rbe_ctx* c) { return c ? c->S : 0.0; }

size_t rbe_workspace_bytes(const rbe_ctx* cc) {
    if (!cc) return 0;
    rbe_ctx* c = const_cast<rbe_ctx*>(cc);   // the launch geometry is a lazily filled cache of the context
    if (init_device(c) != RBE_OK) return 0;
    return c->ws_bytes;
}

rbe_status rbe_set_workspace(rbe_ctx* c, void* d_ws, size_t bytes) {
    if (!c) return RBE_ERR_INVALID_ARG;
    rbe_status s = init_device(c);
    if (s != RBE_OK) return s;
    if (!d_ws || bytes < c->ws_bytes || (reinterpret_cast<uintptr_t>(d_ws) & 255u))
        return fail(c, RBE_ERR_WORKSPACE, "workspace must be non-null, 256-byte aligned and >= rbe_workspace_bytes");
    // only the bytes this context uses are claimed: a caller may carve several workspaces out of one allocation
    if (!ws_claim(c, c->device, reinterpret_cast<uintptr_t>(d_ws), reinterpret_cast<uintptr_t>(d_ws) + c->ws_bytes))
        return fail(c, RBE_ERR_WORKSPACE, "rbe_set_workspace: the buffer overlaps the workspace of another live context "
                                          "(a workspace belongs to one context until that context is destroyed or given another buffer)");
    c->ws = static_cast<unsigned char*>(d_ws);
    c->have_k = c->have_w = c->have_rho = false;
    // the structure-factor kernel's completion ticket starts at zero and resets itself
    RBE_CUDA(c, cudaMemset(c->ws + c->off_ticket, 0, (size_t)(c->sf_ngroups + 1) * sizeof(unsigned int)));
    if (!c->sampler_T.empty())
        RBE_CUDA(c, cudaMemcpy(c->ws + c->off_T, c->sampler_T.data(), c->sampler_T.size() * sizeof(uint32_t), cudaMemcpyHostToDevice));
    RBE_CUDA(c, cudaMemset(c->ws + c->off_state, 0, 2 * sizeof(unsigned long long)));
    RBE_CUDA(c, cudaMemset(c->ws + c->off_xch_err, 0, sizeof(int32_t)));
    RBE_CUDA(c, cudaMemset(c->ws + c->off_bar, 0, sizeof(unsigned long long)));
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }   // bound to the old workspace
    if (c->graph) { cudaGraphDestroy(c->graph); c->graph = nullptr; }
    RBE_CUDA(c, cudaDeviceSynchronize());
    return RBE_OK;
}

rbe_status rbe_set_pairing(rbe_ctx* c, int32_t mode) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if (mode != 0 && mode != 1 && mode != 3) return fail(c, RBE_ERR_INVALID_ARG, "rbe_set_pairing: mode must be 0, 1 or 3");
    c->sf_pairing = mode;
    return RBE_OK;
}

rbe_status rbe_set_pair_kernel(rbe_ctx* c, int32_t kind) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if (kind != 0 && kind != 1) return fail(c, RBE_ERR_INVALID_ARG, "rbe_set_pair_kernel: kind must be 0 or 1");
    c->sr_kernel = kind;
    return RBE_OK;
}

rbe_status rbe_pair_table_host(const rbe_ctx* c, double rs, float* h_tf, float* h_te, int32_t capacity, int32_t* n_out) {
    if (!c || !(rs > 0.0) || !std::isfinite(rs) || !n_out) return RBE_ERR_INVALID_ARG;
    const int emax = (int)std::floor(std::log2(rs * rs)) + 1;
    int ntab = (emax - rbe::SR_TAB_EMIN) << rbe::SR_TAB_BITS;
    if (ntab < (1 << rbe::SR_TAB_BITS)) ntab = 1 << rbe::SR_TAB_BITS;
    if (ntab > rbe::SR_TAB_MAX) return RBE_ERR_INVALID_ARG;
    *n_out = ntab;
    if (!h_tf && !h_te) return RBE_OK;                       // size query
    if (capacity < ntab) return RBE_ERR_INVALID_ARG;
    for (int i = 0; i < ntab; ++i) {
        float4 f, e;
        rbe::sr_table_entry(i, c->alpha, f, e);
        if (h_tf) { h_tf[4 * i] = f.x; h_tf[4 * i + 1] = f.y; h_tf[4 * i + 2] = f.z; h_tf[4 * i + 3] = f.w; }
        if (h_te) { h_te[4 * i] = e.x; h_te[4 * i + 1] = e.y; h_te[4 * i + 2] = e.z; h_te[4 * i + 3] = e.w; }
    }
    return RBE_OK;
}

rbe_status rbe_set_pair_table(rbe_ctx* c, int32_t on) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if (on != 0 && on != 1) return fail(c, RBE_ERR_INVALID_ARG, "rbe_set_pair_table: on must be 0 or 1");
    c->sr_table = on;
    return RBE_OK;
}

rbe_status rbe_get_launch_info(const rbe_ctx* c, rbe_launch_info* out) {
    if (!c || !out) return RBE_ERR_INVALID_ARG;
    if (!c->dev_ready) return RBE_ERR_NOT_READY;
    *out = c->li;
    return RBE_OK;
}

rbe_status rbe_set_kvectors(rbe_ctx* c, const int32_t* h_m, const double* h_w, void* stream) {
    if (!c || !h_m) return fail(c, RBE_ERR_INVALID_ARG, "rbe_set_kvectors: null argument");
    // validate first: independent of the device state
    const rbe_status vs = check_kvectors(c, h_m, h_w);
    if (vs != RBE_OK) return vs;
    if (!c->ws) return fail(c, RBE_ERR_NOT_READY, "rbe_set_kvectors before rbe_set_workspace");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int slot = c->stage_next;
    c->stage_next = (slot + 1) % NSTAGE;
    if (!c->stage[slot]) {
        RBE_CUDA(c, cudaMallocHost(&c->stage[slot], c->stage_bytes));
        RBE_CUDA(c, cudaEventCreateWithFlags(&c->stage_ev[slot], cudaEventDisableTiming));
    } else if (c->stage_used[slot]) {
        RBE_CUDA(c, cudaEventSynchronize(c->stage_ev[slot]));
    }
    int4* hm = static_cast<int4*>(c->stage[slot]);
    for (int32_t l = 0; l < c->P; ++l) hm[l] = make_int4(h_m[3 * l], h_m[3 * l + 1], h_m[3 * l + 2], 0);
    size_t bytes = (size_t)c->P * sizeof(int4);
    RBE_CUDA(c, cudaMemcpyAsync(c->ws + c->off_kvec, hm, bytes, cudaMemcpyHostToDevice, st));
    if (h_w) {
        double* hw = reinterpret_cast<double*>(hm + c->P);
        std::memcpy(hw, h_w, (size_t)c->P * sizeof(double));
        RBE_CUDA(c, cudaMemcpyAsync(c->ws + c->off_w, hw, (size_t)c->P * sizeof(double), cudaMemcpyHostToDevice, st));
    }
    RBE_CUDA(c, cudaEventRecord(c->stage_ev[slot], st));
    c->stage_used[slot] = true;
    c->have_k = true;
    c->have_w = (h_w != nullptr);
    c->have_rho = false;
    return RBE_OK;
}

rbe_status rbe_structure_factor(rbe_ctx* c, const void* d_xyzq, void* d_rho, void* stream) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if (!c->ws || !c->have_k) return fail(c, RBE_ERR_NOT_READY, "rbe_structure_factor needs a workspace and k-vectors");
    if ((c->N > 0 && !d_xyzq) || (reinterpret_cast<uintptr_t>(d_xyzq) & 15u) || (reinterpret_cast<uintptr_t>(d_rho) & 15u))
        return fail(c, RBE_ERR_INVALID_ARG, "rbe_structure_factor: null or misaligned pointer");
    rbe_status s = launch_sf(c, d_xyzq, c->N, 0, 1, d_rho, static_cast<cudaStream_t>(stream));
    if (s != RBE_OK) return s;
    c->have_rho = true;
    return RBE_OK;
}

rbe_status rbe_set_rho(rbe_ctx* c, const void* d_rho, void* stream) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if (!c->ws || !c->have_k) return fail(c, RBE_ERR_NOT_READY, "rbe_set_rho needs a workspace and k-vectors");
    if (!d_rho || (reinterpret_cast<uintptr_t>(d_rho) & 15u))
        return fail(c, RBE_ERR_INVALID_ARG, "rbe_set_rho: null or misaligned pointer");
    if (c->xch_world > 0) return fail(c, RBE_ERR_INVALID_ARG, "rbe_set_rho: a fused exchange is configured (rbe_set_exchange)");
    RBE_CUDA(c, cudaMemcpyAsync(c->ws + c->off_rho, d_rho, (size_t)c->P * sizeof(double2), cudaMemcpyDeviceToDevice,
                                static_cast<cudaStream_t>(stream)));
    c->have_rho = true;
    return RBE_OK;
}

rbe_status rbe_forces(rbe_ctx* c, const void* d_xyzq, void* d_force, int32_t with_energy, void* stream) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if (!c->ws || !c->have_k || !c->have_rho)
        return fail(c, RBE_ERR_NOT_READY, "rbe_forces needs rbe_structure_factor (or rbe_set_rho) after rbe_set_kvectors");
    if (c->N == 0) return RBE_OK;
    if (!d_xyzq || !d_force || (reinterpret_cast<uintptr_t>(d_xyzq) & 15u) || (reinterpret_cast<uintptr_t>(d_force) & 15u))
        return fail(c, RBE_ERR_INVALID_ARG, "rbe_forces: null or misaligned pointer");
    return launch_f(c, d_xyzq, d_force, c->N, with_energy, static_cast<cudaStream_t>(stream));
}

rbe_status rbe_step(rbe_ctx* c, const int32_t* h_m, const double* h_w, const void* d_xyzq, void* d_force, int32_t with_energy,
                    void* d_rho, void* stream) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if (!c->ws) return fail(c, RBE_ERR_NOT_READY, "rbe_step before rbe_set_workspace");
    if (!h_m && h_w) return fail(c, RBE_ERR_INVALID_ARG, "rbe_step: weights without wavevectors");
    if (!h_m && !c->have_k) return fail(c, RBE_ERR_NOT_READY, "rbe_step: no k-set (pass h_m, or call rbe_set_kvectors / rbe_sample_kvectors first)");
    if ((c->N > 0 && (!d_xyzq || !d_force)) || (reinterpret_cast<uintptr_t>(d_xyzq) & 15u) || (reinterpret_cast<uintptr_t>(d_force) & 15u) ||
        (reinterpret_cast<uintptr_t>(d_rho) & 15u))
        return fail(c, RBE_ERR_INVALID_ARG, "rbe_step: null or misaligned pointer");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const bool fused = c->step_fused && c->xch_world == 0;
    rbe_status s = RBE_OK;
    if (h_m) {
        if (fused && !h_w && c->P <= rbe::STEP_KPARAM_MAX) {
            // the wavevectors travel in the kernel parameters: validate here, no copy, no staging
            s = check_kvectors(c, h_m, nullptr);
            if (s != RBE_OK) return s;
            c->have_k = true; c->have_w = false; c->have_rho = false;
            s = launch_step(c, h_m, d_xyzq, d_force, with_energy, d_rho, st);
            if (s == RBE_OK) c->have_rho = true;
            return s;
        }
        s = rbe_set_kvectors(c, h_m, h_w, stream);
        if (s != RBE_OK) return s;
    }
    if (fused) {
        s = launch_step(c, nullptr, d_xyzq, d_force, with_energy, d_rho, st);
        if (s == RBE_OK) c->have_rho = true;
        return s;
    }
    // several k-chunks (P > 4096), a multi-GPU exchange, or no cooperative launch: the two-launch path
    s = rbe_structure_factor(c, d_xyzq, d_rho, stream);
    if (s != RBE_OK) return s;
    return rbe_forces(c, d_xyzq, d_force, with_energy, stream);
}

rbe_status rbe_kspace_energy(rbe_ctx* c, double* h_U, void* stream) {
    if (!c || !h_U) return fail(c, RBE_ERR_INVALID_ARG, "rbe_kspace_energy: null argument");
    if (!c->ws || !c->have_k || !c->have_rho) return fail(c, RBE_ERR_NOT_READY, "rbe_kspace_energy needs a structure factor");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (!c->h_U_pinned) RBE_CUDA(c, cudaMallocHost(reinterpret_cast<void**>(&c->h_U_pinned), sizeof(double)));
    rbe::energy_kernel<<<1, 256, 0, st>>>(k_table(c), c->P, ws_ptr<double>(c, c->off_U));
    RBE_CUDA(c, cudaGetLastError());
    RBE_CUDA(c, cudaMemcpyAsync(c->h_U_pinned, c->ws + c->off_U, sizeof(double), cudaMemcpyDeviceToHost, st));
    RBE_CUDA(c, cudaStreamSynchronize(st));
    *h_U = *c->h_U_pinned;
    return RBE_OK;
}

rbe_status rbe_sample_kvectors(rbe_ctx* c, uint64_t seed, uint64_t step, void* stream) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if (!c->ws) return fail(c, RBE_ERR_NOT_READY, "rbe_sample_kvectors before rbe_set_workspace");
    if (c->sampler_T.empty()) return fail(c, RBE_ERR_INVALID_ARG, "rbe_sample_kvectors: the inverse-CDF table for this L, alpha is too large");
    rbe_status s = launch_sampler(c, false, seed, step, static_cast<cudaStream_t>(stream));
    if (s != RBE_OK) return s;
    c->have_k = true; c->have_w = false; c->have_rho = false;
    return RBE_OK;
}

rbe_status rbe_get_kvectors(rbe_ctx* c, int32_t* h_m, void* stream) {
    if (!c || !h_m) return fail(c, RBE_ERR_INVALID_ARG, "rbe_get_kvectors: null argument");
    if (!c->ws || !c->have_k) return fail(c, RBE_ERR_NOT_READY, "rbe_get_kvectors: no k-set");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    std::vector<int4> tmp((size_t)c->P);
    RBE_CUDA(c, cudaMemcpyAsync(tmp.data(), c->ws + c->off_kvec, tmp.size() * sizeof(int4), cudaMemcpyDeviceToHost, st));
    RBE_CUDA(c, cudaStreamSynchronize(st));
    for (int32_t l = 0; l < c->P; ++l) { h_m[3 * l] = tmp[l].x; h_m[3 * l + 1] = tmp[l].y; h_m[3 * l + 2] = tmp[l].z; }
    return RBE_OK;
}

rbe_status rbe_graph_capture(rbe_ctx* c, const void* d_xyzq, void* d_force, int32_t with_energy, uint64_t seed,
                             uint64_t first_step) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if (!c->ws) return fail(c, RBE_ERR_NOT_READY, "rbe_graph_capture before rbe_set_workspace");
    if (c->sampler_T.empty()) return fail(c, RBE_ERR_INVALID_ARG, "rbe_graph_capture: the device sampler is unavailable for this L, alpha");
    if (c->xch_world > 0) return fail(c, RBE_ERR_INVALID_ARG, "rbe_graph_capture: not available with a fused exchange (the epoch is a launch argument)");
    if (c->N > 0 && (!d_xyzq || !d_force || (reinterpret_cast<uintptr_t>(d_xyzq) & 15u) || (reinterpret_cast<uintptr_t>(d_force) & 15u)))
        return fail(c, RBE_ERR_INVALID_ARG, "rbe_graph_capture: null or misaligned pointer");
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    if (c->graph) { cudaGraphDestroy(c->graph); c->graph = nullptr; }
    if (!c->s_cap) RBE_CUDA(c, cudaStreamCreateWithFlags(&c->s_cap, cudaStreamNonBlocking));
    const unsigned long long st8[2] = {seed, first_step};
    RBE_CUDA(c, cudaMemcpy(c->ws + c->off_state, st8, sizeof(st8), cudaMemcpyHostToDevice));
    RBE_CUDA(c, cudaStreamBeginCapture(c->s_cap, cudaStreamCaptureModeThreadLocal));
    rbe_status s = launch_sampler(c, true, 0, 0, c->s_cap);
    c->have_w = false;   // the graph's batch carries the uniform weights S / P
    if (s == RBE_OK) s = launch_kspace(c, d_xyzq, d_force, with_energy, c->s_cap);
    cudaGraph_t g = nullptr;
    const cudaError_t e = cudaStreamEndCapture(c->s_cap, &g);
    if (s != RBE_OK) { if (g) cudaGraphDestroy(g); return s; }
    if (e != cudaSuccess) return cuda_fail(c, "cudaStreamEndCapture", e);
    c->graph = g;
    c->graph_have_w = false;
    RBE_CUDA(c, cudaGraphInstantiate(&c->graph_exec, c->graph, 0));
    return RBE_OK;
}

rbe_status rbe_graph_launch(rbe_ctx* c, void* stream) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if (!c->graph_exec) return fail(c, RBE_ERR_NOT_READY, "rbe_graph_launch before rbe_graph_capture");
    RBE_CUDA(c, cudaGraphLaunch(c->graph_exec, static_cast<cudaStream_t>(stream)));
    c->have_k = true; c->have_w = c->graph_have_w; c->have_rho = true;
    return RBE_OK;
}

size_t rbe_exchange_bytes(const rbe_ctx* c, int32_t world) {
    if (!c || world < 1 || world > rbe::MAX_WORLD) return 0;
    return xch_flags_offset(world, c->P) + align_up((size_t)2 * world * sizeof(uint32_t), 256);
}

rbe_status rbe_set_exchange(rbe_ctx* c, int32_t rank, int32_t world, void* const* d_bufs, size_t bytes) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if (world < 1 || !d_bufs) {   // switch the exchange off
        c->xch_world = 0; c->xch_rank = 0;
        return RBE_OK;
    }
    if (world > rbe::MAX_WORLD || rank < 0 || rank >= world)
        return fail(c, RBE_ERR_INVALID_ARG, "rbe_set_exchange: need 0 <= rank < world <= " + std::to_string(rbe::MAX_WORLD));
    if (bytes < rbe_exchange_bytes(c, world)) return fail(c, RBE_ERR_WORKSPACE, "rbe_set_exchange: buffers smaller than rbe_exchange_bytes");
    for (int r = 0; r < world; ++r)
        if (!d_bufs[r] || (reinterpret_cast<uintptr_t>(d_bufs[r]) & 255u))
            return fail(c, RBE_ERR_INVALID_ARG, "rbe_set_exchange: null or misaligned buffer of rank " + std::to_string(r));
    for (int r = 0; r < world; ++r) c->xch_buf[r] = static_cast<unsigned char*>(d_bufs[r]);
    c->xch_world = world; c->xch_rank = rank; c->xch_epoch = 0;
    c->have_rho = false;
    return RBE_OK;
}

rbe_status rbe_exchange_check(rbe_ctx* c, void* stream) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if (!c->ws) return fail(c, RBE_ERR_NOT_READY, "rbe_exchange_check before rbe_set_workspace");
    int32_t e = 0;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    RBE_CUDA(c, cudaMemcpyAsync(&e, c->ws + c->off_xch_err, sizeof(e), cudaMemcpyDeviceToHost, st));
    RBE_CUDA(c, cudaStreamSynchronize(st));
    if (e) return fail(c, RBE_ERR_CUDA, "fused exchange: a peer's structure factors did not arrive within 10 s");
    return RBE_OK;
}

// ---- real-space partner (Eq. 2.10 truncated at r_s): workspace layout and launches
namespace {
struct SrLayout {
    int nc = 0;
    int64_t ncell = 0;
    size_t off_turns = 0, off_sorted = 0, off_cell = 0, off_order = 0, off_sidx = 0, off_count = 0, off_cursor = 0, off_start = 0;
    size_t off_acc = 0, off_gbox = 0, off_tab = 0;
    size_t bytes = 0;
};
// cells of side >= cell_min; `need` distinct cells per dimension (the stencil must not meet itself around the box)
bool sr_layout(const rbe_ctx* c, double cell_min, int need, SrLayout& l) {
    if (!c || !(cell_min > 0.0) || !std::isfinite(cell_min) || c->N >= ((int64_t)1 << 32)) return false;
    const double ncd = std::floor(c->L / cell_min);
    if (ncd < (double)need) return false;
    l.nc = ncd > 512.0 ? 512 : (int)ncd;               // larger cells are still correct (side >= cell_min)
    l.ncell = (int64_t)l.nc * l.nc * l.nc;
    const size_t N = (size_t)c->N, nce = (size_t)l.ncell;
    size_t off = 0;
    l.off_turns = off;  off = align_up(off + N * sizeof(uint4), 256);
    l.off_sorted = off; off = align_up(off + N * sizeof(uint4), 256);
    l.off_cell = off;   off = align_up(off + N * sizeof(int32_t), 256);
    l.off_order = off;  off = align_up(off + N * sizeof(uint32_t), 256);
    l.off_sidx = off;   off = align_up(off + N * sizeof(uint32_t), 256);
    l.off_count = off;  off = align_up(off + nce * sizeof(uint32_t), 256);
    l.off_cursor = off; off = align_up(off + nce * sizeof(uint32_t), 256);
    l.off_start = off;  off = align_up(off + (nce + 1) * sizeof(uint32_t), 256);
    l.off_acc = off;    off = align_up(off + N * 4 * sizeof(long long), 256);
    l.off_gbox = off;   off = align_up(off + nce * rbe::SR_GMAX * 6 * sizeof(float), 256);
    l.off_tab = off;    off = align_up(off + 2 * (size_t)rbe::SR_TAB_MAX * sizeof(float4), 256);   // pair-term tables (force, energy)
    l.bytes = off;
    return true;
}
}  // namespace

namespace {
// The cell kernel's list: cells of side >= r_s / 2 (125-cell stencil, R = 2) where the box holds five of them per dimension,
// else cells of side >= r_s (27-cell stencil, R = 1): the stencil must not meet itself around the box.
bool sr_cell_layout(const rbe_ctx* c, double rs, SrLayout& l, int& R) {
    if (!c || !(rs > 0.0) || !std::isfinite(rs)) return false;
    if (sr_layout(c, 0.5 * rs, 5, l)) R = 2;
    else if (sr_layout(c, rs, 3, l)) R = 1;
    else return false;
    return true;
}
}  // namespace

size_t rbe_short_range_bytes(const rbe_ctx* c, double rs) {
    SrLayout l, l2;
    int R;
    if (!sr_layout(c, rs, 3, l)) return 0;             // the 27-cell stencil needs 3 distinct cells per dimension
    if (sr_cell_layout(c, rs, l2, R) && l2.bytes > l.bytes) return l2.bytes;   // enough for either kernel (rbe_set_pair_kernel)
    return l.bytes;
}

namespace {
// Random batch list: cells of side >= r_c as Algorithm 2 says, but never so small that the stencil
// exceeds 9^3 cells; R = cells the shell reaches beyond the atom's own; 2R + 1 distinct cells per dimension.
bool rbl_layout(const rbe_ctx* c, double rc, double rs, SrLayout& l, int& R) {
    if (!c || !(rc > 0.0) || !(rc < rs) || !std::isfinite(rs)) return false;
    const double cell_min = rc > rs / 4.0 ? rc : rs / 4.0;
    if (!sr_layout(c, cell_min, 3, l)) return false;
    R = (int)std::ceil(rs / (c->L / l.nc) - 1e-12);
    if (R < 1) R = 1;
    if (R > 4 || 2 * R + 1 > l.nc) return false;
    return true;
}
}  // namespace

size_t rbe_rbl_bytes(const rbe_ctx* c, double rc, double rs) {
    SrLayout l;
    int R;
    return rbl_layout(c, rc, rs, l, R) ? l.bytes : 0;
}

namespace {
struct SrBuffers {
    uint4 *turns, *sorted;
    int32_t* cell_of;
    uint32_t *order, *sidx, *count, *cursor, *start;
    long long* acc;
    float* gbox;
    float4* tab;
};
// argument checks + the linked-cell list (bin, scan, scatter, sort) shared by rbe_short_range and rbe_rbl_forces
rbe_status sr_build_cells(rbe_ctx* c, const char* who, const void* d_xyzq, void* d_force, void* d_ws,
                          size_t ws_bytes, cudaStream_t st, const SrLayout& l, SrBuffers& b) {
    rbe_status s0 = init_device(c);
    if (s0 != RBE_OK) return s0;
    if (c->N == 0) return RBE_OK;
    if (!d_xyzq || !d_force || (reinterpret_cast<uintptr_t>(d_xyzq) & 15u) || (reinterpret_cast<uintptr_t>(d_force) & 15u))
        return fail(c, RBE_ERR_INVALID_ARG, std::string(who) + ": null or misaligned pointer");
    if (!d_ws || ws_bytes < l.bytes || (reinterpret_cast<uintptr_t>(d_ws) & 255u))
        return fail(c, RBE_ERR_WORKSPACE, std::string(who) + ": d_ws must hold rbe_short_range_bytes bytes, 256-byte aligned");
    unsigned char* w = static_cast<unsigned char*>(d_ws);
    b.turns = reinterpret_cast<uint4*>(w + l.off_turns);
    b.sorted = reinterpret_cast<uint4*>(w + l.off_sorted);
    b.cell_of = reinterpret_cast<int32_t*>(w + l.off_cell);
    b.order = reinterpret_cast<uint32_t*>(w + l.off_order);
    b.sidx = reinterpret_cast<uint32_t*>(w + l.off_sidx);
    b.count = reinterpret_cast<uint32_t*>(w + l.off_count);
    b.cursor = reinterpret_cast<uint32_t*>(w + l.off_cursor);
    b.start = reinterpret_cast<uint32_t*>(w + l.off_start);
    b.acc = reinterpret_cast<long long*>(w + l.off_acc);
    b.gbox = reinterpret_cast<float*>(w + l.off_gbox);
    b.tab = reinterpret_cast<float4*>(w + l.off_tab);
    const unsigned nb = (unsigned)((c->N + 255) / 256);
    RBE_CUDA(c, cudaMemsetAsync(b.count, 0, (size_t)l.ncell * sizeof(uint32_t), st));
    rbe::sr_bin_kernel<<<nb, 256, 0, st>>>(static_cast<const float4*>(d_xyzq), c->N, rbe::TWO32 / c->L, l.nc, b.turns, b.cell_of, b.count);
    rbe::sr_scan_kernel<<<1, 1024, 0, st>>>(b.count, (int)l.ncell, b.start, b.cursor);
    rbe::sr_scatter_kernel<<<nb, 256, 0, st>>>(b.cell_of, c->N, b.start, b.cursor, b.order);
    rbe::sr_sort_kernel<<<(unsigned)((l.ncell * 32 + 255) / 256), 256, 0, st>>>(b.order, b.start, (int)l.ncell, l.nc, b.turns, b.sorted, b.sidx);
    RBE_CUDA(c, cudaGetLastError());
    return RBE_OK;
}
}  // namespace

namespace {
// rbe_short_range with the cell kernel (rbe_set_pair_kernel(ctx, 1)): the same linked-cell build on finer cells, then ONE
// force kernel that writes the caller's array directly.
rbe_status short_range_cells(rbe_ctx* c, const void* d_xyzq, double rs, void* d_force, int32_t accumulate, int32_t with_energy,
                             void* d_ws, size_t ws_bytes, cudaStream_t st) {
    SrLayout l;
    SrBuffers b;
    int R = 0;
    if (!sr_cell_layout(c, rs, l, R)) return fail(c, RBE_ERR_INVALID_ARG, "rbe_short_range: invalid r_s");
    rbe_status s = sr_build_cells(c, "rbe_short_range", d_xyzq, d_force, d_ws, ws_bytes, st, l, b);
    if (s != RBE_OK || c->N == 0) return s;
    rbe::SrCellParams pp;
    pp.sorted = b.sorted; pp.sidx = b.sidx; pp.start = b.start;
    pp.force = static_cast<float4*>(d_force);
    pp.nc = l.nc; pp.R = R; pp.accumulate = accumulate;
    pp.len_unit = (float)(c->L / rbe::TWO32);
    const double cell_len = c->L / l.nc;
    pp.rs2 = (float)(rs * rs);
    // margin of the tensor-core cutoff test: the own atom is rounded to TF32 (<= 2^-12 cell sides per component, i.e.
    // |dr| <= sqrt(3) 2^-12 cell sides), plus 2e-5 |x|^2_max for the fp32 / TF32 rounding of the sums (candidates lie within
    // R + 1/2 cell sides of the cell centre per component)
    const double dr = std::sqrt(3.0) * cell_len / 4096.0, xmax = (R + 0.5) * cell_len;
    const double margin = 1.5 * (2.0 * rs * dr + dr * dr) + 2e-5 * 3.0 * xmax * xmax;
    pp.thr = (float)(rs * rs + margin);
    pp.sqrt_alpha = (float)std::sqrt(c->alpha);
    pp.nalpha_log2e = (float)(-c->alpha * 1.4426950408889634);
    // the pair-term table: up to past r_s^2 + 2 margins (what can pass the test; the exact test then zeroes it)
    const int emax = (int)std::floor(std::log2(rs * rs + 2.0 * margin)) + 1;
    int ntab = (emax - rbe::SR_TAB_EMIN) << rbe::SR_TAB_BITS;
    if (ntab < (1 << rbe::SR_TAB_BITS)) ntab = 1 << rbe::SR_TAB_BITS;
    if (ntab > rbe::SR_TAB_MAX) return fail(c, RBE_ERR_INVALID_ARG, "rbe_short_range: r_s too large for the pair-term table");
    pp.ntab = ntab;
    pp.tab_f = b.tab; pp.tab_e = b.tab + rbe::SR_TAB_MAX;
    pp.tab_umin = (float)std::ldexp(1.0, rbe::SR_TAB_EMIN);
    // candidate list in shared memory: 1.5 x the mean number of candidates of a cell, in steps of 256
    const int side = 2 * R + 1;
    const double mean_cand = (double)c->N / (double)l.ncell * (double)(side * side * side);
    int cap = (int)std::ceil(1.5 * mean_cand / 256.0) * 256 + 256;
    if (cap > rbe::SR_CAP_MAX) cap = rbe::SR_CAP_MAX;
    pp.cap = cap;
    const bool table = c->sr_table != 0;
    const size_t dyn = rbe::sr_cell_smem_bytes(ntab, table, with_energy != 0, cap);
    const int dyn_max = (int)rbe::sr_cell_smem_bytes(rbe::SR_TAB_MAX, true, true, rbe::SR_CAP_MAX);
    const unsigned grid = (unsigned)l.ncell, block = 32 * rbe::SR_W;
    if (table) rbe::sr_table_kernel<<<(unsigned)((ntab + 127) / 128), 128, 0, st>>>(b.tab, b.tab + rbe::SR_TAB_MAX, ntab, c->alpha);
#define RBE_SR_CELL_LAUNCH(E, T)                                                                                              \
    do {                                                                                                                      \
        RBE_CUDA(c, cudaFuncSetAttribute(rbe::sr_cell_kernel<E, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn_max));   \
        rbe::sr_cell_kernel<E, T><<<grid, block, dyn, st>>>(pp);                                                              \
    } while (0)
    if (with_energy) { if (table) RBE_SR_CELL_LAUNCH(true, true); else RBE_SR_CELL_LAUNCH(true, false); }
    else { if (table) RBE_SR_CELL_LAUNCH(false, true); else RBE_SR_CELL_LAUNCH(false, false); }
#undef RBE_SR_CELL_LAUNCH
    RBE_CUDA(c, cudaGetLastError());
    return RBE_OK;
}
}  // namespace

rbe_status rbe_short_range(rbe_ctx* c, const void* d_xyzq, double rs, void* d_force, int32_t accumulate,
                           int32_t with_energy, void* d_ws, size_t ws_bytes, void* stream) {
    if (!c) return RBE_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    SrLayout l;
    SrBuffers b;
    if (!sr_layout(c, rs, 3, l))
        return fail(c, RBE_ERR_INVALID_ARG, "rbe_short_range: need 0 < r_s <= L/3 (three cells of side >= r_s per dimension) and N < 2^32");
    if (c->sr_kernel == 1) return short_range_cells(c, d_xyzq, rs, d_force, accumulate, with_energy, d_ws, ws_bytes, st);
    rbe_status s = sr_build_cells(c, "rbe_short_range", d_xyzq, d_force, d_ws, ws_bytes, st, l, b);
    if (s != RBE_OK || c->N == 0) return s;
    const unsigned nb = (unsigned)((c->N + 255) / 256);
    const float len_unit = (float)(c->L / rbe::TWO32);
    RBE_CUDA(c, cudaMemsetAsync(b.acc, 0, (size_t)c->N * 4 * sizeof(long long), st));
    rbe::sr_gbox_kernel<<<(unsigned)((l.ncell * 32 + 255) / 256), 256, 0, st>>>(b.sorted, b.start, (int)l.ncell, l.nc, len_unit, b.gbox);
    rbe::SrPairParams pp;
    pp.sorted = b.sorted; pp.start = b.start; pp.gbox = b.gbox; pp.acc = b.acc;
    pp.nc = l.nc;
    pp.len_unit = len_unit;
    pp.cell_len = (float)(c->L / l.nc);
    pp.rs2 = (float)(rs * rs);
    pp.sqrt_alpha = (float)std::sqrt(c->alpha);
    pp.nalpha_log2e = (float)(-c->alpha * 1.4426950408889634);
    // the pair-term table: the octaves of u = r^2 from 2^EMIN up to r_s^2 (only pairs with r^2 < r_s^2 look it up)
    const int emax = (int)std::floor(std::log2(rs * rs)) + 1;
    int ntab = (emax - rbe::SR_TAB_EMIN) << rbe::SR_TAB_BITS;
    if (ntab < (1 << rbe::SR_TAB_BITS)) ntab = 1 << rbe::SR_TAB_BITS;
    if (ntab > rbe::SR_TAB_MAX) return fail(c, RBE_ERR_INVALID_ARG, "rbe_short_range: r_s too large for the pair-term table");
    pp.ntab = ntab;
    pp.tab_f = b.tab; pp.tab_e = b.tab + rbe::SR_TAB_MAX;
    pp.tab_umin = (float)std::ldexp(1.0, rbe::SR_TAB_EMIN);
    const bool table = c->sr_table != 0;
    const size_t dyn = rbe::sr_pair_smem_bytes(ntab, table, with_energy != 0);
    const unsigned grid = (unsigned)l.ncell, block = 32 * rbe::SR_PAIR_WARPS;
    if (table) {
        rbe::sr_table_kernel<<<(unsigned)((ntab + 127) / 128), 128, 0, st>>>(b.tab, b.tab + rbe::SR_TAB_MAX, ntab, c->alpha);
        RBE_CUDA(c, cudaFuncSetAttribute(rbe::sr_pair_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * rbe::SR_TAB_MAX * (int)sizeof(float4)));
        RBE_CUDA(c, cudaFuncSetAttribute(rbe::sr_pair_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, rbe::SR_TAB_MAX * (int)sizeof(float4)));
        if (with_energy) rbe::sr_pair_kernel<true, true><<<grid, block, dyn, st>>>(pp);
        else rbe::sr_pair_kernel<false, true><<<grid, block, dyn, st>>>(pp);
    } else {
        if (with_energy) rbe::sr_pair_kernel<true, false><<<grid, block, 0, st>>>(pp);
        else rbe::sr_pair_kernel<false, false><<<grid, block, 0, st>>>(pp);
    }
    rbe::sr_finalize_kernel<<<nb, 256, 0, st>>>(b.acc, b.sorted, b.sidx, c->N, static_cast<float4*>(d_force), accumulate, with_energy);
    RBE_CUDA(c, cudaGetLastError());
    return RBE_OK;
}

rbe_status rbe_rbl_forces(rbe_ctx* c, const void* d_xyzq, double rc, double rs, int32_t p, uint64_t seed, uint64_t step,
                          void* d_force, int32_t accumulate, void* d_ws, size_t ws_bytes, void* stream) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if (!(rc > 0.0) || !(rc < rs) || p < 1 || p > rbe::RBL_PMAX)
        return fail(c, RBE_ERR_INVALID_ARG, "rbe_rbl_forces: need 0 < r_c < r_s and 1 <= p <= " + std::to_string(rbe::RBL_PMAX));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    SrLayout l;
    SrBuffers b;
    int R = 0;
    if (!rbl_layout(c, rc, rs, l, R))
        return fail(c, RBE_ERR_INVALID_ARG, "rbe_rbl_forces: the shell must span at most 9 cells of side max(r_c, r_s/4) per dimension, and they must fit the box");
    rbe_status s = sr_build_cells(c, "rbe_rbl_forces", d_xyzq, d_force, d_ws, ws_bytes, st, l, b);
    if (s != RBE_OK || c->N == 0) return s;
    RBE_CUDA(c, cudaMemsetAsync(b.acc, 0, 4 * sizeof(long long), st));
    rbe::RblParams rp;
    rp.sorted = b.sorted; rp.sidx = b.sidx; rp.start = b.start;
    rp.force = static_cast<float4*>(d_force);
    rp.fsum = b.acc;
    rp.nc = l.nc; rp.R = R; rp.p = p; rp.accumulate = accumulate;
    rp.len_unit = (float)(c->L / rbe::TWO32);
    rp.rc2 = (float)(rc * rc); rp.rs2 = (float)(rs * rs);
    rp.sqrt_alpha = (float)std::sqrt(c->alpha);
    // reading Q20: the per-step salt of the pair keys, one Philox4x32-10 call (counter (step, 0, 0), key seed)
    uint32_t salt[4];
    philox4x32_10_host((uint32_t)step, (uint32_t)(step >> 32), 0u, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), salt);
    rp.salt0 = salt[0]; rp.salt1 = salt[1];
    // tile: 1.3 x the mean number of candidates of a cell, in steps of 256 (candidate indices are 15-bit: <= 8192)
    const double mean_cand = (double)c->N / (double)l.ncell * (double)((2 * R + 1) * (2 * R + 1) * (2 * R + 1));
    int tc = (int)std::ceil(1.3 * mean_cand / 256.0) * 256 + 256;
    if (tc > rbe::RBL_TC_MAX) tc = rbe::RBL_TC_MAX;
    rp.tc = tc;
    RBE_CUDA(c, cudaFuncSetAttribute(rbe::rbl_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rbe::rbl_smem_bytes(rbe::RBL_TC_MAX)));
    rbe::rbl_kernel<<<(unsigned)l.ncell, rbe::RBL_THREADS, rbe::rbl_smem_bytes(tc), st>>>(rp);
    rbe::rbl_correct_kernel<<<(unsigned)((c->N + 255) / 256), 256, 0, st>>>(b.acc, c->N, static_cast<float4*>(d_force));
    RBE_CUDA(c, cudaGetLastError());
    return RBE_OK;
}

rbe_status rbe_kspace_virial(rbe_ctx* c, double* h_W, void* stream) {
    if (!c || !h_W) return fail(c, RBE_ERR_INVALID_ARG, "rbe_kspace_virial: null argument");
    if (!c->ws || !c->have_k || !c->have_rho) return fail(c, RBE_ERR_NOT_READY, "rbe_kspace_virial needs a structure factor");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    double* d_W = ws_ptr<double>(c, c->off_U) + 1;
    rbe::virial_kernel<<<1, 256, 0, st>>>(k_table(c), c->P, c->alpha, d_W);
    RBE_CUDA(c, cudaGetLastError());
    RBE_CUDA(c, cudaMemcpyAsync(h_W, d_W, 6 * sizeof(double), cudaMemcpyDeviceToHost, st));
    RBE_CUDA(c, cudaStreamSynchronize(st));
    return RBE_OK;
}

size_t rbe_step_host_bytes(const rbe_ctx* c, int32_t compact) {
    if (!c) return 0;
    const size_t nb = (size_t)c->N * sizeof(float4), nb3 = (size_t)c->N * 3 * sizeof(float);
    return align_up(nb, 256) + align_up(nb, 256) + (compact ? align_up(nb3, 256) + align_up(nb3, 256) : 0);
}

namespace {
// The end-to-end step from host buffers.  compact = false: float4 {x,y,z,q} in, float4 {F, e} out.
// compact = true: float3 positions in, float3 forces out, charges from rbe_set_charges; a pack and an
// unpack kernel sit between the copies and the two hot kernels.
rbe_status step_host_impl(rbe_ctx* c, const float* h_in, const int32_t* h_m, const double* h_w, float* h_out,
                          int32_t with_energy, double* h_U, void* d_scratch, size_t scratch_bytes, void* stream, bool compact) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if ((c->N > 0 && (!h_in || !h_out)) || !h_m) return fail(c, RBE_ERR_INVALID_ARG, "rbe_step_host: null argument");
    if (compact && c->N > 0 && !c->d_q) return fail(c, RBE_ERR_NOT_READY, "rbe_step_host_xyz needs rbe_set_charges");
    const size_t nb = (size_t)c->N * sizeof(float4), nb3 = (size_t)c->N * 3 * sizeof(float);
    const size_t need = rbe_step_host_bytes(c, compact ? 1 : 0);
    if (c->N > 0 && (!d_scratch || scratch_bytes < need || (reinterpret_cast<uintptr_t>(d_scratch) & 255u)))
        return fail(c, RBE_ERR_WORKSPACE, "rbe_step_host: d_scratch must hold rbe_step_host_bytes bytes, 256-byte aligned");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    unsigned char* base = static_cast<unsigned char*>(d_scratch);
    float4* d_x = reinterpret_cast<float4*>(base);
    float4* d_f = reinterpret_cast<float4*>(base + align_up(nb, 256));
    float* d_x3 = reinterpret_cast<float*>(base + 2 * align_up(nb, 256));
    float* d_f3 = reinterpret_cast<float*>(base + 2 * align_up(nb, 256) + align_up(nb3, 256));
    // bytes per atom on the wire and the two copy helpers (a chunk [lo, lo + n) of atoms)
    auto copy_in = [&](int64_t lo, int64_t n, cudaStream_t s_) -> cudaError_t {
        return compact ? cudaMemcpyAsync(d_x3 + 3 * lo, h_in + 3 * lo, (size_t)n * 3 * sizeof(float), cudaMemcpyHostToDevice, s_)
                       : cudaMemcpyAsync(d_x + lo, reinterpret_cast<const float4*>(h_in) + lo, (size_t)n * sizeof(float4), cudaMemcpyHostToDevice, s_);
    };
    auto copy_out = [&](int64_t lo, int64_t n, cudaStream_t s_) -> cudaError_t {
        return compact ? cudaMemcpyAsync(h_out + 3 * lo, d_f3 + 3 * lo, (size_t)n * 3 * sizeof(float), cudaMemcpyDeviceToHost, s_)
                       : cudaMemcpyAsync(reinterpret_cast<float4*>(h_out) + lo, d_f + lo, (size_t)n * sizeof(float4), cudaMemcpyDeviceToHost, s_);
    };
    auto pack = [&](int64_t lo, int64_t n) {      // on st, after the chunk has arrived
        if (compact && n > 0) rbe::pack_xyzq_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d_x3 + 3 * lo, c->d_q + lo, n, d_x + lo);
    };
    auto unpack = [&](int64_t lo, int64_t n) {    // on st, after the chunk's forces
        if (compact && n > 0) rbe::unpack_force_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d_f + lo, n, d_f3 + 3 * lo);
    };
    rbe_status s = rbe_set_kvectors(c, h_m, h_w, stream);
    if (s != RBE_OK) return s;

    // Chunked pipeline: the transfers are the long pole (32 B per atom over PCIe against ~0.2 ns
    // per atom of kernels), so the atoms travel in chunks on two copy streams and the kernels of a
    // chunk run as soon as it has arrived: H2D(c+1) overlaps SF(c); D2H(c) overlaps F(c+1).  Every
    // chunk adds to the same per-CTA fp64 rows in stream order (deterministic); the last structure-
    // factor launch runs the second pass; the force launches need the complete rho, so they start
    // after it.
    int64_t nchunk = c->N / HOST_MIN_CHUNK;
    if (nchunk > HOST_MAX_CHUNKS) nchunk = HOST_MAX_CHUNKS;
    if (nchunk < 1) nchunk = 1;
    // Chunk boundaries (whole 32-atom windows).  What stays exposed is the structure-factor launch of
    // the LAST input chunk and the force launch of the FIRST output chunk, so the input chunks shrink
    // (weights nchunk .. 1) and the output chunks grow (1 .. nchunk); the two splits are independent.
    int64_t in_lo[HOST_MAX_CHUNKS + 1], out_lo[HOST_MAX_CHUNKS + 1];
    {
        const int64_t wsum = nchunk * (nchunk + 1) / 2, units = (c->N + 31) / 32;
        int64_t acc_in = 0, acc_out = 0;
        for (int64_t i = 0; i < nchunk; ++i) {
            in_lo[i] = units * acc_in / wsum * 32;
            out_lo[i] = units * acc_out / wsum * 32;
            acc_in += nchunk - i;
            acc_out += i + 1;
        }
        in_lo[nchunk] = out_lo[nchunk] = c->N;
    }
    const unsigned evflag = cudaEventDisableTiming;
    if (nchunk > 1 && !c->s_h2d) {
        RBE_CUDA(c, cudaStreamCreateWithFlags(&c->s_h2d, cudaStreamNonBlocking));
        RBE_CUDA(c, cudaStreamCreateWithFlags(&c->s_d2h, cudaStreamNonBlocking));
        RBE_CUDA(c, cudaEventCreateWithFlags(&c->ev_start, evflag));
        RBE_CUDA(c, cudaEventCreateWithFlags(&c->ev_done, evflag));
        for (int i = 0; i < HOST_MAX_CHUNKS; ++i) {
            RBE_CUDA(c, cudaEventCreateWithFlags(&c->ev_in[i], evflag));
            RBE_CUDA(c, cudaEventCreateWithFlags(&c->ev_f[i], evflag));
        }
    }
    if (nchunk == 1) {
        if (c->N > 0) RBE_CUDA(c, copy_in(0, c->N, st));
        pack(0, c->N);
        s = rbe_structure_factor(c, d_x, nullptr, stream);
        if (s != RBE_OK) return s;
        s = rbe_forces(c, d_x, d_f, with_energy, stream);
        if (s != RBE_OK) return s;
        unpack(0, c->N);
        if (c->N > 0) RBE_CUDA(c, copy_out(0, c->N, st));
    } else {
        auto pipeline = [&]() -> rbe_status {
            RBE_CUDA(c, cudaEventRecord(c->ev_start, st));          // the copies start after the caller's earlier work
            RBE_CUDA(c, cudaStreamWaitEvent(c->s_h2d, c->ev_start, 0));
            RBE_CUDA(c, cudaStreamWaitEvent(c->s_d2h, c->ev_start, 0));
            for (int64_t i = 0; i < nchunk; ++i) {
                const int64_t lo = in_lo[i], n = in_lo[i + 1] - lo;
                RBE_CUDA(c, copy_in(lo, n, c->s_h2d));
                RBE_CUDA(c, cudaEventRecord(c->ev_in[i], c->s_h2d));
                RBE_CUDA(c, cudaStreamWaitEvent(st, c->ev_in[i], 0));
                pack(lo, n);
                s = launch_sf(c, d_x + lo, n, i > 0, i == nchunk - 1, nullptr, st);
                if (s != RBE_OK) return s;
            }
            c->have_rho = true;
            for (int64_t i = 0; i < nchunk; ++i) {
                const int64_t lo = out_lo[i], n = out_lo[i + 1] - lo;
                s = launch_f(c, d_x + lo, d_f + lo, n, with_energy, st);
                if (s != RBE_OK) return s;
                unpack(lo, n);
                RBE_CUDA(c, cudaEventRecord(c->ev_f[i], st));
                RBE_CUDA(c, cudaStreamWaitEvent(c->s_d2h, c->ev_f[i], 0));
                RBE_CUDA(c, copy_out(lo, n, c->s_d2h));
            }
            RBE_CUDA(c, cudaEventRecord(c->ev_done, c->s_d2h));
            RBE_CUDA(c, cudaStreamWaitEvent(st, c->ev_done, 0));
            return RBE_OK;
        };
        s = pipeline();
        if (s != RBE_OK) {      // never return with the library's copy streams still running into the caller's buffers
            cudaStreamSynchronize(c->s_h2d);
            cudaStreamSynchronize(c->s_d2h);
            return s;
        }
    }
    if (h_U) return rbe_kspace_energy(c, h_U, stream);
    RBE_CUDA(c, cudaStreamSynchronize(st));
    return RBE_OK;
}
}  // namespace

rbe_status rbe_step_host(rbe_ctx* c, const float* h_xyzq, const int32_t* h_m, const double* h_w, float* h_force,
                         int32_t with_energy, double* h_U, void* d_scratch, size_t scratch_bytes, void* stream) {
    return step_host_impl(c, h_xyzq, h_m, h_w, h_force, with_energy, h_U, d_scratch, scratch_bytes, stream, false);
}

rbe_status rbe_set_charges(rbe_ctx* c, const void* d_q) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if (d_q && (reinterpret_cast<uintptr_t>(d_q) & 3u)) return fail(c, RBE_ERR_INVALID_ARG, "rbe_set_charges: misaligned pointer");
    c->d_q = static_cast<const float*>(d_q);
    return RBE_OK;
}

rbe_status rbe_step_host_xyz(rbe_ctx* c, const float* h_xyz, const int32_t* h_m, const double* h_w, float* h_force3,
                             double* h_U, void* d_scratch, size_t scratch_bytes, void* stream) {
    return step_host_impl(c, h_xyz, h_m, h_w, h_force3, 0, h_U, d_scratch, scratch_bytes, stream, true);
}

rbe_status rbe_nve_kick(rbe_ctx* c, void* d_vel, const void* d_inv_mass, const void* d_force, double half_dt, void* d_pos,
                        void* d_xyzq, double dt, void* stream) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if (c->N == 0) return RBE_OK;
    if (!d_vel || !d_inv_mass || !d_force || (d_pos && !d_xyzq) || (reinterpret_cast<uintptr_t>(d_force) & 15u) ||
        (reinterpret_cast<uintptr_t>(d_xyzq) & 15u) || (reinterpret_cast<uintptr_t>(d_vel) & 7u) || (reinterpret_cast<uintptr_t>(d_pos) & 7u) ||
        (reinterpret_cast<uintptr_t>(d_inv_mass) & 7u) || !std::isfinite(half_dt) || !std::isfinite(dt))
        return fail(c, RBE_ERR_INVALID_ARG, "rbe_nve_kick: null or misaligned pointer, or a non-finite time step");
    rbe::nve_kick_kernel<<<(unsigned)((c->N + 255) / 256), 256, 0, static_cast<cudaStream_t>(stream)>>>(
        static_cast<double*>(d_vel), static_cast<const double*>(d_inv_mass), static_cast<const float4*>(d_force), half_dt,
        static_cast<double*>(d_pos), static_cast<float4*>(d_xyzq), dt, c->N);
    RBE_CUDA(c, cudaGetLastError());
    return RBE_OK;
}

rbe_status rbe_nve_energies(rbe_ctx* c, const void* d_vel, const void* d_inv_mass, const void* d_force, double* h_out, void* stream) {
    if (!c || !h_out) return fail(c, RBE_ERR_INVALID_ARG, "rbe_nve_energies: null argument");
    if (!c->ws) return fail(c, RBE_ERR_NOT_READY, "rbe_nve_energies before rbe_set_workspace");
    if ((d_vel && !d_inv_mass) || (reinterpret_cast<uintptr_t>(d_force) & 15u))
        return fail(c, RBE_ERR_INVALID_ARG, "rbe_nve_energies: velocities without masses, or a misaligned pointer");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    double2* part = ws_ptr<double2>(c, c->off_nve);
    double* out = reinterpret_cast<double*>(part + rbe::NVE_RED_CTAS);
    rbe::nve_energy_partial_kernel<<<rbe::NVE_RED_CTAS, 256, 0, st>>>(static_cast<const double*>(d_vel), static_cast<const double*>(d_inv_mass),
                                                                      static_cast<const float4*>(d_force), c->N, part);
    rbe::nve_energy_final_kernel<<<1, rbe::NVE_RED_CTAS, 0, st>>>(part, rbe::NVE_RED_CTAS, out);
    RBE_CUDA(c, cudaGetLastError());
    RBE_CUDA(c, cudaMemcpyAsync(h_out, out, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
    RBE_CUDA(c, cudaStreamSynchronize(st));
    return RBE_OK;
}

rbe_status rbe_md_capture(rbe_ctx* c, void* d_pos, void* d_vel, const void* d_inv_mass, void* d_xyzq, void* d_force, double rs, double dt,
                          void* d_sr_ws, size_t sr_bytes, int32_t sampled, uint64_t seed, uint64_t first_step, int32_t with_energy) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if (!c->ws) return fail(c, RBE_ERR_NOT_READY, "rbe_md_capture before rbe_set_workspace");
    if (sampled && c->sampler_T.empty()) return fail(c, RBE_ERR_INVALID_ARG, "rbe_md_capture: the device sampler is unavailable for this L, alpha");
    if (!sampled && !c->have_k) return fail(c, RBE_ERR_NOT_READY, "rbe_md_capture: no k-set (rbe_set_kvectors first, or sampled != 0)");
    if (c->xch_world > 0) return fail(c, RBE_ERR_INVALID_ARG, "rbe_md_capture: not available with a fused exchange");
    if (c->N < 1 || !d_pos || !d_vel || !d_inv_mass || !d_xyzq || !d_force || !(dt > 0.0) || !std::isfinite(dt))
        return fail(c, RBE_ERR_INVALID_ARG, "rbe_md_capture: null pointer, empty system or bad time step");
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    if (c->graph) { cudaGraphDestroy(c->graph); c->graph = nullptr; }
    if (!c->s_cap) RBE_CUDA(c, cudaStreamCreateWithFlags(&c->s_cap, cudaStreamNonBlocking));
    if (sampled) {
        const unsigned long long st8[2] = {seed, first_step};
        RBE_CUDA(c, cudaMemcpy(c->ws + c->off_state, st8, sizeof(st8), cudaMemcpyHostToDevice));
    }
    RBE_CUDA(c, cudaStreamBeginCapture(c->s_cap, cudaStreamCaptureModeThreadLocal));
    // v(t+dt/2), x(t+dt)  ->  [a fresh batch]  ->  F_long  ->  + F_short  ->  v(t+dt)
    rbe_status s = rbe_nve_kick(c, d_vel, d_inv_mass, d_force, 0.5 * dt, d_pos, d_xyzq, dt, c->s_cap);
    if (s == RBE_OK && sampled) { s = launch_sampler(c, true, 0, 0, c->s_cap); c->have_w = false; }
    if (s == RBE_OK) s = launch_kspace(c, d_xyzq, d_force, with_energy, c->s_cap);
    if (s == RBE_OK) s = rbe_short_range(c, d_xyzq, rs, d_force, 1, with_energy, d_sr_ws, sr_bytes, c->s_cap);
    if (s == RBE_OK) s = rbe_nve_kick(c, d_vel, d_inv_mass, d_force, 0.5 * dt, nullptr, nullptr, dt, c->s_cap);
    cudaGraph_t g = nullptr;
    const cudaError_t e = cudaStreamEndCapture(c->s_cap, &g);
    if (s != RBE_OK) { if (g) cudaGraphDestroy(g); return s; }
    if (e != cudaSuccess) return cuda_fail(c, "cudaStreamEndCapture", e);
    c->graph = g;
    c->graph_have_w = c->have_w;     // sampled: cleared above; else the weights of the k-set the caller uploaded
    RBE_CUDA(c, cudaGraphInstantiate(&c->graph_exec, c->graph, 0));
    return RBE_OK;
}

rbe_status rbe_probe_pipe_rates(rbe_ctx* c, double* h_out, void* stream) {
    if (!c || !h_out) return fail(c, RBE_ERR_INVALID_ARG, "rbe_probe_pipe_rates: null argument");
    if (!c->ws) return fail(c, RBE_ERR_NOT_READY, "rbe_probe_pipe_rates before rbe_set_workspace");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int sms = c->li.num_sms, iters = 2048, chains = 8;
    // scratch: the grid-barrier-free tail of the workspace is not touched; the group rows are (>= 16 B * P per group)
    if ((size_t)sms * sizeof(long long) > (size_t)c->li.sf_grid_x * c->P * sizeof(double2) + (c->off_rho - c->off_part))
        return fail(c, RBE_ERR_WORKSPACE, "rbe_probe_pipe_rates: workspace too small");
    long long* d_cyc = ws_ptr<long long>(c, c->off_part);
    std::vector<long long> cyc((size_t)sms);
    cudaEvent_t e0, e1;
    RBE_CUDA(c, cudaEventCreate(&e0));
    RBE_CUDA(c, cudaEventCreate(&e1));
    double clock_mhz = 0.0;
    for (int mode = 0; mode < 4; ++mode) {
        for (int rep = 0; rep < 2; ++rep) {   // rep 0 warms up
            RBE_CUDA(c, cudaEventRecord(e0, st));
            switch (mode) {
                case 0: rbe::probe_kernel<0><<<sms, 1024, 0, st>>>(d_cyc, iters, 1.0001f, 0.5f, 3, 7); break;
                case 1: rbe::probe_kernel<1><<<sms, 1024, 0, st>>>(d_cyc, iters, 1.0001f, 0.5f, 3, 7); break;
                case 2: rbe::probe_kernel<2><<<sms, 1024, 0, st>>>(d_cyc, iters, 1.0001f, 0.5f, 3, 7); break;
                default: rbe::probe_kernel<3><<<sms, 1024, 0, st>>>(d_cyc, iters, 1.0001f, 0.5f, 3, 7); break;
            }
            RBE_CUDA(c, cudaEventRecord(e1, st));
            RBE_CUDA(c, cudaGetLastError());
        }
        RBE_CUDA(c, cudaMemcpyAsync(cyc.data(), d_cyc, cyc.size() * sizeof(long long), cudaMemcpyDeviceToHost, st));
        RBE_CUDA(c, cudaStreamSynchronize(st));
        std::sort(cyc.begin(), cyc.end());
        const double med = (double)cyc[cyc.size() / 2];
        h_out[mode] = 1024.0 * chains * iters / med;          // lanes (thread-instructions) per SM per clock
        if (mode == 3) {                                       // the longest kernel: clock = cycles / elapsed time
            float ms = 0.f;
            RBE_CUDA(c, cudaEventElapsedTime(&ms, e0, e1));
            clock_mhz = (double)cyc.back() / (ms * 1e3);
        }
    }
    h_out[4] = clock_mhz;
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return RBE_OK;
}

rbe_status rbe_host_alloc(void** out, size_t bytes) {
    if (!out || bytes == 0) return RBE_ERR_INVALID_ARG;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return RBE_ERR_NO_DEVICE;
    }
    if (cudaHostAlloc(out, bytes, cudaHostAllocDefault) != cudaSuccess) {
        cudaGetLastError();
        *out = nullptr;
        return RBE_ERR_CUDA;
    }
    return RBE_OK;
}

rbe_status rbe_host_free(void* h_ptr) {
    if (!h_ptr) return RBE_OK;
    if (cudaFreeHost(h_ptr) != cudaSuccess) {
        cudaGetLastError();
        return RBE_ERR_CUDA;
    }
    return RBE_OK;
}

const char* rbe_last_error(const rbe_ctx* c) { return c ? c->err.c_str() : "null context"; }

const char* rbe_status_string(rbe_status s) {
    switch (s) {
        case RBE_OK: return "RBE_OK";
        case RBE_ERR_INVALID_ARG: return "RBE_ERR_INVALID_ARG";
        case RBE_ERR_BAD_KVECTOR: return "RBE_ERR_BAD_KVECTOR";
        case RBE_ERR_NOT_READY: return "RBE_ERR_NOT_READY";
        case RBE_ERR_WORKSPACE: return "RBE_ERR_WORKSPACE";
        case RBE_ERR_CUDA: return "RBE_ERR_CUDA";
        case RBE_ERR_NO_DEVICE: return "RBE_ERR_NO_DEVICE";
    }
    return "RBE_ERR_UNKNOWN";
}

int32_t rbe_version(void) { return 100; }

}  // extern "C"

// ------------------------------------------------------------------------------------------------------------
// rbe_step_static: the k-space step without a caller-provided workspace (include/rbe.h gives the reasons: a
// plug-in inside a host program that owns all device memory, or a loop that cannot take cudaMalloc's stall).
// The scratch of step_kernel -- per-CTA fp64 rows, k-set copy, rho, the per-k force records, the barrier
// counter -- is carved from ONE array that is part of this library's device image.  Nothing on this path
// allocates; the array holds its contents from call to call and is shared by every caller on the device.
namespace {

constexpr size_t ST_OFF_PART = 0;                                                                         // double2 [rows][P]
constexpr size_t ST_OFF_KVEC = ST_OFF_PART + (size_t)RBE_STATIC_MAX_CTAS * RBE_STATIC_MAX_P * sizeof(double2);   // int4 [P]
constexpr size_t ST_OFF_RHO = ST_OFF_KVEC + (size_t)RBE_STATIC_MAX_P * sizeof(int4);                      // double2 [P]
constexpr size_t ST_OFF_KA = ST_OFF_RHO + (size_t)RBE_STATIC_MAX_P * sizeof(double2);                     // int4 [P]
constexpr size_t ST_OFF_KB = ST_OFF_KA + (size_t)RBE_STATIC_MAX_P * sizeof(int4);                         // float4 [P]
constexpr size_t ST_OFF_BAR = ST_OFF_KB + (size_t)RBE_STATIC_MAX_P * sizeof(float4);                      // u64, on a line of its own
constexpr size_t ST_BYTES = ST_OFF_BAR + 256;
static_assert(ST_BYTES == RBE_STATIC_SCRATCH_BYTES, "rbe.h states the size of the built-in scratch");
static_assert(RBE_STATIC_MAX_P <= rbe::STEP_KPARAM_MAX, "the wavevectors must fit the kernel parameters");
static_assert(ST_OFF_KVEC % 256 == 0 && ST_OFF_BAR % 256 == 0, "sub-arrays stay 256-byte aligned");

}  // namespace

// In HOST code this name is only a handle for cudaGetSymbolAddress: it is not a device address, and a kernel
// handed `g_static_scratch` itself would fault (or scribble over host memory where the GPU can reach it).
static __device__ __align__(256) unsigned char g_static_scratch[ST_BYTES];

namespace {

constexpr int STATIC_MAX_DEVICES = 64;
struct StaticDevice {
    unsigned char* base = nullptr;   // device address of g_static_scratch on this device (nullptr: set-up not done)
    int smem_max = 0;                // dynamic shared memory the step kernels may use there
    int coop = 0;
};
StaticDevice g_static_dev[STATIC_MAX_DEVICES];
std::mutex g_static_mu;

// Once per device, with that device current: the address of the array as the GPU sees it, and the kernel
// attributes rbe_step would have set through the context.  No allocation; not to be run under stream capture.
rbe_status static_setup(rbe_ctx* c, int dev, StaticDevice* out) {
    std::lock_guard<std::mutex> lock(g_static_mu);
    StaticDevice& d = g_static_dev[dev];
    if (!d.base) {
        void* ptr = nullptr;
        RBE_CUDA(c, cudaGetSymbolAddress(&ptr, g_static_scratch));
        if (!ptr || (reinterpret_cast<uintptr_t>(ptr) & 255u))
            return fail(c, RBE_ERR_CUDA, "rbe_step_static: cudaGetSymbolAddress returned a null or misaligned address");
        int optin = 0, coop = 0;
        RBE_CUDA(c, cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
        RBE_CUDA(c, cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
        const int smem_max = optin - 4 * 1024;   // as init_device: the kernels' static shared memory stays under 4 KB
        RBE_CUDA(c, cudaFuncSetAttribute(rbe::step_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max));
        RBE_CUDA(c, cudaFuncSetAttribute(rbe::step_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max));
        RBE_CUDA(c, cudaFuncSetAttribute(rbe::step_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max));
        RBE_CUDA(c, cudaFuncSetAttribute(rbe::step_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max));
        d.smem_max = smem_max;
        d.coop = coop;
        d.base = static_cast<unsigned char*>(ptr);   // last: marks the set-up as done
    }
    *out = d;
    return RBE_OK;
}

}  // namespace

extern "C" rbe_status rbe_step_static(rbe_ctx* c, const int32_t* h_m, const void* d_xyzq, void* d_force, int32_t with_energy,
                                      void* d_rho, void* stream) {
    if (!c) return RBE_ERR_INVALID_ARG;
    if (!h_m) return fail(c, RBE_ERR_INVALID_ARG, "rbe_step_static: h_m is null (the wavevectors travel with the call)");
    if ((c->N > 0 && (!d_xyzq || !d_force)) || (reinterpret_cast<uintptr_t>(d_xyzq) & 15u) || (reinterpret_cast<uintptr_t>(d_force) & 15u) ||
        (reinterpret_cast<uintptr_t>(d_rho) & 15u))
        return fail(c, RBE_ERR_INVALID_ARG, "rbe_step_static: null or misaligned pointer");
    // the limits of the built-in array come first: they do not depend on the device
    if (c->P > RBE_STATIC_MAX_P)
        return fail(c, RBE_ERR_WORKSPACE, "rbe_step_static: P = " + std::to_string(c->P) + " exceeds the built-in scratch (P <= " +
                                              std::to_string(RBE_STATIC_MAX_P) + "); use rbe_step with a caller-allocated workspace");
    rbe_status s = check_kvectors(c, h_m, nullptr);
    if (s != RBE_OK) return s;
    s = init_device(c);   // launch geometry for this (N, P) on the current device: queries only
    if (s != RBE_OK) return s;
    int dev = -1;
    RBE_CUDA(c, cudaGetDevice(&dev));
    if (dev != c->device) return fail(c, RBE_ERR_INVALID_ARG, "rbe_step_static: the context was first used on another device");
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return fail(c, RBE_ERR_NO_DEVICE, "rbe_step_static: device ordinal beyond 63");
    StaticDevice sd;
    s = static_setup(c, dev, &sd);
    if (s != RBE_OK) return s;
    const int G = c->li.sf_grid_x;
    if (G > RBE_STATIC_MAX_CTAS || G > c->li.num_sms)
        return fail(c, RBE_ERR_WORKSPACE, "rbe_step_static: a grid of " + std::to_string(G) + " CTAs exceeds the built-in scratch (<= " +
                                              std::to_string(RBE_STATIC_MAX_CTAS) + " rows)");
    if (!sd.coop || c->li.sf_grid_y != 1 || c->step_smem > (size_t)sd.smem_max)
        return fail(c, RBE_ERR_CUDA, "rbe_step_static: the device cannot run the one-launch step kernel for this P");

    cudaStream_t st = static_cast<cudaStream_t>(stream);
    unsigned char* base = sd.base;
    // The array still holds the previous call's contents.  Only the barrier counter has to start from a known
    // value (a multiple of this call's grid size; zero is one): rows, rho and records are rewritten before use.
    RBE_CUDA(c, cudaMemsetAsync(base + ST_OFF_BAR, 0, sizeof(unsigned long long), st));

    rbe::StepParams sp;
    sp.sf.xyzq = static_cast<const float4*>(d_xyzq);
    sp.sf.N = c->N;
    sp.sf.part = reinterpret_cast<double2*>(base + ST_OFF_PART);
    sp.sf.two32_over_L = rbe::TWO32 / c->L;
    sp.sf.P = c->P; sp.sf.gs = c->sf_gs; sp.sf.ng = c->sf_ng;
    sp.sf.pairing = c->sf_pairing;
    sp.sf.accumulate = 0;
    sp.f.xyzq = static_cast<const float4*>(d_xyzq);
    sp.f.force = static_cast<float4*>(d_force);
    sp.f.N = c->N;
    sp.f.two32_over_L = rbe::TWO32 / c->L;
    sp.kvec = reinterpret_cast<const int4*>(base + ST_OFF_KVEC);
    sp.w = nullptr;
    sp.w_uniform = c->S / (double)c->P;
    sp.L = c->L;
    sp.rho = reinterpret_cast<double2*>(base + ST_OFF_RHO);
    sp.rho_user = static_cast<double2*>(d_rho);
    sp.ka = reinterpret_cast<int4*>(base + ST_OFF_KA);
    sp.kb = reinterpret_cast<float4*>(base + ST_OFF_KB);
    sp.bar = reinterpret_cast<unsigned long long*>(base + ST_OFF_BAR);
    sp.kparam = 1;
    for (int32_t i = 0; i < 3 * c->P; ++i) sp.km[i] = (int16_t)h_m[i];   // validated above: |m_d| < 2^15

    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)G);
    cfg.blockDim = dim3((unsigned)c->li.sf_threads);
    cfg.dynamicSmemBytes = c->step_smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeCooperative;
    attr[0].val.cooperative = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (c->sf_deep) {
        if (with_energy) RBE_CUDA(c, cudaLaunchKernelEx(&cfg, rbe::step_kernel<true, true>, sp));
        else RBE_CUDA(c, cudaLaunchKernelEx(&cfg, rbe::step_kernel<true, false>, sp));
    } else {
        if (with_energy) RBE_CUDA(c, cudaLaunchKernelEx(&cfg, rbe::step_kernel<false, true>, sp));
        else RBE_CUDA(c, cudaLaunchKernelEx(&cfg, rbe::step_kernel<false, false>, sp));
    }
    return RBE_OK;
}
