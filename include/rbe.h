/*
 * rbe.h -- C ABI of librbe: the random batch Ewald (RBE) Fourier-space Coulomb force of
 * arxiv 2407.09315 (RBMD) on one NVIDIA B200 (sm_100a).
 *
 * "P:nnn" below = line nnn of the paper text (/root/reference/PAPER.md at build time).
 *
 * What the library computes, for N atoms {r_i, q_i} in a cubic periodic box of side L
 * (V = L^3) and a batch of P integer wavevectors m_l in Z^3 \ {0}, k_l = 2 pi m_l / L
 * (P:115):
 *
 *   rho(k_l) = sum_j q_j exp(i k_l . r_j)                                  Eq. (2.9),
 *   F_i      = - sum_l w_l (4 pi q_i k_l / (V k_l^2)) Im(exp(-i k_l . r_i) rho(k_l))
 *                                                                           Eq. (2.12)
 *   U        = (2 pi / V) sum_l w_l |rho(k_l)|^2 / k_l^2      (2nd term of Eq. (2.8),  P:112)
 *
 * with w_l = S / P by default, S = sum_{m != 0} exp(-|k_m|^2 / 4 alpha) the paper's
 * normalisation constant Q.  The k-set is drawn by the caller (Algorithm 1 step 1,
 * P:202) and handed over as integers; steps 2-4 of Algorithm 1 run on the GPU.
 *
 * Units are Gaussian (Eq. 2.5): charges in e, lengths in A, forces in e^2/A^2, energy
 * in e^2/A; alpha in A^-2 (erfc(sqrt(alpha) r)).  No Coulomb constant is applied.
 *
 * Conventions
 *  - `d_*` pointers are DEVICE memory owned by the caller, 16-byte aligned, never retained
 *    after the call returns (except the workspace, retained until rbe_destroy or the next
 *    rbe_set_workspace).  `h_*` pointers are HOST memory owned by the caller.
 *  - `stream` is a cudaStream_t passed as void* (0 = the legacy default stream).  Every call
 *    that takes a stream only enqueues work on it and returns; the exceptions, which synchronise
 *    that stream (or, where they take none, the device) before returning, are rbe_kspace_energy,
 *    rbe_kspace_virial, rbe_get_kvectors, rbe_exchange_check, rbe_step_host, rbe_step_host_xyz,
 *    rbe_probe_pipe_rates, rbe_set_workspace and rbe_graph_capture.
 *  - The library allocates no device memory.  Host memory: the context and a small pinned
 *    staging ring for the k-vectors, both freed by rbe_destroy.
 *  - Every function returns an rbe_status (or a value documented below); nothing aborts,
 *    throws across the boundary, or prints.  rbe_last_error gives the text of the last failure.
 *  - Results are bitwise reproducible run to run on the same device: no floating-point atomics,
 *    every reduction in a fixed order.
 *  - Positions may lie outside [0, L): exp(i k . r) is exactly periodic because k . nL = 2 pi m . n.
 *    Non-finite positions or charges are undefined behaviour (not checked on the hot path).
 *  - A context is not thread-safe; use one per host thread / stream.
 */
#ifndef RBE_H_
#define RBE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rbe_ctx rbe_ctx; /* opaque; created by rbe_create, freed by rbe_destroy */

typedef enum {
    RBE_OK = 0,
    RBE_ERR_INVALID_ARG = 1,  /* null pointer, N < 0, L <= 0, alpha <= 0, P < 1, misaligned pointer */
    RBE_ERR_BAD_KVECTOR = 2,  /* some m_l == (0,0,0) or |m_l,d| >= 2^15; or a weight is not finite */
    RBE_ERR_NOT_READY = 3,    /* call order: workspace / k-vectors / structure factor missing */
    RBE_ERR_WORKSPACE = 4,    /* workspace too small or misaligned */
    RBE_ERR_CUDA = 5,         /* a CUDA runtime call failed (text in rbe_last_error) */
    RBE_ERR_NO_DEVICE = 6     /* no usable sm_100 device: there is no CPU fallback */
} rbe_status;

/* Launch geometry of the two k-space kernels, for benchmarks and profiles (read-only information). */
typedef struct {
    int32_t num_sms;
    int32_t sf_grid_x, sf_grid_y, sf_threads, sf_smem_bytes; /* structure-factor kernel */
    int32_t sf_k_per_thread, sf_atom_groups, sf_tile_atoms;
    int32_t sf_red_group, sf_red_groups;                     /* in-kernel two-level fixed-order reduction */
    int32_t f_grid, f_threads, f_smem_bytes, f_atoms_per_thread; /* force kernel */
    int32_t step_fused, step_smem_bytes;                     /* rbe_step runs as ONE cooperative launch (grid sf_grid_x) */
} rbe_launch_info;

/* Create a context for N atoms (on this GPU), box side L [A], splitting parameter alpha [A^-2]
 * (Eq. 2.6) and batch size P.  Computes S(L, alpha) in fp64 on the host
 * (S = H^3 - 1, H = sum_m exp(-pi^2 m^2 / (alpha L^2))).  Makes no CUDA call, so it works
 * on a machine without a GPU.  N = 0 is allowed (all outputs are then zero / empty).
 * Errors: RBE_ERR_INVALID_ARG. */
rbe_status rbe_create(rbe_ctx** out, int64_t N, double L, double alpha, int32_t P);

/* Free the context, its pinned staging buffers and events.  NULL is accepted. */
rbe_status rbe_destroy(rbe_ctx* ctx);

/* The paper's normalisation constant Q == S for this context's L and alpha. */
double rbe_normaliser_S(const rbe_ctx* ctx);

/* Bytes of device scratch the context needs (per-CTA fp64 partials, rho, the k-set).
 * Queries the current CUDA device on first use.  Returns 0 on error (see rbe_last_error). */
size_t rbe_workspace_bytes(const rbe_ctx* ctx);

/* Hand the context a device buffer of at least rbe_workspace_bytes bytes, 256-byte aligned,
 * allocated on the current CUDA device.  Caller keeps ownership and must keep it alive.  The buffer belongs to
 * THIS context alone for as long as it is set (it holds state that survives from launch to launch: the k-set,
 * rho, the step counter of the device sampler, the arrival counter of rbe_step's grid barrier, which the call
 * zeroes and which must stay a multiple of the context's grid size): never share it between contexts.  The library keeps
 * a list of the buffers its live contexts hold and refuses (RBE_ERR_WORKSPACE) a buffer whose first
 * rbe_workspace_bytes bytes overlap another live context's; rbe_destroy, or giving that context another buffer, frees
 * the claim.  Several workspaces may be carved out of one allocation as long as they do not overlap.
 * Errors: RBE_ERR_WORKSPACE, RBE_ERR_NO_DEVICE, RBE_ERR_CUDA. */
rbe_status rbe_set_workspace(rbe_ctx* ctx, void* d_ws, size_t bytes);

/* How the structure-factor kernel may combine atoms (default 3).  For two atoms with q_2 = +-q_1
 * the kernel evaluates q_1 e^{i phi_1} + q_2 e^{i phi_2} = 2 q_1 cos(d) e^{i a} (a, d = half sum and
 * half difference of the phases; a quarter-turn offset for opposite signs): 3 special-function
 * evaluations for two (atom, k) pairs instead of 4.  Atoms are matched by the bit pattern of |q|
 * inside windows of 32 consecutive atoms; unmatched atoms, and every atom when mode = 0, take the
 * plain path, so any charge assignment is handled and the result is the same sum (to rounding).
 *   mode 0: never pair;  1: pair equal charges only;  3: pair equal and opposite charges.
 * Errors: RBE_ERR_INVALID_ARG. */
rbe_status rbe_set_pairing(rbe_ctx* ctx, int32_t mode);

/* Which force kernel rbe_short_range runs (default 0).  Same definition, same tolerances, both bitwise reproducible.
 *   kind 0: cells of side >= r_s; a warp ring over 32 x 32 blocks of atoms, every unordered pair once (Newton's third
 *           law), partial sums of different warps combined in 64-bit fixed point with integer atomics;
 *   kind 1: cells of side >= r_s / 2 (125-cell stencil), one CTA per cell; the cutoff test runs on the tensor cores
 *           (r^2 as a K = 8 TF32 product with a margin, the exact fp32 test repeated at evaluation), every ordered pair
 *           is evaluated by one lane and F_i is written directly: no atomics, no fixed point, no finalise pass.
 * rbe_short_range_bytes covers either.  Errors: RBE_ERR_INVALID_ARG. */
rbe_status rbe_set_pair_kernel(rbe_ctx* ctx, int32_t kind);

/* How rbe_short_range evaluates the pair term of Eq. (2.10) (default 0).
 *   on 0: erfc by a degree-8 polynomial fit (3.4e-7 relative error), exp and 1/r by the special-function unit;
 *   on 1: the paper's method: a table over u = r^2 with interpolation above a small radius, the
 *         analytic form below it.  Tabulated are e^{alpha u} g(r)/r and e^{alpha u} erfc(sqrt(alpha) r)/r (the Gaussian
 *         factored out: one exp2 per pair), 32 intervals per octave of u from 2^-6 A^2 up to r_s^2, a cubic through four
 *         Chebyshev nodes per interval (<= 2e-7 relative interpolation error), rebuilt on the device by every call
 *         (one more kernel) and copied into the shared memory of every CTA.  r_s^2 must stay below 2^26 A^2.
 * Both meet the same tolerance; measured on B200 at N = 1e6, r_s = 10 A: 2.70 ms (0) against 2.73 ms (1).
 * Errors: RBE_ERR_INVALID_ARG. */
rbe_status rbe_set_pair_table(rbe_ctx* ctx, int32_t on);

/* The same table computed on the HOST (the device kernel and this call run one function), for inspection and for tests
 * that need no GPU.  *n_out = number of intervals for this r_s: (floor(log2 r_s^2) + 1 + 6) * 32; interval i covers
 * u = r^2 in u0 + [0, h), u0 = 2^e (1 + m/32), h = 2^e / 32, e = -6 + i / 32, m = i % 32.  h_tf / h_te: float [capacity][4]
 * (host) or NULL, entry i = {c0, c1, c2, c3} with T(u) ~ c0 + c1 d + c2 d^2 + c3 d^3, d = u - u0, where
 * T_f(u) = e^{alpha u} g(r)/r (g of Eq. 2.10) and T_e(u) = e^{alpha u} erfc(sqrt(alpha) r)/r.  Both NULL: size query.
 * Errors: RBE_ERR_INVALID_ARG (also when capacity < *n_out or the table would exceed 1024 intervals). */
rbe_status rbe_pair_table_host(const rbe_ctx* ctx, double rs, float* h_tf, float* h_te, int32_t capacity, int32_t* n_out);

/* Fill *out with the launch geometry chosen for this context (valid after rbe_set_workspace). */
rbe_status rbe_get_launch_info(const rbe_ctx* ctx, rbe_launch_info* out);

/* Algorithm 1 step 1 hand-over: upload the batch of wavevectors.
 *   h_m  int32 [P][3], host: integer triples m_l, k_l = 2 pi m_l / L.  Duplicates allowed.
 *   h_w  double [P], host, or NULL.  NULL: w_l = S / P (Eq. 2.12).  Otherwise w_l = h_w[l];
 *        with w_l = exp(-k_l^2 / 4 alpha) and the k-set = every grid vector the same kernels
 *        evaluate the deterministic sum of Eq. (2.11).
 * The arrays are copied before the call returns (they may be reused immediately); the
 * host-to-device copy is enqueued on `stream`.  Invalidates any previous structure factor.
 * Errors: RBE_ERR_BAD_KVECTOR, RBE_ERR_NOT_READY (no workspace), RBE_ERR_CUDA. */
rbe_status rbe_set_kvectors(rbe_ctx* ctx, const int32_t* h_m, const double* h_w, void* stream);

/* Algorithm 1 step 1 on the device: draw this context's batch of P wavevectors on the GPU,
 * m != 0 with probability ~ exp(-|2 pi m / L|^2 / 4 alpha), weights w_l = S / P.  Exact iid
 * draws (the paper's Metropolis chain is under-specified): each m_d by inverse CDF of
 * the 1-D discrete Gaussian, the zero triple rejected.  Counter-based, so the batch is a pure
 * function of (L, alpha, P, seed, step):
 *   candidate j = 0, 1, ... : words (x, y, z) = first three outputs of Philox4x32-10 with counter
 *   (j mod 2^32, j >> 32, step mod 2^32, step >> 32) and key (seed mod 2^32, seed >> 32);
 *   m_d = #{ i : T_i <= word_d } - M, where c = pi^2 / (alpha L^2), M = ceil(sqrt(40 ln 2 / c)),
 *   T_i = min(2^32 - 1, floor(2^32 * sum_{i' <= i} exp(-c (i' - M)^2) / sum_{all})), i = 0 .. 2M - 1
 *   (fp64, host);
 *   the batch = the first P candidates != (0, 0, 0), in order of j.
 * No host-to-device traffic; replaces rbe_set_kvectors for this step (and invalidates any previous
 * structure factor).  Errors: RBE_ERR_NOT_READY (no workspace), RBE_ERR_INVALID_ARG (M > 2^20:
 * table too large for this L, alpha), RBE_ERR_CUDA. */
rbe_status rbe_sample_kvectors(rbe_ctx* ctx, uint64_t seed, uint64_t step, void* stream);

/* Copy the current k-set back to the host: h_m int32 [P][3].  Synchronises `stream`.
 * Errors: RBE_ERR_NOT_READY (no k-set), RBE_ERR_INVALID_ARG, RBE_ERR_CUDA. */
rbe_status rbe_get_kvectors(rbe_ctx* ctx, int32_t* h_m, void* stream);

/* One whole step -- rbe_sample_kvectors(seed, step) + rbe_structure_factor + rbe_forces -- captured
 * once as a CUDA graph bound to d_xyzq / d_force (float4 [N], device, caller-owned, must stay valid)
 * and replayed with ONE launch per step and no host-to-device traffic: (seed, step) live in the
 * workspace and every replay advances the step by one, starting at first_step.  Meant for the
 * launch-bound small systems and for MD loops that keep positions on the device.
 * rbe_graph_capture synchronises (it uploads the step counter and instantiates the graph);
 * rbe_graph_launch only enqueues on `stream`.  After a replay rbe_kspace_energy and
 * rbe_get_kvectors refer to that step.  A new rbe_set_workspace discards the graph.
 * Errors: RBE_ERR_NOT_READY, RBE_ERR_INVALID_ARG, RBE_ERR_CUDA. */
rbe_status rbe_graph_capture(rbe_ctx* ctx, const void* d_xyzq, void* d_force, int32_t with_energy,
                             uint64_t seed, uint64_t first_step);
rbe_status rbe_graph_launch(rbe_ctx* ctx, void* stream);

/* Algorithm 1 steps 2-3, Eq. (2.9): rho(k_l) for l = 0..P-1 over this context's
 * N atoms, then the per-k force coefficients for rbe_forces.
 *   d_xyzq  float4 [N] = {x, y, z, q} (AoS), device.
 *   d_rho   double2 [P] = {Re, Im}, device, or NULL if the caller does not want a copy.
 * fp32 phases from 32-bit fixed-point fractional coordinates (m . s mod 1 is exact), fp32
 * sincos, fp32 partial sums over at most ~64 atoms, fp64 above that; per-CTA fp64 partials
 * summed in a fixed order (two-level tree) by the last CTAs of the same launch.
 * Errors: RBE_ERR_NOT_READY, RBE_ERR_INVALID_ARG, RBE_ERR_CUDA. */
rbe_status rbe_structure_factor(rbe_ctx* ctx, const void* d_xyzq, void* d_rho, void* stream);

/* Replace the context's structure factors by d_rho (double2 [P], device; copied).  This is the multi-GPU exchange point: each rank computes rho over its
 * own atoms, the ranks sum the P complex numbers (rank order), and each rank injects the
 * global sum here before rbe_forces.  Requires rbe_set_kvectors.
 * Errors: RBE_ERR_NOT_READY, RBE_ERR_INVALID_ARG, RBE_ERR_CUDA. */
rbe_status rbe_set_rho(rbe_ctx* ctx, const void* d_rho, void* stream);

/* Fused multi-GPU exchange of the structure factors (one process per GPU, atoms sharded over the
 * ranks, the k-set replicated: same seed or same host k-set on every rank).  The paper has no
 * multi-GPU path (future work); what must be exchanged is the sum of P complex numbers
 * (P:137).  Each rank owns one exchange buffer of rbe_exchange_bytes(ctx, world) bytes that every
 * peer can address (NVLink peer mapping, e.g. a torch symmetric-memory allocation), zero-filled
 * before the first step.  With an exchange configured, rbe_structure_factor's last CTA writes
 * this rank's partial rho into its slot of EVERY rank's buffer and releases a per-rank flag;
 * rbe_forces / rbe_kspace_energy wait for all `world` flags of the step and add the slots in rank
 * order (bitwise the same rho on every rank): no collective call, no extra launch.  The d_rho copy
 * of rbe_structure_factor then holds this rank's PARTIAL sum.  All ranks must run the same
 * sequence of steps.  A kernel that waits longer than 10 s for a peer gives up and raises a flag
 * that rbe_exchange_check reports (it never hangs the GPU).
 *   d_bufs  host array of `world` device pointers, d_bufs[r] = rank r's buffer as mapped in THIS
 *           process (d_bufs[rank] is the local one), each 256-byte aligned, `bytes` long.
 * Every rbe_set_exchange restarts the step epoch at zero: the buffers of ALL ranks must be zero-filled again
 * (and the ranks synchronised) before the first step after it.  A consumer that gives up waiting writes NaN
 * forces / energy, so a missed rbe_exchange_check cannot pass silently.
 * rbe_set_exchange with world < 1 or d_bufs == NULL switches the exchange off.  Not combinable with
 * rbe_set_rho or rbe_graph_capture (RBE_ERR_INVALID_ARG).
 * Errors: RBE_ERR_INVALID_ARG, RBE_ERR_WORKSPACE (bytes too small), RBE_ERR_CUDA. */
size_t     rbe_exchange_bytes(const rbe_ctx* ctx, int32_t world);
rbe_status rbe_set_exchange(rbe_ctx* ctx, int32_t rank, int32_t world, void* const* d_bufs, size_t bytes);
rbe_status rbe_exchange_check(rbe_ctx* ctx, void* stream);   /* synchronises `stream` */

/* Algorithm 1 step 4, Eq. (2.12): forces on this context's N atoms from the
 * current k-set and structure factors.
 *   d_xyzq   float4 [N], device: the same positions the structure factor was computed from.  The kernel is
 *            launched with programmatic stream serialisation; before it waits for the preceding kernel of the
 *            stream it only issues L2 prefetches for d_xyzq (no value is consumed early), so a preceding
 *            kernel may still be writing the positions.
 *   d_force  float4 [N], device: {F_x, F_y, F_z, e_i}; e_i = 0 unless with_energy != 0, then
 *            e_i = (2 pi q_i / V) sum_l w_l Re(exp(-i k_l . r_i) rho(k_l)) / k_l^2 (sum_i e_i = U).
 * Errors: RBE_ERR_NOT_READY (no structure factor since the last rbe_set_kvectors),
 *         RBE_ERR_INVALID_ARG, RBE_ERR_CUDA. */
rbe_status rbe_forces(rbe_ctx* ctx, const void* d_xyzq, void* d_force, int32_t with_energy,
                      void* stream);

/* Algorithm 1 steps 2-4 -- Eq. (2.9) P:117 then Eq. (2.12) P:131 -- as ONE cooperative kernel launch:
 * structure-factor phase, a grid-wide barrier, a fixed-order reduction of the per-CTA fp64 rows distributed
 * over the CTAs (which also builds every wavevector's force record once), a second barrier, force phase.
 *   h_m, h_w   as rbe_set_kvectors, or h_m == NULL: keep the k-set already on the device (rbe_set_kvectors /
 *              rbe_sample_kvectors).  With h_w == NULL and P <= 512 the wavevectors travel in the kernel
 *              parameters: the step is one launch and no host-to-device copy.
 *   d_xyzq     float4 [N] device;  d_force  float4 [N] device (as rbe_forces);  with_energy as rbe_forces
 *   d_rho      double2 [P] device, or NULL
 * Equivalent to rbe_set_kvectors + rbe_structure_factor + rbe_forces: the same arithmetic per (atom, k) pair,
 * the same tolerances against the definitions; rho differs from rbe_structure_factor's in the last bits only
 * (another fixed order of the per-CTA rows).  Bitwise reproducible.  Afterwards rbe_kspace_energy /
 * rbe_kspace_virial / rbe_forces refer to this step.  Takes the two launches instead when P > 4096, when a
 * multi-GPU exchange is configured, when the device cannot launch cooperatively, or when the system is so large
 * (N * P > 4e6 per SM) that the two-launch kernels are the faster form (rbe_launch_info.step_fused tells).
 * d_xyzq must not be written by other work while the launch runs; no other kernel may share the GPU's SMs with
 * it in a way that keeps part of the grid from becoming resident (the cooperative launch fails rather than hangs).
 * Errors: RBE_ERR_NOT_READY, RBE_ERR_BAD_KVECTOR, RBE_ERR_INVALID_ARG, RBE_ERR_CUDA. */
rbe_status rbe_step(rbe_ctx* ctx, const int32_t* h_m, const double* h_w, const void* d_xyzq, void* d_force,
                    int32_t with_energy, void* d_rho, void* stream);

/* rbe_step for a caller that has no device memory to give, and no way to get any.
 *
 * Everywhere else in this header the scratch a kernel needs (per-CTA partial sums, the reduced rho, the per-k
 * force records, the grid-barrier counter) sits in a workspace the CALLER allocates and hands over with
 * rbe_set_workspace.  That does not suit every host program.  A force plug-in loaded into an MD engine, or into
 * any application whose own pool has already claimed the GPU's memory, may be given the position and force
 * arrays and nothing else: cudaMalloc there either fails outright or takes memory the host program counted on.
 * Code in a time-step loop with a latency budget cannot afford it either, because cudaMalloc and cudaFree
 * stall the whole device while they run.  For such callers this one call computes the same k-space step --
 * Algorithm 1 steps 2-4, Eq. (2.9) P:117 then Eq. (2.12), one cooperative launch of the same
 * kernel as rbe_step -- with its scratch in an array that is part of the library image (a file-scope
 * `static __device__` array in rbe_api.cu).  The call itself, and everything it calls, uses no cudaMalloc,
 * cudaFree, cudaMallocHost or other allocating routine; it needs a context from rbe_create (host memory only,
 * no CUDA call) but NO rbe_set_workspace, and it neither reads nor changes the context's workspace or k-set state
 * (rbe_kspace_energy, rbe_forces etc. do not see this step).
 *
 *   h_m        int32 [P][3], host: the batch of wavevectors, as rbe_set_kvectors (uniform weights S / P only);
 *              they travel in the kernel parameters, so there is no host-to-device copy to stage
 *   d_xyzq     float4 [N] device (caller-owned input);  d_force  float4 [N] device (caller-owned output, as
 *              rbe_forces; .w = e_i if with_energy != 0, else 0);  d_rho  double2 [P] device or NULL (output)
 *
 * Limits.  The array is RBE_STATIC_SCRATCH_BYTES = 1 605 888 bytes (about 1.5 MiB): room for
 * P <= RBE_STATIC_MAX_P = 512 wavevectors and a grid of at most RBE_STATIC_MAX_CTAS = 192 CTAs (the kernel runs
 * one CTA per SM: 148 on B200).  N is not limited by it (the scratch does not grow with N).  A larger P, or a
 * device with more SMs than that, is refused with RBE_ERR_WORKSPACE and a message naming the limit; nothing is
 * launched.  Every GPU on which a process has loaded librbe.so holds one copy of the array, from the moment the
 * library's code is loaded onto it until the process exits, whether or not this call is ever made.
 *
 * First call on a device.  The first rbe_step_static on each device (with that device current) also does a
 * one-time set-up on the host: it looks up the array's device address (cudaGetSymbolAddress) and raises the
 * kernel's shared-memory limit.  Make that first call outside any stream capture; later calls only enqueue a
 * 8-byte memset (the barrier counter must start at zero, and the array keeps whatever the previous call left
 * in it) and the kernel on `stream`.
 *
 * Sharing.  There is ONE array per device, shared by every context, host thread and stream of the process.  Calls
 * that follow one another on one stream are safe.  Two rbe_step_static calls whose kernels could run at the same
 * time on one device -- different streams without an event between them, or two host threads -- race on it: wrong
 * forces, or a grid barrier that never opens.  Serialise them.  It is independent of every workspace, so it may
 * overlap with the other calls of this header.
 * Results: the same arithmetic, launch geometry and summation order as the one-launch form of rbe_step with h_m given.
 * Errors: RBE_ERR_INVALID_ARG (null / misaligned pointer, or the context was first used on another device),
 *         RBE_ERR_BAD_KVECTOR, RBE_ERR_WORKSPACE (beyond the limits above), RBE_ERR_NO_DEVICE, RBE_ERR_CUDA. */
#define RBE_STATIC_MAX_P 512
#define RBE_STATIC_MAX_CTAS 192
#define RBE_STATIC_SCRATCH_BYTES 1605888
rbe_status rbe_step_static(rbe_ctx* ctx, const int32_t* h_m, const void* d_xyzq, void* d_force, int32_t with_energy,
                           void* d_rho, void* stream);

/* Real-space partner of the RBE force: the short-range part of the Ewald-split Coulomb force,
 * Eq. (2.10), truncated at the cutoff radius r_s, over a linked-cell list of cubic
 * cells of side >= r_s (a one-shot cell list; Algorithm 2's own list has cells of side r_c):
 *   F_i = - q_i sum_{j != i, r < r_s} q_j ( erfc(sqrt(alpha) r) / r^2
 *            + 2 sqrt(alpha) exp(-alpha r^2) / (sqrt(pi) r) ) d / r,   d = nearest image of r_j - r_i
 *   e_i = 1/2 q_i sum_{j != i, r < r_s} q_j erfc(sqrt(alpha) r) / r      (first term of Eq. 2.8)
 * with this context's L and alpha.  Coincident atoms (r = 0) are skipped.  Independent of the
 * k-set; needs no rbe_set_workspace.  fp32 arithmetic on cell-relative coordinates derived from exact
 * fixed-point separations; erfc by a degree-8 polynomial fit with 3.4e-7 RELATIVE error for x <= 10, or the pair term
 * from a table (rbe_set_pair_table).  Every unordered pair
 * is evaluated once (Newton's third law); partial sums of different warps are combined in 64-bit
 * fixed point with integer atomics (scale 2^40: |F_i / q_i| must stay below 8.4e6 e/A^2, and partial sums
 * below 9e-13 e/A^2 are lost), so the result
 * is bitwise reproducible.
 *   d_xyzq      float4 [N] device;  rs  cutoff radius [A], 0 < rs <= L/3
 *   d_force     float4 [N] device: {F_x, F_y, F_z, e_i}; e_i = 0 unless with_energy != 0
 *   accumulate  != 0: add to what d_force holds (e.g. the k-space force of rbe_forces)
 *   d_ws        caller-owned device scratch of rbe_short_range_bytes(ctx, rs) bytes (~76 B per atom
 *               + 204 B per cell), 256-byte aligned; its contents are rebuilt by every call
 * rbe_short_range_bytes returns 0 for an invalid rs.  Enqueues seven kernels (eight with rbe_set_pair_table) and two memsets on `stream`.
 * Errors: RBE_ERR_INVALID_ARG, RBE_ERR_WORKSPACE, RBE_ERR_NO_DEVICE, RBE_ERR_CUDA. */
size_t     rbe_short_range_bytes(const rbe_ctx* ctx, double rs);
rbe_status rbe_short_range(rbe_ctx* ctx, const void* d_xyzq, double rs, void* d_force, int32_t accumulate,
                           int32_t with_energy, void* d_ws, size_t ws_bytes, void* stream);

/* Random batch list (RBL) estimate of the same short-range force: section 2.3, Eqs. (2.13)-(2.16)
 * P:145-166, Algorithm 2, with F_ij the electrostatic pair force of Eq. (2.10):
 *   F_i = sum_{j: r < r_c} F_ij + (N_s / p) sum_{j in B(i)} F_ij + F^corr,  F^corr = -(1/N) sum_i (...)
 * where N_s counts the shell r_c <= r < r_s of atom i and B(i) holds the min(p, N_s) shell members with the
 * smallest keys u_ij.  The paper does not say how the p members are drawn; here (reading Q20)
 *   (s0, s1) = first two words of Philox4x32-10 with counter (step mod 2^32, step >> 32, 0, 0) and key
 *              (seed mod 2^32, seed >> 32)                       [once per call, on the host]
 *   u_ij     = fmix32( (i * 0x9E3779B1 + s0) xor (j * 0x85EBCA77 + s1) )   mod 2^32, i and j atom indices,
 *   fmix32(h): h ^= h >> 16; h *= 0x85EBCA6B; h ^= h >> 13; h *= 0xC2B2AE35; h ^= h >> 16
 * -- a uniformly random p-subset, a pure function of (seed, step), distinct keys for distinct j.  N_s <= p:
 * the whole shell, scale 1.  Cell list with cells of side max(r_c, r_s / 4) (Algorithm 2: side r_c),
 * one CTA per cell, a warp per atom.  Forces only (d_force[i].w = 0, or unchanged with accumulate).
 * 1 <= p <= 32, 0 < rc < rs, and the 2R + 1 cells of side c = L / floor(L / max(r_c, r_s / 4)) that the shell spans
 * (R = ceil(r_s / c) <= 4) must fit the box (r_s below about 0.44 L).  d_ws: caller-owned scratch of rbe_rbl_bytes(ctx, rc, rs) bytes (~76 B per atom
 * + 204 B per cell), 256-byte aligned; rbe_rbl_bytes returns 0 for invalid radii.  Bitwise reproducible.
 * Errors: RBE_ERR_INVALID_ARG, RBE_ERR_WORKSPACE, RBE_ERR_NO_DEVICE, RBE_ERR_CUDA. */
size_t     rbe_rbl_bytes(const rbe_ctx* ctx, double rc, double rs);
rbe_status rbe_rbl_forces(rbe_ctx* ctx, const void* d_xyzq, double rc, double rs, int32_t p, uint64_t seed,
                          uint64_t step, void* d_force, int32_t accumulate, void* d_ws, size_t ws_bytes,
                          void* stream);

/* U = (2 pi / V) sum_l w_l |rho(k_l)|^2 / k_l^2 for the current k-set and structure factors,
 * summed in fp64 in a fixed order; written to *h_U (host).  Synchronises `stream`.
 * Errors: RBE_ERR_NOT_READY, RBE_ERR_INVALID_ARG, RBE_ERR_CUDA. */
rbe_status rbe_kspace_energy(rbe_ctx* ctx, double* h_U, void* stream);

/* k-space virial of the current k-set and structure factors (for the pressure of the isothermal-
 * isobaric variant the paper names; the paper gives no estimator): minus the strain derivative
 * of the second term of Eq. (2.8) P:112 with the weights of Eq. (2.12),
 *   W_ab = sum_l (2 pi w_l / V) |rho_l|^2 / k_l^2 [ delta_ab - 2 k_la k_lb / k_l^2 (1 + k_l^2 / 4 alpha) ],
 * h_W double [6] (host) = W_xx, W_yy, W_zz, W_xy, W_xz, W_yz in e^2/A; fp64, fixed order.
 * Synchronises `stream`.  Errors: RBE_ERR_NOT_READY, RBE_ERR_INVALID_ARG, RBE_ERR_CUDA. */
rbe_status rbe_kspace_virial(rbe_ctx* ctx, double* h_W, void* stream);

/* One whole step from HOST buffers (the end-to-end path): copies h_xyzq (float [N][4]) to the
 * device, uploads the k-set, runs rbe_structure_factor and rbe_forces, copies the forces back
 * into h_force (float [N][4]) and, if h_U != NULL, the energy into *h_U; synchronises `stream`.
 * d_scratch: caller-owned device buffer of at least rbe_step_host_bytes(ctx, 0) bytes (positions + forces:
 * about 32 B per atom), 256-byte aligned.
 * With N >= 131 072 the atoms travel in up to 4 chunks on two internal copy streams so that the
 * transfers overlap the kernels (every chunk adds to the same per-CTA fp64 partial rows in stream
 * order: the result stays bitwise reproducible).  Pinned host buffers (rbe_host_alloc) make the
 * copies asynchronous; pageable ones work but are slower.
 * Errors: as the calls it is made of, plus RBE_ERR_WORKSPACE if d_scratch is too small. */
size_t     rbe_step_host_bytes(const rbe_ctx* ctx, int32_t compact);   /* d_scratch size: compact = 0 rbe_step_host, 1 rbe_step_host_xyz */
rbe_status rbe_step_host(rbe_ctx* ctx, const float* h_xyzq, const int32_t* h_m, const double* h_w,
                         float* h_force, int32_t with_energy, double* h_U, void* d_scratch,
                         size_t scratch_bytes, void* stream);

/* Compact end-to-end step for MD loops, where the charges never change: only POSITIONS travel to the
 * device (h_xyz float [N][3]) and only force vectors travel back (h_force3 float [N][3]): 24 B per
 * atom over PCIe instead of 32.  The charges live on the device: rbe_set_charges(ctx, d_q) registers a
 * caller-owned device array float [N] (retained until replaced; NULL unregisters).  Same chunked
 * pipeline and the same two hot kernels as rbe_step_host, plus a pack and an unpack kernel per chunk;
 * the forces are bitwise those of rbe_step_host.  d_scratch: at least rbe_step_host_bytes(ctx, 1)
 * bytes (about 56 B per atom), 256-byte aligned.  Per-atom energies are not returned; h_U (optional) receives the k-space energy.
 * Synchronises `stream`.  Errors: as rbe_step_host, plus RBE_ERR_NOT_READY without rbe_set_charges. */
rbe_status rbe_set_charges(rbe_ctx* ctx, const void* d_q);
rbe_status rbe_step_host_xyz(rbe_ctx* ctx, const float* h_xyz, const int32_t* h_m, const double* h_w,
                             float* h_force3, double* h_U, void* d_scratch, size_t scratch_bytes,
                             void* stream);

/* NVE velocity-Verlet loop (the paper integrates with velocity-Verlet, and runs the NVE ensemble among
 * others).  State in fp64, owned by the caller, on the device: positions
 * d_pos double [N][3], velocities d_vel double [N][3], inverse masses d_inv_mass double [N]; the force kernels
 * read d_xyzq float4 [N] = positions rounded to fp32 + charges, which rbe_nve_kick keeps in step.  Units: A, e,
 * amu, hence times in tau = sqrt(amu A^3 / e^2) = 2.68285 fs (reading Q21).
 *
 * rbe_nve_kick:  v += half_dt * F / m  from d_force float4 [N] (.w ignored); then, if d_pos != NULL, the drift
 *   x += dt * v and d_xyzq[i].xyz = (float) x[i] (d_xyzq[i].w, the charge, is kept).  One step of the scheme is
 *   kick(dt/2, drift dt) -> forces at the new positions -> kick(dt/2, no drift).  Enqueues one kernel.
 *   An inverse mass of 0 freezes an atom's velocity.  Positions are NOT wrapped into the box: the fp64 positions stay
 *   continuous (handy for displacements), and the force kernels are exactly periodic, but the fp32 copy in d_xyzq
 *   loses resolution as |x| grows (ulp(x) = 2^-23 |x|), so in runs where atoms diffuse over many box lengths the caller
 *   should subtract whole box vectors from d_pos now and then.
 * rbe_nve_energies:  h_out double [2] (host) = { sum_i 1/2 m_i v_i^2 over the atoms with inverse mass > 0 (0 if d_vel == NULL), sum_i d_force[i].w
 *   (0 if d_force == NULL: with_energy forces carry the per-atom potential energies there) }, fp64, fixed order;
 *   synchronises `stream`; needs the workspace.
 * rbe_md_capture:  one whole MD step -- kick + drift, [a fresh batch from the device sampler if sampled != 0:
 *   (seed, step) as rbe_graph_capture; else the k-set and weights already on the device, e.g. the full grid with
 *   w_l = exp(-k_l^2 / 4 alpha): deterministic Ewald], the k-space step (rbe_step's kernels), rbe_short_range
 *   with accumulate = 1 and cutoff rs (d_sr_ws of rbe_short_range_bytes(ctx, rs) bytes), kick -- captured ONCE as
 *   a CUDA graph bound to these arrays and replayed by rbe_graph_launch with one launch per step, positions and
 *   velocities resident on the device.  Before the first replay d_force must hold the forces of the current
 *   positions (rbe_step + rbe_short_range(accumulate)).  with_energy != 0: d_force[i].w carries the per-atom
 *   k-space + short-range potential energy after every step.  Synchronises; replaces any rbe_graph_capture graph.
 * Nothing on this path keeps unlike charges apart (the paper's Lennard-Jones term, Eq. 2.2, is out of scope):
 * meant for short horizons from a perturbed crystal.
 * Errors: RBE_ERR_INVALID_ARG, RBE_ERR_NOT_READY, RBE_ERR_WORKSPACE, RBE_ERR_CUDA. */
rbe_status rbe_nve_kick(rbe_ctx* ctx, void* d_vel, const void* d_inv_mass, const void* d_force, double half_dt,
                        void* d_pos, void* d_xyzq, double dt, void* stream);
rbe_status rbe_nve_energies(rbe_ctx* ctx, const void* d_vel, const void* d_inv_mass, const void* d_force,
                            double* h_out, void* stream);
rbe_status rbe_md_capture(rbe_ctx* ctx, void* d_pos, void* d_vel, const void* d_inv_mass, void* d_xyzq, void* d_force,
                          double rs, double dt, void* d_sr_ws, size_t sr_bytes, int32_t sampled, uint64_t seed,
                          uint64_t first_step, int32_t with_energy);

/* Measure, on this device and now, the issue rates that bound this path (there is no vendor-stated figure to
 * take them from): h_out double [5] (host) = thread-instructions per SM per clock of FFMA, IMAD, I2FP.F32.S32
 * and MUFU.SIN (dependent-free chains, 32 warps per SM, in-kernel clock64), and the SM clock in MHz observed
 * while the MUFU probe ran (its cycles / its CUDA-event time).  Four short launches (~0.2 ms in all) that use the
 * workspace as scratch: call it between steps (it invalidates the per-CTA rows of a chunked host step in
 * flight, nothing else).  Synchronises `stream`.  Errors: RBE_ERR_NOT_READY, RBE_ERR_INVALID_ARG, RBE_ERR_CUDA. */
rbe_status rbe_probe_pipe_rates(rbe_ctx* ctx, double* h_out, void* stream);

/* Page-locked (pinned) HOST memory for the end-to-end path: cudaHostAlloc'ed, so that the copies of
 * rbe_step_host are asynchronous DMA transfers at full PCIe rate (measured on B200 hosts: 55 GB/s
 * from such a buffer, 15-40 GB/s and erratic from memory pinned after allocation).  The caller
 * owns the buffer until rbe_host_free.  No context is needed.
 * Errors: RBE_ERR_INVALID_ARG (out == NULL or bytes == 0), RBE_ERR_NO_DEVICE, RBE_ERR_CUDA. */
rbe_status rbe_host_alloc(void** out, size_t bytes);
rbe_status rbe_host_free(void* h_ptr);

/* Text of the last error on this context (owned by the context; "" if none).  For ctx == NULL
 * returns a static string. */
const char* rbe_last_error(const rbe_ctx* ctx);

/* Static name of a status code. */
const char* rbe_status_string(rbe_status s);

/* Library version: major * 10000 + minor * 100 + patch. */
int32_t rbe_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RBE_H_ */
