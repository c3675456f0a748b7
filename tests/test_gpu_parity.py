"""Parity of the CUDA path (through the C ABI) against the fp64 oracle, element by element on
the same seeded inputs and the same k-set.  Tolerances are BASELINE.json north_star's
(reading Q15):

  rho : max_l |rho_gpu,l - rho_or,l|            <= 1e-6 * sum_j |q_j|
  F   : ||F_gpu - F_or||_2 / ||F_or||_2          <= 2e-5   (all 3N components, or the sample)
  U   : |U_gpu - U_or| / |U_or|                  <= 1e-5
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2407_09315_b200 import inputs, rbe

pytestmark = pytest.mark.gpu

RHO_TOL, F_TOL, U_TOL = 1e-6, 2e-5, 1e-5


def gpu_step(atoms, L, alpha, m, w=None, with_energy=False):
    N, P = atoms.shape[0], m.shape[0]
    ctx = rbe.Rbe(N, L, alpha, P)
    xyzq = torch.from_numpy(atoms).cuda()
    rho = torch.empty((P, 2), dtype=torch.float64, device="cuda")
    force = torch.full((N, 4), float("nan"), dtype=torch.float32, device="cuda")
    ctx.rbe_set_kvectors(m, w)
    ctx.rbe_structure_factor(xyzq, rho)
    ctx.rbe_forces(xyzq, force, with_energy)
    U = ctx.rbe_kspace_energy()
    torch.cuda.synchronize()
    return ctx, rho.cpu().numpy(), force.cpu().numpy(), U


def gpu_fused_step(atoms, L, alpha, m, w=None, with_energy=False):
    """The same step through rbe_step: ONE cooperative launch (SF phase, grid barrier, distributed
    fixed-order reduction, grid barrier, F phase)."""
    N, P = atoms.shape[0], m.shape[0]
    ctx = rbe.Rbe(N, L, alpha, P)
    xyzq = torch.from_numpy(atoms).cuda()
    rho = torch.full((P, 2), float("nan"), dtype=torch.float64, device="cuda")
    force = torch.full((N, 4), float("nan"), dtype=torch.float32, device="cuda")
    ctx.rbe_step(m, xyzq, force, w=w, with_energy=with_energy, rho=rho)
    U = ctx.rbe_kspace_energy()
    torch.cuda.synchronize()
    return ctx, rho.cpu().numpy(), force.cpu().numpy(), U


def check(atoms, L, alpha, m, w=None, with_energy=False, sel=None, f_tol=F_TOL):
    """Both product paths against the oracle: the two launches (rbe_structure_factor + rbe_forces) and the
    one-launch rbe_step.  Returns the errors of the one-launch path (what bench.py times)."""
    cache = {}
    _check_path(gpu_step, cache, atoms, L, alpha, m, w, with_energy, sel, f_tol)
    return _check_path(gpu_fused_step, cache, atoms, L, alpha, m, w, with_energy, sel, f_tol)


def _check_path(run, cache, atoms, L, alpha, m, w, with_energy, sel, f_tol):
    ctx, rho_g, F_g, U_g = run(atoms, L, alpha, m, w, with_energy)
    S = oracle.S(L, alpha)
    assert abs(ctx.rbe_normaliser_S() - S) <= 1e-13 * S
    if "rho" not in cache:
        cache["rho"] = oracle.rho(atoms, L, m)
        cache["F"] = oracle.force(atoms, L, m, S, cache["rho"], w=w, sel=sel, with_energy=with_energy)
    rho_o = cache["rho"]
    qsum = np.abs(atoms[:, 3].astype(np.float64)).sum()
    err_rho = np.abs(rho_g - rho_o).max() if len(m) else 0.0
    assert err_rho <= RHO_TOL * max(qsum, 1e-300), (err_rho, qsum)
    out = cache["F"]
    F_o, e_o = out if with_energy else (out, None)
    Fg = F_g[:, :3].astype(np.float64)
    if sel is not None:
        Fg = Fg[sel]
    nrm = np.linalg.norm(F_o)
    err_F = np.linalg.norm(Fg - F_o) / nrm if nrm > 0 else np.abs(Fg).max()
    assert err_F <= f_tol, err_F
    U_o = oracle.energy(L, m, S, rho_o, w=w)
    assert abs(U_g - U_o) <= U_TOL * abs(U_o) + 1e-300, (U_g, U_o)
    eg = F_g[:, 3].astype(np.float64)
    if with_energy:
        egs = eg if sel is None else eg[sel]
        assert np.linalg.norm(egs - e_o) <= 2e-5 * np.linalg.norm(e_o) + 1e-12
    else:
        assert np.all(eg == 0.0)
    assert np.isfinite(F_g).all()
    return dict(rho=err_rho / max(qsum, 1e-300), F=err_F, U=abs(U_g - U_o) / max(abs(U_o), 1e-300),
                F_gpu=F_g, rho_gpu=rho_g)


# ------------------------------------------------------------------ BASELINE.json configs
@pytest.mark.parametrize("name", ["water_3k", "water_96k"])
@pytest.mark.parametrize("with_energy", [False, True])
def test_config_small(name, with_energy):
    cfg = inputs.CONFIGS[name]
    atoms = inputs.make_atoms(cfg)
    m = inputs.sample_kset(cfg.L, cfg.alpha, cfg.P, cfg.seed, 0)
    r = check(atoms, cfg.L, cfg.alpha, m, with_energy=with_energy)
    # momentum conservation on the GPU result: |sum_i F_i|_inf <= 1e-6 * sum_i |F_i|_inf
    F = r["F_gpu"][:, :3].astype(np.float64)
    assert np.abs(F.sum(0)).max() <= 1e-6 * np.abs(F).max(1).sum()


def _momentum_ok(F_gpu):
    F = F_gpu[:, :3].astype(np.float64)
    assert np.abs(F.sum(0)).max() <= 1e-6 * np.abs(F).max(1).sum()


def test_config_1m_full_size_bench_configuration():
    """Config 3 (N = 999 999, P = 200) in the launch configuration bench.py times: rho and ALL 3N
    force components against the full oracle (Eq. 2.9, Eq. 2.12), sum F = 0."""
    cfg = inputs.CONFIGS["water_nacl_1m"]
    atoms = inputs.make_atoms(cfg)
    m = inputs.sample_kset(cfg.L, cfg.alpha, cfg.P, cfg.seed, 0)
    r = check(atoms, cfg.L, cfg.alpha, m, with_energy=False)
    _momentum_ok(r["F_gpu"])


def test_config_10m_full():
    """Config 4 (N = 9 999 999, P = 200): every force component against the oracle (~7 s of oracle time)."""
    cfg = inputs.CONFIGS["water_10m"]
    atoms = inputs.make_atoms(cfg)
    m = inputs.sample_kset(cfg.L, cfg.alpha, cfg.P, cfg.seed, 0)
    r = check(atoms, cfg.L, cfg.alpha, m)
    _momentum_ok(r["F_gpu"])


@pytest.mark.parametrize("P", [50, 100, 200, 400, 800, 1600])
def test_ion_sweep_batch_sizes_at_1m(P):
    """Config 5, the P sweep at its own N = 1e6: rho and all 3N force components against the oracle."""
    cfg = inputs.ions_config(10 ** 6, P=P)
    atoms = inputs.make_atoms(cfg)
    m = inputs.sample_kset(cfg.L, cfg.alpha, cfg.P, cfg.seed, 0)
    r = check(atoms, cfg.L, cfg.alpha, m, with_energy=(P == 100))
    _momentum_ok(r["F_gpu"])


@pytest.mark.parametrize("N", [10 ** 4, 10 ** 5, 10 ** 7])
def test_ion_sweep_sizes_at_p200(N):
    """Config 5, the N sweep at P = 200 (N = 1e6 is in the P sweep above, 1e8 below): full oracle."""
    cfg = inputs.ions_config(N, P=200)
    atoms = inputs.make_atoms(cfg)
    m = inputs.sample_kset(cfg.L, cfg.alpha, cfg.P, cfg.seed, 0)
    r = check(atoms, cfg.L, cfg.alpha, m)
    _momentum_ok(r["F_gpu"])


def test_ions_1e8_max_size_at_p200():
    """The largest sweep point at its own batch size (N = 1e8, L = 1000 A, P = 200: the hardest case
    for fp32 phases), as SURVEY.md s8(d) prescribes: oracle rho for all 200 wavevectors once, oracle
    forces on a seeded subset of 1e5 atoms (plus the ragged tail)."""
    cfg = inputs.ions_config(10 ** 8, P=200)
    atoms = inputs.make_atoms(cfg)
    m = inputs.sample_kset(cfg.L, cfg.alpha, cfg.P, cfg.seed, 0)
    sel = np.sort(np.random.default_rng(2).choice(cfg.N, 100_000, replace=False)).astype(np.int64)
    sel[-2:] = [cfg.N - 2, cfg.N - 1]
    check(atoms, cfg.L, cfg.alpha, m, sel=sel)


# ------------------------------------------------------------------------ ragged / edge
@pytest.mark.parametrize("N", [1, 2, 31, 32, 33, 1000, 4097, 20011])
def test_ragged_atom_counts(N):
    cfg = inputs.ions_config(20_012)
    atoms = inputs.make_atoms(cfg)[:N].copy()
    m = inputs.sample_kset(cfg.L, cfg.alpha, 100, 11, N)
    check(atoms, cfg.L, cfg.alpha, m, with_energy=True)


@pytest.mark.parametrize("P", [1, 3, 4, 5, 50, 127, 200, 257, 400, 800, 1600, 2049, 4500])
def test_ragged_batch_sizes(P):
    cfg = inputs.ions_config(10_000)
    atoms = inputs.make_atoms(cfg)
    m = inputs.sample_kset(cfg.L, cfg.alpha, P, 12, P)
    check(atoms, cfg.L, cfg.alpha, m, with_energy=(P % 2 == 1))


# ------------------------------------------------------------ equal-|q| pairing (sf_kernel)
def _charge_case(kind, n, rng):
    if kind == "all_distinct":          # nothing pairs: every atom takes the plain path
        return (rng.random(n) * 2 - 1 + 1e-3).astype(np.float32)
    if kind == "all_equal":             # one class, non-neutral
        return np.full(n, 0.75, dtype=np.float32)
    if kind == "with_zeros":            # zero charges are dropped, the rest pair
        q = np.where(np.arange(n) % 3 == 0, 0.0, np.where(np.arange(n) % 2 == 0, 1.0, -1.0))
        return q.astype(np.float32)
    if kind == "odd_classes":           # class sizes are odd inside most 32-atom windows
        return np.array([0.5, -0.5, 0.5, 1.25, -0.5, 0.5, 2.0], dtype=np.float32)[np.arange(n) % 7]
    if kind == "negative_zero":
        q = np.where(np.arange(n) % 2 == 0, 1.0, -1.0).astype(np.float32)
        q[::5] = -0.0
        return q
    raise ValueError(kind)


@pytest.mark.parametrize("kind", ["all_distinct", "all_equal", "with_zeros", "odd_classes", "negative_zero"])
def test_pairing_handles_any_charge_assignment(kind):
    rng = np.random.default_rng(21)
    n, L, alpha = 9_001, 40.0, 0.09
    atoms = np.empty((n, 4), dtype=np.float32)
    atoms[:, :3] = rng.random((n, 3)) * L
    atoms[:, 3] = _charge_case(kind, n, rng)
    m = inputs.sample_kset(L, alpha, 100, 22)
    check(atoms, L, alpha, m, with_energy=True)


@pytest.mark.parametrize("name", ["water_96k", "ions_20000"])
def test_pairing_modes_agree(name):
    """rbe_set_pairing 0 / 1 / 3 evaluate the same sum: rho agrees to rounding, well inside the
    tolerance, whichever atoms the kernel combines."""
    cfg = inputs.CONFIGS[name] if name in inputs.CONFIGS else inputs.ions_config(20_000)
    atoms = inputs.make_atoms(cfg)
    m = inputs.sample_kset(cfg.L, cfg.alpha, cfg.P, cfg.seed, 3)
    xyzq = torch.from_numpy(atoms).cuda()
    out = {}
    for mode in (0, 1, 3):
        ctx = rbe.Rbe(cfg.N, cfg.L, cfg.alpha, cfg.P)
        ctx.rbe_set_pairing(mode)
        rho = torch.empty((cfg.P, 2), dtype=torch.float64, device="cuda")
        ctx.rbe_set_kvectors(m)
        ctx.rbe_structure_factor(xyzq, rho)
        out[mode] = rho.cpu().numpy()
    qsum = np.abs(atoms[:, 3].astype(np.float64)).sum()
    rho_o = oracle.rho(atoms, cfg.L, m)
    for mode in (0, 1, 3):
        assert np.abs(out[mode] - rho_o).max() <= RHO_TOL * qsum
        # far tighter than the bar: relative to |rho| itself (cancellation in neutral molecules kept)
        rel = np.hypot(*(out[mode] - rho_o).T) / np.hypot(*rho_o.T)
        assert np.median(rel) <= 2e-5, (mode, np.median(rel))
    with pytest.raises(rbe.RbeError):
        ctx.rbe_set_pairing(2)


def test_empty_system():
    m = inputs.sample_kset(20.0, 0.09, 16, 1)
    ctx, rho, F, U = gpu_step(np.zeros((0, 4), dtype=np.float32), 20.0, 0.09, m)
    assert np.all(rho == 0.0) and F.shape == (0, 4) and U == 0.0


def test_positions_far_outside_the_box_and_extreme_m():
    """Periodic wrap is implicit (reading Q6); |m_d| up to 2^15 - 1 is accepted (reading Q10)."""
    L, alpha = 64.0, 0.09
    rng = np.random.default_rng(3)
    n = 50_000  # the fixed-point phase error |m| 2^-33 turns adds up like sqrt(N); the bar like N
    atoms = np.empty((n, 4), dtype=np.float32)
    atoms[:, :3] = (rng.random((n, 3)) * 40 - 20) * L  # up to 20 boxes away
    atoms[:, 3] = np.where(np.arange(n) % 2 == 0, 1.0, -1.0)
    m = inputs.sample_kset(L, alpha, 64, 5)
    m[0] = [32767, -32767, 32767]
    m[1] = [-32767, 0, 1]
    # |x| ~ 1280 A carries an fp32 ulp of 1.2e-4 A; the oracle sees the same fp32 values
    check(atoms, L, alpha, m, with_energy=True)


def test_weighted_full_grid_reproduces_deterministic_ewald():
    """w_l = exp(-k_l^2/4alpha) over every grid vector: the GPU kernels evaluate Eq. (2.11) and
    the second term of Eq. (2.8) -- compared with oracle.ewald_full, not with the RBE oracle."""
    L, alpha, mmax = 12.0, 0.3, 7
    cfg = inputs.ions_config(400)
    atoms = inputs.make_atoms(cfg)
    atoms[:, :3] *= np.float32(L / cfg.L)
    m = inputs.full_kgrid(mmax)
    k2 = (2 * np.pi / L) ** 2 * (m.astype(np.float64) ** 2).sum(1)
    w = np.exp(-k2 / (4 * alpha))
    ctx, rho, F, U = gpu_step(atoms, L, alpha, m, w=w, with_energy=True)
    Uref, _, Fl = oracle.ewald_full(atoms[:, :3].astype(np.float64), atoms[:, 3].astype(np.float64),
                                    L, alpha, nreal=0, mmax=mmax)
    assert np.linalg.norm(F[:, :3] - Fl) / np.linalg.norm(Fl) <= F_TOL
    assert abs(U - Uref[1]) <= U_TOL * abs(Uref[1])
    assert abs(F[:, 3].astype(np.float64).sum() - Uref[1]) <= 1e-4 * abs(Uref[1])


def test_bitwise_reproducible_and_k_resubmission():
    cfg = inputs.CONFIGS["water_96k"]
    atoms = inputs.make_atoms(cfg)
    xyzq = torch.from_numpy(atoms).cuda()
    ctx = rbe.Rbe(cfg.N, cfg.L, cfg.alpha, cfg.P)
    outs = []
    for step in (0, 1, 0):
        m = inputs.sample_kset(cfg.L, cfg.alpha, cfg.P, cfg.seed, step)
        rho = torch.empty((cfg.P, 2), dtype=torch.float64, device="cuda")
        F = torch.empty((cfg.N, 4), dtype=torch.float32, device="cuda")
        ctx.rbe_set_kvectors(m)
        ctx.rbe_structure_factor(xyzq, rho)
        ctx.rbe_forces(xyzq, F)
        outs.append((rho.cpu().numpy().copy(), F.cpu().numpy().copy(), ctx.rbe_kspace_energy()))
    assert np.array_equal(outs[0][0], outs[2][0]) and np.array_equal(outs[0][1], outs[2][1])
    assert outs[0][2] == outs[2][2]
    assert not np.array_equal(outs[0][0], outs[1][0])


def test_call_order_errors_on_device():
    ctx = rbe.Rbe(64, 10.0, 0.3, 4)
    xyzq = torch.zeros((64, 4), dtype=torch.float32, device="cuda")
    F = torch.zeros((64, 4), dtype=torch.float32, device="cuda")
    with pytest.raises(rbe.RbeError) as e:
        ctx.rbe_structure_factor(xyzq)
    assert e.value.status == 3
    ctx.rbe_set_kvectors(np.array([[1, 0, 0], [0, 1, 0], [0, 0, 1], [1, 1, 1]], dtype=np.int32))
    with pytest.raises(rbe.RbeError) as e:
        ctx.rbe_forces(xyzq, F)
    assert e.value.status == 3
    ctx.rbe_structure_factor(xyzq)
    ctx.rbe_forces(xyzq, F)
    ctx.rbe_set_kvectors(np.array([[2, 0, 0], [0, 1, 0], [0, 0, 1], [1, 1, 1]], dtype=np.int32))
    with pytest.raises(rbe.RbeError):  # a new k-set invalidates the structure factor
        ctx.rbe_forces(xyzq, F)
    info = ctx.rbe_get_launch_info()
    assert info["num_sms"] >= 100 and info["sf_grid_x"] >= 1


def test_two_shards_with_rank_ordered_sum_match_single_context():
    """Multi-GPU data path on one device: two contexts own half the atoms each; the partial
    structure factors are summed in rank order and injected with rbe_set_rho."""
    cfg = inputs.CONFIGS["water_96k"]
    atoms = inputs.make_atoms(cfg)
    m = inputs.sample_kset(cfg.L, cfg.alpha, cfg.P, cfg.seed, 0)
    parts, ctxs, xs = [], [], []
    for rank in range(2):
        lo, hi = inputs.shard_bounds(cfg.N, 2, rank, align=32)
        x = torch.from_numpy(atoms[lo:hi].copy()).cuda()
        c = rbe.Rbe(hi - lo, cfg.L, cfg.alpha, cfg.P)
        rho = torch.empty((cfg.P, 2), dtype=torch.float64, device="cuda")
        c.rbe_set_kvectors(m)
        c.rbe_structure_factor(x, rho)
        parts.append(rho); ctxs.append(c); xs.append(x)
    total = parts[0] + parts[1]
    Fs = []
    for c, x in zip(ctxs, xs):
        F = torch.empty((x.shape[0], 4), dtype=torch.float32, device="cuda")
        c.rbe_set_rho(total)
        c.rbe_forces(x, F)
        Fs.append(F.cpu().numpy())
    F_g = np.concatenate(Fs)[:, :3].astype(np.float64)
    S = oracle.S(cfg.L, cfg.alpha)
    rho_o = oracle.rho(atoms, cfg.L, m)
    F_o = oracle.force(atoms, cfg.L, m, S, rho_o)
    assert np.abs(total.cpu().numpy() - rho_o).max() <= RHO_TOL * np.abs(atoms[:, 3]).sum()
    assert np.linalg.norm(F_g - F_o) / np.linalg.norm(F_o) <= F_TOL


def test_host_buffer_step_matches_device_path():
    cfg = inputs.CONFIGS["water_3k"]
    atoms = inputs.make_atoms(cfg)
    m = inputs.sample_kset(cfg.L, cfg.alpha, cfg.P, cfg.seed, 0)
    ctx, rho_g, F_g, U_g = gpu_step(atoms, cfg.L, cfg.alpha, m, with_energy=True)
    h_x = torch.from_numpy(atoms).pin_memory()
    h_f = torch.empty((cfg.N, 4), dtype=torch.float32).pin_memory()
    U = ctx.rbe_step_host(h_x, m, h_f, with_energy=True, want_energy=True)
    assert np.array_equal(h_f.numpy(), F_g) and U == U_g


@pytest.mark.parametrize("N", [131_073, 300_000])
def test_host_buffer_step_chunked_pipeline(N):
    """rbe_step_host splits N >= 131 072 atoms into up to 4 chunks (copy/compute pipeline); every chunk
    adds to the same per-CTA rows in stream order, so the result is the oracle's to the usual
    tolerances and bitwise reproducible run to run (the fp32 partial sums group the atoms differently
    from the one-launch device path, so the two agree to fp32 rounding of those, not bitwise)."""
    cfg = inputs.ions_config(300_000)
    atoms = inputs.make_atoms(cfg)[:N].copy()
    m = inputs.sample_kset(cfg.L, cfg.alpha, 64, 31)
    ctx, rho_g, F_g, U_g = gpu_step(atoms, cfg.L, cfg.alpha, m, with_energy=True)
    h_x = torch.from_numpy(atoms).pin_memory()
    outs = []
    for rep in range(2):
        h_f = torch.full((N, 4), float("nan"), dtype=torch.float32).pin_memory()
        U = ctx.rbe_step_host(h_x, m, h_f, with_energy=True, want_energy=True)
        outs.append((h_f.numpy().copy(), U))
    assert np.array_equal(outs[0][0], outs[1][0]) and outs[0][1] == outs[1][1]
    F_h, U_h = outs[0]
    S = oracle.S(cfg.L, cfg.alpha)
    rho_o = oracle.rho(atoms, cfg.L, m)
    F_o, e_o = oracle.force(atoms, cfg.L, m, S, rho_o, with_energy=True)
    assert np.linalg.norm(F_h[:, :3] - F_o) / np.linalg.norm(F_o) <= F_TOL
    assert np.linalg.norm(F_h[:, 3] - e_o) <= 2e-5 * np.linalg.norm(e_o)
    assert abs(U_h - oracle.energy(cfg.L, m, S, rho_o)) <= U_TOL * abs(U_g)
    assert abs(U_h - U_g) <= 1e-6 * abs(U_g)
    # the library's own page-locked buffers (rbe_host_alloc), as bench.py's e2e leg uses them
    a_x, a_f = rbe.rbe_host_alloc((N, 4)), rbe.rbe_host_alloc((N, 4))
    a_x[:] = atoms
    a_f[:] = np.nan
    ctx.rbe_step_host(a_x, m, a_f, with_energy=True)
    assert np.array_equal(a_f, F_h)
    # pageable host memory takes the same path (the copies are then staged by the driver)
    h_f2 = np.full((N, 4), np.nan, dtype=np.float32)
    ctx.rbe_step_host(atoms, m, h_f2, with_energy=True)
    assert np.array_equal(h_f2, F_h)


@pytest.mark.parametrize("name,weighted", [("water_3k", False), ("water_96k", False), ("ions_400", True)])
def test_kspace_virial_matches_oracle(name, weighted):
    """rbe_kspace_virial against oracle/virial.py (reading Q19): fp64 on both sides from the GPU's rho,
    so the bar is the energy's (1e-5 relative to the largest component)."""
    from oracle import virial
    if weighted:
        L, alpha, mmax = 12.0, 0.3, 7
        cfg = inputs.ions_config(400)
        atoms = inputs.make_atoms(cfg)
        atoms[:, :3] *= np.float32(L / cfg.L)
        m = inputs.full_kgrid(mmax)
        w = np.exp(-(2 * np.pi / L) ** 2 * (m.astype(np.float64) ** 2).sum(1) / (4 * alpha))
    else:
        cfg = inputs.CONFIGS[name]
        atoms, L, alpha, w = inputs.make_atoms(cfg), cfg.L, cfg.alpha, None
        m = inputs.sample_kset(L, alpha, cfg.P, cfg.seed, 0)
    ctx = rbe.Rbe(atoms.shape[0], L, alpha, m.shape[0])
    with pytest.raises(rbe.RbeError):
        ctx.rbe_kspace_virial()
    ctx.rbe_set_kvectors(m, w)
    ctx.rbe_structure_factor(torch.from_numpy(atoms).cuda())
    W = ctx.rbe_kspace_virial()
    S = oracle.S(L, alpha)
    W_o = virial.kspace_virial(L, alpha, m, S, oracle.rho(atoms, L, m), w=w)
    assert np.abs(W - W_o).max() <= U_TOL * np.abs(W_o).max()
    assert np.array_equal(W, ctx.rbe_kspace_virial())          # fixed order: bitwise reproducible


def test_deterministic_ewald_mode_with_a_large_k_grid():
    """SURVEY.md s8(f) row 4, deterministic mode at scale: every grid vector with |m_d| <= 12 (P = 15 624:
    several k-chunks in both kernels) with weights exp(-k^2/4alpha) on BASELINE config 1 reproduces the
    full long-range force and energy of Eqs. (2.11) / (2.8), computed by oracle.ewald_full."""
    cfg = inputs.CONFIGS["water_3k"]
    atoms = inputs.make_atoms(cfg)
    mmax = 12                                             # exp(-k^2/4alpha) < 3e-8 beyond it at L = 31 A
    m = inputs.full_kgrid(mmax)
    k2 = (2 * np.pi / cfg.L) ** 2 * (m.astype(np.float64) ** 2).sum(1)
    w = np.exp(-k2 / (4 * cfg.alpha))
    ctx, rho, F, U = gpu_step(atoms, cfg.L, cfg.alpha, m, w=w, with_energy=True)
    Uref, _, Fl = oracle.ewald_full(atoms[:, :3].astype(np.float64), atoms[:, 3].astype(np.float64),
                                    cfg.L, cfg.alpha, nreal=0, mmax=mmax)
    assert np.linalg.norm(F[:, :3] - Fl) / np.linalg.norm(Fl) <= F_TOL
    assert abs(U - Uref[1]) <= U_TOL * abs(Uref[1])
    assert abs(F[:, 3].astype(np.float64).sum() - Uref[1]) <= 1e-4 * abs(Uref[1])


@pytest.mark.parametrize("N", [3000, 300_000])
def test_compact_host_step_matches_the_float4_host_step(N):
    """rbe_step_host_xyz (positions in, force vectors out, charges resident on the device) runs the same
    kernels over the same chunks as rbe_step_host: bitwise the same forces and energy."""
    cfg = inputs.ions_config(300_000)
    atoms = inputs.make_atoms(cfg)[:N].copy()
    m = inputs.sample_kset(cfg.L, cfg.alpha, 64, 41)
    ctx = rbe.Rbe(N, cfg.L, cfg.alpha, 64)
    h_x, h_f = rbe.rbe_host_alloc((N, 4)), rbe.rbe_host_alloc((N, 4))
    h_x[:] = atoms
    U4 = ctx.rbe_step_host(h_x, m, h_f, want_energy=True)
    h_x3, h_f3 = rbe.rbe_host_alloc((N, 3)), rbe.rbe_host_alloc((N, 3))
    h_x3[:] = atoms[:, :3]
    h_f3[:] = np.nan
    with pytest.raises(rbe.RbeError) as e:
        ctx.rbe_step_host_xyz(h_x3, m, h_f3)
    assert e.value.status == 3                                   # charges not registered yet
    ctx.rbe_set_charges(torch.from_numpy(atoms[:, 3].copy()).cuda())
    U3 = ctx.rbe_step_host_xyz(h_x3, m, h_f3, want_energy=True)
    assert np.array_equal(h_f3, h_f[:, :3]) and U3 == U4


def test_contexts_of_different_sizes_coexist():
    """Found by a randomised sweep: the dynamic-shared-memory limit is an attribute of the kernel FUNCTION; a
    small context created after a large one must not lower it under the large one's launches."""
    big_cfg, small_cfg = inputs.CONFIGS["water_96k"], inputs.CONFIGS["water_3k"]
    big_atoms, small_atoms = inputs.make_atoms(big_cfg), inputs.make_atoms(small_cfg)
    big = rbe.Rbe(big_cfg.N, big_cfg.L, big_cfg.alpha, big_cfg.P)
    small = rbe.Rbe(64, small_cfg.L, small_cfg.alpha, 3)                # created second: tiny tile, tiny k-table
    xb, xs = torch.from_numpy(big_atoms).cuda(), torch.from_numpy(small_atoms[:64].copy()).cuda()
    Fb, Fs = torch.empty_like(xb), torch.empty_like(xs)
    mb = inputs.sample_kset(big_cfg.L, big_cfg.alpha, big_cfg.P, 1, 0)
    ms = inputs.sample_kset(small_cfg.L, small_cfg.alpha, 3, 1, 0)
    for _ in range(2):                                                   # alternate the two contexts
        small.rbe_set_kvectors(ms); small.rbe_structure_factor(xs); small.rbe_forces(xs, Fs)
        big.rbe_set_kvectors(mb); big.rbe_structure_factor(xb); big.rbe_forces(xb, Fb)
    S = oracle.S(big_cfg.L, big_cfg.alpha)
    F_o = oracle.force(big_atoms, big_cfg.L, mb, S, oracle.rho(big_atoms, big_cfg.L, mb))
    assert np.linalg.norm(Fb.cpu().numpy()[:, :3] - F_o) / np.linalg.norm(F_o) <= F_TOL
