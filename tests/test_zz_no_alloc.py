"""rbe_step_static: the k-space step for callers that cannot allocate device memory.

Who needs it: a force routine loaded as a plug-in into an MD engine (or any program) whose own memory pool has
already taken the GPU's memory -- it is handed the position and force arrays and may not cudaMalloc a workspace
beside them -- and code inside a time-step loop that cannot accept the device-wide stall a cudaMalloc / cudaFree
causes.  The regular rbe_step wants a caller-allocated workspace (rbe_set_workspace); rbe_step_static keeps the
same scratch in a fixed 1.5 MiB array built into librbe.so instead, for P <= 512 (include/rbe.h).

What is checked here: its forces, per-atom energies and structure factors against the EXISTING path (rbe_step with
a workspace) on the same inputs, within the tolerances the parity tests use (tests/test_gpu_parity.py) -- on two
calls in a row, because the array is shared and keeps what the previous call left behind (the second call must not
be disturbed by the first, also when the two use different grid sizes).  Both paths launch the same kernel with the
same geometry, so the results are in fact expected to be bit-identical; that is asserted too.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It passes alone in a fresh process (the first call on the device then does the one-time set-up) and
after the other tests.
"""
import numpy as np
import pytest

from paper_2407_09315_b200 import inputs, rbe

RHO_TOL, F_TOL = 1e-6, 2e-5   # as tests/test_gpu_parity.py (reading Q15)


def _case(N, P, seed):
    """Seeded synthetic ions at the BASELINE density: float32 [N,4] atoms, box side, alpha.  Odd N: the even system
    one atom larger with its last atom dropped (neutrality does not matter when two GPU paths are compared)."""
    cfg = inputs.ions_config(N + (N & 1), P)
    atoms = np.ascontiguousarray(inputs.make_atoms(cfg)[:N])
    assert atoms.shape == (N, 4)
    return atoms, cfg.L, cfg.alpha, seed


def _compare(got_F, got_rho, ref_F, ref_rho, qsum, with_energy):
    assert np.isfinite(got_F).all() and np.isfinite(got_rho).all()
    assert np.abs(got_rho - ref_rho).max() <= RHO_TOL * qsum
    d = got_F[:, :3].astype(np.float64) - ref_F[:, :3].astype(np.float64)
    assert np.linalg.norm(d) <= F_TOL * np.linalg.norm(ref_F[:, :3].astype(np.float64))
    if with_energy:
        e_ref = ref_F[:, 3].astype(np.float64)
        assert np.linalg.norm(got_F[:, 3].astype(np.float64) - e_ref) <= 2e-5 * np.linalg.norm(e_ref) + 1e-12
    else:
        assert np.all(got_F[:, 3] == 0.0)
    # same kernel, same launch geometry, same summation order: nothing may differ at all
    assert np.array_equal(got_rho, ref_rho)
    assert np.array_equal(got_F, ref_F)


@pytest.mark.gpu
@pytest.mark.parametrize("N,P,with_energy", [(3000, 100, False), (96000, 100, True), (1237, 37, False),
                                             (999_999, 200, False), (50_001, 512, True)])
def test_two_calls_in_a_row_match_the_workspace_path(N, P, with_energy):
    import torch
    atoms, L, alpha, seed = _case(N, P, 11)
    m1 = inputs.sample_kset(L, alpha, P, seed, 0)
    m2 = inputs.sample_kset(L, alpha, P, seed, 1)
    qsum = float(np.abs(atoms[:, 3].astype(np.float64)).sum())
    xyzq = torch.from_numpy(atoms).cuda()

    # the existing path: a context with a caller-allocated workspace
    ref = rbe.Rbe(N, L, alpha, P)
    ref_out = []
    for m in (m1, m2):
        F = torch.full((N, 4), float("nan"), dtype=torch.float32, device="cuda")
        rho = torch.full((P, 2), float("nan"), dtype=torch.float64, device="cuda")
        ref.rbe_step(m, xyzq, F, with_energy=with_energy, rho=rho)
        torch.cuda.synchronize()
        ref_out.append((F.cpu().numpy(), rho.cpu().numpy()))
    assert not np.array_equal(ref_out[0][0], ref_out[1][0])   # the two batches really differ

    # the new entry point: a context that never gets a workspace; outputs prefilled with NaN
    ctx = rbe.Rbe(N, L, alpha, P, allocate=False)
    Fs = [torch.full((N, 4), float("nan"), dtype=torch.float32, device="cuda") for _ in range(2)]
    rhos = [torch.full((P, 2), float("nan"), dtype=torch.float64, device="cuda") for _ in range(2)]
    ctx.rbe_step_static(m1, xyzq, Fs[0], with_energy=with_energy, rho=rhos[0])   # (first call on the device: set-up)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    # two calls back to back on one stream, no synchronisation between them: the second starts from whatever
    # the first left in the shared array
    ctx.rbe_step_static(m1, xyzq, Fs[0], with_energy=with_energy, rho=rhos[0])
    ctx.rbe_step_static(m2, xyzq, Fs[1], with_energy=with_energy, rho=rhos[1])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before   # the calls took no device memory
    for k in range(2):
        _compare(Fs[k].cpu().numpy(), rhos[k].cpu().numpy(), ref_out[k][0], ref_out[k][1], qsum, with_energy)
    # the context still has no workspace, and the static step did not pretend otherwise
    with pytest.raises(rbe.RbeError) as ei:
        ctx.rbe_kspace_energy()
    assert ei.value.status == 3   # RBE_ERR_NOT_READY


@pytest.mark.gpu
def test_alternating_sizes_share_the_array():
    """Contexts of different sizes (different grids, different P) take turns on the one array, without a
    synchronisation in between: every call must clear what has to start from zero (the barrier counter) itself."""
    import torch
    cases = [_case(700, 64, 3), _case(96000, 200, 4), _case(5000, 512, 5)]
    work = []
    for atoms, L, alpha, seed in cases:
        N = atoms.shape[0]
        P = {700: 64, 96000: 200, 5000: 512}[N]
        m = inputs.sample_kset(L, alpha, P, seed, 0)
        xyzq = torch.from_numpy(atoms).cuda()
        ref = rbe.Rbe(N, L, alpha, P)
        F_ref = torch.empty((N, 4), dtype=torch.float32, device="cuda")
        rho_ref = torch.empty((P, 2), dtype=torch.float64, device="cuda")
        ref.rbe_step(m, xyzq, F_ref, rho=rho_ref)
        torch.cuda.synchronize()
        work.append(dict(ctx=rbe.Rbe(N, L, alpha, P, allocate=False), m=m, xyzq=xyzq, N=N, P=P,
                         qsum=float(np.abs(atoms[:, 3].astype(np.float64)).sum()),
                         F_ref=F_ref.cpu().numpy(), rho_ref=rho_ref.cpu().numpy(), out=[]))
    for rnd in range(3):
        for w in work:
            F = torch.full((w["N"], 4), float("nan"), dtype=torch.float32, device="cuda")
            rho = torch.full((w["P"], 2), float("nan"), dtype=torch.float64, device="cuda")
            w["ctx"].rbe_step_static(w["m"], w["xyzq"], F, rho=rho)
            w["out"].append((F, rho))
    torch.cuda.synchronize()
    for w in work:
        for F, rho in w["out"]:
            _compare(F.cpu().numpy(), rho.cpu().numpy(), w["F_ref"], w["rho_ref"], w["qsum"], False)


def test_sizes_beyond_the_array_are_refused_with_a_clear_error():
    """P above RBE_STATIC_MAX_P = 512 does not fit the built-in array: refused before any CUDA call (so this runs
    without a GPU), with a message that names the limit.  Bad wavevectors and a missing k-set are refused too."""
    import ctypes
    L = rbe.lib()
    h = ctypes.c_void_p()
    assert L.rbe_create(ctypes.byref(h), 1000, 21.5, 0.09, 513) == 0
    m = np.ones((513, 3), dtype=np.int32)
    dummy = ctypes.c_void_p(4096)   # never dereferenced: the size check comes first
    st = L.rbe_step_static(h, ctypes.c_void_p(m.ctypes.data), dummy, dummy, 0, None, None)
    assert st == 4   # RBE_ERR_WORKSPACE
    msg = L.rbe_last_error(h).decode()
    assert "512" in msg and "513" in msg and "rbe_step_static" in msg
    L.rbe_destroy(h)

    h = ctypes.c_void_p()
    assert L.rbe_create(ctypes.byref(h), 1000, 21.5, 0.09, 4) == 0
    assert L.rbe_step_static(h, None, dummy, dummy, 0, None, None) == 1          # no wavevectors: RBE_ERR_INVALID_ARG
    m = np.ones((4, 3), dtype=np.int32)
    assert L.rbe_step_static(h, ctypes.c_void_p(m.ctypes.data), ctypes.c_void_p(4100), dummy, 0, None, None) == 1   # misaligned
    m[2] = 0
    assert L.rbe_step_static(h, ctypes.c_void_p(m.ctypes.data), dummy, dummy, 0, None, None) == 2   # RBE_ERR_BAD_KVECTOR
    L.rbe_destroy(h)
