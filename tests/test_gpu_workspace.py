"""rbe_set_workspace refuses a buffer that another live context holds (include/rbe.h): a workspace carries state from
launch to launch -- the k-set, rho, the sampler's step counter, the arrival counter of the one-launch step's grid
barrier -- so two contexts on one buffer corrupt each other or leave a barrier waiting.  No sanitizer can be run on this
pool to catch such a caller, hence the check in the library."""
import numpy as np
import pytest
import torch

from paper_2407_09315_b200 import inputs, rbe

pytestmark = pytest.mark.gpu


def test_a_workspace_belongs_to_one_live_context():
    L, alpha, P, N = 40.0, 0.09, 64, 5000
    a = rbe.Rbe(N, L, alpha, P, allocate=False)
    b = rbe.Rbe(N, L, alpha, P, allocate=False)
    n = a.rbe_workspace_bytes()
    assert n == b.rbe_workspace_bytes() and n % 256 == 0
    buf = torch.empty(3 * n, dtype=torch.uint8, device="cuda")
    a.rbe_set_workspace(buf[:n])
    for clash in (buf[:n], buf[n - 256:2 * n - 256], buf):          # the same bytes, a partial overlap, a superset
        with pytest.raises(rbe.RbeError) as ei:
            b.rbe_set_workspace(clash)
        assert ei.value.status == 4 and "another live context" in str(ei.value)       # RBE_ERR_WORKSPACE
    b.rbe_set_workspace(buf[n:2 * n])                                # carved from the same allocation, disjoint: fine
    a.rbe_set_workspace(buf[:n])                                     # a context may be given its own buffer again
    a.rbe_set_workspace(buf[2 * n:])                                 # moving on frees the old claim ...
    c = rbe.Rbe(N, L, alpha, P, allocate=False)
    c.rbe_set_workspace(buf[:n])                                     # ... for somebody else
    c.close()
    b.close()                                                        # and so does rbe_destroy
    d = rbe.Rbe(N, L, alpha, P, allocate=False)
    d.rbe_set_workspace(buf[:2 * n])

    # the three survivors still compute: one step each on disjoint workspaces, identical results
    atoms = inputs.make_atoms(inputs.ions_config(N, P))
    atoms[:, :3] *= np.float32(L / inputs.ion_box(N))
    m = inputs.sample_kset(L, alpha, P, 5, 0)
    x = torch.from_numpy(atoms).cuda()
    out = []
    for ctx in (a, d):
        f = torch.empty((N, 4), dtype=torch.float32, device="cuda")
        ctx.rbe_step(m, x, f)
        out.append(f)
    torch.cuda.synchronize()
    assert torch.equal(out[0], out[1]) and torch.isfinite(out[0]).all()
