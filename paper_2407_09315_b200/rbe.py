"""ctypes binding of librbe (include/rbe.h): argument marshalling only.

Same names as the C ABI.  torch supplies device memory and the CUDA stream; every step of
the path runs in the library's own kernels.  There is no CPU fallback: if librbe.so is
missing, or there is no sm_100 device, the calls raise.
"""
from __future__ import annotations

import ctypes
import os

HERE = os.path.dirname(os.path.abspath(__file__))
SO_PATH = os.path.join(HERE, "librbe.so")

RBE_OK = 0
STATUS_NAMES = {
    0: "RBE_OK", 1: "RBE_ERR_INVALID_ARG", 2: "RBE_ERR_BAD_KVECTOR", 3: "RBE_ERR_NOT_READY",
    4: "RBE_ERR_WORKSPACE", 5: "RBE_ERR_CUDA", 6: "RBE_ERR_NO_DEVICE",
}


class RbeError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {msg}")
        self.status = status


class LaunchInfo(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in (
        "num_sms", "sf_grid_x", "sf_grid_y", "sf_threads", "sf_smem_bytes", "sf_k_per_thread",
        "sf_atom_groups", "sf_tile_atoms", "sf_red_group", "sf_red_groups", "f_grid", "f_threads",
        "f_smem_bytes", "f_atoms_per_thread", "step_fused", "step_smem_bytes")]

    def as_dict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_}


_lib = None


def lib():
    """Load librbe.so (built in-tree by build.py).  Fails loudly if it is not there."""
    global _lib
    if _lib is None:
        if not os.path.exists(SO_PATH):
            raise ImportError(
                f"{SO_PATH} not found: build it with `python -m paper_2407_09315_b200.build` "
                "(or __graft_entry__.build()); there is no fallback path")
        L = ctypes.CDLL(SO_PATH)
        vp, i32, i64, dbl, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_double, ctypes.c_size_t
        L.rbe_create.restype = ctypes.c_int
        L.rbe_create.argtypes = [ctypes.POINTER(vp), i64, dbl, dbl, i32]
        L.rbe_destroy.restype = ctypes.c_int
        L.rbe_destroy.argtypes = [vp]
        L.rbe_normaliser_S.restype = dbl
        L.rbe_normaliser_S.argtypes = [vp]
        L.rbe_workspace_bytes.restype = sz
        L.rbe_workspace_bytes.argtypes = [vp]
        L.rbe_set_workspace.restype = ctypes.c_int
        L.rbe_set_workspace.argtypes = [vp, vp, sz]
        L.rbe_set_pairing.restype = ctypes.c_int
        L.rbe_set_pairing.argtypes = [vp, i32]
        L.rbe_set_pair_table.restype = ctypes.c_int
        L.rbe_set_pair_table.argtypes = [vp, i32]
        L.rbe_set_pair_kernel.restype = ctypes.c_int
        L.rbe_set_pair_kernel.argtypes = [vp, i32]
        L.rbe_pair_table_host.restype = ctypes.c_int
        L.rbe_pair_table_host.argtypes = [vp, dbl, vp, vp, i32, ctypes.POINTER(i32)]
        L.rbe_get_launch_info.restype = ctypes.c_int
        L.rbe_get_launch_info.argtypes = [vp, ctypes.POINTER(LaunchInfo)]
        L.rbe_set_kvectors.restype = ctypes.c_int
        L.rbe_set_kvectors.argtypes = [vp, vp, vp, vp]
        u64 = ctypes.c_uint64
        L.rbe_sample_kvectors.restype = ctypes.c_int
        L.rbe_sample_kvectors.argtypes = [vp, u64, u64, vp]
        L.rbe_get_kvectors.restype = ctypes.c_int
        L.rbe_get_kvectors.argtypes = [vp, vp, vp]
        L.rbe_graph_capture.restype = ctypes.c_int
        L.rbe_graph_capture.argtypes = [vp, vp, vp, i32, u64, u64]
        L.rbe_graph_launch.restype = ctypes.c_int
        L.rbe_graph_launch.argtypes = [vp, vp]
        L.rbe_exchange_bytes.restype = sz
        L.rbe_exchange_bytes.argtypes = [vp, i32]
        L.rbe_set_exchange.restype = ctypes.c_int
        L.rbe_set_exchange.argtypes = [vp, i32, i32, ctypes.POINTER(vp), sz]
        L.rbe_exchange_check.restype = ctypes.c_int
        L.rbe_exchange_check.argtypes = [vp, vp]
        L.rbe_short_range_bytes.restype = sz
        L.rbe_short_range_bytes.argtypes = [vp, dbl]
        L.rbe_short_range.restype = ctypes.c_int
        L.rbe_short_range.argtypes = [vp, vp, dbl, vp, i32, i32, vp, sz, vp]
        L.rbe_rbl_bytes.restype = sz
        L.rbe_rbl_bytes.argtypes = [vp, dbl, dbl]
        L.rbe_rbl_forces.restype = ctypes.c_int
        L.rbe_rbl_forces.argtypes = [vp, vp, dbl, dbl, i32, ctypes.c_uint64, ctypes.c_uint64, vp, i32, vp, sz, vp]
        L.rbe_structure_factor.restype = ctypes.c_int
        L.rbe_structure_factor.argtypes = [vp, vp, vp, vp]
        L.rbe_set_rho.restype = ctypes.c_int
        L.rbe_set_rho.argtypes = [vp, vp, vp]
        L.rbe_forces.restype = ctypes.c_int
        L.rbe_forces.argtypes = [vp, vp, vp, i32, vp]
        L.rbe_step.restype = ctypes.c_int
        L.rbe_step.argtypes = [vp, vp, vp, vp, vp, i32, vp, vp]
        L.rbe_step_static.restype = ctypes.c_int
        L.rbe_step_static.argtypes = [vp, vp, vp, vp, i32, vp, vp]
        L.rbe_step_host_bytes.restype = sz
        L.rbe_step_host_bytes.argtypes = [vp, i32]
        L.rbe_probe_pipe_rates.restype = ctypes.c_int
        L.rbe_probe_pipe_rates.argtypes = [vp, vp, vp]
        L.rbe_nve_kick.restype = ctypes.c_int
        L.rbe_nve_kick.argtypes = [vp, vp, vp, vp, dbl, vp, vp, dbl, vp]
        L.rbe_nve_energies.restype = ctypes.c_int
        L.rbe_nve_energies.argtypes = [vp, vp, vp, vp, vp, vp]
        L.rbe_md_capture.restype = ctypes.c_int
        L.rbe_md_capture.argtypes = [vp, vp, vp, vp, vp, vp, dbl, dbl, vp, sz, i32, ctypes.c_uint64, ctypes.c_uint64, i32]
        L.rbe_kspace_energy.restype = ctypes.c_int
        L.rbe_kspace_energy.argtypes = [vp, ctypes.POINTER(dbl), vp]
        L.rbe_kspace_virial.restype = ctypes.c_int
        L.rbe_kspace_virial.argtypes = [vp, vp, vp]
        L.rbe_set_charges.restype = ctypes.c_int
        L.rbe_set_charges.argtypes = [vp, vp]
        L.rbe_step_host_xyz.restype = ctypes.c_int
        L.rbe_step_host_xyz.argtypes = [vp, vp, vp, vp, vp, ctypes.POINTER(dbl), vp, sz, vp]
        L.rbe_step_host.restype = ctypes.c_int
        L.rbe_step_host.argtypes = [vp, vp, vp, vp, vp, i32, ctypes.POINTER(dbl), vp, sz, vp]
        L.rbe_host_alloc.restype = ctypes.c_int
        L.rbe_host_alloc.argtypes = [ctypes.POINTER(vp), sz]
        L.rbe_host_free.restype = ctypes.c_int
        L.rbe_host_free.argtypes = [vp]
        L.rbe_last_error.restype = ctypes.c_char_p
        L.rbe_last_error.argtypes = [vp]
        L.rbe_status_string.restype = ctypes.c_char_p
        L.rbe_status_string.argtypes = [ctypes.c_int]
        L.rbe_version.restype = i32
        _lib = L
    return _lib


class _HostBlock:
    """Owner of one rbe_host_alloc block: freed when the last numpy view of it is gone."""

    def __init__(self, nbytes):
        self.ptr = ctypes.c_void_p()
        st = lib().rbe_host_alloc(ctypes.byref(self.ptr), nbytes)
        if st != RBE_OK:
            raise RbeError(st, "rbe_host_alloc failed")

    def __del__(self):
        if getattr(self, "ptr", None) is not None and self.ptr.value and _lib is not None:
            _lib.rbe_host_free(self.ptr)
            self.ptr = ctypes.c_void_p()


def rbe_host_alloc(shape, dtype="float32"):
    """numpy array in page-locked host memory from the library's rbe_host_alloc (cudaHostAlloc): the
    buffers to hand to rbe_step_host.  Freed (rbe_host_free) when the array and its views are gone."""
    import numpy as np
    dt = np.dtype(dtype)
    count = int(np.prod(shape))
    nbytes = max(count * dt.itemsize, 1)
    blk = _HostBlock(nbytes)
    buf = (ctypes.c_ubyte * nbytes).from_address(blk.ptr.value)
    buf._rbe_owner = blk          # numpy keeps `buf` alive through .base; `buf` keeps the owner alive
    return np.frombuffer(buf, dtype=dt, count=count).reshape(shape)


def _stream_ptr(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(int(getattr(stream, "cuda_stream", stream)))


def _np_ptr(a):
    return None if a is None else ctypes.c_void_p(a.ctypes.data)


class Rbe:
    """One RBE context: N atoms on the current device, box L, alpha, batch size P."""

    def __init__(self, N: int, L: float, alpha: float, P: int, *, allocate: bool = True):
        self._h = ctypes.c_void_p()
        self.N, self.L, self.alpha, self.P = int(N), float(L), float(alpha), int(P)
        st = lib().rbe_create(ctypes.byref(self._h), self.N, self.L, self.alpha, self.P)
        if st != RBE_OK:
            self._h = ctypes.c_void_p()
            raise RbeError(st, "rbe_create: invalid argument")
        self._ws = None
        self._scratch = None
        if allocate:
            self.rbe_set_workspace()

    # ---- plumbing
    def _check(self, st):
        if st != RBE_OK:
            raise RbeError(st, lib().rbe_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value and _lib is not None:
            _lib.rbe_destroy(self._h)
            self._h = ctypes.c_void_p()

    __del__ = close

    # ---- the C ABI, same names
    def rbe_normaliser_S(self) -> float:
        return float(lib().rbe_normaliser_S(self._h))

    def rbe_workspace_bytes(self) -> int:
        n = int(lib().rbe_workspace_bytes(self._h))
        if n == 0:
            raise RbeError(6, lib().rbe_last_error(self._h).decode())
        return n

    def rbe_set_workspace(self, ws=None):
        import torch
        if ws is None:
            ws = torch.empty(self.rbe_workspace_bytes(), dtype=torch.uint8, device="cuda")
        self._check(lib().rbe_set_workspace(self._h, ctypes.c_void_p(ws.data_ptr()), ws.numel() * ws.element_size()))
        self._ws = ws  # keep alive

    def rbe_set_pairing(self, mode: int):
        self._check(lib().rbe_set_pairing(self._h, int(mode)))

    def rbe_set_pair_kernel(self, kind: int):
        self._check(lib().rbe_set_pair_kernel(self._h, int(kind)))

    def rbe_pair_table_host(self, rs: float):
        """(tf, te): float32 [n, 4] cubic coefficients of the pair-term tables, computed on the host (needs no GPU)."""
        import numpy as np
        n = ctypes.c_int32(0)
        self._check(lib().rbe_pair_table_host(self._h, float(rs), None, None, 0, ctypes.byref(n)))
        tf = np.zeros((n.value, 4), dtype=np.float32)
        te = np.zeros((n.value, 4), dtype=np.float32)
        self._check(lib().rbe_pair_table_host(self._h, float(rs), ctypes.c_void_p(tf.ctypes.data), ctypes.c_void_p(te.ctypes.data),
                                              n.value, ctypes.byref(n)))
        return tf, te

    def rbe_set_pair_table(self, on: bool):
        self._check(lib().rbe_set_pair_table(self._h, int(bool(on))))

    def rbe_get_launch_info(self) -> dict:
        li = LaunchInfo()
        self._check(lib().rbe_get_launch_info(self._h, ctypes.byref(li)))
        return li.as_dict()

    def rbe_set_kvectors(self, m, w=None, stream=None):
        """m: numpy int32 [P,3] (host); w: numpy float64 [P] (host) or None."""
        import numpy as np
        mm = np.ascontiguousarray(m, dtype=np.int32)
        assert mm.shape == (self.P, 3), mm.shape
        ww = None if w is None else np.ascontiguousarray(w, dtype=np.float64)
        assert ww is None or ww.shape == (self.P,)
        self._check(lib().rbe_set_kvectors(self._h, _np_ptr(mm), _np_ptr(ww), _stream_ptr(stream)))

    def rbe_sample_kvectors(self, seed: int, step: int, stream=None):
        self._check(lib().rbe_sample_kvectors(self._h, int(seed), int(step), _stream_ptr(stream)))

    def rbe_get_kvectors(self, stream=None):
        """numpy int32 [P,3]: the current k-set (synchronises)."""
        import numpy as np
        m = np.empty((self.P, 3), dtype=np.int32)
        self._check(lib().rbe_get_kvectors(self._h, _np_ptr(m), _stream_ptr(stream)))
        return m

    def rbe_graph_capture(self, xyzq, force, with_energy: bool, seed: int, first_step: int):
        _check_tensor(xyzq, (self.N, 4), "float32")
        _check_tensor(force, (self.N, 4), "float32")
        self._graph_buffers = (xyzq, force)   # the graph is bound to these: keep them alive
        self._check(lib().rbe_graph_capture(self._h, ctypes.c_void_p(xyzq.data_ptr()), ctypes.c_void_p(force.data_ptr()),
                                            int(bool(with_energy)), int(seed), int(first_step)))

    def rbe_graph_launch(self, stream=None):
        self._check(lib().rbe_graph_launch(self._h, _stream_ptr(stream)))

    def rbe_exchange_bytes(self, world: int) -> int:
        return int(lib().rbe_exchange_bytes(self._h, int(world)))

    def rbe_set_exchange(self, rank: int, world: int, buf_ptrs, nbytes: int, keep_alive=None):
        """buf_ptrs: `world` device pointers (ints), buf_ptrs[r] = rank r's exchange buffer as mapped
        in this process; None switches the exchange off."""
        if buf_ptrs is None:
            self._check(lib().rbe_set_exchange(self._h, 0, 0, None, 0))
            self._xch_keep = None
            return
        arr = (ctypes.c_void_p * int(world))(*[int(p) for p in buf_ptrs])
        self._check(lib().rbe_set_exchange(self._h, int(rank), int(world), arr, int(nbytes)))
        self._xch_keep = keep_alive

    def rbe_exchange_check(self, stream=None):
        self._check(lib().rbe_exchange_check(self._h, _stream_ptr(stream)))

    def rbe_structure_factor(self, xyzq, rho=None, stream=None):
        """xyzq: cuda float32 [N,4]; rho: cuda float64 [P,2] or None."""
        _check_tensor(xyzq, (self.N, 4), "float32")
        if rho is not None:
            _check_tensor(rho, (self.P, 2), "float64")
        self._check(lib().rbe_structure_factor(
            self._h, ctypes.c_void_p(xyzq.data_ptr()),
            None if rho is None else ctypes.c_void_p(rho.data_ptr()), _stream_ptr(stream)))

    def rbe_set_rho(self, rho, stream=None):
        _check_tensor(rho, (self.P, 2), "float64")
        self._check(lib().rbe_set_rho(self._h, ctypes.c_void_p(rho.data_ptr()), _stream_ptr(stream)))

    def rbe_forces(self, xyzq, force, with_energy: bool = False, stream=None):
        """xyzq, force: cuda float32 [N,4]."""
        _check_tensor(xyzq, (self.N, 4), "float32")
        _check_tensor(force, (self.N, 4), "float32")
        self._check(lib().rbe_forces(self._h, ctypes.c_void_p(xyzq.data_ptr()),
                                     ctypes.c_void_p(force.data_ptr()), int(bool(with_energy)),
                                     _stream_ptr(stream)))

    def rbe_step(self, m, xyzq, force, w=None, with_energy: bool = False, rho=None, stream=None):
        """Algorithm 1 steps 2-4 in one cooperative launch.  m: numpy int32 [P,3] (host) or None (keep the
        k-set on the device); xyzq, force: cuda float32 [N,4]; rho: cuda float64 [P,2] or None."""
        import numpy as np
        _check_tensor(xyzq, (self.N, 4), "float32")
        _check_tensor(force, (self.N, 4), "float32")
        if rho is not None:
            _check_tensor(rho, (self.P, 2), "float64")
        mm = None if m is None else np.ascontiguousarray(m, dtype=np.int32)
        assert mm is None or mm.shape == (self.P, 3), mm.shape
        ww = None if w is None else np.ascontiguousarray(w, dtype=np.float64)
        assert ww is None or ww.shape == (self.P,)
        self._check(lib().rbe_step(self._h, _np_ptr(mm), _np_ptr(ww), ctypes.c_void_p(xyzq.data_ptr()),
                                   ctypes.c_void_p(force.data_ptr()), int(bool(with_energy)),
                                   None if rho is None else ctypes.c_void_p(rho.data_ptr()), _stream_ptr(stream)))

    def rbe_step_static(self, m, xyzq, force, with_energy: bool = False, rho=None, stream=None):
        """rbe_step for callers that cannot allocate device memory (a plug-in inside a program whose pool owns the
        GPU's memory; a loop that cannot take cudaMalloc's device-wide stall): the kernel's scratch is an array built
        into librbe.so, so the context needs no workspace (`Rbe(..., allocate=False)` works).  m: numpy int32 [P,3]
        (host, required); xyzq, force: cuda float32 [N,4]; rho: cuda float64 [P,2] or None.  P <= 512.  One array per
        device, shared by all callers: keep calls on one stream, or order them with events.  The first call on a
        device does a one-time set-up and should be made outside stream capture.  See include/rbe.h."""
        import numpy as np
        _check_tensor(xyzq, (self.N, 4), "float32")
        _check_tensor(force, (self.N, 4), "float32")
        if rho is not None:
            _check_tensor(rho, (self.P, 2), "float64")
        mm = np.ascontiguousarray(m, dtype=np.int32)
        assert mm.shape == (self.P, 3), mm.shape
        self._check(lib().rbe_step_static(self._h, _np_ptr(mm), ctypes.c_void_p(xyzq.data_ptr()),
                                          ctypes.c_void_p(force.data_ptr()), int(bool(with_energy)),
                                          None if rho is None else ctypes.c_void_p(rho.data_ptr()), _stream_ptr(stream)))

    def rbe_step_bound(self, xyzq, force, with_energy: bool = False, rho=None, stream=None):
        """rbe_step with everything but the k-set marshalled ONCE: returns call(m) for m a C-contiguous numpy int32
        [P,3] array.  For loops whose per-step host cost matters (small systems are launch-bound): the call is one
        ctypes transition, no tensor checks."""
        import numpy as np
        _check_tensor(xyzq, (self.N, 4), "float32")
        _check_tensor(force, (self.N, 4), "float32")
        if rho is not None:
            _check_tensor(rho, (self.P, 2), "float64")
        fn, h, st = lib().rbe_step, self._h, _stream_ptr(stream)
        px, pf = ctypes.c_void_p(xyzq.data_ptr()), ctypes.c_void_p(force.data_ptr())
        pr = None if rho is None else ctypes.c_void_p(rho.data_ptr())
        we, shape = int(bool(with_energy)), (self.P, 3)
        keep = (xyzq, force, rho)

        def call(m):
            assert m.dtype == np.int32 and m.shape == shape and m.flags["C_CONTIGUOUS"] and keep is not None
            status = fn(h, m.ctypes.data, None, px, pf, we, pr, st)
            if status != RBE_OK:
                self._check(status)
        return call

    def rbe_step_host_bytes(self, compact: bool) -> int:
        return int(lib().rbe_step_host_bytes(self._h, int(bool(compact))))

    def rbe_probe_pipe_rates(self, stream=None) -> dict:
        """Measured issue rates (thread-instructions per SM per clock) and the SM clock seen (synchronises)."""
        import numpy as np
        out = np.zeros(5, dtype=np.float64)
        self._check(lib().rbe_probe_pipe_rates(self._h, _np_ptr(out), _stream_ptr(stream)))
        return {"ffma": float(out[0]), "imad": float(out[1]), "i2fp": float(out[2]), "mufu": float(out[3]),
                "sm_mhz": float(out[4])}

    def rbe_nve_kick(self, vel, inv_mass, force, half_dt: float, pos=None, xyzq=None, dt: float = 0.0, stream=None):
        """v += half_dt F / m; with pos (cuda float64 [N,3]) also x += dt v and xyzq[:, :3] = float32(x)."""
        _check_tensor(vel, (self.N, 3), "float64")
        _check_tensor(inv_mass, (self.N,), "float64")
        _check_tensor(force, (self.N, 4), "float32")
        if pos is not None:
            _check_tensor(pos, (self.N, 3), "float64")
            _check_tensor(xyzq, (self.N, 4), "float32")
        self._check(lib().rbe_nve_kick(self._h, ctypes.c_void_p(vel.data_ptr()), ctypes.c_void_p(inv_mass.data_ptr()),
                                       ctypes.c_void_p(force.data_ptr()), float(half_dt),
                                       None if pos is None else ctypes.c_void_p(pos.data_ptr()),
                                       None if pos is None else ctypes.c_void_p(xyzq.data_ptr()), float(dt), _stream_ptr(stream)))

    def rbe_nve_energies(self, vel=None, inv_mass=None, force=None, stream=None):
        """(kinetic energy, sum of force[:, 3]) in fp64, fixed order (synchronises)."""
        import numpy as np
        out = np.zeros(2, dtype=np.float64)
        self._check(lib().rbe_nve_energies(self._h, None if vel is None else ctypes.c_void_p(vel.data_ptr()),
                                           None if inv_mass is None else ctypes.c_void_p(inv_mass.data_ptr()),
                                           None if force is None else ctypes.c_void_p(force.data_ptr()), _np_ptr(out),
                                           _stream_ptr(stream)))
        return float(out[0]), float(out[1])

    def rbe_md_capture(self, pos, vel, inv_mass, xyzq, force, rs: float, dt: float, sampled: bool, seed: int = 0,
                       first_step: int = 0, with_energy: bool = False):
        import torch
        _check_tensor(pos, (self.N, 3), "float64")
        _check_tensor(vel, (self.N, 3), "float64")
        _check_tensor(inv_mass, (self.N,), "float64")
        _check_tensor(xyzq, (self.N, 4), "float32")
        _check_tensor(force, (self.N, 4), "float32")
        n = self.rbe_short_range_bytes(rs)
        if n == 0:
            raise RbeError(1, "rbe_md_capture: need 0 < r_s <= L/3")
        # The graph records the ADDRESS of its short-range scratch, so it gets a tensor of its own, kept alive beside
        # the other arrays the graph is bound to and never rebound: rbe_short_range / rbe_rbl_forces may replace the
        # shared self._sr_ws by a larger one at any time (the RBL cell list can need more bytes), which would leave a
        # graph that used it replaying into freed memory.
        graph_sr_ws = torch.empty(n, dtype=torch.uint8, device="cuda")
        self._check(lib().rbe_md_capture(self._h, ctypes.c_void_p(pos.data_ptr()), ctypes.c_void_p(vel.data_ptr()),
                                         ctypes.c_void_p(inv_mass.data_ptr()), ctypes.c_void_p(xyzq.data_ptr()),
                                         ctypes.c_void_p(force.data_ptr()), float(rs), float(dt),
                                         ctypes.c_void_p(graph_sr_ws.data_ptr()), graph_sr_ws.numel(), int(bool(sampled)),
                                         int(seed), int(first_step), int(bool(with_energy))))
        self._graph_buffers = (pos, vel, inv_mass, xyzq, force, graph_sr_ws)   # replaced only after the new graph exists

    def rbe_short_range_bytes(self, rs: float) -> int:
        return int(lib().rbe_short_range_bytes(self._h, float(rs)))

    def rbe_short_range(self, xyzq, rs: float, force, accumulate: bool = False, with_energy: bool = False, stream=None):
        """Real-space partner (Eq. 2.10 truncated at rs).  xyzq, force: cuda float32 [N,4]."""
        import torch
        _check_tensor(xyzq, (self.N, 4), "float32")
        _check_tensor(force, (self.N, 4), "float32")
        n = self.rbe_short_range_bytes(rs)
        if n == 0:
            raise RbeError(1, "rbe_short_range: need 0 < r_s <= L/3")
        if getattr(self, "_sr_ws", None) is None or self._sr_ws.numel() < n:
            self._sr_ws = torch.empty(n, dtype=torch.uint8, device="cuda")
        self._check(lib().rbe_short_range(self._h, ctypes.c_void_p(xyzq.data_ptr()), float(rs),
                                          ctypes.c_void_p(force.data_ptr()), int(bool(accumulate)), int(bool(with_energy)),
                                          ctypes.c_void_p(self._sr_ws.data_ptr()), self._sr_ws.numel(), _stream_ptr(stream)))

    def rbe_rbl_bytes(self, rc: float, rs: float) -> int:
        return int(lib().rbe_rbl_bytes(self._h, float(rc), float(rs)))

    def rbe_rbl_forces(self, xyzq, rc: float, rs: float, p: int, seed: int, step: int, force, accumulate: bool = False, stream=None):
        """Random batch list estimate of the short-range force (Eqs. 2.13-2.16).  xyzq, force: cuda float32 [N,4]."""
        import torch
        _check_tensor(xyzq, (self.N, 4), "float32")
        _check_tensor(force, (self.N, 4), "float32")
        n = self.rbe_rbl_bytes(rc, rs)
        if n == 0:
            raise RbeError(1, "rbe_rbl_forces: need 0 < r_c < r_s <= L/3")
        if getattr(self, "_sr_ws", None) is None or self._sr_ws.numel() < n:
            self._sr_ws = torch.empty(n, dtype=torch.uint8, device="cuda")
        self._check(lib().rbe_rbl_forces(self._h, ctypes.c_void_p(xyzq.data_ptr()), float(rc), float(rs), int(p), int(seed),
                                         int(step), ctypes.c_void_p(force.data_ptr()), int(bool(accumulate)),
                                         ctypes.c_void_p(self._sr_ws.data_ptr()), self._sr_ws.numel(), _stream_ptr(stream)))

    def rbe_kspace_energy(self, stream=None) -> float:
        u = ctypes.c_double(0.0)
        self._check(lib().rbe_kspace_energy(self._h, ctypes.byref(u), _stream_ptr(stream)))
        return float(u.value)

    def rbe_kspace_virial(self, stream=None):
        """numpy float64 [6] = W_xx, W_yy, W_zz, W_xy, W_xz, W_yz (synchronises)."""
        import numpy as np
        W = np.empty(6, dtype=np.float64)
        self._check(lib().rbe_kspace_virial(self._h, _np_ptr(W), _stream_ptr(stream)))
        return W

    def rbe_set_charges(self, q):
        """q: cuda float32 [N] (kept alive by this object) or None."""
        if q is None:
            self._check(lib().rbe_set_charges(self._h, None))
        else:
            _check_tensor(q, (self.N,), "float32")
            self._check(lib().rbe_set_charges(self._h, ctypes.c_void_p(q.data_ptr())))
        self._q = q

    def rbe_step_host_xyz(self, h_xyz, m, h_force3, w=None, want_energy=False, stream=None):
        """Compact end-to-end step: h_xyz / h_force3 are host float32 [N,3] (numpy or CPU torch)."""
        import numpy as np
        import torch
        need = self.rbe_step_host_bytes(True)
        if getattr(self, "_scratch3", None) is None or self._scratch3.numel() < need:
            self._scratch3 = torch.empty(max(1, need), dtype=torch.uint8, device="cuda")
        mm = np.ascontiguousarray(m, dtype=np.int32)
        assert mm.shape == (self.P, 3)
        ww = None if w is None else np.ascontiguousarray(w, dtype=np.float64)
        u = ctypes.c_double(0.0)
        self._check(lib().rbe_step_host_xyz(
            self._h, ctypes.c_void_p(_host_ptr3(h_xyz, self.N)), _np_ptr(mm), _np_ptr(ww),
            ctypes.c_void_p(_host_ptr3(h_force3, self.N)), ctypes.byref(u) if want_energy else None,
            ctypes.c_void_p(self._scratch3.data_ptr()), self._scratch3.numel(), _stream_ptr(stream)))
        return float(u.value) if want_energy else None

    def rbe_step_host(self, h_xyzq, m, h_force, w=None, with_energy=False, want_energy=False, stream=None):
        """End-to-end step from HOST buffers: h_xyzq / h_force are CPU float32 [N,4] torch tensors
        (pinned for asynchronous copies) or numpy arrays; m numpy int32 [P,3]."""
        import numpy as np
        import torch
        if self._scratch is None:
            self._scratch = torch.empty(max(1, self.rbe_step_host_bytes(False)), dtype=torch.uint8, device="cuda")
        mm = np.ascontiguousarray(m, dtype=np.int32)
        assert mm.shape == (self.P, 3)
        ww = None if w is None else np.ascontiguousarray(w, dtype=np.float64)
        u = ctypes.c_double(0.0)
        self._check(lib().rbe_step_host(
            self._h, ctypes.c_void_p(_host_ptr(h_xyzq, self.N)), _np_ptr(mm), _np_ptr(ww),
            ctypes.c_void_p(_host_ptr(h_force, self.N)), int(bool(with_energy)),
            ctypes.byref(u) if want_energy else None,
            ctypes.c_void_p(self._scratch.data_ptr()), self._scratch.numel(), _stream_ptr(stream)))
        return float(u.value) if want_energy else None


def _host_ptr3(a, N):
    import numpy as np
    if isinstance(a, np.ndarray):
        assert a.dtype == np.float32 and a.flags["C_CONTIGUOUS"] and a.shape == (N, 3)
        return a.ctypes.data
    assert (not a.is_cuda) and a.is_contiguous() and tuple(a.shape) == (N, 3)
    return a.data_ptr()


def _check_tensor(t, shape, dtype):
    import torch
    if not (t.is_cuda and t.is_contiguous() and tuple(t.shape) == tuple(shape) and t.dtype == getattr(torch, dtype)):
        raise ValueError(f"expected contiguous cuda {dtype} tensor of shape {shape}, got {t.dtype} {tuple(t.shape)} on {t.device}")


def _host_ptr(a, N):
    import numpy as np
    if isinstance(a, np.ndarray):
        assert a.dtype == np.float32 and a.flags["C_CONTIGUOUS"] and a.shape == (N, 4)
        return a.ctypes.data
    assert (not a.is_cuda) and a.is_contiguous() and tuple(a.shape) == (N, 4)
    return a.data_ptr()
