"""fp64 CPU oracle for the RBE k-space path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes marshalling around ``rbe_oracle.c``, ``ewald_ref.c`` and ``short_range.c`` (plain C, fp64, written
from /root/reference/PAPER.md; every function there cites the passage it follows).  No
arithmetic of the method lives in this file.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_2407_09315_b200`` and shares no code with the CUDA path.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_SRC = [os.path.join(_HERE, "rbe_oracle.c"), os.path.join(_HERE, "ewald_ref.c"), os.path.join(_HERE, "short_range.c")]
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle's C sources with gcc (-O2 -fopenmp, no fast-math)."""
    stale = force or not os.path.exists(_SO) or any(
        os.path.getmtime(s) > os.path.getmtime(_SO) for s in _SRC
    )
    if stale:
        tmp = _SO + f".tmp{os.getpid()}"
        cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c11", "-o", tmp] + _SRC + ["-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _SO)
    return _SO


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = ctypes.CDLL(build())
    c_d, c_i32, c_i64 = ctypes.c_double, ctypes.c_int32, ctypes.c_int64
    vp = ctypes.c_void_p
    lib.oracle_max_threads.restype = ctypes.c_int
    lib.oracle_set_threads.argtypes = [ctypes.c_int]
    lib.oracle_S.restype = c_d
    lib.oracle_S.argtypes = [c_d, c_d]
    lib.oracle_S_grid.restype = c_d
    lib.oracle_S_grid.argtypes = [c_d, c_d, ctypes.c_int]
    lib.oracle_rho.restype = None
    lib.oracle_rho.argtypes = [c_i64, vp, c_d, c_i32, vp, vp]
    lib.oracle_force.restype = None
    lib.oracle_force.argtypes = [c_i64, vp, c_d, c_i32, vp, vp, c_d, vp, c_i64, vp, vp, vp]
    lib.oracle_energy.restype = c_d
    lib.oracle_energy.argtypes = [c_d, c_i32, vp, vp, c_d, vp]
    lib.oracle_ewald_full.restype = None
    lib.oracle_ewald_full.argtypes = [c_i32, vp, vp, c_d, c_d, c_i32, c_i32, vp, vp, vp]
    lib.oracle_direct_image_sum.restype = None
    lib.oracle_direct_image_sum.argtypes = [c_i32, vp, vp, c_d, c_i32, vp, vp]
    lib.oracle_short_range.restype = None
    lib.oracle_short_range.argtypes = [c_i64, vp, c_d, c_d, c_d, c_i64, vp, vp, vp]
    _lib = lib
    return lib


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _xyzq(xyzq):
    a = np.ascontiguousarray(xyzq, dtype=np.float32)
    assert a.ndim == 2 and a.shape[1] == 4, "xyzq must be float32 [N,4]"
    return a


def _m(m):
    a = np.ascontiguousarray(m, dtype=np.int32)
    assert a.ndim == 2 and a.shape[1] == 3, "m must be int32 [P,3]"
    return a


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def set_threads(n: int) -> None:
    _load().oracle_set_threads(int(n))


def S(L: float, alpha: float) -> float:
    """Normaliser S = sum_{m != 0} exp(-|k_m|^2/4alpha)."""
    return float(_load().oracle_S(float(L), float(alpha)))


def S_grid(L: float, alpha: float, mmax: int) -> float:
    return float(_load().oracle_S_grid(float(L), float(alpha), int(mmax)))


def rho(xyzq, L: float, m) -> np.ndarray:
    """Structure factors, Eq. (2.9).  Returns float64 [P,2] = (Re, Im)."""
    a, mm = _xyzq(xyzq), _m(m)
    out = np.empty((mm.shape[0], 2), dtype=np.float64)
    _load().oracle_rho(a.shape[0], _p(a), float(L), mm.shape[0], _p(mm), _p(out))
    return out


def force(xyzq, L: float, m, S_: float, rho_, w=None, sel=None, with_energy: bool = False):
    """RBE force, Eq. (2.12).  Returns float64 [nsel,3] (and [nsel] energies if asked)."""
    a, mm = _xyzq(xyzq), _m(m)
    r = np.ascontiguousarray(rho_, dtype=np.float64)
    assert r.shape == (mm.shape[0], 2)
    ww = None if w is None else np.ascontiguousarray(w, dtype=np.float64)
    if ww is not None:
        assert ww.shape == (mm.shape[0],)
    ss = None if sel is None else np.ascontiguousarray(sel, dtype=np.int64)
    nsel = a.shape[0] if ss is None else ss.shape[0]
    F = np.empty((nsel, 3), dtype=np.float64)
    e = np.empty((nsel,), dtype=np.float64) if with_energy else None
    _load().oracle_force(a.shape[0], _p(a), float(L), mm.shape[0], _p(mm), _p(ww), float(S_),
                         _p(r), nsel, _p(ss), _p(F), _p(e))
    return (F, e) if with_energy else F


def energy(L: float, m, S_: float, rho_, w=None) -> float:
    """k-space energy estimate (second term of Eq. 2.8 with the RBE weights)."""
    mm = _m(m)
    r = np.ascontiguousarray(rho_, dtype=np.float64)
    ww = None if w is None else np.ascontiguousarray(w, dtype=np.float64)
    return float(_load().oracle_energy(float(L), mm.shape[0], _p(mm), _p(ww), float(S_), _p(r)))


def ewald_full(r, q, L: float, alpha: float, nreal: int, mmax: int):
    """Full Ewald sum (Eqs. 2.8, 2.10, 2.11).  Returns (U[3]={real,k,self}, Fshort, Flong)."""
    rr = np.ascontiguousarray(r, dtype=np.float64)
    qq = np.ascontiguousarray(q, dtype=np.float64)
    n = qq.shape[0]
    assert rr.shape == (n, 3)
    U = np.empty(3, dtype=np.float64)
    Fs = np.empty((n, 3), dtype=np.float64)
    Fl = np.empty((n, 3), dtype=np.float64)
    _load().oracle_ewald_full(n, _p(rr), _p(qq), float(L), float(alpha), int(nreal), int(mmax),
                              _p(U), _p(Fs), _p(Fl))
    return U, Fs, Fl


def direct_image_sum(r, q, L: float, R: int):
    """Brute-force periodic image sum over the sphere of cells |n| <= R.  Returns (U, F)."""
    rr = np.ascontiguousarray(r, dtype=np.float64)
    qq = np.ascontiguousarray(q, dtype=np.float64)
    n = qq.shape[0]
    U = ctypes.c_double(0.0)
    F = np.empty((n, 3), dtype=np.float64)
    _load().oracle_direct_image_sum(n, _p(rr), _p(qq), float(L), int(R), ctypes.byref(U), _p(F))
    return float(U.value), F


def short_range(xyzq, L: float, alpha: float, rs: float, sel=None):
    """Short-range Ewald force, Eq. (2.10), truncated at r_s (nearest image).  Returns
    (F float64 [nsel,3], e float64 [nsel]) with sum(e) = U_short when sel is None."""
    a = _xyzq(xyzq)
    assert rs <= 0.5 * L + 1e-12, "reading Q18: r_s <= L/2"
    ss = None if sel is None else np.ascontiguousarray(sel, dtype=np.int64)
    nsel = a.shape[0] if ss is None else ss.shape[0]
    F = np.empty((nsel, 3), dtype=np.float64)
    e = np.empty((nsel,), dtype=np.float64)
    _load().oracle_short_range(a.shape[0], _p(a), float(L), float(alpha), float(rs), nsel, _p(ss), _p(F), _p(e))
    return F, e
