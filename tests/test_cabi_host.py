"""Host-side checks of the C ABI (no GPU needed): librbe.so loads, exports every symbol that
include/rbe.h declares, and the calls that make no CUDA call behave as the header says."""
import ctypes
import os
import re

import numpy as np
import pytest

import oracle
from paper_2407_09315_b200 import build as rbe_build
from paper_2407_09315_b200 import inputs, rbe

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    rbe_build.build()
    return rbe.lib()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "rbe.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rbe_[a-z_A-Z0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared_symbols()
    assert {"rbe_create", "rbe_set_kvectors", "rbe_structure_factor", "rbe_forces",
            "rbe_kspace_energy", "rbe_destroy", "rbe_step_host", "rbe_set_rho", "rbe_set_pairing", "rbe_set_pair_table", "rbe_set_pair_kernel",
            "rbe_host_alloc", "rbe_host_free"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
    assert lib.rbe_version() >= 100


def test_no_torch_or_cuda_types_in_header():
    text = open(os.path.join(ROOT, "include", "rbe.h")).read()
    code = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    assert "torch" not in code and "at::" not in code and "#include <cuda" not in code
    assert not re.search(r"\bcuda[A-Z]\w*_t\b|\bCU[a-z]+\b", code)  # no cudaStream_t / CUstream etc.


@pytest.mark.parametrize("name", ["water_3k", "water_96k", "water_nacl_1m", "water_10m"])
def test_normaliser_matches_oracle(lib, name):
    cfg = inputs.CONFIGS[name]
    h = ctypes.c_void_p()
    assert lib.rbe_create(ctypes.byref(h), cfg.N, cfg.L, cfg.alpha, cfg.P) == 0
    S = lib.rbe_normaliser_S(h)
    assert abs(S - oracle.S(cfg.L, cfg.alpha)) <= 1e-13 * S
    # Poisson-resummed closed form  S = (L sqrt(alpha/pi))^3 - 1  (+ exponentially small terms)
    assert abs(S - ((cfg.L * np.sqrt(cfg.alpha / np.pi)) ** 3 - 1)) < 1e-9 * S
    assert lib.rbe_destroy(h) == 0


def test_create_rejects_bad_arguments(lib):
    h = ctypes.c_void_p()
    for args in [(-1, 10.0, 0.1, 8), (10, 0.0, 0.1, 8), (10, 10.0, -1.0, 8), (10, 10.0, 0.1, 0),
                 (10, float("nan"), 0.1, 8), (10, 10.0, float("inf"), 8)]:
        assert lib.rbe_create(ctypes.byref(h), *args) == 1
        assert not h.value
    assert lib.rbe_create(None, 1, 1.0, 1.0, 1) == 1
    assert lib.rbe_destroy(None) == 0
    assert lib.rbe_status_string(2) == b"RBE_ERR_BAD_KVECTOR"


def test_kvector_validation_and_call_order(lib):
    h = ctypes.c_void_p()
    assert lib.rbe_create(ctypes.byref(h), 100, 10.0, 0.3, 4) == 0
    good = np.array([[1, 0, 0], [0, -2, 1], [3, 3, 3], [0, 0, 1]], dtype=np.int32)
    for bad_row in ([0, 0, 0], [32768, 0, 0], [0, -32768, 1]):
        bad = good.copy()
        bad[2] = bad_row
        st = lib.rbe_set_kvectors(h, ctypes.c_void_p(bad.ctypes.data), None, None)
        assert st == 2, bad_row
        assert b"k-vector 2" in lib.rbe_last_error(h)
    w = np.array([1.0, np.nan, 1.0, 1.0])
    assert lib.rbe_set_kvectors(h, ctypes.c_void_p(good.ctypes.data), ctypes.c_void_p(w.ctypes.data), None) == 2
    # valid k-vectors but no workspace yet -> NOT_READY (still no CUDA call made)
    assert lib.rbe_set_kvectors(h, ctypes.c_void_p(good.ctypes.data), None, None) == 3
    assert lib.rbe_structure_factor(h, None, None, None) == 3
    assert lib.rbe_forces(h, None, None, 0, None) == 3
    u = ctypes.c_double()
    assert lib.rbe_kspace_energy(h, ctypes.byref(u), None) == 3
    assert lib.rbe_destroy(h) == 0


def test_size_queries_need_no_device(lib):
    """rbe_step_host_bytes / rbe_short_range_bytes / rbe_rbl_bytes are pure functions of the context (the binding
    sizes its scratch buffers with them instead of repeating the layout)."""
    lib.rbe_step_host_bytes.restype = ctypes.c_size_t
    lib.rbe_rbl_bytes.restype = ctypes.c_size_t
    lib.rbe_short_range_bytes.restype = ctypes.c_size_t
    h = ctypes.c_void_p()
    N = 100_003
    assert lib.rbe_create(ctypes.byref(h), N, 60.0, 0.09, 8) == 0
    b4, b3 = lib.rbe_step_host_bytes(h, 0), lib.rbe_step_host_bytes(h, 1)
    assert 32 * N <= b4 <= 32 * N + 1024 and 56 * N <= b3 <= 56 * N + 2048 and b4 % 256 == 0 and b3 % 256 == 0
    assert lib.rbe_step_host_bytes(None, 0) == 0
    assert lib.rbe_short_range_bytes(h, ctypes.c_double(10.0)) > 76 * N
    assert lib.rbe_short_range_bytes(h, ctypes.c_double(21.0)) == 0                 # r_s > L/3
    # rbe_short_range_bytes covers both of its force kernels: the finer list of rbe_set_pair_kernel(1) is the RBL's at r_c = r_s / 2
    assert lib.rbe_rbl_bytes(h, ctypes.c_double(5.0), ctypes.c_double(10.0)) == lib.rbe_short_range_bytes(h, ctypes.c_double(10.0))
    assert lib.rbe_rbl_bytes(h, ctypes.c_double(4.0), ctypes.c_double(10.0)) > lib.rbe_short_range_bytes(h, ctypes.c_double(10.0))
    assert lib.rbe_rbl_bytes(h, ctypes.c_double(10.0), ctypes.c_double(5.0)) == 0   # r_c >= r_s
    assert lib.rbe_rbl_bytes(h, ctypes.c_double(5.0), ctypes.c_double(21.0)) > 0    # 9 cells of 5.45 A fit the 60 A box
    assert lib.rbe_rbl_bytes(h, ctypes.c_double(5.0), ctypes.c_double(29.0)) == 0   # the stencil would meet itself
    # the one-launch step and the NVE calls refuse to run without a workspace (no CUDA call is made)
    m = np.array([[1, 0, 0]] * 8, dtype=np.int32)
    assert lib.rbe_step(h, ctypes.c_void_p(m.ctypes.data), None, None, None, 0, None, None) == 3
    out = (ctypes.c_double * 2)()
    assert lib.rbe_nve_energies(h, None, None, None, out, None) == 3
    assert lib.rbe_destroy(h) == 0


def test_no_cpu_fallback_without_device(lib):
    """On a box without a GPU the product path must fail loudly, never compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    h = ctypes.c_void_p()
    assert lib.rbe_create(ctypes.byref(h), 100, 10.0, 0.3, 4) == 0
    assert lib.rbe_workspace_bytes(h) == 0
    assert b"no CUDA device" in lib.rbe_last_error(h)
    buf = ctypes.create_string_buffer(1 << 16)
    assert lib.rbe_set_workspace(h, buf, 1 << 16) == 6
    with pytest.raises(rbe.RbeError):
        rbe.Rbe(100, 10.0, 0.3, 4)
    lib.rbe_destroy(h)


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2407_09315_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), f
                assert "liboracle" not in src and "rbe_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2407_09315_b200\b", src, flags=re.M), f
            assert "librbe" not in src and "#include \"rbe" not in src, f


@pytest.mark.parametrize("alpha,rs", [(0.09, 10.0), (0.35, 6.0), (0.02, 11.3), (0.1156, 30.0), (1.0, 30.0)])
def test_pair_table_matches_the_closed_forms(alpha, rs):
    """rbe_pair_table_host (the same function the device kernel runs): the tabulated pair term of P:196 as built here
    (reading Q23).  Evaluated the way the kernels do -- index and origin from the fp32 bit pattern of u = r^2, cubic
    in fp32 -- it must reproduce T_f(u) = e^{alpha u} [erfc(x)/r + 2 sqrt(alpha/pi) e^{-x^2}] / u and
    T_e(u) = e^{alpha u} erfc(x)/r (x = sqrt(alpha) r; written out with scipy) to 1e-6 relative everywhere on
    [2^-6, r_s^2), i.e. the pair force and energy of Eq. (2.10) / Eq. (2.8) once multiplied by e^{-alpha u}."""
    from scipy.special import erfcx

    from paper_2407_09315_b200 import rbe
    ctx = rbe.Rbe(8, 100.0, alpha, 4, allocate=False)
    tf, te = ctx.rbe_pair_table_host(rs)
    n = tf.shape[0]
    assert n == (int(np.floor(np.log2(rs * rs))) + 1 + 6) * 32 and te.shape == (n, 4)
    rng = np.random.default_rng(3)
    u = np.concatenate([np.exp(rng.uniform(np.log(2.0 ** -6), np.log(rs * rs), 200_000)),
                        2.0 ** -6 * (1 + np.arange(64) / 32.0), [np.nextafter(np.float32(rs * rs), np.float32(0))]]).astype(np.float32)
    u = u[(u >= 2.0 ** -6) & (u < rs * rs)]
    bits = u.view(np.uint32)
    idx = (bits >> 18).astype(np.int64) - ((127 - 6) << 5)
    assert idx.min() == 0 and idx.max() < n
    d = u - (bits & np.uint32(0xFFFC0000)).view(np.float32)                          # exact in fp32
    def cubic(t):
        c = t[idx]
        return ((c[:, 3] * d + c[:, 2]) * d + c[:, 1]) * d + c[:, 0]                 # fp32 Horner, as the kernels
    ud = u.astype(np.float64)
    r = np.sqrt(ud)
    x = np.sqrt(alpha) * r
    Te = erfcx(x) / r
    Tf = (Te + 2.0 * np.sqrt(alpha / np.pi)) / ud
    assert np.abs(cubic(tf) / Tf - 1).max() <= 1e-6
    assert np.abs(cubic(te) / Te - 1).max() <= 1e-6
