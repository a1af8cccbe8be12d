"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/sl1m.h declares; argument validation runs before any device work; without a CUDA
device the product path fails loudly (no CPU fallback, no route through the oracle)."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_1310_2078_b200 as sl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    lib = sl.load_library()
    names = sl.exported_symbols()
    assert {"sl1m_plan_create", "sl1m_forward", "sl1m_adjoint", "sl1m_solve", "sl1m_destroy",
            "sl1m_max_eig"} <= set(names)
    for n in names:
        assert hasattr(lib, n), n
        getattr(lib, n)


def test_status_strings_and_null_safety():
    lib = sl.load_library()
    assert lib.sl1m_status_string(0) == b"SL1M_OK"
    assert lib.sl1m_status_string(3) == b"SL1M_ERR_DOMAIN"
    assert lib.sl1m_status_string(99) == b"SL1M_ERR_UNKNOWN"
    lib.sl1m_destroy(None)
    assert lib.sl1m_launch_count(None) == 0 and lib.sl1m_plan_n_pix(None) == 0
    assert lib.sl1m_forward(None, None, None, None) == 1
    assert lib.sl1m_solve(None, None, 0.0, 1.0, 0, 0, None, None, None, None, None) == 1


def test_validation_precedes_device_work():
    """These must fail with their own status even on a box with no GPU."""
    uvw = np.zeros((4, 3))
    with pytest.raises(sl.Sl1mError, match="SL1M_ERR_DOMAIN"):
        sl.Plan(uvw, [0.9], [0.9])
    with pytest.raises(sl.Sl1mError, match="SL1M_ERR_SIZE"):
        sl.Plan(np.zeros((0, 3)), [0.0], [0.0])
    with pytest.raises(sl.Sl1mError, match="SL1M_ERR_INDEX"):
        sl.Plan(uvw, [0.0], [0.0], ant_p=[0, 0, 0, 5], ant_q=[0, 0, 0, 0], gains=np.ones((2, 1), np.complex64))
    with pytest.raises(sl.Sl1mError, match="SL1M_ERR_PARAM"):
        sl.Plan(uvw, [0.0], [0.0], gauss_model=3)


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(sl.Sl1mError, match="SL1M_ERR_CUDA"):
        sl.Plan(np.zeros((4, 3)), [0.0], [0.0])


def test_product_path_never_touches_the_oracle_and_vice_versa():
    """The two sides share no code and neither imports the other (prompt section 3)."""
    pkg = os.path.join(ROOT, "paper_1310_2078_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, re.M), f
                assert "liboracle" not in txt and "sl1m_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1310_2078_b200" not in txt and "from paper_1310_2078_b200" not in txt, f
            assert "libsl1m" not in txt and "#include \"sl1m" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "workloads")):
        if f.endswith(".py"):
            txt = open(os.path.join(ROOT, "workloads", f)).read()
            assert not re.search(r"^\s*(import|from)\s+(oracle|paper_1310_2078_b200)\b", txt, re.M), f


def test_sass_has_tma_bulk_copy_and_mufu():
    """The forward kernel stages pixel tiles with TMA bulk copies (UBLKCP) and generates entries
    with MUFU.SIN/COS; checked on the built library when cuobjdump is available."""
    import shutil
    import subprocess
    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    sl.load_library()
    sass = subprocess.run([cuobjdump, "-sass", sl.library_path()], capture_output=True, text=True).stdout
    assert "UBLKCP" in sass and "MUFU.SIN" in sass and "MUFU.COS" in sass and "MUFU.EX2" in sass
    assert "sm_100a" in sass


def test_quadtree_refine_host_logic_is_bit_exact_against_the_oracle():
    """sl1m_quadtree_refine is pure host code (no GPU needed): on the same fp32 image it must take
    exactly the oracle's decisions (reading R23) -- same leaves, same order, same start values."""
    import numpy as np
    import oracle
    rng = np.random.default_rng(3)
    N, d = 12, 0.004
    k = np.arange(N * N)
    l, m, side = (k % N - N / 2 + 0.5) * d, (k // N - N / 2 + 0.5) * d, np.full(N * N, d)
    I = np.where(rng.uniform(size=N * N) < 0.3, rng.pareto(1.5, N * N), 0.0).astype(np.float32)
    for frac, min_side in ((0.01, 0.0), (0.2, d / 4), (-1.0, 0.0), (0.05, d)):
        for _ in range(3):
            got = sl.quadtree_refine(l, m, side, I, frac, min_side)
            want = oracle.quadtree_refine(l, m, side, I.astype(np.float64), frac, min_side)
            assert got[5] == want[5]
            for a, b in zip(got[:3], want[:3]):
                assert np.array_equal(a, b)
            assert np.array_equal(got[3].astype(np.float64), want[3]) and np.array_equal(got[4], want[4])
            l, m, side = got[0], got[1], got[2]
            I = (got[3] * rng.uniform(0.2, 1.5, got[3].shape[0])).astype(np.float32)
        l, m, side = (k % N - N / 2 + 0.5) * d, (k // N - N / 2 + 0.5) * d, np.full(N * N, d)
        I = np.where(rng.uniform(size=N * N) < 0.3, rng.pareto(1.5, N * N), 0.0).astype(np.float32)
    # capacity too small: refused, nothing else
    lib = sl.load_library()
    import ctypes
    out = np.empty(4), np.empty(4), np.empty(4), np.empty(4, np.float32)
    n_out, n_ref = ctypes.c_int64(), ctypes.c_int64()
    four = np.array([-1.0, 1.0, -1.0, 1.0]), np.array([-1.0, -1.0, 1.0, 1.0]), np.full(4, 2.0), np.ones(4, np.float32)
    st = lib.sl1m_quadtree_refine(4, *(a.ctypes.data_as(ctypes.c_void_p) for a in four), 0.5, 0.0, 4,
                                  *(a.ctypes.data_as(ctypes.c_void_p) for a in out), None, ctypes.byref(n_out),
                                  ctypes.byref(n_ref))
    assert st == 2  # SL1M_ERR_SIZE
    # ... and the failure carries its own detail text (not a stale one from an earlier call)
    assert b"capacity" in lib.sl1m_last_error()
    # an image that is zero everywhere splits nothing, also with frac < 0 (sl1m.h; the oracle agrees)
    zero = np.zeros(4, np.float32)
    got = sl.quadtree_refine(four[0], four[1], four[2], zero, -1.0, 0.0)
    assert got[5] == 0 and got[0].shape[0] == 4
    assert oracle.quadtree_refine(four[0], four[1], four[2], zero.astype(np.float64), -1.0, 0.0)[5] == 0
