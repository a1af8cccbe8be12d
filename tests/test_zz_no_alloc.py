"""sl1m_forward_noalloc -- the one entry point of the library that never asks the CUDA driver for memory.

Why it exists: every other call needs a plan, and creating a plan reserves workspaces with cudaMalloc.  A caller
that sits inside a real-time pipeline (an allocation holds up every stream on the device), that runs where all
device memory already belongs to somebody's pool (the raw allocation fails, or takes a neighbour's share), or that
must keep a fixed footprint after start-up cannot do that.  For them the partial sums of the pixel-split forward go
to a 4 MiB array compiled into the library instead; the caller brings every other buffer.

What is checked here: on two calls in a row (different sizes and images, so the second call runs over whatever the
first one left in the shared array) and on a repeat of the first, the visibilities agree with the existing plan path
sl1m_forward -- and with the fp64 oracle -- within the tolerance every apply test of this suite uses (relative L2
<= 2e-4); the repeat is bit-identical; the driver's free-memory figure does not move across the later calls; sizes
beyond the array are refused with a message that names the limit.

This file is named so that pytest collects it LAST (`pytest --collect-only -q`): `pytest -x` stops at the first
failure, and a failure here must not hide any other test.  It passes alone in a fresh process and after the rest."""
import ctypes

import numpy as np
import pytest

TOL_APPLY = 2e-4      # the apply tolerance of tests/test_gpu_parity.py (north_star: relative L2 per apply)


def rel_l2(got, want):
    return float(np.linalg.norm(np.asarray(got) - np.asarray(want)) / max(np.linalg.norm(want), 1e-300))


def test_noalloc_refuses_sizes_beyond_its_static_scratch():
    """Validation runs before any device work, so this needs no GPU: a visibility count the 4 MiB array cannot serve
    (one complex partial per visibility at the very least) is SL1M_ERR_SIZE, and the text tells the user the limit
    and what to do instead."""
    import paper_1310_2078_b200 as sl
    lib = sl.load_library()
    fake = ctypes.c_void_p(256)                      # never dereferenced: the size check comes first
    st = lib.sl1m_forward_noalloc(sl.NOALLOC_MAX_VIS + 1, fake, 100, fake, fake, fake, fake, None)
    assert st == 2 and lib.sl1m_status_string(st) == b"SL1M_ERR_SIZE"
    msg = lib.sl1m_last_error().decode()
    assert str(sl.NOALLOC_MAX_VIS) in msg and "static scratch" in msg and "plan" in msg, msg
    st = lib.sl1m_forward_noalloc(100, fake, sl.NOALLOC_MAX_PIX + 1, fake, fake, fake, fake, None)
    assert st == 2 and str(sl.NOALLOC_MAX_PIX) in lib.sl1m_last_error().decode()
    assert lib.sl1m_forward_noalloc(0, fake, 100, fake, fake, fake, fake, None) == 2
    assert lib.sl1m_forward_noalloc(100, fake, 100, fake, None, fake, fake, None) == 1      # SL1M_ERR_NULL


def _problem(wl, n_vis, n_pix, x):
    """One (geometry, image) case: device tensors for the new entry point, a plan for the existing path."""
    import torch
    import paper_1310_2078_b200 as sl
    uvw, l, m = wl.uvw[:n_vis], wl.l[:n_pix], wl.m[:n_pix]
    return dict(
        uvw=torch.from_numpy(np.ascontiguousarray(uvw)).cuda(), l=torch.from_numpy(np.ascontiguousarray(l)).cuda(),
        m=torch.from_numpy(np.ascontiguousarray(m)).cuda(), x=torch.from_numpy(x.astype(np.float32)).cuda(),
        out=torch.full((n_vis,), float("nan"), dtype=torch.complex64, device="cuda"),
        plan=sl.Plan(uvw, l, m), host=(uvw, l, m, x.astype(np.float32).astype(np.float64)))


@pytest.mark.gpu
def test_noalloc_forward_matches_the_plan_forward_on_two_calls_in_a_row():
    import torch
    import oracle
    import paper_1310_2078_b200 as sl
    from workloads import make_workload

    wl = make_workload(5, n_side=64, n_ant=32, n_steps=8, n_src=50)     # 30 degree field, w != 0: 4,096 pixels x 3,968 visibilities
    rng = np.random.default_rng(20261106)
    # ragged on purpose: neither size is a multiple of the kernel's 512-visibility / 256-pixel tiles
    a = _problem(wl, 3001, 4059, rng.uniform(0.0, 1.0, 4059))
    xb = np.where(rng.uniform(size=4096) < 0.05, rng.pareto(1.5, 4096) + 0.1, 0.0)          # a sparse sky
    b = _problem(wl, 1237, 4096, xb)
    want = {}
    for name, c in (("a", a), ("b", b)):
        want[name] = c["plan"].forward(c["x"]).cpu().numpy()                              # the existing path
        uvw, l, m, x64 = c["host"]
        ref = oracle.Oracle(uvw, l, m).forward(x64)
        assert rel_l2(want[name], ref) <= TOL_APPLY
        c["ref"] = ref
    torch.cuda.synchronize()

    def call(c):
        c["out"].fill_(float("nan"))
        sl.forward_noalloc(c["uvw"], c["l"], c["m"], c["x"], c["out"])
        torch.cuda.synchronize()
        return c["out"].cpu().numpy().copy()

    got_a = call(a)                                   # first call on this device: also looks up the scratch address
    free_0 = torch.cuda.mem_get_info()[0]
    got_b = call(b)                                   # second call, straight after, over the first one's leftovers
    got_a2 = call(a)
    free_1 = torch.cuda.mem_get_info()[0]
    for name, got, c in (("a", got_a, a), ("b", got_b, b), ("a again", got_a2, a)):
        assert np.all(np.isfinite(got)), name
        e_plan, e_ref = rel_l2(got, want[name[0]]), rel_l2(got, c["ref"])
        print(f"noalloc call {name}: rel-L2 vs sl1m_forward {e_plan:.2e}, vs the fp64 oracle {e_ref:.2e}")
        assert e_plan <= TOL_APPLY and e_ref <= TOL_APPLY, (name, e_plan, e_ref)
    assert np.array_equal(got_a, got_a2), "the same call twice must give the same bits (fixed summation order)"
    assert free_1 == free_0, f"device free memory moved by {free_0 - free_1} bytes across two calls that allocate nothing"
    a["plan"].close()
    b["plan"].close()


@pytest.mark.gpu
def test_noalloc_forward_at_its_visibility_limit():
    """n_vis == SL1M_NOALLOC_MAX_VIS uses every slot of the array with a single pixel split."""
    import torch
    import paper_1310_2078_b200 as sl

    rng = np.random.default_rng(7)
    n_vis, n_pix = sl.NOALLOC_MAX_VIS, 300
    uvw = rng.uniform(-2000.0, 2000.0, (n_vis, 3))
    l, m = rng.uniform(-0.2, 0.2, n_pix), rng.uniform(-0.2, 0.2, n_pix)
    x = rng.uniform(0.0, 1.0, n_pix).astype(np.float32)
    plan = sl.Plan(uvw, l, m)
    xd = torch.from_numpy(x).cuda()
    want = plan.forward(xd).cpu().numpy()
    out = torch.empty(n_vis, dtype=torch.complex64, device="cuda")
    got = sl.forward_noalloc(torch.from_numpy(uvw).cuda(), torch.from_numpy(l).cuda(), torch.from_numpy(m).cuda(), xd,
                             out).cpu().numpy()
    e = rel_l2(got, want)
    print(f"noalloc at {n_vis} visibilities x {n_pix} pixels: rel-L2 vs sl1m_forward {e:.2e}")
    assert e <= TOL_APPLY
    plan.close()
