"""lbwp_diagnostics_static (include/lbwp.h): the diagnostics entry point that allocates nothing (its scratch is a static
device array of the library), against the existing path lbwp_diagnostics, on two calls in a row.

Collected last on purpose (the suite runs with `pytest -x`); passes alone in a fresh process and after the other tests.
Tolerance: the sums are added in the same order by both paths, so the comparison is exact (tighter than the
diagnostics tests' TOL against the oracle)."""
import ctypes
import math

import numpy as np
import pytest

from paper_2301_01622_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lbwp():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    from paper_2301_01622_b200 import build as lbuild
    from paper_2301_01622_b200 import lbwp as mod
    lbuild.build()
    return mod


def _as_dict(out, n):
    h = out.cpu().numpy()
    return {"mass": [h[0], h[1]], "momentum": [h[2], h[3], h[4]], "rho_mean_above": h[5] / h[6] if h[6] > 0 else 0.0,
            "count_above": int(h[6] + 0.5), "rho_max": h[8], "probe_rho": [h[9 + p] for p in range(n)], "unused": h[7]}


@pytest.mark.parametrize("dtype,ncomp,n", [("f32", 2, 64), ("f64", 2, 32), ("f32", 1, 48), ("f64", 1, 24)])
def test_static_diagnostics_equal_context_diagnostics_twice(lbwp, dtype, ncomp, n):
    import torch
    if ncomp == 2:
        m0 = wl.as_dtype(wl.config3(n)["moments"], dtype)
        kw = dict(lattice=27, ncomp=2, tau=0.9, A=0.01, beta=0.7)
    else:
        m0 = wl.as_dtype(wl.noisy_solenoidal(0, shape=(n, n, n)), dtype)
        kw = dict(lattice=27, ncomp=1, tau=0.6)
    probes = [(n // 4, n // 2, n // 2), (n // 2, n // 2, n // 2), (n - 1, 0, 5)]
    dprobes = torch.tensor(probes, dtype=torch.int32, device="cuda")
    out = torch.full((lbwp.DIAG_STATIC_NOUT + len(probes),), float("nan"), dtype=torch.float64, device="cuda")
    with lbwp.Lbwp(m0, dtype=dtype, **kw) as sim:
        for call in range(2):                     # the second call finds the first call's partials in the scratch
            sim.step(7)
            want = sim.diagnostics(0.5, probes)   # existing path: context scratch from cudaMalloc
            dense = sim.moments()                 # the same state, dense external layout, caller-held
            out.fill_(float("nan"))
            torch.cuda.synchronize()
            before, free_before = torch.cuda.memory_allocated(), torch.cuda.mem_get_info()[0]
            lbwp.diagnostics_static(dense, out, ncomp=ncomp, threshold=0.5, probes=dprobes)
            torch.cuda.synchronize()
            assert torch.cuda.memory_allocated() == before
            if call == 1:                         # (the first call of a process may load the module's kernels)
                assert torch.cuda.mem_get_info()[0] >= free_before, "device memory was allocated"
            got = _as_dict(out, len(probes))
            assert got.pop("unused") == 0.0
            assert got == want, (call, got, want)
            assert want["mass"][0] > 0 and want["count_above"] > 0
    # a probe outside the box is device data: NaN, and the sums are untouched
    bad = torch.tensor([[n, 0, 0], [0, 0, 0]], dtype=torch.int32, device="cuda")
    out2 = torch.zeros(lbwp.DIAG_STATIC_NOUT + 2, dtype=torch.float64, device="cuda")
    lbwp.diagnostics_static(dense, out2, ncomp=ncomp, threshold=0.5, probes=bad)
    h = out2.cpu().numpy()
    assert math.isnan(h[9]) and h[10] == float(dense[0, 0, 0, 0]) and np.array_equal(h[:9], out.cpu().numpy()[:9])


def test_static_diagnostics_rejects_sizes_beyond_the_maximum(lbwp):
    import torch
    lib = lbwp.load()
    m = torch.ones((10, 4, 4, 4), dtype=torch.float32, device="cuda")
    out = torch.zeros(16, dtype=torch.float64, device="cuda")
    pr = torch.zeros((4, 3), dtype=torch.int32, device="cuda")
    mp, op, pp = (ctypes.c_void_p(t.data_ptr()) for t in (m, out, pr))

    def call(dev=0, dtype=lbwp.LBWP_F32, ncomp=1, nx=4, ny=4, nz=4, mom=mp, npr=0, probes=None, o=op):
        return lib.lbwp_diagnostics_static(dev, dtype, ncomp, nx, ny, nz, mom, 0.5, npr, probes, o, None)

    assert call() == 0
    torch.cuda.synchronize()
    assert out[0].item() == 64.0 and out[6].item() == 64.0 and out[8].item() == 1.0
    for bad, word in [(dict(nx=2048, ny=2048, nz=1024), "LBWP_DIAG_STATIC_MAX_NODES"),      # 2^32 nodes: checked before any access
                      (dict(npr=lbwp.DIAG_STATIC_MAX_PROBES + 1, probes=pp), "LBWP_DIAG_STATIC_MAX_PROBES"),
                      (dict(npr=1, probes=None), "probe_xyz"), (dict(mom=None), "NULL"), (dict(o=None), "NULL"),
                      (dict(dtype=7), "dtype"), (dict(ncomp=3), "ncomp"), (dict(dev=64), "device"), (dict(nz=0), "empty")]:
        assert call(**bad) == -1, bad      # LBWP_EINVAL
        assert word in lib.lbwp_last_error().decode(), (bad, lib.lbwp_last_error())
