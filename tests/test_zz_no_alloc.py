"""gp_kappa_noalloc (include/gpupegas.h) against gp_kappa (pytest -m gpu).

gp_kappa_noalloc is the correctness check kappa for programs that cannot let this library take
device memory: their own pool already holds the card's HBM, or they run a loop in which a cudaMalloc would stall
every stream.  It needs no context; its partial sums live in one fixed array compiled into the library, which all
calls share and which keeps whatever the previous call left in it.  So the thing to check is not only that one call
gives gp_kappa's numbers, but that a SECOND call, on other data of another size, is not disturbed by the first
call's left-overs: the second state below has fewer blocks than the first, so stale slots of the first call lie
right behind the ones it uses.  Tolerance: kappa_close of tests/test_gpu_overdetermined.py (1e-10 relative), the
bar every kappa comparison of the suite uses; the two paths differ only in summation order.

The file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests.  It runs the same alone in a fresh process (where its first call is also the first use of the
library on the device) and after the rest of the suite.
"""
import numpy as np
import pytest

from paper_1311_0861_b200 import workloads as W
from tests.test_gpu_overdetermined import GP_OD, kappa_close, perturbation
from tests.test_gpu_parity import pkg  # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu

GAS = ["rho", "mx", "my", "mz", "E", "eps"]
STARS = ["n", "nux", "nuy", "nuz", "Exx", "Exy", "Exz", "Eyy", "Eyz", "Ezz", "Pxx", "Pxy", "Pxz", "Pyy", "Pyz", "Pzz"]


def od_context(pkg, dims, components, seed):
    """A GP_OD context (the existing path) whose carried fields are a few per cent off what the conserved fields
    imply, so that both kappa have a scale; built with the library's own calls only."""
    w = W.smooth_gas(dims=dims, kmax=2, amp=0.2, components=components, seed=seed)
    sim = pkg.Simulation(w.nx, w.ny, w.nz, w.h, w.components | GP_OD, w.poisson, w.G, w.gamma, w.bc)
    sim.set_state(w.state())
    sim.od_derive()
    for i, k in enumerate(sim.od_field_names()):
        sim.set(k, sim.get(k) * perturbation(w, seed + i))
    return w, sim


def fields_on_device(sim, names):
    """The caller's own copies of the fields (plain contiguous arrays, as the ABI defines a field)."""
    import torch
    return [sim.get(k, out=torch.empty(sim.cells, dtype=torch.float64, device="cuda")) for k in names]


def test_noalloc_kappa_matches_gp_kappa_on_two_calls_in_a_row(pkg):
    import torch
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    # 40*24*36 = 34560 cells: 9 blocks of 4096 with a ragged last one; then 36*10*12 = 4320 cells: 2 blocks
    cases = [((40, 24, 36), W.GAS | W.STARS, 300), ((36, 10, 12), W.GAS | W.STARS, 400)]
    first = None
    for dims, comp, seed in cases:
        w, sim = od_context(pkg, dims, comp, seed)
        expect = sim.kappa()                                   # the existing path: context, allocated storage
        assert min(expect) > 1e-4, expect                      # the perturbation gave both sums a scale
        gas, stars = fields_on_device(sim, GAS), fields_on_device(sim, STARS)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        got = pkg.binding.kappa_noalloc(w.h, gas=gas, stars=stars, out=out)
        torch.cuda.synchronize()
        if first is not None:      # (the very first call may make the driver load the module that holds the array)
            assert torch.cuda.mem_get_info()[0] == free_before
        got = tuple(got.cpu().tolist())
        assert kappa_close(got, expect, 1e-30), (dims, got, expect)
        if first is None:
            first = (w, gas, stars, got)
        sim.close()
    # a third call, on the first state again, after the smaller one ran in between: the same bits as before
    w, gas, stars, got0 = first
    again = tuple(pkg.binding.kappa_noalloc(w.h, gas=gas, stars=stars, out=out).cpu().tolist())
    assert again == got0, (again, got0)


def test_noalloc_kappa_one_component_and_its_limit(pkg):
    import ctypes as C
    import torch
    B = pkg.binding
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    w, sim = od_context(pkg, (70, 19, 9), W.GAS, 500)
    expect = sim.kappa()
    gas = fields_on_device(sim, GAS)
    got = tuple(B.kappa_noalloc(w.h, gas=gas, out=out).cpu().tolist())
    assert kappa_close(got, expect, 1e-30) and got[1] == 0.0 and expect[1] == 0.0, (got, expect)
    # beyond the size the fixed array was built for the call refuses, before touching any pointer
    ptrs = (C.c_void_p * 6)(*[t.data_ptr() for t in gas])
    rc = B.lib().gp_kappa_noalloc(B.KAPPA_NOALLOC_MAX_CELLS + 1, w.h, ptrs, None, out.data_ptr(), None)
    assert rc == B.GP_ERR_ARG and b"exceed the limit" in B.lib().gp_last_error()
    assert B.lib().gp_kappa_noalloc(0, w.h, ptrs, None, out.data_ptr(), None) == B.GP_ERR_ARG
    assert B.lib().gp_kappa_noalloc(16, w.h, None, None, out.data_ptr(), None) == B.GP_ERR_ARG
    torch.cuda.synchronize()
    assert np.isfinite(out.cpu().numpy()).all()
