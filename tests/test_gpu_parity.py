"""GPU-vs-oracle parity through the C ABI (pytest -m gpu), SURVEY.md 8(d) "parity protocol".

Both sides get the same seeded inputs, compute their own dt (relative difference <= 1e-13),
then both step with the ORACLE's dt so that rounding in dt does not compound.  Bars
(BASELINE.json north_star): per field group, max|diff|/max|ref| <= 1e-11 after one step;
sum|diff|/sum|ref| <= 1e-8 after the config's step count.  Momenta and the six nE_ij are
compared as vector groups (a component that is ~0 by symmetry has no scale of its own).
"""
import numpy as np
import pytest

from paper_1311_0861_b200 import workloads as W

pytestmark = pytest.mark.gpu

GROUPS_GAS = [("rho",), ("mx", "my", "mz"), ("E",)]
GROUPS_BME = [("n",), ("nux", "nuy", "nuz"), ("Exx", "Exy", "Exz", "Eyy", "Eyz", "Ezz")]
TOL_1STEP = 1e-11
TOL_NSTEP = 1e-8


@pytest.fixture(scope="module")
def pkg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1311_0861_b200 as p
    p.lib()
    return p


def groups(w):
    return (GROUPS_GAS if w.components & W.GAS else []) + (GROUPS_BME if w.components & W.STARS else [])


def err_max(sim, ref, names):
    num = max(np.abs(sim.get(k) - ref.get(k)).max() for k in names)
    den = max(np.abs(ref.get(k)).max() for k in names)
    return num / den


def err_l1(sim, ref, names):
    num = sum(np.abs(sim.get(k) - ref.get(k)).sum() for k in names)
    den = sum(np.abs(ref.get(k)).sum() for k in names)
    return num / den


def make_pair(pkg, orc, w):
    state = w.state()
    sim = pkg.Simulation.from_workload(w)
    sim.set_state(state)
    ref = orc.Oracle(w.nx, w.ny, w.nz, w.h, w.components, w.poisson, w.G, w.gamma, w.bc)
    ref.set_state(state)
    return sim, ref


def full_step(sim, ref, w, dt_cap=None):
    if w.poisson != W.POISSON_NONE:
        sim.solve_poisson()
        ref.solve_poisson()
    dt_g, dt_r = sim.max_dt(w.cfl), ref.max_dt(w.cfl)
    assert abs(dt_g - dt_r) <= 1e-13 * dt_r, (dt_g, dt_r)
    dt = dt_r if dt_cap is None else min(dt_r, dt_cap)
    sim.step(dt)
    ref.step(dt)
    return dt


REPORT = []          # (workload, grid, kind, field group, error) of every comparison, dumped at module teardown


@pytest.fixture(scope="module", autouse=True)
def parity_report():
    yield
    import json
    import os
    out = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "gpurun_out")
    os.makedirs(out, exist_ok=True)
    with open(os.path.join(out, "parity_report.json"), "w") as f:
        json.dump(REPORT, f, indent=0)


def check(sim, ref, w, tol, err):
    kind = "max_1step" if err is err_max else "l1_nstep"
    for g in groups(w):
        e = err(sim, ref, g)
        REPORT.append([w.name, [w.nx, w.ny, w.nz], kind, "+".join(g), float(e)])
        assert e <= tol, (w.name, g, e)
    if w.poisson != W.POISSON_NONE:
        e = err_max(sim, ref, ("phi",))
        REPORT.append([w.name, [w.nx, w.ny, w.nz], kind, "phi", float(e)])
        assert e <= TOL_1STEP, (w.name, "phi", e)


def run_parity(pkg, orc, w, steps):
    sim, ref = make_pair(pkg, orc, w)
    full_step(sim, ref, w)
    check(sim, ref, w, TOL_1STEP, err_max)
    for _ in range(steps - 1):
        full_step(sim, ref, w)
    check(sim, ref, w, TOL_NSTEP, err_l1)
    return sim, ref


# ------------------------------------------------------------------------------------------------
# the five configs at sizes the oracle finishes in seconds
# ------------------------------------------------------------------------------------------------
def test_config1_sod_full_run_and_exact_solution(pkg, orc):
    from tests import exact_riemann as ER
    w = W.sod()                                                 # 128x4x4, the config's own size
    sim, ref = make_pair(pkg, orc, w)
    t, n = 0.0, 0
    while t < w.t_end * (1 - 1e-14):
        dt = full_step(sim, ref, w, dt_cap=w.t_end - t)
        if n == 0:
            check(sim, ref, w, TOL_1STEP, err_max)
        t += dt
        n += 1
    assert n == 274
    check(sim, ref, w, TOL_NSTEP, err_l1)
    rho = sim.get("rho")
    assert np.all(rho == rho[0:1, 0:1, :])                      # 1-D problem stays 1-D, bitwise
    x = (np.arange(w.nx) + 0.5) * w.h
    re, ue, pe = ER.sample((x - 0.5) / t, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, w.gamma)
    u = sim.get("mx")[0, 0] / rho[0, 0]
    p = (w.gamma - 1) * (sim.get("E")[0, 0] - 0.5 * rho[0, 0] * u * u)
    assert np.abs(rho[0, 0] - re).mean() < 2.5e-2 and np.abs(u - ue).mean() < 4.5e-2 and np.abs(p - pe).mean() < 2.5e-2


def test_config2_smooth_gas_reduced(pkg, orc):
    run_parity(pkg, orc, W.smooth_gas(n=64, steps=100), 100)


def test_config2_ragged_dims_gas_and_stars(pkg, orc):
    # sizes that are no multiple of any tile, both components, no gravity
    run_parity(pkg, orc, W.smooth_gas(dims=(70, 19, 9), kmax=2, amp=0.2, components=W.GAS | W.STARS), 20)


def test_config3_collapse_isolated_reduced(pkg, orc):
    run_parity(pkg, orc, W.collapse(n=32, steps=200), 200)


def test_config4_disk_periodic_reduced(pkg, orc):
    run_parity(pkg, orc, W.disk(n=64, rd_cells=3.2, zd_cells=1.28), 100)


def test_config5_two_disks_periodic_reduced(pkg, orc):
    run_parity(pkg, orc, W.two_disks(n=64, rd_cells=3.2, zd_cells=1.28), 50)


def test_config5_two_disks_isolated_reduced(pkg, orc):
    run_parity(pkg, orc, W.two_disks(n=32, rd_cells=3.2, zd_cells=1.28, poisson=W.POISSON_ISOLATED), 20)


# ------------------------------------------------------------------------------------------------
# edge cases
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 1, 1), (1, 0, 1), (0, 1, 0)])
def test_minimum_grid_and_boundary_mixes(pkg, orc, bc):
    w = W.smooth_gas(dims=(4, 4, 4), kmax=1, amp=0.2, components=W.GAS | W.STARS)
    w.bc = bc
    run_parity(pkg, orc, w, 5)


@pytest.mark.parametrize("bc", [(1, 0, 1), (0, 1, 0), (1, 1, 0), (1, 1, 1)])
def test_mixed_hydro_boundaries_under_the_periodic_solve(pkg, orc, bc):
    """Periodic Poisson solve (Phi and its ghosts wrap on every axis) with outflow hydro boundaries on some
    axes: the U* of a periodic ghost cell next to an outflow face takes grad Phi from the wrapped Phi."""
    w = W.two_disks(n=32, rd_cells=3.2, zd_cells=1.28)
    w.bc = bc
    run_parity(pkg, orc, w, 6)


def test_user_set_phi_with_mixed_boundaries(pkg, orc):
    """GP_POISSON_NONE with a Phi handed in by the caller: its ghosts follow the hydro rule per axis."""
    w = W.smooth_gas(dims=(36, 10, 12), kmax=2, amp=0.2, components=W.GAS | W.STARS)
    w.bc = (1, 0, 1)
    rng = np.random.default_rng(77)
    phi = 0.3 * rng.standard_normal((w.nz, w.ny, w.nx))
    sim, ref = make_pair(pkg, orc, w)
    sim.set("phi", phi)
    ref.set("phi", phi)
    for _ in range(4):
        full_step(sim, ref, w)
    check(sim, ref, w, TOL_1STEP * 10, err_max)


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_tubes_along_each_axis_with_outflow(pkg, orc, axis):
    for comp in (W.GAS, W.STARS):
        w = W.sod(n=48, nt=5, axis=axis, components=comp)
        w.steps = 30
        run_parity(pkg, orc, w, 30)


def test_state_round_trip_is_bit_exact_and_restartable(pkg, orc):
    w = W.smooth_gas(dims=(24, 12, 10), kmax=2, components=W.GAS | W.STARS)
    state = w.state()
    a = pkg.Simulation.from_workload(w)
    a.set_state(state)
    for k in a.field_names():
        assert np.array_equal(a.get(k), state[k])
    a.step(1e-3)
    b = pkg.Simulation.from_workload(w)
    b.set_state(a.get_state())
    a.step(1e-3)
    b.step(1e-3)
    for k in a.field_names():
        assert np.array_equal(a.get(k), b.get(k))


def test_device_resident_dt_equals_host_dt(pkg, orc):
    w = W.smooth_gas(dims=(32, 16, 8), kmax=2, components=W.GAS | W.STARS)
    a = pkg.Simulation.from_workload(w)
    b = pkg.Simulation.from_workload(w)
    a.set_state(w.state())
    b.set_state(w.state())
    dt = a.max_dt(w.cfl)
    a.step(dt)
    b.max_dt(w.cfl, to_host=False)
    b.step(0.0)
    for k in a.field_names():
        assert np.array_equal(a.get(k), b.get(k))


def test_device_pointers_and_own_allocation(pkg, orc):
    import torch
    w = W.smooth_gas(dims=(16, 8, 8), kmax=1)
    a = pkg.Simulation.from_workload(w, use_torch_memory=False)     # library-owned cudaMalloc
    b = pkg.Simulation.from_workload(w)
    st = w.state()
    for k, v in st.items():
        a.set(k, v)
        b.set(k, torch.from_numpy(v).cuda())                        # device-to-device set
    a.step(1e-3)
    b.step(1e-3)
    out = torch.empty(w.cells, dtype=torch.float64, device="cuda")
    for k in st:
        assert np.array_equal(a.get(k), b.get(k, out=out).cpu().numpy().reshape(a.shape))


def test_bad_state_and_bad_arguments_are_reported(pkg, orc):
    w = W.smooth_gas(dims=(8, 8, 8), kmax=1)
    s = pkg.Simulation.from_workload(w)
    st = w.state()
    st["E"] = st["E"].copy()
    st["E"][1, 2, 3] = 0.0                                           # negative pressure there
    s.set_state(st)
    with pytest.raises(pkg.GpError) as e:
        s.max_dt(0.3)
    assert e.value.code == pkg.GP_ERR_STATE
    st["E"][1, 2, 3] = np.nan
    s.set_state(st)
    with pytest.raises(pkg.GpError) as e:
        s.max_dt(0.3)
    assert e.value.code == pkg.GP_ERR_STATE
    with pytest.raises(pkg.GpError):                                 # stars are not enabled
        s.set("n", st["rho"])
    with pytest.raises(pkg.GpError):                                 # no Poisson mode
        s.solve_poisson()
    with pytest.raises(pkg.GpError):                                 # too small
        pkg.Simulation(3, 8, 8, 0.1)
    with pytest.raises(pkg.GpError):                                 # odd size with a Poisson mode
        pkg.Simulation(9, 8, 8, 0.1, poisson=pkg.GP_POISSON_PERIODIC)


def test_poisson_non_power_of_two_against_stencil(pkg, orc):
    """The CUDA path accepts any even size; where the oracle's radix-2 FFT cannot follow, the
    27-point stencil residual (a property that holds at any size) is the check."""
    nx, ny, nz, h, G = 24, 12, 20, 0.1, 1.3
    rng = np.random.default_rng(7)
    rho = rng.uniform(0.5, 1.5, (nz, ny, nx))
    s = pkg.Simulation(nx, ny, nz, h, pkg.GP_GAS, pkg.GP_POISSON_PERIODIC, G=G)
    s.set("rho", rho)
    s.solve_poisson()
    phi = s.get("phi")
    a = phi
    for ax in range(3):
        a = (np.roll(a, 1, ax) + 4.0 * a + np.roll(a, -1, ax)) / 6.0
    res = 6.0 * (a - phi) / (h * h) - 4 * np.pi * G * (rho - rho.mean())
    assert np.abs(res).max() < 1e-11 * 4 * np.pi * G * rho.max()
    assert abs(phi.mean()) < 1e-12 * np.abs(phi).max()


def test_device_reciprocal_and_rsqrt_are_accurate_to_a_few_ulp(pkg):
    """The hydro kernels use 1/x and 1/sqrt(x) built from the hardware seed plus one cubic
    correction; bound their error over 60 decades against numpy's correctly rounded results."""
    rng = np.random.default_rng(11)
    x = np.concatenate([10.0 ** rng.uniform(-30, 30, 200000), rng.uniform(0.5, 2.0, 200000),
                        np.array([1.0, 2.0, 4.0, 0.25, 3.0, 1e-4, 1e4])])
    r, s = pkg.math_selftest(x)
    ulp = np.finfo(np.float64).eps
    assert np.abs(r * x - 1.0).max() <= 4 * ulp
    exact = 1.0 / np.sqrt(x)
    assert (np.abs(s - exact) / exact).max() <= 4 * ulp


# ------------------------------------------------------------------------------------------------
# periodic Poisson: fused z pass (every radix mix 2^3 .. 2^10, non-cubic grids) and the source
# rho + n that rides in the step's epilogue
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [(16, 8, 8), (8, 16, 16), (32, 8, 32), (16, 32, 64), (8, 8, 128), (12, 6, 256),
                                  (8, 4, 512), (4, 4, 1024)])
def test_periodic_poisson_fused_z_pass_against_oracle(pkg, orc, dims):
    nx, ny, nz = dims
    h, G = 0.05, 0.7
    rng = np.random.default_rng(100 + nz)
    rho = rng.uniform(0.5, 1.5, (nz, ny, nx))
    n = rng.uniform(0.1, 0.4, (nz, ny, nx))
    s = pkg.Simulation(nx, ny, nz, h, pkg.GP_GAS | pkg.GP_STARS, pkg.GP_POISSON_PERIODIC, G=G)
    s.set("rho", rho)
    s.set("n", n)
    s.solve_poisson()
    phi = s.get("phi")
    # property that holds at any size: the 27-point stencil residual
    a = phi
    for ax in range(3):
        a = (np.roll(a, 1, ax) + 4.0 * a + np.roll(a, -1, ax)) / 6.0
    src = rho + n
    res = 6.0 * (a - phi) / (h * h) - 4 * np.pi * G * (src - src.mean())
    assert np.abs(res).max() < 1e-11 * 4 * np.pi * G * src.max()
    if all(d & (d - 1) == 0 for d in dims):                     # the oracle's FFT is radix 2
        r = orc.Oracle(nx, ny, nz, h, orc.GAS | orc.STARS, orc.POISSON_PERIODIC, G)
        r.set("rho", rho)
        r.set("n", n)
        r.solve_poisson()
        ref = r.get("phi")
        assert np.abs(phi - ref).max() <= TOL_1STEP * np.abs(ref).max()


def test_source_from_step_epilogue_equals_fresh_assembly(pkg, orc):
    """After gp_step the next solve uses rho + n written by the gas kernel's epilogue;
    a solve after a get/set round trip reassembles it with k_source.  Both must agree bitwise."""
    w = W.two_disks(n=32, rd_cells=3.2, zd_cells=1.28)
    a = pkg.Simulation.from_workload(w)
    a.set_state(w.state())
    a.solve_poisson()
    a.step(a.max_dt(w.cfl))
    b = pkg.Simulation.from_workload(w)
    b.set_state({k: a.get(k) for k in a.field_names()})
    a.solve_poisson()
    b.solve_poisson()
    assert np.array_equal(a.get("phi"), b.get("phi"))


# ------------------------------------------------------------------------------------------------
# isolated Poisson: pruned transforms (power-of-two ny, nz) and the full-cuFFT fallback, against
# direct summation (the definition, PAPER.md:186 with the boundary reading G3) and the oracle
# ------------------------------------------------------------------------------------------------
# the thin grids reach the column transforms the full-size configs run: 256-point (P=8), 512-point
# (k_colfft<9,4,2>, config 3 at 256^3) and 1024-point columns (k_colfft<10,4,1>, config 5 isolated at 512^3),
# with their zero-pruned input (nin), the kept-rows remap (nkeep, row 2^P-1) and 4-column tiles
@pytest.mark.parametrize("dims", [(4, 4, 4), (16, 8, 32), (8, 32, 4), (10, 16, 8), (6, 4, 64), (10, 12, 6), (8, 6, 8),
                                  (8, 128, 8), (8, 8, 128), (8, 256, 8), (8, 8, 256), (8, 4, 512), (4, 512, 8),
                                  (12, 256, 4)])
def test_isolated_poisson_against_direct_summation(pkg, orc, dims):
    nx, ny, nz = dims
    h, G = 0.1, 1.7
    rng = np.random.default_rng(300 + nx + 7 * nz)
    rho = rng.uniform(0.0, 1.0, (nz, ny, nx))
    s = pkg.Simulation(nx, ny, nz, h, pkg.GP_GAS, pkg.GP_POISSON_ISOLATED, G=G, bc=(1, 1, 1))
    s.set("rho", rho)
    s.solve_poisson()
    phi = s.get("phi")
    ref = orc.poisson_direct(rho, h, G)
    assert np.abs(phi - ref).max() <= 1e-11 * np.abs(ref).max()
    s.set("rho", 2.0 * rho)                       # a second solve reuses plans, tables and work arrays
    s.solve_poisson()
    assert np.abs(s.get("phi") - 2.0 * ref).max() <= 2e-11 * np.abs(ref).max()


def test_isolated_poisson_ghost_faces_drive_the_same_step_as_the_oracle(pkg, orc):
    """The six ghost faces of Phi come from padded indices 2N-1 and N; a step of a cloud that touches
    every face of a non-cubic box uses all of them."""
    w = W.collapse(n=16, steps=1)
    nx, ny, nz = 16, 8, 32
    rng = np.random.default_rng(5)
    st = {"rho": rng.uniform(0.5, 1.5, (nz, ny, nx))}
    st["mx"] = 0.1 * st["rho"] * rng.uniform(-1, 1, (nz, ny, nx))
    st["my"] = 0.1 * st["rho"] * rng.uniform(-1, 1, (nz, ny, nx))
    st["mz"] = 0.1 * st["rho"] * rng.uniform(-1, 1, (nz, ny, nx))
    st["E"] = 1.5 * st["rho"] + 0.5 * (st["mx"] ** 2 + st["my"] ** 2 + st["mz"] ** 2) / st["rho"]
    sim = pkg.Simulation(nx, ny, nz, 0.05, pkg.GP_GAS, pkg.GP_POISSON_ISOLATED, G=1.0, gamma=w.gamma, bc=(1, 1, 1))
    ref = orc.Oracle(nx, ny, nz, 0.05, orc.GAS, orc.POISSON_ISOLATED, 1.0, w.gamma, (1, 1, 1))
    sim.set_state(st)
    ref.set_state(st)
    sim.solve_poisson()
    ref.solve_poisson()
    dt = ref.max_dt(0.2)
    sim.step(dt)
    ref.step(dt)
    for g in GROUPS_GAS:
        assert err_max(sim, ref, g) <= TOL_1STEP, g


def test_fp64_issue_rate_self_test_backs_the_alu_peak(pkg):
    """bench.py's roofline_alu takes 148 SMs x 64 fp64 lanes x the SM clock as the peak; the DFMA self test of the
    library (csrc/selftest.cu) must reach most of it and cannot exceed it."""
    import torch
    rate, ms = pkg.fp64_rate_selftest()
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    nominal = sms * 64 * 1.965e9
    assert 0.75 * nominal <= rate <= 1.02 * nominal, (rate, nominal, ms)
