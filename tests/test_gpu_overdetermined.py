"""The overdetermined system (PAPER.md:41 4th equation, 65, 194-202) through the CUDA path against
the oracle (pytest -m gpu): contexts created with GP_OD carry rho*eps and Pi_ij inside the fused kernels, take the
pressure and the dispersion tensor from the carried fields, fold kappa and apply the energy balance (G15)
in the kernels' epilogue.

Same protocol and bars as tests/test_gpu_parity.py: same seeded inputs, both sides step with the oracle's dt;
max|diff|/max|ref| <= 1e-11 per field group after one step, sum|diff|/sum|ref| <= 1e-8 after N steps.  The carried
fields are perturbed away from what the conserved fields imply (seeded, smooth, a few per cent), so that a kernel
taking p or Pi from the wrong description fails, and so that kappa has a scale.
"""
import numpy as np
import pytest

from paper_1311_0861_b200 import workloads as W
from tests.test_gpu_parity import GROUPS_BME, GROUPS_GAS, TOL_1STEP, TOL_NSTEP, err_l1, err_max
from tests.test_gpu_parity import pkg  # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu

GP_OD = 4
OD_GAS = [("eps",)]
OD_BME = [("Pxx", "Pxy", "Pxz", "Pyy", "Pyz", "Pzz")]
PI = ["Pxx", "Pxy", "Pxz", "Pyy", "Pyz", "Pzz"]


def groups(w):
    return ((GROUPS_GAS + OD_GAS) if w.components & W.GAS else []) + ((GROUPS_BME + OD_BME) if w.components & W.STARS else [])


def perturbation(w, seed):
    """Smooth seeded factor 1 + 0.04 cos(...) on the grid of w."""
    rng = np.random.default_rng(seed)
    k = rng.integers(1, 3, size=3)
    ph = rng.uniform(0, 2 * np.pi)
    z, y, x = np.meshgrid(np.arange(w.nz) / w.nz, np.arange(w.ny) / w.ny, np.arange(w.nx) / w.nx, indexing="ij")
    return 1.0 + 0.04 * np.cos(2 * np.pi * (k[0] * x + k[1] * y + k[2] * z) + ph)


def make_pair(pkg, orc, w, perturb=True, state=None):
    """A GP_OD context and an oracle with the overdetermined system enabled, same state; carried fields derived on
    each side by its own code, then (perturb) overwritten on both with the oracle's derived values times a factor."""
    state = w.state() if state is None else state
    sim = pkg.Simulation(w.nx, w.ny, w.nz, w.h, w.components | GP_OD, w.poisson, w.G, w.gamma, w.bc)
    sim.set_state(state)
    sim.od_derive()
    ref = orc.Oracle(w.nx, w.ny, w.nz, w.h, w.components, w.poisson, w.G, w.gamma, w.bc)
    ref.set_state(state)
    ref.od_enable()
    if perturb:
        for i, k in enumerate(ref.od_field_names()):
            a = ref.get(k) * perturbation(w, 100 + i)
            ref.set(k, a)
            sim.set(k, a)
    return sim, ref


def check(sim, ref, w, tol, err):
    for g in groups(w):
        e = err(sim, ref, g)
        assert e <= tol, (w.name, g, e)


def od_step(sim, ref, w, balance, dt=None):
    if w.poisson != W.POISSON_NONE:
        sim.solve_poisson()
        ref.solve_poisson()
    if dt is None:
        dt_g, dt = sim.max_dt(w.cfl), ref.max_dt(w.cfl)
        assert abs(dt_g - dt) <= 1e-13 * dt, (dt_g, dt)
    sim.od_step(dt, balance=balance)
    ref.od_step(dt, balance=balance)
    return dt


def kappa_close(a, b, scale):
    return all(abs(x - y) <= 1e-10 * max(abs(y), scale) for x, y in zip(a, b))


# ------------------------------------------------------------------------------------------------
def test_derive_matches_the_oracle(pkg, orc):
    w = W.smooth_gas(dims=(36, 10, 12), kmax=2, amp=0.2, components=W.GAS | W.STARS)
    sim, ref = make_pair(pkg, orc, w, perturb=False)
    for k in ref.od_field_names():
        a, b = sim.get(k), ref.get(k)
        assert np.abs(a - b).max() <= 4e-16 * np.abs(b).max(), k
    # derived fields: kappa is zero to round-off on both sides
    kg, kb = sim.kappa()
    scale = w.h ** 3 * w.cells
    assert kg <= 1e-14 * scale and kb <= 1e-14 * scale


@pytest.mark.parametrize("components", [W.GAS, W.STARS, W.GAS | W.STARS])
@pytest.mark.parametrize("balance", [False, True])
def test_od_step_parity_smooth_periodic(pkg, orc, components, balance):
    w = W.smooth_gas(dims=(40, 24, 36), kmax=2, amp=0.2, components=components)
    sim, ref = make_pair(pkg, orc, w)
    k0 = ref.kappa()
    assert kappa_close(sim.kappa(), k0, 1e-30) and max(k0) > 1e-3      # the perturbation gives kappa a scale
    od_step(sim, ref, w, balance)
    check(sim, ref, w, TOL_1STEP, err_max)
    if not balance:
        # the kernels' folded kappa is that of the state they produced
        assert kappa_close(sim.od_last_kappa(), ref.kappa(), 1e-30)
        assert kappa_close(sim.kappa(), ref.kappa(), 1e-30)
    else:
        scale = w.h ** 3 * w.cells
        assert max(sim.kappa()) <= 1e-13 * scale and max(ref.kappa()) <= 1e-13 * scale
    for _ in range(11):
        od_step(sim, ref, w, balance)
    check(sim, ref, w, TOL_NSTEP, err_l1)


def test_od_step_grid_with_interior_tiles(pkg, orc):
    """Large enough that some footprints lie inside the grid (staged by TMA boxes, 16 fields in 8 pair maps) and that
    the z extent is cut into chunks; outflow along y exercises the U* ghost copies of the wider ring slots."""
    w = W.smooth_gas(dims=(96, 48, 40), kmax=3, amp=0.2, components=W.GAS | W.STARS)
    w.bc = (0, 1, 0)
    sim, ref = make_pair(pkg, orc, w)
    od_step(sim, ref, w, False)
    check(sim, ref, w, TOL_1STEP, err_max)
    assert kappa_close(sim.od_last_kappa(), ref.kappa(), 1e-30)
    for _ in range(3):
        od_step(sim, ref, w, True)
    check(sim, ref, w, TOL_NSTEP, err_l1)


def test_od_step_ragged_outflow_and_mixed_boundaries(pkg, orc):
    for bc in [(1, 1, 1), (1, 0, 1), (0, 1, 0)]:
        w = W.smooth_gas(dims=(70, 19, 9), kmax=2, amp=0.2, components=W.GAS | W.STARS)
        w.bc = bc
        sim, ref = make_pair(pkg, orc, w)
        od_step(sim, ref, w, False)
        check(sim, ref, w, TOL_1STEP, err_max)
        for _ in range(5):
            od_step(sim, ref, w, True)
        check(sim, ref, w, TOL_NSTEP, err_l1)


def test_od_minimum_grid(pkg, orc):
    w = W.smooth_gas(dims=(4, 4, 4), kmax=1, amp=0.2, components=W.GAS | W.STARS)
    for bc in [(0, 0, 0), (1, 1, 1)]:
        w.bc = bc
        sim, ref = make_pair(pkg, orc, w)
        od_step(sim, ref, w, False)
        check(sim, ref, w, TOL_1STEP, err_max)


@pytest.mark.parametrize("n", [32, 64])
def test_od_step_with_gravity_two_disks(pkg, orc, n):
    w = W.two_disks(n=n, rd_cells=0.1 * n, zd_cells=0.04 * n)
    sim, ref = make_pair(pkg, orc, w)
    od_step(sim, ref, w, False)
    check(sim, ref, w, TOL_1STEP, err_max)
    assert kappa_close(sim.od_last_kappa(), ref.kappa(), 1e-30)
    for _ in range(9):
        od_step(sim, ref, w, True)
    check(sim, ref, w, TOL_NSTEP, err_l1)


def test_od_isolated_collapse(pkg, orc):
    w = W.collapse(n=32)
    sim, ref = make_pair(pkg, orc, w)
    od_step(sim, ref, w, True)
    check(sim, ref, w, TOL_1STEP, err_max)
    for _ in range(5):
        od_step(sim, ref, w, True)
    check(sim, ref, w, TOL_NSTEP, err_l1)


BLK_YY = (slice(0, 2), slice(3, 8), slice(5, 20))       # (z, y, x) blocks of the (32, 12, 10) grid, disjoint from blk
BLK_ZZ = (slice(2, 6), slice(9, 12), slice(5, 20))


def unphysical_state(w):
    """Conserved fields whose total-energy description is NOT physical in a block of cells (rho E - rho v^2/2 < 0,
    n E_xx - n u_x^2 < 0, far from zero), as happens at gas-vacuum borders; the carried fields stay positive."""
    s = w.state()
    blk = (slice(2, 6), slice(3, 8), slice(5, 20))
    if "E" in s:
        kin = 0.5 * (s["mx"] ** 2 + s["my"] ** 2 + s["mz"] ** 2) / s["rho"]
        s["E"][blk] = 0.6 * kin[blk]                       # E < kinetic energy, but positive
        blk2 = (slice(6, 9), slice(3, 8), slice(5, 20))
        s["E"][blk2] = -0.05                               # even E - rho eps < 0: the velocity is zeroed
    if "Exx" in s:
        s["Exx"][blk] = 0.3 * (s["nux"] ** 2 / s["n"])[blk]
        # blocks that violate Pi_yy > 0 ALONE and Pi_zz > 0 ALONE (implied value -0.2): all three diagonals of the
        # condition are exercised (fused_impl.cuh lag epilogue, od.cu k_od_cell)
        s["Eyy"][BLK_YY] = (s["nuy"] ** 2 / s["n"])[BLK_YY] - 0.2
        s["Ezz"][BLK_ZZ] = (s["nuz"] ** 2 / s["n"])[BLK_ZZ] - 0.2
    return s


def carried_from(w, orc):
    """Carried fields of the ORIGINAL (physical) state, from the oracle's derive; in the first block the carried
    internal energy is set below the (too small) total energy, 0.3 x kinetic, so that the gas rule rescales |v| there
    (rho v^2/2 := rho E - rho eps = 0.3 x kinetic); in the second block rho E - rho eps < 0 and the rule zeroes v."""
    ref = orc.Oracle(w.nx, w.ny, w.nz, w.h, w.components, w.poisson, w.G, w.gamma, w.bc)
    s = w.state()
    ref.set_state(s)
    ref.od_enable()
    out = {k: ref.get(k) for k in ref.od_field_names()}
    if "eps" in out:
        kin = 0.5 * (s["mx"] ** 2 + s["my"] ** 2 + s["mz"] ** 2) / s["rho"]
        blk = (slice(2, 6), slice(3, 8), slice(5, 20))
        out["eps"][blk] = 0.3 * kin[blk]
    return out


def test_balance_alone_on_unphysical_cells(pkg, orc):
    w = W.smooth_gas(dims=(32, 12, 10), kmax=2, amp=0.4, components=W.GAS | W.STARS)
    carried = carried_from(w, orc)
    sim, ref = make_pair(pkg, orc, w, perturb=False, state=unphysical_state(w))
    for k, a in carried.items():
        sim.set(k, a)
        ref.set(k, a)
    assert kappa_close(sim.kappa(), ref.kappa(), 1e-30) and min(ref.kappa()) > 1e-4
    sim.od_balance()
    ref.od_balance()
    check(sim, ref, w, 1e-14, err_max)
    # all three branches of the gas rule and both of the collisionless rule were taken
    assert np.any(sim.get("mx")[7, 5, 5:20] == 0.0) and np.all(sim.get("E")[7, 5, 5:20] == carried["eps"][7, 5, 5:20])
    # ... also where Pi_yy or Pi_zz alone is the unphysical one: the carried tensor is kept and all six n E_ij follow it
    for blk in (BLK_YY, BLK_ZZ):
        nn, uu = sim.get("n")[blk], [sim.get(k)[blk] / sim.get("n")[blk] for k in ("nux", "nuy", "nuz")]
        for p, e, (i, j) in zip(PI, ["Exx", "Exy", "Exz", "Eyy", "Eyz", "Ezz"], [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]):
            assert np.array_equal(sim.get(p)[blk], carried[p][blk]), p
            assert np.abs(sim.get(e)[blk] - (carried[p][blk] + nn * uu[i] * uu[j])).max() <= 1e-14, e
    scale = w.h ** 3 * w.cells
    assert max(sim.kappa()) <= 1e-13 * scale


def test_step_with_balance_on_unphysical_cells(pkg, orc):
    """The stages run on the carried (positive) fields where the total-energy description is unphysical, and the
    balance inside the kernel's epilogue repairs the conserved fields; the CFL reduction of an OD context runs on the
    carried fields as well (reading G16)."""
    w = W.smooth_gas(dims=(32, 12, 10), kmax=2, amp=0.4, components=W.GAS | W.STARS)
    carried = carried_from(w, orc)
    sim, ref = make_pair(pkg, orc, w, perturb=False, state=unphysical_state(w))
    for k, a in carried.items():
        sim.set(k, a)
        ref.set(k, a)
    # reading G16: in a GP_OD context the CFL reduction takes the carried (positive) fields, so it yields a dt here,
    # the oracle's; the same state in a base context is rightly reported as unphysical
    dt_g, dt_r = sim.max_dt(w.cfl), ref.max_dt(w.cfl)
    assert abs(dt_g - dt_r) <= 1e-13 * dt_r
    base = pkg.Simulation.from_workload(w)
    base.set_state(unphysical_state(w))
    with pytest.raises(pkg.binding.GpError) as e:
        base.max_dt(w.cfl)
    assert e.value.code == pkg.binding.GP_ERR_STATE
    a = carried["Pyy"].copy()
    a[4, 5, 6] *= -1.0                         # a non-positive CARRIED value is what an OD context reports
    sim.set("Pyy", a)
    with pytest.raises(pkg.binding.GpError):
        sim.max_dt(w.cfl)
    sim.set("Pyy", carried["Pyy"])
    dt = 0.05 * w.h
    # an unbalanced step of a twin pair: the max folded in the kernels' epilogue sees the carried fields too
    sim2, ref2 = make_pair(pkg, orc, w, perturb=False, state=unphysical_state(w))
    for k, a in carried.items():
        sim2.set(k, a)
        ref2.set(k, a)
    sim2.od_step(dt, balance=False)
    ref2.od_step(dt, balance=False)
    dt_g, dt_r = sim2.max_dt(w.cfl), ref2.max_dt(w.cfl)
    assert abs(dt_g - dt_r) <= 1e-13 * dt_r
    sim.od_step(dt, balance=True)
    ref.od_step(dt, balance=False)
    k_pre = ref.kappa()                       # what the two stages left, before the balance
    ref.od_balance()
    check(sim, ref, w, TOL_1STEP, err_max)
    assert kappa_close(sim.od_last_kappa(), k_pre, 1e-30) and min(k_pre) > 1e-4
    # after the balance the state is physical again on both sides: the CFL reductions agree
    dt_g, dt_r = sim.max_dt(w.cfl), ref.max_dt(w.cfl)
    assert abs(dt_g - dt_r) <= 1e-13 * dt_r
    for _ in range(4):
        od_step(sim, ref, w, True)
    check(sim, ref, w, TOL_NSTEP, err_l1)


def test_gp_step_on_an_od_context_is_the_balanced_step(pkg, orc):
    w = W.smooth_gas(dims=(24, 12, 10), kmax=2, components=W.GAS | W.STARS)
    sim, ref = make_pair(pkg, orc, w)
    dt = ref.max_dt(w.cfl)
    sim.step(dt)
    ref.od_step(dt, balance=True)
    check(sim, ref, w, TOL_1STEP, err_max)


def test_balanced_od_run_follows_the_base_scheme(pkg, orc):
    """With derived carried fields and the balance on, the overdetermined run is the base scheme (the oracle pins this
    bit for bit; the CUDA kernels differ by rounding only)."""
    w = W.smooth_gas(dims=(32, 16, 24), kmax=2, amp=0.2, components=W.GAS | W.STARS)
    sim, _ = make_pair(pkg, orc, w, perturb=False)
    base = pkg.Simulation.from_workload(w)
    base.set_state(w.state())
    for _ in range(10):
        dt = base.max_dt(w.cfl)
        base.step(dt)
        sim.step(dt)
    for g in GROUPS_GAS + GROUPS_BME:
        assert err_l1(sim, base, g) <= 1e-12, g


def test_od_calls_need_an_od_context(pkg):
    B = pkg.binding
    sim = pkg.Simulation(8, 8, 8, 0.125, W.GAS)
    for call in (sim.od_derive, sim.od_balance, sim.kappa, sim.od_last_kappa, lambda: sim.od_step(1e-3)):
        with pytest.raises(B.GpError) as e:
            call()
        assert e.value.code == B.GP_ERR_UNSUPPORTED
    with pytest.raises(B.GpError):
        sim.set("eps", np.ones((8, 8, 8)))
    od = pkg.Simulation(8, 8, 8, 0.125, W.GAS | GP_OD)
    od.set_state(W.smooth_gas(dims=(8, 8, 8), kmax=1).state())
    od.od_derive()
    with pytest.raises(B.GpError) as e:
        od.od_last_kappa()
    assert e.value.code == B.GP_ERR_STATE
    with pytest.raises(B.GpError):
        od.set("Pxx", np.ones((8, 8, 8)))       # no collisionless component in this context


def test_od_fields_round_trip(pkg):
    rng = np.random.default_rng(7)
    od = pkg.Simulation(12, 6, 10, 0.1, W.GAS | W.STARS | GP_OD)
    data = {k: rng.uniform(0.5, 1.5, size=(10, 6, 12)) for k in od.field_names() + od.od_field_names()}
    for k, a in data.items():
        od.set(k, a)
    for k, a in data.items():
        assert np.array_equal(od.get(k), a), k


def test_restart_of_an_od_context_needs_its_carried_fields(pkg, orc):
    """Restart path: a GP_OD context whose conserved fields were written without the carried ones (or that was never
    given any) refuses to step, to reduce dt and to balance, instead of running on the pressure of another state;
    once all fields of the saved state are in, it continues bit for bit like the run it was saved from."""
    B = pkg.binding
    w = W.smooth_gas(dims=(24, 12, 10), kmax=2, amp=0.2, components=W.GAS | W.STARS)
    sim, ref = make_pair(pkg, orc, w)
    for _ in range(2):
        od_step(sim, ref, w, False)
    names = sim.field_names() + sim.od_field_names()
    saved = {k: sim.get(k) for k in names}
    fresh = pkg.Simulation(w.nx, w.ny, w.nz, w.h, w.components | GP_OD, w.poisson, w.G, w.gamma, w.bc)
    for call in (lambda: fresh.od_step(1e-3), lambda: fresh.max_dt(w.cfl), fresh.od_balance, lambda: fresh.step(1e-3)):
        with pytest.raises(B.GpError) as e:       # fresh storage: no carried fields at all
            call()
        assert e.value.code == B.GP_ERR_STATE and "stale" in str(e.value)
    for k in sim.field_names():
        fresh.set(k, saved[k])
    with pytest.raises(B.GpError) as e:           # conserved fields only: still stale
        fresh.od_step(1e-3, balance=False)
    assert e.value.code == B.GP_ERR_STATE
    fresh.set("eps", saved["eps"])
    with pytest.raises(B.GpError):                # the gas is complete, the collisionless component is not
        fresh.max_dt(w.cfl)
    for k in PI:
        fresh.set(k, saved[k])
    dt = sim.max_dt(w.cfl)                         # folded by the last step's epilogue
    dt_fresh = fresh.max_dt(w.cfl)                 # stand-alone reduction over the same state (other rounding of the root)
    assert abs(dt_fresh - dt) <= 1e-13 * dt
    fresh.od_step(dt, balance=False)
    sim.od_step(dt, balance=False)
    for k in names:
        assert np.array_equal(fresh.get(k), sim.get(k)), k
    # writing a conserved field afterwards makes that component's carried fields lag again; gp_od_derive clears it
    sim.set("rho", sim.get("rho"))
    with pytest.raises(B.GpError):
        sim.od_step(dt)
    sim.od_derive()
    sim.od_step(dt)
