"""The paper's own verification problems run through the CUDA path (pytest -m gpu), SURVEY.md 8(f)-2:
Godunov tubes of Table 2, the collisionless tube (reading G9),
the Aksenov test and the equilibrium sphere rho = 1 - r.

Each problem is checked twice: against the CPU oracle on every step (same bars as test_gpu_parity.py)
and against what the paper fixes in closed form (exact Riemann solution, the implicit Aksenov
solution, the printed Phi_0(r) and the hydrostatic balance), with the acceptance the oracle's own
pins use (tests/test_oracle_hydro.py).
"""
import numpy as np
import pytest

from paper_1311_0861_b200 import workloads as W
from tests import exact_riemann as ER

pytestmark = pytest.mark.gpu

TOL_1STEP, TOL_NSTEP = 1e-11, 1e-8


@pytest.fixture(scope="module")
def pkg():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1311_0861_b200 as p
    p.lib()
    return p


def pair(pkg, orc, nx, ny, nz, h, comps, state, gamma, bc, poisson=0, G=1.0):
    sim = pkg.Simulation(nx, ny, nz, h, comps, poisson, G=G, gamma=gamma, bc=bc)
    ref = orc.Oracle(nx, ny, nz, h, comps, poisson, G, gamma, bc)
    sim.set_state(state)
    ref.set_state(state)
    return sim, ref


def worst(sim, ref, names, l1=False):
    if l1:
        return sum(np.abs(sim.get(k) - ref.get(k)).sum() for k in names) / sum(np.abs(ref.get(k)).sum() for k in names)
    return max(np.abs(sim.get(k) - ref.get(k)).max() for k in names) / max(np.abs(ref.get(k)).max() for k in names)


def march(sim, ref, cfl, t_end, groups):
    """Both sides to t_end with the oracle's dt (last step clipped); parity after step 1 and at the end."""
    t, n = 0.0, 0
    while t < t_end * (1 - 1e-14):
        dt_g, dt_r = sim.max_dt(cfl), ref.max_dt(cfl)
        assert abs(dt_g - dt_r) <= 1e-13 * dt_r
        dt = min(dt_r, t_end - t)
        sim.step(dt)
        ref.step(dt)
        if n == 0:
            for g in groups:
                assert worst(sim, ref, g) <= TOL_1STEP, g
        t += dt
        n += 1
    for g in groups:
        assert worst(sim, ref, g, l1=True) <= TOL_NSTEP, g
    return t, n


GAS_GROUPS = [("rho",), ("mx", "my", "mz"), ("E",)]
BME_GROUPS = [("n",), ("nux", "nuy", "nuz"), ("Exx", "Exy", "Exz", "Eyy", "Eyz", "Ezz")]


@pytest.mark.parametrize("left,right,t_end,bound", [
    ((2.0, 0.0, 2.0), (1.0, 0.0, 1.0), 0.2, 0.03),          # PAPER.md:497-508, Table 2 test 1
    ((1.0, -2.0, 0.4), (1.0, 2.0, 0.4), 0.15, 0.1),         # test 2
    ((1.0, 0.0, 1000.0), (1.0, 0.0, 0.01), 0.012, 0.25),    # test 3
])
def test_table2_godunov_tubes(pkg, orc, left, right, t_end, bound):
    w = W.sod(n=128, left=left, right=right, t_end=t_end)
    sim, ref = pair(pkg, orc, w.nx, w.ny, w.nz, w.h, w.components, w.state(), w.gamma, w.bc)
    t, _ = march(sim, ref, w.cfl, t_end, GAS_GROUPS)
    rho = sim.get("rho")
    assert np.all(rho > 0) and np.all(rho == rho[0:1, 0:1, :])
    x = (np.arange(w.nx) + 0.5) * w.h
    re, _, _ = ER.sample((x - 0.5) / t, *left, *right, w.gamma)
    assert np.abs(rho[0, 0] - re).mean() / np.abs(re).mean() < bound


def test_collisionless_tube_reading_G9(pkg, orc):
    """PAPER.md:231 as read in DESIGN.md G9: left n = 2, Pi = (2,1,1,1,1,1); right n = 1, Pi = 1; u = 0.
    Its (n, n u_x, nE_xx) must equal (rho, rho v, 2 rho E) of the gamma = 3 gas tube with p = Pi_xx
    (same wave speed, PAPER.md:86 vs 140), which in turn follows the exact Riemann solution."""
    n, nt, t_end = 128, 4, 0.15
    h = 1.0 / n
    x = (np.arange(n) + 0.5) * h
    L = np.broadcast_to((x < 0.5)[None, None, :], (nt, nt, n))
    dens = np.where(L, 2.0, 1.0)
    one, zero = np.ones_like(dens), np.zeros_like(dens)
    Pi = [np.where(L, 2.0, 1.0), one, one, one, one, one]
    bc = (W.BC_OUTFLOW, W.BC_PERIODIC, W.BC_PERIODIC)
    stars = W._pack_stars(dens, [zero, zero, zero], Pi)
    gas = W._pack_gas(dens, zero, zero, zero, Pi[0], 3.0)
    sim, ref = pair(pkg, orc, n, nt, nt, h, W.STARS, stars, 3.0, bc)
    gsim, gref = pair(pkg, orc, n, nt, nt, h, W.GAS, gas, 3.0, bc)
    t, steps = march(sim, ref, 0.2, t_end, BME_GROUPS)
    tg, gsteps = march(gsim, gref, 0.2, t_end, GAS_GROUPS)
    assert steps == gsteps and abs(t - tg) <= 1e-12
    assert np.allclose(sim.get("n"), gsim.get("rho"), rtol=1e-12, atol=0)
    assert np.allclose(sim.get("nux"), gsim.get("mx"), rtol=1e-11, atol=1e-13)
    assert np.allclose(sim.get("Exx"), 2.0 * gsim.get("E"), rtol=1e-12, atol=0)
    re, _, _ = ER.sample((x - 0.5) / t, 2.0, 0.0, 2.0, 1.0, 0.0, 1.0, 3.0)
    assert np.abs(sim.get("n")[0, 0] - re).mean() / re.mean() < 0.05


def test_aksenov_smooth_periodic_flow(pkg, orc):
    """gamma = 3, rho = 1 + 0.5 cos x, u = 0, p = rho^3/3 on [0, 2 pi]; at t = pi/2
    rho = 1 and u solves u = 0.5 sin(x - u t)."""
    n = 128
    h = 2 * np.pi / n
    x = (np.arange(n) + 0.5) * h
    rho = (1.0 + 0.5 * np.cos(x))[None, None, :] * np.ones((4, 4, n))
    zero = np.zeros_like(rho)
    st = W._pack_gas(rho, zero, zero, zero, rho ** 3 / 3.0, 3.0)
    sim, ref = pair(pkg, orc, n, 4, 4, h, W.GAS, st, 3.0, (0, 0, 0))
    t_end = np.pi / 2
    march(sim, ref, 0.2, t_end, GAS_GROUPS)
    u = (sim.get("mx") / sim.get("rho"))[0, 0]
    ue = np.zeros(n)
    for _ in range(200):
        ue = 0.5 * np.sin(x - ue * t_end)
    assert np.abs(u - ue).mean() < 0.035
    assert np.abs(sim.get("rho")[0, 0] - 1.0).mean() < 0.05


def sphere(n, L=2.4):
    h = L / n
    x = (np.arange(n) + 0.5) * h - L / 2
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    r = np.sqrt(X * X + Y * Y + Z * Z)
    phi0 = np.where(r <= 1, -np.pi / 3 * (r ** 3 - 2 * r * r) - 2 * np.pi / 3, -np.pi / (3 * np.maximum(r, 1e-9)))
    p0 = np.where(r <= 1, -np.pi * r * r / 36 * (9 * r * r - 28 * r + 24) + 5 * np.pi / 36, 0.0)
    return h, r, phi0, p0


def test_equilibrium_sphere_potential_and_balance(pkg, orc):
    """rho_0 = 1 - r with the printed Phi_0(r) and p_0(r).  The isolated solve must
    reach Phi_0 at second order, and a step from the equilibrium must leave it at rest up to the
    truncation error of the pressure and potential gradients."""
    errs = []
    for n in (32, 64):
        h, r, phi0, _ = sphere(n)
        s = pkg.Simulation(n, n, n, h, pkg.GP_GAS, pkg.GP_POISSON_ISOLATED, G=1.0, bc=(1, 1, 1))
        s.set("rho", np.maximum(1.0 - r, 0.0))
        s.solve_poisson()
        errs.append(np.abs(s.get("phi") - phi0).max() / np.abs(phi0).max())
    assert errs[1] < 1.5e-3 and errs[0] > 3.0 * errs[1]
    n = 64
    h, r, phi0, p0 = sphere(n)
    rho = np.maximum(1.0 - r, 1e-3)
    zero = np.zeros_like(r)
    st = W._pack_gas(rho, zero, zero, zero, p0 + 1e-3, 5 / 3)
    sim, ref = pair(pkg, orc, n, n, n, h, W.GAS, st, 5 / 3, (1, 1, 1))
    sim.set("phi", phi0)
    ref.set("phi", phi0)
    dt = 1e-3
    sim.step(dt)
    ref.step(dt)
    for g in GAS_GROUPS:
        assert worst(sim, ref, g) <= TOL_1STEP, g
    force = np.sqrt(sum(sim.get(k) ** 2 for k in ("mx", "my", "mz"))) / dt
    inside = r < 0.85
    gravity = (rho * np.pi / 3 * np.abs(3 * r * r - 4 * r))[inside].max()
    assert force[inside].max() / gravity < 0.02
