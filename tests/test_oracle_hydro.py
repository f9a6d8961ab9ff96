"""Pins P3-P8, P12 and the Lagrangian-stage pins: the oracle's hydro step against closed forms,
invariants and textbook special cases."""
import os

import numpy as np
import pytest

from paper_1311_0861_b200 import workloads as W
from tests import exact_riemann as ER

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def make(orc, w):
    o = orc.Oracle(w.nx, w.ny, w.nz, w.h, w.components, w.poisson, w.G, w.gamma, w.bc)
    o.set_state(w.state())
    return o


def run_to(o, w, t_end=None, steps=None):
    t, n = 0.0, 0
    while (t_end is not None and t < t_end * (1 - 1e-14)) or (steps is not None and n < steps):
        dt = o.max_dt(w.cfl)
        if t_end is not None:
            dt = min(dt, t_end - t)
        o.step(dt)
        t += dt
        n += 1
    return t, n


# ------------------------------------------------------------------------------------------------
# the exact Riemann solver used as the yardstick is itself pinned to the quoted textbook values
# ------------------------------------------------------------------------------------------------
def test_exact_riemann_matches_quoted_sod_values():
    ps_ref, us_ref, shock_ref = np.loadtxt(os.path.join(GOLD, "sod_star_state.txt"))
    ps, us = ER.star(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, 1.4)
    assert ps == pytest.approx(ps_ref, abs=5e-6)
    assert us == pytest.approx(us_ref, abs=5e-6)
    shock = np.sqrt(1.4 * 0.1 / 0.125) * np.sqrt(2.4 / 2.8 * ps / 0.1 + 0.4 / 2.8)
    assert shock == pytest.approx(shock_ref, abs=5e-5)


def sod_errors(orc, n):
    w = W.sod(n=n)
    o = make(orc, w)
    t, steps = run_to(o, w, t_end=w.t_end)
    rho, mx, E = o.get("rho")[0, 0], o.get("mx")[0, 0], o.get("E")[0, 0]
    u = mx / rho
    p = (w.gamma - 1) * (E - 0.5 * rho * u * u)
    x = (np.arange(n) + 0.5) * w.h
    re, ue, pe = ER.sample((x - 0.5) / t, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, w.gamma)
    return [np.abs(a - b).mean() for a, b in ((rho, re), (u, ue), (p, pe))], steps


def test_P4_sod_converges_to_exact_solution(orc):
    """Config 1 against the exact Riemann solution: first-order convergence (L1 error falls
    monotonically under refinement) and the N=128 errors sit where a first-order scheme's do."""
    e128, steps = sod_errors(orc, 128)
    e256, _ = sod_errors(orc, 256)
    e512, _ = sod_errors(orc, 512)
    assert steps == 274                      # CFL 0.2 to t = 0.2 takes 274 steps
    for a, b, c in zip(e128, e256, e512):
        assert b < 0.75 * a and c < 0.75 * b
    assert e128[0] < 2.5e-2 and e128[1] < 4.5e-2 and e128[2] < 2.5e-2
    # plateau values between the contact and the shock
    w = W.sod(n=512)
    o = make(orc, w)
    run_to(o, w, t_end=0.2)
    rho, mx, E = o.get("rho")[0, 0], o.get("mx")[0, 0], o.get("E")[0, 0]
    i = int((0.5 + 0.5 * (0.92745 + 1.7522) * 0.2) * 512)     # midway between contact and shock
    u = mx[i] / rho[i]
    assert u == pytest.approx(0.92745, abs=5e-3)
    assert 0.4 * (E[i] - 0.5 * rho[i] * u * u) == pytest.approx(0.30313, abs=3e-3)


@pytest.mark.parametrize("left,right,t_end", [
    ((2.0, 0.0, 2.0), (1.0, 0.0, 1.0), 0.2),          # PAPER.md:497-508, Table 2 test 1
    ((1.0, -2.0, 0.4), (1.0, 2.0, 0.4), 0.15),        # test 2
    ((1.0, 0.0, 1000.0), (1.0, 0.0, 0.01), 0.012),    # test 3
])
def test_P5_table2_shock_tubes(orc, left, right, t_end):
    errs = []
    for n in (128, 256):
        w = W.sod(n=n, left=left, right=right, t_end=t_end)
        o = make(orc, w)
        t, _ = run_to(o, w, t_end=t_end)
        rho = o.get("rho")[0, 0]
        assert np.all(rho > 0)
        x = (np.arange(n) + 0.5) * w.h
        re, _, _ = ER.sample((x - 0.5) / t, *left, *right, w.gamma)
        errs.append(np.abs(rho - re).mean() / np.abs(re).mean())
    assert errs[1] < 0.8 * errs[0]
    # test 1 is mild; test 2's near-vacuum centre and test 3's thin dense shell (6x compression
    # over ~2% of the tube) are smeared by a first-order scheme at N=128
    assert errs[0] < (0.25 if left[2] > 100 else (0.1 if left[1] < 0 else 0.03))


def test_P3_bme_tube_equals_gamma3_gas_tube(orc):
    """A 1-D collisionless problem's (n, n u_d, nE_dd) is a gamma = 3 gas problem's
    (rho, rho v, 2 rho E): same wave speed (PAPER.md:86 vs 140), same face formulas."""
    for axis in range(3):
        wg = W.sod(n=64, axis=axis, gamma=3.0, components=W.GAS)
        ws = W.sod(n=64, axis=axis, gamma=3.0, components=W.STARS)
        og, os_ = make(orc, wg), make(orc, ws)
        for _ in range(60):
            dtg, dts = og.max_dt(0.2), os_.max_dt(0.2)
            assert dts == pytest.approx(dtg, rel=1e-14)
            og.step(dtg)
            os_.step(dtg)
        mom = ["mx", "my", "mz"][axis], ["nux", "nuy", "nuz"][axis]
        ed = ["Exx", "Eyy", "Ezz"][axis]
        assert np.allclose(os_.get("n"), og.get("rho"), rtol=1e-13, atol=0)
        assert np.allclose(os_.get(mom[1]), og.get(mom[0]), rtol=1e-12, atol=1e-14)
        assert np.allclose(os_.get(ed), 2.0 * og.get("E"), rtol=1e-13, atol=0)


def total(o, name):
    return o.get(name).sum()


def test_P6_conservation_periodic_no_gravity(orc):
    """'The mass of gas and total impulse are conserved because of the selected numerical
    scheme': with periodic boundaries every conserved field's sum is constant
    to round-off (flux form of both stages)."""
    w = W.smooth_gas(n=16, kmax=2, amp=0.3, components=W.GAS | W.STARS, cfl=0.3)
    o = make(orc, w)
    names = o.field_names()
    t0 = {k: total(o, k) for k in names}
    scale = {k: np.abs(o.get(k)).sum() for k in names}
    run_to(o, w, steps=40)
    for k in names:
        assert abs(total(o, k) - t0[k]) <= 2e-14 * scale[k], k
    assert np.abs(o.get("rho") - w.state()["rho"]).max() > 1e-3      # the state did evolve


def test_P6_momentum_conserved_with_periodic_gravity(orc):
    """Centred gradient of the inverse 27-point Laplacian is antisymmetric, so with the source
    rho + n also being the density the force acts on, total momentum (gas + stars) is conserved
    and mass is untouched."""
    w = W.disk(n=32, rd_cells=4.0, zd_cells=1.5, background=1e-2, steps=10)
    o = make(orc, w)
    m0 = total(o, "rho"), total(o, "n")
    p0 = np.array([total(o, a) + total(o, b) for a, b in (("mx", "nux"), ("my", "nuy"), ("mz", "nuz"))])
    pscale = sum(np.abs(o.get(k)).sum() for k in ("mx", "my", "nux", "nuy"))
    for _ in range(10):
        o.solve_poisson()
        o.step(o.max_dt(0.2))
    assert abs(total(o, "rho") - m0[0]) <= 1e-13 * m0[0]
    assert abs(total(o, "n") - m0[1]) <= 1e-13 * m0[1]
    p1 = np.array([total(o, a) + total(o, b) for a, b in (("mx", "nux"), ("my", "nuy"), ("mz", "nuz"))])
    assert np.abs(p1 - p0).max() <= 1e-12 * pscale


def test_P7_tube_is_the_same_along_x_y_z(orc):
    prof = {}
    for comp in (W.GAS, W.STARS):
        for axis in range(3):
            w = W.sod(n=48, nt=4, axis=axis, components=comp)
            o = make(orc, w)
            for _ in range(30):
                o.step(o.max_dt(0.2))
            a = o.get("rho" if comp == W.GAS else "n")
            a = np.moveaxis(a, 2 - axis, -1)            # tube axis last
            assert np.all(a == a[0:1, 0:1, :])          # no transverse variation, bitwise
            prof[(comp, axis)] = a[0, 0]
        for axis in (1, 2):
            assert np.allclose(prof[(comp, axis)], prof[(comp, 0)], rtol=2e-15, atol=0)


def test_P7_blast_keeps_mirror_and_permutation_symmetry(orc):
    n = 16
    h = 1.0 / n
    x = (np.arange(n) + 0.5) * h - 0.5
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    r2 = X * X + Y * Y + Z * Z
    rho = 1.0 + 2.0 * np.exp(-r2 / 0.02)
    p = 1.0 + 20.0 * np.exp(-r2 / 0.02)
    zero = np.zeros_like(rho)
    for comp in (W.GAS, W.STARS):
        o = orc.Oracle(n, n, n, h, comp, gamma=1.4)
        if comp == W.GAS:
            o.set_state(W._pack_gas(rho, zero, zero, zero, p, 1.4))
            names = ("rho", "mx", "my", "mz", "E")
        else:
            o.set_state(W._pack_stars(rho, [zero, zero, zero], [p, zero, zero, p, zero, p]))
            names = ("n", "nux", "nuy", "nuz", "Exx")
        for _ in range(12):
            o.step(o.max_dt(0.3))
        d, mx, my, mz = (o.get(k) for k in names[:4])
        tol = 1e-13 * np.abs(mx).max()
        assert np.abs(mx).max() > 1e-2
        assert np.allclose(d, d[::-1, :, :], rtol=1e-13) and np.allclose(d, d[:, :, ::-1], rtol=1e-13)
        assert np.allclose(mx, -mx[:, :, ::-1], atol=tol)                      # mirror in x
        assert np.allclose(d, d.transpose(2, 1, 0), rtol=1e-13)                # swap x <-> z
        assert np.allclose(mx, mz.transpose(2, 1, 0), atol=tol)
        assert np.allclose(my, mx.transpose(0, 2, 1), atol=tol)                # swap x <-> y
        if comp == W.STARS:
            exy, eyz = o.get("Exy"), o.get("Eyz")
            assert np.abs(exy).max() > 1e-6                                    # shear stress did develop
            assert np.allclose(o.get("Exz"), o.get("Exz").transpose(2, 1, 0), atol=1e-13)   # xz symmetric under x<->z
            assert np.allclose(exy, eyz.transpose(2, 1, 0), atol=1e-13)        # x<->z maps xy -> zy


def test_P8_uniform_gravity_leaves_pressure_and_stress_unchanged(orc):
    n = 8
    h = 0.1
    g = np.array([0.3, -0.7, 0.45])
    x = (np.arange(n) + 0.5) * h
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    phi = g[0] * X + g[1] * Y + g[2] * Z
    one = np.ones_like(phi)
    o = orc.Oracle(n, n, n, h, W.GAS | W.STARS, gamma=5 / 3)
    Pi0 = [1.1, 0.2, -0.1, 0.9, 0.05, 1.3]
    st = W._pack_gas(1.3 * one, 0.2 * one, -0.4 * one, 0.1 * one, 0.7 * one, 5 / 3)
    st.update(W._pack_stars(0.8 * one, [0.3 * one, 0.1 * one, -0.2 * one], [P * one for P in Pi0]))
    o.set_state(st)
    o.set("phi", phi)
    dt = 0.05
    o.step(dt)
    s = (slice(2, -2),) * 3                      # away from the (periodic) jump of the linear potential
    rho, E = o.get("rho")[s], o.get("E")[s]
    v = [o.get(k)[s] / rho for k in ("mx", "my", "mz")]
    for d in range(3):
        assert np.allclose(v[d], [0.2, -0.4, 0.1][d] - dt * g[d], rtol=0, atol=1e-15)     # the kick
    p = (5 / 3 - 1) * (E - 0.5 * rho * sum(a * a for a in v))
    assert np.allclose(p, 0.7, rtol=0, atol=2e-15)
    nn = o.get("n")[s]
    u = [o.get(k)[s] / nn for k in ("nux", "nuy", "nuz")]
    pairs = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]
    for name, (i, j), P in zip(W.STAR_FIELDS[4:], pairs, Pi0):
        assert np.allclose(o.get(name)[s] - nn * u[i] * u[j], P, rtol=0, atol=3e-15), name


# ------------------------------------------------------------------------------------------------
# Lagrangian stage alone
# ------------------------------------------------------------------------------------------------
def test_lagrangian_uniform_velocity_is_donor_cell_upwind(orc):
    """With a uniform velocity the 18-cell face velocity is that velocity, and (124)+(128)
    reduce to the textbook first-order donor-cell scheme, here written with np.roll."""
    n = 12
    h = 1.0 / n
    rng = np.random.default_rng(5)
    rho = rng.uniform(0.5, 2.0, (n, n, n))
    vel = np.array([0.7, -0.4, 0.25])
    one = np.ones_like(rho)
    o = orc.Oracle(n, n, n, h, W.GAS, gamma=1.4)
    o.set_state(W._pack_gas(rho, vel[0] * one, vel[1] * one, vel[2] * one, one, 1.4))
    dt = 0.3 * h
    o.lagrangian_only(dt)
    for name in ("rho", "mx", "E"):
        f = W._pack_gas(rho, vel[0] * one, vel[1] * one, vel[2] * one, one, 1.4)[name]
        ref = f.copy()
        for d, ax in ((0, 2), (1, 1), (2, 0)):          # array axes are (z, y, x)
            if vel[d] > 0:
                ref -= dt / h * vel[d] * (f - np.roll(f, 1, axis=ax))
            else:
                ref -= dt / h * vel[d] * (np.roll(f, -1, axis=ax) - f)
        assert np.allclose(o.get(name), ref, rtol=1e-13, atol=1e-15), name


def test_lagrangian_face_velocity_weights(orc):
    """Reading G2: vertex velocity = mean of 8 cells, face velocity = mean of 4 vertices.  For a
    velocity that is a polynomial in the transverse coordinates this has a closed form:
    linear -> the value at the face centre; y^2 -> y^2 + h^2/2 (weights 1/4,1/2,1/4).  Checked
    through the mass flux of a uniform-density gas: rho' = 1 - dt * (discrete divergence)."""
    n = 16
    h = 1.0
    x = np.arange(n) + 0.5
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    one = np.ones_like(X)
    dt = 0.01
    s = (slice(3, -3),) * 3
    # v_x = a*y^2 + b*z + c*x: div of face-averaged v = c exactly (the y^2 + h^2/2 terms cancel across x-faces)
    o = orc.Oracle(n, n, n, h, W.GAS, gamma=1.4, bc=(W.BC_OUTFLOW,) * 3)
    o.set_state(W._pack_gas(one, 0.01 * Y * Y + 0.02 * Z + 0.03 * X + 1.0, 0 * one, 0 * one, one, 1.4))
    o.lagrangian_only(dt)
    assert np.allclose(o.get("rho")[s], 1.0 - dt * 0.03, rtol=0, atol=1e-15)
    # a density step across an x-face makes the face velocity itself visible:
    # cell left of the step at i0 loses dt/h * w_f * rho_L through its right face and gains through its left.
    rho = np.where(X < 8.0, 2.0, 1.0)
    vx = 0.01 * Y * Y + 0.5
    o.set_state(W._pack_gas(rho, vx, 0 * one, 0 * one, one, 1.4))
    o.lagrangian_only(dt)
    got = o.get("rho")
    wf = 0.01 * (Y * Y + 0.5 * h * h) + 0.5                  # closed form of the 18-cell average at an x-face
    # cell i=8 (first cell right of the step): inflow w_f*2 through its left face, outflow w_f*1 through its right
    exp8 = 1.0 - dt / h * (wf[:, :, 8] * 1.0 - wf[:, :, 8] * 2.0)
    assert np.allclose(got[3:-3, 3:-3, 8], exp8[3:-3, 3:-3], rtol=0, atol=1e-15)


def test_lagrangian_upwind_side_follows_sign(orc):
    n = 8
    h = 1.0
    rho = np.ones((n, n, n))
    rho[:, :, 4] = 3.0
    one = np.ones_like(rho)
    for sgn in (+1.0, -1.0):
        o = orc.Oracle(n, n, n, h, W.GAS, gamma=1.4)
        o.set_state(W._pack_gas(rho, sgn * 0.5 * one, 0 * one, 0 * one, one, 1.4))
        o.lagrangian_only(0.1)
        r = o.get("rho")[0, 0]
        down = 5 if sgn > 0 else 3
        assert r[4] == pytest.approx(3.0 - 0.1 * 0.5 * 2.0, rel=1e-15)
        assert r[down] == pytest.approx(1.0 + 0.1 * 0.5 * 2.0, rel=1e-15)
        assert r[8 - down] == pytest.approx(1.0, rel=1e-15)


# ------------------------------------------------------------------------------------------------
# Eulerian stage alone
# ------------------------------------------------------------------------------------------------
def test_eulerian_stage_by_hand_on_one_jump(orc):
    """One x-face with a pressure jump: momentum and energy of the two adjacent cells change by
    the face values of (112)/(114); density is untouched."""
    n = 8
    h = 0.5
    g = 1.4
    one = np.ones((n, n, n))
    rho = np.where(np.arange(n)[None, None, :] < 4, 1.0, 0.125) * one
    p = np.where(np.arange(n)[None, None, :] < 4, 1.0, 0.1) * one
    o = orc.Oracle(n, n, n, h, W.GAS, gamma=g, bc=(W.BC_OUTFLOW, W.BC_PERIODIC, W.BC_PERIODIC))
    o.set_state(W._pack_gas(rho, 0 * one, 0 * one, 0 * one, p, g))
    dt = 0.1
    o.eulerian(dt)
    Z = np.sqrt(1.0 * 0.125 * g * 1.1 / 1.125)
    V, P = 0.45 / Z, 0.55
    assert np.array_equal(o.get_star("rho"), rho)
    mx, E = o.get_star("mx")[0, 0], o.get_star("E")[0, 0]
    assert mx[3] == pytest.approx(-dt / h * (P - 1.0), rel=1e-14)
    assert mx[4] == pytest.approx(-dt / h * (0.1 - P), rel=1e-14)
    assert E[3] == pytest.approx(1.0 / 0.4 - dt / h * (P * V), rel=1e-14)
    assert E[4] == pytest.approx(0.1 / 0.4 + dt / h * (P * V), rel=1e-14)
    assert np.all(mx[[0, 1, 2, 5, 6, 7]] == 0.0)


def test_P11_hydrostatic_sphere_balance(orc):
    """rho0 = 1 - r with the printed p0(r) and Phi0(r) is an equilibrium, so the
    Eulerian-stage momentum change -grad P - rho grad Phi vanishes at second order in h."""
    res = []
    for n in (32, 64):
        L = 2.4
        h = L / n
        x = (np.arange(n) + 0.5) * h - L / 2
        Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
        r = np.sqrt(X * X + Y * Y + Z * Z)
        rho = np.maximum(1.0 - r, 1e-3)
        p = np.where(r <= 1, -np.pi * r * r / 36 * (9 * r * r - 28 * r + 24) + 5 * np.pi / 36, 0.0) + 1e-3
        phi = np.where(r <= 1, -np.pi / 3 * (r ** 3 - 2 * r * r) - 2 * np.pi / 3, -np.pi / (3 * np.maximum(r, 1e-9)))
        zero = np.zeros_like(r)
        o = orc.Oracle(n, n, n, h, W.GAS, gamma=5 / 3, bc=(W.BC_OUTFLOW,) * 3)
        o.set_state(W._pack_gas(rho, zero, zero, zero, p, 5 / 3))
        o.set("phi", phi)
        dt = 1e-3
        o.eulerian(dt)
        force = np.sqrt(sum(o.get_star(k) ** 2 for k in ("mx", "my", "mz"))) / dt
        inside = r < 0.85
        gravity = (rho * np.pi / 3 * np.abs(3 * r * r - 4 * r))[inside].max()
        res.append(force[inside].max() / gravity)
    assert res[0] < 0.05
    assert res[1] < 0.3 * res[0]               # second order: 4x smaller per halving of h


def test_P12_aksenov_smooth_flow(orc):
    """gamma = 3, rho = 1 + 0.5 cos x, u = 0, p = rho^3/3 on [0, 2 pi]; at
    t = pi/2 the exact solution is rho = 1 and u = 0.5 sin(x - u t).  First-order convergence."""
    errs = []
    for n in (64, 128, 256):
        h = 2 * np.pi / n
        x = (np.arange(n) + 0.5) * h
        rho = (1.0 + 0.5 * np.cos(x))[None, None, :] * np.ones((4, 4, n))
        o = orc.Oracle(n, 4, 4, h, W.GAS, gamma=3.0)
        zero = np.zeros_like(rho)
        o.set_state(W._pack_gas(rho, zero, zero, zero, rho ** 3 / 3.0, 3.0))
        t, t_end = 0.0, np.pi / 2
        while t < t_end * (1 - 1e-14):
            dt = min(o.max_dt(0.2), t_end - t)
            o.step(dt)
            t += dt
        u = (o.get("mx") / o.get("rho"))[0, 0]
        ue = np.zeros(n)
        for _ in range(200):
            ue = 0.5 * np.sin(x - ue * t_end)
        errs.append(np.abs(u - ue).mean())
    assert errs[0] < 0.05
    assert errs[1] < 0.7 * errs[0] and errs[2] < 0.7 * errs[1]


def test_P13_cfl_is_the_brute_force_max(orc):
    w = W.smooth_gas(n=16, kmax=2, amp=0.3, components=W.GAS | W.STARS)
    o = make(orc, w)
    st = w.state()
    rho = st["rho"]
    v = [st[k] / rho for k in ("mx", "my", "mz")]
    p = (w.gamma - 1) * (st["E"] - 0.5 * rho * sum(a * a for a in v))
    s_gas = max((np.abs(a) + np.sqrt(w.gamma * p / rho)).max() for a in v)
    n = st["n"]
    u = [st[k] / n for k in ("nux", "nuy", "nuz")]
    s_st = max((np.abs(u[d]) + np.sqrt(3 * (st[e] - n * u[d] * u[d]) / n)).max() for d, e in enumerate(("Exx", "Eyy", "Ezz")))
    assert o.max_dt(0.3) == pytest.approx(0.3 * w.h / max(s_gas, s_st), rel=1e-14)
    # a non-positive pressure is reported, never clamped (reading G10)
    bad = st["E"].copy()
    bad[3, 4, 5] = 0.0
    o.set("E", bad)
    with pytest.raises(orc.OracleError) as e:
        o.max_dt(0.3)
    assert e.value.code == orc.ERR_STATE


def test_P14_get_set_round_trip_is_bit_exact(orc):
    w = W.smooth_gas(n=16, kmax=2, components=W.GAS | W.STARS)
    a, b = make(orc, w), make(orc, w)
    a.step(1e-3)
    b.step(1e-3)
    c = orc.Oracle(w.nx, w.ny, w.nz, w.h, w.components, w.poisson, w.G, w.gamma, w.bc)
    c.set_state(a.get_state())
    a.step(1e-3)
    c.step(1e-3)
    for k in a.field_names():
        assert np.array_equal(a.get(k), c.get(k))
