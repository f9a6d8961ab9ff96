"""Pins of the overdetermined system the oracle carries as an extension: rho*eps beside rho*E
(4th equation), Pi_ij beside n*E_ij, the correctness check kappa and the
build's own energy-balance rule (PAPER.md:202 cites it only; G15).  Closed forms and invariants only."""
import numpy as np
import pytest

from paper_1311_0861_b200 import workloads as W

PAIRS = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]
PN = ["Pxx", "Pxy", "Pxz", "Pyy", "Pyz", "Pzz"]
EN = ["Exx", "Exy", "Exz", "Eyy", "Eyz", "Ezz"]


def make(orc, w):
    o = orc.Oracle(w.nx, w.ny, w.nz, w.h, w.components, w.poisson, w.G, w.gamma, w.bc)
    o.set_state(w.state())
    return o


def test_enable_derives_the_carried_fields_and_kappa_is_zero(orc):
    w = W.smooth_gas(n=12, kmax=2, amp=0.3, components=W.GAS | W.STARS)
    o = make(orc, w)
    o.od_enable()
    st = w.state()
    v2 = sum(st[k] ** 2 for k in ("mx", "my", "mz")) / st["rho"] ** 2
    assert np.allclose(o.get("eps"), st["E"] - 0.5 * st["rho"] * v2, rtol=1e-15)
    u = [st[k] / st["n"] for k in ("nux", "nuy", "nuz")]
    for name, e, (i, j) in zip(PN, EN, PAIRS):
        assert np.allclose(o.get(name), st[e] - st["n"] * u[i] * u[j], rtol=1e-14, atol=1e-16)
    kg, kb = o.kappa()
    assert kg <= 1e-15 * np.abs(st["E"]).sum() * w.h ** 3 and kb <= 1e-15 * np.abs(st["Exx"]).sum() * w.h ** 3


def test_kappa_is_the_riemann_sum_of_the_printed_integrands(orc):
    """PAPER.md:198-200 by hand: perturb rho*eps in one cell and Pi_xy in another."""
    w = W.smooth_gas(n=8, kmax=1, amp=0.2, components=W.GAS | W.STARS)
    o = make(orc, w)
    o.od_enable()
    eps = o.get("eps")
    eps[1, 2, 3] += 0.25
    o.set("eps", eps)
    pxy = o.get("Pxy")
    pxy[4, 5, 6] -= 0.5
    o.set("Pxy", pxy)
    kg, kb = o.kappa()
    assert kg == pytest.approx(0.25 * w.h ** 3, rel=1e-12)
    assert kb == pytest.approx(0.5 * w.h ** 3, rel=1e-12)


def test_balanced_overdetermined_step_is_the_base_scheme_bit_for_bit(orc):
    """Where the total-energy description is physical the balance resets rho*eps and Pi_ij from it after every step, so
    the pressure and the dispersion tensor the next step takes from the carried fields are those the base scheme derives:
    both runs must agree bit for bit (gas + collisionless component, with gravity)."""
    w = W.two_disks(n=16, rd_cells=3.2, zd_cells=1.28)
    a, b = make(orc, w), make(orc, w)
    b.od_enable()
    for _ in range(4):
        a.solve_poisson()
        b.solve_poisson()
        dt = a.max_dt(w.cfl)
        a.step(dt)
        b.od_step(dt, balance=True)
    for k in a.field_names():
        assert np.array_equal(a.get(k), b.get(k)), k
    kg, kb = b.kappa()                       # round-off of E - (E - k) - k only
    assert kg <= 1e-15 * np.abs(a.get("E")).sum() * w.h ** 3 and kb <= 1e-15 * np.abs(a.get("Exx")).sum() * w.h ** 3


@pytest.mark.parametrize("rates", [(0.3, 0.0, 0.0), (0.0, -0.2, 0.0), (0.1, 0.2, -0.4)])
def test_internal_energy_under_uniform_compression_closed_form(orc, rates):
    """Uniform rho and p, v_d = -a_d x_d: every face velocity of PAPER.md:112 is the plain mean (pL = pR), so
    div V = -(a_x + a_y + a_z) exactly and PAPER.md:41 (4th equation, Eulerian stage) gives
    (rho eps)* = rho eps (1 + tau (gamma-1) sum a_d); the total energy changes by -tau/h sum delta(P V) with P = p."""
    n, h, g, tau, p0, rho0 = 10, 0.1, 1.4, 0.01, 2.0, 1.5
    x = (np.arange(n) + 0.5) * h
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    one = np.ones_like(X)
    v = [-rates[0] * X, -rates[1] * Y, -rates[2] * Z]
    o = orc.Oracle(n, n, n, h, W.GAS, gamma=g, bc=(W.BC_OUTFLOW,) * 3)
    o.set_state(W._pack_gas(rho0 * one, v[0], v[1], v[2], p0 * one, g))
    o.od_enable()
    o.od_eulerian(tau)
    inner = (slice(1, -1),) * 3
    eps0 = p0 / (g - 1)
    assert np.allclose(o.get_star("eps")[inner], eps0 * (1 + tau * (g - 1) * sum(rates)), rtol=1e-13)
    # gravity does not enter the 4th equation: a uniform pull leaves (rho eps)* where it was
    o.set("phi", 0.7 * X + 0.2 * Z)
    o.od_eulerian(tau)
    assert np.allclose(o.get_star("eps")[inner], eps0 * (1 + tau * (g - 1) * sum(rates)), rtol=1e-13)


def test_dispersion_tensor_under_linear_shear_and_compression_closed_form(orc):
    """Uniform n and isotropic Pi = p, u = (-a x, s x, 0): the face velocities of PAPER.md:170-172 are plain means, so
    PAPER.md:65 (Eulerian stage) gives Pi_xx* = p (1 + 2 tau a), Pi_xy* = -tau p s, the rest unchanged to first order in
    tau; none of them feels gravity."""
    n, h, tau, p0, n0, a, s = 10, 0.1, 0.01, 2.0, 1.5, 0.3, 0.4
    x = (np.arange(n) + 0.5) * h
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    one, zero = np.ones_like(X), np.zeros_like(X)
    o = orc.Oracle(n, n, n, h, W.STARS, bc=(W.BC_OUTFLOW,) * 3)
    o.set_state(W._pack_stars(n0 * one, [-a * X, s * X, zero], [p0 * one, zero, zero, p0 * one, zero, p0 * one]))
    o.od_enable()
    o.set("phi", 0.3 * Y)
    o.od_eulerian(tau)
    inner = (slice(1, -1),) * 3
    exp = {"Pxx": p0 * (1 + 2 * tau * a), "Pxy": -tau * p0 * s, "Pxz": 0.0, "Pyy": p0, "Pyz": 0.0, "Pzz": p0}
    for k, v in exp.items():
        assert np.allclose(o.get_star(k)[inner], v, rtol=1e-13, atol=1e-15), k


def test_carried_fields_ride_the_lagrangian_stage_like_the_density(orc):
    """PAPER.md:118-130 is linear in the advected field and uses one velocity per component: a carried field that starts as
    a constant multiple of the density stays that multiple."""
    w = W.smooth_gas(n=12, kmax=2, amp=0.3, components=W.GAS | W.STARS)
    o = make(orc, w)
    o.od_enable()
    o.set("eps", 3.0 * w.state()["rho"])
    for q, name in enumerate(PN):
        o.set(name, (q + 1.5) * w.state()["n"])
    o.od_lagrangian_only(0.2 * w.h)
    assert np.allclose(o.get("eps"), 3.0 * o.get("rho"), rtol=1e-14)
    for q, name in enumerate(PN):
        assert np.allclose(o.get(name), (q + 1.5) * o.get("n"), rtol=1e-14)


def aksenov_drift(orc, n, balance):
    h = 2 * np.pi / n
    x = (np.arange(n) + 0.5) * h
    rho = (1.0 + 0.5 * np.cos(x))[None, None, :] * np.ones((4, 4, n))
    o = orc.Oracle(n, 4, 4, h, W.GAS, gamma=3.0)
    zero = np.zeros_like(rho)
    o.set_state(W._pack_gas(rho, zero, zero, zero, rho ** 3 / 3.0, 3.0))
    o.od_enable()
    t, t_end, kmax = 0.0, np.pi / 4, 0.0
    while t < t_end * (1 - 1e-14):
        dt = min(o.max_dt(0.2), t_end - t)
        o.od_step(dt, balance=balance)
        kmax = max(kmax, o.kappa()[0])
        t += dt
    r, m, E, eps = (o.get(k)[0, 0] for k in ("rho", "mx", "E", "eps"))
    return np.abs((E - 0.5 * m * m / r) - eps).mean() / eps.mean(), kmax


def test_two_energy_descriptions_agree_on_smooth_flow_and_converge(orc):
    """PAPER.md:243-248 (smooth until t = pi/2): without any balancing the internal energy carried by the 4th equation
    and the one implied by the total energy stay within the scheme's first-order truncation error of each other, and
    that gap halves with h.  This is what kappa_gas measures."""
    d = [aksenov_drift(orc, n, balance=False)[0] for n in (64, 128, 256)]
    assert d[0] < 0.03
    assert 0.35 < d[1] / d[0] < 0.65 and 0.35 < d[2] / d[1] < 0.65
    gap, kmax = aksenov_drift(orc, 64, balance=True)
    assert gap <= 1e-15 and kmax <= 1e-15 * (2 * np.pi) ** 3


def test_kappa_at_a_shock_is_bounded_and_the_balance_removes_it(orc):
    """Sod tube (config 1): the non-conservative 4th equation misses the shock heating, so kappa_gas grows where the
    shock has passed; it stays a bounded fraction of the total energy, and with the balance the run is the base scheme."""
    w = W.sod(n=128)
    a, b, c = make(orc, w), make(orc, w), make(orc, w)
    b.od_enable()
    c.od_enable()
    for _ in range(120):
        dt = a.max_dt(w.cfl)
        a.step(dt)
        b.od_step(dt, balance=True)
        c.od_step(dt, balance=False)
    assert np.array_equal(a.get("E"), b.get("E")) and np.array_equal(a.get("rho"), b.get("rho"))
    etot = np.abs(c.get("E")).sum() * w.h ** 3
    kg = c.kappa()[0]
    assert 1e-4 * etot < kg < 0.05 * etot
    assert np.all(c.get("eps") > 0)


def test_balance_at_a_vacuum_border_keeps_pressure_positive(orc):
    """G15 by hand on single cells: (1) healthy cell: rho eps := rho E - rho v^2/2, momentum untouched; (2) border cell
    whose total energy lies below its kinetic energy: rho eps kept, |v| rescaled, direction kept, so that the identity of
    PAPER.md:41 (last line) holds again; (3) total energy below even rho eps: velocity zeroed, rho E raised to rho eps."""
    n = 4
    one = np.ones((n, n, n))
    o = orc.Oracle(n, n, n, 1.0, W.GAS, gamma=1.4)
    rho = 2.0 * one
    mx, my, mz = 2.0 * one, -1.0 * one, 0.5 * one
    kin = 0.5 * (mx ** 2 + my ** 2 + mz ** 2) / rho
    E = kin + 1.0
    o.set_state({"rho": rho, "mx": mx, "my": my, "mz": mz, "E": E})
    o.od_enable()
    eps = o.get("eps")
    eps[:] = 0.4                       # the carried value drifted everywhere
    E2 = E.copy()
    E2[0, 0, 1] = kin[0, 0, 1] - 0.3   # border cell: rho E - kin < 0, but rho E - rho eps > 0
    E2[0, 0, 2] = 0.1                  # hopeless cell: rho E < rho eps
    o.set("eps", eps)
    o.set("E", E2)
    o.od_balance()
    e, m = o.get("eps"), [o.get(k) for k in ("mx", "my", "mz")]
    assert e[0, 0, 0] == pytest.approx(1.0, rel=1e-14) and m[0][0, 0, 0] == 2.0
    knew = 0.5 * sum(a[0, 0, 1] ** 2 for a in m) / 2.0
    assert e[0, 0, 1] == 0.4 and knew == pytest.approx(E2[0, 0, 1] - 0.4, rel=1e-13)
    assert m[0][0, 0, 1] / m[1][0, 0, 1] == pytest.approx(-2.0, rel=1e-14)          # direction kept
    assert all(a[0, 0, 2] == 0.0 for a in m) and o.get("E")[0, 0, 2] == 0.4 and e[0, 0, 2] == 0.4
    assert o.kappa()[0] <= 1e-14


def test_balance_of_the_collisionless_component_by_hand(orc):
    """G15 by hand on single cells of a STARS context with uniform n, u != 0 and a carried Pi that drifted everywhere:
    (a) a healthy cell (all three implied Pi_dd > 0): Pi_ij := n E_ij - n u_i u_j, n E_ij untouched; (b), (c), (d) one
    cell each whose implied Pi_xx, Pi_yy, Pi_zz ALONE is not positive: the carried tensor wins there and all six
    n E_ij := Pi_ij + n u_i u_j exactly, n, n u and Pi untouched.  kappa_bme is zero afterwards."""
    N = 4
    one = np.ones((N, N, N))
    nn = 2.0 * one
    u = [0.5 * one, -0.25 * one, 0.75 * one]
    Pi_implied = [1.0, 0.2, -0.1, 0.8, 0.05, 1.2]          # xx xy xz yy yz zz, what n E_ij will imply
    o = orc.Oracle(N, N, N, 1.0, W.STARS)
    st = W._pack_stars(nn, u, [v * one for v in Pi_implied])
    o.set_state(st)
    o.od_enable()
    carried = [0.6, 0.1, 0.02, 0.5, -0.04, 0.9]             # the drifted carried tensor, different in every component
    for name, v in zip(PN, carried):
        o.set(name, v * one)
    E = {e: st[e].copy() for e in EN}
    nuu = {e: 2.0 * u[i][0, 0, 0] * u[j][0, 0, 0] for e, (i, j) in zip(EN, PAIRS)}
    bad = {"Exx": (0, 0, 1), "Eyy": (0, 0, 2), "Ezz": (0, 0, 3)}   # one diagonal each: implied Pi_dd = -0.3
    for e, cell in bad.items():
        E[e][cell] = nuu[e] - 0.3
    for e in EN:
        o.set(e, E[e])
    o.od_balance()
    got_E = {e: o.get(e) for e in EN}
    got_P = {p: o.get(p) for p in PN}
    # (a) healthy cell: total-energy description wins, nE untouched bit for bit
    for p, e, v in zip(PN, EN, Pi_implied):
        assert got_P[p][0, 0, 0] == pytest.approx(v, rel=1e-14, abs=1e-15)
        assert got_E[e][0, 0, 0] == E[e][0, 0, 0]
    assert np.array_equal(got_E["Exx"][1:], E["Exx"][1:])
    # (b), (c), (d): carried tensor wins in the whole cell
    for cell in bad.values():
        for p, e, v in zip(PN, EN, carried):
            assert got_P[p][cell] == v, (cell, p)
            assert got_E[e][cell] == v + nuu[e], (cell, e)
    assert np.array_equal(o.get("n"), nn)
    for k, a in zip(("nux", "nuy", "nuz"), u):
        assert np.array_equal(o.get(k), nn * a)
    assert o.kappa()[1] <= 1e-14


def test_cfl_of_an_overdetermined_context_uses_the_carried_fields(orc):
    """Reading G16: with the overdetermined system on, the signal speeds are those of the pressure and dispersion the
    stages use, p = (gamma-1) rho*eps and the carried Pi_dd.  A state whose total-energy description is unphysical in
    a block (gas-vacuum border) but whose carried fields are positive yields a finite dt, equal to the brute-force
    maximum over the carried-field wave speeds; a non-positive CARRIED value is what gets reported."""
    g = 1.4
    w = W.smooth_gas(dims=(12, 8, 6), kmax=2, amp=0.3, components=W.GAS | W.STARS, gamma=g)
    st = w.state()
    base = make(orc, w)
    o = make(orc, w)
    o.od_enable()
    dt0 = base.max_dt(0.3)
    assert o.max_dt(0.3) == pytest.approx(dt0, rel=1e-14)        # derived carried fields: the same speeds
    rng = np.random.default_rng(11)
    eps = o.get("eps") * rng.uniform(0.5, 2.0, size=st["rho"].shape)
    P = {k: o.get(k) * rng.uniform(0.5, 2.0, size=st["rho"].shape) for k in ("Pxx", "Pyy", "Pzz")}
    E = st["E"].copy()
    E[1:3, 2:5, 3:9] = 1e-3                                     # far below the kinetic energy there
    Exx = st["Exx"].copy()
    Exx[3:5, 2:5, 3:9] = 1e-3
    o.set("eps", eps); o.set("E", E); o.set("Exx", Exx)
    for k, a in P.items():
        o.set(k, a)
    base.set("E", E)
    with pytest.raises(Exception):
        base.max_dt(0.3)                                        # the base scheme rightly reports the state
    v = [np.abs(st[k] / st["rho"]) for k in ("mx", "my", "mz")]
    u = [np.abs(st[k] / st["n"]) for k in ("nux", "nuy", "nuz")]
    cs = np.sqrt(g * (g - 1.0) * eps / st["rho"])
    smax = max(max((a + cs).max() for a in v),
               max((a + np.sqrt(3.0 * P[k] / st["n"])).max() for a, k in zip(u, ("Pxx", "Pyy", "Pzz"))))
    assert o.max_dt(0.3) == pytest.approx(0.3 * w.h / smax, rel=1e-14)
    assert abs(o.max_dt(0.3) - dt0) > 1e-3 * dt0                # and it is not the base scheme's number
    for name in ("eps", "Pyy"):
        a = o.get(name)
        keep = a[2, 3, 4]
        a[2, 3, 4] = -keep
        o.set(name, a)
        with pytest.raises(Exception):
            o.max_dt(0.3)
        a[2, 3, 4] = keep
        o.set(name, a)
    assert np.isfinite(o.max_dt(0.3))


def test_dispersion_equation_agrees_with_the_energy_tensor_on_smooth_shear(orc):
    """One unbalanced step of a smooth state with all six Pi components and all velocities varying: the Pi_ij carried by
    PAPER.md:65 and the one implied by n E_ij differ by the truncation error only, first order in h."""
    gaps = []
    for N in (32, 64, 128):
        h = 1.0 / N
        s = 2 * np.pi * (np.arange(N) + 0.5) * h
        lift = lambda a: np.broadcast_to(a[None, None, :], (4, 4, N)).copy()
        n = lift(1.0 + 0.2 * np.sin(s + 0.3))
        u = [lift(0.30 * np.sin(s + 0.1)), lift(-0.20 * np.sin(s + 1.3)), lift(0.25 * np.cos(s + 0.7))]
        Pi = [lift((1.0 if i == j else 0.2) + 0.1 * np.sin(s + 0.9 * q + 0.2)) for q, (i, j) in enumerate(PAIRS)]
        o = orc.Oracle(N, 4, 4, h, W.STARS)
        o.set_state(W._pack_stars(n, u, Pi))
        o.od_enable()
        dt = 0.2 * o.max_dt(1.0)
        o.od_step(dt, balance=False)
        nn = o.get("n")
        uu = [o.get(k) / nn for k in ("nux", "nuy", "nuz")]
        gap = 0.0
        for name, e, (i, j) in zip(PN, EN, PAIRS):
            gap = max(gap, np.abs(o.get(e) - nn * uu[i] * uu[j] - o.get(name)).max())
        gaps.append(gap / dt)
        assert o.kappa()[1] > 0
    assert gaps[0] < 0.5
    assert 0.35 < gaps[1] / gaps[0] < 0.65 and 0.35 < gaps[2] / gaps[1] < 0.65


def test_the_stages_take_pressure_and_dispersion_from_the_carried_fields(orc):
    """Uniform conserved state (so the total energy implies a uniform pressure and n E_ij a uniform Pi), but a jump in the
    CARRIED rho*eps / Pi_xx between cells 3 and 4: the momentum of the two adjacent cells must change by the face value of
    PAPER.md:114 / 174 evaluated with p = (gamma-1) rho*eps and the carried Pi_xx."""
    N, h, g, dt = 8, 0.5, 1.4, 0.1
    one = np.ones((4, 4, N))
    zero = 0 * one
    o = orc.Oracle(N, 4, 4, h, W.GAS | W.STARS, gamma=g, bc=(W.BC_OUTFLOW, W.BC_PERIODIC, W.BC_PERIODIC))
    st = W._pack_gas(one, zero, zero, zero, one, g)
    st.update(W._pack_stars(one, [zero, zero, zero], [one, zero, zero, one, zero, one]))
    o.set_state(st)
    o.od_enable()
    jump = np.where(np.arange(N)[None, None, :] < 4, 1.0, 0.1) * one
    o.set("eps", jump / (g - 1))
    o.set("Pxx", jump)
    o.od_eulerian(dt)
    P = 0.55                                       # (114) and (174) with equal velocities: the mean of the two sides
    mx, nux = o.get_star("mx")[0, 0], o.get_star("nux")[0, 0]
    for m in (mx, nux):
        assert m[3] == pytest.approx(-dt / h * (P - 1.0), rel=1e-14)
        assert m[4] == pytest.approx(-dt / h * (0.1 - P), rel=1e-14)
        assert np.all(m[[0, 1, 2, 5, 6, 7]] == 0.0)
