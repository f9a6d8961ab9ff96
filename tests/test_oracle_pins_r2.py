"""Round-2 pins for the two parts of the oracle that no round-1 test fixed ("Survivors"):

* the shear (transverse) fluxes of the collisionless Eulerian stage -- the Pi*_{td} flux of (nu_t)* and
  the 2 Pi*_{td} u*_t / Pi*_{jd} u*_i + Pi*_{id} u*_j fluxes of nE_ij (2nd and 3rd equation);
* the LOW-side outflow ghost cell ("one-layer overlapping", readings a-1 / H6).

The yardstick of the first is the continuous system PAPER.md:63 itself without its advective terms
(the Eulerian stage), differentiated spectrally -- no face formula is retyped here.
"""
import numpy as np
import pytest

from paper_1311_0861_b200 import workloads as W

PAIRS = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]
ENAMES = ["Exx", "Exy", "Exz", "Eyy", "Eyz", "Ezz"]
MNAMES = ["nux", "nuy", "nuz"]


def _spectral_ddx(f, L):
    """d/ds of a periodic band-limited sample f (cell centres, period L): exact up to Nyquist."""
    n = f.shape[0]
    k = 2j * np.pi * np.fft.fftfreq(n, d=L / n)
    return np.real(np.fft.ifft(k * np.fft.fft(f)))


def _shear_state(N, d):
    """All ten BME primitives vary smoothly along axis d only; every Pi_ij and u_i is live."""
    h = 1.0 / N
    s = (np.arange(N) + 0.5) * h
    w = 2 * np.pi * s
    n = 1.0 + 0.2 * np.sin(w + 0.3)
    u = [0.30 * np.sin(w + 0.1), -0.20 * np.sin(w + 1.3), 0.25 * np.cos(w + 0.7)]
    Pi = {}
    for q, (i, j) in enumerate(PAIRS):
        Pi[(i, j)] = (1.0 if i == j else 0.2) + 0.1 * np.sin(w + 0.9 * q + 0.2) + 0.05 * np.cos(2 * w + 0.4 * q)
        Pi[(j, i)] = Pi[(i, j)]
    return h, s, n, u, Pi


def _eulerian_increments(orc, N, d):
    h, s, n, u, Pi = _shear_state(N, d)
    dims = [4, 4, 4]
    dims[d] = N
    nx, ny, nz = dims
    shape = (nz, ny, nx)
    ax = 2 - d                                   # numpy axis of coordinate d in (z, y, x) arrays

    def lift(a):
        sh = [1, 1, 1]
        sh[ax] = N
        return np.broadcast_to(a.reshape(sh), shape).copy()

    st = W._pack_stars(lift(n), [lift(a) for a in u], [lift(Pi[p]) for p in PAIRS])
    o = orc.Oracle(nx, ny, nz, h, W.STARS, gamma=5.0 / 3.0)
    o.set_state(st)
    dt = 1e-3
    o.eulerian(dt)
    sel = [0, 0, 0]
    sel[ax] = slice(None)
    inc = {k: ((o.get_star(k) - st[k]) / dt)[tuple(sel)] for k in MNAMES + ENAMES}
    assert np.array_equal(o.get_star("n"), st["n"])          # density untouched
    # PAPER.md:63 without advection, fields depending on x_d only:
    #   d/dt (n u_i) = -d/dx_d Pi_{id};   d/dt (n E_ij) = -d/dx_d (Pi_{jd} u_i + Pi_{id} u_j)
    exact = {}
    for i in range(3):
        exact[MNAMES[i]] = -_spectral_ddx(Pi[(i, d)], 1.0)
    for name, (i, j) in zip(ENAMES, PAIRS):
        exact[name] = -_spectral_ddx(Pi[(j, d)] * u[i] + Pi[(i, d)] * u[j], 1.0)
    return inc, exact


@pytest.mark.parametrize("d", [0, 1, 2])
def test_bme_eulerian_stage_converges_to_the_moment_equations_including_shear(orc, d):
    """Every one of the nine updated BME fields, with all six Pi components and all three velocities
    varying along axis d, converges at first order to the right-hand side of PAPER.md:63.  Dropping or
    halving any flux term (normal or shear) leaves an O(1) residual."""
    errs = {}
    for N in (64, 128, 256):
        inc, exact = _eulerian_increments(orc, N, d)
        errs[N] = {k: np.abs(inc[k] - exact[k]).max() / np.abs(exact[k]).max() for k in exact}
    for k in errs[64]:
        assert errs[256][k] < 0.05, (k, errs[256][k])
        for fine, coarse in ((128, 64), (256, 128)):          # first order: the error halves with h
            assert 0.4 < errs[fine][k] / errs[coarse][k] < 0.6, (k, [errs[N][k] for N in errs])


def test_bme_shear_flux_by_hand_on_a_pure_shear_jump(orc):
    """A tangential-velocity jump u_y: +a | -a across one x-face with uniform n, isotropic Pi = p.
    PAPER.md:176 gives Pi*_xy = a sqrt(n p) there, u*_y = 0, Pi*_xx = p, u*_x = 0; so by PAPER.md:63 the two
    adjacent cells change (nu_y) by -+ tau/h Pi*_xy and nE_yy by -+ tau/h 2 Pi*_xy u*_y = 0.  The flux of
    nE_xy, Pi*_xy u*_x + Pi*_xx u*_y, is 0 on the jump face and p*(+-a) on the uniform faces either side,
    so both adjacent cells gain tau/h p a; one cell further away nothing changes."""
    N, h, a, p, nn, dt = 8, 0.5, 0.3, 2.0, 1.5, 0.05
    one = np.ones((4, 4, N))
    uy = np.where(np.arange(N)[None, None, :] < 4, a, -a) * one
    zero = 0 * one
    st = W._pack_stars(nn * one, [zero, uy, zero], [p * one, zero, zero, p * one, zero, p * one])
    o = orc.Oracle(N, 4, 4, h, W.STARS, bc=(W.BC_OUTFLOW, W.BC_PERIODIC, W.BC_PERIODIC))
    o.set_state(st)
    o.eulerian(dt)
    Pxy = a * np.sqrt(nn * p)                                 # (176): (u_y^L - u_y^R)/2 * sqrt([n][Pi_xx])
    dnuy = (o.get_star("nuy") - st["nuy"])[0, 0]
    assert dnuy[3] == pytest.approx(-dt / h * Pxy, rel=1e-14)
    assert dnuy[4] == pytest.approx(+dt / h * Pxy, rel=1e-14)
    assert np.all(dnuy[[0, 1, 2, 5, 6, 7]] == 0.0)
    # nE_yy = Pi_yy + n u_y^2 keeps its value: the shear flux 2 Pi*_xy u*_y vanishes with u*_y = 0 ...
    assert np.allclose((o.get_star("Eyy") - st["Eyy"])[0, 0], 0.0, atol=1e-15)
    # ... while nE_xy loses the flux Pi*_xx u*_y = p*(+-a) of the uniform faces and nothing through the jump face
    dExy = (o.get_star("Exy") - st["Exy"])[0, 0]
    assert dExy[3] == pytest.approx(dt / h * p * a, rel=1e-14)
    assert dExy[4] == pytest.approx(dt / h * p * a, rel=1e-14)
    assert np.all(dExy[[0, 1, 2, 5, 6, 7]] == 0.0)
    # add a uniform drift u_x = c: u*_x = c, so nE_xy now receives the flux Pi*_xy c (3rd eq.)
    c = 0.7
    st2 = W._pack_stars(nn * one, [c * one, uy, zero], [p * one, zero, zero, p * one, zero, p * one])
    o.set_state(st2)
    o.eulerian(dt)
    dExy = (o.get_star("Exy") - st2["Exy"])[0, 0]
    assert dExy[3] == pytest.approx(-dt / h * (Pxy * c - p * a), rel=1e-13)
    assert dExy[4] == pytest.approx(+dt / h * (Pxy * c + p * a), rel=1e-13)
    # and a uniform drift u_y = c on top of the jump: u*_y = c, so nE_yy receives 2 Pi*_xy c
    st3 = W._pack_stars(nn * one, [zero, uy + c, zero], [p * one, zero, zero, p * one, zero, p * one])
    o.set_state(st3)
    o.eulerian(dt)
    dEyy = (o.get_star("Eyy") - st3["Eyy"])[0, 0]
    assert dEyy[3] == pytest.approx(-dt / h * 2 * Pxy * c, rel=1e-13)
    assert dEyy[4] == pytest.approx(+dt / h * 2 * Pxy * c, rel=1e-13)


# ------------------------------------------------------------------------------------------------
# outflow ghost cells, LOW and high side, on every axis (reading a-1: copy of the nearest interior cell)
# ------------------------------------------------------------------------------------------------
def _tube(axis, N, prof):
    dims = [4, 4, 4]
    dims[axis] = N
    nx, ny, nz = dims
    sh = [1, 1, 1]
    sh[2 - axis] = N
    return (nx, ny, nz), np.broadcast_to(np.asarray(prof, dtype=float).reshape(sh), (nz, ny, nx)).copy()


def _line(a, axis):
    sel = [1, 1, 1]
    sel[2 - axis] = slice(None)
    return a[tuple(sel)]


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("side", ["low", "high"])
def test_outflow_ghost_of_the_eulerian_stage_is_the_adjacent_cell(orc, axis, side):
    """Pressure jump between the boundary cell and its inner neighbour.  With ghost := boundary cell the
    outer face of the boundary cell sees L = R, so P = p, V = 0 there (PAPER.md:112-114 with equal states)
    and the boundary cell changes by the inner face alone; a ghost copied from one cell further in (or a
    wrapped one) would put a second jump on the outer face."""
    N, h, g, dt = 8, 0.5, 1.4, 0.1
    jump = 1 if side == "low" else N - 1                      # first cell of the right-hand state
    idx = np.arange(N)
    rho_p, p_p = np.where(idx < jump, 1.0, 0.125), np.where(idx < jump, 1.0, 0.1)
    (nx, ny, nz), rho = _tube(axis, N, rho_p)
    _, p = _tube(axis, N, p_p)
    zero = np.zeros_like(rho)
    bc = [W.BC_PERIODIC] * 3
    bc[axis] = W.BC_OUTFLOW
    o = orc.Oracle(nx, ny, nz, h, W.GAS, gamma=g, bc=tuple(bc))
    o.set_state(W._pack_gas(rho, zero, zero, zero, p, g))
    o.eulerian(dt)
    Z = np.sqrt(1.0 * 0.125 * g * 1.1 / 1.125)
    V, P = 0.45 / Z, 0.55                                     # (112), (114) on the jump
    m = _line(o.get_star(["mx", "my", "mz"][axis]), axis)
    E = _line(o.get_star("E"), axis)
    exp_m, exp_E = np.zeros(N), p_p / (g - 1)
    exp_m[jump - 1] = -dt / h * (P - 1.0)
    exp_m[jump] = -dt / h * (0.1 - P)
    exp_E[jump - 1] -= dt / h * (P * V)
    exp_E[jump] += dt / h * (P * V)
    assert np.allclose(m, exp_m, rtol=1e-14, atol=1e-16)
    assert np.allclose(E, exp_E, rtol=1e-14, atol=0)


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("side", ["low", "high"])
def test_outflow_ghost_of_the_lagrangian_stage_is_the_adjacent_cell(orc, axis, side):
    """Uniform velocity blowing INTO the box through an outflow boundary whose boundary cell differs from
    its inner neighbour: the inflow carries the ghost value (upwind f+), which must be the
    boundary cell's own, so that cell keeps what it had plus the exchange with its inner neighbour."""
    N, h, dt, w = 8, 1.0, 0.1, 0.5
    idx = np.arange(N)
    prof = np.where(idx == (0 if side == "low" else N - 1), 3.0, 1.0)
    (nx, ny, nz), rho = _tube(axis, N, prof)
    vel = [np.zeros_like(rho) for _ in range(3)]
    vel[axis] = (w if side == "low" else -w) * np.ones_like(rho)
    bc = [W.BC_PERIODIC] * 3
    bc[axis] = W.BC_OUTFLOW
    o = orc.Oracle(nx, ny, nz, h, W.GAS, gamma=1.4, bc=tuple(bc))
    o.set_state(W._pack_gas(rho, vel[0], vel[1], vel[2], np.ones_like(rho), 1.4))
    o.lagrangian_only(dt)
    r = _line(o.get("rho"), axis)
    b, inner = (0, 1) if side == "low" else (N - 1, N - 2)
    # boundary cell: inflow w*ghost(=3) through the outer face, outflow w*3 through the inner face -> unchanged;
    # its inner neighbour: inflow w*3, outflow w*1
    assert r[b] == pytest.approx(3.0, rel=1e-15)
    assert r[inner] == pytest.approx(1.0 + dt / h * w * (3.0 - 1.0), rel=1e-15)
    others = [i for i in range(N) if i not in (b, inner)]
    assert np.allclose(r[others], 1.0, rtol=1e-15)
