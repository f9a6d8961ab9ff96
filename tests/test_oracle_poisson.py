"""Pins P9, P10 and the FFT pin: the oracle's Poisson solvers against library FFTs, the
27-point stencil they invert, brute-force summation and closed forms."""
import numpy as np
import pytest

from paper_1311_0861_b200 import workloads as W


def test_fft1d_against_numpy(orc):
    rng = np.random.default_rng(3)
    for n in (1, 2, 8, 64, 1024):
        x = rng.normal(size=n) + 1j * rng.normal(size=n)
        assert np.allclose(orc.fft1d(x, -1), np.fft.fft(x), rtol=0, atol=1e-12 * n)
        assert np.allclose(orc.fft1d(x, +1), np.fft.ifft(x) * n, rtol=0, atol=1e-12 * n)


def laplacian27(phi, h):
    """The 27-point Laplacian PAPER.md:190 inverts: weights centre -38/9... expressed through
    its factorised symbol 6(1 - prod_d(1 - (2/3) sin^2)) <-> (6/h^2)(A_x A_y A_z - 1) with the
    1-D average A = (1/6, 2/3, 1/6)."""
    a = phi
    for ax in range(3):
        a = (np.roll(a, 1, ax) + 4.0 * a + np.roll(a, -1, ax)) / 6.0
    return 6.0 * (a - phi) / (h * h)


def laplacian27_weights(phi, h):
    """Same operator written with explicit weights: centre -64/15?  No: built from the outer
    product of (1/6, 4/6, 1/6) minus the identity, times 6/h^2 — centre 6*(8/27 - 1) = -38/9,
    face 6*(2/27) = 4/9, edge 6*(1/54) = 1/9, corner 6*(1/216) = 1/36."""
    out = np.zeros_like(phi)
    for dz in (-1, 0, 1):
        for dy in (-1, 0, 1):
            for dx in (-1, 0, 1):
                k = abs(dx) + abs(dy) + abs(dz)
                wgt = {0: -38.0 / 9.0, 1: 4.0 / 9.0, 2: 1.0 / 9.0, 3: 1.0 / 36.0}[k]
                out += wgt * np.roll(phi, (-dz, -dy, -dx), (0, 1, 2))
    return out / (h * h)


def test_laplacian_helpers_agree():
    rng = np.random.default_rng(0)
    phi = rng.normal(size=(6, 8, 10))
    assert np.allclose(laplacian27(phi, 0.3), laplacian27_weights(phi, 0.3), rtol=1e-12, atol=1e-12)


def test_P9_periodic_solve_inverts_the_27_point_stencil(orc):
    nx, ny, nz, h, G = 16, 8, 32, 0.25, 1.7
    rng = np.random.default_rng(1)
    rho = rng.uniform(0.5, 1.5, (nz, ny, nx))
    n = rng.uniform(0.1, 0.4, (nz, ny, nx))
    o = orc.Oracle(nx, ny, nz, h, W.GAS | W.STARS, W.POISSON_PERIODIC, G=G)
    o.set("rho", rho)
    o.set("n", n)
    o.solve_poisson()
    phi = o.get("phi")
    src = rho + n                                    # one solve of the summed density
    assert abs(phi.mean()) < 1e-13 * np.abs(phi).max()                     # k = 0 mode set to zero
    res = laplacian27_weights(phi, h) - 4 * np.pi * G * (src - src.mean())
    assert np.abs(res).max() < 1e-12 * 4 * np.pi * G * np.abs(src).max()
    pad = o.phi_padded()                             # ghost ring wraps
    assert np.array_equal(pad[1:-1, 1:-1, 0], phi[:, :, -1]) and np.array_equal(pad[-1, 1:-1, 1:-1], phi[0])


def test_P9_single_mode_and_sign(orc):
    """One Fourier mode in -> the same mode out times the factor of PAPER.md:190 with the sign
    of reading G3: an over-density sits in a potential well (Phi < 0 where rho is largest)."""
    n, h = 16, 1.0 / 16
    x = (np.arange(n) + 0.5) * h
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    k = (2, 1, 3)
    mode = np.cos(2 * np.pi * (k[0] * X + k[1] * Y + k[2] * Z))
    o = orc.Oracle(n, n, n, h, W.GAS, W.POISSON_PERIODIC, G=1.0)
    o.set("rho", 1.0 + 0.5 * mode)
    o.solve_poisson()
    s2 = [np.sin(np.pi * kk / n) ** 2 for kk in k]
    fac = -4 * np.pi * h * h / (6 * (1 - (1 - 2 / 3 * s2[0]) * (1 - 2 / 3 * s2[1]) * (1 - 2 / 3 * s2[2])))
    assert np.allclose(o.get("phi"), 0.5 * fac * mode, rtol=0, atol=1e-13 * abs(fac))
    assert fac < 0
    # long-wave limit: the solve tends to the continuum Phi_k = -4 pi G rho_k / |k|^2
    n, h = 32, 1.0 / 32
    x = (np.arange(n) + 0.5) * h
    o = orc.Oracle(n, 4, 4, h, W.GAS, W.POISSON_PERIODIC, G=1.0)
    o.set("rho", (1.0 + 0.5 * np.cos(2 * np.pi * x))[None, None, :] * np.ones((4, 4, n)))
    o.solve_poisson()
    assert np.allclose(o.get("phi")[0, 0], -0.5 * 4 * np.pi / (2 * np.pi) ** 2 * np.cos(2 * np.pi * x), rtol=0, atol=5e-3 * 0.16)


def test_kernel_self_is_the_cube_centre_potential(orc):
    """K(0) h = potential at the centre of a uniform unit cube of unit mass =
    int_cube 1/|r| d^3r.  Checked by Gauss-Legendre quadrature on the octant in spherical-like
    (Duffy) coordinates, independent of the closed form the oracle uses."""
    # int over [0,1/2]^3 of 1/r, times 8.  Duffy: split the octant in 3 pyramids by the largest coordinate;
    # on x >= y,z: y = x s, z = x t, dV = x^2 dx ds dt, 1/r = 1/(x sqrt(1+s^2+t^2)).
    g, wq = np.polynomial.legendre.leggauss(40)
    s = 0.5 * (g + 1)
    ws = 0.5 * wq
    S, T = np.meshgrid(s, s, indexing="ij")
    inner = (np.outer(ws, ws) / np.sqrt(1 + S * S + T * T)).sum()
    val = 8 * 3 * inner * (0.5 ** 2 / 2)            # int_0^{1/2} x dx = 1/8
    assert orc.kernel_self() == pytest.approx(val, rel=1e-12)
    assert orc.kernel_self() == pytest.approx(2.3800773640, abs=1e-9)


def test_P10_isolated_solve_equals_direct_summation_including_ghost_ring(orc):
    nx, ny, nz, h, G = 8, 4, 16, 0.5, 2.0
    rng = np.random.default_rng(2)
    rho = rng.uniform(0.0, 1.0, (nz, ny, nx))
    o = orc.Oracle(nx, ny, nz, h, W.GAS, W.POISSON_ISOLATED, G=G, bc=(W.BC_OUTFLOW,) * 3)
    o.set("rho", rho)
    o.solve_poisson()
    pad = o.phi_padded()
    ref = orc.poisson_direct(rho, h, G, lo=(-1, -1, -1), hi=(nz + 1, ny + 1, nx + 1))
    scale = np.abs(ref).max()
    assert np.allclose(pad[1:-1, 1:-1, 1:-1], ref[1:-1, 1:-1, 1:-1], rtol=0, atol=1e-13 * scale)
    for sl in ((0, slice(1, -1), slice(1, -1)), (-1, slice(1, -1), slice(1, -1)),
               (slice(1, -1), 0, slice(1, -1)), (slice(1, -1), -1, slice(1, -1)),
               (slice(1, -1), slice(1, -1), 0), (slice(1, -1), slice(1, -1), -1)):
        assert np.allclose(pad[sl], ref[sl], rtol=0, atol=1e-13 * scale)
    # second call reuses the cached kernel spectrum and gives the same answer
    o.solve_poisson()
    assert np.array_equal(o.phi_padded(), pad)


def test_P10_direct_sum_is_the_plain_definition(orc):
    """The direct summation itself, on a 3-cell example by hand: Phi_i = -G sum_j m_j / r_ij,
    self term K(0)."""
    rho = np.zeros((2, 2, 4))
    rho[0, 0, 0], rho[1, 1, 3] = 2.0, 5.0
    h, G = 0.5, 3.0
    phi = orc.poisson_direct(rho, h, G)
    m0, m1 = 2.0 * h ** 3, 5.0 * h ** 3
    d01 = h * np.sqrt(9 + 1 + 1)
    assert phi[0, 0, 0] == pytest.approx(-G * (m0 * orc.kernel_self() / h + m1 / d01), rel=1e-14)
    assert phi[0, 0, 1] == pytest.approx(-G * (m0 / h + m1 / (h * np.sqrt(4 + 1 + 1))), rel=1e-14)


def test_P10_point_mass_and_sphere(orc):
    n, h = 32, 2.4 / 32
    o = orc.Oracle(n, n, n, h, W.GAS, W.POISSON_ISOLATED, G=1.0, bc=(W.BC_OUTFLOW,) * 3)
    rho = np.zeros((n, n, n))
    rho[10, 12, 14] = 3.0
    o.set("rho", rho)
    o.solve_poisson()
    phi = o.get("phi")
    k, j, i = np.meshgrid(*(np.arange(n),) * 3, indexing="ij")
    r = h * np.sqrt((i - 14.0) ** 2 + (j - 12.0) ** 2 + (k - 10.0) ** 2)
    mask = r > 0
    assert np.allclose(phi[mask], -3.0 * h ** 3 / r[mask], rtol=1e-12, atol=0)
    # rho = 1 - r sphere: the printed Phi0(r), second-order convergence
    errs = []
    for n in (16, 32):
        h = 2.4 / n
        x = (np.arange(n) + 0.5) * h - 1.2
        Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
        r = np.sqrt(X * X + Y * Y + Z * Z)
        o = orc.Oracle(n, n, n, h, W.GAS, W.POISSON_ISOLATED, G=1.0, bc=(W.BC_OUTFLOW,) * 3)
        o.set("rho", np.maximum(1.0 - r, 0.0))
        o.solve_poisson()
        exact = np.where(r <= 1, -np.pi / 3 * (r ** 3 - 2 * r * r) - 2 * np.pi / 3, -np.pi / (3 * r))
        errs.append(np.abs(o.get("phi") - exact).max())
    assert errs[0] < 2e-2 and errs[1] < 0.3 * errs[0]
