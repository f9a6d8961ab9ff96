"""Pins P1 and P2: the oracle's face solvers against what the paper and linear algebra fix.

The paper states that the face values are the exact solution of the linearised
Eulerian-stage system dq/dt + B dq/dx = 0 at the cell boundary: characteristic decomposition,
upwinding by the sign of each eigenvalue.  For a constant matrix B that solution at x/t = 0 is
    q* = (qL + qR)/2 + sign(B) (qL - qR)/2,   sign(B) = R sign(Lambda) R^-1,
computed here by numerical eigendecomposition — independent of the printed formulas
 the oracle implements.
"""
import numpy as np
import pytest


def matrix_sign(B):
    lam, R = np.linalg.eig(B)
    assert np.abs(lam.imag).max() < 1e-9
    return (R @ np.diag(np.sign(lam.real)) @ np.linalg.inv(R)).real


def test_gas_face_equals_characteristic_solution(orc):
    rng = np.random.default_rng(11)
    for _ in range(200):
        g = rng.uniform(1.1, 3.0)
        rl, rr = rng.uniform(0.1, 5.0, 2)
        pl, pr = rng.uniform(0.1, 5.0, 2)
        vl, vr = rng.uniform(-2, 2, 2)
        # PAPER.md:84 with the first row/column ruled out (86): q = (v, p); averaged parameters
        # as they appear in (112)-(114): harmonic mean of rho, arithmetic mean of p.
        rho = 2 * rl * rr / (rl + rr)
        p = 0.5 * (pl + pr)
        B = np.array([[0.0, 1.0 / rho], [g * p, 0.0]])
        q = 0.5 * (np.array([vl, pl]) + np.array([vr, pr])) + 0.5 * matrix_sign(B) @ (np.array([vl, pl]) - np.array([vr, pr]))
        V, P = orc.gas_face(g, rl, vl, pl, rr, vr, pr)
        assert V == pytest.approx(q[0], rel=1e-12, abs=1e-13)
        assert P == pytest.approx(q[1], rel=1e-12, abs=1e-13)


def test_gas_face_special_cases(orc):
    # L = R: the face carries the common state
    V, P = orc.gas_face(1.4, 0.7, 0.3, 2.0, 0.7, 0.3, 2.0)
    assert (V, P) == (0.3, 2.0)
    # mirror: swapping L and R and flipping the velocity sign flips V and keeps P
    V1, P1 = orc.gas_face(1.4, 1.0, 0.4, 1.0, 0.125, -0.2, 0.1)
    V2, P2 = orc.gas_face(1.4, 0.125, 0.2, 0.1, 1.0, -0.4, 1.0)
    assert V1 == -V2 and P1 == P2
    # Sod's initial jump, by hand from (112)/(114): Z = sqrt(1*0.125*1.4*1.1/1.125)
    Z = np.sqrt(1.0 * 0.125 * 1.4 * 1.1 / 1.125)
    V, P = orc.gas_face(1.4, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1)
    assert V == pytest.approx(0.45 / Z, rel=1e-15)
    assert P == pytest.approx(0.55, rel=1e-15)


def bme_matrix(n, Pxx, Pxy, Pxz):
    """Eulerian-stage matrix for q = (ux, uy, uz, Pxx, Pxy, Pxz), x-direction, re-derived from
    PAPER.md:63 and 65 with the advective terms ruled out (the printed matrix at 136 is garbled):
        du_i/dt   = -(1/n) dPi_ix/dx
        dPi_xx/dt = -3 Pi_xx dux/dx
        dPi_xy/dt = -2 Pi_xy dux/dx - Pi_xx duy/dx      (xz likewise)
    """
    B = np.zeros((6, 6))
    B[0, 3] = B[1, 4] = B[2, 5] = 1.0 / n
    B[3, 0] = 3.0 * Pxx
    B[4, 0], B[4, 1] = 2.0 * Pxy, Pxx
    B[5, 0], B[5, 2] = 2.0 * Pxz, Pxx
    return B


def test_bme_matrix_eigenvalues_match_paper():
    # +-sqrt(3 Pi_xx/rho), +-sqrt(Pi_xx/rho) (the latter double)
    lam = np.sort(np.linalg.eigvals(bme_matrix(2.0, 1.5, 0.3, -0.2)).real)
    a, b = np.sqrt(3 * 1.5 / 2.0), np.sqrt(1.5 / 2.0)
    assert np.allclose(lam, [-a, -b, -b, b, b, a], rtol=1e-12)


PERM = {0: (0, 1, 2), 1: (1, 2, 0), 2: (2, 0, 1)}   # axis d -> (d, t1, t2)
SYM = [[0, 1, 2], [1, 3, 4], [2, 4, 5]]


@pytest.mark.parametrize("d", [0, 1, 2])
def test_bme_face_equals_characteristic_solution(orc, d):
    rng = np.random.default_rng(100 + d)
    dd, t1, t2 = PERM[d]
    for _ in range(300):
        nL, nR = rng.uniform(0.2, 4.0, 2)
        uL, uR = rng.uniform(-2, 2, 3), rng.uniform(-2, 2, 3)
        PiL, PiR = rng.uniform(-0.8, 0.8, 6), rng.uniform(-0.8, 0.8, 6)
        for P in (PiL, PiR):
            for i in range(3):
                P[SYM[i][i]] = rng.uniform(0.5, 3.0)
        nb = 2 * nL * nR / (nL + nR)                                  # averaging of PAPER.md:180 (reading G7)
        a = 0.5 * (PiL[SYM[dd][dd]] + PiR[SYM[dd][dd]])
        b1 = 0.5 * (PiL[SYM[dd][t1]] + PiR[SYM[dd][t1]])
        b2 = 0.5 * (PiL[SYM[dd][t2]] + PiR[SYM[dd][t2]])
        S = matrix_sign(bme_matrix(nb, a, b1, b2))
        qL = np.array([uL[dd], uL[t1], uL[t2], PiL[SYM[dd][dd]], PiL[SYM[dd][t1]], PiL[SYM[dd][t2]]])
        qR = np.array([uR[dd], uR[t1], uR[t2], PiR[SYM[dd][dd]], PiR[SYM[dd][t1]], PiR[SYM[dd][t2]]])
        q = 0.5 * (qL + qR) + 0.5 * S @ (qL - qR)
        us, Pid = orc.bme_face(d, nL, uL, PiL, nR, uR, PiR)
        got = np.array([us[dd], us[t1], us[t2], Pid[dd], Pid[t1], Pid[t2]])
        assert np.allclose(got, q, rtol=1e-10, atol=1e-11), (got, q)


def test_bme_face_special_cases(orc):
    u = np.array([0.3, -0.1, 0.7])
    Pi = np.array([1.2, 0.1, -0.2, 0.9, 0.05, 1.5])
    for d in range(3):
        us, Pid = orc.bme_face(d, 1.3, u, Pi, 1.3, u, Pi)          # L = R
        assert np.array_equal(us, u)
        assert np.array_equal(Pid, [Pi[SYM[i][d]] for i in range(3)])
    # vanishing off-diagonal stress: the transverse cross terms vanish and the normal pair
    # (u_d, Pi_dd) is the gas solver with gamma = 3, p = Pi_dd (PAPER.md:140 vs 86)
    PiL = np.array([2.0, 0, 0, 1.0, 0, 1.5])
    PiR = np.array([1.0, 0, 0, 3.0, 0, 0.5])
    uL, uR = np.array([0.5, 0.2, -0.3]), np.array([-0.4, 0.1, 0.6])
    us, Pid = orc.bme_face(0, 2.0, uL, PiL, 1.0, uR, PiR)
    V, P = orc.gas_face(3.0, 2.0, uL[0], PiL[0], 1.0, uR[0], PiR[0])
    assert us[0] == V and Pid[0] == P
    Z1 = np.sqrt(2 * 2.0 * 1.0 / 3.0 * 1.5)
    assert us[1] == pytest.approx(0.5 * (0.2 + 0.1), rel=1e-15)
    assert Pid[1] == pytest.approx(0.5 * (0.2 - 0.1) * Z1, rel=1e-14)
