"""Full-size checks (pytest -m gpu) of BASELINE.json config 5 in the launch configuration bench.py
times: 512^3, gas + collisionless component + periodic FFT gravity, one full timestep through the
C ABI (gp_solve_poisson + gp_max_dt + gp_step).

The CPU oracle cannot step 512^3 in seconds, so the step is checked
  * on SAMPLED outputs the oracle computes one by one: cut-outs of (U^n, Phi) of 24^3 cells
    around the two disk centres, in the background and across the periodic box edge are stepped
    by the oracle with the same dt; the scheme's domain of dependence is two cells (Eulerian then
    Lagrangian stage) plus one for the centred grad Phi, so the inner 16^3 cells of
    a cut-out are exactly what the full grid computes there -- tolerance 1e-11 per field group;
  * through properties that hold at any size: mass of each component and total momentum conserved
    to round-off (periodic box, "mass ... and total impulse are conserved"),
    27-point stencil residual of Phi, positivity, and the dt folded by the
    step's epilogue equal to the dt of the stand-alone reduction over the same state.
"""
import numpy as np
import pytest

from paper_1311_0861_b200 import workloads as W

pytestmark = pytest.mark.gpu

N = 512
M, MARGIN = 24, 4
GROUPS = [("rho",), ("mx", "my", "mz"), ("E",), ("n",), ("nux", "nuy", "nuz"),
          ("Exx", "Exy", "Exz", "Eyy", "Eyz", "Ezz")]
# (x, y, z) corners of the cut-outs: disk A centre, disk B centre, background, across the box edge
CORNERS = [(154 - 12, 256 - 12, 256 - 12), (358 - 12, 256 - 12, 256 - 12), (40, 60, 80), (N - 10, N - 7, N - 12)]


def cut(a, corner):
    x0, y0, z0 = corner
    ix = [np.arange(c, c + M) % N for c in (z0, y0, x0)]
    return np.ascontiguousarray(a[np.ix_(*ix)])


@pytest.fixture(scope="module")
def run():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1311_0861_b200 as pkg
    pkg.lib()
    w = W.two_disks(n=N)
    names = w.field_names
    sim = pkg.Simulation.from_workload(w)
    buf = np.empty((N, N, N))
    before, after, sums0, sums1 = {}, {}, {}, {}
    host = {k: np.empty((N, N, N)) for k in names}
    w.fill(host)
    for k in names:
        sim.set(k, host[k])
        sums0[k] = float(host[k].sum(dtype=np.longdouble))
        before[k] = [cut(host[k], c) for c in CORNERS]
    scale = {k: float(np.abs(host[k]).sum(dtype=np.longdouble)) for k in names}
    del host
    sim.solve_poisson()
    dt = sim.max_dt(w.cfl)                       # stand-alone reduction (state was set from outside)
    phi = sim.get("phi", out=buf).copy()
    before["phi"] = [cut(phi, c) for c in CORNERS]
    sim.step(dt)
    dt_epilogue = sim.max_dt(w.cfl)              # folded by the step's epilogue
    pos = {}
    for k in names:
        a = sim.get(k, out=buf)
        sums1[k] = float(a.sum(dtype=np.longdouble))
        after[k] = [cut(a, c) for c in CORNERS]
        if k in ("rho", "n", "E", "Exx", "Eyy", "Ezz"):
            pos[k] = float(a.min())
    # the stand-alone reduction over the same (new) state: a get/set round trip drops the cached value
    sim.set("rho", sim.get("rho", out=buf))
    dt_standalone = sim.max_dt(w.cfl)
    return dict(w=w, dt=dt, before=before, after=after, sums0=sums0, sums1=sums1, scale=scale, phi=phi, pos=pos,
                dt_epilogue=dt_epilogue, dt_standalone=dt_standalone)


def test_sampled_cutouts_match_the_oracle(run, orc):
    w, dt = run["w"], run["dt"]
    inner = (slice(MARGIN, M - MARGIN),) * 3
    for ci in range(len(CORNERS)):
        ref = orc.Oracle(M, M, M, w.h, w.components, orc.POISSON_NONE, w.G, w.gamma, (1, 1, 1))
        for k in w.field_names:
            ref.set(k, run["before"][k][ci])
        ref.set("phi", run["before"]["phi"][ci])
        ref.step(dt)
        for g in GROUPS:
            num = max(np.abs(run["after"][k][ci][inner] - ref.get(k)[inner]).max() for k in g)
            den = max(np.abs(ref.get(k)[inner]).max() for k in g)
            assert num <= 1e-11 * den, (CORNERS[ci], g, num / den)


def test_mass_and_total_momentum_are_conserved(run):
    s0, s1, sc = run["sums0"], run["sums1"], run["scale"]
    for k in ("rho", "n"):
        assert abs(s1[k] - s0[k]) <= 1e-13 * sc[k], k
    # periodic FFT gravity: the centred gradient of the inverse Laplacian is antisymmetric, so the
    # momentum the two components exchange with the field cancels
    for g, s in (("mx", "nux"), ("my", "nuy"), ("mz", "nuz")):
        drift = (s1[g] + s1[s]) - (s0[g] + s0[s])
        assert abs(drift) <= 1e-12 * (sc[g] + sc[s]), (g, drift / (sc[g] + sc[s]))


def test_state_stays_physical_and_dt_paths_agree(run):
    for k, v in run["pos"].items():
        assert v > 0.0, k
    assert abs(run["dt_epilogue"] - run["dt_standalone"]) <= 1e-13 * run["dt_standalone"]


def test_potential_inverts_the_27_point_stencil(run):
    w, phi = run["w"], run["phi"]
    # Phi was solved for rho + n of the INITIAL state; rebuild that source from the workload
    src = np.empty((N, N, N))
    for z0 in range(0, N, 64):
        f = w.fields(z0, z0 + 64)
        src[z0:z0 + 64] = f["rho"] + f["n"]
    a = phi
    for ax in range(3):
        a = (np.roll(a, 1, ax) + 4.0 * a + np.roll(a, -1, ax)) / 6.0
    res = 6.0 * (a - phi) / (w.h * w.h) - 4 * np.pi * w.G * (src - src.mean())
    assert np.abs(res).max() < 1e-10 * 4 * np.pi * w.G * src.max()
    assert abs(phi.mean()) < 1e-12 * np.abs(phi).max()
