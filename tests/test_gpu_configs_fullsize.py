"""Configs 2, 3, 4 of BASELINE.json at their OWN grid (256^3) against the oracle, element by element
(pytest -m gpu), SURVEY.md 8(d) "parity protocol": both sides compute their own dt (<= 1e-13 apart), both step
with the oracle's; max|diff|/max|ref| <= 1e-11 per field group after one step, sum|diff|/sum|ref| <= 1e-8 after
the steps run, Phi <= 1e-11 of max|Phi|.

The default suite runs as many steps as keep it inside the driver's time limit (config 2: all 100; config 3: 40,
through the 512^3 padded isolated solve of the oracle, i.e. the pruned 512-point column transforms
k_colfft<9,4,2>; config 4: all 100; config 5: 3 steps at 512^3, the WHOLE grid element by element -- the oracle
needs about 20 s per step and 35 GB of host memory there, so the test is skipped, with that reason, on a host
with less than 45 GB available).  With GP_SLOW=1 in the environment config 3 runs its 200 steps and config 5 its
50 steps at 512^3 (GP_SLOW_N5 overrides the grid if host memory is short); the error table of that run is
recorded in profiles/parity_r2.md.
"""
import os

import numpy as np
import pytest

from paper_1311_0861_b200 import workloads as W
from tests.test_gpu_parity import REPORT, check, err_l1, err_max, full_step, make_pair, TOL_1STEP, TOL_NSTEP
from tests.test_gpu_parity import pkg, parity_report  # noqa: F401  (fixtures)

pytestmark = pytest.mark.gpu

SLOW = os.environ.get("GP_SLOW", "0") == "1"


def run(pkg, orc, w, steps):
    sim, ref = make_pair(pkg, orc, w)
    full_step(sim, ref, w)
    check(sim, ref, w, TOL_1STEP, err_max)
    for _ in range(steps - 1):
        full_step(sim, ref, w)
    check(sim, ref, w, TOL_NSTEP, err_l1)
    REPORT.append([w.name, [w.nx, w.ny, w.nz], "steps", "", steps])


def test_config2_smooth_gas_256_all_100_steps(pkg, orc):
    run(pkg, orc, W.smooth_gas(n=256, steps=100), 100)


def test_config3_collapse_256_isolated(pkg, orc):
    run(pkg, orc, W.collapse(n=256), 200 if SLOW else 40)


def test_config4_disk_256_periodic_all_100_steps(pkg, orc):
    run(pkg, orc, W.disk(n=256), 100)


def host_memory_gb():
    import psutil
    return psutil.virtual_memory().available / 2 ** 30


def test_config5_two_disks_512_whole_grid_3_steps(pkg, orc):
    """BASELINE.json config 5 at its own size, every cell of every field against the oracle, three full timesteps."""
    if host_memory_gb() < 45:
        pytest.skip(f"the oracle needs about 35 GB of host memory at 512^3; {host_memory_gb():.0f} GB available")
    run(pkg, orc, W.two_disks(n=512), 3)


@pytest.mark.skipif(not SLOW, reason="config 5 for its 50 steps at 512^3 takes the oracle ~15 minutes: GP_SLOW=1")
def test_config5_two_disks_512_all_50_steps(pkg, orc):
    n = int(os.environ.get("GP_SLOW_N5", "512"))
    run(pkg, orc, W.two_disks(n=n), 50)


@pytest.mark.skipif(not SLOW, reason="one isolated solve at 512^3 (1024-point pruned columns): GP_SLOW=1")
def test_config5_isolated_solve_512_against_oracle(pkg, orc):
    """k_colfft<10,4,1> with pruning, against the oracle's 1024^3 padded convolution."""
    n = int(os.environ.get("GP_SLOW_N5", "512"))
    w = W.two_disks(n=n, poisson=W.POISSON_ISOLATED)
    sim, ref = make_pair(pkg, orc, w)
    sim.solve_poisson()
    ref.solve_poisson()
    e = err_max(sim, ref, ("phi",))
    REPORT.append([w.name + "_isolated", [w.nx, w.ny, w.nz], "max_1step", "phi", float(e)])
    assert e <= TOL_1STEP
