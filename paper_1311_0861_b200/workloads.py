"""Seeded synthetic inputs for the five BASELINE.json configs (numpy only).

This module serves both the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic: it only evaluates analytic initial conditions at cell centres and packs
them into the conserved fields the scheme carries (PAPER.md:41 last line, rho*E = rho*eps +
rho*v^2/2, nE_ij = Pi_ij + n*u_i*u_j).  It imports neither the CUDA binding nor
oracle/.  The paper uses no dataset: its workloads are analytic initial states,
so these configs stand in for them (recipe and the choices BASELINE.json leaves open: DESIGN.md).

Every workload can be generated slab by slab along z (`fields(z0, z1)`), bit-identically to
generating it whole, so a 512^3 state never has to exist on the host in one piece.
Arrays are float64 with shape (z, y, x), x fastest.
"""
from dataclasses import dataclass, field

import numpy as np

GAS, STARS = 1, 2
POISSON_NONE, POISSON_PERIODIC, POISSON_ISOLATED = 0, 1, 2
BC_PERIODIC, BC_OUTFLOW = 0, 1

GAS_FIELDS = ["rho", "mx", "my", "mz", "E"]
STAR_FIELDS = ["n", "nux", "nuy", "nuz", "Exx", "Exy", "Exz", "Eyy", "Eyz", "Ezz"]


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    h: float
    components: int
    poisson: int
    gamma: float
    bc: tuple
    cfl: float
    steps: int
    G: float = 1.0
    t_end: float = None
    _gen: object = field(default=None, repr=False)

    @property
    def cells(self):
        return self.nx * self.ny * self.nz

    @property
    def field_names(self):
        return (GAS_FIELDS if self.components & GAS else []) + (STAR_FIELDS if self.components & STARS else [])

    def fields(self, z0=0, z1=None):
        """Conserved fields of the z-slab [z0, z1) as {name: array (z1-z0, ny, nx)}."""
        z1 = self.nz if z1 is None else z1
        return self._gen(z0, z1)

    def state(self):
        return self.fields(0, self.nz)

    def fill(self, out, slab=8, threads=None):
        """Generate the state slab by slab (in a thread pool) into preallocated arrays
        out[name] of shape (nz, ny, nx), e.g. views of pinned host tensors."""
        import os
        from concurrent.futures import ThreadPoolExecutor

        def work(z0):
            z1 = min(self.nz, z0 + slab)
            for k, v in self.fields(z0, z1).items():
                out[k][z0:z1] = v

        threads = threads or min(32, os.cpu_count() or 1)
        with ThreadPoolExecutor(max_workers=threads) as ex:
            list(ex.map(work, range(0, self.nz, slab)))
        return out


def _centres(n, h, lo=0, hi=None):
    hi = n if hi is None else hi
    return (np.arange(lo, hi, dtype=np.float64) + 0.5) * h


def _pack_gas(rho, vx, vy, vz, p, gamma):
    return {"rho": rho, "mx": rho * vx, "my": rho * vy, "mz": rho * vz,
            "E": p / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy + vz * vz)}


# ------------------------------------------------------------------------------------------------
# config 1: Sod shock tube along an axis, embedded in 3-D (PAPER.md:223-225 kind of test)
# ------------------------------------------------------------------------------------------------
def sod(n=128, nt=4, axis=0, gamma=1.4, left=(1.0, 0.0, 1.0), right=(0.125, 0.0, 0.1), x0=0.5,
        t_end=0.2, cfl=0.2, components=GAS):
    """Tube of n cells along `axis` (0=x,1=y,2=z), nt cells across; states are (rho, v, p).

    With components=STARS the same tube is set up for the collisionless component with
    n=rho, u=v along the axis and Pi = p * identity (used for the gas<->BME equivalence pin).
    """
    dims = [nt, nt, nt]
    dims[axis] = n
    nx, ny, nz = dims
    h = 1.0 / n
    bc = [BC_PERIODIC] * 3
    bc[axis] = BC_OUTFLOW

    def gen(z0, z1):
        shape = (z1 - z0, ny, nx)
        if axis == 0:
            s = _centres(nx, h)[None, None, :]
        elif axis == 1:
            s = _centres(ny, h)[None, :, None]
        else:
            s = _centres(nz, h, z0, z1)[:, None, None]
        L = np.broadcast_to(s < x0, shape)
        rho = np.where(L, left[0], right[0]).astype(np.float64)
        v = np.where(L, left[1], right[1]).astype(np.float64)
        p = np.where(L, left[2], right[2]).astype(np.float64)
        zero = np.zeros(shape)
        vel = [zero, zero, zero]
        vel[axis] = v
        out = {}
        if components & GAS:
            out.update(_pack_gas(rho, vel[0], vel[1], vel[2], p, gamma))
        if components & STARS:
            out.update(_pack_stars(rho, vel, [p, zero, zero, p, zero, p]))
        return out

    return Workload("sod", nx, ny, nz, h, components, POISSON_NONE, gamma, tuple(bc), cfl,
                    steps=0, t_end=t_end, _gen=gen)


def _pack_stars(n, u, Pi):
    """n, u[3], Pi[6] (xx,xy,xz,yy,yz,zz) -> conserved BME fields."""
    out = {"n": n, "nux": n * u[0], "nuy": n * u[1], "nuz": n * u[2]}
    pairs = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]
    for name, P, (i, j) in zip(STAR_FIELDS[4:], Pi, pairs):
        out[name] = P + n * u[i] * u[j]
    return out


# ------------------------------------------------------------------------------------------------
# config 2: smooth periodic gas perturbation, sum of 8 seeded Fourier modes
# ------------------------------------------------------------------------------------------------
def _fourier_field(seed, kmax, nmodes=8):
    rng = np.random.default_rng(seed)
    ks = []
    while len(ks) < nmodes:
        k = rng.integers(-kmax, kmax + 1, size=3)
        if 0 < (k * k).sum() <= kmax * kmax:
            ks.append(k)
    phases = rng.uniform(0.0, 2.0 * np.pi, size=nmodes)
    return np.array(ks), phases


def smooth_gas(n=256, gamma=5.0 / 3.0, kmax=8, amp=0.1, seed=2000, steps=100, cfl=0.3, dims=None,
               components=GAS):
    """rho = 1 + amp*S_0, v_d = amp*S_d, p = 1 on the periodic unit box (cubic cells, h = 1/nx).

    With STARS enabled the collisionless component gets its own seeded fields (seeds +4..+7):
    n = 1 + amp*S_4, u_d = amp*S_{4+d}, and a smooth anisotropic Pi built from one more field.
    """
    nx, ny, nz = dims or (n, n, n)
    h = 1.0 / nx
    modes = [_fourier_field(seed + q, kmax) for q in range(9)]

    def S(q, z0, z1):
        ks, ph = modes[q]
        x = _centres(nx, h)[None, None, :]
        y = _centres(ny, h)[None, :, None]
        z = _centres(nz, h, z0, z1)[:, None, None]
        acc = np.zeros((z1 - z0, ny, nx))
        for (kx, ky, kz), p in zip(ks, ph):
            acc += np.cos(2.0 * np.pi * (kx * x + ky * y + kz * z) + p)
        return acc / len(ph)

    def gen(z0, z1):
        out = {}
        if components & GAS:
            rho = 1.0 + amp * S(0, z0, z1)
            out.update(_pack_gas(rho, amp * S(1, z0, z1), amp * S(2, z0, z1), amp * S(3, z0, z1),
                                 np.ones_like(rho), gamma))
        if components & STARS:
            nn = 1.0 + amp * S(4, z0, z1)
            u = [amp * S(5, z0, z1), amp * S(6, z0, z1), amp * S(7, z0, z1)]
            a = amp * S(8, z0, z1)
            # symmetric positive-definite, smoothly varying, all six components distinct
            Pi = [1.0 + a, 0.2 * a + 0.05, -0.15 * a + 0.02, 0.8 - 0.5 * a, 0.1 * a - 0.03, 1.2 + 0.3 * a]
            out.update(_pack_stars(nn, u, Pi))
        return out

    return Workload("smooth_gas", nx, ny, nz, h, components, POISSON_NONE, gamma,
                    (BC_PERIODIC,) * 3, cfl, steps, _gen=gen)


# ------------------------------------------------------------------------------------------------
# config 3: cold self-gravitating sphere, rho ~ 1/r, isolated Poisson (stand-in for PAPER.md:296-298)
# ------------------------------------------------------------------------------------------------
def collapse(n=256, gamma=5.0 / 3.0, radius=0.25, eint=0.05, background=1e-4, mass=1.0, steps=200,
             cfl=0.2, poisson=POISSON_ISOLATED):
    h = 1.0 / n
    bc = (BC_OUTFLOW,) * 3 if poisson == POISSON_ISOLATED else (BC_PERIODIC,) * 3

    def shape_fn(z0, z1):
        x = _centres(n, h)[None, None, :] - 0.5
        y = _centres(n, h)[None, :, None] - 0.5
        z = _centres(n, h, z0, z1)[:, None, None] - 0.5
        r = np.sqrt(x * x + y * y + z * z)
        inner = 1.0 / np.maximum(r, 0.5 * h)
        taper = (1.0 / radius) * np.exp(-(r - radius) / h)     # one-cell e-fold taper
        return np.where(r <= radius, inner, taper)

    total = 0.0
    for z0 in range(0, n, 32):
        total += float(shape_fn(z0, min(n, z0 + 32)).sum())
    A = mass / (total * h ** 3)

    def gen(z0, z1):
        rho = np.maximum(A * shape_fn(z0, z1), background)
        zero = np.zeros_like(rho)
        return _pack_gas(rho, zero, zero, zero, (gamma - 1.0) * eint * rho, gamma)

    return Workload("collapse", n, n, n, h, GAS, poisson, gamma, bc, cfl, steps, _gen=gen)


# ------------------------------------------------------------------------------------------------
# configs 4 and 5: exponential disks of gas + stars in circular rotation
# ------------------------------------------------------------------------------------------------
def _freeman_vc2_table(G, mass, rd, rmax, npts=4096):
    """v_c^2(R) of a razor-thin exponential disk (Freeman 1970), tabulated for np.interp."""
    from scipy.special import i0e, i1e, k0e, k1e
    R = np.linspace(0.0, rmax, npts)
    y = np.maximum(R / (2.0 * rd), 1e-12)
    sigma0 = mass / (2.0 * np.pi * rd * rd)
    # I0K0 - I1K1 with the exponentially scaled functions: the scalings cancel
    vc2 = 4.0 * np.pi * G * sigma0 * rd * y * y * (i0e(y) * k0e(y) - i1e(y) * k1e(y))
    vc2[0] = 0.0
    return R, vc2


@dataclass
class _Disk:
    centre: tuple       # box units
    axis: tuple         # unit normal
    bulk: tuple         # bulk velocity
    mass: float
    seed: int


def _disks(name, n, disks, steps, cfl, poisson, gamma, rd_cells, zd_cells, gas_fraction, eint,
           background, sigma2_frac, sigma2_min, noise, G, trunc=5.0):
    h = 1.0 / n
    rd, zd = rd_cells * h, zd_cells * h
    bc = (BC_PERIODIC,) * 3 if poisson != POISSON_ISOLATED else (BC_OUTFLOW,) * 3
    tables = [_freeman_vc2_table(G, d.mass, rd, 2.0) for d in disks]

    def geometry(d, z0, z1):
        x = _centres(n, h)[None, None, :] - d.centre[0]
        y = _centres(n, h)[None, :, None] - d.centre[1]
        z = _centres(n, h, z0, z1)[:, None, None] - d.centre[2]
        ax = np.asarray(d.axis, dtype=np.float64)
        ax = ax / np.sqrt((ax * ax).sum())
        zeta = x * ax[0] + y * ax[1] + z * ax[2]                 # height above the disk plane
        px, py, pz = x - zeta * ax[0], y - zeta * ax[1], z - zeta * ax[2]   # in-plane position
        R = np.sqrt(px * px + py * py + pz * pz)
        # exponential disk, smoothly truncated at ~5 scale lengths so that it is far below the
        # background where it meets the periodic seam or the box edge (no sharp jumps)
        prof = np.exp(-R / rd - np.abs(zeta) / zd - (R / (trunc * rd)) ** 4)
        # phi-hat = axis x (in-plane unit vector)
        Rs = np.maximum(R, 1e-300)
        ex, ey, ez = px / Rs, py / Rs, pz / Rs
        phix = ax[1] * ez - ax[2] * ey
        phiy = ax[2] * ex - ax[0] * ez
        phiz = ax[0] * ey - ax[1] * ex
        return prof, R, (phix, phiy, phiz)

    # analytic normalisation of the untruncated double-exponential profile: M = 4 pi A rd^2 zd
    norms = [d.mass / (4.0 * np.pi * rd * rd * zd) for d in disks]

    def gen(z0, z1):
        shape = (z1 - z0, n, n)
        rho = np.full(shape, background)
        nn = np.full(shape, background)
        gm = [np.zeros(shape) for _ in range(3)]                 # gas momentum
        sm = [np.zeros(shape) for _ in range(3)]                 # stellar momentum
        ekin_s = [np.zeros(shape) for _ in range(6)]             # sum_k n_k u_ki u_kj
        therm_s = np.full(shape, background * sigma2_min)        # sum_k n_k sigma_k^2
        pairs = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]
        for d, A, (Rt, vc2t) in zip(disks, norms, tables):
            prof, R, phat = geometry(d, z0, z1)
            dens = A * prof
            vc2 = np.interp(R, Rt, vc2t)
            vc = np.sqrt(vc2)
            xi = np.stack([np.random.default_rng([d.seed, k]).uniform(-1.0, 1.0, size=(n, n))
                           for k in range(z0, z1)])
            rho_d = gas_fraction * dens
            n_d = (1.0 - gas_fraction) * dens * (1.0 + noise * xi)
            vel = [vc * phat[i] + d.bulk[i] for i in range(3)]
            rho += rho_d
            nn += n_d
            for i in range(3):
                gm[i] += rho_d * vel[i]
                sm[i] += n_d * vel[i]
            for q, (i, j) in enumerate(pairs):
                ekin_s[q] += n_d * vel[i] * vel[j]
            therm_s += n_d * np.maximum(sigma2_frac * vc2, sigma2_min)
        out = {"rho": rho, "mx": gm[0], "my": gm[1], "mz": gm[2],
               "E": rho * eint + 0.5 * (gm[0] ** 2 + gm[1] ** 2 + gm[2] ** 2) / rho}
        out.update({"n": nn, "nux": sm[0], "nuy": sm[1], "nuz": sm[2]})
        for q, name in enumerate(STAR_FIELDS[4:]):
            out[name] = ekin_s[q] + (therm_s if pairs[q][0] == pairs[q][1] else 0.0)
        return out

    return Workload(name, n, n, n, h, GAS | STARS, poisson, gamma, bc, cfl, steps, G=G, _gen=gen)


def _disk_scales(n, rd_cells, zd_cells):
    # BASELINE.json: scale length 0.05 and scale height 0.005 box lengths; reduced-size cases
    # pass the scales in cells instead so that the structure stays resolved.
    return (0.05 * n if rd_cells is None else rd_cells), (0.005 * n if zd_cells is None else zd_cells)


def disk(n=256, steps=100, cfl=0.2, poisson=POISSON_PERIODIC, gamma=5.0 / 3.0, rd_cells=None,
         zd_cells=None, gas_fraction=0.2, eint=0.05, background=1e-4, sigma2_frac=0.1, sigma2_min=0.01,
         noise=0.01, G=1.0, seed=4):
    rd_cells, zd_cells = _disk_scales(n, rd_cells, zd_cells)
    d = [_Disk((0.5, 0.5, 0.5), (0.0, 0.0, 1.0), (0.0, 0.0, 0.0), 1.0, seed)]
    return _disks("disk", n, d, steps, cfl, poisson, gamma, rd_cells, zd_cells, gas_fraction, eint,
                  background, sigma2_frac, sigma2_min, noise, G)


def two_disks(n=512, steps=50, cfl=0.2, poisson=POISSON_PERIODIC, gamma=5.0 / 3.0, rd_cells=None,
              zd_cells=None, gas_fraction=0.2, eint=0.05, background=1e-4, sigma2_frac=0.1,
              sigma2_min=0.01, noise=0.01, G=1.0, seeds=(5, 6)):
    rd_cells, zd_cells = _disk_scales(n, rd_cells, zd_cells)
    s, c = np.sin(np.pi / 6.0), np.cos(np.pi / 6.0)
    d = [_Disk((0.3, 0.5, 0.5), (0.0, 0.0, 1.0), (+0.15, 0.0, 0.0), 0.5, seeds[0]),
         _Disk((0.7, 0.5, 0.5), (s, 0.0, c), (-0.15, 0.0, 0.0), 0.5, seeds[1])]
    return _disks("two_disks", n, d, steps, cfl, poisson, gamma, rd_cells, zd_cells, gas_fraction, eint,
                  background, sigma2_frac, sigma2_min, noise, G)


def config(i, **kw):
    """The i-th BASELINE.json config (1-based) at its full size unless overridden."""
    return {1: sod, 2: smooth_gas, 3: collapse, 4: disk, 5: two_disks}[i](**kw)
