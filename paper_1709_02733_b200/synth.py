"""Seeded synthetic inputs for the elastic-FDTD forward/adjoint pair (H, H^T).

This module holds NONE of the method's arithmetic: it only builds material volumes, initial
pressure volumes, receiver coordinates and the parameter record, which the CUDA path
(`paper_1709_02733_b200.binding`) and the CPU oracle (`oracle/`) both consume.  Neither of those
imports the other; both may import this.

The inputs STAND IN for the paper's CT-derived skull, cortical-vessel phantom and 11x400-ring
scanner (Sec. 6.1.1), which are not available; shapes and value ranges follow
BASELINE.json's configs and the paper's parameter sets.  The recipe is
restated in DESIGN.md ("Input recipe").

Conventions
-----------
* volumes are float32, C-order ``[nz][ny][nx]`` (x fastest; x,y,z = paper directions 1,2,3);
* node (x,y,z) sits at physical (x*h, y*h, z*h); receiver coordinates are float64 metres, ``[L][3]``
  in (x,y,z) order;
* ``lam``/``mu`` in Pa, ``rho`` in kg/m^3, ``alpha`` in 1/s (paper's diffusive absorption, Eq. 3a).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, asdict

import numpy as np

SEED_BASE = 170902733


@dataclass
class Params:
    """Mirror of the C `pact_params` record (include/pact.h)."""
    nx: int
    ny: int
    nz: int
    h: float
    dt: float
    nt: int
    npml: int
    pml_R: float = 1e-4
    pml_cref: float = 1500.0
    pml_beta_max: float = math.pi * 0.25e6

    @property
    def N(self) -> int:
        return self.nx * self.ny * self.nz

    def as_dict(self):
        return asdict(self)


@dataclass
class Problem:
    """One synthetic workload: parameters, medium, receivers, a p0 volume."""
    name: str
    prm: Params
    lam: np.ndarray      # float32 [nz][ny][nx]
    mu: np.ndarray       # float32
    rho: np.ndarray      # float32
    alpha: np.ndarray    # float32
    rcv: np.ndarray      # float64 [L][3] metres
    p0: np.ndarray       # float32 [nz][ny][nx]
    meta: dict = field(default_factory=dict)

    @property
    def L(self) -> int:
        return int(self.rcv.shape[0])


# --------------------------------------------------------------------------- helpers

CFL_LIMIT = 6.0 / (7.0 * math.sqrt(3.0))   # c_max*dt/h <= 6/(7*sqrt(3))


def stable_dt(h: float, c_max: float, fraction: float = 0.5) -> float:
    """Time step at `fraction` of the scheme's stability limit (reading G16)."""
    return fraction * CFL_LIMIT * h / c_max


def lame_from_speeds(cp, cs, rho):
    """(lambda, mu) from compressional / shear speeds and density; Eq. 2."""
    cp = np.asarray(cp, dtype=np.float64)
    cs = np.asarray(cs, dtype=np.float64)
    rho = np.asarray(rho, dtype=np.float64)
    mu = rho * cs * cs
    lam = rho * (cp * cp - 2.0 * cs * cs)
    return lam, mu


def grid_coords(prm: Params):
    """Physical node coordinates as broadcastable (z,y,x) arrays."""
    z = (np.arange(prm.nz, dtype=np.float64) * prm.h)[:, None, None]
    y = (np.arange(prm.ny, dtype=np.float64) * prm.h)[None, :, None]
    x = (np.arange(prm.nx, dtype=np.float64) * prm.h)[None, None, :]
    return x, y, z


def centre(prm: Params) -> np.ndarray:
    return 0.5 * prm.h * np.array([prm.nx - 1, prm.ny - 1, prm.nz - 1], dtype=np.float64)


def fibonacci_sphere(L: int, radius: float, c: np.ndarray) -> np.ndarray:
    i = np.arange(L, dtype=np.float64)
    zz = 1.0 - (2.0 * i + 1.0) / L
    ph = i * math.pi * (3.0 - math.sqrt(5.0))
    rr = np.sqrt(np.maximum(0.0, 1.0 - zz * zz))
    pts = np.stack([rr * np.cos(ph), rr * np.sin(ph), zz], axis=1)
    return c[None, :] + radius * pts


def fibonacci_hemisphere(L: int, radius: float, c: np.ndarray) -> np.ndarray:
    i = np.arange(L, dtype=np.float64)
    zz = (i + 0.5) / L
    ph = i * math.pi * (3.0 - math.sqrt(5.0))
    rr = np.sqrt(np.maximum(0.0, 1.0 - zz * zz))
    pts = np.stack([rr * np.cos(ph), rr * np.sin(ph), zz], axis=1)
    return c[None, :] + radius * pts


def radius_field(prm: Params, c: np.ndarray) -> np.ndarray:
    x, y, z = grid_coords(prm)
    return np.sqrt((x - c[0]) ** 2 + (y - c[1]) ** 2 + (z - c[2]) ** 2)


def _gaussian_blob(prm: Params, c, sigma, amp, cut=3.5, out=None):
    """Add amp*exp(-r^2/(2 sigma^2)), zeroed beyond cut*sigma, into `out` (float64 volume)."""
    if out is None:
        out = np.zeros((prm.nz, prm.ny, prm.nx), dtype=np.float64)
    h = prm.h
    rad = cut * sigma
    lo = [max(0, int(math.floor((c[a] - rad) / h))) for a in range(3)]
    hi = [min(n - 1, int(math.ceil((c[a] + rad) / h))) for a, n in zip(range(3), (prm.nx, prm.ny, prm.nz))]
    xs = np.arange(lo[0], hi[0] + 1) * h
    ys = np.arange(lo[1], hi[1] + 1) * h
    zs = np.arange(lo[2], hi[2] + 1) * h
    r2 = ((zs[:, None, None] - c[2]) ** 2 + (ys[None, :, None] - c[1]) ** 2
          + (xs[None, None, :] - c[0]) ** 2)
    g = amp * np.exp(-r2 / (2.0 * sigma * sigma))
    g[r2 > rad * rad] = 0.0
    out[lo[2]:hi[2] + 1, lo[1]:hi[1] + 1, lo[0]:hi[0] + 1] += g
    return out


def _catmull_rom(ctrl: np.ndarray, samples_per_seg: int) -> np.ndarray:
    """Uniform Catmull-Rom curve through ctrl[0..n-1] (end points duplicated)."""
    P = np.vstack([ctrl[0], ctrl, ctrl[-1]])
    out = []
    t = np.linspace(0.0, 1.0, samples_per_seg, endpoint=False)[:, None]
    for i in range(1, len(P) - 2):
        p0, p1, p2, p3 = P[i - 1], P[i], P[i + 1], P[i + 2]
        out.append(0.5 * ((2 * p1) + (-p0 + p2) * t + (2 * p0 - 5 * p1 + 4 * p2 - p3) * t * t
                          + (-p0 + 3 * p1 - 3 * p2 + p3) * t ** 3))
    out.append(P[-2][None, :])
    return np.vstack(out)


def _paint_tubes(prm: Params, curves, tube_r: float) -> np.ndarray:
    """p0 = 1 within tube_r of any curve sample (float32 volume)."""
    vol = np.zeros((prm.nz, prm.ny, prm.nx), dtype=np.float32)
    h = prm.h
    k = int(math.ceil(tube_r / h)) + 1
    off = np.arange(-k, k + 1)
    for curve in curves:
        for p in curve:
            ic = np.round(p / h).astype(int)
            xs = ic[0] + off
            ys = ic[1] + off
            zs = ic[2] + off
            xs = xs[(xs >= 0) & (xs < prm.nx)]
            ys = ys[(ys >= 0) & (ys < prm.ny)]
            zs = zs[(zs >= 0) & (zs < prm.nz)]
            if len(xs) == 0 or len(ys) == 0 or len(zs) == 0:
                continue
            r2 = ((zs[:, None, None] * h - p[2]) ** 2 + (ys[None, :, None] * h - p[1]) ** 2
                  + (xs[None, None, :] * h - p[0]) ** 2)
            sub = vol[zs[0]:zs[-1] + 1, ys[0]:ys[-1] + 1, xs[0]:xs[-1] + 1]
            sub[r2 <= tube_r * tube_r] = 1.0
    return vol


def _smooth_local(vol: np.ndarray, sigma_cells: float) -> np.ndarray:
    """Gaussian smoothing restricted to the bounding box of the support (+4 sigma)."""
    from scipy.ndimage import gaussian_filter
    nzs = np.nonzero(vol)
    if len(nzs[0]) == 0:
        return vol
    pad = int(math.ceil(4 * sigma_cells)) + 1
    sl = tuple(slice(max(0, int(a.min()) - pad), min(n, int(a.max()) + pad + 1))
               for a, n in zip(nzs, vol.shape))
    out = vol.copy()
    out[sl] = gaussian_filter(vol[sl].astype(np.float32), sigma=sigma_cells, mode="constant")
    return out


def _clear_near_pml(prm: Params, vol: np.ndarray, guard: int = 2):
    """Enforce 'support at least 2 grid positions away from the PML'."""
    m = prm.npml + guard
    if m <= 0:
        return vol
    vol[:m, :, :] = 0
    vol[-m:, :, :] = 0
    vol[:, :m, :] = 0
    vol[:, -m:, :] = 0
    vol[:, :, :m] = 0
    vol[:, :, -m:] = 0
    return vol


# --------------------------------------------------------------------------- BASELINE configs

WATER = dict(cp=1500.0, cs=0.0, rho=1000.0)
BONE = dict(cp=3000.0, cs=1600.0, rho=2000.0)      # G18 end point (porosity 0)
_GRID = {
    1: dict(n=64, h=0.25e-3, npml=10, nt=300, L=128),
    2: dict(n=128, h=0.20e-3, npml=10, nt=1000, L=512),
    3: dict(n=256, h=0.15e-3, npml=10, nt=2000, L=2048, shell=(11e-3, 14e-3), cap=(8e-3, 10e-3),
            tubes=6, rcv_r=16e-3),
    4: dict(n=512, h=0.15e-3, npml=16, nt=4000, L=4096, shell=(24e-3, 30e-3), cap=(17e-3, 19e-3),
            tubes=12, rcv_r=33.5e-3),
    5: dict(n=384, h=0.15e-3, npml=10, nt=3000, L=2048, shell=(18e-3, 22.5e-3), cap=(11e-3, 13e-3),
            tubes=8, rcv_r=25.5e-3),
}


def _finish(name, prm, cp, cs, rho, alpha, rcv, p0, meta=None) -> Problem:
    lam, mu = lame_from_speeds(cp, cs, rho)
    shape = (prm.nz, prm.ny, prm.nx)
    f32 = lambda a: np.ascontiguousarray(np.broadcast_to(np.asarray(a, dtype=np.float64), shape)
                                         .astype(np.float32))
    return Problem(name=name, prm=prm, lam=f32(lam), mu=f32(mu), rho=f32(rho), alpha=f32(alpha),
                   rcv=np.ascontiguousarray(rcv, dtype=np.float64),
                   p0=np.ascontiguousarray(p0, dtype=np.float32), meta=meta or {})


def config1(nt: int | None = None) -> Problem:
    """64^3 homogeneous water, one Gaussian ball, 128 receivers on a Fibonacci sphere r=7 mm."""
    g = _GRID[1]
    rng = np.random.default_rng(SEED_BASE + 1)
    n, h = g["n"], g["h"]
    prm = Params(n, n, n, h, stable_dt(h, WATER["cp"]), nt or g["nt"], g["npml"],
                 pml_cref=WATER["cp"])
    c = centre(prm)
    cb = c + rng.uniform(-1e-3, 1e-3, size=3)
    p0 = _gaussian_blob(prm, cb, 1e-3, 1.0)
    p0 = _clear_near_pml(prm, p0)
    rcv = fibonacci_sphere(g["L"], 7e-3, c)
    return _finish("C1", prm, WATER["cp"], 0.0, WATER["rho"], 0.0, rcv, p0, dict(blob=cb))


def skull_alpha_from_db(cp: float, db_per_mhz_cm: float = 0.5, f0_mhz: float = 1.0) -> float:
    """Reading G17: amplitude decay alpha/(2 c_l) Np/m at f0 = 1 MHz."""
    np_per_m = db_per_mhz_cm * f0_mhz * 100.0 / 8.686
    return 2.0 * cp * np_per_m


def config2(nt: int | None = None) -> Problem:
    """128^3 water + 2 mm homogeneous skull shell around brain; 8 Gaussian blobs; 512 receivers."""
    g = _GRID[2]
    rng = np.random.default_rng(SEED_BASE + 2)
    n, h = g["n"], g["h"]
    cmax = 2800.0
    prm = Params(n, n, n, h, stable_dt(h, cmax), nt or g["nt"], g["npml"], pml_cref=cmax)
    c = centre(prm)
    r = radius_field(prm, c)
    shell = (r >= 6e-3) & (r <= 8e-3)
    inside = r < 6e-3
    cp = np.where(shell, 2800.0, np.where(inside, 1540.0, 1500.0))
    cs = np.where(shell, 1500.0, 0.0)
    rho = np.where(shell, 1900.0, np.where(inside, 1040.0, 1000.0))
    alpha = np.where(shell, skull_alpha_from_db(2800.0), 0.0)
    p0 = np.zeros((n, n, n), dtype=np.float64)
    blobs = []
    for _ in range(8):
        while True:
            d = rng.uniform(-4.5e-3, 4.5e-3, size=3)
            if np.linalg.norm(d) < 4.5e-3:
                break
        amp = rng.uniform(0.5, 1.0)
        _gaussian_blob(prm, c + d, 0.5e-3, amp, out=p0)
        blobs.append((c + d, amp))
    p0[~inside] = 0.0
    rcv = fibonacci_sphere(g["L"], 9.5e-3, c)
    return _finish("C2", prm, cp, cs, rho, alpha, rcv, p0, dict(blobs=blobs))


def _porous_skull(k: int, nt: int | None = None, n_override: int | None = None) -> Problem:
    """Configs 3-5: porosity-mapped skull shell, vessel-like tubes, hemispherical receivers."""
    from scipy.ndimage import gaussian_filter
    g = _GRID[k]
    rng = np.random.default_rng(SEED_BASE + k)
    n, h = g["n"], g["h"]
    cmax = BONE["cp"]
    prm = Params(n, n, n, h, stable_dt(h, cmax), nt or g["nt"], g["npml"], pml_cref=cmax)
    c = centre(prm)
    r = radius_field(prm, c).astype(np.float32)
    r_in, r_out = g["shell"]
    shell = (r >= r_in) & (r <= r_out)
    # porosity: U(0,1) noise -> Gaussian filter (0.5 mm) -> min-max over the shell to [0, 0.6]
    noise = rng.random((n, n, n), dtype=np.float32)
    sm = gaussian_filter(noise, sigma=0.5e-3 / h, mode="wrap")
    del noise
    lo, hi = float(sm[shell].min()), float(sm[shell].max())
    por = np.clip((sm - lo) / (hi - lo), 0.0, 1.0) * 0.6
    del sm
    por = np.where(shell, por, 1.0).astype(np.float32)     # outside the shell: pure water
    # G18: q = bone*(1-phi) + water*phi
    cp = BONE["cp"] * (1 - por) + WATER["cp"] * por
    cs = BONE["cs"] * (1 - por) + WATER["cs"] * por
    rho = BONE["rho"] * (1 - por) + WATER["rho"] * por
    alpha = np.where(shell, 0.1e6 * (1 - por), 0.0)          # paper's skull 0.1 /us
    # tubes on the upper cap, radius in `cap`
    c0, c1 = g["cap"]
    curves = []
    for _ in range(g["tubes"]):
        az0 = rng.uniform(0, 2 * math.pi)
        ctrl = []
        for j in range(4):
            rad = rng.uniform(c0, c1)
            polar = rng.uniform(0.05, 0.9)                   # angle from +z, radians
            az = az0 + rng.uniform(-0.8, 0.8)
            ctrl.append(c + rad * np.array([math.sin(polar) * math.cos(az),
                                            math.sin(polar) * math.sin(az), math.cos(polar)]))
        curves.append(_catmull_rom(np.array(ctrl), 96))
    p0 = _paint_tubes(prm, curves, 0.3e-3)
    p0 = _smooth_local(p0, 1.0)
    p0[r >= r_in - 2 * h] = 0.0                              # p0 lives in the fluid inside the skull
    p0 = _clear_near_pml(prm, p0)
    rcv = fibonacci_hemisphere(g["L"], g["rcv_r"], c)
    return _finish(f"C{k}", prm, cp, cs, rho, alpha, rcv, p0, dict(tubes=len(curves)))


def config3(nt=None): return _porous_skull(3, nt)
def config4(nt=None): return _porous_skull(4, nt)
def config5(nt=None): return _porous_skull(5, nt)


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def make_config(k: int, nt: int | None = None) -> Problem:
    """BASELINE.json config k (1-based). `nt` overrides the number of samples (truncated runs)."""
    return CONFIGS[k](nt)


# --------------------------------------------------------------------------- small test problems

def random_problem(nx=16, ny=12, nz=14, nt=25, npml=3, L=7, seed=0, fluid_fraction=0.4,
                   lossy=True, cfl_fraction=0.9, h=0.2e-3, smooth=False) -> Problem:
    """Random heterogeneous medium with fluid (mu=0) cells, absorption and off-node receivers.

    Used by the adjoint dot test, the brute-force pins and the GPU parity tests (ragged sizes)."""
    rng = np.random.default_rng(SEED_BASE + 1000 + seed)
    shape = (nz, ny, nx)
    cp = rng.uniform(1500.0, 3000.0, size=shape)
    cs = rng.uniform(600.0, 0.5 * cp)
    fluid = rng.random(shape) < fluid_fraction
    cs = np.where(fluid, 0.0, cs)
    rho = rng.uniform(1000.0, 2000.0, size=shape)
    alpha = rng.uniform(0.0, 1e5, size=shape) if lossy else np.zeros(shape)
    if smooth:
        from scipy.ndimage import gaussian_filter
        cp = gaussian_filter(cp, 1.5)
        rho = gaussian_filter(rho, 1.5)
        cs = np.where(fluid, 0.0, gaussian_filter(cs, 1.5))
    cmax = float(cp.max())
    prm = Params(nx, ny, nz, h, stable_dt(h, cmax, cfl_fraction), nt, npml, pml_cref=cmax)
    ext = np.array([nx - 1, ny - 1, nz - 1], dtype=np.float64) * h
    rcv = rng.uniform(0.02, 0.98, size=(L, 3)) * ext[None, :]
    if L >= 2:
        rcv[1] = np.round(rcv[1] / h) * h          # one receiver exactly on a node
    if L >= 3:
        rcv[2] = rcv[0] + 0.1 * h * rng.uniform(-1, 1, 3)   # two receivers sharing a cell
        rcv[2] = np.clip(rcv[2], 0.0, ext)
    if L >= 4:
        rcv[3] = ext                                # the far corner (clamped cell)
    p0 = rng.standard_normal(shape)
    return _finish(f"rand{seed}", prm, cp, cs, rho, alpha, rcv, p0, dict(seed=seed))


def random_vectors(prob: Problem, seed=0):
    """x ~ N(0,1)^N and y ~ N(0,1)^{M x L} for the inner-product test."""
    rng = np.random.default_rng(SEED_BASE + 2000 + seed)
    prm = prob.prm
    x = rng.standard_normal((prm.nz, prm.ny, prm.nx))
    y = rng.standard_normal((prm.nt, prob.L))
    return x, y


def custom_problem(name, prm: Params, cp, cs, rho, alpha, rcv, p0) -> Problem:
    """Problem from speed/density volumes or scalars (broadcast to the grid)."""
    return _finish(name, prm, cp, cs, rho, alpha, np.asarray(rcv, dtype=np.float64).reshape(-1, 3),
                   np.broadcast_to(np.asarray(p0, dtype=np.float64), (prm.nz, prm.ny, prm.nx)))


def gaussian_ball(prm: Params, c, sigma, amp=1.0, cut=3.5) -> np.ndarray:
    """amp*exp(-r^2/(2 sigma^2)) on the nodes, zero beyond cut*sigma (float64 volume)."""
    return _gaussian_blob(prm, np.asarray(c, dtype=np.float64), sigma, amp, cut)


def fluid_version(prob: Problem) -> Problem:
    """The same workload with the shear modulus set to zero everywhere and the longitudinal speed kept
    (lambda' = lambda + 2 mu = rho c_l^2): the medium of the paper's H^dagger_{mu=0} ("the shear
    modulus of the elastic medium was set to zero", the skull's longitudinal speed being a free parameter)."""
    from dataclasses import replace
    lam = (prob.lam.astype(np.float64) + 2.0 * prob.mu.astype(np.float64)).astype(np.float32)
    return replace(prob, name=prob.name + "-fluid", lam=lam, mu=np.zeros_like(prob.mu))


def crop(prob: Problem, origin, n, nt: int) -> Problem:
    """Sub-block [z0:z0+n, y0:y0+n, x0:x0+n] of a problem's volumes with the receivers that fall
    inside it (shifted to the block's origin) and `nt` samples — a bounded sample of the same
    workload for timing the CPU oracle (bench.py `cpu_baseline`, `--impl reference`)."""
    from dataclasses import replace
    x0, y0, z0 = (int(v) for v in origin)
    sl = (slice(z0, z0 + n), slice(y0, y0 + n), slice(x0, x0 + n))
    prm = replace(prob.prm, nx=n, ny=n, nz=n, nt=nt)
    r = prob.rcv - np.array([x0, y0, z0], dtype=np.float64) * prob.prm.h
    keep = np.all((r >= 0.0) & (r <= (n - 1) * prob.prm.h), axis=1)
    cut = lambda a: None if a is None else np.ascontiguousarray(a[sl])
    return Problem(name=f"{prob.name}-crop{n}", prm=prm, lam=cut(prob.lam), mu=cut(prob.mu), rho=cut(prob.rho),
                   alpha=cut(prob.alpha), rcv=np.ascontiguousarray(r[keep]), p0=cut(prob.p0),
                   meta=dict(origin=(x0, y0, z0), parent=prob.name))
