"""Pins for the CPU oracle (oracle/) against what the paper and the mathematics fix.

Each test names the passage it pins.  None of them touches the CUDA path.
"""
import math
import os
from dataclasses import replace

import numpy as np
import pytest

from paper_1709_02733_b200 import synth
from oracle.oracle import Oracle
from oracle import bruteforce as bf

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")) as fh:
    for line in fh:
        if line.strip() and not line.startswith("#"):
            k, v = line.split()[:2]
            GOLD[k] = float(v)


def rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / max(np.linalg.norm(np.ravel(b)), 1e-300)


# ----------------------------------------------------------------------------- adjointness

@pytest.mark.parametrize("seed,npml,lossy", [(0, 3, True), (1, 0, False), (2, 2, True)])
def test_dot_product_identity(seed, npml, lossy):
    """<Hx,y> = <x,H^T y>, random heterogeneous medium with fluid cells,
    absorption, C-PML and off-node receivers; north_star bar 1e-12."""
    pb = synth.random_problem(nx=16, ny=12, nz=14, nt=25, npml=npml, L=7, seed=seed, lossy=lossy)
    o = Oracle.from_problem(pb)
    x, y = synth.random_vectors(pb, seed)
    a = np.vdot(o.forward(x), y)
    b = np.vdot(x, o.adjoint(y))
    assert abs(a - b) <= 1e-12 * abs(a)


def test_bruteforce_entrywise():
    """H from pact_oracle.c (columns via forward, rows via adjoint) equals the independent
    Kronecker assembly of Eq. 49/54/56 multiplied out (Eq. 58), entry by entry."""
    pb = synth.random_problem(nx=7, ny=6, nz=5, nt=5, npml=2, L=3, seed=3)
    H = bf.system_matrix(pb)
    o = Oracle.from_problem(pb)
    N, R = pb.prm.N, H.shape[0]
    Hf = np.stack([o.forward(np.eye(1, N, j).ravel()).ravel() for j in range(N)], axis=1)
    Ha = np.stack([o.adjoint(np.eye(1, R, i).ravel()).ravel() for i in range(R)], axis=0)
    sc = np.abs(H).max()
    assert np.abs(Hf - H).max() <= 1e-13 * sc
    assert np.abs(Ha - H).max() <= 1e-13 * sc


def test_bruteforce_no_pml_ragged():
    pb = synth.random_problem(nx=5, ny=7, nz=6, nt=4, npml=0, L=4, seed=4)
    H = bf.system_matrix(pb)
    o = Oracle.from_problem(pb)
    N = pb.prm.N
    Hf = np.stack([o.forward(np.eye(1, N, j).ravel()).ravel() for j in range(N)], axis=1)
    assert np.abs(Hf - H).max() <= 1e-13 * np.abs(H).max()


# ----------------------------------------------------------------------------- IC and sampling

def test_first_sample_is_trilinear_p0():
    """tau = -1/3 I (Eq. 21) with Theta = -R (Eq. 23) gives p^_0 = R p0 (reading G1); R is
    trilinear interpolation, exact for a field affine in each coordinate."""
    assert GOLD["tau_scale"] * 3 * GOLD["theta_scale"] == pytest.approx(1.0)
    pb = synth.random_problem(nx=9, ny=8, nz=7, nt=2, npml=0, L=12, seed=5)
    prm = pb.prm
    z, y, x = np.meshgrid(np.arange(prm.nz), np.arange(prm.ny), np.arange(prm.nx), indexing="ij")
    aff = lambda X, Y, Z: 0.3 + 1.5 * X - 0.7 * Y + 0.2 * Z + 0.11 * X * Y * Z   # trilinear
    p0 = aff(x * prm.h, y * prm.h, z * prm.h)
    o = Oracle.from_problem(pb)
    d0 = o.forward(p0)[0]
    expect = aff(pb.rcv[:, 0], pb.rcv[:, 1], pb.rcv[:, 2])
    assert np.abs(d0 - expect).max() <= 1e-14 * np.abs(expect).max()
    for l in range(pb.L):
        nodes, w = o.receiver_row(l)
        assert abs(w.sum() - 1.0) < 1e-14 and (w >= 0).all()


# ----------------------------------------------------------------------------- one step, closed form

def test_one_step_polynomial_closed_form():
    """Eq. 8 is exact on cubics, so one step of Eq. 10 on a homogeneous lossless solid with a
    polynomial p0 has a closed form at interior points:
      u^i_{1/2} = -(dt/(3 rho)) d_i p0 at u^i's staggered position,
      s^ii_1 = -p0/3 - dt^2/(3 rho) (lam lap p0 + 2 mu d_i^2 p0) at nodes,
      s^ij_1 = -dt^2 mu/(3 rho) 2 d_i d_j p0 at the shear position.
    Pins the stencil weights and 1/h (Eq. 8), the staggered positions (Fig. 1 reading), the
    signs, the lambda/2mu mixing (Eq. 7c) and the -1/3 (Eq. 21)."""
    n, h = 14, 0.2e-3
    lam, mu, rho = GOLD["valid_solid_lambda"], GOLD["valid_solid_mu"], GOLD["valid_solid_rho"]
    cp = math.sqrt((lam + 2 * mu) / rho)
    cs = math.sqrt(mu / rho)
    prm = synth.Params(n, n + 1, n + 2, h, synth.stable_dt(h, cp, 0.5), 2, 0)
    dt = prm.dt
    X = lambda i: i * h * 1e3    # work in mm to keep numbers O(1)
    s = 1e3                       # d/dx in 1/m of a polynomial in mm
    P = lambda x, y, z: 1 + x + 2 * y - z + x * y - 0.5 * y * z + 0.3 * x * z + x * x * y - y * y * z \
        + 0.2 * x ** 3 - 0.1 * y ** 3 + 0.05 * z ** 3 + 0.4 * x * y * z
    Px = lambda x, y, z: 1 + y + 0.3 * z + 2 * x * y + 0.6 * x * x + 0.4 * y * z
    Py = lambda x, y, z: 2 + x - 0.5 * z + x * x - 2 * y * z - 0.3 * y * y + 0.4 * x * z
    Pz = lambda x, y, z: -1 - 0.5 * y + 0.3 * x - y * y + 0.15 * z * z + 0.4 * x * y
    Pxx = lambda x, y, z: 2 * y + 1.2 * x
    Pyy = lambda x, y, z: -2 * z - 0.6 * y
    Pzz = lambda x, y, z: 0.3 * z
    Pxy = lambda x, y, z: 1 + 2 * x + 0.4 * z
    Pxz = lambda x, y, z: 0.3 + 0.4 * y
    Pyz = lambda x, y, z: -0.5 - 2 * y + 0.4 * x
    zi, yi, xi = np.meshgrid(np.arange(prm.nz), np.arange(prm.ny), np.arange(prm.nx), indexing="ij")
    x, y, z = X(xi), X(yi), X(zi)
    hm = h * 1e3
    p0 = P(x, y, z)
    pb = synth.custom_problem("poly", prm, cp, cs, rho, 0.0, np.zeros((0, 3)), p0)
    lam32, mu32, rho32 = float(pb.lam.flat[0]), float(pb.mu.flat[0]), float(pb.rho.flat[0])
    o = Oracle.from_problem(pb)
    o.set_p0(p0)
    o.step()
    I = (slice(4, -4),) * 3
    k = -dt / (3 * rho32) * s
    chk = lambda got, want: np.abs(got[I] - want[I]).max() <= 1e-11 * np.abs(want[I]).max()
    assert chk(o.field("u1"), k * Px(x + hm / 2, y, z))
    assert chk(o.field("u2"), k * Py(x, y + hm / 2, z))
    assert chk(o.field("u3"), k * Pz(x, y, z + hm / 2))
    k2 = -dt * dt / (3 * rho32) * s * s
    lap = Pxx(x, y, z) + Pyy(x, y, z) + Pzz(x, y, z)
    base = GOLD["tau_scale"] * p0
    assert chk(o.field("s11"), base + k2 * (lam32 * lap + 2 * mu32 * Pxx(x, y, z)))
    assert chk(o.field("s22"), base + k2 * (lam32 * lap + 2 * mu32 * Pyy(x, y, z)))
    assert chk(o.field("s33"), base + k2 * (lam32 * lap + 2 * mu32 * Pzz(x, y, z)))
    assert chk(o.field("s12"), k2 * mu32 * 2 * Pxy(x + hm / 2, y + hm / 2, z))
    assert chk(o.field("s13"), k2 * mu32 * 2 * Pxz(x + hm / 2, y, z + hm / 2))
    assert chk(o.field("s23"), k2 * mu32 * 2 * Pyz(x, y + hm / 2, z + hm / 2))
    assert GOLD["stencil_inner"] + 3 * GOLD["stencil_outer"] == pytest.approx(1.0)  # consistency of Eq. 8


# ----------------------------------------------------------------------------- staggered coefficients

def test_staggered_coefficients():
    """rho, alpha: 2-point arithmetic means; mu at shear points: 4-point
    harmonic mean, zero next to fluid (reading G10)."""
    pb = synth.random_problem(nx=6, ny=5, nz=4, nt=2, npml=0, L=1, seed=6)
    o = Oracle.from_problem(pb)
    rho, al, mu = (pb.rho.astype(np.float64), pb.alpha.astype(np.float64), pb.mu.astype(np.float64))
    cl = lambda i, n: min(i, n - 1)
    prm = pb.prm
    for (x, y, z) in [(0, 0, 0), (2, 3, 1), (5, 4, 3), (5, 0, 3), (1, 4, 2)]:
        assert o.coef(0, 0, 0, x, y, z) == 0.5 * (rho[z, y, x] + rho[z, y, cl(x + 1, prm.nx)])
        assert o.coef(0, 1, 0, x, y, z) == 0.5 * (rho[z, y, x] + rho[z, cl(y + 1, prm.ny), x])
        assert o.coef(1, 2, 0, x, y, z) == 0.5 * (al[z, y, x] + al[cl(z + 1, prm.nz), y, x])
        four = [mu[z, y, x], mu[z, y, cl(x + 1, prm.nx)], mu[cl(z + 1, prm.nz), y, x],
                mu[cl(z + 1, prm.nz), y, cl(x + 1, prm.nx)]]
        want = 0.0 if min(four) == 0 else 4.0 / sum(1.0 / m for m in four)
        assert o.coef(2, 0, 2, x, y, z) == pytest.approx(want, rel=1e-15)


# ----------------------------------------------------------------------------- energy invariant

def _staggered_np(pb):
    return bf.staggered(pb)


def _energy(o, pb, u_prev):
    """E = 1/2 s^T C^-1 s + 1/2 u_{m+1/2}^T Q u_{m-1/2}; isotropic compliance per point."""
    rho_s, _, mu_s = _staggered_np(pb)
    lam = pb.lam.astype(np.float64)
    mu = pb.mu.astype(np.float64)
    s11, s22, s33 = o.field("s11"), o.field("s22"), o.field("s33")
    tr = s11 + s22 + s33
    if (mu > 0).all():
        # e_ii = (s_ii - lam/(3 lam + 2 mu) tr)/(2 mu)
        k = lam / (3 * lam + 2 * mu)
        en = 0.5 * ((s11 * (s11 - k * tr) + s22 * (s22 - k * tr) + s33 * (s33 - k * tr)) / (2 * mu)).sum()
        en += 0.5 * (o.field("s12") ** 2 / mu_s[(0, 1)]).sum()
        en += 0.5 * (o.field("s13") ** 2 / mu_s[(0, 2)]).sum()
        en += 0.5 * (o.field("s23") ** 2 / mu_s[(1, 2)]).sum()
    else:
        en = 0.5 * (s11 ** 2 / lam).sum()
    for a, name in enumerate(("u1", "u2", "u3")):
        en += 0.5 * (o.field(name) * rho_s[a] * u_prev[a]).sum()
    return en


@pytest.mark.parametrize("fluid", [False, True])
def test_energy_invariant(fluid):
    """Without PML and absorption the leapfrog of Eq. 10 conserves
    E_m = 1/2 s_m^T C^-1 s_m + 1/2 u_{m+1/2}^T Q u_{m-1/2} exactly (Psi = -dt C D^T, Phi = dt Q^-1 D
    with zero padding).  Pins Phi/Psi (Eq. 7b,c), the Lame mixing and the staggered coefficients."""
    pb = synth.random_problem(nx=12, ny=11, nz=10, nt=2, npml=0, L=1, seed=7,
                              fluid_fraction=1.0 if fluid else 0.0, lossy=False, cfl_fraction=0.9)
    o = Oracle.from_problem(pb)
    rng = np.random.default_rng(11)
    o.set_p0(rng.standard_normal(pb.p0.shape))
    if not fluid:   # general stress state, not only the isotropic initial one
        for nme in ("s11", "s22", "s33", "s12", "s13", "s23"):
            o.field(nme)[...] = rng.standard_normal(pb.p0.shape)
    u_prev = [o.field(n).copy() for n in ("u1", "u2", "u3")]
    E = []
    for m in range(1000):
        sig = {n: o.field(n).copy() for n in ("s11", "s22", "s33", "s12", "s13", "s23")}
        # E_m needs s_m with u_{m+1/2}: advance, then evaluate with the saved s_m
        o.step()
        u_new = [o.field(n).copy() for n in ("u1", "u2", "u3")]
        sig_new = {n: o.field(n).copy() for n in sig}
        for n in sig:
            o.field(n)[...] = sig[n]
        E.append(_energy(o, pb, u_prev))
        for n in sig:
            o.field(n)[...] = sig_new[n]
        u_prev = u_new
    E = np.array(E)
    assert np.abs(E - E[0]).max() <= 1e-12 * abs(E[0])


# ----------------------------------------------------------------------------- mu = 0 special case

def _acoustic_textbook(pb, nt):
    """Textbook staggered acoustic leapfrog (p at nodes, v at half points) with the Eq. 8
    stencil, zero padding, arithmetic rho: the system H reduces to when mu = 0."""
    prm = pb.prm
    h, dt = prm.h, prm.dt
    lam = pb.lam.astype(np.float64)
    rho_s, _, _ = bf.staggered(pb)
    c1, c2 = GOLD["stencil_inner"], GOLD["stencil_outer"]

    def pad(f, ax):
        w = [(0, 0)] * 3
        w[ax] = (2, 2)
        return np.pad(f, w)

    def sl(f, ax, o):
        n = f.shape[ax] - 4
        idx = [slice(None)] * 3
        idx[ax] = slice(2 + o, 2 + o + n)
        return f[tuple(idx)]

    def dplus(f, ax):
        g = pad(f, ax)
        return (c1 * (sl(g, ax, 1) - sl(g, ax, 0)) + c2 * (sl(g, ax, 2) - sl(g, ax, -1))) / h

    def dminus(f, ax):
        g = pad(f, ax)
        return (c1 * (sl(g, ax, 0) - sl(g, ax, -1)) + c2 * (sl(g, ax, 1) - sl(g, ax, -2))) / h

    p = pb.p0.astype(np.float64).copy()
    v = [np.zeros_like(p) for _ in range(3)]
    out = [p.copy()]
    for m in range(nt - 1):
        for a in range(3):
            v[a] -= dt / rho_s[a] * dplus(p, bf.AX[a])
        div = sum(dminus(v[a], bf.AX[a]) for a in range(3))
        p -= dt * lam * div
        out.append(p.copy())
    return out


def test_fluid_special_case_matches_textbook_acoustics():
    """mu = 0 everywhere: shear stresses stay exactly 0, s11 = s22 = s33 bit-identically, and
    p = -s11 follows the textbook acoustic staggered scheme."""
    pb = synth.random_problem(nx=13, ny=10, nz=11, nt=12, npml=0, L=5, seed=8, fluid_fraction=1.0,
                              lossy=False)
    o = Oracle.from_problem(pb)
    ref = _acoustic_textbook(pb, pb.prm.nt)
    o.set_p0(pb.p0.astype(np.float64))
    for m in range(pb.prm.nt):
        assert np.array_equal(o.field("s11"), o.field("s22"))
        assert np.array_equal(o.field("s11"), o.field("s33"))
        for nme in ("s12", "s13", "s23"):
            assert not o.field(nme).any()
        # -(s11+s22+s33)/3 ... with s_ii = -p/3 each, p = -(s11+s22+s33)
        p = -(o.field("s11") + o.field("s22") + o.field("s33"))
        assert np.abs(p - ref[m]).max() <= 1e-12 * np.abs(ref[m]).max()
        if m < pb.prm.nt - 1:
            o.step()


# ----------------------------------------------------------------------------- closed form (d'Alembert)

def _dalembert_gauss(r, t, c, sigma):
    """p(r,t) = [(r-ct) p0(|r-ct|) + (r+ct) p0(r+ct)]/(2r), p0 = exp(-r^2/(2 sigma^2))."""
    g = lambda s: np.exp(-s * s / (2 * sigma * sigma))
    return ((r - c * t) * g(np.abs(r - c * t)) + (r + c * t) * g(r + c * t)) / (2 * r)


def _closed_form_error(n, h, nt_factor):
    c, rho, sigma = GOLD["water_cl"], GOLD["water_rho"], 1e-3
    dt = synth.stable_dt(0.25e-3, c, 0.5) / nt_factor     # C1's dt, halved with h
    nt = int(110 * nt_factor)
    prm = synth.Params(n, n, n, h, dt, nt, 8 * nt_factor, pml_cref=c)
    ctr = synth.centre(prm)
    ang = np.linspace(0.3, 2.6, 6)
    rcv = np.stack([ctr + 3e-3 * np.array([math.sin(a) * math.cos(2 * a), math.sin(a) * math.sin(2 * a),
                                           math.cos(a)]) for a in ang])
    p0 = synth.gaussian_ball(prm, ctr, sigma, cut=6.0)
    pb = synth.custom_problem("cf", prm, c, 0.0, rho, 0.0, rcv, p0)
    d = Oracle.from_problem(pb).forward(pb.p0.astype(np.float64))
    t = (np.arange(nt) + 0.5) * dt              # reading G15: p^_m ~ p((m+1/2) dt) for m >= 1
    r = np.linalg.norm(rcv - ctr, axis=1)
    ex = _dalembert_gauss(r[None, :], t[:, None], c, sigma)
    ex_unshifted = _dalembert_gauss(r[None, :], (t - 0.5 * dt)[:, None], c, sigma)
    return rel(d[1:], ex[1:]), rel(d[1:], ex_unshifted[1:])


def test_closed_form_spherical_wave():
    """Homogeneous lossless fluid: spherically symmetric d'Alembert solution for a Gaussian
    ball (replaces the Cagniard-de Hoop comparison, whose numbers are not
    printed).  Pins physical units, dt, h and the time indexing (G12, G15)."""
    e1, e1_unshifted = _closed_form_error(48, 0.25e-3, 1)
    assert e1 <= 1.5e-2, e1
    # against p(m dt) instead of p((m+1/2) dt) the error is several times larger (G15)
    assert e1_unshifted >= 2.5 * e1, (e1, e1_unshifted)
    # second-order convergence when h and dt are halved together: measured 7.81e-3 -> 2.23e-3, ratio 3.49
    # (SURVEY 8(c) quotes "ratio >= 3.5" from a prototype with other receivers; DESIGN.md section 3 records 3.4)
    e2, _ = _closed_form_error(96, 0.125e-3, 2)
    assert e2 <= e1 / 3.4, (e1, e2)


def test_closed_form_uniform_sphere_n_pulse():
    """north_star's pin: a uniform sphere (p0 = 1 for r <= a, a = 10 h) in homogeneous lossless fluid radiates the
    N-shaped pulse p(r,t) = (r - ct)/(2r) for |r - ct| < a, 0 otherwise (r > a).  The jumps at |r - ct| = a ring
    on any grid (raw relative L2 27 % here: Gibbs / numerical dispersion of a staircase sphere), so the pin is on
    what the N shape fixes: the slope -c/(2r) of the ramp, its zero crossing at r = ct, and the time integral of
    the trace (a parabola arc, insensitive to the ringing).  Compared at t_m + dt/2 (reading G15).  A wrong tau or
    Theta scale, a time-index slip or a wrong c (lambda, rho, h, dt) moves slope or crossing far outside the bars."""
    c, rho, h = GOLD["water_cl"], GOLD["water_rho"], 0.25e-3
    a = 10 * h
    dt = synth.stable_dt(h, c, 0.5)
    r_rcv = 2.0 * a
    nt = int((r_rcv + a + 6 * h) / c / dt) + 4
    prm = synth.Params(64, 64, 64, h, dt, nt, 8, pml_cref=c)
    ctr = synth.centre(prm)
    ang = np.linspace(0.3, 2.6, 6)
    rcv = np.stack([ctr + r_rcv * np.array([math.sin(t) * math.cos(2 * t), math.sin(t) * math.sin(2 * t), math.cos(t)])
                    for t in ang])
    p0 = (synth.radius_field(prm, ctr) <= a).astype(np.float64)
    pb = synth.custom_problem("npulse", prm, c, 0.0, rho, 0.0, rcv, p0)
    d = Oracle.from_problem(pb).forward(pb.p0.astype(np.float64))
    t = (np.arange(nt) + 0.5) * dt
    rr = np.linalg.norm(rcv - ctr, axis=1)
    s = rr[None, :] - c * t[:, None]
    ex = np.where(np.abs(s) < a, s / (2 * rr[None, :]), 0.0)
    assert rel(d[1:], ex[1:]) <= 0.35                       # qualitative: the shape is there (measured 0.27)
    I, Iex = np.cumsum(d[1:], axis=0) * dt, np.cumsum(ex[1:], axis=0) * dt
    assert rel(I, Iex) <= 5e-2                              # measured 3.6e-2 (2.2e-2 at a = 16 h)
    for l in range(rr.size):
        m = np.abs(s[:, l]) < a - 3 * h                     # the ramp, away from the jumps
        A = np.stack([t[m], np.ones(int(m.sum()))], 1)
        (slope, icpt), *_ = np.linalg.lstsq(A, d[m, l], rcond=None)
        assert abs(slope / (-c / (2 * rr[l])) - 1.0) <= 3e-2        # measured <= 1.9e-2
        assert abs((-icpt / slope) * c / rr[l] - 1.0) <= 5e-3       # zero crossing at r = ct: measured <= 2.6e-3
        # sign pattern of an N: compression first (r - ct > 0), then rarefaction
        assert d[m, l][0] > 0 > d[m, l][-1]
        # support: long after the pulse has passed the trace is back near zero
        late = s[:, l] < -(a + 5 * h)
        assert np.abs(d[late, l]).max() <= 0.25 * d[:, l].max()


# ----------------------------------------------------------------------------- C-PML behaviour

def test_pml_tables_eq38():
    """b = exp(-(d+beta) dt), a = d/(d+beta) (b-1) (Eq. 38, kappa=1): a = 0, b = 1 outside the
    slabs; inside -1 < a < 0 < b < 1 and a/(b-1) = d/(d+beta) in (0,1], growing with depth."""
    pb = synth.random_problem(nx=40, ny=30, nz=26, nt=2, npml=6, L=1, seed=9)
    o = Oracle.from_problem(pb)
    for ax, n in enumerate((40, 30, 26)):
        t = o.pml_tables(ax)
        P = 6
        assert (t["a_int"][P:n - P] == 0).all() and (t["b_int"][P:n - P] == 1).all()
        assert (t["a_half"][P:n - 1 - P] == 0).all() and (t["b_half"][P:n - 1 - P] == 1).all()
        assert (t["a_int"][:P] < 0).all() and (t["a_int"][n - P:] < 0).all()
        assert (t["a_half"][:P] < 0).all() and (t["a_half"][n - 1 - P:] < 0).all()
        ratio = t["a_int"][:P] / (t["b_int"][:P] - 1)
        assert ((ratio > 0) & (ratio <= 1)).all() and (np.diff(ratio) < 0).all()
        # mirror symmetry of the profile: int table is symmetric, half table about n-1.5
        assert np.allclose(t["a_int"], t["a_int"][::-1], rtol=0, atol=1e-15)
        assert np.allclose(t["a_half"][:n - 1], t["a_half"][:n - 1][::-1], rtol=0, atol=1e-15)
    # Eq. 38 against the independently typed profile of bruteforce.py (the profile d(x), beta(x)
    # itself is reading G8: "parity unpinned" by the paper)
    a_i, b_i, a_h, b_h = bf.pml_profile(pb.prm, 40)
    t = o.pml_tables(0)
    assert np.allclose(t["a_int"], a_i, rtol=1e-14) and np.allclose(t["b_half"], b_h, rtol=1e-14)


def test_pml_eq38_worked_values():
    """Eq. 38a,b (kappa = 1 PAPER.md:422) against values worked by hand (tests/golden/
    paper_constants.txt).  With P = 2, R = 1/e, c_ref = 1600 m/s, h = 3 mm the profile of reading G8 has
    d0 = 3 c_ref / (2 P h) = 4e5 1/s; with beta_max = 4e5 1/s the int table holds (d, beta) = (4e5, 0) at
    depth 2 and (1e5, 2e5) at depth 1, the half table (2.25e5, 1e5) at depth 1.5 and (2.5e4, 3e5) at depth 0.5.
    Dropping beta from the exponent, inverting d/(d+beta), or using b - 1 with the wrong sign all fail here."""
    n, P = 12, 2
    prm = synth.Params(n, n, n, 3e-3, GOLD["eq38_dt"], 2, P, pml_R=math.exp(-1.0), pml_cref=1600.0, pml_beta_max=4e5)
    pb = synth.custom_problem("eq38", prm, 1500.0, 0.0, 1000.0, 0.0, synth.centre(prm)[None, :], np.zeros((n, n, n)))
    o = Oracle.from_problem(pb)
    want = {("int", 0): "d4e5_beta0", ("int", 1): "d1e5_beta2e5", ("half", 0): "d2.25e5_beta1e5",
            ("half", 1): "d2.5e4_beta3e5"}
    for ax in range(3):
        t = o.pml_tables(ax)
        for (kind, i), key in want.items():
            a, b = GOLD["eq38_a_" + key], GOLD["eq38_b_" + key]
            mirror = n - 1 - i if kind == "int" else n - 2 - i      # same depth in the far slab
            for j in (i, mirror):
                assert abs(t["a_" + kind][j] - a) <= 1e-13 * abs(a), (ax, kind, j)
                assert abs(t["b_" + kind][j] - b) <= 1e-13 * b, (ax, kind, j)


def test_pml_absorbs_and_is_transparent_early():
    """A Gaussian pulse in water: with a 10-cell C-PML the trace at a receiver equals (<=5e-4 of
    peak) the trace in a box so large that no reflection arrives; with no PML it does not; and
    before any boundary arrival PML and no-PML runs agree.  Memory variables stay zero while p0's
    support is >= 2 cells from the PML."""
    c, rho, h = 1500.0, 1000.0, 0.25e-3
    dt = synth.stable_dt(h, c, 0.5)
    nt = 200

    def run(n, npml):
        prm = synth.Params(n, n, n, h, dt, nt, npml, pml_cref=c)
        ctr = synth.centre(prm)
        rcv = np.stack([ctr + np.array([4e-3, 0.3e-3, -0.2e-3]), ctr + np.array([-1e-3, 3.7e-3, 1e-3])])
        p0 = synth.gaussian_ball(prm, ctr, 1e-3)
        pb = synth.custom_problem("pml", prm, c, 0.0, rho, 0.0, rcv, p0)
        o = Oracle.from_problem(pb)
        d = o.forward(pb.p0.astype(np.float64))
        return d, o, pb

    d_pml, o, pb = run(64, 10)
    d_big, _, _ = run(112, 0)        # reflection needs > 2*(56-16)*h/c = 13.3 us > nt*dt = 8.2 us
    d_none, _, _ = run(64, 0)
    peak = np.abs(d_big).max()
    assert np.abs(d_pml - d_big).max() <= 5e-4 * peak
    assert np.abs(d_none - d_big).max() >= 0.1 * peak
    early = int((32 - 16 - 14) * h / c / dt)   # nothing has reached the PML yet
    assert np.abs(d_pml[:early] - d_none[:early]).max() <= 1e-12 * peak
    o.set_p0(pb.p0.astype(np.float64))
    o.step()
    assert o.memvar_energy("phi") == 0.0 and o.memvar_energy("psi") == 0.0


# ----------------------------------------------------------------------------- absorption

def test_diffusive_absorption_decay():
    """Uniform alpha in Eq. 3a gives p_tt + alpha p_t = c^2 lap p.  With p = exp(-alpha t/2) q,
    q obeys the lossless wave equation up to alpha^2/4 (1e-3 of omega^2 here) with q(0) = p0,
    q_t(0) = (alpha/2) p0, whose spherically symmetric solution for a Gaussian ball is
    d'Alembert's plus alpha sigma^2/(4 c r) (g(r-ct) - g(r+ct)).  Pins J = I - dt A (Eq. 7a)."""
    c, rho, h, sigma = 1500.0, 1000.0, 0.25e-3, 1e-3
    alpha = GOLD["skull_alpha"]
    dt = synth.stable_dt(h, c, 0.5)
    nt = 130
    prm = synth.Params(56, 56, 56, h, dt, nt, 8, pml_cref=c)
    ctr = synth.centre(prm)
    rcv = np.stack([ctr + np.array([3.5e-3, 0.1e-3, 0.2e-3])])
    p0 = synth.gaussian_ball(prm, ctr, sigma, cut=6.0)
    d1 = Oracle.from_problem(synth.custom_problem("a1", prm, c, 0.0, rho, alpha, rcv, p0)).forward(p0)
    d0 = Oracle.from_problem(synth.custom_problem("a0", prm, c, 0.0, rho, 0.0, rcv, p0)).forward(p0)
    t = (np.arange(nt) + 0.5) * dt
    r = np.linalg.norm(rcv[0] - ctr)
    g = lambda s: np.exp(-s * s / (2 * sigma * sigma))
    lossless = _dalembert_gauss(r, t, c, sigma)
    q = lossless + alpha * sigma ** 2 / (4 * c * r) * (g(r - c * t) - g(r + c * t))
    # measured 1.60e-2, of which 1.47e-2 is the O(h^2) error the lossless run (alpha = 0, same grid) has against its
    # own closed form: what absorption adds is 1.3e-3 (the neglected alpha^2/4 term is 1.1e-3 of omega^2), inside
    # SURVEY 8(c)'s 1 % bar for J
    e_lossy = rel(d1[1:, 0], (np.exp(-alpha * t / 2) * q)[1:])
    e_lossless = rel(d0[1:, 0], lossless[1:])
    assert e_lossy <= 2e-2 and e_lossy - e_lossless <= 3e-3, (e_lossy, e_lossless)
    assert rel(d1[1:, 0], lossless[1:]) >= 0.1      # and the loss is not negligible
    # a wrong decay rate (alpha instead of alpha/2) is far outside the bar
    assert rel(d1[1:, 0], (np.exp(-alpha * t) * q)[1:]) >= 0.1


# ----------------------------------------------------------------------------- linearity, symmetry

def test_linearity_and_mirror_symmetry():
    pb = synth.random_problem(nx=12, ny=10, nz=9, nt=15, npml=2, L=6, seed=10)
    o = Oracle.from_problem(pb)
    rng = np.random.default_rng(3)
    x1, x2 = rng.standard_normal(pb.p0.shape), rng.standard_normal(pb.p0.shape)
    lhs = o.forward(2.0 * x1 - 0.5 * x2)
    rhs = 2.0 * o.forward(x1) - 0.5 * o.forward(x2)
    assert np.abs(lhs - rhs).max() <= 1e-12 * np.abs(lhs).max()


@pytest.mark.parametrize("perm", [(1, 0, 2), (2, 1, 0), (1, 2, 0)])
def test_axis_permutation_symmetry(perm):
    """Eq. 3 and its discretisation treat the three directions alike: permuting the axes of the
    medium, p0 and receiver coordinates permutes nothing in the data.  Catches a table, offset or
    coefficient applied along the wrong axis."""
    pb = synth.random_problem(nx=12, ny=10, nz=9, nt=15, npml=2, L=6, seed=10)
    d = Oracle.from_problem(pb).forward(pb.p0)
    prm = pb.prm
    n = (prm.nx, prm.ny, prm.nz)
    # new direction a is old direction perm[a]; numpy axis of direction a is 2 - a
    tr = lambda v: np.ascontiguousarray(np.transpose(v, [2 - perm[2 - k] for k in range(3)]))
    prm_p = replace(prm, nx=n[perm[0]], ny=n[perm[1]], nz=n[perm[2]])
    pb_p = synth.Problem("perm", prm_p, tr(pb.lam), tr(pb.mu), tr(pb.rho), tr(pb.alpha),
                         np.ascontiguousarray(pb.rcv[:, list(perm)]), tr(pb.p0))
    dp = Oracle.from_problem(pb_p).forward(pb_p.p0)
    assert np.abs(d - dp).max() <= 1e-12 * np.abs(d).max()


# ----------------------------------------------------------------------------- stability

def test_stability_limit():
    """c_max dt / h <= 6/(7 sqrt 3) (von Neumann for Eq. 8 + leapfrog, reading G11): a
    water/skull-shell medium stays bounded at 0.99x the limit, a homogeneous solid at 1.02x blows
    up.  Arithmetic rho/alpha averaging at the interfaces is what PAPER.md:289 prescribes 'to
    avoid instability'."""
    n, h = 28, 0.2e-3
    prm0 = synth.Params(n, n, n, h, 1.0, 1500, 0)
    r = synth.radius_field(prm0, synth.centre(prm0))
    shell = (r > 1.6e-3) & (r < 2.4e-3)
    cp = np.where(shell, GOLD["skull_cl"], GOLD["water_cl"])
    cs = np.where(shell, GOLD["skull_cs"], 0.0)
    rho = np.where(shell, GOLD["skull_rho"], GOLD["water_rho"])
    prm = replace(prm0, dt=synth.stable_dt(h, GOLD["skull_cl"], 0.99))
    rng = np.random.default_rng(5)
    p0 = rng.standard_normal((n, n, n))          # excites every mode, including Nyquist
    rcv = synth.centre(prm)[None, :] + 0.3e-3
    pb = synth.custom_problem("stab", prm, cp, cs, rho, 0.0, rcv, p0)
    d = Oracle.from_problem(pb).forward(p0)
    assert np.isfinite(d).all() and np.abs(d[-200:]).max() <= 10 * np.abs(d[:200]).max()
    prm_bad = replace(prm0, nt=300, dt=synth.stable_dt(h, GOLD["skull_cl"], 1.02))
    pb2 = synth.custom_problem("unst", prm_bad, GOLD["skull_cl"], GOLD["skull_cs"], GOLD["skull_rho"],
                               0.0, rcv, p0)
    d2 = Oracle.from_problem(pb2).forward(p0)
    assert (not np.isfinite(d2).all()) or np.abs(d2[-20:]).max() > 1e6 * np.abs(d2[:20]).max()


# ----------------------------------------------------------------------------- adjoint recursion order

def test_adjoint_recursion_matches_eq27():
    """Eq. 27: v_{M-1} = Theta^T p_{M-1}; v_{m-1} = Theta^T p_{m-1} + W^T v_m; p_adj = tau^T v_0,
    driven step by step through the oracle's stepper, equals oracle.adjoint."""
    pb = synth.random_problem(nx=9, ny=8, nz=7, nt=6, npml=2, L=4, seed=12)
    o = Oracle.from_problem(pb)
    _, y = synth.random_vectors(pb, 1)
    want = o.adjoint(y)
    o.adj_begin()
    M = pb.prm.nt
    o.adj_source(y[M - 1])
    for m in range(M - 1, 0, -1):
        o.adj_step()
        o.adj_source(y[m - 1])
    assert np.array_equal(o.adj_image(), want)


# ----------------------------------------------------------------------------- projected gradient (oracle/pgd.py)

def test_pgd_oracle_against_dense_matrix():
    """oracle/pgd.py against plain linear algebra on the dense H of a tiny grid
    (independent Kronecker assembly, oracle/bruteforce.py): the power iteration converges to the largest eigenvalue
    of H^T H (numpy SVD), every projected-gradient iterate equals max(0, p - s H^T (H p - d)) computed with the dense
    matrix, the reported norms are those of the dense residual / update, and with s = 1/||H||^2 the residual never
    grows (the step is non-expansive)."""
    from oracle import pgd as opgd
    pb = synth.random_problem(nx=7, ny=6, nz=5, nt=6, npml=2, L=4, seed=17)
    H = bf.system_matrix(pb)                                  # (nt L) x N
    o = Oracle.from_problem(pb)
    rng = np.random.default_rng(17)
    shape = pb.p0.shape
    s2_true = np.linalg.svd(H, compute_uv=False)[0] ** 2
    s2, v = opgd.power_iteration(o, rng.standard_normal(shape), iters=200)
    assert abs(s2 - s2_true) <= 1e-6 * s2_true                # converged (gap-dependent, hence 200 iterations)
    assert abs(np.linalg.norm(v) - 1.0) <= 1e-12
    s2_8, _ = opgd.power_iteration(o, rng.standard_normal(shape), iters=8)
    assert 0.5 * s2_true <= s2_8 <= s2_true * (1 + 1e-12)     # a Rayleigh-type estimate never exceeds the true value
    p_true = np.maximum(rng.standard_normal(shape), 0.0)
    d = (H @ p_true.ravel()).reshape(pb.prm.nt, pb.L) + 0.01 * rng.standard_normal((pb.prm.nt, pb.L))
    step = 1.0 / s2_true
    its, res, upd = opgd.pgd(o, np.zeros(shape), d, step, 5)
    p = np.zeros(H.shape[1])
    for k in range(5):
        r = H @ p - d.ravel()
        q = np.maximum(p - step * (H.T @ r), 0.0)
        assert abs(res[k] - np.linalg.norm(r)) <= 1e-12 * np.linalg.norm(r)
        assert abs(upd[k] - np.linalg.norm(q - p)) <= 1e-10 * max(np.linalg.norm(q - p), 1e-30)
        assert np.abs(its[k].ravel() - q).max() <= 1e-12 * max(np.abs(q).max(), 1e-30)
        p = q
    assert all(res[k + 1] <= res[k] * (1 + 1e-12) for k in range(4))
    # without the projection the same code is plain gradient descent (Landweber)
    its_u, _, _ = opgd.pgd(o, np.zeros(shape), d, step, 1, nonneg=False)
    assert np.abs(its_u[0].ravel() - (-step) * (H.T @ (-d.ravel()))).max() <= 1e-12 * np.abs(its_u[0]).max()
