"""Dense/sparse-matrix brute force for tiny grids — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Assembles the propagator W' of Eq. 49 block by block from the operator
definitions of Eq. 7, 43, 45, 47, the initial-value
map tau' (Eq. 54 with the 1/3 of Eq. 21, reading G1) and the sampling rows s'_l (Eq. 56), and
multiplies them out:  H = [Theta' ; Theta' W' ; ... ; Theta' W'^(M-1)] tau'   (Eq. 50-58).

It is written independently of pact_oracle.c (different language, Kronecker-product assembly
instead of loops) so that agreement of the two pins every index, sign and coefficient placement.
Only usable for N of a few hundred.
"""
from __future__ import annotations

import math

import numpy as np
import scipy.sparse as sp

C1, C2 = 9.0 / 8.0, -1.0 / 24.0      # Eq. 8


def d_plus(n, h):
    """integer -> half positions: (D+ f)[i] = (C1 (f[i+1]-f[i]) + C2 (f[i+2]-f[i-1]))/h, zero padded."""
    D = sp.diags([-C2, -C1, C1, C2], [-1, 0, 1, 2], shape=(n, n), format="csr")
    return D / h


def d_minus(n, h):
    """half -> integer positions: (D- g)[i] = (C1 (g[i]-g[i-1]) + C2 (g[i+1]-g[i-2]))/h."""
    D = sp.diags([-C2, -C1, C1, C2], [-2, -1, 0, 1], shape=(n, n), format="csr")
    return D / h


def kron3(Az, Ay, Ax):
    return sp.kron(Az, sp.kron(Ay, Ax, format="csr"), format="csr")


def pml_profile(prm, n):
    """Eq. 38 (kappa=1) on the reading-G8 profile; returns (a_int, b_int, a_half, b_half)."""
    P = prm.npml
    out = []
    for half in (0.0, 0.5):
        a = np.zeros(n)
        b = np.ones(n)
        for i in range(n):
            if P == 0:
                continue
            s = i + half
            depth = max(P - s, s - (n - 1 - P), 0.0)
            if depth > 0:
                xi = depth / P
                d = -3.0 * prm.pml_cref * math.log(prm.pml_R) / (2.0 * P * prm.h) * xi * xi
                beta = prm.pml_beta_max * (1.0 - xi)
                b[i] = math.exp(-(d + beta) * prm.dt)
                a[i] = d / (d + beta) * (b[i] - 1.0) if d > 0 else 0.0
        out += [a, b]
    return out[0], out[1], out[2], out[3]


def _shift_clamped(v, axis):
    """v sampled at index+1 along `axis`, last index repeated (clamp)."""
    last = np.take(v, [-1], axis=axis)
    return np.concatenate([np.delete(v, 0, axis=axis), last], axis=axis)


AX = {0: 2, 1: 1, 2: 0}    # paper direction (0=x,1=y,2=z) -> numpy axis of a [z][y][x] volume


def staggered(prob):
    """rho_b, alpha_b (2-point arithmetic) and mu_bc (4-point harmonic, 0 if any is 0)."""
    rho = prob.rho.astype(np.float64)
    al = prob.alpha.astype(np.float64)
    mu = prob.mu.astype(np.float64)
    rho_s = [0.5 * (rho + _shift_clamped(rho, AX[b])) for b in range(3)]
    al_s = [0.5 * (al + _shift_clamped(al, AX[b])) for b in range(3)]
    mu_s = {}
    for (b, c) in ((0, 1), (0, 2), (1, 2)):
        m0 = mu
        m1 = _shift_clamped(mu, AX[b])
        m2 = _shift_clamped(mu, AX[c])
        m3 = _shift_clamped(m1, AX[c])
        stack = np.stack([m0, m1, m2, m3])
        anyzero = (stack == 0).any(axis=0)
        with np.errstate(divide="ignore"):
            hm = 4.0 / (1.0 / stack).sum(axis=0)
        mu_s[(b, c)] = np.where(anyzero, 0.0, hm)
    return rho_s, al_s, mu_s


def trilinear_rows(prob):
    prm = prob.prm
    n = (prm.nx, prm.ny, prm.nz)
    N = prm.N
    rows = sp.lil_matrix((prob.L, N))
    for l in range(prob.L):
        i0, t = [], []
        for b in range(3):
            f = min(max(prob.rcv[l, b] / prm.h, 0.0), n[b] - 1.0)
            i = min(int(math.floor(f)), n[b] - 2)
            i0.append(i)
            t.append(f - i)
        for cz in (0, 1):
            for cy in (0, 1):
                for cx in (0, 1):
                    w = ((t[0] if cx else 1 - t[0]) * (t[1] if cy else 1 - t[1])
                         * (t[2] if cz else 1 - t[2]))
                    j = (i0[0] + cx) + prm.nx * ((i0[1] + cy) + prm.ny * (i0[2] + cz))
                    rows[l, j] += w
    return rows.tocsr()


def assemble(prob):
    """Return (Wp, taup, Thetap): 27N x 27N, 27N x N, L x 27N sparse matrices."""
    prm = prob.prm
    nx, ny, nz, h, dt = prm.nx, prm.ny, prm.nz, prm.h, prm.dt
    N = prm.N
    n = (nx, ny, nz)
    I1 = [sp.identity(k, format="csr") for k in n]

    def D3(b, plus):
        D1 = d_plus(n[b], h) if plus else d_minus(n[b], h)
        mats = [I1[2], I1[1], I1[0]]          # (z, y, x)
        mats[2 - b] = D1
        return kron3(*mats)

    def diag1(b, table):
        """1-D table along axis b broadcast to the volume, as a diagonal matrix."""
        shape = [1, 1, 1]
        shape[AX[b]] = n[b]
        vol = np.broadcast_to(np.asarray(table).reshape(shape), (nz, ny, nx))
        return sp.diags(vol.reshape(-1))

    def dg(vol):
        return sp.diags(np.asarray(vol, dtype=np.float64).reshape(-1))

    tabs = [pml_profile(prm, n[b]) for b in range(3)]     # per axis: a_int, b_int, a_half, b_half
    rho_s, al_s, mu_s = staggered(prob)
    lam = prob.lam.astype(np.float64)
    mu = prob.mu.astype(np.float64)
    Z = sp.csr_matrix((N, N))
    I = sp.identity(N, format="csr")

    voigt = [(0, 0), (1, 1), (2, 2), (1, 2), (0, 2), (0, 1)]     # Eq. 9c order 11,22,33,23,13,12

    def sig_col(a, b):
        return voigt.index((min(a, b), max(a, b)))

    # derivative that acts on sigma^{ab} along b inside the u^a equation: D+ if a == b else D-
    # its memory variable phi^{ab} sits at u^a's position: "half" table if a == b else "int"
    def phi_tab(a, b):
        ta = tabs[b]
        return (ta[2], ta[3]) if a == b else (ta[0], ta[1])

    # derivative of u^a along b inside the sigma^{ab} equation: D- if a == b else D+
    # psi^{ab} sits at sigma^{ab}'s position: "int" table if a == b else "half"
    def psi_tab(a, b):
        ta = tabs[b]
        return (ta[0], ta[1]) if a == b else (ta[2], ta[3])

    pairs = [(a, b) for a in range(3) for b in range(3)]        # Eq. 44 order 11,12,13,21,...

    # B, B~ (Eq. 45a,b), E (45c), E~ (45d)
    B = sp.block_diag([diag1(b, phi_tab(a, b)[1]) for (a, b) in pairs], format="csr")
    Bt = sp.block_diag([diag1(b, psi_tab(a, b)[1]) for (a, b) in pairs], format="csr")
    E_rows, Et_rows = [], []
    for (a, b) in pairs:
        row = [Z] * 6
        row[sig_col(a, b)] = diag1(b, phi_tab(a, b)[0]) @ D3(b, plus=(a == b))
        E_rows.append(row)
        rowt = [Z] * 3
        rowt[a] = diag1(b, psi_tab(a, b)[0]) @ D3(b, plus=(a != b))
        Et_rows.append(rowt)
    E = sp.bmat(E_rows, format="csr")
    Et = sp.bmat(Et_rows, format="csr")

    # J (7a), Phi (7b), Gamma (45e)
    J = sp.block_diag([dg(1.0 - dt * al_s[a]) for a in range(3)], format="csr")
    Phi_rows, Gam_rows = [], []
    for a in range(3):
        Qinv = dg(dt / rho_s[a])
        row = [Z] * 6
        for b in range(3):
            k = sig_col(a, b)
            row[k] = row[k] + Qinv @ D3(b, plus=(a == b))
        Phi_rows.append(row)
        g = [Z] * 9
        for b in range(3):
            g[pairs.index((a, b))] = Qinv
        Gam_rows.append(g)
    Phi = sp.bmat(Phi_rows, format="csr")
    Gam = sp.bmat(Gam_rows, format="csr")

    # Psi (7c), Delta (45f), rows in Voigt order
    Psi_rows, Del_rows = [], []
    for (i, j) in voigt:
        prow = [Z] * 3
        drow = [Z] * 9
        if i == j:
            for k in range(3):
                prow[k] = prow[k] + dg(dt * lam) @ D3(k, plus=False)
                drow[pairs.index((k, k))] = drow[pairs.index((k, k))] + dg(dt * lam)
            prow[i] = prow[i] + dg(dt * 2.0 * mu) @ D3(i, plus=False)
            drow[pairs.index((i, i))] = drow[pairs.index((i, i))] + dg(dt * 2.0 * mu)
        else:
            M = dg(dt * mu_s[(i, j)])
            prow[j] = prow[j] + M @ D3(i, plus=True)       # d_i u^j
            prow[i] = prow[i] + M @ D3(j, plus=True)       # d_j u^i
            drow[pairs.index((i, j))] = M                  # psi^{ij}: d_j u^i
            drow[pairs.index((j, i))] = M                  # psi^{ji}: d_i u^j
        Psi_rows.append(prow)
        Del_rows.append(drow)
    Psi = sp.bmat(Psi_rows, format="csr")
    Del = sp.bmat(Del_rows, format="csr")

    F = Phi + Gam @ E            # Eq. 47g
    G = Psi + Del @ Et           # Eq. 47h
    I6 = sp.identity(6 * N, format="csr")
    # Eq. 49; state order [phi (9N); u (3N); psi (9N); sigma (6N)]
    Wp = sp.bmat([
        [B, None, None, E],
        [Gam @ B, J, None, F],
        [Et @ Gam @ B, Et @ J, Bt, Et @ F],
        [G @ Gam @ B, G @ J, Del @ Bt, I6 + G @ F],
    ], format="csr")

    # tau' (Eq. 54 with Eq. 21's 1/3, reading G1): sigma11 = sigma22 = sigma33 = -p0/3
    third = -I / 3.0
    taup = sp.vstack([sp.csr_matrix((21 * N, N)), third, third, third, sp.csr_matrix((3 * N, N))],
                     format="csr")
    # Theta' (Eq. 56): s'_l = [0_{21N}, -R_l, -R_l, -R_l, 0_{3N}]
    R = trilinear_rows(prob)
    Thetap = sp.hstack([sp.csr_matrix((prob.L, 21 * N)), -R, -R, -R, sp.csr_matrix((prob.L, 3 * N))],
                       format="csr")
    return Wp, taup, Thetap


def system_matrix(prob):
    """Dense H (nt*L x N), time-major rows (Eq. 12)."""
    Wp, taup, Thetap = assemble(prob)
    V = taup.toarray()                       # 27N x N
    blocks = []
    for m in range(prob.prm.nt):
        blocks.append(Thetap @ V)
        if m < prob.prm.nt - 1:
            V = Wp @ V
    return np.vstack(blocks)
