"""Brute-force NumPy restatement of ONE IMEX-SSP2(2,2,2) step on a small fully periodic grid.

Written independently of oracle/rgrmhd_oracle.cpp (different language, different data layout:
interior-only arrays with np.roll instead of ghost zones; matrix inverses from numpy.linalg
instead of adjugates; tensor algebra through einsum; the stage solves through scipy.optimize.root
on the full 4-unknown nonlinear system with the 3x3 Ohm system solved by numpy.linalg.solve; the
stiff source R and the conduction current evaluated LITERALLY from Ohm's law, Eq. 29/41, instead of
the oracle's difference quotient).  It is test infrastructure for the 'whole step' pin of
SURVEY.md Sec. 8(c) and shares no code with either implementation.

Arrays: fields have shape (nz, ny, nx); tensors carry leading index axes, e.g. g[i, j, z, y, x].
"""
import numpy as np
from scipy import optimize

LEVI = np.zeros((3, 3, 3))
LEVI[0, 1, 2] = LEVI[1, 2, 0] = LEVI[2, 0, 1] = 1.0
LEVI[0, 2, 1] = LEVI[2, 1, 0] = LEVI[1, 0, 2] = -1.0
AX = {0: 2, 1: 1, 2: 0}     # direction k -> numpy axis of a (z,y,x) array
SYM = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]


def sh(a, k, o):
    """a shifted so that result[i] = a[i + o] along direction k (periodic)."""
    return np.roll(a, -o, axis=a.ndim - 3 + AX[k])


def full_metric(metric16):
    alpha = metric16[0]
    beta = metric16[1:4]
    g = np.empty((3, 3) + alpha.shape); K = np.empty_like(g)
    for q, (i, j) in enumerate(SYM):
        g[i, j] = g[j, i] = metric16[4 + q]
        K[i, j] = K[j, i] = metric16[10 + q]
    return alpha, beta, g, K


def geom(g):
    gm = np.moveaxis(g, (0, 1), (-2, -1))
    ginv = np.moveaxis(np.linalg.inv(gm), (-2, -1), (0, 1))
    sg = np.sqrt(np.linalg.det(gm))
    return ginv, sg


def prim2cons(P, g, sg, Gam):
    rho, p = P[0], P[1]; v, E, B = P[2:5], P[5:8], P[8:11]
    vD = np.einsum("ij...,j...->i...", g, v)
    v2 = np.einsum("i...,i...->...", v, vD)
    W = 1 / np.sqrt(1 - v2)
    h = rho + Gam / (Gam - 1) * p
    E2 = np.einsum("ij...,i...,j...->...", g, E, E); B2 = np.einsum("ij...,i...,j...->...", g, B, B)
    ExB = sg * np.einsum("ijk,j...,k...->i...", LEVI, E, B)
    U = np.empty_like(P)
    U[0] = sg * rho * W
    U[1:4] = sg * (h * W * W * vD + ExB)
    U[4] = sg * (h * W * W - p + 0.5 * (E2 + B2)) - U[0]
    U[5:8] = sg * E; U[8:11] = sg * B; U[11:14] = sg * P[11:14]
    return U


def flux(P, Jc, k, alpha, beta, g, ginv, sg, Gam):
    """U and F^k for the state P with conduction current density Jc (densitised, 3 components)."""
    U = prim2cons(P, g, sg, Gam)
    rho, p = P[0], P[1]; v, E, B = P[2:5], P[5:8], P[8:11]
    vD = np.einsum("ij...,j...->i...", g, v); ED = np.einsum("ij...,j...->i...", g, E); BD = np.einsum("ij...,j...->i...", g, B)
    W2 = 1 / (1 - np.einsum("i...,i...->...", v, vD))
    h = rho + Gam / (Gam - 1) * p
    E2 = np.einsum("i...,i...->...", E, ED); B2 = np.einsum("i...,i...->...", B, BD)
    F = np.empty_like(P)
    F[0] = (alpha * v[k] - beta[k]) * U[0]
    for j in range(3):
        T = h * W2 * v[k] * vD[j] - E[k] * ED[j] - B[k] * BD[j] + (p + 0.5 * (E2 + B2) if j == k else 0.0)
        F[1 + j] = alpha * sg * T - beta[k] * U[1 + j]
    SU = np.einsum("ij...,j...->i...", ginv, U[1:4])
    F[4] = alpha * (SU[k] - v[k] * U[0]) - beta[k] * U[4]
    for i in range(3):
        F[8 + i] = alpha * (np.einsum("j,j...->...", LEVI[i, k], ED) + ginv[i, k] * U[12]) - beta[k] * U[8 + i]
        F[5 + i] = -alpha * (np.einsum("j,j...->...", LEVI[i, k], BD) - ginv[i, k] * U[11]) - beta[k] * U[5 + i]
    F[12] = alpha * U[8 + k] - beta[k] * U[12]
    F[11] = alpha * U[5 + k] - beta[k] * U[11]
    F[13] = alpha * (U[13] * v[k] + Jc[k]) - beta[k] * U[13]
    return U, F


def recon(u, k, scheme, eps_w=1e-26):
    """(value at the cell's lower face, value at its upper face) from the 5-cell stencil."""
    m2, m1, c, p1, p2 = sh(u, k, -2), sh(u, k, -1), u, sh(u, k, 1), sh(u, k, 2)
    if scheme == 2:
        def plus(a0, a1, a2, a3, a4):
            q = [(2 * a0 - 7 * a1 + 11 * a2) / 6, (-a1 + 5 * a2 + 2 * a3) / 6, (2 * a2 + 5 * a3 - a4) / 6]
            b = [13 / 12 * (a0 - 2 * a1 + a2) ** 2 + 0.25 * (a0 - 4 * a1 + 3 * a2) ** 2,
                 13 / 12 * (a1 - 2 * a2 + a3) ** 2 + 0.25 * (a1 - a3) ** 2,
                 13 / 12 * (a2 - 2 * a3 + a4) ** 2 + 0.25 * (3 * a2 - 4 * a3 + a4) ** 2]
            w = [d / (eps_w + bb) ** 2 for d, bb in zip((0.1, 0.6, 0.3), b)]
            return (w[0] * q[0] + w[1] * q[1] + w[2] * q[2]) / (w[0] + w[1] + w[2])
        return plus(p2, p1, c, m1, m2), plus(m2, m1, c, p1, p2)
    a, b = c - m1, p1 - c
    if scheme == 0:
        s = np.where(a * b <= 0, 0.0, np.sign(a) * np.minimum(np.abs(a), np.abs(b)))
    else:
        cand = np.stack([2 * a, 2 * b, 0.5 * (a + b)])
        s = np.where(np.all(cand > 0, 0), cand.min(0), np.where(np.all(cand < 0, 0), cand.max(0), 0.0))
    return c - 0.5 * s, c + 0.5 * s


def ohm_current(P, alpha, g, sg, sigma):
    """Densitised conduction current Jc^i = W sigma [calE^i + sqrt(g)(v x B)^i - (v.E) sqrt(g) v^i] (Eq. 29)."""
    v, E, B = P[2:5], P[5:8], P[8:11]
    vD = np.einsum("ij...,j...->i...", g, v); BD = np.einsum("ij...,j...->i...", g, B)
    W = 1 / np.sqrt(1 - np.einsum("i...,i...->...", v, vD))
    vxB = np.einsum("ijk,j...,k...->i...", LEVI, vD, BD) / sg
    vE = np.einsum("i...,i...->...", vD, E)
    return W * sigma * sg * (E + vxB - vE * v)


def rhs(P, Jc, metric16, dx, Gam, kappa, scheme, active=(True, True, True)):
    alpha, beta, g, K = full_metric(metric16)
    ginv, sg = geom(g)
    out = np.zeros_like(P)
    for k in range(3):
        if not active[k]:
            continue
        # face between cell i-1 and i, stored at i
        am = 0.5 * (alpha + sh(alpha, k, -1)); bm = 0.5 * (beta + sh(beta, k, -1)); gmf = 0.5 * (g + sh(g, k, -1))
        ginvf, sgf = geom(gmf)
        PL = np.empty_like(P); PR = np.empty_like(P)
        for vv in range(14):
            lo, hi = recon(P[vv], k, scheme)
            PL[vv] = sh(hi, k, -1); PR[vv] = lo
        lo, hi = recon(Jc[k] / sg, k, scheme)
        JL = np.zeros((3,) + alpha.shape); JR = np.zeros_like(JL)
        JL[k] = sgf * sh(hi, k, -1); JR[k] = sgf * lo
        UL, FL = flux(PL, JL, k, am, bm, gmf, ginvf, sgf, Gam)
        UR, FR = flux(PR, JR, k, am, bm, gmf, ginvf, sgf, Gam)
        c = am * np.sqrt(ginvf[k, k])
        lp = np.maximum(0.0, c - bm[k]); lm = np.minimum(0.0, -c - bm[k])
        Fh = (lp * FL - lm * FR + lp * lm * (UR - UL)) / (lp - lm)
        out -= (sh(Fh, k, 1) - Fh) / dx[k]
    # sources
    d = lambda f, k: (-sh(f, k, 2) + 8 * sh(f, k, 1) - 8 * sh(f, k, -1) + sh(f, k, -2)) / (12 * dx[k]) if active[k] else np.zeros_like(f)
    dal = np.stack([d(alpha, k) for k in range(3)])                 # [k]
    dbe = np.stack([d(beta, k) for k in range(3)])                  # [k, i]
    dg = np.stack([d(g, k) for k in range(3)])                      # [k, i, j]
    U = prim2cons(P, g, sg, Gam)
    rho, p = P[0], P[1]; v, E, B = P[2:5], P[5:8], P[8:11]
    vD = np.einsum("ij...,j...->i...", g, v)
    W2 = 1 / (1 - np.einsum("i...,i...->...", v, vD))
    h = rho + Gam / (Gam - 1) * p
    E2 = np.einsum("ij...,i...,j...->...", g, E, E); B2 = np.einsum("ij...,i...,j...->...", g, B, B)
    T = h * W2 * np.einsum("i...,j...->ij...", v, v) + ginv * (p + 0.5 * (E2 + B2)) - np.einsum("i...,j...->ij...", E, E) - np.einsum("i...,j...->ij...", B, B)
    S = np.zeros_like(P)
    S[1:4] = 0.5 * alpha * sg * np.einsum("jk...,ijk...->i...", T, dg) + np.einsum("j...,ij...->i...", U[1:4], dbe) - (U[4] + U[0]) * dal
    SU = np.einsum("ij...,j...->i...", ginv, U[1:4])
    S[4] = alpha * sg * np.einsum("ij...,ij...->...", T, K) - np.einsum("j...,j...->...", SU, dal)
    christ = np.einsum("il...,jk...,jlk...->i...", ginv, ginv, dg) - 0.5 * np.einsum("il...,jk...,ljk...->i...", ginv, ginv, dg)
    Gi = np.einsum("ij...,j...->i...", ginv, dal) - alpha * christ
    trK = np.einsum("ij...,ij...->...", ginv, K)
    S[8:11] = -np.einsum("k...,ki...->i...", U[8:11], dbe) + U[12] * Gi
    S[5:8] = -np.einsum("k...,ki...->i...", U[5:8], dbe) + U[11] * Gi - alpha * U[13] * v
    S[12] = -alpha * U[12] * trK + np.einsum("k...,k...->...", U[8:11], dal) - alpha * kappa * U[12]
    S[11] = -alpha * U[11] * trK + np.einsum("k...,k...->...", U[5:8], dal) + alpha * U[13] - alpha * kappa * U[11]
    return out + S


def solve_stage(Ustar, Pguess, metric16, adt, sigma, Gam):
    """Cell by cell: root of the full system in (v^i, p) with E from the 3x3 linear Ohm system."""
    alpha, beta, g, K = full_metric(metric16)
    ginv, sg = geom(g)
    P = np.empty_like(Pguess)
    shape = alpha.shape
    for idx in np.ndindex(shape):
        gg = g[(slice(None), slice(None)) + idx]; s_g = sg[idx]; al = alpha[idx]
        U = Ustar[(slice(None),) + idx] / s_g
        D, SD, tau, Es, B = U[0], U[1:4], U[4], U[5:8], U[8:11]
        BD = gg @ B; B2 = B @ BD
        sig = sigma[idx] if np.ndim(sigma) else sigma

        def fields(x):
            v, p = x[:3], x[3]
            vD = gg @ v; W = 1 / np.sqrt(1 - v @ vD); s = adt * al * sig * W
            vxB = np.einsum("ijk,j,k->i", LEVI, vD, BD) / s_g
            M = (1 + s) * np.eye(3) - s * np.outer(v, vD)
            E = np.linalg.solve(M, Es - s * vxB)
            return v, p, vD, W, E

        def F(x):
            v, p, vD, W, E = fields(x)
            E2 = E @ gg @ E
            Z = tau + D + p - 0.5 * (E2 + B2)
            ExB = s_g * np.einsum("ijk,j,k->i", LEVI, E, B)
            r = np.empty(4)
            r[:3] = (Z * vD - (SD - ExB)) / Z
            r[3] = (p - (Gam - 1) / Gam * (Z / W ** 2 - D / W)) / p
            return r

        x0 = np.concatenate([Pguess[(slice(2, 5),) + idx], [Pguess[(1,) + idx]]])
        sol = optimize.root(F, x0, method="hybr", tol=1e-15, options=dict(xtol=1e-15, maxfev=2000))
        x = sol.x
        for _ in range(3):          # polish with Newton on a finite-difference Jacobian
            J = np.empty((4, 4)); f0 = F(x)
            for c in range(4):
                hstep = 1e-7 * max(abs(x[c]), 1e-3); xp = x.copy(); xp[c] += hstep; xm = x.copy(); xm[c] -= hstep
                J[:, c] = (F(xp) - F(xm)) / (2 * hstep)
            x = x - np.linalg.solve(J, f0)
        v, p, vD, W, E = fields(x)
        P[(slice(None),) + idx] = np.concatenate([[D / W, p], v, E, B, U[11:14]])
    return P


def imex_step(P0, metric16, dx, dt, Gam, sigma, kappa, scheme, active=(True, True, True)):
    """Eq. 35-37 evaluated literally, with R = -alpha * Jc from Ohm's law (Eq. 41)."""
    alpha, beta, g, K = full_metric(metric16)
    ginv, sg = geom(g)
    gam = 1 - 1 / np.sqrt(2)
    Un = prim2cons(P0, g, sg, Gam)
    # stage 1
    P1 = solve_stage(Un, P0, metric16, gam * dt, sigma, Gam)
    Jc1 = ohm_current(P1, alpha, g, sg, sigma); R1 = -alpha * Jc1
    F1 = rhs(P1, Jc1, metric16, dx, Gam, kappa, scheme, active)
    # stage 2
    Us = Un + dt * F1
    Us[5:8] += dt * (1 - 2 * gam) * R1
    P2 = solve_stage(Us, P1, metric16, gam * dt, sigma, Gam)
    Jc2 = ohm_current(P2, alpha, g, sg, sigma); R2 = -alpha * Jc2
    F2 = rhs(P2, Jc2, metric16, dx, Gam, kappa, scheme, active)
    Unew = Un + 0.5 * dt * (F1 + F2)
    Unew[5:8] += 0.5 * dt * (R1 + R2)
    Pnew = solve_stage(Unew, P2, metric16, 0.0, 0.0, Gam)
    return Pnew, Unew
