"""Oracle: the factored, time-marginalised extrinsic likelihood (TEST INFRASTRUCTURE ONLY).

Follows PAPER.md section II.A (lines 55-98), Eq. (4), (5), (7) and Appendix A Eq. (A2)
(lines 466-471), with the readings G1-G13, G28, G38 of DESIGN.md section 3.  Plain numpy in
float64/complex128, vectorised over samples only: the loops over time bins j, detectors k
and modes m are written out in the paper's order.  No blocking, no fusion.
"""
from __future__ import annotations

import math

import numpy as np

C_LIGHT = 299792458.0  # m/s (G5: the paper writes t_k = t_c - x_k.n with c = 1)


# --------------------------------------------------------------------------- step 1
def antenna(D, pos, gmst, ra, dec, psi):
    """F_{+,k}, F_{x,k}, tau_k for each sample ("response functions F+ and Fx ...
    arrival time t_k = t_c - x_k . n"; reading G5/G6: textbook detector-tensor contraction).

    D [K,3,3] symmetric traceless response tensors, pos [K,3] metres (Earth-fixed),
    ra/dec/psi arrays [N].  Returns Fp [K,N], Fx [K,N], tau [K,N] (seconds)."""
    D = np.asarray(D, dtype=np.float64)
    pos = np.asarray(pos, dtype=np.float64)
    ra = np.asarray(ra, dtype=np.float64)
    dec = np.asarray(dec, dtype=np.float64)
    psi = np.asarray(psi, dtype=np.float64)
    g = gmst - ra
    cg, sg = np.cos(g), np.sin(g)
    cd, sd = np.cos(dec), np.sin(dec)
    cp, sp = np.cos(psi), np.sin(psi)
    nhat = np.stack([cd * cg, -cd * sg, sd])                         # Earth -> source
    X = np.stack([-cp * sg - sp * cg * sd, -cp * cg + sp * sg * sd, sp * cd])
    Y = np.stack([sp * sg - cp * cg * sd, sp * cg + cp * sg * sd, cp * cd])
    K = D.shape[0]
    N = ra.shape[0]
    Fp = np.zeros((K, N))
    Fx = np.zeros((K, N))
    tau = np.zeros((K, N))
    for k in range(K):
        for a in range(3):
            for b in range(3):
                Fp[k] += X[a] * D[k, a, b] * X[b] - Y[a] * D[k, a, b] * Y[b]
                Fx[k] += X[a] * D[k, a, b] * Y[b] + Y[a] * D[k, a, b] * X[b]
        tau[k] = -(pos[k, 0] * nhat[0] + pos[k, 1] * nhat[1] + pos[k, 2] * nhat[2]) / C_LIGHT
    return Fp, Fx, tau


# --------------------------------------------------------------------------- step 2
def swsh(s, l, m, theta, phi):
    """Spin-weighted spherical harmonic sY_lm(theta, phi) by Goldberg's closed form, written as
    a polynomial in cos(theta/2), sin(theta/2) (never via cot).  PAPER.md:67-70 (Eq. 4) uses
    s = -2."""
    theta = np.asarray(theta, dtype=np.float64)
    phi = np.asarray(phi, dtype=np.float64)
    ch = np.cos(0.5 * theta)
    sh = np.sin(0.5 * theta)
    norm = math.sqrt(math.factorial(l + m) * math.factorial(l - m) * (2 * l + 1)
                     / (4.0 * math.pi * math.factorial(l + s) * math.factorial(l - s)))
    acc = np.zeros_like(theta)
    for r in range(0, l - s + 1):
        kk = r + s - m
        if kk < 0 or kk > l + s:
            continue
        pc = 2 * r + s - m              # power of cos(theta/2)
        ps = 2 * l - 2 * r - s + m      # power of sin(theta/2)
        term = math.comb(l - s, r) * math.comb(l + s, kk) * ch ** pc * sh ** ps
        acc = acc + (term if r % 2 == 0 else -term)
    sign = 1.0 if (l + m - s) % 2 == 0 else -1.0
    return sign * norm * acc * np.exp(1j * m * phi)


def ylm(ell, m, incl, phi):
    """-2Y_lm(incl, phi) for the mode list (ell[i], m[i]); returns [M, N] complex."""
    return np.stack([swsh(-2, int(l), int(mm), incl, phi) for l, mm in zip(ell, m)])


# --------------------------------------------------------------------------- steps 3-6
def bilinear_table(table, A, B):
    """Distance-marginalised lnT(A, B): bilinear in the regular (A, B) grid, clamped to its
    edges (G28)."""
    nA, nB = table["nA"], table["nB"]
    T = table["lnT"]
    a = (A - table["A_lo"]) / (table["A_hi"] - table["A_lo"]) * (nA - 1)
    b = (B - table["B_lo"]) / (table["B_hi"] - table["B_lo"]) * (nB - 1)
    a = np.minimum(np.maximum(a, 0.0), float(nA - 1))
    b = np.minimum(np.maximum(b, 0.0), float(nB - 1))
    ia = np.minimum(np.floor(a).astype(np.int64), nA - 2)
    ib = np.minimum(np.floor(b).astype(np.int64), nB - 2)
    fa = a - ia
    fb = b - ib
    t0 = (1.0 - fa) * T[ib, ia] + fa * T[ib, ia + 1]
    t1 = (1.0 - fa) * T[ib + 1, ia] + fa * T[ib + 1, ia + 1]
    return (1.0 - fb) * t0 + fb * t1


def quadratic_term(F, Y, U, V):
    """B = 1/4 sum_k [ |F_k|^2 Y^H U_k Y + Re(F_k^2 Y^T V_k Y) ]  (Eq. 7, G1-G3).
    F [K,N] complex, Y [M,N] complex, U,V [K,M,M]."""
    K, N = F.shape
    M = Y.shape[0]
    B = np.zeros(N)
    for k in range(K):
        yUy = np.zeros(N, dtype=np.complex128)
        yVy = np.zeros(N, dtype=np.complex128)
        for a in range(M):
            for b in range(M):
                yUy += np.conj(Y[a]) * U[k, a, b] * Y[b]
                yVy += Y[a] * V[k, a, b] * Y[b]
        B += (np.abs(F[k]) ** 2) * yUy.real + (F[k] * F[k] * yVy).real
    return 0.25 * B


def lnL_angles(D, pos, gmst, ell, m, Q, U, V, D_ref, fs, t_Q0, t_lo, dt, N_t,
               ra, dec, psi, phi_ref, incl, dist, interp=1, table=None, return_series=False):
    """Time-marginalised lnL for each sample (Eq. 5/7; time marginalisation
    PAPER.md:94, 333, 547 with reading G9: uniform prior over the grid, rectangle rule).

    Q [K,M,N_Q] complex, U,V [K,M,M] complex for one intrinsic point.  `dist` is ignored when
    a distance table is given (G28).  Returns lnL_marg [N] (and lnL(t_j) [N,N_t])."""
    Fp, Fx, tau = antenna(D, pos, gmst, ra, dec, psi)
    F = Fp - 1j * Fx
    Y = ylm(ell, m, incl, -np.asarray(phi_ref))        # Eq. A2 with phi_* = 0 (G7)
    K = F.shape[0]
    M = Y.shape[0]
    N = F.shape[1]
    N_Q = Q.shape[2]
    B = quadratic_term(F, Y, U, V)
    if table is None:
        x = D_ref / np.asarray(dist, dtype=np.float64)
    lnLt = np.empty((N, N_t))
    for j in range(N_t):
        t_j = t_lo + j * dt
        A_j = np.zeros(N)
        for k in range(K):
            u = (t_j + tau[k] - t_Q0) * fs
            if interp:
                n = np.floor(u).astype(np.int64)
                f = u - n
            else:
                n = np.floor(u + 0.5).astype(np.int64)
                f = np.zeros(N)
            if n.min() < 0 or n.max() + 1 > N_Q - 1:
                raise ValueError("time grid + delays leave the stored Q span")
            z = np.zeros(N, dtype=np.complex128)
            for im in range(M):
                Qr = (1.0 - f) * Q[k, im, n].real + f * Q[k, im, n + 1].real
                Qi = (1.0 - f) * Q[k, im, n].imag + f * Q[k, im, n + 1].imag
                z += np.conj(Y[im]) * (Qr + 1j * Qi)
            A_j += (np.conj(F[k]) * z).real
        if table is None:
            lnLt[:, j] = x * A_j - x * x * B
        else:
            lnLt[:, j] = bilinear_table(table, A_j, B)
    mx = lnLt.max(axis=1)
    lnL = mx + np.log(np.exp(lnLt - mx[:, None]).sum(axis=1)) - math.log(N_t)
    if return_series:
        return lnL, lnLt
    return lnL


def z_to_angles(z):
    """Integrator coordinates z = (RA, sin Dec, psi, phi_ref, cos incl[, D]) -> angles (G38)."""
    ra = z[0]
    dec = np.arcsin(z[1])
    psi = z[2]
    phi_ref = z[3]
    incl = np.arccos(z[4])
    dist = z[5] if z.shape[0] > 5 else None
    return ra, dec, psi, phi_ref, incl, dist


def ln_prior_z(z, D_min, D_max):
    """ln p(z) in the flat coordinates (SURVEY 8(c) "Prior", G13): isotropic sky and
    orientation, p(D) = 3 D^2 / (D_max^3 - D_min^3).  d = 5: the distance factor is inside the
    table."""
    lnp = -math.log(2.0 * math.pi) - math.log(2.0) - math.log(math.pi) - math.log(2.0 * math.pi) \
        - math.log(2.0)
    out = np.full(z.shape[1], lnp)
    if z.shape[0] > 5:
        out = out + np.log(3.0 * z[5] * z[5] / (D_max ** 3 - D_min ** 3))
    return out


def lnL_z(D, pos, gmst, ell, m, Q, U, V, D_ref, fs, t_Q0, t_lo, dt, N_t, z, interp=1, table=None):
    """lnL at integrator coordinates z [d,N] (same definition as lnL_angles through z_to_angles)."""
    ra, dec, psi, phi_ref, incl, dist = z_to_angles(np.asarray(z))
    return lnL_angles(D, pos, gmst, ell, m, Q, U, V, D_ref, fs, t_Q0, t_lo, dt, N_t,
                      ra, dec, psi, phi_ref, incl, dist, interp=interp, table=table)
