"""Seeded synthetic workloads shaped like the paper's ILE jobs.

The paper's data (GWOSC strain, PSDs, waveform models) are not
available, so every input is synthetic: a 2- or 3-detector network sampled at 4096 Hz
(PAPER.md:371, 555-559), l_max = 2 or 4 mode sets (Table II), loud and
weak sources, many intrinsic points per job.

Nothing here evaluates the likelihood or an integrator.  The injected-signal coefficients
(F_k(theta_0), Y_lm(theta_0), tau_k(theta_0)) come from ``injections.json``, written by
``oracle/make_injections.py``.
"""
from __future__ import annotations

import json
import os
from dataclasses import dataclass, field

import numpy as np

C_LIGHT = 299792458.0          # m/s
FS = 4096.0                    # Hz, "4096 Hz"
R_EARTH = 6.371e6              # m, BASELINE.json configs[0]
SEED_BASE = 20250511 * 10**4
SIGMA_T = 2.0e-3               # s, template envelope width
F0 = 60.0                      # Hz, template phase rate per unit m
D0_MPC = 500.0                 # injected distance

_HERE = os.path.dirname(os.path.abspath(__file__))

# Per-config shape table; N and n_iter are the full BASELINE.json sizes.
CONFIGS = {
    1: dict(K=2, lmax=2, N_Q=410, N_t=41, stride=2, snr=10.0, kind="UNIFORM", d=6,
            N=1 << 16, n_iter=1, P=1, table=False, two_templates=False),
    2: dict(K=3, lmax=4, N_Q=820, N_t=400, stride=1, snr=20.0, kind="AC", d=6,
            N=1 << 20, n_iter=10, P=1, table=False, two_templates=False),
    3: dict(K=3, lmax=4, N_Q=820, N_t=400, stride=1, snr=100.0, kind="AV", d=6,
            N=1 << 22, n_iter=20, P=1, table=False, two_templates=False),
    4: dict(K=3, lmax=4, N_Q=820, N_t=200, stride=1, snr=20.0, kind="UNIFORM", d=6,
            N=1 << 18, n_iter=1, P=512, table=False, two_templates=False),
    5: dict(K=3, lmax=4, N_Q=820, N_t=400, stride=1, snr=50.0, kind="PORTFOLIO", d=5,
            N=1 << 21, n_iter=30, P=1, table=True, two_templates=True),
}


def config_seed(cfg: int, p: int = 0) -> int:
    """seed = 20250511e4 + 1000*cfg + p."""
    return SEED_BASE + 1000 * cfg + p


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(seed))


def make_modes(lmax: int):
    """Mode list, l ascending then m ascending: M = 5 (l=2) or 21 (l=2..4)."""
    ell, m = [], []
    for l in range(2, lmax + 1):
        for mm in range(-l, l + 1):
            ell.append(l)
            m.append(mm)
    return np.asarray(ell, dtype=np.int32), np.asarray(m, dtype=np.int32)


def make_network(K: int, rng: np.random.Generator):
    """Random symmetric traceless response tensors with Tr(D^2) = 1/2 and detector
    positions on a 6371 km sphere (BASELINE.json configs[0])."""
    D = np.empty((K, 3, 3))
    pos = np.empty((K, 3))
    for k in range(K):
        A = rng.standard_normal((3, 3))
        S = 0.5 * (A + A.T)
        S -= np.trace(S) / 3.0 * np.eye(3)
        S *= np.sqrt(0.5 / np.trace(S @ S))
        D[k] = S
        v = rng.standard_normal(3)
        pos[k] = R_EARTH * v / np.linalg.norm(v)
    return D, pos


def mode_amplitudes(ell, m, profile: int = 0):
    """a_lm = 0.4^(l-2) * 0.5^|l-|m||; profile 1 favours |m| < l (config 5's second template)."""
    ell = np.asarray(ell, dtype=float)
    am = np.abs(np.asarray(m, dtype=float))
    if profile == 0:
        return 0.4 ** (ell - 2.0) * 0.5 ** np.abs(ell - am)
    return 0.6 ** (ell - 2.0) * 0.5 ** np.abs(ell - 1.0 - am)


def make_uv(K: int, ell, m, rng: np.random.Generator, profile: int = 0):
    """U_k = G^H G (Hermitian positive definite), V_k = G^T G (complex symmetric), from a
    seeded complex Gaussian G (2M x M) with columns scaled by the mode amplitudes; both
    divided by U_k[(2,2),(2,2)] (BASELINE.json configs[0]; PAPER.md:339-341 symmetries).
    Also returns the scaled G_k [K, 2M, M] (its rows play the part of whitened frequency bins
    of the modes), from which make_q colours the noise."""
    M = len(ell)
    amp = mode_amplitudes(ell, m, profile)
    i22 = int(np.nonzero((np.asarray(ell) == 2) & (np.asarray(m) == 2))[0][0])
    U = np.empty((K, M, M), dtype=np.complex128)
    V = np.empty((K, M, M), dtype=np.complex128)
    Gs = np.empty((K, 2 * M, M), dtype=np.complex128)
    for k in range(K):
        G = (rng.standard_normal((2 * M, M)) + 1j * rng.standard_normal((2 * M, M))) / np.sqrt(2.0)
        G = G * amp[None, :]
        Uk = G.conj().T @ G
        Vk = G.T @ G
        Uk = 0.5 * (Uk + Uk.conj().T)      # exact Hermitian / symmetric bit patterns
        Vk = 0.5 * (Vk + Vk.T)
        s = Uk[i22, i22].real
        U[k] = Uk / s
        V[k] = Vk / s
        Gs[k] = G / np.sqrt(s)
    return U, V, Gs


def load_injection(cfg: int):
    """Injected-signal fixture for one config: theta_0 and, per template, F[K], Y[M], tau[K]."""
    with open(os.path.join(_HERE, "injections.json")) as fh:
        data = json.load(fh)
    ent = data[str(cfg)]
    out = []
    for tpl in ent["templates"]:
        out.append(dict(
            theta0=tpl["theta0"],
            F=np.array([complex(float.fromhex(a), float.fromhex(b)) for a, b in tpl["F"]]),
            Y=np.array([complex(float.fromhex(a), float.fromhex(b)) for a, b in tpl["Y"]]),
            tau=np.array([float.fromhex(a) for a in tpl["tau"]]),
        ))
    return out


def matched_q0(U, V, c0):
    """q0_k = (U_k c0_k + conj(V_k) conj(c0_k)) / 2: the noise-free Q of a signal with mode
    coefficients c0_k (the data-synthesis identity behind pin P4)."""
    return 0.5 * (np.einsum("kab,kb->ka", U, c0) + np.einsum("kab,kb->ka", V.conj(), c0.conj()))


def network_rho2(U, V, c0):
    """rho^2 = sum_k (c0^H U c0 + Re c0^T V c0)/2 of the synthesised signal."""
    t1 = np.einsum("ka,kab,kb->", c0.conj(), U, c0).real
    t2 = np.einsum("ka,kab,kb->", c0, V, c0).real
    return 0.5 * (t1 + t2)


def make_q(U, V, G, ell, m, templates, snr, N_Q, t_Q0, rng, noise=True, x0=None):
    """Q_{k,m}[n] = sum_templates q0_{k,m} * A_m(t_n - tau_k(theta_0)) + eta, with
    A_m(s) = exp(-s^2 / 2 sigma_t^2) exp(2 pi i m f0 s).  The noise is eta_k[n] = G_k^H w[n]
    with w a real standard-normal 2M-vector per bin, so that E[eta eta^H] = U_k and
    E[eta eta^T] = conj(V_k): exactly the statistics <h_lm|n> has for real Gaussian detector
    noise (Eq. 6a), with unit variance in the (2,2) mode (BASELINE.json configs[0] "unit complex
    Gaussian noise").  White-across-modes noise would let weak modes fit noise without bound.
    The overall scale x0 = D_ref/D0 is solved so the first template has network SNR `snr`
    (or taken from `x0` when given: every intrinsic point of one event shares D_ref).  A second
    template (config 5) is scaled by 0.7 and re-weighted across m by the ratio of the two
    amplitude profiles.  Returns Q [K, M, N_Q], D_ref, rho2 (of the first template)."""
    K, M = U.shape[0], U.shape[1]
    t = t_Q0 + np.arange(N_Q) / FS
    Q = np.zeros((K, M, N_Q), dtype=np.complex128)
    rho2 = None
    for it, tpl in enumerate(templates):
        c_unit = tpl["F"][:, None] * tpl["Y"][None, :]           # c0 / x0
        if it == 0:
            r2_unit = network_rho2(U, V, c_unit)
            if x0 is None:
                x0 = snr / np.sqrt(r2_unit)
            rho2 = x0 * x0 * r2_unit
        c0 = x0 * c_unit * (1.0 if it == 0 else 0.7)
        q0 = matched_q0(U, V, c0)
        if it > 0:
            q0 = q0 * (mode_amplitudes(ell, m, 1) / mode_amplitudes(ell, m, 0))[None, :]
        for k in range(K):
            s = t - tpl["tau"][k]
            env = np.exp(-0.5 * (s / SIGMA_T) ** 2)
            for im in range(M):
                Q[k, im] += q0[k, im] * env * np.exp(2j * np.pi * float(m[im]) * F0 * s)
    if noise:
        for k in range(K):
            w = rng.standard_normal((G.shape[1], N_Q))
            Q[k] += G[k].conj().T @ w
    D_ref = x0 * D0_MPC
    return Q, float(D_ref), float(rho2)


def make_distance_table(D_ref, D_min, D_max, A_lo, A_hi, B_lo, B_hi, nA=256, nB=256, nodes=4097):
    """lnT[b][a] = ln int_{D_min}^{D_max} p(D) exp(x A - x^2 B) dD, x = D_ref/D,
    p(D) = 3 D^2 / (D_max^3 - D_min^3), by composite Simpson on `nodes` points in D, in
    log-sum-exp form.  The table is *input data* for both the oracle and the
    CUDA path (BASELINE.json configs[4]: "seeded 2-D lookup table (256x256, bilinear)")."""
    Dn = np.linspace(D_min, D_max, nodes)
    h = (D_max - D_min) / (nodes - 1)
    wS = np.ones(nodes)
    wS[1:-1:2] = 4.0
    wS[2:-1:2] = 2.0
    wS *= h / 3.0
    x = D_ref / Dn
    lnp = np.log(3.0 * Dn * Dn / (D_max ** 3 - D_min ** 3)) + np.log(wS)
    A = np.linspace(A_lo, A_hi, nA)
    B = np.linspace(B_lo, B_hi, nB)
    lnT = np.empty((nB, nA))
    for ib in range(nB):
        e = A[:, None] * x[None, :] - B[ib] * (x * x)[None, :] + lnp[None, :]
        mx = e.max(axis=1)
        lnT[ib] = mx + np.log(np.exp(e - mx[:, None]).sum(axis=1))
    return dict(nA=nA, nB=nB, A_lo=float(A_lo), A_hi=float(A_hi), B_lo=float(B_lo),
                B_hi=float(B_hi), lnT=lnT)


@dataclass
class Problem:
    cfg: int
    K: int
    M: int
    P: int
    N_Q: int
    fs: float
    t_Q0: float
    D: np.ndarray
    pos: np.ndarray
    gmst: float
    ell: np.ndarray
    m: np.ndarray
    Q: np.ndarray            # [P, K, M, N_Q] complex128
    U: np.ndarray            # [P, K, M, M] complex128
    V: np.ndarray            # [P, K, M, M] complex128
    D_ref: float
    rho2: float
    t_lo: float
    dt: float
    N_t: int
    interp: int
    D_min: float
    D_max: float
    d: int
    lo: np.ndarray           # integrator box, z = (RA, sin Dec, psi, phi_ref, cos incl[, D])
    hi: np.ndarray
    kind: str
    N: int
    n_iter: int
    opts: dict = field(default_factory=dict)
    table: dict | None = None
    inj: list | None = None


def make_problem(cfg: int, P: int | None = None, N: int | None = None, n_iter: int | None = None,
                 noise: bool = True, d: int | None = None, with_table: bool | None = None) -> Problem:
    """Build config `cfg` (1..5) of BASELINE.json.  P / N / n_iter override the full sizes for
    tests; `noise=False` gives the zero-noise variant used by pin P4."""
    c = CONFIGS[cfg]
    K, lmax, N_Q, N_t, stride = c["K"], c["lmax"], c["N_Q"], c["N_t"], c["stride"]
    P = c["P"] if P is None else P
    N = c["N"] if N is None else N
    n_iter = c["n_iter"] if n_iter is None else n_iter
    d = c["d"] if d is None else d
    with_table = c["table"] if with_table is None else with_table

    rng0 = _rng(config_seed(cfg, 0))
    D, pos = make_network(K, rng0)
    ell, m = make_modes(lmax)
    M = len(ell)
    t_Q0 = -(N_Q // 2) / FS
    inj = load_injection(cfg)

    Q = np.empty((P, K, M, N_Q), dtype=np.complex128)
    U = np.empty((P, K, M, M), dtype=np.complex128)
    V = np.empty((P, K, M, M), dtype=np.complex128)
    D_ref = None
    rho2 = None
    for p in range(P):
        rng = rng0 if p == 0 else _rng(config_seed(cfg, p))
        U[p], V[p], G = make_uv(K, ell, m, rng, profile=0)
        # one event: every intrinsic point shares D_ref (x0 solved on point 0 only)
        x0 = None if p == 0 else D_ref / D0_MPC
        Qp, D_ref_p, rho2_p = make_q(U[p], V[p], G, ell, m, inj, c["snr"], N_Q, t_Q0, rng,
                                     noise=noise, x0=x0)
        if p == 0:
            D_ref, rho2 = D_ref_p, rho2_p
        Q[p] = Qp

    half = (N_t - 1) // 2 if stride == 2 else N_t // 2
    t_lo = -half * stride / FS
    dt = stride / FS
    D_min, D_max = 100.0, 2000.0
    lo = np.array([0.0, -1.0, 0.0, 0.0, -1.0, D_min])[:d].copy()
    hi = np.array([2.0 * np.pi, 1.0, np.pi, 2.0 * np.pi, 1.0, D_max])[:d].copy()

    opts = dict(seed=config_seed(cfg, 0) & 0xFFFFFFFFFFFFFFFF)
    if c["kind"] == "AC":
        opts.update(n_bins=100, eps=0.1, beta=1.0)
    elif c["kind"] == "AV":
        opts.update(P_thr=0.999, N_min_star=4096)
    elif c["kind"] == "PORTFOLIO":
        opts.update(members=["AC", "AV", "GMM"], n_bins=100, eps=0.1, beta=1.0, P_thr=0.999,
                    N_min_star=4096, n_gmm=8)

    table = None
    if with_table:
        x0 = D_ref / D0_MPC
        A_pk = rho2 / x0
        B_pk = rho2 / (2.0 * x0 * x0)
        table = make_distance_table(D_ref, D_min, D_max, 0.0, 1.3 * A_pk, 0.02 * B_pk, 3.0 * B_pk)

    return Problem(cfg=cfg, K=K, M=M, P=P, N_Q=N_Q, fs=FS, t_Q0=t_Q0, D=D, pos=pos, gmst=0.0,
                   ell=ell, m=m, Q=Q, U=U, V=V, D_ref=D_ref, rho2=rho2, t_lo=t_lo, dt=dt, N_t=N_t,
                   interp=1, D_min=D_min, D_max=D_max, d=d, lo=lo, hi=hi, kind=c["kind"], N=N,
                   n_iter=n_iter, opts=opts, table=table, inj=inj)


def make_custom_problem(K: int, lmax: int, snr: float, seed: int, N_Q: int = 820, N_t: int = 300, modes=None) -> Problem:
    """A one-point problem with a detector / mode count outside the five configs (parity of the kernels' other
    shapes).  The template's mode coefficients are seeded random numbers with the usual amplitude law, not a
    physical signal (no injection fixture is needed): Q = q0 A_m(t - tau_k) + coloured noise as in make_q."""
    rng = _rng(SEED_BASE + 900000 + seed)
    D, pos = make_network(K, rng)
    ell, m = make_modes(lmax)
    if modes is not None:                                   # an explicit (l, m) list instead of all modes up to lmax
        ell = np.array([lm[0] for lm in modes], dtype=ell.dtype)
        m = np.array([lm[1] for lm in modes], dtype=m.dtype)
    M = len(ell)
    t_Q0 = -(N_Q // 2) / FS
    U, V, G = make_uv(K, ell, m, rng, profile=0)
    tpl = dict(F=(rng.standard_normal(K) + 1j * rng.standard_normal(K)) * 0.5,
               Y=(rng.standard_normal(M) + 1j * rng.standard_normal(M)) * 0.3,
               tau=rng.uniform(-0.5, 0.5, K) * R_EARTH / C_LIGHT)
    Q, D_ref, rho2 = make_q(U, V, G, ell, m, [tpl], snr, N_Q, t_Q0, rng)
    t_lo = -(N_t // 2) / FS
    D_min, D_max = 100.0, 2000.0
    lo = np.array([0.0, -1.0, 0.0, 0.0, -1.0, D_min])
    hi = np.array([2.0 * np.pi, 1.0, np.pi, 2.0 * np.pi, 1.0, D_max])
    return Problem(cfg=0, K=K, M=M, P=1, N_Q=N_Q, fs=FS, t_Q0=t_Q0, D=D, pos=pos, gmst=0.0, ell=ell, m=m,
                   Q=Q[None], U=U[None], V=V[None], D_ref=D_ref, rho2=rho2, t_lo=t_lo, dt=1.0 / FS, N_t=N_t, interp=1,
                   D_min=D_min, D_max=D_max, d=6, lo=lo, hi=hi, kind="UNIFORM", N=1 << 12, n_iter=1,
                   opts=dict(seed=seed), table=None, inj=None)


def uniform_box_samples(lo, hi, N, seed):
    """N points uniform in the box [lo, hi) (numpy Philox; for parity inputs, not the
    integrators' own counter-based draws)."""
    rng = _rng(seed)
    d = len(lo)
    z = np.empty((d, N))
    for c in range(d):
        z[c] = lo[c] + rng.random(N) * (hi[c] - lo[c])
    return z
