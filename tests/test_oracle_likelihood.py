"""Pins P1-P6, P8 for oracle/likelihood.py (closed forms, invariants, special cases)."""
import math

import numpy as np
import pytest

from oracle import likelihood as lk
from synth import make_modes, make_network, make_problem
from synth.workloads import matched_q0, network_rho2


def _rng(seed):
    return np.random.Generator(np.random.Philox(seed))


# ------------------------------------------------------------------------------- P1: Y_lm
def test_ylm_l2_closed_forms():
    # -2Y_{2,+-2} = sqrt(5/64pi)(1 +- cos t)^2 e^{+-2i phi}; -2Y_{2,+-1} = sqrt(5/16pi) sin t (1 +- cos t) e^{+-i phi};
    # -2Y_{20} = sqrt(15/32pi) sin^2 t  (textbook; SURVEY pin P1)
    rng = _rng(1)
    th = rng.uniform(0, math.pi, 50)
    ph = rng.uniform(0, 2 * math.pi, 50)
    c, s = np.cos(th), np.sin(th)
    ref = {
        2: math.sqrt(5 / (64 * math.pi)) * (1 + c) ** 2 * np.exp(2j * ph),
        -2: math.sqrt(5 / (64 * math.pi)) * (1 - c) ** 2 * np.exp(-2j * ph),
        1: math.sqrt(5 / (16 * math.pi)) * s * (1 + c) * np.exp(1j * ph),
        -1: math.sqrt(5 / (16 * math.pi)) * s * (1 - c) * np.exp(-1j * ph),
        0: math.sqrt(15 / (32 * math.pi)) * s * s + 0j,
    }
    for m, r in ref.items():
        np.testing.assert_allclose(lk.swsh(-2, 2, m, th, ph), r, rtol=0, atol=2e-15)


def test_ylm_sum_rule_and_symmetries():
    rng = _rng(2)
    th = rng.uniform(0, math.pi, 20)
    ph = rng.uniform(0, 2 * math.pi, 20)
    for l in (2, 3, 4):
        tot = sum(np.abs(lk.swsh(-2, l, m, th, ph)) ** 2 for m in range(-l, l + 1))
        np.testing.assert_allclose(tot, (2 * l + 1) / (4 * math.pi), rtol=1e-13)
        for m in range(-l, l + 1):
            a = np.conj(lk.swsh(-2, l, m, th, ph))
            b = (-1) ** (-2 + m) * lk.swsh(2, l, -m, th, ph)
            np.testing.assert_allclose(a, b, atol=1e-14)
            a = lk.swsh(-2, l, m, math.pi - th, ph + math.pi)
            b = (-1) ** l * lk.swsh(2, l, m, th, ph)
            np.testing.assert_allclose(a, b, atol=1e-14)


def test_ylm_orthonormal_by_quadrature():
    ell, m = make_modes(4)
    xg, wg = np.polynomial.legendre.leggauss(40)
    th = np.arccos(xg)
    nph = 64
    ph = 2 * math.pi * np.arange(nph) / nph
    TH, PH = np.meshgrid(th, ph, indexing="ij")
    W = (wg[:, None] * (2 * math.pi / nph) * np.ones((1, nph))).ravel()
    Y = lk.ylm(ell, m, TH.ravel(), PH.ravel())
    G = (Y.conj() * W[None, :]) @ Y.T
    np.testing.assert_allclose(G, np.eye(len(ell)), atol=1e-13)


def test_ylm_poles_finite():
    ell, m = make_modes(4)
    Y = lk.ylm(ell, m, np.array([0.0, math.pi]), np.array([0.3, 0.3]))
    assert np.isfinite(Y).all()
    # at iota = 0 only m = +2 survives, at pi only m = -2
    for i, (l, mm) in enumerate(zip(ell, m)):
        if mm != 2:
            assert abs(Y[i, 0]) < 1e-15
        if mm != -2:
            assert abs(Y[i, 1]) < 1e-15


# ------------------------------------------------------------------------------- P2: antenna
def test_antenna_psi_rotation_and_average():
    rng = _rng(3)
    D, pos = make_network(3, rng)
    N = 200000
    ra = rng.uniform(0, 2 * math.pi, N)
    dec = np.arcsin(rng.uniform(-1, 1, N))
    psi = rng.uniform(0, math.pi, N)
    Fp, Fx, tau = lk.antenna(D, pos, 0.3, ra, dec, psi)
    Fp0, Fx0, _ = lk.antenna(D, pos, 0.3, ra, dec, np.zeros(N))
    # F+ + iFx at psi = e^{-2 i psi} (value at psi = 0)
    np.testing.assert_allclose(Fp + 1j * Fx, np.exp(-2j * psi) * (Fp0 + 1j * Fx0), atol=1e-14)
    # sky+psi average of F+^2 + Fx^2 = (4/5) Tr(D^2) = 2/5 for Tr(D^2) = 1/2
    for k in range(3):
        avg = np.mean(Fp[k] ** 2 + Fx[k] ** 2)
        assert abs(avg - 0.8 * np.trace(D[k] @ D[k])) < 4e-3
    assert np.all(np.abs(tau) <= np.linalg.norm(pos, axis=1)[:, None] / lk.C_LIGHT * (1 + 1e-14))


def test_antenna_L_shaped_and_delay_extremes():
    # L-shaped interferometer D = (xx - yy)/2: source overhead (+z), psi=0 -> |F| = 1
    D = np.zeros((1, 3, 3))
    D[0, 0, 0], D[0, 1, 1] = 0.5, -0.5
    pos = np.array([[0.0, 0.0, 6.0e6]])
    Fp, Fx, tau = lk.antenna(D, pos, 0.0, np.array([0.7]), np.array([math.pi / 2]), np.array([0.0]))
    assert abs(math.hypot(Fp[0, 0], Fx[0, 0]) - 1.0) < 1e-14
    # source along +x_k: the detector hears it earlier by |x_k|/c
    assert abs(tau[0, 0] + 6.0e6 / lk.C_LIGHT) < 1e-18
    # detector at the geocentre: no delay
    _, _, tau0 = lk.antenna(D, np.zeros((1, 3)), 0.0, np.array([1.0]), np.array([0.2]), np.array([0.0]))
    assert tau0[0, 0] == 0.0
    # n-hat for (ra, dec) with gmst: source at ra = gmst, dec = 0 lies along +x (Earth-fixed)
    _, _, t2 = lk.antenna(D, np.array([[1.0e6, 0.0, 0.0]]), 1.1, np.array([1.1]), np.array([0.0]), np.array([0.0]))
    assert abs(t2[0, 0] + 1.0e6 / lk.C_LIGHT) < 1e-18


def test_polarisation_basis_orthonormal():
    # rebuild X, Y, n from the formulas' outputs: F for D = n n^T must vanish (transverse basis)
    rng = _rng(4)
    ra, dec, psi = rng.uniform(0, 6, 5), rng.uniform(-1.5, 1.5, 5), rng.uniform(0, 3, 5)
    for i in range(5):
        g = 0.4 - ra[i]
        n = np.array([math.cos(dec[i]) * math.cos(g), -math.cos(dec[i]) * math.sin(g), math.sin(dec[i])])
        D = np.outer(n, n)[None]
        Fp, Fx, _ = lk.antenna(D, np.zeros((1, 3)), 0.4, ra[i:i + 1], dec[i:i + 1], psi[i:i + 1])
        assert abs(Fp[0, 0]) < 1e-15 and abs(Fx[0, 0]) < 1e-15
        # identity tensor: X.X - Y.Y = 0 and 2 X.Y = 0
        Fp, Fx, _ = lk.antenna(np.eye(3)[None], np.zeros((1, 3)), 0.4, ra[i:i + 1], dec[i:i + 1], psi[i:i + 1])
        assert abs(Fp[0, 0]) < 1e-15 and abs(Fx[0, 0]) < 1e-15


# ------------------------------------------------------------------------------- P3: Eq. 7 scalar case
def test_single_detector_single_mode_closed_form():
    rng = _rng(5)
    D, pos = make_network(1, rng)
    pos[:] = 0.0                                   # no delay: Q index is exact
    ell, m = np.array([2]), np.array([2])
    N_Q, fs, t_Q0 = 64, 4096.0, -32 / 4096.0
    Q = (rng.standard_normal((1, 1, N_Q)) + 1j * rng.standard_normal((1, 1, N_Q)))
    Us, Vs = 1.7, 0.3 - 0.4j
    U = np.array([[[Us + 0j]]])
    V = np.array([[[Vs]]])
    D_ref = 100.0
    N = 7
    ra, dec, psi = rng.uniform(0, 6, N), rng.uniform(-1.5, 1.5, N), rng.uniform(0, 3, N)
    phi, incl, dist = rng.uniform(0, 6, N), rng.uniform(0.1, 3, N), rng.uniform(50, 300, N)
    N_t, t_lo, dt = 9, -4 / fs, 1 / fs
    lnL, lnLt = lk.lnL_angles(D, pos, 0.0, ell, m, Q, U, V, D_ref, fs, t_Q0, t_lo, dt, N_t,
                              ra, dec, psi, phi, incl, dist, return_series=True)
    Fp, Fx, _ = lk.antenna(D, pos, 0.0, ra, dec, psi)
    for i in range(N):
        F = complex(Fp[0, i], -Fx[0, i])
        Y = math.sqrt(5 / (64 * math.pi)) * (1 + math.cos(incl[i])) ** 2 * np.exp(-2j * phi[i])
        FY = F * Y
        x = D_ref / dist[i]
        for j in range(N_t):
            q = Q[0, 0, 32 - 4 + j]
            want = x * (np.conj(FY) * q).real - 0.25 * x * x * (abs(FY) ** 2 * Us + (FY * FY * Vs).real)
            assert abs(lnLt[i, j] - want) <= 1e-12 * max(1.0, abs(want))
        want_m = math.log(np.mean(np.exp(lnLt[i] - lnLt[i].max()))) + lnLt[i].max()
        assert abs(lnL[i] - want_m) < 1e-12


# ------------------------------------------------------------------------------- P4: zero-noise injection
@pytest.mark.parametrize("cfg", [1, 2])
def test_zero_noise_injection_peak_is_half_rho2(cfg):
    prob = make_problem(cfg, noise=False)
    prob.pos[:] = 0.0                             # co-located detectors: arrival on a stored bin
    inj = prob.inj[0]
    th = inj["theta0"]
    # rebuild Q without delays (tau = 0) from the same injection coefficients
    x0 = prob.D_ref / th["dist"]
    c0 = x0 * inj["F"][:, None] * inj["Y"][None, :]
    q0 = matched_q0(prob.U[0], prob.V[0], c0)
    rho2 = network_rho2(prob.U[0], prob.V[0], c0)
    assert abs(rho2 - prob.rho2) < 1e-9 * rho2
    Q = np.repeat(q0[:, :, None], prob.N_Q, axis=2)          # constant in time (also pins P5)
    args = dict(D=prob.D, pos=prob.pos, gmst=0.0, ell=prob.ell, m=prob.m, Q=Q, U=prob.U[0], V=prob.V[0],
                D_ref=prob.D_ref, fs=prob.fs, t_Q0=prob.t_Q0, t_lo=prob.t_lo, dt=prob.dt, N_t=prob.N_t)
    one = lambda v: np.array([v])
    lnL0 = lk.lnL_angles(ra=one(th["ra"]), dec=one(th["dec"]), psi=one(th["psi"]), phi_ref=one(th["phi_ref"]),
                         incl=one(th["incl"]), dist=one(th["dist"]), **args)
    assert abs(lnL0[0] - 0.5 * rho2) < 1e-10 * rho2
    # Cauchy-Schwarz: lnL(theta) <= rho^2 / 2 everywhere
    rng = _rng(6)
    N = 400
    lnL = lk.lnL_angles(ra=rng.uniform(0, 2 * math.pi, N), dec=np.arcsin(rng.uniform(-1, 1, N)),
                        psi=rng.uniform(0, math.pi, N), phi_ref=rng.uniform(0, 2 * math.pi, N),
                        incl=np.arccos(rng.uniform(-1, 1, N)), dist=rng.uniform(100, 2000, N), **args)
    assert lnL.max() <= 0.5 * rho2 * (1 + 1e-12)
    # maximum over D at fixed angles is A^2 / 4B at x* = A / 2B
    F = inj["F"]
    Y = inj["Y"]
    B = lk.quadratic_term(F[:, None], Y[:, None], prob.U[0], prob.V[0])[0]
    A = sum((np.conj(F[k]) * np.sum(np.conj(Y) * q0[k])).real for k in range(prob.K))
    assert abs(A * A / (4 * B) - 0.5 * rho2) < 1e-10 * rho2


# ------------------------------------------------------------------------------- P5: time LSE
def test_time_lse_shift_and_dominant_bin():
    rng = _rng(7)
    prob = make_problem(1)
    N = 16
    z = np.stack([rng.uniform(l, h, N) for l, h in zip(prob.lo, prob.hi)])
    args = dict(D=prob.D, pos=prob.pos, gmst=0.0, ell=prob.ell, m=prob.m, U=prob.U[0], V=prob.V[0],
                D_ref=prob.D_ref, fs=prob.fs, t_Q0=prob.t_Q0, t_lo=prob.t_lo, dt=prob.dt, N_t=prob.N_t)
    ang = lk.z_to_angles(z)
    lnL, lnLt = lk.lnL_angles(*([None] * 0), Q=prob.Q[0], ra=ang[0], dec=ang[1], psi=ang[2], phi_ref=ang[3],
                              incl=ang[4], dist=ang[5], return_series=True, **args)
    # definition
    want = np.log(np.mean(np.exp(lnLt - 5.0), axis=1)) + 5.0
    np.testing.assert_allclose(lnL, want, rtol=1e-12)
    # one huge spike in Q at one stored bin -> dominated by one (or two, interpolated) bins
    assert np.all(lnL <= lnLt.max(axis=1) + 1e-12)
    assert np.all(lnL >= lnLt.max(axis=1) - math.log(prob.N_t) - 1e-12)


# ------------------------------------------------------------------------------- P6: interpolation
def test_interpolation_exact_on_linear_q_and_nearest_mode():
    rng = _rng(8)
    prob = make_problem(1)
    K, M, N_Q = prob.K, prob.M, prob.N_Q
    a = rng.standard_normal((K, M)) + 1j * rng.standard_normal((K, M))
    b = rng.standard_normal((K, M)) + 1j * rng.standard_normal((K, M))
    t = prob.t_Q0 + np.arange(N_Q) / prob.fs
    Qlin = a[:, :, None] + b[:, :, None] * t[None, None, :] * 100.0
    N = 5
    z = np.stack([rng.uniform(l, h, N) for l, h in zip(prob.lo, prob.hi)])
    ang = lk.z_to_angles(z)
    args = dict(D=prob.D, pos=prob.pos, gmst=0.0, ell=prob.ell, m=prob.m, U=prob.U[0], V=prob.V[0],
                D_ref=prob.D_ref, fs=prob.fs, t_Q0=prob.t_Q0, t_lo=prob.t_lo, dt=prob.dt, N_t=prob.N_t,
                ra=ang[0], dec=ang[1], psi=ang[2], phi_ref=ang[3], incl=ang[4], dist=ang[5])
    _, lnLt = lk.lnL_angles(Q=Qlin, return_series=True, **args)
    # direct evaluation with Q(t) evaluated analytically at t_j + tau_k
    Fp, Fx, tau = lk.antenna(prob.D, prob.pos, 0.0, ang[0], ang[1], ang[2])
    F = Fp - 1j * Fx
    Y = lk.ylm(prob.ell, prob.m, ang[4], -ang[3])
    B = lk.quadratic_term(F, Y, prob.U[0], prob.V[0])
    x = prob.D_ref / ang[5]
    for j in range(prob.N_t):
        A = np.zeros(N)
        for k in range(K):
            tt = prob.t_lo + j * prob.dt + tau[k]
            Qe = a[k][:, None] + b[k][:, None] * tt[None, :] * 100.0
            A += (np.conj(F[k]) * np.sum(np.conj(Y) * Qe, axis=0)).real
        np.testing.assert_allclose(lnLt[:, j], x * A - x * x * B, rtol=1e-9, atol=1e-9)
    # nearest mode == linear mode when delays are zero (f = 0)
    args0 = dict(args, pos=np.zeros_like(prob.pos))
    l1 = lk.lnL_angles(Q=prob.Q[0], interp=1, **args0)
    l0 = lk.lnL_angles(Q=prob.Q[0], interp=0, **args0)
    np.testing.assert_array_equal(l1, l0)


def test_out_of_span_raises():
    prob = make_problem(1)
    z = np.array([[1.0], [0.1], [0.5], [1.0], [0.2], [500.0]])
    ang = lk.z_to_angles(z)
    with pytest.raises(ValueError):
        lk.lnL_angles(prob.D, prob.pos, 0.0, prob.ell, prob.m, prob.Q[0], prob.U[0], prob.V[0], prob.D_ref,
                      prob.fs, prob.t_Q0, -0.06, prob.dt, prob.N_t, *ang)


# ------------------------------------------------------------------------------- z <-> angles (G38)
def test_lnL_z_matches_angles():
    prob = make_problem(1)
    rng = _rng(9)
    N = 8
    z = np.stack([rng.uniform(l, h, N) for l, h in zip(prob.lo, prob.hi)])
    args = (prob.D, prob.pos, 0.0, prob.ell, prob.m, prob.Q[0], prob.U[0], prob.V[0], prob.D_ref,
            prob.fs, prob.t_Q0, prob.t_lo, prob.dt, prob.N_t)
    a = lk.lnL_z(*args, z)
    b = lk.lnL_angles(*args, z[0], np.arcsin(z[1]), z[2], z[3], np.arccos(z[4]), z[5])
    np.testing.assert_array_equal(a, b)
    lp = lk.ln_prior_z(z, prob.D_min, prob.D_max)
    want = np.log(3 * z[5] ** 2 / (2000.0 ** 3 - 100.0 ** 3) / (2 * math.pi * 2 * math.pi * 2 * math.pi * 2))
    np.testing.assert_allclose(lp, want, rtol=1e-14)


# ------------------------------------------------------------------------------- P12: distance table
def test_distance_table_against_quadrature_and_laplace():
    from scipy import integrate
    from synth import make_distance_table
    D_ref, D_min, D_max = 800.0, 100.0, 2000.0
    tab = make_distance_table(D_ref, D_min, D_max, 0.0, 500.0, 50.0, 400.0, nA=33, nB=17)
    rng = _rng(10)
    for _ in range(6):
        ia, ib = rng.integers(0, 33), rng.integers(0, 17)
        A = tab["A_lo"] + ia * (tab["A_hi"] - tab["A_lo"]) / 32
        B = tab["B_lo"] + ib * (tab["B_hi"] - tab["B_lo"]) / 16
        xs = max(min(A / (2 * B), D_ref / D_min), D_ref / D_max) if A > 0 else D_ref / D_max
        pk = xs * A - xs * xs * B
        f = lambda Dd: 3 * Dd * Dd / (D_max ** 3 - D_min ** 3) * math.exp(D_ref / Dd * A - (D_ref / Dd) ** 2 * B - pk)
        pts = [D_ref / xs] if D_min < D_ref / xs < D_max else None
        val, _ = integrate.quad(f, D_min, D_max, points=pts, epsabs=0, epsrel=1e-12, limit=400)
        assert abs(tab["lnT"][ib, ia] - (math.log(val) + pk)) < 1e-8
        # node lookup reproduces the node
        assert abs(lk.bilinear_table(tab, np.array([A]), np.array([B]))[0] - tab["lnT"][ib, ia]) < 1e-10
    # Laplace limit: A = 400, B = 300 -> 131.03 vs asymptotic 131.06
    A, B = 400.0, 300.0
    xs = A / (2 * B)
    lap = A * A / (4 * B) + 0.5 * math.log(math.pi / B) + math.log(3 * D_ref ** 3 / ((D_max ** 3 - D_min ** 3) * xs ** 4))
    got = lk.bilinear_table(make_distance_table(D_ref, D_min, D_max, 399.0, 401.0, 299.0, 301.0, nA=3, nB=3),
                            np.array([A]), np.array([B]))[0]
    assert abs(got - lap) < 5.0 / (B * xs * xs) * 2
    # clamping
    t = make_distance_table(D_ref, D_min, D_max, 0.0, 10.0, 1.0, 2.0, nA=5, nB=5)
    assert lk.bilinear_table(t, np.array([-5.0]), np.array([0.5]))[0] == t["lnT"][0, 0]
    assert lk.bilinear_table(t, np.array([50.0]), np.array([9.0]))[0] == t["lnT"][4, 4]
    # bilinear midpoint
    mid = lk.bilinear_table(t, np.array([1.25]), np.array([1.125]))[0]
    assert abs(mid - 0.25 * (t["lnT"][0, 0] + t["lnT"][0, 1] + t["lnT"][1, 0] + t["lnT"][1, 1])) < 1e-12
