"""GPU parity: CUDA path (through the C ABI) vs the oracle, element by element (-m gpu)."""
import math

import numpy as np
import pytest

from synth import make_problem
from synth.workloads import uniform_box_samples

pytestmark = pytest.mark.gpu


VARIANTS = (0, 1, 2, 3)        # every value ile_set_lnL_variant accepts
FUSED = (0, 2)                 # the two fused kernels (tcgen05 digits, FP64 DMMA)


def _tol(ref):
    return 1e-9 * np.maximum(1.0, np.abs(ref))      # north_star: per-sample lnL within 1e-9 relative (fp64)


@pytest.fixture(scope="module")
def torch_mod():
    import torch
    return torch


def _ile(prob):
    from paper_2505_11655_b200 import Ile
    ile = Ile(0)
    ile.load_problem(prob)
    return ile


def _dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def test_antenna_and_ylm_parity(torch_mod):
    from oracle import likelihood as lk
    torch = torch_mod
    prob = make_problem(2)
    ile = _ile(prob)
    rng = np.random.default_rng(5)
    N = 4099
    ra, dec, psi = rng.uniform(0, 2 * math.pi, N), np.arcsin(rng.uniform(-1, 1, N)), rng.uniform(0, math.pi, N)
    incl, phi = np.arccos(rng.uniform(-1, 1, N)), rng.uniform(0, 2 * math.pi, N)
    incl[:2] = [0.0, math.pi]
    Fp, Fx, tau = ile.antenna(_dev(torch, ra), _dev(torch, dec), _dev(torch, psi), prob.K)
    rFp, rFx, rtau = lk.antenna(prob.D, prob.pos, prob.gmst, ra, dec, psi)
    np.testing.assert_allclose(Fp.cpu().numpy(), rFp, rtol=0, atol=1e-14)
    np.testing.assert_allclose(Fx.cpu().numpy(), rFx, rtol=0, atol=1e-14)
    np.testing.assert_allclose(tau.cpu().numpy(), rtau, rtol=0, atol=1e-17)
    Y = ile.ylm(_dev(torch, incl), _dev(torch, phi), prob.M).cpu().numpy()
    rY = lk.ylm(prob.ell, prob.m, incl, phi)
    np.testing.assert_allclose(Y[..., 0] + 1j * Y[..., 1], rY, rtol=0, atol=2e-15)


@pytest.mark.parametrize("cfg,N", [(1, 5000), (2, 1531)])
def test_lnL_parity_all_entry_points(torch_mod, cfg, N):
    from oracle import likelihood as lk
    torch = torch_mod
    prob = make_problem(cfg)
    ile = _ile(prob)
    z = uniform_box_samples(prob.lo, prob.hi, N, seed=77 + cfg)
    ref = lk.lnL_z(prob.D, prob.pos, prob.gmst, prob.ell, prob.m, prob.Q[0], prob.U[0], prob.V[0], prob.D_ref, prob.fs,
                   prob.t_Q0, prob.t_lo, prob.dt, prob.N_t, z)
    zd = _dev(torch, z)
    # every kernel the ABI can select: 0 = tcgen05 integer-digit kernel where the shape allows (config 1's stride-2
    # grid runs the DMMA kernel), 1 = plain, 2 = DMMA kernel behind the delay-cell sort, 3 = DMMA kernel, unsorted
    for variant in VARIANTS:
        ile.set_lnL_variant(variant)
        got, lp = ile.lnL_z(0, zd, want_prior=True)
        got = got.cpu().numpy()
        assert np.all(np.abs(got - ref) <= _tol(ref)), (variant, np.abs(got - ref).max())
        np.testing.assert_allclose(lp.cpu().numpy(), lk.ln_prior_z(z, prob.D_min, prob.D_max), rtol=1e-14)
    ang = lk.z_to_angles(z)
    got2, dump = ile.lnL(0, *[_dev(torch, a) for a in ang], N_t_dump=prob.N_t)
    assert np.all(np.abs(got2.cpu().numpy() - ref) <= _tol(ref))
    _, ref_t = lk.lnL_angles(prob.D, prob.pos, prob.gmst, prob.ell, prob.m, prob.Q[0], prob.U[0], prob.V[0], prob.D_ref,
                             prob.fs, prob.t_Q0, prob.t_lo, prob.dt, prob.N_t, *[a[:64] for a in ang], return_series=True)
    d = dump.cpu().numpy()[:64]
    assert np.all(np.abs(d - ref_t) <= 1e-9 * np.maximum(1.0, np.abs(ref_t)))


def test_lnL_localised_samples_single_round(torch_mod):
    """Samples concentrated on the sky (what the adapted samplers produce): one round per tile."""
    from oracle import likelihood as lk
    torch = torch_mod
    prob = make_problem(3)
    ile = _ile(prob)
    N = 2048 + 17
    z = uniform_box_samples(prob.lo, prob.hi, N, seed=5)
    th = prob.inj[0]["theta0"]
    z[0] = th["ra"] + 0.01 * (z[0] / (2 * math.pi) - 0.5)
    z[1] = math.sin(th["dec"]) + 0.01 * z[1]
    z[:, 7] = [7.0, 0.0, 1.0, 1.0, 0.0, 500.0]                        # one out-of-box sample
    ref = lk.lnL_z(prob.D, prob.pos, prob.gmst, prob.ell, prob.m, prob.Q[0], prob.U[0], prob.V[0], prob.D_ref, prob.fs,
                   prob.t_Q0, prob.t_lo, prob.dt, prob.N_t, np.delete(z, 7, axis=1))
    assert ref.max() > 1000.0                                         # loud source: lnL dynamic range
    for variant in FUSED:
        ile.set_lnL_variant(variant)
        got = ile.lnL_z(0, _dev(torch, z)).cpu().numpy()
        assert got[7] == -np.inf
        got = np.delete(got, 7)
        assert np.all(np.abs(got - ref) <= _tol(ref)), (variant, np.abs(got - ref).max())


def test_lnL_nearest_bin_and_table(torch_mod):
    from oracle import likelihood as lk
    torch = torch_mod
    prob = make_problem(5, N=1)
    ile = _ile(prob)
    N = 777
    z = uniform_box_samples(prob.lo, prob.hi, N, seed=9)
    args = (prob.D, prob.pos, prob.gmst, prob.ell, prob.m, prob.Q[0], prob.U[0], prob.V[0], prob.D_ref, prob.fs,
            prob.t_Q0, prob.t_lo, prob.dt, prob.N_t)
    ref = lk.lnL_z(*args, z, table=prob.table)
    zd = _dev(torch, z)
    ref0 = lk.lnL_z(*args, z, interp=0, table=prob.table)
    for variant in FUSED:
        ile.set_lnL_variant(variant)
        ile.set_time_grid(prob.t_lo, prob.dt, prob.N_t, 1)
        got = ile.lnL_z(0, zd).cpu().numpy()
        assert np.all(np.abs(got - ref) <= _tol(ref)), (variant, np.abs(got - ref).max())
        ile.set_time_grid(prob.t_lo, prob.dt, prob.N_t, 0)            # nearest-bin mode
        got0 = ile.lnL_z(0, zd).cpu().numpy()
        assert np.all(np.abs(got0 - ref0) <= _tol(ref0)), (variant, np.abs(got0 - ref0).max())


@pytest.mark.parametrize("nA,nB,a_lo,a_hi", [(256, 256, 0.05, 0.2), (40, 7, -0.1, 0.5), (5, 3, 0.0, 1.3), (2, 2, 0.0, 0.1), (33, 2, 0.0, 0.02)])
def test_lnL_table_edges(torch_mod, nA, nB, a_lo, a_hi):
    """Distance tables whose A range is left on both sides (lookups clamped to the edges, G28) and whose rows are shorter
    than, equal to and longer than the part of a row the fused kernel keeps in shared memory; B range narrower than the
    samples' B."""
    from oracle import likelihood as lk
    from synth.workloads import make_distance_table, D0_MPC
    torch = torch_mod
    prob = make_problem(5, N=1)
    x0 = prob.D_ref / D0_MPC
    A_pk, B_pk = prob.rho2 / x0, prob.rho2 / (2.0 * x0 * x0)
    table = make_distance_table(prob.D_ref, prob.D_min, prob.D_max, a_lo * A_pk, a_hi * A_pk, 0.4 * B_pk, 0.9 * B_pk, nA=nA, nB=nB, nodes=257)
    ile = _ile(prob)
    ile.load_distance_table(table)
    N = 1301
    z = uniform_box_samples(prob.lo, prob.hi, N, seed=21)
    # a few samples at the injected parameters' neighbourhood, so that rows near the arrival time reach the top of the table
    th = prob.inj[0]["theta0"]
    inj = np.array([th["ra"], math.sin(th["dec"]), th["psi"], th["phi_ref"], math.cos(th["incl"])])[: z.shape[0]]
    z[:, :64] = inj[:, None] + 1e-3 * (z[:, :64] - inj[:, None])
    z = np.minimum(np.maximum(z, np.asarray(prob.lo)[:, None]), np.nextafter(np.asarray(prob.hi), -np.inf)[:, None])
    args = (prob.D, prob.pos, prob.gmst, prob.ell, prob.m, prob.Q[0], prob.U[0], prob.V[0], prob.D_ref, prob.fs,
            prob.t_Q0, prob.t_lo, prob.dt, prob.N_t)
    ref = lk.lnL_z(*args, z, table=table)
    zd = _dev(torch, z)
    for variant in FUSED:
        ile.set_lnL_variant(variant)
        got = ile.lnL_z(0, zd).cpu().numpy()
        assert np.all(np.abs(got - ref) <= _tol(ref)), (variant, np.abs(got - ref).max())


@pytest.mark.parametrize("cfg", [1, 2, 4, 5])
def test_lnL_repeatable(torch_mod, cfg):
    """The fused kernels on the same batch again and again: bit-identical results.  Nothing in them depends on the order in
    which warps run, so any difference is a race (the quartets of a tile are not in step with each other, and shared-memory
    arrays are reused between the phases); the first call is compared with the oracle on a subset."""
    from oracle import likelihood as lk
    torch = torch_mod
    prob = make_problem(cfg, N=1) if cfg in (4, 5) else make_problem(cfg)
    ile = _ile(prob)
    N = 60013
    z = uniform_box_samples(prob.lo, prob.hi, N, seed=101 + cfg)
    th = prob.inj[0]["theta0"]
    inj = np.array([th["ra"], math.sin(th["dec"]), th["psi"], th["phi_ref"], math.cos(th["incl"]), th["dist"]])[: z.shape[0]]
    half = N // 2                                                     # half of the batch around the injected parameters
    z[:, :half] = inj[:, None] + 0.05 * (z[:, :half] - inj[:, None])
    z = np.minimum(np.maximum(z, np.asarray(prob.lo)[:, None]), np.nextafter(np.asarray(prob.hi), -np.inf)[:, None])
    zd = _dev(torch, z)
    for variant in FUSED:
        ile.set_lnL_variant(variant)
        first = ile.lnL_z(0, zd).cpu().numpy()
        for rep in range(6):
            again = ile.lnL_z(0, zd).cpu().numpy()
            assert np.array_equal(first, again, equal_nan=True), (variant, rep, np.nanmax(np.abs(first - again)))
        sub = np.r_[0:96, half - 48:half + 48, N - 96:N]
        ref = lk.lnL_z(prob.D, prob.pos, prob.gmst, prob.ell, prob.m, prob.Q[0], prob.U[0], prob.V[0], prob.D_ref, prob.fs,
                       prob.t_Q0, prob.t_lo, prob.dt, prob.N_t, z[:, sub], table=prob.table)
        assert np.all(np.abs(first[sub] - ref) <= _tol(ref)), (variant, np.abs(first[sub] - ref).max())


def test_reduce_parity(torch_mod):
    from oracle.reduce import reduce_lnw
    torch = torch_mod
    prob = make_problem(1)
    ile = _ile(prob)
    rng = np.random.default_rng(3)
    for N in (1, 31, 100003):
        lnw = rng.normal(0, 30, N) + 4000.0
        if N > 50:
            lnw[5] = -np.inf
            lnw[6] = np.nan
        ref = reduce_lnw(lnw)
        got = ile.reduce(_dev(torch, lnw))
        assert abs(got["ln_integral"] - ref["ln_integral"]) <= 1e-8                 # north_star: log-integral within 1e-8
        for k in ("n_eff", "n_ess", "rel_variance"):
            assert abs(got[k] - ref[k]) <= 1e-9 * max(1.0, abs(ref[k]))
        assert got["n_samples"] == N and got["n_nonfinite"] == ref["n_nonfinite"]
        assert got["ln_w_max"] == ref["ln_w_max"]
    got = ile.reduce(_dev(torch, np.full(10, -np.inf)))
    assert got["ln_integral"] == -np.inf and got["n_eff"] == 0


def test_error_paths(torch_mod):
    from paper_2505_11655_b200 import Ile, IleError
    prob = make_problem(1)
    ile = Ile(0)
    with pytest.raises(IleError):
        ile.set_time_grid(prob.t_lo, prob.dt, prob.N_t)              # ESTATE: nothing loaded
    ile.set_network(prob.D, prob.pos, 0.0)
    ile.set_modes(prob.ell, prob.m)
    Ubad = prob.U.copy()
    Ubad[0, 0, 0, 1] += 1e-6
    with pytest.raises(IleError):
        ile.load_quv(prob.Q, Ubad, prob.V, prob.fs, prob.t_Q0, prob.D_ref)   # Eq. 17 violated
    ile.load_quv(prob.Q, prob.U, prob.V, prob.fs, prob.t_Q0, prob.D_ref)
    with pytest.raises(IleError):
        ile.set_time_grid(-0.045, prob.dt, prob.N_t)                 # ERANGE: window + delays leave Q
    with pytest.raises(IleError):
        ile.set_time_grid(prob.t_lo, 1.5 / prob.fs, 10)              # non-integer stride


@pytest.mark.parametrize("variant", FUSED)
@pytest.mark.parametrize("N_t,stride", [(1, 1), (7, 1), (15, 1), (16, 1), (17, 1), (63, 1), (64, 1), (65, 1), (129, 1), (333, 1), (50, 2), (131, 3)])
def test_time_grid_shapes(torch_mod, N_t, stride, variant):
    """Window lengths around the 64-output phases of the DMMA kernel and the 16-bin work items of the tcgen05 kernel
    (one phase, exactly full, one bin over, a short tail) and time steps of 2 and 3 stored bins (DMMA kernel in
    both variants), on the l <= 4 three-detector problem."""
    from oracle import likelihood as lk
    torch = torch_mod
    prob = make_problem(2)
    ile = _ile(prob)
    ile.set_lnL_variant(variant)
    dt = stride / prob.fs
    t_lo = -0.5 * (N_t - 1) * dt
    t_lo = round(t_lo * prob.fs) / prob.fs                              # on the stored grid
    ile.set_time_grid(t_lo, dt, N_t, 1)
    N = 32 * 9 + 5
    z = uniform_box_samples(prob.lo, prob.hi, N, seed=100 + N_t)
    ref = lk.lnL_z(prob.D, prob.pos, prob.gmst, prob.ell, prob.m, prob.Q[0], prob.U[0], prob.V[0], prob.D_ref, prob.fs,
                   prob.t_Q0, t_lo, dt, N_t, z)
    got = ile.lnL_z(0, _dev(torch, z)).cpu().numpy()
    assert np.all(np.abs(got - ref) <= _tol(ref)), np.abs(got - ref).max()


@pytest.mark.parametrize("K,lmax", [(1, 2), (2, 3), (3, 3), (3, 4)])
def test_lnL_other_shapes(torch_mod, K, lmax):
    """Detector and mode counts other than the configs': K = 1..3, l <= 2, 3, 4 (M = 5, 12, 21) through the tcgen05
    kernel (any M <= 24) and whatever the DMMA variant falls back to."""
    from oracle import likelihood as lk
    from synth.workloads import make_custom_problem
    torch = torch_mod
    prob = make_custom_problem(K=K, lmax=lmax, snr=30.0, seed=40 + 10 * K + lmax)
    ile = _ile(prob)
    N = 700
    z = uniform_box_samples(prob.lo, prob.hi, N, seed=3)
    ref = lk.lnL_z(prob.D, prob.pos, prob.gmst, prob.ell, prob.m, prob.Q[0], prob.U[0], prob.V[0], prob.D_ref, prob.fs,
                   prob.t_Q0, prob.t_lo, prob.dt, prob.N_t, z)
    for variant in FUSED:
        ile.set_lnL_variant(variant)
        got = ile.lnL_z(0, _dev(torch, z)).cpu().numpy()
        assert np.all(np.abs(got - ref) <= _tol(ref)), (variant, np.abs(got - ref).max())


_L4 = [(l, mm) for l in (2, 3, 4) for mm in range(-l, l + 1)]


@pytest.mark.parametrize("K,modes", [(3, _L4 + [(5, 5)]),                                         # M = 22: the most ile_load_quv takes
                                     (2, [lm for lm in _L4 if lm[1] != 0]),                       # M = 18: even row lengths in step 4
                                     (3, [(2, 2), (2, -2), (3, 3), (3, -3), (4, 4), (4, -4), (2, 1)]),   # M = 7
                                     (1, [(2, 2)])])                                              # one mode
def test_lnL_mode_lists(torch_mod, K, modes):
    """Mode sets that are not 'all modes up to l_max': the largest the library takes, an even count, a short odd list and a
    single mode (step 4's rows are dealt to the thread groups per (M, K); digits are cut in groups of four reals)."""
    from oracle import likelihood as lk
    from synth.workloads import make_custom_problem
    torch = torch_mod
    prob = make_custom_problem(K=K, lmax=2, snr=30.0, seed=70 + len(modes), modes=modes)
    ile = _ile(prob)
    N = 900
    z = uniform_box_samples(prob.lo, prob.hi, N, seed=11)
    ref = lk.lnL_z(prob.D, prob.pos, prob.gmst, prob.ell, prob.m, prob.Q[0], prob.U[0], prob.V[0], prob.D_ref, prob.fs,
                   prob.t_Q0, prob.t_lo, prob.dt, prob.N_t, z)
    for variant in FUSED:
        ile.set_lnL_variant(variant)
        got = ile.lnL_z(0, _dev(torch, z)).cpu().numpy()
        assert np.all(np.abs(got - ref) <= _tol(ref)), (variant, np.abs(got - ref).max())


@pytest.mark.parametrize("K,lmax", [(1, 2), (2, 3), (2, 4)])
def test_lnL_table_other_shapes(torch_mod, K, lmax):
    """Distance marginalisation through the table with one and two detectors (the fused kernels are instantiated per detector
    count and table mode; config 5 covers three detectors only)."""
    from oracle import likelihood as lk
    from synth.workloads import make_custom_problem, make_distance_table, D0_MPC
    torch = torch_mod
    prob = make_custom_problem(K=K, lmax=lmax, snr=25.0, seed=300 + 10 * K + lmax)
    x0 = prob.D_ref / D0_MPC
    A_pk, B_pk = prob.rho2 / x0, prob.rho2 / (2.0 * x0 * x0)
    table = make_distance_table(prob.D_ref, prob.D_min, prob.D_max, 0.0, 1.3 * A_pk, 0.02 * B_pk, 3.0 * B_pk, nA=96, nB=64, nodes=513)
    ile = _ile(prob)
    ile.load_distance_table(table)
    N = 1100
    z = uniform_box_samples(prob.lo[:5], prob.hi[:5], N, seed=17)
    ref = lk.lnL_z(prob.D, prob.pos, prob.gmst, prob.ell, prob.m, prob.Q[0], prob.U[0], prob.V[0], prob.D_ref, prob.fs,
                   prob.t_Q0, prob.t_lo, prob.dt, prob.N_t, z, table=table)
    for variant in FUSED:
        ile.set_lnL_variant(variant)
        got = ile.lnL_z(0, _dev(torch, z)).cpu().numpy()
        assert np.all(np.abs(got - ref) <= _tol(ref)), (variant, np.abs(got - ref).max())


def test_too_many_modes_rejected(torch_mod):
    from paper_2505_11655_b200 import Ile
    from paper_2505_11655_b200.binding import IleError
    from synth.workloads import make_custom_problem
    prob = make_custom_problem(K=2, lmax=2, snr=30.0, seed=99, modes=_L4 + [(5, 5), (5, -5)])           # M = 23
    ile = Ile(0)
    ile.set_network(prob.D, prob.pos, prob.gmst)
    ile.set_modes(prob.ell, prob.m)
    with pytest.raises(IleError, match="at most 22 modes"):
        ile.load_quv(prob.Q, prob.U, prob.V, prob.fs, prob.t_Q0, prob.D_ref)


def test_two_contexts_in_one_process(torch_mod):
    """Two contexts alive at once (different networks, mode sets and time grids), calls interleaved: each answers as it
    does alone.  The kernels' shared-memory opt-in and every other piece of launch state is per call, not per process."""
    from oracle import likelihood as lk
    torch = torch_mod
    probs = [make_problem(1), make_problem(2)]
    iles = [_ile(p) for p in probs]
    zs = [uniform_box_samples(p.lo, p.hi, 900 + 37 * i, seed=500 + i) for i, p in enumerate(probs)]
    refs = [lk.lnL_z(p.D, p.pos, p.gmst, p.ell, p.m, p.Q[0], p.U[0], p.V[0], p.D_ref, p.fs, p.t_Q0, p.t_lo, p.dt, p.N_t, z)
            for p, z in zip(probs, zs)]
    for variant in FUSED:
        for ile in iles:
            ile.set_lnL_variant(variant)
        for rnd in range(2):
            outs = [ile.lnL_z(0, _dev(torch, z)) for ile, z in zip(iles, zs)]           # both queued before either is read
            for out, ref in zip(outs, refs):
                got = out.cpu().numpy()
                assert np.all(np.abs(got - ref) <= _tol(ref)), (variant, rnd, np.abs(got - ref).max())
    # an integrator on each, stepped alternately (same kernel as the solo runs: the default)
    for ile in iles:
        ile.set_lnL_variant(0)
    from paper_2505_11655_b200 import Integrator
    from paper_2505_11655_b200.binding import result_from_device

    def make(ile, p, i):
        return Integrator(ile, "AC", p.d, p.lo, p.hi, seed=9 + i, max_batch=4096)

    def step(it, g):
        return float(result_from_device(it.step(0, 4096, g))["ln_integral"][0])

    solo = []
    for i, p in enumerate(probs):
        it = make(_ile(p), p, i)
        solo.append([step(it, g) for g in range(3)])
    its = [make(ile, p, i) for i, (ile, p) in enumerate(zip(iles, probs))]
    both = [[], []]
    for g in range(3):
        for i, it in enumerate(its):
            both[i].append(step(it, g))
    assert both == solo
