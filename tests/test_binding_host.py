"""Host-side logic of the binding (no GPU): state blob layout round trip, option defaults through
the C ABI, error codes of calls that must fail without touching a device."""
import ctypes as C

import numpy as np

from paper_2505_11655_b200 import binding as b


def _ac(d=3, nb=7, seed=0):
    rng = np.random.default_rng(seed)
    return dict(kind=b.KINDS["AC"], d=d, n_bins=nb, H=rng.integers(0, 1 << 60, (d, nb)).astype(np.uint64),
                pi=rng.random((d, nb)), cdf=rng.random((d, nb + 1)))


def _av(d=3, C_=11, seed=1):
    rng = np.random.default_rng(seed)
    return dict(kind=b.KINDS["AV"], d=d, n=9, C=C_, N_min=123, L_thr=-4.5, keys=np.sort(rng.integers(0, 9 ** d, C_)).astype(np.uint64))


def _gmm(d=3, C_=4, seed=2):
    rng = np.random.default_rng(seed)
    return dict(kind=b.KINDS["GMM"], d=d, n_comp=C_, gd=d, omega=rng.random(C_), mu=rng.random((C_, d)), Sigma=rng.random((C_, d, d)),
                L=rng.random((C_, d, d)))


def _same(x, y):
    assert x.keys() == y.keys()
    for k in x:
        if isinstance(x[k], np.ndarray):
            assert x[k].dtype == y[k].dtype and np.array_equal(x[k], y[k]), k
        elif isinstance(x[k], list):
            for p, q in zip(x[k], y[k]):
                _same(p, q)
        else:
            assert x[k] == y[k], k


def test_member_blobs_round_trip():
    for st in (_ac(), _av(), _gmm()):
        blob = b.pack_state(st)
        assert len(blob) % 8 == 0
        _same(b.parse_state(blob), st)
    ac = _ac()
    assert len(b.pack_state(ac)) == 16 + 8 + 3 * 7 * 16 + 3 * 8 * 8           # header, n_bins, H + pi, cdf (include/ile.h)
    av = _av()
    assert len(b.pack_state(av)) == 16 + 32 + 11 * 8


def test_portfolio_blob_round_trip():
    W = np.zeros(8)
    W[:3] = [0.2, 0.3, 0.5]
    st = dict(kind=b.KINDS["PORTFOLIO"], d=3, n_members=3, W=W, frozen=np.array([0, 1, 0, 0, 0, 0, 0, 0], dtype=np.int64),
              alloc=np.array([10, 20, 30, 0, 0, 0, 0, 0], dtype=np.int64), active=np.array([1, 1, 1, 0, 0, 0, 0, 0], dtype=np.int64),
              members=[_ac(), _av(), _gmm()])
    _same(b.parse_state(b.pack_state(st)), st)


def test_opts_default_through_the_abi():
    lib = b.load_library()
    o = b.IntegratorOpts()
    assert lib.ile_integrator_opts_default(C.byref(o), b.KINDS["PORTFOLIO"], 5) == 0
    assert (o.kind, o.d, o.n_bins, o.n_gmm, o.n_members) == (4, 5, 100, 8, 3)
    assert list(o.member_kind)[:3] == [b.KINDS["AC"], b.KINDS["AV"], b.KINDS["GMM"]]
    assert abs(o.eps - 0.1) < 1e-15 and o.beta == 1.0 and o.P_thr == 0.999 and o.N_min_star == 4096
    assert abs(o.hi[0] - 2 * np.pi) < 1e-15 and o.lo[1] == -1.0 and abs(o.hi[2] - np.pi) < 1e-15
    assert lib.ile_integrator_opts_default(C.byref(o), 9, 5) == -1 and lib.ile_integrator_opts_default(C.byref(o), 1, 0) == -1
    assert lib.ile_integrator_opts_default(C.byref(o), 1, 9) == -1


def test_null_handles_are_rejected():
    lib = b.load_library()
    assert lib.ile_sync(None) == -1 and lib.ile_destroy(None) == -1
    assert lib.ile_integrator_destroy(None) == -1 and lib.ile_integrator_reset(None) == -1
    assert lib.ile_set_prior(None, C.c_double(1.0), C.c_double(2.0)) == -1
    lib.ile_last_error.restype = C.c_char_p
    assert lib.ile_last_error(None) == b"null context"
