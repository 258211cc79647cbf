"""GPU parity of ile_precompute_quv (Eq. 6a-c) against the oracle (-m gpu)."""
import numpy as np
import pytest

from synth import make_modes, make_network
from synth.spectra import make_spectra

pytestmark = pytest.mark.gpu


def _close(got, ref, rel):
    assert np.all(np.abs(got - ref) <= rel * np.abs(ref).max()), np.abs(got - ref).max() / np.abs(ref).max()


# window of 300 bins -> 512-point transforms of the spectrum decimated by 4, 2, 32, 128 and 1; 1536: not a power of two, by the definition
@pytest.mark.parametrize("lmax,K,N_f,P", [(2, 2, 2048, 2), (3, 3, 1024, 1), (2, 2, 16384, 2), (2, 1, 65536, 1), (2, 2, 1536, 1)])
def test_precompute_parity_and_lnL_from_it(lmax, K, N_f, P):
    import torch
    from paper_2505_11655_b200 import Ile
    from oracle import likelihood as lk
    from oracle.precompute import precompute_q, precompute_uv
    from synth.workloads import uniform_box_samples
    fs = 4096.0
    ell, m = make_modes(lmax)
    M = len(ell)
    rng = np.random.Generator(np.random.Philox(99))
    D, pos = make_network(K, rng)
    h, d, S, df = make_spectra(K, ell, m, N_f, fs, seed=4242 + lmax, P=P)
    f_low, N_Q, n0 = 20.0, 300, -150
    ile = Ile(0)
    ile.set_network(D, pos, 0.0)
    ile.set_modes(ell, m)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    ile.precompute_quv(dev(h), dev(d), dev(S), df, f_low, n0 / fs, N_Q, D_ref=500.0)
    for p in range(P):
        Q, U, V = ile.get_quv(p, K, M, N_Q)
        rU, rV = precompute_uv(h[p], S, df, f_low)
        rQ = precompute_q(h[p], d, S, df, f_low, n0 / fs, N_Q)
        _close(U, rU, 1e-12)
        _close(V, rV, 1e-12)
        _close(Q, rQ, 1e-11)
        for k in range(K):                                                         # Eq. 17-18 on the device result
            assert np.abs(U[k] - U[k].conj().T).max() <= 1e-13 * np.abs(U).max()
            assert np.abs(V[k] - V[k].T).max() <= 1e-13 * np.abs(V).max()
    # the likelihood evaluated from the device-made Q/U/V equals the oracle's from its own
    t_lo, N_t = -40 / fs, 81
    ile.set_time_grid(t_lo, 1.0 / fs, N_t)
    ile.set_prior(100.0, 2000.0)
    lo = np.array([0.0, -1.0, 0.0, 0.0, -1.0, 100.0])
    hi = np.array([2 * np.pi, 1.0, np.pi, 2 * np.pi, 1.0, 2000.0])
    z = uniform_box_samples(lo, hi, 700, seed=8)
    got = ile.lnL_z(P - 1, dev(z)).cpu().numpy()
    rU, rV = precompute_uv(h[P - 1], S, df, f_low)
    rQ = precompute_q(h[P - 1], d, S, df, f_low, n0 / fs, N_Q)
    ref = lk.lnL_z(D, pos, 0.0, ell, m, rQ, rU, rV, 500.0, fs, n0 / fs, t_lo, 1.0 / fs, N_t, z)
    assert np.all(np.abs(got - ref) <= 1e-9 * np.maximum(1.0, np.abs(ref))), np.abs(got - ref).max()


def test_precompute_parity_at_the_bench_shape():
    """The shape bench.py --precompute times (M = 21, K = 3, N_f = 32768, N_Q = 1024: the eight-column FFT
    instantiation and the tiled U/V grid), P = 2.  The oracle's Q is O(N_Q N_f K M): compared on two 32-bin windows
    (the first stored bins and the last), U and V in full."""
    import torch
    from paper_2505_11655_b200 import Ile
    from oracle.precompute import precompute_q, precompute_uv
    fs, N_f, K, P, N_Q = 4096.0, 32768, 3, 2, 1024
    ell, m = make_modes(4)
    M = len(ell)
    D, pos = make_network(K, np.random.Generator(np.random.Philox(99)))
    h, d, S, df = make_spectra(K, ell, m, N_f, fs, seed=77, P=P)
    f_low, n0 = 20.0, -(N_Q // 2)
    ile = Ile(0)
    ile.set_network(D, pos, 0.0)
    ile.set_modes(ell, m)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    ile.precompute_quv(dev(h), dev(d), dev(S), df, f_low, n0 / fs, N_Q, D_ref=500.0)
    for p in range(P):
        Q, U, V = ile.get_quv(p, K, M, N_Q)
        rU, rV = precompute_uv(h[p], S, df, f_low)
        _close(U, rU, 1e-12)
        _close(V, rV, 1e-12)
        scale = np.abs(Q).max()
        for first in (0, N_Q // 2 - 16, N_Q - 32):
            rQ = precompute_q(h[p], d, S, df, f_low, (n0 + first) / fs, 32)
            assert np.all(np.abs(Q[:, :, first:first + 32] - rQ) <= 1e-11 * scale), np.abs(Q[:, :, first:first + 32] - rQ).max() / scale

@pytest.mark.parametrize("N_f,N_Q,n0", [(4096, 200, -100), (2048, 1024, -700), (4096, 1500, 3000), (8192, 2048, -1024), (8192, 2500, -10)])
def test_precompute_q_window_shapes(N_f, N_Q, n0):
    """The transform sizes the pruned FFT instantiates (windows of 200 -> 256 points: the register tail, one output per
    thread; 1024 points with a spectrum decimated by 2 only: half-empty groups; 1500 and 2048 -> 2048 points: odd log2, eight
    outputs per thread), windows that wrap around the segment (n0 > 0 near the end), and a window above 2048 bins, which the
    definition kernel takes.  Q in full against the oracle's definition; K = 1, l = 2."""
    import torch
    from paper_2505_11655_b200 import Ile
    from oracle.precompute import precompute_q, precompute_uv
    fs, K = 4096.0, 1
    ell, m = make_modes(2)
    M = len(ell)
    D, pos = make_network(K, np.random.Generator(np.random.Philox(99)))
    h, d, S, df = make_spectra(K, ell, m, N_f, fs, seed=31 + N_Q, P=1)
    ile = Ile(0)
    ile.set_network(D, pos, 0.0)
    ile.set_modes(ell, m)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    ile.precompute_quv(dev(h), dev(d), dev(S), df, 20.0, n0 / fs, N_Q, D_ref=500.0)
    Q, U, V = ile.get_quv(0, K, M, N_Q)
    rQ = precompute_q(h[0], d, S, df, 20.0, n0 / fs, N_Q)
    rU, rV = precompute_uv(h[0], S, df, 20.0)
    _close(Q, rQ, 1e-11)
    _close(U, rU, 1e-12)
    _close(V, rV, 1e-12)


def test_precompute_argument_errors():
    import torch
    from paper_2505_11655_b200 import Ile, IleError
    ell, m = make_modes(2)
    rng = np.random.Generator(np.random.Philox(1))
    D, pos = make_network(2, rng)
    h, d, S, df = make_spectra(2, ell, m, 256, 4096.0, seed=5)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    ile = Ile(0)
    with pytest.raises(IleError):
        ile.precompute_quv(dev(h), dev(d), dev(S), df, 20.0, 0.0, 64, 500.0)          # ESTATE: no network / modes
    ile.set_network(D, pos, 0.0)
    ile.set_modes(ell, m)
    with pytest.raises(IleError):
        ile.precompute_quv(dev(h), dev(d), dev(S), df, 20.0, 0.3 / 4096.0, 64, 500.0)  # t_Q0 off the sample grid
    with pytest.raises(IleError):
        ile.precompute_quv(dev(h), dev(d), dev(S), df, 20.0, 0.0, 1024, 500.0)         # window longer than the segment
    ile.precompute_quv(dev(h), dev(d), dev(S), df, 20.0, -32 / 4096.0, 64, 500.0)
