"""Pins of the Q/U/V precompute oracle (Eq. 6a-c; symmetries Eq. 17-18)."""
import numpy as np

from oracle.precompute import precompute_q, precompute_uv, weights


def _setup(M=4, K=2, N_f=512, seed=0):
    rng = np.random.default_rng(seed)
    ht = rng.standard_normal((M, N_f)) + 1j * rng.standard_normal((M, N_f))       # complex time-domain modes
    ht *= np.hanning(N_f)[None, :]
    h = np.fft.fft(ht, axis=1)
    S = 1.0 + rng.random((K, N_f // 2 + 1))
    return rng, ht, h, S


def test_symmetries_eq17_18_and_positive_norms():
    rng, ht, h, S = _setup()
    U, V = precompute_uv(h, S, df=0.25, f_low=3.0)
    for k in range(U.shape[0]):
        assert np.allclose(U[k], U[k].conj().T, rtol=0, atol=1e-12 * np.abs(U).max())          # Eq. 17
        assert np.allclose(V[k], V[k].T, rtol=0, atol=1e-12 * np.abs(V).max())                 # Eq. 18
        assert np.all(np.linalg.eigvalsh(U[k]) > 0)


def test_white_noise_parseval():
    """S = const, f_low < 0: <a|b> = (2 df / S) sum_f a~* b~ = (2 df N_f / S) sum_t a*(t) b(t)."""
    rng, ht, h, S = _setup()
    N_f, df, S0 = h.shape[1], 0.5, 3.0
    Sc = np.full_like(S, S0)
    U, V = precompute_uv(h, Sc, df, f_low=-1.0)
    ref_U = 2 * df * N_f / S0 * np.einsum("at,bt->ab", ht.conj(), ht)
    ref_V = 2 * df * N_f / S0 * np.einsum("at,bt->ab", ht, ht)                                  # <a*|b> = sum a b
    assert np.allclose(U[0], ref_U, rtol=1e-12) and np.allclose(V[0], ref_V, rtol=1e-12)


def test_q_is_the_inverse_fft_of_the_weighted_product():
    rng, ht, h, S = _setup()
    N_f, df = h.shape[1], 0.25
    d = np.fft.fft(rng.standard_normal((2, N_f)), axis=1)
    fs = N_f * df
    n0, N_Q = -20, 48
    Q = precompute_q(h, d, S, df, 2.0, n0 / fs, N_Q)
    w = weights(S, N_f, df, 2.0)
    for k in range(2):
        for a in range(h.shape[0]):
            full = N_f * np.fft.ifft(w[k] * np.conj(h[a]) * d[k])                                # library routine
            ref = full[(np.arange(N_Q) + n0) % N_f]
            assert np.allclose(Q[k, a], ref, rtol=0, atol=1e-10 * np.abs(full).max())


def test_noise_free_data_equal_to_a_delayed_mode_peaks_at_the_delay_with_height_U():
    """d = h_a delayed by an integer number of samples: Q_a(delay) = <h_a|h_a> = U_aa, |Q_a(t)| <= U_aa."""
    rng, ht, h, S = _setup(M=3, K=1)
    N_f, df = h.shape[1], 0.25
    fs = N_f * df
    delay = 7
    j = np.arange(N_f)
    d = (h[1] * np.exp(-2j * np.pi * j * delay / N_f))[None, :]                                  # shift theorem
    U, V = precompute_uv(h, S, df, 1.0)
    Q = precompute_q(h, d, S, df, 1.0, -16 / fs, 40)
    q = Q[0, 1]
    assert abs(q[16 + delay] - U[0, 1, 1]) < 1e-10 * abs(U[0, 1, 1])
    assert np.all(np.abs(q) <= abs(U[0, 1, 1]) * (1 + 1e-12)) and np.argmax(np.abs(q)) == 16 + delay


def test_band_limit_excludes_low_frequencies():
    rng, ht, h, S = _setup()
    N_f, df = h.shape[1], 0.25
    w = weights(S, N_f, df, f_low=10.0)
    f = np.abs(np.fft.fftfreq(N_f, d=1.0 / (N_f * df)))
    assert np.all(w[:, f <= 10.0] == 0.0) and np.all(w[:, f > 10.0] > 0.0)
    assert np.allclose(w[:, 1:], w[:, 1:][:, ::-1])                                              # even in f
