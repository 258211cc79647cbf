"""Seeded synthetic frequency-domain inputs for the Q/U/V precompute.

Stand-ins for what RIFT feeds its inner products: mode spectra h~_lm(f) of
a chirp-like signal, detector data spectra d~_k(f) = signal + coloured noise, one-sided PSDs S_k(|f|).
Inputs only: no inner product is evaluated here.  numpy FFT bin order, fs = N_f * df.
"""
from __future__ import annotations

import numpy as np


def make_spectra(K, ell, m, N_f, fs, seed, P=1, amp=30.0):
    """Returns h [P, M, N_f] complex128, d [K, N_f] complex128, S [K, N_f/2+1] float64, df.

    Continuous-transform convention (spectrum = dt x DFT), so that <h|h> is of order amp^2 / 3 and a
    noise bin contributes order one to <n|n>: signal-to-noise ratios of tens, as in the paper's events.
    """
    rng = np.random.Generator(np.random.Philox(seed))
    M = len(ell)
    dt = 1.0 / fs
    t = (np.arange(N_f) - N_f // 2) * dt
    df = fs / N_f
    T = N_f * dt
    h = np.empty((P, M, N_f), dtype=np.complex128)
    h_t0 = None
    for p in range(P):
        f0 = 40.0 + 10.0 * rng.random()
        chirp = 60.0 + 40.0 * rng.random()
        env = np.exp(-0.5 * (t / (0.08 + 0.04 * rng.random())) ** 2)
        h_t = np.empty((M, N_f), dtype=np.complex128)
        for a in range(M):
            phase = 2.0 * np.pi * float(m[a]) * (f0 * t + 0.5 * chirp * t * t) / 2.0 + rng.uniform(0, 2 * np.pi)
            rel = 0.4 ** (float(ell[a]) - 2.0) * 0.5 ** abs(float(ell[a]) - abs(float(m[a])))
            h_t[a] = amp * rel * env * np.exp(-1j * phase)
            h[p, a] = dt * np.fft.fft(np.fft.ifftshift(h_t[a]))
        if p == 0:
            h_t0 = h_t
    f = np.arange(N_f // 2 + 1) * df
    S = np.empty((K, N_f // 2 + 1))
    for k in range(K):
        S[k] = (1.0 + (30.0 / np.maximum(f, 5.0)) ** 4 + (f / (0.4 * fs)) ** 2) * (0.8 + 0.4 * rng.random())
    d = np.empty((K, N_f), dtype=np.complex128)
    for k in range(K):
        coef = 0.3 * (rng.standard_normal(M) + 1j * rng.standard_normal(M))
        sig_t = np.real((coef[:, None] * h_t0).sum(axis=0))                            # a real strain built from point 0's modes
        half = np.sqrt(S[k] * T / 4.0) * (rng.standard_normal(N_f // 2 + 1) + 1j * rng.standard_normal(N_f // 2 + 1))
        noise_t = np.fft.irfft(half, n=N_f)                                           # real noise series (in spectrum units)
        d[k] = dt * np.fft.fft(np.fft.ifftshift(sig_t)) + np.fft.fft(noise_t)
    return h, d, S, df
