"""Seeded synthetic frequency-domain inputs for the Q/U/V precompute.

Stand-ins for what RIFT feeds its inner products: mode spectra h~_lm(f) of
a chirp-like signal, detector data spectra d~_k(f) = signal + coloured noise, one-sided PSDs S_k(|f|).
Inputs only: no inner product is evaluated here.  numpy FFT bin order, fs = N_f * df.
"""
from __future__ import annotations

import numpy as np


def make_spectra(K, ell, m, N_f, fs, seed, P=1, snr_scale=5.0):
    """Returns h [P, M, N_f] complex128, d [K, N_f] complex128, S [K, N_f/2+1] float64, df."""
    rng = np.random.Generator(np.random.Philox(seed))
    M = len(ell)
    t = (np.arange(N_f) - N_f // 2) / fs
    df = fs / N_f
    h = np.empty((P, M, N_f), dtype=np.complex128)
    for p in range(P):
        f0 = 40.0 + 10.0 * rng.random()
        chirp = 60.0 + 40.0 * rng.random()
        env = np.exp(-0.5 * (t / (0.08 + 0.04 * rng.random())) ** 2)
        for a in range(M):
            phase = 2.0 * np.pi * float(m[a]) * (f0 * t + 0.5 * chirp * t * t) / 2.0 + rng.uniform(0, 2 * np.pi)
            amp = 0.4 ** (float(ell[a]) - 2.0) * 0.5 ** abs(float(ell[a]) - abs(float(m[a])))
            h[p, a] = np.fft.fft(np.fft.ifftshift(amp * env * np.exp(-1j * phase)))
    f = np.arange(N_f // 2 + 1) * df
    S = np.empty((K, N_f // 2 + 1))
    for k in range(K):
        S[k] = (1.0 + (30.0 / np.maximum(f, 5.0)) ** 4 + (f / (0.4 * fs)) ** 2) * (0.8 + 0.4 * rng.random())
    d = np.empty((K, N_f), dtype=np.complex128)
    for k in range(K):
        coef = (rng.standard_normal(M) + 1j * rng.standard_normal(M)) * snr_scale
        sig = np.real(np.fft.ifft((coef[:, None] * h[0]).sum(axis=0)))                 # a real strain built from point 0's modes
        noise = np.fft.irfft(np.sqrt(S[k] * fs / 2.0) * (rng.standard_normal(N_f // 2 + 1) + 1j * rng.standard_normal(N_f // 2 + 1)), n=N_f)
        d[k] = np.fft.fft(sig + noise)
    return h, d, S, df
