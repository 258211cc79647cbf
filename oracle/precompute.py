"""Oracle: the inner products Q, U, V of Eq. (6a-c) (TEST INFRASTRUCTURE ONLY).

PAPER.md:78-87:  <a|b>_k = 2 int_{|f| > f_low} df a~*(f) b~(f) / S_k(|f|)  (two-sided, complex);
Q_{k,lm}(t) = <h_lm(t)|d>_k = 2 int df/S_k(|f|) e^{2 pi i f t} h~*_lm(f) d~(f)   (6a)
U_{k,lm,l'm'} = <h_lm|h_l'm'>_k                                                   (6b)
V_{k,lm,l'm'} = <h_lm^*|h_l'm'>_k = 2 int df h~_lm(-f) h~_l'm'(f) / S_k(|f|)      (6c)
(the Fourier transform of h^* at f is the conjugate of h~ at -f).

Discretisation (reading G40): frequency bins in numpy FFT order,
f_j = j df for j <= N_f/2 and (j - N_f) df above; integrals -> sums times df; the time grid of Q is
t_n = t_Q0 + n / fs with fs = N_f df and t_Q0 fs an integer, so e^{2 pi i f_j t_n} =
exp(2 pi i j (n + n0) / N_f).  Plain sums, written as the definition.
"""
from __future__ import annotations

import numpy as np


def weights(S, N_f, df, f_low):
    """w_k[j] = 2 df / S_k(|f_j|) for |f_j| > f_low, else 0.  S [K, N_f/2 + 1] one-sided over |f|."""
    j = np.arange(N_f)
    jabs = np.where(j <= N_f // 2, j, N_f - j)
    f = jabs * df
    w = 2.0 * df / S[:, jabs]
    return np.where(f[None, :] > f_low, w, 0.0)


def precompute_uv(h, S, df, f_low):
    """h [M, N_f] complex (one intrinsic point) -> U, V [K, M, M]."""
    M, N_f = h.shape
    w = weights(S, N_f, df, f_low)
    neg = (N_f - np.arange(N_f)) % N_f
    K = S.shape[0]
    U = np.empty((K, M, M), dtype=np.complex128)
    V = np.empty((K, M, M), dtype=np.complex128)
    for k in range(K):
        for a in range(M):
            for b in range(M):
                U[k, a, b] = np.sum(w[k] * np.conj(h[a]) * h[b])
                V[k, a, b] = np.sum(w[k] * h[a][neg] * h[b])
    return U, V


def precompute_q(h, d, S, df, f_low, t_Q0, N_Q):
    """h [M, N_f], d [K, N_f] complex -> Q [K, M, N_Q] on t_n = t_Q0 + n / (N_f df)."""
    M, N_f = h.shape
    K = d.shape[0]
    w = weights(S, N_f, df, f_low)
    n0 = int(round(t_Q0 * N_f * df))
    assert abs(t_Q0 * N_f * df - n0) < 1e-9, "t_Q0 must sit on the sample grid"
    j = np.arange(N_f)
    Q = np.empty((K, M, N_Q), dtype=np.complex128)
    for n in range(N_Q):
        ph = np.exp(2j * np.pi * ((j * (n + n0)) % N_f) / N_f)
        for k in range(K):
            x = w[k] * d[k] * ph
            for a in range(M):
                Q[k, a, n] = np.sum(np.conj(h[a]) * x)
    return Q
