"""Oracle: adaptive Monte Carlo integrators (TEST INFRASTRUCTURE ONLY).

UNIFORM, AC (adaptive cartesian), AV (adaptive volume, PAPER.md:234-283,
Eq. 11-16), GMM (as a portfolio member) and PORTFOLIO.
The paper defers the algorithms' details to refs [23], [37-39], [64]; every step below
follows the readings G18-G26, G30, G35 of DESIGN.md section 3 in the order stated there.
**Parity unpinned w.r.t. RIFT's own constants** (eps, beta, P_thr, N_min*, EM schedule); the
integrators are pinned through closed-form integrals and invariants (pins P7, P9-P11).

All integrators share one interface:
    draw(N, g, i0=0)   -> z [d,N], ln_ps [N]   Philox counter = (i0+i, g), key = seed
    ln_pdf(z)          -> ln p_s(z) at arbitrary points (-inf outside the support)
    update(z, lnw, ln_ps=None)                 train on one batch (teacher-forced)
Bit-exact quantities (AC histograms, AV n_bins / N_min / key set, draws z) use only IEEE
+ - * / floor rint sqrt comparisons, no fused multiply-add and no libm transcendental.
"""
from __future__ import annotations

import math

import numpy as np

from .philox import uniforms

LOG2E = float.fromhex("0x1.71547652b82fep+0")
LN2 = float.fromhex("0x1.62e42fefa39efp-1")
FIX_ONE = 40            # fixed-point scale 2^40
T_CUT = -29.0           # exp(t) * 2^40 rounds to 0 below this


def qfix(t):
    """Fixed-point weight q = rint(sexp(t) * 2^40) as uint64 for t <= 0, where sexp is the
    *specified* exponential of DESIGN.md section 3 ("Determinism"): y = t*log2(e); n = rint(y);
    f = y - n; zz = f*ln2; p = Horner(sum_{k<=13} zz^k / k!) with separate multiply and add;
    result p * 2^n.  NaN and t < -29 give 0; t > 0 is clamped to 0 (cannot occur: t = ln w - max)."""
    t = np.asarray(t, dtype=np.float64)
    ok = ~np.isnan(t) & (t >= T_CUT)
    tt = np.where(ok, np.minimum(t, 0.0), 0.0)
    y = tt * LOG2E
    n = np.rint(y)
    f = y - n
    zz = f * LN2
    p = np.full(tt.shape, 1.0 / math.factorial(13))
    for k in range(12, -1, -1):
        p = p * zz
        p = p + 1.0 / math.factorial(k)
    q = np.rint(np.ldexp(p, (n + FIX_ONE).astype(np.int64)))
    return np.where(ok, q, 0.0).astype(np.uint64)


def bin_index(zc, lo, hi, n):
    """b = min(n-1, floor((z - lo) / (hi - lo) * n)), clipped at 0 (SURVEY 8(c) AC)."""
    t = (zc - lo) / (hi - lo) * float(n)
    b = np.floor(t)
    b = np.minimum(np.maximum(b, 0.0), float(n - 1))
    return b.astype(np.int64)


def in_box(z, lo, hi):
    ok = np.ones(z.shape[1], dtype=bool)
    for c in range(z.shape[0]):
        ok &= (z[c] >= lo[c]) & (z[c] < hi[c])
    return ok


def _below(hi, lo):
    return np.nextafter(hi, lo)


def box_volume(lo, hi):
    V0 = 1.0
    for c in range(len(lo)):
        V0 = V0 * (hi[c] - lo[c])
    return V0


def _finite_max(lnw):
    ok = np.isfinite(lnw)
    return (lnw[ok].max() if ok.any() else None), ok


# =============================================================================== UNIFORM
class Uniform:
    kind = "UNIFORM"

    def __init__(self, lo, hi, seed):
        self.lo = np.asarray(lo, dtype=np.float64)
        self.hi = np.asarray(hi, dtype=np.float64)
        self.d = len(lo)
        self.seed = seed

    def draw(self, N, g, i0=0):
        u = uniforms(self.seed, i0 + np.arange(N, dtype=np.uint64), g, 2 + self.d)
        z = np.empty((self.d, N))
        for c in range(self.d):
            zc = self.lo[c] + u[2 + c] * (self.hi[c] - self.lo[c])
            z[c] = np.minimum(zc, _below(self.hi[c], self.lo[c]))
        return z, self.ln_pdf(z)

    def ln_pdf(self, z):
        out = np.full(z.shape[1], -math.log(box_volume(self.lo, self.hi)))
        out[~in_box(z, self.lo, self.hi)] = -np.inf
        return out

    def update(self, z, lnw, ln_ps=None):
        return


# =============================================================================== AC
class AC:
    """Adaptive cartesian: product of per-dimension piecewise-constant pdfs (PAPER.md:107:
    "sampling prior p_s which has product form ... after a large block of evaluations, each
    one-dimensional marginal sampling prior can be updated")."""
    kind = "AC"

    def __init__(self, lo, hi, seed, n_bins=100, eps=0.1, beta=1.0):
        self.lo = np.asarray(lo, dtype=np.float64)
        self.hi = np.asarray(hi, dtype=np.float64)
        self.d = len(lo)
        self.seed = seed
        self.n_bins = int(n_bins)
        self.eps = float(eps)
        self.beta = float(beta)
        self.H = np.zeros((self.d, self.n_bins), dtype=np.uint64)
        self.pi = np.full((self.d, self.n_bins), 1.0 / self.n_bins)     # iteration 0: uniform
        self.cdf = np.zeros((self.d, self.n_bins + 1))
        self._scan()

    def _scan(self):
        for c in range(self.d):
            acc = 0.0
            self.cdf[c, 0] = 0.0
            for b in range(self.n_bins):
                acc = acc + self.pi[c, b]
                self.cdf[c, b + 1] = acc

    def draw(self, N, g, i0=0):
        u = uniforms(self.seed, i0 + np.arange(N, dtype=np.uint64), g, 2 + self.d)
        nb = self.n_bins
        z = np.empty((self.d, N))
        for c in range(self.d):
            uc = u[2 + c]
            b = np.searchsorted(self.cdf[c, :nb], uc, side="right") - 1   # last b: cdf[b] <= u
            r = (uc - self.cdf[c, b]) / self.pi[c, b]
            r = np.minimum(r, 1.0 - 2.0 ** -53)
            delta = (self.hi[c] - self.lo[c]) / float(nb)
            zc = self.lo[c] + (b.astype(np.float64) + r) * delta
            z[c] = np.minimum(zc, _below(self.hi[c], self.lo[c]))
        return z, self.ln_pdf(z)

    def ln_pdf(self, z):
        nb = self.n_bins
        out = np.zeros(z.shape[1])
        for c in range(self.d):
            b = bin_index(z[c], self.lo[c], self.hi[c], nb)
            pdf = self.pi[c, b] * float(nb) / (self.hi[c] - self.lo[c])
            out = out + np.log(pdf)
        out[~in_box(z, self.lo, self.hi)] = -np.inf
        return out

    def histogram(self, z, lnw):
        """H_c[b] = sum of fixed-point weights q_i of the in-box samples in bin b."""
        m, fin = _finite_max(lnw)
        nb = self.n_bins
        H = np.zeros((self.d, nb), dtype=np.uint64)
        if m is None:
            return H
        ok = fin & in_box(z, self.lo, self.hi)
        q = qfix(self.beta * (np.where(ok, lnw, -np.inf) - m))
        for c in range(self.d):
            b = bin_index(z[c], self.lo[c], self.hi[c], nb)
            np.add.at(H[c], b[ok], q[ok])
        return H

    def update(self, z, lnw, ln_ps=None):
        H = self.histogram(z, lnw)
        self.H = H
        nb = self.n_bins
        for c in range(self.d):
            tot = int(H[c].sum(dtype=np.uint64))
            if tot == 0:
                continue                                   # keep the old pi
            for b in range(nb):
                a = float(H[c, b]) / float(tot)
                self.pi[c, b] = (1.0 - self.eps) * a + self.eps / float(nb)
        self._scan()


# =============================================================================== AV
def av_n_max(d):
    """Largest n with n^d < 2^62 (exact integers)."""
    n = int(round(2.0 ** (62.0 / d))) + 2
    while n ** d >= 1 << 62:
        n -= 1
    return n


def pow_d(n, d):
    p = 1.0
    for _ in range(d):
        p = p * float(n)
    return p


class AV:
    """Adaptive volume: n_bins per dimension, a set of active cells, uniform
    sampling over their union; threshold for enclosed probability P_thr;
    V_{g+1} = V_g N_min / N_live, Delta V = V_{g+1} / sqrt(N_min); n_bins from
    Eq. (13).  Readings G19-G24, G35."""
    kind = "AV"

    def __init__(self, lo, hi, seed, P_thr=0.999, N_min_star=4096):
        self.lo = np.asarray(lo, dtype=np.float64)
        self.hi = np.asarray(hi, dtype=np.float64)
        self.d = len(lo)
        self.seed = seed
        self.P_thr = float(P_thr)
        self.N_min_star = int(N_min_star)
        self.n = 1                                           # iteration 0: one cell
        self.keys = np.zeros(1, dtype=np.uint64)
        self.n_max = av_n_max(self.d)
        self.N_min = 0
        self.L_thr = -math.inf

    @property
    def v(self):
        return float(len(self.keys)) / pow_d(self.n, self.d)

    def key_of(self, z, n):
        key = np.zeros(z.shape[1], dtype=np.uint64)
        mul = 1
        for c in range(self.d):
            key = key + bin_index(z[c], self.lo[c], self.hi[c], n).astype(np.uint64) * np.uint64(mul)
            mul *= n
        return key

    def draw(self, N, g, i0=0):
        u = uniforms(self.seed, i0 + np.arange(N, dtype=np.uint64), g, 2 + self.d)
        C = len(self.keys)
        cell = np.minimum(np.floor(u[0] * float(C)).astype(np.int64), C - 1)
        key = self.keys[cell]
        z = np.empty((self.d, N))
        n64 = np.uint64(self.n)
        for c in range(self.d):
            ic = key % n64
            key = key // n64
            y = (ic.astype(np.float64) + u[2 + c]) / float(self.n)
            zc = self.lo[c] + y * (self.hi[c] - self.lo[c])
            z[c] = np.minimum(zc, _below(self.hi[c], self.lo[c]))
        ln_ps = np.full(N, -math.log(self.v * box_volume(self.lo, self.hi)))
        return z, ln_ps

    def ln_pdf(self, z):
        key = self.key_of(z, self.n)
        pos = np.searchsorted(self.keys, key)
        pos = np.minimum(pos, len(self.keys) - 1)
        member = (self.keys[pos] == key) & in_box(z, self.lo, self.hi)
        return np.where(member, -math.log(self.v * box_volume(self.lo, self.hi)), -np.inf)

    def update(self, z, lnw, ln_ps=None):
        N = z.shape[1]
        lnw = np.asarray(lnw, dtype=np.float64)
        ok = np.isfinite(lnw) & in_box(z, self.lo, self.hi)
        if ln_ps is not None:
            ok &= np.isfinite(ln_ps)
        if not ok.any():
            return
        lnf = np.where(ok, lnw + (ln_ps if ln_ps is not None else 0.0), -np.inf)
        m = lnw[ok].max()
        q = qfix(np.where(ok, lnw, -np.inf) - m)
        total = int(q.sum(dtype=np.uint64))
        if total == 0:
            return
        order = np.lexsort((np.arange(N), -lnf))            # ln f descending, index ascending
        T = int(math.ceil(self.P_thr * float(total)))
        pre = np.cumsum(q[order], dtype=np.uint64)
        N_P = int(np.searchsorted(pre, np.uint64(T), side="left")) + 1
        n_valid = int(ok.sum())
        N_min = min(n_valid, max(N_P, self.N_min_star))
        kept = order[:N_min]
        self.N_min = N_min
        self.L_thr = float(lnf[kept[-1]])
        if ln_ps is None:
            v_new = self.v * float(N_min) / float(N)
        else:
            # portfolio member: importance estimate of the kept volume
            mn = ln_ps[ok].min()
            r = qfix(mn - np.where(ok, ln_ps, np.inf))
            R = int(r[kept].sum(dtype=np.uint64))
            v_new = (float(R) * 2.0 ** -FIX_ONE) * math.exp(-mn) / (float(N) * box_volume(self.lo, self.hi))
        dv = v_new / math.sqrt(float(N_min))
        self.v_new, self.dv = v_new, dv                      # kept for inspection (tests); not used by the method
        inv = 1.0 / dv
        lo_n, hi_n = 1, self.n_max                           # largest n with n^d <= 1/dv (Eq. 13)
        while lo_n < hi_n:
            mid = (lo_n + hi_n + 1) // 2
            if pow_d(mid, self.d) <= inv:
                lo_n = mid
            else:
                hi_n = mid - 1
        self.n = lo_n
        self.keys = np.unique(self.key_of(z[:, kept], self.n))


# =============================================================================== GMM
class GMM:
    """Gaussian-mixture sampling prior ("Gaussian mixture models (GMMs) to generate sampling priors
    for any user-specified subset of dimensions"), one weighted EM step per batch (G26).  `dims` = the modelled
    dimensions (default: all d); the others are sampled uniformly over the box and their density factor is
    1/(hi - lo) inside it, 0 outside (reading G43).  Not bit-exact (exp / log / sincos); compared to 1e-10 relative."""
    kind = "GMM"
    REG = 1.0e-6

    def __init__(self, lo, hi, seed, n_comp=8, dims=None):
        self.lo = np.asarray(lo, dtype=np.float64)
        self.hi = np.asarray(hi, dtype=np.float64)
        self.d = len(lo)
        self.dims = list(range(self.d)) if dims is None else sorted(int(c) for c in dims)
        self.other = [c for c in range(self.d) if c not in self.dims]
        self.gd = len(self.dims)
        self.seed = seed
        self.C = int(n_comp)
        u = uniforms(seed, np.arange(self.C, dtype=np.uint64), 0xFFFFFFFF, self.d)
        self.omega = np.full(self.C, 1.0 / self.C)
        self.mu = (self.lo[:, None] + u * (self.hi - self.lo)[:, None]).T[:, self.dims].copy()     # [C, gd]
        self.Sigma = np.stack([np.diag((0.5 * (self.hi - self.lo)[self.dims]) ** 2) for _ in range(self.C)])
        self._chol()

    def _chol(self):
        d = self.gd
        self.L = np.zeros((self.C, d, d))
        for c in range(self.C):
            S = self.Sigma[c]
            L = self.L[c]
            for i in range(d):
                for j in range(i + 1):
                    s = S[i, j]
                    for k in range(j):
                        s = s - L[i, k] * L[j, k]
                    L[i, j] = math.sqrt(s) if i == j else s / L[j, j]

    def _ln_comp(self, z):
        """ln N(z_dims; mu_c, Sigma_c) for every component: [C, N]."""
        d = self.gd
        zg = z[self.dims]
        N = z.shape[1]
        out = np.empty((self.C, N))
        for c in range(self.C):
            L = self.L[c]
            y = np.empty((d, N))
            for i in range(d):                                 # forward substitution L y = z - mu
                s = zg[i] - self.mu[c, i]
                for k in range(i):
                    s = s - L[i, k] * y[k]
                y[i] = s / L[i, i]
            quad = np.zeros(N)
            lndet = 0.0
            for i in range(d):
                quad = quad + y[i] * y[i]
                lndet = lndet + math.log(L[i, i])
            out[c] = -0.5 * quad - lndet - 0.5 * d * math.log(2.0 * math.pi)
        return out

    def ln_pdf(self, z):
        e = self._ln_comp(z) + np.log(self.omega)[:, None]
        mx = e.max(axis=0)
        out = mx + np.log(np.exp(e - mx).sum(axis=0))
        if self.other:                                         # uniform factor of the dimensions the mixture leaves alone
            lnu = 0.0
            ok = np.ones(z.shape[1], dtype=bool)
            for c in self.other:
                lnu = lnu + math.log(self.hi[c] - self.lo[c])
                ok &= (z[c] >= self.lo[c]) & (z[c] < self.hi[c])
            out = np.where(ok, out - lnu, -np.inf)
        return out

    def draw(self, N, g, i0=0):
        d = self.gd
        npair = (d + 1) // 2
        u = uniforms(self.seed, i0 + np.arange(N, dtype=np.uint64), g, 2 + 2 * npair + len(self.other))
        cw = np.cumsum(self.omega)
        comp = np.minimum(np.searchsorted(cw, u[0], side="right"), self.C - 1)
        nrm = np.empty((2 * npair, N))
        for p in range(npair):                                 # Box-Muller
            r = np.sqrt(-2.0 * np.log(1.0 - u[2 + 2 * p]))
            ang = 2.0 * math.pi * u[3 + 2 * p]
            nrm[2 * p] = r * np.cos(ang)
            nrm[2 * p + 1] = r * np.sin(ang)
        z = np.empty((self.d, N))
        for i in range(d):
            s = self.mu[comp, i]
            for k in range(i + 1):
                s = s + self.L[comp, i, k] * nrm[k]
            z[self.dims[i]] = s
        for q, c in enumerate(self.other):                     # the other dimensions: uniform over the box, as Uniform.draw
            zc = self.lo[c] + u[2 + 2 * npair + q] * (self.hi[c] - self.lo[c])
            z[c] = np.minimum(zc, _below(self.hi[c], self.lo[c]))
        return z, self.ln_pdf(z)

    def update(self, z, lnw, ln_ps=None):
        lnw = np.asarray(lnw, dtype=np.float64)
        ok = np.isfinite(lnw) & in_box(z, self.lo, self.hi)
        if not ok.any():
            return
        m = lnw[ok].max()
        wt = np.where(ok, np.exp(np.where(ok, lnw, -np.inf) - m), 0.0)
        e = self._ln_comp(z) + np.log(self.omega)[:, None]
        mx = e.max(axis=0)
        resp = np.exp(e - mx)
        resp = resp / resp.sum(axis=0)
        a = resp * wt[None, :]                                  # [C, N]
        s0 = a.sum(axis=1)
        if not (s0.sum() > 0.0):
            return
        new_omega = s0 / s0.sum()
        rng2 = ((self.hi - self.lo) ** 2)[self.dims]
        zg = z[self.dims]
        for c in range(self.C):
            if not (s0[c] > 1.0e-300):
                continue                                       # dead component: keep it
            dz = zg - self.mu[c][:, None]                      # shifted moments about the old mean
            s1 = (a[c][None, :] * dz).sum(axis=1)
            s2 = np.einsum("n,in,jn->ij", a[c], dz, dz)
            mean = s1 / s0[c]
            self.Sigma[c] = s2 / s0[c] - np.outer(mean, mean) + self.REG * np.diag(rng2)
            self.mu[c] = self.mu[c] + mean
        self.omega = new_omega
        self._chol()


# =============================================================================== PORTFOLIO
class Portfolio:
    """Mixture of member samplers (p_s = sum_a W_a p_s,a / sum_a W_a), weights
    adapted from the per-member n_ESS of the last batch, floor 0.05/N_s, members below 5 %
    frozen, every other member trained on all samples with the overall weights.
    Reading G25.

    Options of PAPER.md:297 (readings G41, G42): `first_iter[a]` = "the first iteration for which a given
    sampler is activated within the portfolio" (member 0 is always active): before it the member gets no
    samples, has no term in p_s, is not trained, and N_s counts the activated members only, so the portfolio
    behaves exactly as if the member were not there; when the activated set changes the weights restart
    uniform and no member is frozen on that batch.  `silent[a]`: the member "contribute[s] silently, only contributing training data for other
    samplers without directly influencing the integral": it draws N // N_active samples per batch (fixed
    share, its weight is not adapted), it has no term in p_s, its samples are left out of the estimate
    (they sit after the contributing members' samples: silent members are listed last) and every
    trained member, itself included, sees all samples with the weights L p / p_s."""
    kind = "PORTFOLIO"

    def __init__(self, members, first_iter=None, silent=None):
        self.members = list(members)
        self.Ns = len(self.members)
        self.first_iter = np.zeros(self.Ns, dtype=np.int64) if first_iter is None else np.asarray(first_iter, dtype=np.int64)
        self.silent = np.zeros(self.Ns, dtype=bool) if silent is None else np.asarray(silent, dtype=bool)
        if self.first_iter[0] != 0 or self.silent[0]:
            raise ValueError("member 0 is active from iteration 0 and contributes")
        if np.any(self.silent[:-1] & ~self.silent[1:]):
            raise ValueError("silent members are listed after the contributing ones")
        self.lo, self.hi, self.d = members[0].lo, members[0].hi, members[0].d
        self.alloc = None
        self.frozen = np.zeros(self.Ns, dtype=bool)
        self.active = np.zeros(self.Ns, dtype=bool)           # activated set of the last draw
        self.W = np.zeros(self.Ns)
        self._activate(0)
        self.restarted = False

    def _activate(self, g):
        """Activated set at iteration g; when it differs from the last draw's the weights restart uniform over the
        contributing activated members."""
        act = self.first_iter <= g
        if not np.array_equal(act, self.active):
            self.active = act
            con = act & ~self.silent
            self.W = np.where(con, 1.0 / float(con.sum()), 0.0)
            self.frozen = np.zeros(self.Ns, dtype=bool)
            self.restarted = True

    @property
    def contributing(self):
        return self.active & ~self.silent

    def allocation(self, N):
        con, sil = self.contributing, self.active & self.silent
        n_act = int(self.active.sum())
        each = N // n_act if sil.any() else 0
        Nc = N - int(sil.sum()) * each
        Na = np.where(con, np.floor(float(Nc) * self.W), 0.0).astype(np.int64)
        rem = Nc - int(Na.sum())
        idx = np.nonzero(con)[0]
        a = 0
        while rem > 0:
            Na[idx[a % len(idx)]] += 1
            rem -= 1
            a += 1
        Na[sil] = each
        self.n_contrib_samples = Nc
        return Na

    def ln_pdf(self, z):
        terms = [math.log(self.W[a]) + self.members[a].ln_pdf(z) for a in range(self.Ns) if self.contributing[a]]
        e = np.stack(terms)
        mx = e.max(axis=0)
        mxs = np.where(np.isfinite(mx), mx, 0.0)
        with np.errstate(divide="ignore"):
            return np.where(np.isfinite(mx), mxs + np.log(np.exp(e - mxs).sum(axis=0)), -np.inf)

    def draw(self, N, g, i0=0):
        self._activate(g)
        Na = self.allocation(N)
        self.alloc = Na
        z = np.empty((self.d, N))
        off = 0
        for a in range(self.Ns):
            if Na[a] > 0:
                za, _ = self.members[a].draw(int(Na[a]), g, i0=i0 + off)
                z[:, off:off + Na[a]] = za
            off += int(Na[a])
        return z, self.ln_pdf(z)

    def update(self, z, lnw, ln_ps):
        lnw = np.asarray(lnw, dtype=np.float64)
        con = self.contributing
        n_con = int(con.sum())
        ness = np.zeros(self.Ns)
        off = 0
        for a in range(self.Ns):
            seg = lnw[off:off + int(self.alloc[a])]
            off += int(self.alloc[a])
            if not con[a]:
                continue
            fin = np.isfinite(seg)
            if fin.any():
                mm = seg[fin].max()
                e = np.exp(seg[fin] - mm)
                ness[a] = e.sum() ** 2 / (e * e).sum()
        if ness.sum() > 0.0:
            raw = ness / ness.sum()
            # the batch after a restart was drawn with uniform weights (none below 5 %): nobody is frozen on it, so a
            # member that has just been activated is trained at least once
            self.frozen = con & (raw < 0.05) & (not self.restarted)
            W = np.where(con, np.maximum(raw, 0.05 / n_con), 0.0)
            self.W = W / W.sum()
        self.restarted = False
        # a one-member portfolio *is* that member (pin P11): it trains as the member would alone
        ln_ps_arg = ln_ps if self.Ns > 1 else None
        for a in range(self.Ns):
            if self.active[a] and not self.frozen[a]:
                self.members[a].update(z, lnw, ln_ps_arg)


def make_integrator(kind, lo, hi, seed, **o):
    """Factory mirroring ile_integrator_create's options."""
    if kind == "UNIFORM":
        return Uniform(lo, hi, seed)
    if kind == "AC":
        return AC(lo, hi, seed, o.get("n_bins", 100), o.get("eps", 0.1), o.get("beta", 1.0))
    if kind == "AV":
        return AV(lo, hi, seed, o.get("P_thr", 0.999), o.get("N_min_star", 4096))
    if kind == "GMM":
        return GMM(lo, hi, seed, o.get("n_gmm", 8), o.get("gmm_dims"))
    if kind == "PORTFOLIO":
        names = o.get("members", ["AC", "AV", "GMM"])
        per = o.get("member_opts") or [{}] * len(names)           # options unique to each sampler realization
        mem = [make_integrator(k, lo, hi, seed, **{**o, **per[a]}) for a, k in enumerate(names)]
        return Portfolio(mem, o.get("first_iter"), o.get("silent"))
    raise ValueError(kind)
