"""Thin ctypes binding over libile.so (include/ile.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch is used for device
memory and the stream.  There is no CPU fallback: loading fails loudly when the library is
missing, and ile_create fails when there is no CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libile.so")

ILE_MAX_D = 8
ILE_MAX_MEMBERS = 8
KINDS = {"UNIFORM": 0, "AC": 1, "AV": 2, "GMM": 3, "PORTFOLIO": 4}


class IleError(RuntimeError):
    pass


class Result(C.Structure):
    _fields_ = [("ln_integral", C.c_double), ("rel_variance", C.c_double), ("n_eff", C.c_double), ("n_ess", C.c_double),
                ("ln_w_max", C.c_double), ("S1", C.c_double), ("S2", C.c_double), ("n_samples", C.c_uint64),
                ("n_nonfinite", C.c_uint64), ("n_cells", C.c_uint64), ("n_bins", C.c_int64), ("N_min", C.c_uint64),
                ("ln_volume", C.c_double), ("L_thr", C.c_double), ("W", C.c_double * ILE_MAX_MEMBERS),
                ("cum_ln_integral", C.c_double), ("cum_rel_variance", C.c_double), ("cum_n_eff", C.c_double),
                ("cum_n_ess", C.c_double), ("cum_ln_w_max", C.c_double), ("cum_S1", C.c_double), ("cum_S2", C.c_double),
                ("cum_n_samples", C.c_uint64)]


RESULT_DTYPE = np.dtype([("ln_integral", "f8"), ("rel_variance", "f8"), ("n_eff", "f8"), ("n_ess", "f8"), ("ln_w_max", "f8"),
                         ("S1", "f8"), ("S2", "f8"), ("n_samples", "u8"), ("n_nonfinite", "u8"), ("n_cells", "u8"),
                         ("n_bins", "i8"), ("N_min", "u8"), ("ln_volume", "f8"), ("L_thr", "f8"), ("W", "f8", (ILE_MAX_MEMBERS,)),
                         ("cum_ln_integral", "f8"), ("cum_rel_variance", "f8"), ("cum_n_eff", "f8"), ("cum_n_ess", "f8"),
                         ("cum_ln_w_max", "f8"), ("cum_S1", "f8"), ("cum_S2", "f8"), ("cum_n_samples", "u8")])
assert RESULT_DTYPE.itemsize == C.sizeof(Result)


class Integrand(C.Structure):
    """ile_integrand (include/ile.h): built-in test integrands."""
    _fields_ = [("kind", C.c_int32), ("n_comp", C.c_int32), ("par", C.c_double * (4 * (ILE_MAX_D + 2)))]

    @classmethod
    def gaussian_mix(cls, centers, sigmas, ln_amps):
        f = cls()
        f.kind, f.n_comp = 0, len(sigmas)
        for c, (ctr, sg, la) in enumerate(zip(centers, sigmas, ln_amps)):
            for k, v in enumerate(ctr):
                f.par[c * (ILE_MAX_D + 2) + k] = float(v)
            f.par[c * (ILE_MAX_D + 2) + ILE_MAX_D] = float(sg)
            f.par[c * (ILE_MAX_D + 2) + ILE_MAX_D + 1] = float(la)
        return f

    @classmethod
    def rosenbrock(cls, a=1.0, b=100.0, T=1.0):
        f = cls()
        f.kind, f.n_comp = 1, 0
        f.par[0], f.par[1], f.par[2] = float(a), float(b), float(T)
        return f


class IntegratorOpts(C.Structure):
    _fields_ = [("kind", C.c_int32), ("d", C.c_int32), ("lo", C.c_double * ILE_MAX_D), ("hi", C.c_double * ILE_MAX_D),
                ("seed", C.c_uint64), ("max_batch", C.c_int64), ("n_bins", C.c_int32), ("pad0", C.c_int32), ("eps", C.c_double),
                ("beta", C.c_double), ("P_thr", C.c_double), ("N_min_star", C.c_int64), ("n_gmm", C.c_int32),
                ("n_members", C.c_int32), ("member_kind", C.c_int32 * ILE_MAX_MEMBERS),
                ("member_first_iter", C.c_int32 * ILE_MAX_MEMBERS), ("member_silent", C.c_int32 * ILE_MAX_MEMBERS),
                ("member_n_bins", C.c_int32 * ILE_MAX_MEMBERS), ("gmm_dims_mask", C.c_uint32), ("pad1", C.c_int32)]


_lib = None


def load_library():
    """dlopen libile.so (built by paper_2505_11655_b200.build); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise IleError(f"{LIB_PATH} is missing: run `python -m paper_2505_11655_b200.build` (no CPU fallback exists)")
        _lib = C.CDLL(LIB_PATH)
        _lib.ile_last_error.restype = C.c_char_p
        _lib.ile_version.restype = C.c_char_p
    return _lib


def _ptr(t):
    """Device pointer of a torch CUDA float64/int tensor (or None)."""
    if t is None:
        return C.c_void_p(0)
    assert t.is_cuda and t.is_contiguous(), "device pointers must be contiguous CUDA tensors"
    return C.c_void_p(t.data_ptr())


def _host(a, dtype=np.float64):
    a = np.ascontiguousarray(a, dtype=dtype)
    return a, a.ctypes.data_as(C.c_void_p)


def _complex_host(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a, a.ctypes.data_as(C.c_void_p)


class Ile:
    """Context handle: one per (device, stream).  Method names follow include/ile.h."""

    def __init__(self, device: int = 0, stream=None):
        import torch
        self.lib = load_library()
        self.torch = torch
        if stream is None:
            stream = torch.cuda.current_stream(device)
        self.stream = stream
        self.device = device
        self.ctx = C.c_void_p()
        rc = self.lib.ile_create(C.byref(self.ctx), C.c_int(device), C.c_void_p(stream.cuda_stream))
        if rc != 0:
            raise IleError(f"ile_create failed with {rc} (a CUDA device is required; there is no CPU fallback)")

    def _ck(self, rc):
        if rc != 0:
            raise IleError(f"ile error {rc}: {self.lib.ile_last_error(self.ctx).decode()}")

    def close(self):
        if self.ctx:
            self.lib.ile_destroy(self.ctx)
            self.ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- problem definition
    def set_network(self, D, pos_m, gmst=0.0):
        D, pD = _host(D)
        pos, pp = _host(pos_m)
        self._ck(self.lib.ile_set_network(self.ctx, C.c_int(D.shape[0]), pD, pp, C.c_double(gmst)))

    def set_modes(self, ell, m):
        ell, pe = _host(ell, np.int32)
        m, pm = _host(m, np.int32)
        self._ck(self.lib.ile_set_modes(self.ctx, C.c_int(len(ell)), pe, pm))

    def load_quv(self, Q, U, V, fs, t_Q0, D_ref):
        """Q [P,K,M,N_Q], U, V [P,K,M,M] complex128 host arrays."""
        Q, pQ = _complex_host(Q)
        U, pU = _complex_host(U)
        V, pV = _complex_host(V)
        self._ck(self.lib.ile_load_quv(self.ctx, C.c_int(Q.shape[0]), C.c_int(Q.shape[3]), C.c_double(fs), C.c_double(t_Q0),
                                       pQ, pU, pV, C.c_double(D_ref), C.c_int(0)))

    def precompute_quv(self, h, d, S, df, f_low, t_Q0, N_Q, D_ref):
        """ile_precompute_quv from CUDA tensors: h [P,M,N_f] complex128, d [K,N_f] complex128, S [K,N_f/2+1] float64."""
        P, M, N_f = h.shape
        self._ck(self.lib.ile_precompute_quv(self.ctx, C.c_int(P), C.c_int(N_f), C.c_double(df), C.c_double(f_low), _ptr(h), _ptr(d), _ptr(S),
                                             C.c_double(t_Q0), C.c_int(N_Q), C.c_double(D_ref)))

    def get_quv(self, p, K, M, N_Q):
        Q = np.empty((K, M, N_Q), dtype=np.complex128)
        U = np.empty((K, M, M), dtype=np.complex128)
        V = np.empty((K, M, M), dtype=np.complex128)
        self._ck(self.lib.ile_get_quv(self.ctx, C.c_int(p), Q.ctypes.data_as(C.c_void_p), U.ctypes.data_as(C.c_void_p), V.ctypes.data_as(C.c_void_p)))
        return Q, U, V

    def set_time_grid(self, t_lo, dt, N_t, interp=1):
        self._ck(self.lib.ile_set_time_grid(self.ctx, C.c_double(t_lo), C.c_double(dt), C.c_int(N_t), C.c_int(interp)))

    def set_prior(self, D_min, D_max):
        self._ck(self.lib.ile_set_prior(self.ctx, C.c_double(D_min), C.c_double(D_max)))

    def load_distance_table(self, table):
        if table is None:
            self._ck(self.lib.ile_load_distance_table(self.ctx, 0, 0, C.c_double(0), C.c_double(0), C.c_double(0), C.c_double(0), None))
            return
        T, pT = _host(table["lnT"])
        self._ck(self.lib.ile_load_distance_table(self.ctx, C.c_int(table["nA"]), C.c_int(table["nB"]), C.c_double(table["A_lo"]),
                                                  C.c_double(table["A_hi"]), C.c_double(table["B_lo"]), C.c_double(table["B_hi"]), pT))

    def load_problem(self, prob):
        """Convenience: all of the above from a synth.Problem-like object."""
        self.set_network(prob.D, prob.pos, prob.gmst)
        self.set_modes(prob.ell, prob.m)
        self.load_quv(prob.Q, prob.U, prob.V, prob.fs, prob.t_Q0, prob.D_ref)
        self.set_time_grid(prob.t_lo, prob.dt, prob.N_t, prob.interp)
        self.set_prior(prob.D_min, prob.D_max)
        self.load_distance_table(prob.table)

    def set_lnL_variant(self, variant):
        self._ck(self.lib.ile_set_lnL_variant(self.ctx, C.c_int(variant)))

    def sync(self):
        self._ck(self.lib.ile_sync(self.ctx))

    # ---- measurement helpers (include/ile.h "measurement")
    def kernel_launches(self) -> int:
        self.lib.ile_kernel_launches.restype = C.c_uint64
        return int(self.lib.ile_kernel_launches(self.ctx))

    def kernel_timing(self, on: bool):
        self._ck(self.lib.ile_kernel_timing(self.ctx, C.c_int(1 if on else 0)))

    def kernel_time(self):
        """(total device ms, launches) of the fused lnL kernel since kernel_timing(True)."""
        ms, n = C.c_double(0.0), C.c_uint64(0)
        self._ck(self.lib.ile_kernel_time(self.ctx, C.byref(ms), C.byref(n)))
        return ms.value, int(n.value)

    def fp64_peak(self, mode: int) -> float:
        tf = C.c_double(0.0)
        self._ck(self.lib.ile_fp64_peak(self.ctx, C.c_int(mode), C.byref(tf)))
        return tf.value

    def int8_mma_peak(self, mode: int = 0) -> float:
        t = C.c_double(0.0)
        self._ck(self.lib.ile_int8_mma_peak(self.ctx, C.c_int(mode), C.byref(t)))
        return t.value

    def load_quv_ptr(self, P, N_Q, fs, t_Q0, Q_ptr, U_ptr, V_ptr, D_ref):
        """ile_load_quv from raw host addresses (e.g. pinned torch tensors): no marshalling copies."""
        self._ck(self.lib.ile_load_quv(self.ctx, C.c_int(P), C.c_int(N_Q), C.c_double(fs), C.c_double(t_Q0), C.c_void_p(Q_ptr),
                                       C.c_void_p(U_ptr), C.c_void_p(V_ptr), C.c_double(D_ref), C.c_int(0)))

    # ---- direct evaluation (torch CUDA float64 tensors)
    def _empty(self, *shape):
        return self.torch.empty(shape, dtype=self.torch.float64, device=f"cuda:{self.device}")

    def antenna(self, ra, dec, psi, K):
        N = ra.numel()
        Fp, Fx, tau = self._empty(K, N), self._empty(K, N), self._empty(K, N)
        self._ck(self.lib.ile_antenna(self.ctx, C.c_int(N), _ptr(ra), _ptr(dec), _ptr(psi), _ptr(Fp), _ptr(Fx), _ptr(tau)))
        return Fp, Fx, tau

    def ylm(self, incl, phi, M):
        N = incl.numel()
        Y = self._empty(M, N, 2)
        self._ck(self.lib.ile_ylm(self.ctx, C.c_int(N), _ptr(incl), _ptr(phi), _ptr(Y)))
        return Y

    def lnL(self, p, ra, dec, psi, phi_ref, incl, dist=None, N_t_dump=0):
        N = ra.numel()
        out = self._empty(N)
        dump = self._empty(N, N_t_dump) if N_t_dump else None
        self._ck(self.lib.ile_lnL(self.ctx, C.c_int(p), C.c_int(N), _ptr(ra), _ptr(dec), _ptr(psi), _ptr(phi_ref), _ptr(incl),
                                  _ptr(dist), _ptr(out), _ptr(dump)))
        return (out, dump) if N_t_dump else out

    def lnL_z(self, p, z, want_prior=False, out=None):
        d, N = z.shape
        out = self._empty(N) if out is None else out
        lp = self._empty(N) if want_prior else None
        self._ck(self.lib.ile_lnL_z(self.ctx, C.c_int(p), C.c_int(N), C.c_int(d), _ptr(z), _ptr(out), _ptr(lp)))
        return (out, lp) if want_prior else out

    def fair_draw(self, lnw, M, seed, it, mode="systematic"):
        """ile_fair_draw: int64 CUDA tensor [M] of sample indices drawn with probability w / sum w."""
        idx = self.torch.empty(M, dtype=self.torch.int64, device=f"cuda:{self.device}")
        self._ck(self.lib.ile_fair_draw(self.ctx, C.c_int(lnw.numel()), _ptr(lnw), C.c_int(M), C.c_uint64(int(seed) & 0xFFFFFFFFFFFFFFFF),
                                        C.c_uint64(it), C.c_int(0 if mode == "systematic" else 1), _ptr(idx)))
        return idx

    def reduce(self, lnw):
        res = self.torch.zeros(C.sizeof(Result), dtype=self.torch.uint8, device=f"cuda:{self.device}")
        self._ck(self.lib.ile_reduce(self.ctx, C.c_int(lnw.numel()), _ptr(lnw), _ptr(res)))
        return result_from_device(res)[0]

    def reduce_noalloc(self, lnw, out=None):
        """ile_reduce_noalloc: the same reduction with its scratch in a static device array (no allocation in the library;
        pass `out` to allocate nothing here either).  Returns the decoded result (synchronises)."""
        res = self.torch.zeros(C.sizeof(Result), dtype=self.torch.uint8, device=f"cuda:{self.device}") if out is None else out
        self._ck(self.lib.ile_reduce_noalloc(self.ctx, C.c_int(lnw.numel()), _ptr(lnw), _ptr(res)))
        return result_from_device(res)[0]


def result_from_device(buf):
    """uint8 CUDA tensor holding ile_result structs -> numpy structured array (synchronises)."""
    return np.frombuffer(buf.cpu().numpy().tobytes(), dtype=RESULT_DTYPE)


def parse_state(blob: bytes):
    """Decode the blob of ile_integrator_get_state (layout in include/ile.h) into a dict."""
    buf = memoryview(blob)
    pos = 0

    def i64(n=1):
        nonlocal pos
        a = np.frombuffer(buf, dtype="<i8", count=n, offset=pos)
        pos += 8 * n
        return a

    def arr(dtype, *shape):
        nonlocal pos
        n = int(np.prod(shape)) if shape else 1
        a = np.frombuffer(buf, dtype=dtype, count=n, offset=pos).reshape(shape).copy()
        pos += a.itemsize * n
        return a

    def member():
        kind, d = (int(v) for v in i64(2))
        out = dict(kind=kind, d=d)
        if kind == KINDS["AC"]:
            nb = int(i64()[0])
            out.update(n_bins=nb, H=arr("<u8", d, nb), pi=arr("<f8", d, nb), cdf=arr("<f8", d, nb + 1))
        elif kind == KINDS["AV"]:
            n, Cn, N_min = (int(v) for v in i64(3))
            out.update(n=n, C=Cn, N_min=N_min, L_thr=float(arr("<f8", 1)[0]), keys=arr("<u8", Cn))
        elif kind == KINDS["GMM"]:
            Cn, gd = int(i64()[0]), int(i64()[0])
            out.update(n_comp=Cn, gd=gd, omega=arr("<f8", Cn), mu=arr("<f8", Cn, gd), Sigma=arr("<f8", Cn, gd, gd), L=arr("<f8", Cn, gd, gd))
        return out

    kind, d = (int(v) for v in np.frombuffer(buf, dtype="<i8", count=2, offset=0))
    if kind != KINDS["PORTFOLIO"]:
        return member()
    pos = 16
    Ns = int(i64()[0])
    out = dict(kind=kind, d=d, n_members=Ns, W=arr("<f8", ILE_MAX_MEMBERS), frozen=arr("<i8", ILE_MAX_MEMBERS),
               alloc=arr("<i8", ILE_MAX_MEMBERS), active=arr("<i8", ILE_MAX_MEMBERS), members=[])
    for _ in range(Ns):
        i64()
        out["members"].append(member())
    return out


def pack_state(st: dict) -> bytes:
    """Inverse of parse_state (for ile_integrator_set_state)."""
    def member(m):
        parts = [np.array([m["kind"], m["d"]], dtype="<i8").tobytes()]
        if m["kind"] == KINDS["AC"]:
            parts += [np.array([m["n_bins"]], dtype="<i8").tobytes(), np.ascontiguousarray(m["H"], dtype="<u8").tobytes(),
                      np.ascontiguousarray(m["pi"], dtype="<f8").tobytes(), np.ascontiguousarray(m["cdf"], dtype="<f8").tobytes()]
        elif m["kind"] == KINDS["AV"]:
            keys = np.ascontiguousarray(m["keys"], dtype="<u8")
            parts += [np.array([m["n"], len(keys), m.get("N_min", 0)], dtype="<i8").tobytes(),
                      np.array([m.get("L_thr", -np.inf)], dtype="<f8").tobytes(), keys.tobytes()]
        elif m["kind"] == KINDS["GMM"]:
            parts += [np.array([len(m["omega"]), np.asarray(m["mu"]).shape[1]], dtype="<i8").tobytes()]
            parts += [np.ascontiguousarray(m[k], dtype="<f8").tobytes() for k in ("omega", "mu", "Sigma", "L")]
        return b"".join(parts)

    if st["kind"] != KINDS["PORTFOLIO"]:
        return member(st)
    parts = [np.array([st["kind"], st["d"], st["n_members"]], dtype="<i8").tobytes(),
             np.ascontiguousarray(st["W"], dtype="<f8").tobytes(), np.ascontiguousarray(st["frozen"], dtype="<i8").tobytes(),
             np.ascontiguousarray(st["alloc"], dtype="<i8").tobytes(),
             np.ascontiguousarray(st.get("active", np.ones(ILE_MAX_MEMBERS)), dtype="<i8").tobytes()]
    for m in st["members"]:
        b = member(m)
        parts += [np.array([len(b)], dtype="<i8").tobytes(), b]
    return b"".join(parts)


class _DevView:
    """__cuda_array_interface__ holder for a library-owned float64 device buffer."""

    def __init__(self, ptr, shape):
        self.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": "<f8", "data": (int(ptr), False), "version": 2}


class Integrator:
    """Handle over ile_integrator_* (include/ile.h).  Buffers are torch CUDA float64 tensors."""

    def __init__(self, ile: Ile, kind: str, d: int, lo, hi, seed: int, max_batch: int, n_bins=100, eps=0.1, beta=1.0,
                 P_thr=0.999, N_min_star=4096, n_gmm=8, members=("AC", "AV", "GMM"), first_iter=None, silent=None, member_opts=None,
                 gmm_dims=None):
        self.ile = ile
        self.lib = ile.lib
        self.torch = ile.torch
        self.kind, self.d = kind, int(d)
        o = IntegratorOpts()
        self.ile._ck(self.lib.ile_integrator_opts_default(C.byref(o), C.c_int(KINDS[kind]), C.c_int(d)))
        for c in range(d):
            o.lo[c], o.hi[c] = float(lo[c]), float(hi[c])
        o.seed, o.max_batch = int(seed) & 0xFFFFFFFFFFFFFFFF, int(max_batch)
        o.n_bins, o.eps, o.beta, o.P_thr, o.N_min_star, o.n_gmm = int(n_bins), float(eps), float(beta), float(P_thr), int(N_min_star), int(n_gmm)
        if kind == "PORTFOLIO":
            o.n_members = len(members)
            for a, k in enumerate(members):
                o.member_kind[a] = KINDS[k]
                o.member_first_iter[a] = int(first_iter[a]) if first_iter is not None else 0
                o.member_silent[a] = int(bool(silent[a])) if silent is not None else 0
                o.member_n_bins[a] = int((member_opts[a] or {}).get("n_bins", 0)) if member_opts is not None else 0
        if gmm_dims is not None:
            o.gmm_dims_mask = sum(1 << int(c) for c in gmm_dims)
        self.opts = o
        self.h = C.c_void_p()
        self.ile._ck(self.lib.ile_integrator_create(ile.ctx, C.byref(o), C.byref(self.h)))

    @classmethod
    def from_problem(cls, ile: Ile, prob, max_batch=None, kind=None):
        o = {k: v for k, v in prob.opts.items() if k != "seed"}
        return cls(ile, kind or prob.kind, prob.d, prob.lo, prob.hi, prob.opts["seed"], max_batch or prob.N, **o)

    def close(self):
        if self.h:
            self.lib.ile_integrator_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, rc):
        self.ile._ck(rc)

    def reset(self):
        self._ck(self.lib.ile_integrator_reset(self.h))

    def draw(self, N, it, z=None, ln_ps=None):
        z = self.ile._empty(self.d, N) if z is None else z
        ln_ps = self.ile._empty(N) if ln_ps is None else ln_ps
        self._ck(self.lib.ile_integrator_draw(self.h, C.c_int(N), C.c_uint64(it), _ptr(z), _ptr(ln_ps)))
        return z, ln_ps

    def ln_pdf(self, z):
        out = self.ile._empty(z.shape[1])
        self._ck(self.lib.ile_integrator_ln_pdf(self.h, C.c_int(z.shape[1]), _ptr(z), _ptr(out)))
        return out

    def update(self, z, lnw, ln_ps=None):
        self._ck(self.lib.ile_integrator_update(self.h, C.c_int(z.shape[1]), _ptr(z), _ptr(lnw), _ptr(ln_ps)))

    def _results(self, n):
        return self.torch.zeros(n * C.sizeof(Result), dtype=self.torch.uint8, device=f"cuda:{self.ile.device}")

    def step(self, p, N, it, out=None):
        """One iteration; returns the device result buffer (decode with result_from_device)."""
        out = self._results(1) if out is None else out
        self._ck(self.lib.ile_integrator_step(self.h, C.c_int(p), C.c_int(N), C.c_uint64(it), _ptr(out)))
        return out

    def step_integrand(self, f, N, it, out=None):
        """One iteration on a built-in test integrand (Integrand.gaussian_mix / .rosenbrock)."""
        out = self._results(1) if out is None else out
        self._ck(self.lib.ile_integrator_step_integrand(self.h, C.byref(f), C.c_int(N), C.c_uint64(it), _ptr(out)))
        return out

    def run(self, p_first, p_count, n_iter, N, out=None):
        out = self._results(p_count * n_iter) if out is None else out
        self._ck(self.lib.ile_integrator_run(self.h, C.c_int(p_first), C.c_int(p_count), C.c_int(n_iter), C.c_int(N), _ptr(out)))
        return out

    def last_batch(self, N):
        """Zero-copy torch views of the last batch's z [d,N], ln_ps, lnL, lnw (library-owned memory,
        valid until the next draw/step)."""
        ptrs = [C.c_void_p() for _ in range(4)]
        self._ck(self.lib.ile_integrator_last_batch(self.h, *[C.byref(p) for p in ptrs]))
        out = []
        for p, shape in zip(ptrs, ((self.d, N), (N,), (N,), (N,))):
            out.append(self.torch.as_tensor(_DevView(p.value, shape), device=f"cuda:{self.ile.device}"))
        return out

    def get_state(self):
        n = C.c_size_t(0)
        self._ck(self.lib.ile_integrator_get_state(self.h, None, C.byref(n)))
        buf = (C.c_ubyte * n.value)()
        self._ck(self.lib.ile_integrator_get_state(self.h, buf, C.byref(n)))
        return parse_state(bytes(buf)[:n.value])

    def set_state(self, st):
        blob = pack_state(st)
        self._ck(self.lib.ile_integrator_set_state(self.h, blob, C.c_size_t(len(blob))))
