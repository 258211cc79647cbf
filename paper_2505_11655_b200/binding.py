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


class IntegratorOpts(C.Structure):
    _fields_ = [("kind", C.c_int32), ("d", C.c_int32), ("lo", C.c_double * ILE_MAX_D), ("hi", C.c_double * ILE_MAX_D),
                ("seed", C.c_uint64), ("max_batch", C.c_int64), ("n_bins", C.c_int32), ("pad0", C.c_int32), ("eps", C.c_double),
                ("beta", C.c_double), ("P_thr", C.c_double), ("N_min_star", C.c_int64), ("n_gmm", C.c_int32),
                ("n_members", C.c_int32), ("member_kind", C.c_int32 * ILE_MAX_MEMBERS)]


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

    def reduce(self, lnw):
        res = self.torch.zeros(C.sizeof(Result), dtype=self.torch.uint8, device=f"cuda:{self.device}")
        self._ck(self.lib.ile_reduce(self.ctx, C.c_int(lnw.numel()), _ptr(lnw), _ptr(res)))
        return result_from_device(res)[0]


def result_from_device(buf):
    """uint8 CUDA tensor holding ile_result structs -> numpy structured array (synchronises)."""
    return np.frombuffer(buf.cpu().numpy().tobytes(), dtype=RESULT_DTYPE)
