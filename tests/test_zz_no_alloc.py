"""ile_reduce_noalloc (include/ile.h): the weight reduction of step 7 with its scratch in a static device array, for callers
that must not allocate.  Checked against the existing path, ile_reduce, on the same inputs, on two calls in a row (the
array keeps the last call's contents).  Collected last on purpose (file name): a failure here hides nothing behind it."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

FIELDS = ("ln_integral", "rel_variance", "n_eff", "n_ess", "ln_w_max", "S1", "S2", "cum_ln_integral", "cum_rel_variance", "cum_n_eff")


def _same(got, ref):
    # the tolerances of tests/test_gpu_lnl.py::test_reduce (the two paths run the same kernels on the same grid: in fact equal)
    assert abs(got["ln_integral"] - ref["ln_integral"]) <= 1e-8
    for k in FIELDS:
        assert abs(got[k] - ref[k]) <= 1e-9 * max(1.0, abs(ref[k])), k
    for k in ("n_samples", "n_nonfinite", "cum_n_samples"):
        assert got[k] == ref[k], k


def test_reduce_noalloc_matches_reduce_on_consecutive_calls():
    import torch
    from paper_2505_11655_b200 import Ile, IleError
    from paper_2505_11655_b200.binding import Result
    ile = Ile(0)
    rng = np.random.default_rng(11)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    out = torch.zeros(C.sizeof(Result), dtype=torch.uint8, device="cuda:0")
    # a long batch first (every partial of the grid written), then short ones (fewer blocks: what the long call left in the
    # array must not be read), the peaked weights of a loud source, and a batch with nothing finite
    batches = []
    for N in (3_000_017, 1, 31, 100_003, 2048 * 40):
        lnw = rng.normal(0, 30, N) + 4000.0
        if N > 50:
            lnw[5], lnw[6], lnw[7] = -np.inf, np.nan, np.inf
        batches.append(lnw)
    batches.append(np.full(10, -np.inf))
    for rnd in range(2):                                   # two passes over the list: every call follows another one
        for lnw in batches:
            d = dev(lnw)
            ref = ile.reduce(d)                            # existing path: partials in the context's scratch
            got = ile.reduce_noalloc(d, out)
            again = ile.reduce_noalloc(d, out)             # the same call twice in a row
            if np.isfinite(ref["ln_integral"]):
                _same(got, ref)
                _same(again, ref)
            else:
                for r in (got, again):
                    assert r["ln_integral"] == -np.inf and r["n_eff"] == 0 and r["n_samples"] == lnw.size
    # beyond the stated maximum: a clear error, nothing launched
    big = torch.zeros((1 << 24) + 1, dtype=torch.float64, device="cuda:0")
    before = ile.kernel_launches()
    with pytest.raises(IleError, match="exceeds the maximum"):
        ile.reduce_noalloc(big, out)
    assert ile.kernel_launches() == before
    at_max = ile.reduce_noalloc(big[: 1 << 24], out)       # the maximum itself is served
    assert at_max["n_samples"] == 1 << 24 and abs(at_max["ln_integral"]) <= 1e-12


def test_reduce_noalloc_allocates_nothing():
    """Device memory in use does not move across calls (cudaMemGetInfo before and after, buffers made beforehand)."""
    import torch
    from paper_2505_11655_b200 import Ile
    from paper_2505_11655_b200.binding import Result
    ile = Ile(0)
    lnw = torch.randn(1 << 20, dtype=torch.float64, device="cuda:0")
    out = torch.zeros(C.sizeof(Result), dtype=torch.uint8, device="cuda:0")
    ile.reduce_noalloc(lnw, out)                           # first call on this device: symbol address looked up
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(5):
        ile.lib.ile_reduce_noalloc(ile.ctx, C.c_int(lnw.numel()), C.c_void_p(lnw.data_ptr()), C.c_void_p(out.data_ptr()))
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
