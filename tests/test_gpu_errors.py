"""Error behaviour of the C ABI on the device box (-m gpu): every misuse returns a negative status
with a message and leaves the handle usable."""
import numpy as np
import pytest

from synth import make_problem

pytestmark = pytest.mark.gpu


def test_integrator_argument_and_state_errors():
    import torch
    from paper_2505_11655_b200 import Ile, IleError, Integrator
    prob = make_problem(1)
    ile = Ile(0)
    lo, hi = prob.lo, prob.hi
    for bad in (dict(n_bins=0), dict(eps=1.5), dict(beta=0.0)):
        with pytest.raises(IleError):
            Integrator(ile, "AC", 6, lo, hi, 1, 1000, **bad)
    with pytest.raises(IleError):
        Integrator(ile, "AV", 6, lo, hi, 1, 1000, P_thr=0.0)
    with pytest.raises(IleError):
        Integrator(ile, "GMM", 6, lo, hi, 1, 1000, n_gmm=17)
    with pytest.raises(IleError):
        Integrator(ile, "AC", 6, hi, lo, 1, 1000)                    # empty box
    with pytest.raises(IleError):
        Integrator(ile, "PORTFOLIO", 6, lo, hi, 1, 1000, members=())
    g = Integrator(ile, "PORTFOLIO", 3, lo[:3], hi[:3], 1, 1000, members=("AC", "AV"))
    z = torch.zeros((3, 100), dtype=torch.float64, device="cuda")
    w = torch.zeros(100, dtype=torch.float64, device="cuda")
    with pytest.raises(IleError):
        g.update(z, w, w)                                            # ESTATE: this batch was not drawn by the portfolio
    with pytest.raises(IleError):
        g.draw(1001, 0)                                              # beyond max_batch
    with pytest.raises(IleError):
        g.step(0, 100, 0)                                            # ESTATE: no problem loaded (and d = 3)
    st = g.get_state()
    st["members"][0]["n_bins"] = 7                                   # blob of another shape
    st["members"][0]["H"] = st["members"][0]["H"][:, :7]
    st["members"][0]["pi"] = st["members"][0]["pi"][:, :7]
    st["members"][0]["cdf"] = st["members"][0]["cdf"][:, :8]
    with pytest.raises(IleError):
        g.set_state(st)
    zz, lp = g.draw(1000, 0)                                         # the handle still works
    assert torch.isfinite(lp).all()


def test_lnL_dimension_and_point_checks():
    import torch
    from paper_2505_11655_b200 import Ile, IleError
    prob = make_problem(1)
    ile = Ile(0)
    ile.load_problem(prob)
    z5 = torch.zeros((5, 10), dtype=torch.float64, device="cuda")
    with pytest.raises(IleError):
        ile.lnL_z(0, z5)                                             # d = 5 without a distance table
    z6 = torch.zeros((6, 10), dtype=torch.float64, device="cuda")
    with pytest.raises(IleError):
        ile.lnL_z(3, z6)                                             # intrinsic point out of range
    with pytest.raises(IleError):
        ile.set_prior(5.0, 1.0)
    with pytest.raises(IleError):
        ile.set_lnL_variant(99)
    assert ile.lnL_z(0, z6).shape == (10,)
