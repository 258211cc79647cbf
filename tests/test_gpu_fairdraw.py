"""GPU parity of ile_fair_draw against the oracle (-m gpu): indices are integers, so bit-exact."""
import numpy as np
import pytest

from synth import make_problem

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("mode", ["systematic", "independent"])
@pytest.mark.parametrize("N,M", [(1, 7), (2049, 300), (100003, 50000), (1 << 21, 4096)])
def test_fair_draw_bit_exact(mode, N, M):
    import torch
    from paper_2505_11655_b200 import Ile
    from oracle.fairdraw import fair_draw
    ile = Ile(0)
    rng = np.random.default_rng(N + M)
    lnw = rng.normal(0.0, 6.0, N) + 4000.0
    if N > 10:
        lnw[3] = np.nan
        lnw[4] = -np.inf
        lnw[5] = np.inf
    got = ile.fair_draw(torch.from_numpy(lnw).cuda(), M, seed=0xABCDEF12345, it=3, mode=mode).cpu().numpy()
    ref = fair_draw(lnw, M, 0xABCDEF12345, 3, mode)
    assert np.array_equal(got, ref)
    if mode == "systematic":
        assert np.all(np.diff(got) >= 0)


def test_fair_draw_degenerate_weights():
    import torch
    from paper_2505_11655_b200 import Ile
    ile = Ile(0)
    none = ile.fair_draw(torch.full((500,), -float("inf"), dtype=torch.float64, device="cuda"), 16, 1, 0)
    assert torch.all(none == -1)
    lnw = torch.full((5000,), -800.0, dtype=torch.float64, device="cuda")
    lnw[4321] = 12.0
    assert torch.all(ile.fair_draw(lnw, 100, 7, 1) == 4321)


def test_fair_extrinsic_samples_from_an_integrator_batch():
    """extrinsic samples drawn fairly from the weighted ILE samples of one batch."""
    import torch
    from paper_2505_11655_b200 import Ile, Integrator, result_from_device
    from oracle.fairdraw import fair_draw
    prob = make_problem(1)
    ile = Ile(0)
    ile.load_problem(prob)
    g = Integrator.from_problem(ile, prob, max_batch=prob.N)
    res = result_from_device(g.step(0, prob.N, 0))[0]
    z, lp, lnL, lnw = g.last_batch(prob.N)
    M = max(4, int(4 * res["n_eff"]))
    idx = ile.fair_draw(lnw, M, seed=5, it=0)
    assert np.array_equal(idx.cpu().numpy(), fair_draw(lnw.cpu().numpy(), M, 5, 0))
    theta = z[:, idx]                                                   # the fair extrinsic samples
    assert theta.shape == (6, M) and torch.isfinite(lnL[idx]).all()
    # drawn samples are the heavy ones: their mean ln w exceeds the batch's by far
    assert lnw[idx].mean() > lnw[torch.isfinite(lnw)].mean() + 3.0
