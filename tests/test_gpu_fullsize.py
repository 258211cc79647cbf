"""Full BASELINE.json sizes in the launch configuration bench.py times (-m gpu): the oracle cannot
evaluate 2^20..2^22 samples, so per-sample lnL is checked on a seeded subset of the batch the
device drew itself, and the reductions through properties that hold at any size."""
import numpy as np
import pytest

from synth import make_problem

pytestmark = pytest.mark.gpu


def _tol(ref):
    return 1e-9 * np.maximum(1.0, np.abs(ref))


def _strata(prob, z, rng, n_random=192):
    """Indices of the batch to compare with the oracle, chosen where the fused kernel's full-size paths are
    (DESIGN.md section 6): it orders the samples by the cell (16 stored bins per detector) of their first-bin
    indices n_k = floor((t_lo + tau_k - t_Q0) fs) and cuts the order into tiles at every multiple of 128 and at every
    cell change.  Taken: every sample of the first and of the last tile of the order, of the three smallest (ragged)
    tiles and of the tile with the widest spread of n_k; the samples with the extreme n_k of each detector; the
    samples nearest the edges of the prior box; and a random set."""
    from oracle import likelihood as lk
    N = z.shape[1]
    ang = lk.z_to_angles(np.clip(z, prob.lo[:, None], prob.hi[:, None]))         # GMM draws may leave the box (lnL = -inf there)
    _, _, tau = lk.antenna(prob.D, prob.pos, prob.gmst, ang[0], ang[1], ang[2])
    n = np.floor((prob.t_lo + tau - prob.t_Q0) * prob.fs).astype(np.int64)               # [K, N]
    inbox = np.all((z >= prob.lo[:, None]) & (z < prob.hi[:, None]), axis=0)
    cell = (n - n.min()) >> 4
    key = np.where(inbox, 0, 1 << 40)
    for k in range(prob.K):
        key = key * 4096 + np.where(inbox, cell[k], 0)
    order = np.argsort(key, kind="stable")
    ks = key[order]
    start = np.nonzero((np.arange(N) % 128 == 0) | (np.r_[True, ks[1:] != ks[:-1]]))[0]
    cnt = np.diff(np.r_[start, N])
    spread = np.array([(n[:, order[s:s + c]].max(axis=1) - n[:, order[s:s + c]].min(axis=1)).max() for s, c in zip(start, cnt)])
    tiles = {0, len(start) - 1, int(np.argmax(spread))} | set(np.argsort(cnt, kind="stable")[:3].tolist())
    pick = [order[start[t]:start[t] + cnt[t]] for t in tiles]
    for k in range(prob.K):
        pick.append(np.array([np.argmin(np.where(inbox, n[k], 1 << 30)), np.argmax(np.where(inbox, n[k], -1))]))
    y = (z - prob.lo[:, None]) / (prob.hi - prob.lo)[:, None]
    pick.append(np.argsort(np.minimum(y, 1 - y).min(axis=0))[:32])                          # nearest the box edges
    pick.append(rng.choice(N, size=n_random, replace=False))
    return np.unique(np.concatenate(pick))


@pytest.mark.parametrize("cfg,P,n_iter", [(2, 1, 3), (3, 1, 3), (4, 3, 1), (5, 1, 3)])
def test_full_batch_sampled_parity(cfg, P, n_iter):
    import torch
    from paper_2505_11655_b200 import Ile, Integrator, result_from_device
    from oracle.ile import IleProblem
    from oracle.reduce import reduce_lnw
    prob = make_problem(cfg, P=P)
    N = prob.N                                           # 2^20, 2^22, 2^18, 2^21
    ile = Ile(0)
    ile.load_problem(prob)
    g = Integrator.from_problem(ile, prob, max_batch=N)
    rng = np.random.default_rng(100 + cfg)
    for p in range(P):
        g.reset()
        op = IleProblem(prob, p)
        for it in range(n_iter):
            res = result_from_device(g.step(p, N, it))[0]
            z, lp, lnL, lnw = g.last_batch(N)
            idx = _strata(prob, z.cpu().numpy(), rng)
            assert len(idx) >= 300
            tidx = torch.from_numpy(idx).cuda()
            zs = z[:, tidx].cpu().numpy()
            got = lnL[tidx].cpu().numpy()
            ref = op.lnL_z(zs)
            fin = np.isfinite(ref)
            assert np.array_equal(fin, np.isfinite(got))
            assert np.all(np.abs(got[fin] - ref[fin]) <= _tol(ref[fin])), np.abs(got[fin] - ref[fin]).max()
            # ln w of the sampled entries, then the reduction of the device's own ln w in fp64 on the host
            lw = lnw.cpu().numpy()
            ref_w = np.where(fin, ref + op.ln_prior(zs) - lp[tidx].cpu().numpy(), -np.inf)
            assert np.all(np.abs(lw[idx][fin] - ref_w[fin]) <= 2e-9 * np.maximum(1.0, np.abs(ref_w[fin])))
            red = reduce_lnw(lw)                         # oracle reduction on the full device batch
            assert abs(res["ln_integral"] - red["ln_integral"]) <= 1e-8
            assert abs(res["n_eff"] - red["n_eff"]) <= 1e-7 * max(1.0, red["n_eff"])
            assert abs(res["n_ess"] - red["n_ess"]) <= 1e-7 * max(1.0, red["n_ess"])
            assert 1.0 - 1e-9 <= res["n_eff"] <= res["n_ess"] * (1 + 1e-12) <= N * (1 + 1e-12)
            assert res["n_samples"] == N and res["cum_n_samples"] == N * (it + 1)
            # the whole batch once more through the public entry point: the fused kernel's result does not depend on how
            # its warps interleave, so every one of the N values must come out bit for bit the same (a race would show)
            again = ile.lnL_z(p, z)
            assert torch.equal(again.view(torch.int64), lnL.view(torch.int64))
    if prob.kind == "AV":
        assert res["n_bins"] > 1 and 1 <= res["n_cells"] <= N and res["N_min"] >= 4096
        keys = g.get_state()["keys"]
        assert np.all(np.diff(keys.astype(np.int64)) > 0)          # sorted, unique
    if prob.kind == "PORTFOLIO":
        st = g.get_state()
        assert abs(st["W"][:3].sum() - 1.0) < 1e-12 and st["alloc"][:3].sum() == N


@pytest.mark.parametrize("N", [1, 31, 33, 64, 97])
def test_ragged_and_tiny_batches(N):
    import torch
    from paper_2505_11655_b200 import Ile
    from oracle import likelihood as lk
    from synth.workloads import uniform_box_samples
    prob = make_problem(2, P=1)
    ile = Ile(0)
    ile.load_problem(prob)
    z = uniform_box_samples(prob.lo, prob.hi, N, seed=N)
    ref = lk.lnL_z(prob.D, prob.pos, prob.gmst, prob.ell, prob.m, prob.Q[0], prob.U[0], prob.V[0], prob.D_ref, prob.fs,
                   prob.t_Q0, prob.t_lo, prob.dt, prob.N_t, z)
    got = ile.lnL_z(0, torch.from_numpy(z).cuda()).cpu().numpy()
    assert np.all(np.abs(got - ref) <= _tol(ref))


def test_all_samples_outside_the_box_and_empty_batch():
    import torch
    from paper_2505_11655_b200 import Ile
    prob = make_problem(1)
    ile = Ile(0)
    ile.load_problem(prob)
    z = np.tile(np.array([[7.0], [0.0], [1.0], [1.0], [0.0], [500.0]]), (1, 70))     # RA outside [0, 2 pi)
    got, lp = ile.lnL_z(0, torch.from_numpy(z).cuda(), want_prior=True)
    assert torch.all(got == -float("inf")) and torch.all(lp == -float("inf"))
    red = ile.reduce(got)
    assert red["ln_integral"] == -np.inf and red["n_eff"] == 0 and red["n_samples"] == 70
    empty = torch.empty((6, 0), dtype=torch.float64, device="cuda")
    assert ile.lnL_z(0, empty).numel() == 0


def test_delay_spread_beyond_one_round():
    """Unsorted samples all over the sky in one tile force the DMMA kernel's multi-round path (variant 3: no delay-cell sort)."""
    import torch
    from paper_2505_11655_b200 import Ile
    from oracle import likelihood as lk
    from synth.workloads import uniform_box_samples
    prob = make_problem(3, P=1)
    ile = Ile(0)
    ile.load_problem(prob)
    ile.set_lnL_variant(3)
    z = uniform_box_samples(prob.lo, prob.hi, 257, seed=4)
    ref = lk.lnL_z(prob.D, prob.pos, prob.gmst, prob.ell, prob.m, prob.Q[0], prob.U[0], prob.V[0], prob.D_ref, prob.fs,
                   prob.t_Q0, prob.t_lo, prob.dt, prob.N_t, z)
    got = ile.lnL_z(0, torch.from_numpy(z).cuda()).cpu().numpy()
    assert np.all(np.abs(got - ref) <= _tol(ref))
