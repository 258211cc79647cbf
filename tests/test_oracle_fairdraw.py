"""Pins of the fair-draw oracle: properties fixed by the definition of a
fair draw, none of them computed by the oracle itself."""
import numpy as np

from oracle.fairdraw import fair_draw


def test_systematic_counts_are_within_one_of_their_expectation():
    w = np.array([0.5, 0.25, 0.125, 0.0625, 0.0625])          # exact in fixed point
    lnw = np.log(w) + 300.0
    for M in (16, 1000, 99991):
        idx = fair_draw(lnw, M, seed=3, g=1)
        assert np.all(np.diff(idx) >= 0)                       # equally spaced positions: sorted output
        cnt = np.bincount(idx, minlength=5)
        assert cnt.sum() == M and np.all(np.abs(cnt - M * w) < 1.0 + 1e-9)


def test_equal_weights_draw_every_sample_once():
    idx = fair_draw(np.full(64, -7.0), 64, seed=9, g=0)
    assert np.array_equal(idx, np.arange(64))


def test_zero_weight_and_nonfinite_samples_are_never_drawn():
    lnw = np.array([0.0, -np.inf, np.nan, -1.0, -5000.0, np.inf])
    idx = fair_draw(lnw, 5000, seed=1, g=2, mode="independent")
    assert set(np.unique(idx)) <= {0, 3}                       # -5000 underflows the 2^-40 weight grid
    assert fair_draw(np.full(4, -np.inf), 10, 1, 0).tolist() == [-1] * 10
    frac = (idx == 0).mean()
    p0 = 1.0 / (1.0 + np.exp(-1.0))
    assert abs(frac - p0) < 4 * np.sqrt(p0 * (1 - p0) / 5000)


def test_independent_draws_follow_the_weights():
    rng = np.random.default_rng(0)
    lnw = rng.normal(0, 2, 200)
    p = np.exp(lnw - lnw.max())
    p /= p.sum()
    M = 200000
    cnt = np.bincount(fair_draw(lnw, M, seed=11, g=5, mode="independent"), minlength=200)
    keep = M * p > 20
    chi2 = (((cnt - M * p) ** 2) / (M * p))[keep].sum()
    dof = keep.sum() - 1
    assert abs(chi2 - dof) < 5 * np.sqrt(2 * dof)


def test_one_dominant_weight_takes_every_draw():
    lnw = np.array([-100.0, 5000.0, -3.0])
    assert np.all(fair_draw(lnw, 100, 2, 0) == 1)
