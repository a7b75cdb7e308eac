"""Pins of the sampling oracle (oracle/sampling.py) against things other than itself: the published known-answer
vectors of Philox4x32-10, closed forms (greedy limits, uniform logits, the two-token logistic), invariances, and the
distribution the draws must follow (chi-square against softmax probabilities computed here independently).  CPU only."""
from __future__ import annotations

import numpy as np
import pytest

from oracle import sampling as smp


def test_philox4x32_10_known_answers():
    """Known-answer vectors of the reference implementation (Random123 kat_vectors, philox4x32 with 10 rounds): zero
    counter and key, all-ones counter and key, and the digits-of-pi counter and key."""
    assert smp.philox4x32_10((0, 0, 0, 0), (0, 0)) == (0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8)
    f = 0xffffffff
    assert smp.philox4x32_10((f, f, f, f), (f, f)) == (0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd)
    assert smp.philox4x32_10((0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344), (0xa4093822, 0x299f31d0)) == \
        (0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1)


def test_uniform_is_open_interval_and_roughly_uniform():
    u = np.array([smp.uniform(7, s, r) for s in range(200) for r in range(10)])
    assert np.all(u > 0) and np.all(u < 1)
    hist = np.histogram(u, bins=10, range=(0, 1))[0]
    assert np.all(np.abs(hist - 200) < 5 * np.sqrt(200 * 0.9))
    assert smp.uniform(7, 3, 1) != smp.uniform(7, 3, 2) != smp.uniform(8, 3, 2)
    assert smp.uniform(7, 3, 1) == smp.uniform(7, 3, 1)


def test_greedy_limits_are_the_argmax():
    rng = np.random.default_rng(1)
    for _ in range(20):
        lg = rng.normal(0, 3, 50)
        a = int(np.argmax(lg))
        for u in (0.001, 0.37, 0.999):
            assert smp.sample(lg, 0.0, 0, 1.0, u) == a                 # T = 0
            assert smp.sample(lg, 1.0, 1, 1.0, u) == a                 # top-k = 1
            assert smp.sample(lg, 1.0, 0, 1e-9, u) == a                # top-p -> 0
            assert smp.sample(lg, 1e-4, 0, 1.0, u) == a                # T -> 0
    assert smp.sample(np.array([1.0, 5.0, 5.0, 2.0]), 0.0, 0, 1.0, 0.5) == 1   # lowest index among equals


def test_uniform_logits_without_filters_invert_to_floor_u_v():
    V = 37
    for u in (1e-6, 0.2, 0.4999, 0.5, 0.75, 1 - 1e-6):
        assert smp.sample(np.zeros(V), 1.0, 0, 1.0, u) == int(np.floor(u * V))   # no u * V on an integer here


def test_two_token_closed_form_and_shift_invariance():
    """token 0 iff u < sigmoid((l0 - l1) / T); adding a constant to every logit changes nothing."""
    for l0, l1, T in ((0.3, -1.2, 0.7), (2.0, 2.5, 1.3), (-4.0, 1.0, 2.0)):
        p0 = 1.0 / (1.0 + np.exp(-(l0 - l1) / T))
        for u in np.linspace(0.01, 0.99, 33):
            if abs(u - p0) < 1e-9:
                continue
            want = 0 if u < p0 else 1
            assert smp.sample(np.array([l0, l1]), T, 0, 1.0, u) == want
            assert smp.sample(np.array([l0, l1]) + 11.5, T, 0, 1.0, u) == want


def test_top_k_and_top_p_supports_by_brute_force():
    rng = np.random.default_rng(4)
    for _ in range(30):
        V = int(rng.integers(5, 40))
        lg = rng.normal(0, 2, V)
        T = float(rng.uniform(0.5, 2.0))
        k = int(rng.integers(1, V))
        kept, q = smp.support(lg, T, k, 1.0)
        order = np.argsort(-lg)
        assert set(np.flatnonzero(kept)) == set(order[:k])        # no ties in random normals
        assert abs(q.sum() - 1) < 1e-12 and np.all(q[~kept] == 0)
        # top-p by explicit enumeration of prefixes of the descending order
        p = float(rng.uniform(0.1, 0.95))
        kept2, q2 = smp.support(lg, T, 0, p)
        full = np.exp(lg / T - (lg / T).max())
        full /= full.sum()
        cum, n = 0.0, 0
        for i in np.argsort(-full):
            cum += full[i]
            n += 1
            if cum >= p:
                break
        assert set(np.flatnonzero(kept2)) == set(np.argsort(-full)[:n])
        assert abs(q2.sum() - 1) < 1e-12
        assert np.allclose(q2[kept2], full[kept2] / full[kept2].sum())


@pytest.mark.parametrize("top_k,top_p", [(0, 1.0), (5, 1.0), (0, 0.8), (6, 0.9)])
def test_draws_follow_the_filtered_softmax_chi_square(top_k, top_p):
    """20000 draws over successive steps: frequencies against probabilities computed here (not by the oracle)."""
    rng = np.random.default_rng(9)
    V, T, N = 12, 0.9, 20000
    lg = rng.normal(0, 1.5, V)
    full = np.exp(lg / T - (lg / T).max())
    full /= full.sum()
    keep = np.ones(V, bool)
    if top_k:
        keep[np.argsort(-full)[top_k:]] = False
    pr = np.where(keep, full, 0)
    pr /= pr.sum()
    if top_p < 1:
        o = np.argsort(-pr)
        n = int(np.searchsorted(np.cumsum(pr[o]), top_p)) + 1
        keep2 = np.zeros(V, bool)
        keep2[o[:n]] = True
        pr = np.where(keep2, pr, 0)
        pr /= pr.sum()
    toks = np.array([smp.sample_tokens(lg[None, :], [T], [top_k], [top_p], [1234], step)[0] for step in range(N)])
    cnt = np.bincount(toks, minlength=V)
    assert np.all(cnt[pr == 0] == 0)
    sel = pr > 0
    chi2 = float((((cnt[sel] - N * pr[sel]) ** 2) / (N * pr[sel])).sum())
    dof = int(sel.sum()) - 1
    assert chi2 < dof + 5 * np.sqrt(2 * dof) + 5, (chi2, dof)


def test_cdf_interval_contains_the_uniform_number_of_the_sampled_token():
    rng = np.random.default_rng(12)
    for _ in range(50):
        V = int(rng.integers(3, 60))
        lg = rng.normal(0, 2, V)
        T, k, p, u = float(rng.uniform(0.3, 2)), int(rng.integers(0, V)), float(rng.uniform(0.3, 1.0)), float(rng.uniform())
        t = smp.sample(lg, T, k, p, u)
        ok, lo, hi = smp.cdf_interval(lg, T, k, p, t)
        assert ok and lo - 1e-12 <= u <= hi + 1e-12
