"""Sampling-mode DECS in the oracle (Alg. 2 lines 10-15, App. C.1): pins that do not re-use the
oracle's own formula - the Gumbel-Max sample frequencies against softmax(l/tau) computed directly, the moments
of the noise rows against the Gumbel(0,1) closed forms, independence across positions, and losslessness of the
sampled DEX stream against sampled AR decoding for every exploration set."""
import numpy as np
import pytest

from oracle import gumbel


def test_uniforms_are_uniform_and_rows_differ():
    u = np.concatenate([gumbel.uniform_row(7, 0, p, 4096) for p in range(64)])
    assert 0.0 < u.min() and u.max() < 1.0
    hist, _ = np.histogram(u, bins=32, range=(0.0, 1.0))
    exp = len(u) / 32
    assert ((hist - exp) ** 2 / exp).sum() < 80.0                       # chi-square, 31 dof (p ~ 1e-6 at 80)
    a, b = gumbel.uniform_row(7, 0, 5, 1024), gumbel.uniform_row(7, 0, 6, 1024)
    assert abs(np.corrcoef(a, b)[0, 1]) < 0.1                           # rows of different positions
    assert not np.array_equal(a, gumbel.uniform_row(8, 0, 5, 1024))     # seed matters
    assert not np.array_equal(a, gumbel.uniform_row(7, 1, 5, 1024))     # sequence matters


def test_gumbel_moments():
    g = np.concatenate([gumbel.gumbel_row(3, 0, p, 8192) for p in range(32)])
    assert abs(g.mean() - 0.5772156649) < 0.01                          # Euler-Mascheroni
    assert abs(g.var() - np.pi ** 2 / 6) < 0.03


@pytest.mark.parametrize("tau", [1.0, 0.7])
def test_gumbel_max_samples_softmax(tau):
    """argmax(l/tau + G) ~ softmax(l/tau): frequencies over 40000 independent rows (Gumbel-Max trick)."""
    logits = np.array([2.0, 1.0, 0.5, 0.0, -0.5, -1.0, -3.0, 1.5])
    n = 40000
    counts = np.zeros(8)
    for p in range(n):
        counts[int(np.argmax(gumbel.perturbed(logits, tau, gumbel.gumbel_row(11, 0, p, 8))))] += 1
    prob = np.exp(logits / tau)
    prob /= prob.sum()
    chi2 = ((counts - n * prob) ** 2 / (n * prob)).sum()
    assert chi2 < 40.0, (chi2, counts / n, prob)                        # 7 dof


@pytest.mark.parametrize("decs", [False, True])
@pytest.mark.parametrize("X", [(2, 4, 6, 8), (4, 8), (1, 3, 4, 8)])
def test_sampled_dex_equals_sampled_ar(c1, c1_model, X, decs):
    """Lossless under sampling: the committed stream is the exact Gumbel-Max sample of the final-depth model."""
    from oracle import ar_sample, dex_decode
    wl, _, p = c1
    T, tau, seed = 24, 0.9, 1234
    ar = ar_sample(c1_model, p, T, tau, seed)
    od = dex_decode(c1_model, p, T, X, decs=decs, sample=(tau, seed, 0))
    assert np.array_equal(od["tokens"], ar["tokens"])
    from oracle import ar_greedy
    assert not np.array_equal(ar["tokens"], ar_greedy(c1_model, p, T)["tokens"])   # it does sample
