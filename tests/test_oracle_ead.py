"""Pins for oracle/ead.py against the numbers PAPER.md prints (tests/golden) and the
bounds it proves (Eq. 11, Eq. 14, monotonicity, X=[L])."""
import os

import numpy as np
from hypothesis import given, settings, strategies as st

from oracle import ead

G = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "paper_worked_examples.txt")) as f:
    for line in f:
        line = line.split("#")[0].strip()
        if "=" in line:
            k, v = [s.strip() for s in line.split("=", 1)]
            G[k] = v
X = [int(t) for t in G["X"].split(",")]
L, E = int(G["L"]), int(G["EAD"])


def test_exploration_worked_example():
    assert ead.ceil_X(E, X) == int(G["ceil_X_EAD"])
    assert ead.ceil_X(E, X) - E == int(G["overhead_exp"])
    assert ead.resolution(X, L) == int(G["resolution"])


def test_selection_worked_example():
    s = int(G["sel_conservative_s"])
    assert ead.selection_cost(1.0, s, L, [s]) - E == int(G["sel_conservative_extra"])
    s = int(G["sel_aggressive_s"])
    for s1, s2 in ((3, 9), (11, 2)):
        assert ead.selection_cost(0.0, s, L, [s, s1, s2]) == int(G["sel_aggressive_fixed"]) + s1 + s2
    # Prop. 3 decomposition (Eq. 5) for a fractional acceptance probability
    p, s, disc = 0.3, 6, [6, 7]
    lhs = ead.selection_cost(p, s, L, disc) - E
    rhs = p * (s - E) + (1 - p) * (L + sum(disc) - E)
    assert abs(lhs - rhs) < 1e-12


def test_definitions_small_table():
    # exits at depths 1..6 for 3 tokens; final token in the last column
    e = np.array([[5, 7, 7, 2, 7, 7],      # matches at 2,3 then diverges at 4: EAD 2, stable 5
                  [1, 1, 1, 1, 1, 1],      # EAD 1, stable 1
                  [3, 4, 5, 6, 7, 8]])     # only the final depth: 6, 6
    om = ead.acceptance(e)
    assert om[:, -1].tolist() == [1, 1, 1]               # Omega(t,L)=1 by construction
    assert ead.ead(om).tolist() == [2, 1, 6]
    assert ead.stable_ead(om).tolist() == [5, 1, 6]
    assert ead.stable_acceptance(om)[0].tolist() == [0, 0, 0, 0, 1, 1]
    assert ead.workload_X(ead.stable_acceptance(om)[0], [2, 4, 6]) == 6
    assert ead.first_match_depth(om[0], [2, 4, 6]) == 2
    assert ead.speedup(6, [2, 1, 6]) == 18 / 9


sets = st.integers(4, 24).flatmap(
    lambda L_: st.tuples(st.just(L_), st.sets(st.integers(1, L_ - 1), max_size=6),
                         st.sets(st.integers(1, L_ - 1), max_size=6),
                         st.lists(st.integers(1, L_), min_size=1, max_size=12)))


@settings(max_examples=200, deadline=None)
@given(sets)
def test_bounds_and_monotonicity(args):
    L_, a, b, eads = args
    Xa = sorted(a) + [L_]
    Xb = sorted(a | b) + [L_]                      # Xa subset of Xb
    D = ead.resolution(Xa, L_)
    for e in eads:
        c = ead.ceil_X(e, Xa) - e
        assert 0 <= c <= D                          # Eq. 11
        assert ead.ceil_X(e, Xb) <= ead.ceil_X(e, Xa)   # Eq. 30
    S_ead = ead.speedup(L_, eads)
    Sa, Sb = ead.speedup_X(L_, eads, Xa), ead.speedup_X(L_, eads, Xb)
    lower = ead.speedup_lower(L_, eads, Xa)
    assert 1 <= lower + 1e-12 and lower <= Sa + 1e-12 and Sa <= Sb + 1e-12 and Sb <= S_ead + 1e-12   # Eq. 14
    full = list(range(1, L_ + 1))
    assert abs(ead.speedup_X(L_, eads, full) - S_ead) < 1e-12
    assert ead.resolution(full, L_) == 0


def test_resolution_uniform():
    # uniformly spaced: Delta = spacing - 1 ("less than the adjacent spacing")
    for L_, K in ((32, 4), (32, 8), (40, 8), (8, 4)):
        Xs = list(range(L_ // K, L_ + 1, L_ // K))
        assert ead.resolution(Xs, L_) == L_ // K - 1


def test_check_X_rejects():
    import pytest
    for bad in ([], [4, 4, 8], [8, 4], [2, 4, 6], [0, 8]):
        with pytest.raises(ValueError):
            ead.check_X(bad, 8)
    assert ead.check_X([2, 4, 6, 8], 8) == [2, 4, 6, 8]
