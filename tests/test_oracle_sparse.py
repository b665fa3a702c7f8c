"""Sparse exploration lattice (reading R26; "prune low-value branches or construct sparse exploration
lattices while preserving the final-depth commit invariant"): position look-ahead cap P in the oracle.  Pins: the
commit invariant (DEX == AR for every P), P >= N-1 is the full lattice of Sec. 3.2, binomial node counts of a fresh
lattice, closure under parents, and that the anchor chain (the commit rule's inputs) is never pruned."""
from math import comb

import numpy as np
import pytest

from oracle import dex_decode, lattice as lt


@pytest.mark.parametrize("X", [(2, 4, 6, 8), (1, 3, 4, 8), tuple(range(1, 9))])
@pytest.mark.parametrize("P", [1, 2, 3])
@pytest.mark.parametrize("decs", [True, False])
def test_commit_invariant_and_structure(c1, c1_model, c1_ar, X, P, decs):
    wl, w, p = c1
    T, N = 20, len(X)
    od = dex_decode(c1_model, p, T, X, decs=decs, trace=True, lookahead=P)
    assert np.array_equal(od["tokens"], c1_ar["tokens"][:T])                     # lossless
    full = dex_decode(c1_model, p, T, X, decs=decs, trace=True)
    assert od["layer_evals"] <= full["layer_evals"] or od["n_rounds"] > full["n_rounds"]
    present = set()
    for ri, r in enumerate(od["rounds"]):
        nodes = r["nodes"]
        assert lt.anchor(r["q"]) in nodes                                        # anchors are never pruned
        for i in nodes:
            assert lt.level(i) == r["q"] and lt.pos_offset(i) <= P
            assert i == 0 or lt.parent(i) in present                             # closed under parents
        assert sum(r["rows_per_stage"]) == len(nodes) == r["exit_rows"]
        full_level = [i for i in lt.level_nodes(r["q"]) if lt.pos_offset(i) <= P]
        assert set(nodes) <= set(full_level)
        present |= set(nodes)
        if r["committed"]:                                                       # survivors re-rooted
            q_new, mp = lt.collapse_map(r["match_k"], N)
            present = {j for j, o in mp.items() if o in present}
    if N - 1 > P:
        assert max(len(r["nodes"]) for r in od["rounds"]) < 2 ** (N - 1)         # it is sparser than the full lattice


def test_fresh_lattice_counts_are_binomial(c1, c1_model):
    """From an empty lattice (q = 0 after init) level q holds sum_{j<=P} C(q, j) nodes; stage m of level q holds the
    offsets with m trailing depth moves: brute-force enumeration of the heap ids."""
    wl, w, p = c1
    X = tuple(range(1, 9))
    for P in (1, 2, 3):
        od = dex_decode(c1_model, p, 1, X, trace=True, lookahead=P)
        for q, r in enumerate(od["rounds"][:len(X)]):
            assert r["q"] == q
            assert len(r["nodes"]) == sum(comb(q, j) for j in range(min(P, q) + 1))
            want = [0] * len(X)
            for o in range(2 ** q):
                if bin(o).count("1") <= P:
                    want[lt.stage(2 ** q - 1 + o)] += 1
            assert r["rows_per_stage"] == want


@pytest.mark.parametrize("X", [(2, 4, 6, 8), (4, 8)])
def test_wide_cap_is_the_full_lattice(c1, c1_model, X):
    wl, w, p = c1
    T = 16
    full = dex_decode(c1_model, p, T, X, trace=True)
    for P in (len(X) - 1, len(X) + 3):
        od = dex_decode(c1_model, p, T, X, trace=True, lookahead=P)
        assert [r["nodes"] for r in od["rounds"]] == [r["nodes"] for r in full["rounds"]]
        assert [r["u"] for r in od["rounds"]] == [r["u"] for r in full["rounds"]]
        assert np.array_equal(od["match_k"], full["match_k"])


def test_sampling_mode_stays_exact_on_the_sparse_lattice(c1, c1_model):
    from oracle import ar_sample
    wl, w, p = c1
    T = 16
    ar = ar_sample(c1_model, p, T, 0.8, 3)
    od = dex_decode(c1_model, p, T, (2, 4, 6, 8), sample=(0.8, 3, 0), lookahead=1)
    assert np.array_equal(od["tokens"], ar["tokens"])
