"""Pins for oracle/lattice.py: the counts PAPER.md states and a brute-force enumeration of all
D/P move strings (independent of the heap arithmetic)."""
import itertools
import os

from oracle import lattice as lt


def _golden(key):
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_worked_examples.txt")) as f:
        for line in f:
            line = line.split("#")[0]
            if line.strip().startswith(key):
                return float(line.split("=")[1])
    raise KeyError(key)


def test_paper_counts():
    assert sum(len(lt.level_nodes(q)) for q in range(4)) == int(_golden("nodes_state4"))
    for q in range(1, 9):
        assert sum(len(lt.level_nodes(j)) for j in range(q)) == 2 ** q - 1                    # "first 2^q-1"
    assert len(lt.level_nodes(7)) == int(_golden("max_batch_K8"))
    assert sum(len(lt.level_nodes(j)) for j in range(8)) == int(_golden("max_lattice_K8"))
    # ETK_0 -> ETK_1 by depth expansion, ETK_2 by position expansion
    assert lt.path(1) == ['D'] and lt.path(2) == ['P']
    assert lt.stage(1) == 1 and lt.pos_offset(1) == 0 and lt.slot_root(1) == 0
    assert lt.stage(2) == 0 and lt.pos_offset(2) == 1 and lt.slot_root(2) == 2


def _enumerate(q):
    """All move strings of length q in BFS heap order, depth child first."""
    return list(itertools.product("DP", repeat=q))


def test_heap_matches_bruteforce_enumeration():
    for q in range(0, 8):
        nodes = lt.level_nodes(q)
        strings = _enumerate(q)
        assert len(nodes) == len(strings) == 2 ** q
        for i, s in zip(nodes, strings):
            s = list(s)
            assert lt.path(i) == s
            trailing = len(s) - len("".join(s).rstrip("D"))
            assert lt.stage(i) == trailing
            assert lt.pos_offset(i) == s.count("P")
            assert lt.level(i) == q


def test_rows_per_stage_and_survey_trace():
    assert [lt.rows_per_stage(q, 4) for q in range(4)] == [[1, 0, 0, 0], [1, 1, 0, 0], [2, 1, 1, 0], [4, 2, 1, 1]]
    assert lt.rows_per_stage(7, 8) == [64, 32, 16, 8, 4, 2, 1, 1]
    for N in (2, 3, 4, 8):
        for q in range(N):
            r = lt.rows_per_stage(q, N)
            assert sum(r) == 2 ** q and r[q] == 1
            assert all(r[m] == 2 ** (q - 1 - m) for m in range(q))
    # node 13 = P,P,D: slot root 6, attends to slots of nodes 0 and 2
    assert lt.path(13) == ['P', 'P', 'D'] and lt.slot_root(13) == 6
    assert lt.ancestor_slots(13) == [0, 2] and lt.prefix_tokens_nodes(13) == [0, 2]
    assert lt.ancestor_slots(4) == [0] and lt.prefix_tokens_nodes(4) == [1]      # D,P: prefix token is u(1)
    assert lt.slot_chain_prior(7) == [0, 1, 3] and lt.slot_chain_prior(5) == [2]
    assert [lt.anchor(k) for k in range(4)] == [0, 1, 3, 7]


def test_ancestor_chain_nodes_are_older():
    """The K/V a node reads from an ancestor slot at its own stage was produced in a strictly
    earlier round (so one round never reads what it writes)."""
    N = 6
    for q in range(N):
        for i in lt.level_nodes(q):
            m = lt.stage(i)
            for a in lt.ancestor_slots(i):
                j = a
                for _ in range(m):
                    j = 2 * j + 1           # a's chain node at stage m
                assert lt.level(j) < q and lt.slot_root(j) == a and lt.stage(j) == m


def test_collapse_map():
    # N=4 enumerated in SURVEY.md 8(c): k=0 keeps {2,5,6,11,12,13,14}
    assert lt.collapse_map(0, 4) == (3, {0: 2, 1: 5, 2: 6, 3: 11, 4: 12, 5: 13, 6: 14})
    assert lt.collapse_map(1, 4) == (2, {0: 4, 1: 9, 2: 10})
    assert lt.collapse_map(2, 4) == (1, {0: 8})
    assert lt.collapse_map(3, 4) == (0, {})
    for N in (2, 3, 4, 5, 8):
        for k in range(N):
            qn, mp = lt.collapse_map(k, N)
            assert qn == (N - 1 - k if k < N - 1 else 0)
            assert len(mp) == 2 ** qn - 1                       # survivor count
            r = 2 * lt.anchor(k) + 2 if k < N - 1 else None
            for j, o in mp.items():
                assert o < 2 ** N - 1
                # closed form of SURVEY O4: old = ((r+1) << lam) + off - 1
                lam = lt.level(j)
                assert o == ((r + 1) << lam) + (j + 1 - 2 ** lam) - 1
                # survivors' prefix == committed prefix: old path = path(anchor k) + 'P' + new path
                assert lt.path(o) == ['D'] * k + ['P'] + lt.path(j)
                assert lt.stage(o) == lt.stage(j)                # stage structure preserved
                assert lt.pos_offset(o) == lt.pos_offset(j) + 1  # positions shift by exactly one
            # every node consistent with the new committed prefix survives (none missed)
            if k < N - 1:
                want = [i for i in range(2 ** N - 1) if lt.path(i)[:k + 1] == ['D'] * k + ['P']]
                assert sorted(mp.values()) == want
