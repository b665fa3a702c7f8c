"""Pins for oracle/dex.py (O4): brute-force node values, the paper's invariants
(PAPER.md:204, 208), closed-form counts derived from the AR trace alone, special cases."""
import numpy as np
import pytest

import dex_synth
from oracle import OracleModel, ar_greedy, dex_decode, ead
from oracle import lattice as lt
from oracle.bruteforce import forward_nocache, logits_nocache

XS = [(2, 4, 6, 8), (8,), (4, 8), (1, 2, 3, 4, 5, 6, 7, 8), (3, 5, 8), (2, 8)]


@pytest.fixture(scope="module")
def runs(c1, c1_model):
    wl, _, p = c1
    out = {}
    for X in XS:
        for decs in (False, True):
            T = 64 if X == (2, 4, 6, 8) else 24
            out[(X, decs)] = dex_decode(c1_model, p, T, X, decs=decs, trace=(X == (2, 4, 6, 8)))
    return out


def test_lossless_every_X_and_decs(c1_ar, runs):
    """DEX tokens == AR greedy tokens, every X, DECS on and off."""
    for (X, decs), r in runs.items():
        assert np.array_equal(r["tokens"], c1_ar["tokens"][: len(r["tokens"])]), (X, decs)


def test_committed_token_is_final_depth_argmax(c1, c1_ar, runs):
    """y = u_{N-1}, also when an earlier candidate matches."""
    r = runs[((2, 4, 6, 8), True)]
    commits = [rec for rec in r["rounds"] if rec["committed"]]
    assert len(commits) == 64
    for t, rec in enumerate(commits):
        assert rec["token"] == rec["ref"] == c1_ar["tokens"][t]
        assert int(np.argmax(rec["ref_logits"])) == rec["token"]
        assert np.max(np.abs(rec["ref_logits"] - c1_ar["logits"][t])) < 1e-9     # final-depth state == AR's


def test_node_values_bruteforce(c1, c1_model, runs):
    """Every node's h_out == from-scratch forward of (committed tokens + its path tokens),
    truncated at its stage boundary d_m."""
    wl, _, p = c1
    X = (2, 4, 6, 8)
    for decs in (False, True):
        r = runs[(X, decs)]
        committed = list(p)
        checked = 0
        toks = {}
        for rec in r["rounds"][:40]:
            toks.update(rec["u"])
            for i in rec["nodes"]:
                pref = [toks[j] for j in lt.prefix_tokens_nodes(i)]
                H = forward_nocache(c1_model, committed + pref)
                want = H[X[lt.stage(i)], -1]
                assert np.max(np.abs(rec["h_out"][i] - want)) < 1e-9
                # candidate token = (masked) argmax of the shared exit head at that depth
                lg = logits_nocache(c1_model, want)
                if decs and i != lt.anchor(3):
                    for a in lt.slot_chain_prior(i):
                        lg[toks[a]] = -np.inf
                assert rec["u"][i] == int(np.argmax(lg))
                checked += 1
            if rec["committed"]:
                committed.append(rec["token"])
                _, mp = lt.collapse_map(rec["match_k"], 4)
                toks = {j: toks[o] for j, o in mp.items()}
        assert checked > 100


def test_match_index_vs_ead_table(c1_ar, runs):
    om = ead.acceptance(c1_ar["exit_tokens"])
    for X in XS:
        van, dec = runs[(X, False)], runs[(X, True)]
        T = len(van["tokens"])
        for t in range(T):
            # vanilla: matched depth = shallowest explored depth with plain agreement (R7)
            assert X[van["match_k"][t]] == ead.first_match_depth(om[t], X)
            assert dec["match_k"][t] <= van["match_k"][t]          # DECS can only match earlier
        e, es = ead.ead(om)[:T], ead.stable_ead(om)[:T]
        d = np.array([X[k] for k in van["match_k"]])
        assert np.all(np.array([ead.ceil_X(int(v), X) for v in e]) <= d)
        assert np.all(d <= np.array([ead.ceil_X(int(v), X) for v in es]))


def test_closed_form_counts(runs):
    """rounds = N + sum_{t<T}(k_t+1); per-round rows [2^{q-1-m}..,1]; uniform X: layer-evals of
    a round at level q = (L/N) 2^q."""
    for (X, decs), r in runs.items():
        N, T, k = len(X), len(r["tokens"]), r["match_k"]
        lo = [0] + list(X[:-1])
        for rec in r["rounds"]:
            q = rec["q"]
            assert rec["rows_per_stage"] == lt.rows_per_stage(q, N)
            assert rec["exit_rows"] == 2 ** q
            assert rec["layer_evals"] == sum(n * (X[m] - lo[m]) for m, n in enumerate(rec["rows_per_stage"]))
            assert rec["critical_layers"] == max(X[m] - lo[m] for m in range(q + 1))
            assert rec["committed"] == (q == N - 1)
        uniform = len({X[m] - lo[m] for m in range(N)}) == 1
        if uniform:
            per = X[0]
            assert r["critical_layers"] == X[-1] + sum(X[kk] if kk < N - 1 else X[-1] for kk in k[:-1])
            for rec in r["rounds"]:
                assert rec["layer_evals"] == per * 2 ** rec["q"]


def test_rounds_formula_explicit(runs):
    for (X, decs), r in runs.items():
        N, k = len(X), r["match_k"]
        # after a match at k<N-1 the next commit needs k+1 rounds; after a fallback it needs N
        assert r["n_rounds"] == N + sum((kk + 1) if kk < N - 1 else N for kk in k[:-1])


def test_X_equals_L_is_AR(c1, c1_model, c1_ar):
    wl, _, p = c1
    r = dex_decode(c1_model, p, 10, (8,), trace=True)
    assert r["n_rounds"] == 10 and r["layer_evals"] == 80
    for t, rec in enumerate(r["rounds"]):
        assert rec["committed"] and rec["rows_per_stage"] == [1]
        assert np.array_equal(rec["h_out"][0], c1_ar["hidden"][t][-1])          # step-for-step identical


def test_all_exits_agree_gives_k0(c1):
    """Zero Wo, Wd beyond d_0 => every explored exit equals the final one => k_t = 0 for all t,
    rounds = N + T - 1."""
    wl, w, p = c1
    w0 = {k: v.clone() for k, v in w.items()}
    w0["wo"][2:] = 0
    w0["wdn"][2:] = 0
    m = OracleModel(wl.shape, w0)
    T = 12
    r = dex_decode(m, p, T, (2, 4, 6, 8), decs=False)
    assert np.array_equal(r["tokens"], ar_greedy(m, p, T)["tokens"])
    assert set(r["match_k"].tolist()) == {0} and r["n_rounds"] == 4 + T - 1


def test_collapse_keeps_only_consistent_branches(runs):
    """After every commit the surviving nodes' first prefix token == the committed token
    (PAPER.md:208), and 2^{q'}-1 of them survive."""
    r = runs[((2, 4, 6, 8), True)]
    toks = {}
    for rec in r["rounds"]:
        toks.update(rec["u"])
        if rec["committed"]:
            k = rec["match_k"]
            qn, mp = lt.collapse_map(k, 4)
            assert rec["q_after"] == qn and len(mp) == 2 ** qn - 1
            for j, o in mp.items():
                first_prefix_node = lt.prefix_tokens_nodes(o)[0]
                assert toks[first_prefix_node] == rec["token"]
            toks = {j: toks[o] for j, o in mp.items()}


def test_bf16_kv_and_fp32_variants_still_lossless(c1):
    """Losslessness is a property of the procedure, not of the precision."""
    wl, w, p = c1
    for kw in (dict(dtype=np.float32), dict(kv_round="bf16"), dict(dtype=np.float32, kv_round="bf16")):
        m = OracleModel(wl.shape, w, **kw)
        a = ar_greedy(m, p, 16)["tokens"]
        assert np.array_equal(dex_decode(m, p, 16, (2, 4, 6, 8))["tokens"], a)


def test_exact_fp32_weights_invariants():
    """Config c1's "fp32" leg (R15): unrounded fp32 weights, same invariants."""
    wl = dex_synth.workload("c1")
    w = dex_synth.make_weights(wl.shape, wl.weight_seed, exact_fp32=True)
    m = OracleModel(wl.shape, w)
    p = dex_synth.make_prompt(wl.shape.vocab, wl.prompt_len, wl.prompt_seed)
    a = ar_greedy(m, p, 20)["tokens"]
    assert np.array_equal(dex_decode(m, p, 20, wl.depths)["tokens"], a)


def test_teacher_forcing_hook_matches_selection(c1, c1_model, c1_ar):
    """force_tokens = the AR tokens is a no-op."""
    wl, _, p = c1
    r = dex_decode(c1_model, p, 12, (2, 4, 6, 8), force_tokens=c1_ar["tokens"][:12])
    assert np.array_equal(r["tokens"], c1_ar["tokens"][:12])


def test_force_u_hook(c1, c1_model, runs):
    """dex_decode(force_u=...) (teacher forcing of exit decisions for the GPU parity harness, reading R17b): forcing
    the oracle's own candidates changes nothing and records nothing; forcing another token at one node records the
    logit gap between the oracle's arg-max and the forced token and the lattice continues from the forced token."""
    wl, _, p = c1
    X = (2, 4, 6, 8)
    base = runs[(X, True)]
    T = 12
    own = {(ri, i): t for ri, rec in enumerate(base["rounds"]) for i, t in rec["u"].items()}
    same = dex_decode(c1_model, p, T, X, trace=True, force_u=own)
    assert np.array_equal(same["tokens"], base["tokens"][:T])
    assert all("u_forced" not in rec for rec in same["rounds"])
    # force the second-best token at the final-depth anchor of the first commit round
    ri = next(i for i, rec in enumerate(base["rounds"]) if rec["committed"])
    rec = base["rounds"][ri]
    ref_node = lt.anchor(len(X) - 1)
    lg = rec["ref_logits"]
    second = int(np.argsort(lg)[-2])
    forced = dex_decode(c1_model, p, 3, X, trace=True, force_u={(ri, ref_node): second})
    fr = forced["rounds"][ri]
    a, t, gap = fr["u_forced"][ref_node]
    assert a == rec["u"][ref_node] and t == second
    assert np.isclose(gap, lg[a] - lg[second]) and gap > 0
    assert forced["tokens"][0] == second and fr["token"] == second        # the forced candidate is what gets committed
    # a masked token can never be produced by DECS: infinite gap
    node = next(i for i in base["rounds"][1]["nodes"] if lt.slot_chain_prior(i))
    prior_tok = base["rounds"][0]["u"][lt.slot_chain_prior(node)[0]]
    bad = dex_decode(c1_model, p, 1, X, trace=True, force_u={(1, node): prior_tok})
    if base["rounds"][1]["u"][node] != prior_tok:
        assert bad["rounds"][1]["u_forced"][node][2] == np.inf
