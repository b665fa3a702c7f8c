"""Sparse exploration lattice (dex_config.lookahead = P, reading R26) through the C ABI against the
oracle's trace: which nodes are expanded (rows per stage, exit rows, layer evaluations: bit-exact), every node's
candidate token (flip only at an oracle margin < 1e-2, R17) and stage-boundary hidden state, the explored-branch
mask and the commit rule, and the commit invariant: GPU DEX(P) stream == GPU AR stream, bit-identical."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

MARGIN, HID_TOL = 1e-2, 2e-2


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2606_29223_b200 import build
    build.build()
    import paper_2606_29223_b200 as P
    return P


@pytest.fixture(scope="module")
def c1_bf16(c1):
    from oracle import OracleModel
    wl, w, p = c1
    return OracleModel(wl.shape, w, kv_round="bf16")


@pytest.mark.parametrize("rk", [1, 0, 2])
@pytest.mark.parametrize("X,cap", [((2, 4, 6, 8), 1), ((2, 4, 6, 8), 2), (tuple(range(1, 9)), 1), (tuple(range(1, 9)), 2),
                                   (tuple(range(1, 9)), 3), ((1, 3, 4, 8), 2)])
def test_c1_sparse_lattice_matches_oracle(P, c1, c1_bf16, X, cap, rk):
    """Every round of a 24-token run against the oracle's trace with the same cap (tests/trace_util.py: the oracle
    replays with the GPU's exit decisions forced, so nothing is skipped after a near-tie flip): exactly the oracle's
    nodes are expanded, counts bit-exact, hidden states, the explored-branch mask and the R26 commit rule."""
    from trace_util import gpu_trace, compare_with_oracle
    wl, w, p = c1
    T = 24
    g = P.Dex(wl.shape, w, X, max_ctx=128, debug_taps=1, use_graph=0, lookahead=cap, round_kernel=rk)
    g.prefill(0, p)
    recs = gpu_trace(g, T)
    dex_tokens = g.tokens()[len(p):len(p) + T]
    g.close()
    res = compare_with_oracle(recs, c1_bf16, p, X, T, lookahead=cap)
    assert res["rounds"] == len(recs) >= T and res["nodes"] > 30                # coverage: every round, every node
    assert np.array_equal(res["tokens"], dex_tokens)
    a = P.Dex(wl.shape, w, (wl.shape.n_layers,), max_ctx=128, round_kernel=rk)
    a.prefill(0, p)
    ar_gpu, _ = a.generate(T)
    a.close()
    assert np.array_equal(ar_gpu, dex_tokens)                               # the commit invariant


def test_wide_cap_is_the_full_lattice_and_rows_shrink(P, c1):
    wl, w, p = c1
    X = tuple(range(1, 9))
    runs = {}
    for cap in (0, 7, 9, 2):
        g = P.Dex(wl.shape, w, X, max_ctx=128, lookahead=cap)
        g.prefill(0, p)
        toks, recs = g.generate(32)
        runs[cap] = (toks.tolist(), [(r["q"], r["rows_per_stage"], r["match_k"]) for r in recs],
                     sum(r["layer_evals"] for r in recs))
        g.close()
    assert runs[7][:2] == runs[0][:2] and runs[9][:2] == runs[0][:2]
    assert runs[2][0] == runs[0][0] and runs[2][2] < runs[0][2] // 2


def test_collapse_onto_unexplored_branch_is_refused_and_batched_streams(P, c1):
    import dex_synth
    wl, w, p = c1
    X = (2, 4, 6, 8)
    g = P.Dex(wl.shape, w, X, max_ctx=128, lookahead=1, use_graph=0)
    g.prefill(0, p)
    seen = False
    for _ in range(200):
        r = g.step(0)[0]
        if r.match_k < 0:
            continue
        missing = [k for k in range(len(X) - 1) if not (r.branch_mask >> k) & 1]
        if missing and not seen:
            seen = True
            with pytest.raises(P.DexError) as e:
                g.collapse(0, missing[0], r.anchor_tokens[missing[0]])
            assert e.value.code == P.DEX_EINVAL
        g.collapse(0, r.match_k, r.token)
    assert seen                                                             # holes do appear after a collapse at P = 1
    g.close()
    # two sequences, graph replay, auto-collapse: each stream equals its own single-sequence stream
    p2 = dex_synth.make_prompt(wl.shape.vocab, 19, 5)
    T = 32
    ref = []
    for pr in (p, p2):
        s = P.Dex(wl.shape, w, (wl.shape.n_layers,), max_ctx=128)
        s.prefill(0, pr)
        ref.append(s.generate(T)[0])
        s.close()
    b = P.Dex(wl.shape, w, X, max_seqs=2, max_ctx=128, lookahead=2)
    b.prefill(0, p)
    b.prefill(1, p2)
    for _ in range(4 * T):
        b.step()
    assert np.array_equal(b.tokens(0)[len(p):len(p) + T], ref[0])
    assert np.array_equal(b.tokens(1)[len(p2):len(p2) + T], ref[1])
    b.close()


def test_sparse_lattice_with_adapters_and_sampling(P, c1):
    """All optional pieces together (sampling-mode DECS, inducing adapters, look-ahead cap, two sequences, graph
    replay): the stream is still the GPU AR sampling stream with the same Gumbel rows."""
    import dex_synth
    wl, w, p = c1
    X, T = (1, 2, 3, 4, 6, 8), 32
    ad = dex_synth.make_adapters(wl.shape, len(X) - 1, seed=3, alpha=0.5, m=256)
    p2 = dex_synth.make_prompt(wl.shape.vocab, 23, 9)
    kw = dict(sample=1, temperature=0.9, sample_seed=11)
    a = P.Dex(wl.shape, w, (wl.shape.n_layers,), max_seqs=2, max_ctx=128, **kw)
    g = P.Dex(wl.shape, w, X, max_seqs=2, max_ctx=128, adapters=ad, lookahead=2, **kw)
    out = []
    for d in (a, g):
        d.prefill(0, p)
        d.prefill(1, p2)
        for _ in range(6 * T):
            d.step()
        out.append((d.tokens(0)[len(p):len(p) + T].tolist(), d.tokens(1)[len(p2):len(p2) + T].tolist()))
        d.close()
    assert len(out[0][0]) == T and len(out[0][1]) == T
    assert out[0] == out[1]


@pytest.mark.parametrize("cap", [0, 3])
def test_two_wide_lattices_batched(P, c1, cap):
    """N = 8 with two sequences: 128 stage-0 rows, the pass-task instantiation of the round kernel, sequences at
    different FSM states in the same launches; each stream equals its own AR stream."""
    import dex_synth
    wl, w, p = c1
    X, T = tuple(range(1, 9)), 24
    p2 = dex_synth.make_prompt(wl.shape.vocab, 37, 21)
    ref = []
    for pr in (p, p2):
        s = P.Dex(wl.shape, w, (wl.shape.n_layers,), max_ctx=128)
        s.prefill(0, pr)
        ref.append(s.generate(T)[0])
        s.close()
    b = P.Dex(wl.shape, w, X, max_seqs=2, max_ctx=128, lookahead=cap)
    b.prefill(0, p)
    b.step()
    b.step()                      # sequence 0 is two rounds ahead when sequence 1 joins
    b.prefill(1, p2)
    for _ in range(9 * T):
        b.step()
    assert np.array_equal(b.tokens(0)[len(p):len(p) + T], ref[0])
    assert np.array_equal(b.tokens(1)[len(p2):len(p2) + T], ref[1])
    b.close()
