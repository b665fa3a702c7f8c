"""Full-size checks at the 7B shape of config c2, in the launch configuration bench.py times
(CUDA-graph replay, auto-collapse, act_planes = 2): the oracle is too slow for the whole run, so
(i) sampled GEMM outputs are checked against float64 dot products on the same weights,
(ii) a shortened run (8-token prompt, 3 tokens) is compared with the fp32 oracle end to end,
(iii) properties that hold at any size: GPU DEX stream == GPU AR stream, committed token ==
final-depth anchor token, closed-form round and layer-evaluation counts."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


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
def c2():
    import dex_synth
    wl = dex_synth.workload("c2")
    w = dex_synth.make_weights(wl.shape, wl.weight_seed, threads=16)
    return wl, w


def test_c2_gemm_sampled_outputs(P, c2):
    wl, w = c2
    d = P.Dex(wl.shape, w, wl.depths, max_ctx=256, debug_taps=1, use_graph=0)
    rng = np.random.default_rng(3)
    for which, name in enumerate(("wqkv", "wo", "wgu", "wdn")):
        W = w[name][17].reshape(-1, w[name].shape[-1])
        x = rng.standard_normal((128, W.shape[1])).astype(np.float32)
        y = d.gemm(which, 17, x)
        cols = rng.integers(0, W.shape[0], size=256)
        ref = x.astype(np.float64) @ W[cols].float().numpy().astype(np.float64).T
        err = np.abs(y[:, cols] - ref).max() / np.abs(ref).max()
        assert err < 2e-5, (name, err)
    d.close()


def test_c2_short_run_against_fp32_oracle(P, c2):
    import dex_synth
    from oracle import OracleModel, ar_greedy
    wl, w = c2
    om = OracleModel(wl.shape, w, dtype=np.float32, kv_round="bf16")
    p = dex_synth.make_prompt(wl.shape.vocab, 8, 11)
    T = 3
    ar = ar_greedy(om, p, T, keep_hidden=True, keep_logits=True)
    d = P.Dex(wl.shape, w, (wl.shape.n_layers,), max_ctx=128, debug_taps=1, use_graph=0)
    d.prefill(0, p)
    from trace_util import check_ref_blocks
    for t in range(T):
        r = d.step(0)[0]
        h = d.tap_hidden(0)
        for l in range(wl.shape.n_layers):
            assert np.abs(h[l] - ar["hidden"][t][l]).max() / np.abs(ar["hidden"][t][l]).max() < 2e-2
        assert np.abs(d.tap_logits() - ar["logits"][t]).max() < 5e-2
        check_ref_blocks(d.tap_ref_blocks(), ar["logits"][t])   # the fused exit's own reduction over all 1000 blocks
        if r.token != ar["tokens"][t]:
            assert ar["top1"][t] - ar["top2"][t] < 1e-2
        d.collapse(0, 0, int(ar["tokens"][t]))                 # teacher-forced (R17): every position is compared
    d.close()


def test_c2_dex_equals_ar_and_counts(P, c2):
    import dex_synth
    wl, w = c2
    p = dex_synth.make_prompt(wl.shape.vocab, wl.prompt_len, wl.prompt_seed)
    T = 48
    a = P.Dex(wl.shape, w, (wl.shape.n_layers,), max_ctx=wl.prompt_len + 64)
    a.prefill(0, p)
    ar_toks, _ = a.generate(T)
    a.close()
    g = P.Dex(wl.shape, w, wl.depths, max_ctx=wl.prompt_len + 64)
    g.prefill(0, p)
    toks, recs = g.generate(T)
    g.close()
    assert np.array_equal(toks, ar_toks)                       # H3 / losslessness on the GPU
    N, L = len(wl.depths), wl.shape.n_layers
    ks = [r["match_k"] for r in recs if r["committed"]]
    assert len(recs) == N + sum(k + 1 for k in ks[:-1])        # rounds = N + sum (k_t + 1)
    per = L // N
    assert sum(r["layer_evals"] for r in recs) == per * ((2 ** N - 1) + sum(2 ** N - 2 ** (N - 1 - k) for k in ks[:-1]))
    for r in recs:
        if r["committed"]:
            assert r["rows_per_stage"][:N] == [4, 2, 1, 1]


# ------------------------------------------------------------------------------------------
# c3 / c4 / c5 at full size (BASELINE.json:configs[2..4]): the oracle cannot run these shapes in test
# time, so what is checked is what holds at any size - GPU DEX stream bit-identical to the GPU AR stream
# built from the same kernels (losslessness, PAPER.md:208 / H3), every committed token == the final-depth
# anchor token, closed-form round and layer-evaluation counts, the row counts
# of the last tree level - plus sampled GEMM outputs against float64 dot products.
def _generate_all(g, n_seqs, T):
    """Rounds until every sequence has committed T tokens.  Returns tokens[s], records[s]."""
    toks = [[] for _ in range(n_seqs)]
    recs = [[] for _ in range(n_seqs)]
    for _ in range(100000):
        if all(len(t) >= T for t in toks):
            break
        res = g.step()
        for s in range(n_seqs):
            r = res[s]
            if not r.active or len(toks[s]) >= T:
                continue
            recs[s].append(dict(q=r.q_before, committed=r.committed, token=r.token, k=r.match_k, evals=r.layer_evals,
                                rows=list(r.rows_per_stage), anchor=list(r.anchor_tokens), exit_rows=r.exit_rows,
                                mask=r.branch_mask))
            if r.committed:
                toks[s].append(r.token)
    return toks, recs


@pytest.mark.parametrize("key,T", [("c3", 24), ("c4", 16), ("c5", 48)])
def test_fullsize_dex_equals_ar_counts_and_gemm(P, key, T):
    import dex_synth
    wl = dex_synth.workload(key)
    w = dex_synth.make_weights(wl.shape, wl.weight_seed, threads=16)
    X, L, N, S = wl.depths, wl.shape.n_layers, len(wl.depths), wl.n_seqs
    prompts = [dex_synth.make_prompt(wl.shape.vocab, wl.prompt_len, wl.prompt_seed, seq=s) for s in range(S)]
    import torch
    wd = {k: v.cuda() for k, v in w.items()}
    a = P.Dex(wl.shape, wd, (L,), max_seqs=S, max_ctx=wl.prompt_len + T + 8)
    for s in range(S):
        a.prefill(s, prompts[s])
    ar_toks, _ = _generate_all(a, S, T)
    a.close()
    g = P.Dex(wl.shape, wd, X, max_seqs=S, max_ctx=wl.prompt_len + T + 8)
    for s in range(S):
        g.prefill(s, prompts[s])
    toks, recs = _generate_all(g, S, T)
    lens = [b - a_ for a_, b in zip((0,) + tuple(X[:-1]), X)]
    for s in range(S):
        assert toks[s][:T] == ar_toks[s][:T], (key, s)                        # H3 / losslessness on the GPU
        ks = [r["k"] for r in recs[s] if r["committed"]]
        n_rounds = len(recs[s])
        # rounds: N for the first token, k_t + 1 for every later one (the last commit ends the run)
        assert n_rounds == N + sum(k + 1 for k in ks[:T - 1]), (key, s)
        for r in recs[s]:
            q = r["q"]
            want = [(1 << (q - 1 - m)) if m < q else (1 if m == q else 0) for m in range(N)]
            assert r["rows"][:N] == want and r["exit_rows"] == 1 << q
            assert r["evals"] == sum(n * ln for n, ln in zip(want, lens))
            if r["committed"]:
                assert r["token"] == r["anchor"][N - 1]                       # y = u_{N-1}
                assert r["k"] == next((i for i in range(N) if r["anchor"][i] == r["token"]), N - 1)
    g.close()
    # sparse lattice (R26) at full size: same stream, rows within the binomial bound of the cap,
    # commit = shallowest matching anchor whose continuation was explored
    from math import comb
    cap = 2
    g = P.Dex(wl.shape, wd, X, max_seqs=S, max_ctx=wl.prompt_len + T + 8, lookahead=cap)
    for s in range(S):
        g.prefill(s, prompts[s])
    stoks, srecs = _generate_all(g, S, T)
    for s in range(S):
        assert stoks[s][:T] == ar_toks[s][:T], (key, s, "sparse")
        for r in srecs[s]:
            q = r["q"]
            assert r["exit_rows"] == sum(r["rows"][:N]) <= sum(comb(q, j) for j in range(min(cap, q) + 1))
            assert r["rows"][q] == 1 and r["evals"] == sum(n * ln for n, ln in zip(r["rows"][:N], lens))
            if r["committed"]:
                assert r["token"] == r["anchor"][N - 1]
                assert r["k"] == next((i for i in range(N - 1) if r["anchor"][i] == r["token"] and (r["mask"] >> i) & 1), N - 1)
        assert sum(r["evals"] for r in srecs[s]) < sum(r["evals"] for r in recs[s])
    # sampled GEMM outputs of this shape
    d = P.Dex(wl.shape, wd, X, max_seqs=1, max_ctx=256, debug_taps=1, use_graph=0)
    rng = np.random.default_rng(5)
    for which, name in enumerate(("wqkv", "wo", "wgu", "wdn")):
        W = w[name][L // 2].reshape(-1, w[name].shape[-1])
        x = rng.standard_normal((37, W.shape[1])).astype(np.float32)
        y = d.gemm(which, L // 2, x)
        cols = rng.integers(0, W.shape[0], size=128)
        ref = x.astype(np.float64) @ W[cols].float().numpy().astype(np.float64).T
        assert np.abs(y[:, cols] - ref).max() / np.abs(ref).max() < 2e-5, (key, name)
    d.close()
    g.close()
    del wd
    torch.cuda.empty_cache()


@pytest.mark.parametrize("with_ad", [False, True])
def test_c2_dex_short_run_against_fp32_oracle(P, c2, with_ad):
    """The lattice itself at the 7B shape against the oracle's Alg. 1 trace (8-token prompt, 2 commits), EVERY round
    (tests/trace_util.py): each new node's stage-boundary hidden state (tolerance R16), its candidate token (forced
    into the oracle's replay; a difference only at an oracle logit gap < 1e-2, R17b), rows per stage / layer
    evaluations (bit-exact), the commits.  with_ad: the non-final exits go through inducing adapters of the paper's
    width m = 2 d_model."""
    import dex_synth
    from oracle import OracleModel
    from trace_util import gpu_trace, compare_with_oracle
    wl, w = c2
    ad = dex_synth.make_adapters(wl.shape, len(wl.depths) - 1, seed=7, alpha=0.5) if with_ad else None
    om = OracleModel(wl.shape, w, dtype=np.float32, kv_round="bf16", adapters=ad)
    p = dex_synth.make_prompt(wl.shape.vocab, 8, 11)
    T = 2
    g = P.Dex(wl.shape, w, wl.depths, max_ctx=128, debug_taps=1, use_graph=0, adapters=ad)
    g.prefill(0, p)
    recs = gpu_trace(g, T)
    g.close()
    res = compare_with_oracle(recs, om, p, wl.depths, T)
    assert res["rounds"] == len(recs) >= len(wl.depths) + 1 and res["nodes"] >= 16


@pytest.mark.parametrize("rk", [1, 0])
def test_c2_single_plane_dex_equals_ar(P, c2, rk):
    """H3 with act_planes = 1 (activations enter the MMAs as plain bf16): rounding to bf16 amplifies ANY difference
    between the arithmetic of a DEX round and of the AR pass into token flips, so this run is the sharpest detector of
    a non-identical code path (it found one in round 2: the first norm of a stage was reduced in another order by
    k_gather_norm than by the previous layer's add+norm unit).  200 tokens at the bench context."""
    import dex_synth
    wl, w = c2
    p = dex_synth.make_prompt(wl.shape.vocab, wl.prompt_len, wl.prompt_seed)
    T = 200
    out = {}
    for name, X in (("ar", (wl.shape.n_layers,)), ("dex", wl.depths)):
        d = P.Dex(wl.shape, w, X, max_ctx=wl.prompt_len + T + 8, act_planes=1, round_kernel=rk)
        d.prefill(0, p)
        out[name], _ = d.generate(T)
        d.close()
    assert np.array_equal(out["dex"], out["ar"])


def test_c3_flow_kernel_equals_round_kernel(P):
    """k_flow on the N = 8 lattice of c3 at full size (pass tasks, 128 rows, 512-token context): same stream as k_round."""
    import dex_synth
    import torch
    wl = dex_synth.workload("c3")
    w = dex_synth.make_weights(wl.shape, wl.weight_seed, threads=16)
    wd = {k: v.cuda() for k, v in w.items()}
    p = dex_synth.make_prompt(wl.shape.vocab, wl.prompt_len, wl.prompt_seed)
    out = {}
    for rk in (1, 2):
        g = P.Dex(wl.shape, wd, wl.depths, max_ctx=wl.prompt_len + 32, round_kernel=rk)
        g.prefill(0, p)
        out[rk], _ = g.generate(16)
        g.close()
    del wd
    torch.cuda.empty_cache()
    assert np.array_equal(out[1], out[2])


def test_c2_sampling_dex_equals_ar(P, c2):
    """Sampling-mode DECS at the 7B shape: GPU DEX stream == GPU AR stream (same Gumbel rows), differs from greedy."""
    import dex_synth
    wl, w = c2
    p = dex_synth.make_prompt(wl.shape.vocab, 64, wl.prompt_seed)
    T = 32
    out = {}
    for name, X, kw in (("ar", (wl.shape.n_layers,), dict(sample=1, temperature=1.0, sample_seed=5)),
                        ("dex", wl.depths, dict(sample=1, temperature=1.0, sample_seed=5)),
                        ("greedy", wl.depths, dict())):
        d = P.Dex(wl.shape, w, X, max_ctx=128, **kw)
        d.prefill(0, p)
        out[name], _ = d.generate(T)
        d.close()
    assert np.array_equal(out["dex"], out["ar"])
    assert not np.array_equal(out["dex"], out["greedy"])


def test_c2_adapter_dex_equals_ar(P, c2):
    """Inducing-adapter exits at the 7B shape in the launch configuration bench.py times: the committed stream is the
    GPU AR stream whatever the adapters propose; strong random adapters change the round count."""
    import dex_synth
    wl, w = c2
    p = dex_synth.make_prompt(wl.shape.vocab, 64, wl.prompt_seed)
    T = 32
    ad = dex_synth.make_adapters(wl.shape, len(wl.depths) - 1, seed=7, alpha=0.5)
    out = {}
    for name, X, adapters in (("ar", (wl.shape.n_layers,), None), ("plain", wl.depths, None), ("ad", wl.depths, ad)):
        d = P.Dex(wl.shape, w, X, max_ctx=128, adapters=adapters)
        d.prefill(0, p)
        toks, recs = d.generate(T)
        out[name] = (toks, len(recs))
        d.close()
    assert np.array_equal(out["ad"][0], out["ar"][0]) and np.array_equal(out["plain"][0], out["ar"][0])
    assert out["ad"][1] != out["plain"][1]
