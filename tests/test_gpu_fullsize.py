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
    for t in range(T):
        r = d.step()[0]
        h = d.tap_hidden(0)
        for l in range(wl.shape.n_layers):
            assert np.abs(h[l] - ar["hidden"][t][l]).max() / np.abs(ar["hidden"][t][l]).max() < 2e-2
        assert np.abs(d.tap_logits() - ar["logits"][t]).max() < 5e-2
        if ar["top1"][t] - ar["top2"][t] >= 1e-2:
            assert r.token == ar["tokens"][t]
        if r.token != ar["tokens"][t]:
            break
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
