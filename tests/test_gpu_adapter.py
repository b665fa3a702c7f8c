"""Inducing-adapter exits (App. C.2) through the C ABI against the oracle: every new node's
candidate token (a flip only at an oracle top-2 margin < 1e-2 of that node, R17), the stage-boundary hidden state
(which the adapter must NOT touch), the commit rule and losslessness (GPU DEX stream == GPU AR
stream, bit-identical); gate alpha = 0 must reproduce the adapter-free run exactly."""
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


def _adapters(shape, n_ad, m=0, seed=99):
    """Synthetic adapters with per-depth gates and a non-trivial RMSNorm scale (so a wrong adapter index shows)."""
    import dex_synth
    import torch
    ad = dex_synth.make_adapters(shape, n_ad, seed=seed, alpha=0.5, m=m)
    gen = torch.Generator().manual_seed(seed)
    ad["norm"] = 1.0 + 0.2 * torch.randn(ad["norm"].shape, generator=gen)
    ad["alpha"] = 0.3 + 0.5 * torch.rand(ad["alpha"].shape, generator=gen)
    return ad


@pytest.mark.parametrize("rk", [1, 2])
@pytest.mark.parametrize("X,m", [((2, 4, 6, 8), 0), ((4, 8), 0), ((1, 3, 4, 8), 128), (tuple(range(1, 9)), 0)])
def test_c1_adapter_exits_match_oracle(P, c1, X, m, rk):
    """Every round of a 24-token run (tests/trace_util.py: the oracle replays with the GPU's exit decisions forced)."""
    import dex_synth
    from oracle import OracleModel, ar_greedy, dex_decode
    from trace_util import gpu_trace, compare_with_oracle
    wl, w, p = c1
    T = 24
    ad = _adapters(wl.shape, len(X) - 1, m=m)
    om = OracleModel(wl.shape, w, kv_round="bf16", adapters=ad)
    od = dex_decode(om, p, T, X, trace=True)
    plain = dex_decode(OracleModel(wl.shape, w, kv_round="bf16"), p, T, X, trace=True)
    ar = ar_greedy(om, p, T)
    assert np.array_equal(od["tokens"], ar["tokens"])                   # lossless with adapters
    assert [r["u"] for r in od["rounds"]] != [r["u"] for r in plain["rounds"]]   # ... and they do act
    g = P.Dex(wl.shape, w, X, max_ctx=128, debug_taps=1, use_graph=0, adapters=ad, round_kernel=rk)
    g.prefill(0, p)
    recs = gpu_trace(g, T)
    dex_tokens = g.tokens()[len(p):len(p) + T]
    g.close()
    res = compare_with_oracle(recs, om, p, X, T)
    assert res["rounds"] == len(recs) >= T and res["nodes"] > 20
    a = P.Dex(wl.shape, w, (wl.shape.n_layers,), max_ctx=128, round_kernel=rk)
    a.prefill(0, p)
    ar_gpu, _ = a.generate(T)
    a.close()
    assert np.array_equal(ar_gpu, dex_tokens)                           # H3: the adapters never change the stream


def test_gate_zero_is_bit_identical_to_no_adapter(P, c1):
    import dex_synth
    wl, w, p = c1
    X = (2, 4, 6, 8)
    ad = dex_synth.make_adapters(wl.shape, 3, seed=5, alpha=0.0)
    runs = []
    for adapters in (None, ad):
        g = P.Dex(wl.shape, w, X, max_ctx=128, debug_taps=1, use_graph=0, adapters=adapters)
        g.prefill(0, p)
        Bs = []
        for _ in range(30):
            r = g.step()[0]
            Bs.append((g.tap_B().tolist(), r.token, r.match_k, r.ref_top1))
        runs.append(Bs)
        g.close()
    assert runs[0] == runs[1]


def test_adapter_graph_replay_batched_and_rounds_change(P, c1):
    """Launch configuration of bench.py (graph replay, auto-collapse) with two sequences: each stream equals its
    single-sequence stream; the adapters change how many rounds a token takes, never the tokens."""
    import dex_synth
    wl, w, p = c1
    X = (2, 4, 6, 8)
    T = 40
    ad = _adapters(wl.shape, 3)
    p2 = dex_synth.make_prompt(wl.shape.vocab, 21, 77)
    single = {}
    for name, adapters in (("plain", None), ("ad", ad)):
        g = P.Dex(wl.shape, w, X, max_ctx=128, adapters=adapters)
        g.prefill(0, p)
        toks, recs = g.generate(T)
        single[name] = (toks, len(recs))
        g.close()
    assert np.array_equal(single["plain"][0], single["ad"][0])
    assert single["plain"][1] != single["ad"][1]
    g = P.Dex(wl.shape, w, X, max_seqs=2, max_ctx=128, adapters=ad)
    g.prefill(0, p)
    g.prefill(1, p2)
    for _ in range(4 * T):
        g.step()
    t0 = g.tokens(0)[len(p):len(p) + T]
    t1 = g.tokens(1)[len(p2):len(p2) + T]
    g.close()
    assert np.array_equal(t0, single["ad"][0])
    s = P.Dex(wl.shape, w, X, max_ctx=128, adapters=ad)
    s.prefill(0, p2)
    ref1, _ = s.generate(T)
    s.close()
    assert np.array_equal(t1, ref1)


def test_adapter_argument_checks(P, c1):
    import dex_synth
    wl, w, _ = c1
    ad = dex_synth.make_adapters(wl.shape, 1, seed=1)
    with pytest.raises(P.DexError):                                     # per-op path has no adapter ops
        P.Dex(wl.shape, w, (4, 8), max_ctx=64, adapters=ad, round_kernel=0)
    with pytest.raises(ValueError):                                     # one adapter per non-final depth
        P.Dex(wl.shape, w, (2, 4, 8), max_ctx=64, adapters=ad)
    bad = dex_synth.make_adapters(wl.shape, 1, seed=1, m=96)            # not a multiple of 64
    with pytest.raises(P.DexError):
        P.Dex(wl.shape, w, (4, 8), max_ctx=64, adapters=bad)
    wide = dex_synth.make_adapters(wl.shape, 1, seed=1, m=(wl.shape.d_ffn // 64 + 1) * 64)
    with pytest.raises(P.DexError):
        P.Dex(wl.shape, w, (4, 8), max_ctx=64, adapters=wide)
