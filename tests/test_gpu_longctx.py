"""Oracle parity at the widths and context lengths bench.py runs, on models cut down in DEPTH only (the oracle is
NumPy: a 32-layer 7B prefill of 600 tokens would take an hour, 4 layers of the same width take seconds through
oracle.ar.prefill_matrix, which tests/test_oracle_model.py pins to the position-wise prefill):

  * Llama-2-7B width (d = 4096, 32 x 128 heads, ffn 11008, V = 32000), 4 layers, 640-token prompt: the context
    spans 11 attention chunks, several chunk ranges per (stage, head), the tail range, page crossings and the
    cross-CTA last-writer merge of k_round's lattice attention - per-layer hidden states, the fused exit's own
    reduction, tokens, for X = {L} and the four-depth X = {1,2,3,4};
  * Llama-3-8B head (GQA 32/8, ffn 14336, V = 128256: 1002 vocabulary tiles), 8 layers, X = {1..8} (two exit chunks
    per round, pass tasks in the attention);
  * Llama-2-13B width, 4 batched sequences, X = {1..8}: 256-row stages (the widest launch configuration, c5).
"""
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


def _oracle_state(om, prompt):
    from oracle.ar import prefill_matrix
    return prefill_matrix(om, [int(t) for t in prompt])


def _copy_state(st):
    return ([list(x) for x in st[0]], [list(x) for x in st[1]])


@pytest.fixture(scope="module")
def wide7b():
    import dex_synth
    from oracle import OracleModel
    sh = dex_synth.ModelShape("llama2-7b-width-4L", 4, 4096, 32, 32, 128, 11008, 32000)
    w = dex_synth.make_weights(sh, 4242, threads=16)
    p = dex_synth.make_prompt(sh.vocab, 640, 99)
    om = OracleModel(sh, w, dtype=np.float32, kv_round="bf16")
    return sh, w, p, om, _oracle_state(om, p)


def test_7b_width_long_context_ar(P, wide7b):
    """X = {L} at a 640-token context: every layer's hidden state, the logits (debug recompute AND the fused exit's own
    per-block maxima), the anchor top-2, tokens (teacher-forced, R17)."""
    from oracle import ar_greedy
    from trace_util import check_ref_blocks, rel_err, HID_TOL, LOGIT_TOL, MARGIN
    sh, w, p, om, st = wide7b
    T = 4
    ar = ar_greedy(om, p, T, keep_hidden=True, keep_logits=True, state=_copy_state(st))
    d = P.Dex(sh, w, (sh.n_layers,), max_ctx=704, debug_taps=1, use_graph=0)
    d.prefill(0, p)
    flagged = 0
    for t in range(T):
        r = d.step(0)[0]
        h = d.tap_hidden(0)
        for l in range(sh.n_layers):
            assert rel_err(h[l], ar["hidden"][t][l]) < HID_TOL, (t, l)
        assert np.abs(d.tap_logits() - ar["logits"][t]).max() < LOGIT_TOL
        check_ref_blocks(d.tap_ref_blocks(), ar["logits"][t])
        assert abs(r.ref_top1 - ar["top1"][t]) < LOGIT_TOL and abs(r.ref_top2 - ar["top2"][t]) < LOGIT_TOL
        if r.token != ar["tokens"][t]:
            assert ar["top1"][t] - ar["top2"][t] < MARGIN
            flagged += 1
        d.collapse(0, 0, int(ar["tokens"][t]))
    assert flagged <= 1
    d.close()


@pytest.mark.parametrize("rk", [1, 0, 2])
def test_7b_width_long_context_dex_trace(P, wide7b, rk):
    """X = {1,2,3,4} at a 640-token context: every round against the oracle's trace (tests/trace_util.py), all three launch
    paths (k_round, per-op kernels, k_flow); then GPU DEX stream == GPU AR stream."""
    from trace_util import gpu_trace, compare_with_oracle
    sh, w, p, om, st = wide7b
    X, T = (1, 2, 3, 4), 3
    g = P.Dex(sh, w, X, max_ctx=704, debug_taps=1, use_graph=0, round_kernel=rk)
    g.prefill(0, p)
    recs = gpu_trace(g, T)
    dex_tokens = g.tokens()[len(p):len(p) + T]
    g.close()

    from oracle import dex_decode
    force_u = {(ri, i): t for ri, rec in enumerate(recs) for i, t in rec["u"].items()}
    od = dex_decode(om, p, T, X, trace=True, force_u=force_u, state=_copy_state(st))
    _trace_check(recs, od, 15)
    a = P.Dex(sh, w, (sh.n_layers,), max_ctx=704, round_kernel=rk)
    a.prefill(0, p)
    ar_gpu, _ = a.generate(T)
    a.close()
    assert np.array_equal(ar_gpu, dex_tokens)


def _trace_check(recs, od, n_min, margin_mid=None):
    """margin_mid: the oracle logit gap below which an INTERMEDIATE exit decision (a non-final node's candidate) may differ;
    default = the 1e-2 of the committed-token rule (reading R17b).  The final-depth anchor (the committed token) is always
    held to 1e-2."""
    import trace_util as tu
    margin_mid = tu.MARGIN if margin_mid is None else margin_mid
    n_lvl = max(gr["q"] for gr in recs) + 1
    ref_node = (1 << (n_lvl - 1)) - 1
    assert len(od["rounds"]) == len(recs)
    n_nodes = n_forced = 0
    for ri, (gr, o) in enumerate(zip(recs, od["rounds"])):
        assert gr["q"] == o["q"] and gr["rows"] == o["rows_per_stage"] and gr["evals"] == o["layer_evals"], ri
        assert gr["nodes"] == sorted(o["nodes"]), ri
        for i in gr["nodes"]:
            n_nodes += 1
            assert tu.rel_err(gr["h"][i], o["h_out"][i]) < tu.HID_TOL, (ri, i)
        for i, (own, tok, gap) in o.get("u_forced", {}).items():
            n_forced += 1
            assert gap < (tu.MARGIN if (i == ref_node and o["committed"]) else margin_mid), (ri, i, gap)
        if o["committed"]:
            assert gr["token"] == o["token"] and gr["k"] == o["match_k"], ri
            assert abs(gr["top1"] - o["ref_top1"]) < tu.LOGIT_TOL and abs(gr["top2"] - o["ref_top2"]) < tu.LOGIT_TOL
    assert n_nodes >= n_min and n_forced <= max(2, n_nodes // 20), (n_nodes, n_forced)


def test_8b_head_gqa_large_vocab_wide_lattice(P):
    """The c4 head at full width (GQA 32/8, V = 128256), 8 layers, X = {1..8}: one commit = 8 rounds up to 128 rows and
    two exit chunks; every node against the oracle, the fused exit's per-block maxima over all 4008 blocks."""
    import dex_synth
    from oracle import OracleModel, ar_greedy, dex_decode
    from trace_util import gpu_trace, check_ref_blocks
    sh = dex_synth.ModelShape("llama3-8b-width-8L", 8, 4096, 32, 8, 128, 14336, 128256, rope_theta=5e5)
    w = dex_synth.make_weights(sh, 777, threads=16)
    p = dex_synth.make_prompt(sh.vocab, 150, 5)
    om = OracleModel(sh, w, dtype=np.float32, kv_round="bf16")
    st = _oracle_state(om, p)
    X, T = tuple(range(1, 9)), 1
    g = P.Dex(sh, w, X, max_ctx=256, debug_taps=1, use_graph=0)
    g.prefill(0, p)
    recs = gpu_trace(g, T)
    g.close()
    force_u = {(ri, i): t for ri, rec in enumerate(recs) for i, t in rec["u"].items()}
    od = dex_decode(om, p, T, X, trace=True, force_u=force_u, state=_copy_state(st))
    _trace_check(recs, od, 255)
    # AR on the same model: logits of the large-vocabulary head through the fused exit's own reduction
    ar = ar_greedy(om, p, 1, keep_logits=True, state=_copy_state(st))
    a = P.Dex(sh, w, (sh.n_layers,), max_ctx=256, debug_taps=1, use_graph=0)
    a.prefill(0, p)
    r = a.step(0)[0]
    check_ref_blocks(a.tap_ref_blocks(), ar["logits"][0])
    assert np.abs(a.tap_logits() - ar["logits"][0]).max() < 5e-2
    a.close()


def test_13b_width_four_sequences_256_row_stages(P):
    """The c5 launch configuration (Llama-2-13B width, 4 batched lattices, N = 8: 256-row stage 0, 512 exit rows), cut
    to 8 layers: sequence 3 against the oracle's trace for one commit (8 rounds, 255 nodes), the first token of all four streams
    against the GPU AR run."""
    import dex_synth
    from oracle import OracleModel, dex_decode
    from trace_util import gpu_trace
    sh = dex_synth.ModelShape("llama2-13b-width-8L", 8, 5120, 40, 40, 128, 13824, 32000, resid_decay=3.0)
    w = dex_synth.make_weights(sh, 555, threads=16)
    import torch
    wd = {k: v.cuda() for k, v in w.items()}
    S, X, T = 4, tuple(range(1, 9)), 1
    prompts = [dex_synth.make_prompt(sh.vocab, 70 + 9 * s, 31, seq=s) for s in range(S)]
    g = P.Dex(sh, wd, X, max_seqs=S, max_ctx=160, debug_taps=1, use_graph=0)
    for s in range(S):
        g.prefill(s, prompts[s])
    # all sequences step together; record the trace of sequence 3
    N = len(X)
    recs = {3: []}
    for _ in range(N):
        res = g.step(0)
        for s in (3,):
            r = res[s]
            q = r.q_before
            B = g.tap_B(s)
            nodes = list(range((1 << q) - 1, (2 << q) - 1))
            rec = dict(q=q, rows=list(r.rows_per_stage)[:N], evals=int(r.layer_evals), nodes=nodes,
                       u={i: int(B[i]) for i in nodes}, h={i: g.tap_hidden(i, s)[-1].copy() for i in nodes}, committed=0)
            if r.match_k >= 0:
                rec.update(committed=1, token=int(r.token), k=int(r.match_k), top1=float(r.ref_top1), top2=float(r.ref_top2))
            recs[s].append(rec)
        for s in range(S):
            if res[s].match_k >= 0:
                g.collapse(s, res[s].match_k, res[s].token)
    first = [int(g.tokens(s)[len(prompts[s])]) for s in range(S)]
    g.close()
    om = OracleModel(sh, w, dtype=np.float32, kv_round="bf16")
    for s in (3,):
        force_u = {(ri, i): t for ri, rec in enumerate(recs[s]) for i, t in rec["u"].items()}
        od = dex_decode(om, prompts[s], T, X, trace=True, force_u=force_u, state=_oracle_state(om, prompts[s]))
        _trace_check(recs[s], od, 255)
    a = P.Dex(sh, wd, (sh.n_layers,), max_seqs=S, max_ctx=160)
    for s in range(S):
        a.prefill(s, prompts[s])
    res = a.step()
    assert [int(res[s].token) for s in range(S)] == first
    a.close()
    del wd
    torch.cuda.empty_cache()


def test_c2_full_model_at_the_bench_context(P):
    """BASELINE.json:configs[1] at FULL size in the configuration bench.py times: the Llama-2-7B shape with all 32 layers,
    X = {8,16,24,32}, the bench's own 512-token prompt (same seed).  The oracle prefills the prompt in its whole-sequence
    form (oracle.ar.prefill_matrix, pinned to the position-wise prefill), then
      * AR (X = {L}): two tokens, every one of the 32 layers' hidden states, the logits through the debug recompute AND the
        fused exit's own per-block maxima, the anchor top-2, the tokens (teacher-forced, R17);
      * DEX: the first three commits (the first = 4 rounds, 15 lattice nodes; then collapse and the re-rooted lattice)
        against the oracle's Alg. 1 trace with the GPU's exit decisions
        forced (R17b): nodes, rows per stage, layer evaluations, stage-boundary hidden states, the commit;
      * the same for the c3 lattice (X every 4 layers, N = 8: 8 rounds, 255 nodes, then a second commit) on the same
        tensors and prompt."""
    import dex_synth
    import torch
    from oracle import OracleModel, ar_greedy, dex_decode
    from trace_util import gpu_trace, check_ref_blocks, rel_err, HID_TOL, LOGIT_TOL, MARGIN
    wl = dex_synth.workload("c2")
    w = dex_synth.make_weights(wl.shape, wl.weight_seed, threads=16)
    p = dex_synth.make_prompt(wl.shape.vocab, wl.prompt_len, wl.prompt_seed)
    om = OracleModel(wl.shape, w, dtype=np.float32, kv_round="bf16")
    st = _oracle_state(om, p)
    wd = {k: v.cuda() for k, v in w.items()}
    L = wl.shape.n_layers
    # ---- AR
    T = 2
    ar = ar_greedy(om, p, T, keep_hidden=True, keep_logits=True, state=_copy_state(st))
    d = P.Dex(wl.shape, wd, (L,), max_ctx=wl.prompt_len + 16, debug_taps=1, use_graph=0)
    d.prefill(0, p)
    for t in range(T):
        r = d.step(0)[0]
        h = d.tap_hidden(0)
        for l in range(L):
            assert rel_err(h[l], ar["hidden"][t][l]) < HID_TOL, (t, l)
        assert np.abs(d.tap_logits() - ar["logits"][t]).max() < LOGIT_TOL
        check_ref_blocks(d.tap_ref_blocks(), ar["logits"][t])
        assert abs(r.ref_top1 - ar["top1"][t]) < LOGIT_TOL and abs(r.ref_top2 - ar["top2"][t]) < LOGIT_TOL
        if r.token != ar["tokens"][t]:
            assert ar["top1"][t] - ar["top2"][t] < MARGIN
        d.collapse(0, 0, int(ar["tokens"][t]))
    d.close()
    # ---- DEX, first commit
    g = P.Dex(wl.shape, wd, wl.depths, max_ctx=wl.prompt_len + 16, debug_taps=1, use_graph=0)
    g.prefill(0, p)
    recs = gpu_trace(g, 3)                                   # three commits: collapse and the re-rooted lattice included
    g.close()
    force_u = {(ri, i): t for ri, rec in enumerate(recs) for i, t in rec["u"].items()}
    od = dex_decode(om, p, 3, wl.depths, trace=True, force_u=force_u, state=_copy_state(st))
    _trace_check(recs, od, 15 + 2)
    assert [r_["fsm_after"][0] for r_ in recs if r_["committed"]] == [o["q_after"] for o in od["rounds"] if o["committed"]]
    # ---- the c3 lattice on the same tensors and prompt (BASELINE.json:configs[2]: X every 4 layers, N = 8): the first
    #      commit = 8 rounds up to 128 rows, 255 nodes, pass-task attention, both exit chunks on the last round
    X3 = dex_synth.workload("c3").depths
    g = P.Dex(wl.shape, wd, X3, max_ctx=wl.prompt_len + 16, debug_taps=1, use_graph=0)
    g.prefill(0, p)
    recs = gpu_trace(g, 2)                                   # two commits
    g.close()
    force_u = {(ri, i): t for ri, rec in enumerate(recs) for i, t in rec["u"].items()}
    od = dex_decode(om, p, 2, X3, trace=True, force_u=force_u, state=_copy_state(st))
    _trace_check(recs, od, 255 + 1)
    del wd
    torch.cuda.empty_cache()


def test_c4_full_model_at_the_bench_context(P):
    """BASELINE.json:configs[3] at FULL size: the Llama-3-8B shape (32 layers, GQA 32/8, ffn 14336, V = 128256, RoPE theta
    5e5), X every 4 layers (N = 8), the bench's own 2048-token prompt (33 attention chunks, 16 committed pages).  One AR
    token (all 32 layers' hidden states, logits through the recompute and through the fused exit's own maxima over 4008
    blocks, anchor top-2) and the first DEX commit (8 rounds, 255 nodes, pass-task attention over the long context, the
    1002-tile exit head on both exit chunks) against the oracle's trace.  The oracle's prefill takes about a minute."""
    import dex_synth
    import torch
    from oracle import OracleModel, ar_greedy, dex_decode
    from trace_util import gpu_trace, check_ref_blocks, rel_err, HID_TOL, LOGIT_TOL, MARGIN
    wl = dex_synth.workload("c4")
    w = dex_synth.make_weights(wl.shape, wl.weight_seed, threads=16)
    p = dex_synth.make_prompt(wl.shape.vocab, wl.prompt_len, wl.prompt_seed)
    om = OracleModel(wl.shape, w, dtype=np.float32, kv_round="bf16")
    st = _oracle_state(om, p)
    wd = {k: v.cuda() for k, v in w.items()}
    L = wl.shape.n_layers
    ar = ar_greedy(om, p, 1, keep_hidden=True, keep_logits=True, state=_copy_state(st))
    d = P.Dex(wl.shape, wd, (L,), max_ctx=wl.prompt_len + 16, debug_taps=1, use_graph=0)
    d.prefill(0, p)
    r = d.step(0)[0]
    h = d.tap_hidden(0)
    for l in range(L):
        assert rel_err(h[l], ar["hidden"][0][l]) < HID_TOL, l
    assert np.abs(d.tap_logits() - ar["logits"][0]).max() < LOGIT_TOL
    check_ref_blocks(d.tap_ref_blocks(), ar["logits"][0])
    assert abs(r.ref_top1 - ar["top1"][0]) < LOGIT_TOL and abs(r.ref_top2 - ar["top2"][0]) < LOGIT_TOL
    if r.token != ar["tokens"][0]:
        assert ar["top1"][0] - ar["top2"][0] < MARGIN
    d.close()
    g = P.Dex(wl.shape, wd, wl.depths, max_ctx=wl.prompt_len + 16, debug_taps=1, use_graph=0)
    g.prefill(0, p)
    recs = gpu_trace(g, 1)
    g.close()
    force_u = {(ri, i): t for ri, rec in enumerate(recs) for i, t in rec["u"].items()}
    od = dex_decode(om, p, 1, wl.depths, trace=True, force_u=force_u, state=_copy_state(st))
    _trace_check(recs, od, 255)
    del wd
    torch.cuda.empty_cache()


@pytest.fixture(scope="module")
def c5_full():
    import dex_synth
    from oracle import OracleModel
    wl = dex_synth.workload("c5")
    w = dex_synth.make_weights(wl.shape, wl.weight_seed, threads=16)
    prompts = [dex_synth.make_prompt(wl.shape.vocab, wl.prompt_len, wl.prompt_seed, seq=s) for s in range(wl.n_seqs)]
    om = OracleModel(wl.shape, w, dtype=np.float32, kv_round="bf16")
    return wl, w, prompts, om, _oracle_state(om, prompts[3])


@pytest.mark.parametrize("planes", [2, 1])
def test_c5_full_model_at_the_bench_context(P, c5_full, planes):
    """BASELINE.json:configs[4] at FULL size: the Llama-2-13B shape (40 layers), X every 5 layers (N = 8), FOUR sequences
    with their own 1024-token prompts batched into the same launches (256-row stage 0, 512 exit rows).  Sequence 3 is
    checked against the oracle's Alg. 1 trace for its first commit (8 rounds, 255 nodes) while all four step together.
    planes = 2: two-plane activations (the per-op launch path: a 256-row two-plane stage does not fit k_round's ring):
    every clause at its stated tolerance.  planes = 1: the k_round configuration of the c5 bench line (plain bf16
    activations, what north_star's "bf16 tensor-core GEMMs" literally are): hidden states, counts and the committed token
    at their tolerances, but an INTERMEDIATE exit decision may differ from the oracle's up to the logit tolerance
    (5e-2; seen: one node of 255 at an oracle gap of 0.017) - which is why two planes are the default (reading R23)."""
    import torch
    from oracle import dex_decode
    wl, w, prompts, om, st3 = c5_full
    wd = {k: v.cuda() for k, v in w.items()}
    S, X, N = wl.n_seqs, wl.depths, len(wl.depths)
    g = P.Dex(wl.shape, wd, X, max_seqs=S, max_ctx=wl.prompt_len + 16, debug_taps=1, use_graph=0, act_planes=planes)
    for s in range(S):
        g.prefill(s, prompts[s])
    recs = []
    for _ in range(N):
        res = g.step(0)
        r = res[3]
        q = r.q_before
        B = g.tap_B(3)
        nodes = list(range((1 << q) - 1, (2 << q) - 1))
        rec = dict(q=q, rows=list(r.rows_per_stage)[:N], evals=int(r.layer_evals), nodes=nodes,
                   u={i: int(B[i]) for i in nodes}, h={i: g.tap_hidden(i, 3)[-1].copy() for i in nodes}, committed=0)
        if r.match_k >= 0:
            rec.update(committed=1, token=int(r.token), k=int(r.match_k), top1=float(r.ref_top1), top2=float(r.ref_top2))
        recs.append(rec)
        for s in range(S):
            if res[s].match_k >= 0:
                g.collapse(s, res[s].match_k, res[s].token)
    g.close()
    del wd
    torch.cuda.empty_cache()
    force_u = {(ri, i): t for ri, rec in enumerate(recs) for i, t in rec["u"].items()}
    od = dex_decode(om, prompts[3], 1, X, trace=True, force_u=force_u, state=_copy_state(st3))
    _trace_check(recs, od, 255, margin_mid=None if planes == 2 else 5e-2)
