"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element on
the same seeded inputs.  Tolerances are BASELINE.json:north_star's: per-layer hidden states
max relative error 2e-2 (per row vector: max|g-o| / max|o|, reading R16), logits max abs 5e-2,
token streams identical except where the oracle's top-2 margin < 1e-2 (flagged, counted and
teacher-forced, reading R17); GPU DEX stream bit-identical to GPU AR stream.
Integer work (lattice tables, B, match index, counters) is compared bit-exactly."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

HID_TOL, LOGIT_TOL, MARGIN = 2e-2, 5e-2, 1e-2


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
    """Oracle on the bf16-rounded weights with a bf16 KV cache (what the GPU path stores)."""
    from oracle import OracleModel
    wl, w, p = c1
    return OracleModel(wl.shape, w, kv_round="bf16")


def rel_err(g, o):
    return float(np.abs(g - o).max() / np.abs(o).max())


def gpu_generate_forced(P, dex, oracle_tokens, margins, T):
    """R17: run T commits; a mismatch at an oracle margin < 1e-2 is counted and the oracle's
    token is forced through dex_collapse; any other mismatch fails."""
    out, flagged, recs = [], 0, []
    while len(out) < T:
        r = dex.step(0)[0]          # no auto-collapse: commit through the primitive
        rec = dict(q=r.q_before, rows=list(r.rows_per_stage), evals=r.layer_evals, crit=r.critical_layers,
                   anchor=list(r.anchor_tokens), exit_rows=r.exit_rows)
        recs.append(rec)
        if r.match_k < 0:
            continue
        t = len(out)
        tok, k = r.token, r.match_k
        if tok != oracle_tokens[t]:
            assert margins[t] < MARGIN, f"token {t}: gpu {tok} != oracle {oracle_tokens[t]} at margin {margins[t]:.4f}"
            flagged += 1
            tok = int(oracle_tokens[t])
            N = len(dex.depths)
            k = next((i for i in range(N - 1) if rec["anchor"][i] == tok), N - 1)
        rec.update(token=tok, k=k)
        dex.collapse(0, k, tok)
        out.append(tok)
    return np.array(out), flagged, recs


# ------------------------------------------------------------------------------------------
def test_gemm_matches_definition(P, c1):
    """T2: the tcgen05/TMA weight-streaming GEMM against Y = X W^T in float64, for all four
    projections, rows spanning one box, several boxes and a ragged tail; ffn = 688 gives a
    ragged K tail (down) and a ragged out tile (gate/up)."""
    wl, w, _ = c1
    d = P.Dex(wl.shape, w, (8,), max_ctx=256, debug_taps=1, use_graph=0)
    rng = np.random.default_rng(7)
    for which, name in enumerate(("wqkv", "wo", "wgu", "wdn")):
        for layer in (0, 5):
            W = w[name][layer].float().numpy().astype(np.float64).reshape(-1, w[name].shape[-1])
            for rows in (1, 8, 16, 37, 128):
                x = rng.standard_normal((rows, W.shape[1])).astype(np.float32)
                y = d.gemm(which, layer, x)
                ref = x.astype(np.float64) @ W.T
                assert rel_err(y, ref) < 2e-5, (name, layer, rows)
    d.close()


def test_gemm_single_plane_is_bf16_rounded_input(P, c1):
    """act_planes = 1 feeds bf16(x): must equal the definition applied to the rounded input."""
    import dex_synth
    wl, w, _ = c1
    d = P.Dex(wl.shape, w, (8,), max_ctx=256, debug_taps=1, use_graph=0, act_planes=1)
    rng = np.random.default_rng(8)
    W = w["wqkv"][2].float().numpy().astype(np.float64)
    x = rng.standard_normal((19, 256)).astype(np.float32)
    y = d.gemm(0, 2, x)
    ref = dex_synth.bf16_round_f32(x).astype(np.float64) @ W.T
    assert rel_err(y, ref) < 2e-5
    d.close()


@pytest.mark.parametrize("rk", [1, 0, 2])
def test_c1_ar_hidden_logits_tokens(P, c1, c1_bf16, rk):
    """T3 on config c1 with X = {L} (the AR baseline): every layer's hidden state, the final logits - both the
    debug recompute and the fused exit's OWN per-block maxima (tcgen05 accumulators, DEX_TAP_REF_BLOCKS) - and the
    token stream against oracle AR greedy.  Teacher-forced (R17): a token that differs at an oracle margin < 1e-2
    is counted and the oracle's token is committed, so all T positions are always compared."""
    from oracle import ar_greedy
    from trace_util import check_ref_blocks
    wl, w, p = c1
    T = wl.gen_len
    ar = ar_greedy(c1_bf16, p, T, keep_hidden=True, keep_logits=True)
    margins = np.array(ar["top1"]) - np.array(ar["top2"])
    d = P.Dex(wl.shape, w, (wl.shape.n_layers,), max_ctx=128, debug_taps=1, use_graph=0, round_kernel=rk)
    d.prefill(0, p)
    assert d.tap_fsm().tolist() == [0, len(p) - 1, len(p), 0]
    worst_h = worst_l = worst_b = 0.0
    flagged = 0
    for t in range(T):
        r = d.step(0)[0]
        assert r.committed == 0 and r.match_k == 0 and r.q_before == 0
        assert r.layer_evals == wl.shape.n_layers and r.exit_rows == 1
        h = d.tap_hidden(0)
        for l in range(wl.shape.n_layers):
            worst_h = max(worst_h, rel_err(h[l], ar["hidden"][t][l]))
        lg = d.tap_logits()
        worst_l = max(worst_l, float(np.abs(lg - ar["logits"][t]).max()))
        worst_b = max(worst_b, check_ref_blocks(d.tap_ref_blocks(), ar["logits"][t]))
        assert abs(r.ref_top1 - ar["top1"][t]) < LOGIT_TOL and abs(r.ref_top2 - ar["top2"][t]) < LOGIT_TOL
        if r.token != ar["tokens"][t]:
            assert margins[t] < MARGIN, (t, r.token, ar["tokens"][t], margins[t])
            flagged += 1
        d.collapse(0, 0, int(ar["tokens"][t]))
    assert worst_h < HID_TOL, worst_h
    assert worst_l < LOGIT_TOL and worst_b < LOGIT_TOL, (worst_l, worst_b)
    assert flagged <= 2, flagged
    assert np.array_equal(d.tokens()[len(p):], ar["tokens"])
    d.close()


@pytest.mark.parametrize("rk", [1, 0, 2])
@pytest.mark.parametrize("decs", [0, 1])
@pytest.mark.parametrize("X", [(2, 4, 6, 8), (4, 8), (3, 8), (1, 3, 4, 8), tuple(range(1, 9))])
def test_c1_dex_matches_oracle(P, c1, c1_bf16, decs, X, rk):
    """T3/T4 on c1: EVERY round of a 32-token DEX run against the oracle's Alg. 1 trace (tests/trace_util.py: the GPU
    runs free, the oracle replays with the GPU's exit decisions forced; a forced decision must be a near-tie of the
    oracle's logits): nodes expanded, rows per stage / layer evaluations / critical layers (bit-exact), every new
    node's candidate token and stage-boundary hidden state, every commit (token, branch b_k, anchor top-2 logits, FSM
    state after the collapse); then the GPU DEX stream against the GPU AR stream (bit-identical)."""
    from oracle import ar_greedy
    from trace_util import gpu_trace, compare_with_oracle
    wl, w, p = c1
    T = 32
    g = P.Dex(wl.shape, w, X, max_ctx=128, debug_taps=1, use_graph=0, decs=decs, round_kernel=rk)
    g.prefill(0, p)
    recs = gpu_trace(g, T)
    dex_tokens = g.tokens()[len(p):len(p) + T]
    g.close()
    res = compare_with_oracle(recs, c1_bf16, p, X, T, decs=bool(decs))
    assert res["rounds"] == len(recs) >= T and res["nodes"] >= T                         # coverage: every round, every node
    assert np.array_equal(res["tokens"], dex_tokens)
    # the oracle's free-running AR stream may differ from the GPU's only at a near-tie of the final-depth logits
    ar = ar_greedy(c1_bf16, p, T)
    bad = np.nonzero(dex_tokens != ar["tokens"])[0]
    if len(bad):
        assert ar["top1"][bad[0]] - ar["top2"][bad[0]] < MARGIN, (bad[0],)
    a = P.Dex(wl.shape, w, (wl.shape.n_layers,), max_ctx=128, decs=decs, round_kernel=rk)
    a.prefill(0, p)
    ar_gpu, _ = a.generate(T)
    a.close()
    assert np.array_equal(ar_gpu, dex_tokens)                    # H3: bit-identical streams


@pytest.mark.parametrize("rk", [1, 0, 2])
def test_c1_full_run_graph_replay_and_counts(P, c1, c1_bf16, rk):
    """The bench configuration of c1 (64 tokens, CUDA-graph replay, auto-collapse): tokens ==
    oracle, rounds and layer evaluations equal the closed forms of SURVEY 8(c)."""
    from oracle import dex_decode
    wl, w, p = c1
    od = dex_decode(c1_bf16, p, wl.gen_len, wl.depths, decs=True)
    g = P.Dex(wl.shape, w, wl.depths, max_ctx=128, use_graph=1, round_kernel=rk)
    g.prefill(0, p)
    toks, recs = g.generate(wl.gen_len)
    assert np.array_equal(toks, od["tokens"])
    ks = [r["match_k"] for r in recs if r["committed"]]
    assert ks == od["match_k"].tolist()
    N = len(wl.depths)
    assert len(recs) == od["n_rounds"] == N + sum(k + 1 for k in ks[:-1])
    assert sum(r["layer_evals"] for r in recs) == od["layer_evals"]
    assert sum(r["critical_layers"] for r in recs) == od["critical_layers"]
    g.close()


def test_forced_collapse_and_state_errors(P, c1, c1_bf16):
    """dex_collapse as a primitive: ESTATE / EINVAL behaviour and teacher forcing (R17) against
    the oracle run with the same forced tokens (fallback branch when no candidate matches)."""
    from oracle import dex_decode
    wl, w, p = c1
    X = wl.depths
    T = 10
    free = dex_decode(c1_bf16, p, T, X)["tokens"]
    forced = free.copy()
    forced[2] = (forced[2] + 7) % wl.shape.vocab          # tokens nobody proposed -> fallback b_{N-1}
    forced[5] = (forced[5] + 11) % wl.shape.vocab
    od = dex_decode(c1_bf16, p, T, X, force_tokens=forced)
    g = P.Dex(wl.shape, w, X, max_ctx=128, use_graph=1)
    with pytest.raises(P.DexError) as e:
        g.collapse(0, 0, 1)
    assert e.value.code == P.DEX_ESTATE                    # nothing prefetched / pending yet
    g.prefill(0, p)
    n = 0
    while n < T:
        r = g.step(0)[0]
        if r.match_k < 0:
            with pytest.raises(P.DexError) as e:
                g.collapse(0, 0, 1)
            assert e.value.code == P.DEX_ESTATE
            continue
        with pytest.raises(P.DexError) as e:               # a step while a commit is pending
            g.step(0)
        assert e.value.code == P.DEX_ESTATE
        tok = int(forced[n])
        anchor = list(r.anchor_tokens)[:len(X)]
        k = next((i for i in range(len(X) - 1) if anchor[i] == tok), len(X) - 1)
        if k != 0 and anchor[0] != tok:
            with pytest.raises(P.DexError) as e:
                g.collapse(0, 0, tok)
            assert e.value.code == P.DEX_EINVAL            # B[anchor(0)] != token
        g.collapse(0, k, tok)
        assert k == od["match_k"][n]
        n += 1
    assert np.array_equal(g.tokens()[len(p):], forced)
    g.close()


def test_batched_sequences_are_independent(P, c1):
    """R18: three lattices batched into the same launches (different prompt lengths, so their FSMs
    run out of phase) give exactly the streams they give alone."""
    import dex_synth
    wl, w, _ = c1
    prompts = [dex_synth.make_prompt(wl.shape.vocab, n, 99, s) for s, n in enumerate((16, 5, 150))]
    alone = []
    for p in prompts:
        g = P.Dex(wl.shape, w, wl.depths, max_ctx=256)
        g.prefill(0, p)
        alone.append(g.generate(20)[0])
        g.close()
    g = P.Dex(wl.shape, w, wl.depths, max_seqs=3, max_ctx=256, page_size=64)
    for s, p in enumerate(prompts):
        g.prefill(s, p)
    got = [[] for _ in prompts]
    while min(len(t) for t in got) < 20:
        res = g.step()
        for s in range(3):
            if res[s].committed and len(got[s]) < 20:
                got[s].append(res[s].token)
    for s in range(3):
        assert np.array_equal(got[s], alone[s]), s
    g.close()


def test_edges_prompt_len_one_ragged_prefill_pages_and_max_ctx(P, c1, c1_bf16):
    from oracle import ar_greedy
    wl, w, _ = c1
    import dex_synth
    # prompt of one token: nothing to prefill
    p1 = dex_synth.make_prompt(wl.shape.vocab, 1, 5)
    ar = ar_greedy(c1_bf16, p1, 12)
    g = P.Dex(wl.shape, w, wl.depths, max_ctx=64, page_size=64)
    g.prefill(0, p1)
    assert np.array_equal(g.generate(12)[0], ar["tokens"])
    g.close()
    # 150-token prompt: two prefill chunks with a ragged tail, pages of 64 crossed while decoding
    p2 = dex_synth.make_prompt(wl.shape.vocab, 150, 6)
    ar = ar_greedy(c1_bf16, p2, 50)
    margins = np.array(ar["top1"]) - np.array(ar["top2"])
    g = P.Dex(wl.shape, w, wl.depths, max_ctx=200, page_size=64)
    g.prefill(0, p2)
    toks, flagged, _ = gpu_generate_forced(P, g, ar["tokens"], margins, 50)
    assert np.array_equal(toks, ar["tokens"]) and flagged <= 2
    # max_ctx reached -> done, further steps are no-ops
    r = None
    for _ in range(200):
        r = g.step()[0]
        if r.done or not r.active:
            break
    assert r.done == 1 and r.n_tokens == 200
    assert g.step()[0].active == 0
    with pytest.raises(P.DexError) as e:
        g.prefill(0, np.zeros(201, dtype=np.int32))
    assert e.value.code == P.DEX_ECAPACITY
    g.close()


def test_sequence_prefilled_to_max_ctx_is_done_on_both_sides(P, c1):
    """a sequence whose prompt already fills max_ctx is done on the device as on the host mirror: it takes no
    part in the rounds (no rows, no layer evaluations) while the other sequence of the batch decodes its usual stream."""
    import dex_synth
    wl, w, p = c1
    full = dex_synth.make_prompt(wl.shape.vocab, 64, 9)
    alone = P.Dex(wl.shape, w, wl.depths, max_ctx=64)
    alone.prefill(0, p)
    want, _ = alone.generate(20)
    alone.close()
    g = P.Dex(wl.shape, w, wl.depths, max_seqs=2, max_ctx=64)
    g.prefill(0, full)                                       # n == max_ctx: nothing can be generated
    g.prefill(1, p)
    got = []
    while len(got) < 20:
        res = g.step()
        assert res[0].active == 0 and res[0].done == 1 and res[0].layer_evals == 0 and res[0].n_tokens == 64
        if res[1].committed:
            got.append(res[1].token)
    assert g.tap_fsm(0).tolist()[2] == 64                    # the device FSM did not move either
    assert np.array_equal(got, want)
    g.close()


def test_flow_kernel_more_attention_tasks_than_ctas(P, c1):
    """k_flow (round_kernel = 2) on a wide lattice with a long context: more attention tasks than CTAs.  Its CTAs run
    their tasks in order, each waiting for its head's QKV counter, so the tasks must be dealt stage-major; with
    k_round's heaviest-range-first deal this configuration deadlocked (round 2).  Streams must equal k_round's."""
    import dex_synth
    wl, w, _ = c1
    X = tuple(range(1, 9))
    p = dex_synth.make_prompt(wl.shape.vocab, 300, 17)
    out = {}
    for rk in (1, 2):
        g = P.Dex(wl.shape, w, X, max_ctx=360, page_size=64, round_kernel=rk)
        g.prefill(0, p)
        toks, recs = g.generate(24)
        out[rk] = (toks.tolist(), [r["match_k"] for r in recs])
        g.close()
    assert out[1] == out[2]


def test_256_row_single_plane_stages_run_the_round_kernel(P):
    """The c5 launch geometry (4 sequences x N = 8 -> 256-row stage 0, head_dim 128, act_planes = 1) must fit the round
    kernel's shared-memory ring: ONE segment-GEMM launch per round in the library's own counters (dex_profile), not the
    4 |Pi| launches of the per-op fallback - a budget change once made this fall back silently (round 2).  Also
    DEX == AR on that path."""
    import dex_synth
    sh = dex_synth.ModelShape("mini-hd128-8L", 8, 512, 4, 4, 128, 1024, 1000)
    w = dex_synth.make_weights(sh, 91)
    X, S = tuple(range(1, 9)), 4
    prompts = [dex_synth.make_prompt(sh.vocab, 40 + 7 * s, 92, seq=s) for s in range(S)]
    streams = {}
    for name, depths in (("dex", X), ("ar", (sh.n_layers,))):
        g = P.Dex(sh, w, depths, max_seqs=S, max_ctx=128, act_planes=1, page_size=64)
        for s in range(S):
            g.prefill(s, prompts[s])
        g.profile(0)
        got = [[] for _ in range(S)]
        rounds = 0
        while min(len(t) for t in got) < 10:
            res = g.step()
            rounds += 1
            for s in range(S):
                if res[s].committed and len(got[s]) < 10:
                    got[s].append(res[s].token)
        _, ct = g.profile(-1)
        assert ct[0] == rounds and ct[2] == rounds, (name, ct[:3].tolist(), rounds)   # one k_round launch per round
        streams[name] = got
        g.close()
    assert streams["dex"] == streams["ar"]


def test_gqa_headdim128_ragged_vocab(P):
    """A small GQA model with head_dim 128, a vocabulary that is not a multiple of the 128-row
    tile and d_ffn with ragged tiles: AR and DEX against the oracle (shape family of c4)."""
    import dex_synth
    from oracle import OracleModel, ar_greedy, dex_decode
    sh = dex_synth.ModelShape("mini-gqa", 6, 512, 4, 2, 128, 1000, 2001, rope_theta=5e5)
    w = dex_synth.make_weights(sh, 77)
    p = dex_synth.make_prompt(sh.vocab, 70, 78)
    om = OracleModel(sh, w, kv_round="bf16")
    T = 24
    ar = ar_greedy(om, p, T, keep_hidden=True, keep_logits=True)
    margins = np.array(ar["top1"]) - np.array(ar["top2"])
    a = P.Dex(sh, w, (6,), max_ctx=128, debug_taps=1, use_graph=0, page_size=64)
    a.prefill(0, p)
    r = a.step()[0]
    assert rel_err(a.tap_hidden(0)[-1], ar["hidden"][0][-1]) < HID_TOL
    assert np.abs(a.tap_logits() - ar["logits"][0]).max() < LOGIT_TOL
    a.close()
    for X in ((6,), (2, 4, 6), (1, 2, 3, 6)):
        g = P.Dex(sh, w, X, max_ctx=128, page_size=64)
        g.prefill(0, p)
        toks, flagged, _ = gpu_generate_forced(P, g, ar["tokens"], margins, T)
        assert np.array_equal(toks, ar["tokens"]) and flagged <= 1, X
        g.close()
    assert np.array_equal(dex_decode(om, p, T, (2, 4, 6))["tokens"], ar["tokens"])


@pytest.mark.parametrize("X", [(8,), (2, 4, 6, 8), (1, 3, 4, 8)])
def test_c1_sampling_mode_matches_oracle_and_is_lossless(P, c1, c1_bf16, X):
    """Sampling-mode DECS (Alg. 2 lines 10-15, reading R24): the GPU stream against the oracle's Gumbel-Max AR
    sampling with the same counter-based noise (a mismatch only where the oracle's top-2 margin of the PERTURBED
    final-depth logits is < 1e-2, then teacher-forced), and GPU DEX sampling == GPU AR sampling bit for bit."""
    from oracle import ar_sample
    wl, w, p = c1
    T, tau, seed = 32, 0.8, 77
    ar = ar_sample(c1_bf16, p, T, tau, seed)
    margins = np.array(ar["top1"]) - np.array(ar["top2"])
    g = P.Dex(wl.shape, w, X, max_ctx=128, sample=1, temperature=tau, sample_seed=seed)
    g.prefill(0, p)
    toks, flagged, _ = gpu_generate_forced(P, g, ar["tokens"], margins, T)
    assert np.array_equal(toks, ar["tokens"])
    assert flagged <= 2
    g.close()
    # losslessness on the GPU itself, free-running
    a = P.Dex(wl.shape, w, (wl.shape.n_layers,), max_ctx=128, sample=1, temperature=tau, sample_seed=seed)
    a.prefill(0, p)
    ar_gpu, _ = a.generate(T)
    a.close()
    g = P.Dex(wl.shape, w, X, max_ctx=128, sample=1, temperature=tau, sample_seed=seed)
    g.prefill(0, p)
    dex_gpu, recs = g.generate(T)
    g.close()
    assert np.array_equal(dex_gpu, ar_gpu)
    # the reported anchor top-1 is the perturbed logit
    z = [r["ref_top1"] for r in recs if r["committed"]]
    if np.array_equal(ar_gpu, ar["tokens"]):
        assert np.abs(np.array(z) - np.array(ar["top1"])).max() < 5e-2
    # a different seed gives a different stream; greedy differs too
    b = P.Dex(wl.shape, w, X, max_ctx=128, sample=1, temperature=tau, sample_seed=seed + 1)
    b.prefill(0, p)
    other, _ = b.generate(T)
    b.close()
    assert not np.array_equal(other, dex_gpu)


def test_sampling_mode_argument_checks(P, c1):
    wl, w, _ = c1
    with pytest.raises(P.DexError):
        P.Dex(wl.shape, w, (8,), max_ctx=64, sample=1, temperature=0.0)
    with pytest.raises(P.DexError):
        P.Dex(wl.shape, w, (8,), max_ctx=64, sample=1, temperature=1.0, round_kernel=0)
