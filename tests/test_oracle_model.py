"""Pins for oracle/model.py + oracle/ar.py (O1, O2): brute force, a library implementation
(Hugging Face LlamaForCausalLM on the same tensors), and a closed form."""
import numpy as np
import pytest

import dex_synth
from oracle import OracleModel, ar_greedy
from oracle.ar import prefill
from oracle.bruteforce import forward_nocache, logits_nocache
from oracle.model import bf16_round, rmsnorm, rope


def test_cached_path_equals_cachefree_bruteforce(c1, c1_model, c1_ar):
    wl, _, p = c1
    T = 12
    seq = list(p) + list(c1_ar["tokens"][:T])
    H = forward_nocache(c1_model, seq[:-1])            # [L+1, n, d]
    P = len(p)
    for t in range(T):
        # the t-th generated token was produced from position P-1+t
        want = H[1:, P - 1 + t, :]
        got = c1_ar["hidden"][t]
        assert np.max(np.abs(got - want)) < 1e-10
        lg = logits_nocache(c1_model, want[-1])
        assert np.max(np.abs(lg - c1_ar["logits"][t])) < 1e-10
        assert int(np.argmax(lg)) == c1_ar["tokens"][t]


def test_gqa_cached_equals_bruteforce():
    """Same check on a grouped-query shape (config c4 is GQA) with non-unit norm weights."""
    shp = dex_synth.ModelShape("gqa-mini", 3, 64, 8, 2, 8, 96, 50, rope_theta=5e5)
    w = dex_synth.make_weights(shp, 7, norm_jitter=0.2)
    m = OracleModel(shp, w)
    p = dex_synth.make_prompt(shp.vocab, 9, 3)
    ar = ar_greedy(m, p, 6, keep_hidden=True)
    seq = list(p) + list(ar["tokens"])
    H = forward_nocache(m, seq[:-1])
    for t in range(6):
        assert np.max(np.abs(ar["hidden"][t] - H[1:, len(p) - 1 + t])) < 1e-10


def test_against_huggingface_llama(c1, c1_model, c1_ar):
    """Library special case: transformers' LlamaForCausalLM loaded with the same tensors must
    give the same logits (pins reading R13: eps, rotate-half RoPE, untied head, SwiGLU order)."""
    torch = pytest.importorskip("torch")
    tr = pytest.importorskip("transformers")
    wl, w, p = c1
    s = wl.shape
    cfg = tr.LlamaConfig(vocab_size=s.vocab, hidden_size=s.d_model, intermediate_size=s.d_ffn,
                         num_hidden_layers=s.n_layers, num_attention_heads=s.n_heads,
                         num_key_value_heads=s.n_kv_heads, head_dim=s.head_dim, rms_norm_eps=s.rms_eps,
                         rope_theta=s.rope_theta, max_position_embeddings=256, tie_word_embeddings=False,
                         attention_bias=False, mlp_bias=False, hidden_act="silu")
    cfg._attn_implementation = "eager"
    hf = tr.LlamaForCausalLM(cfg).double().eval()
    nq, nk = s.n_heads * s.head_dim, s.n_kv_heads * s.head_dim
    sd = {"model.embed_tokens.weight": w["embed"], "lm_head.weight": w["lm_head"], "model.norm.weight": w["norm_final"]}
    for l in range(s.n_layers):
        pre = f"model.layers.{l}."
        sd[pre + "self_attn.q_proj.weight"] = w["wqkv"][l, :nq]
        sd[pre + "self_attn.k_proj.weight"] = w["wqkv"][l, nq:nq + nk]
        sd[pre + "self_attn.v_proj.weight"] = w["wqkv"][l, nq + nk:]
        sd[pre + "self_attn.o_proj.weight"] = w["wo"][l]
        sd[pre + "mlp.gate_proj.weight"] = w["wgu"][l, 0]
        sd[pre + "mlp.up_proj.weight"] = w["wgu"][l, 1]
        sd[pre + "mlp.down_proj.weight"] = w["wdn"][l]
        sd[pre + "input_layernorm.weight"] = w["norm_attn"][l]
        sd[pre + "post_attention_layernorm.weight"] = w["norm_ffn"][l]
    missing, unexpected = hf.load_state_dict({k: v.double() for k, v in sd.items()}, strict=False)
    assert not [m for m in missing if "rotary" not in m] and not unexpected
    T = 8
    seq = list(p) + list(c1_ar["tokens"][:T - 1])
    with torch.no_grad():
        out = hf(torch.tensor([seq], dtype=torch.long), output_hidden_states=True)
    P = len(p)
    for t in range(T):
        lg = out.logits[0, P - 1 + t].numpy()
        assert np.max(np.abs(lg - c1_ar["logits"][t])) < 1e-6   # HF keeps its rotary tables in fp32
        for l in range(1, s.n_layers):                  # HF hidden_states[L] is post-final-norm
            hs = out.hidden_states[l][0, P - 1 + t].numpy()
            assert np.max(np.abs(hs - c1_ar["hidden"][t][l - 1])) < 1e-6


def test_zero_residual_branches_closed_form(c1):
    """Wo = Wd = 0  =>  h_l = Embed[tok] at every depth l, so every exit decodes the same token."""
    wl, w, p = c1
    w0 = dict(w)
    w0["wo"] = w["wo"] * 0
    w0["wdn"] = w["wdn"] * 0
    m = OracleModel(wl.shape, w0)
    ar = ar_greedy(m, p, 5, keep_hidden=True)
    toks = list(p) + list(ar["tokens"])
    for t in range(5):
        e = m.embed[toks[len(p) - 1 + t]]
        assert np.array_equal(ar["hidden"][t], np.broadcast_to(e, ar["hidden"][t].shape))
        lg = m.lm_head @ (e / np.sqrt(np.mean(e * e) + 1e-5))
        assert ar["tokens"][t] == int(np.argmax(lg))
        assert len(set(ar["exit_tokens"][t])) == 1


def test_primitives():
    x = np.array([3.0, -4.0, 0.0, 12.0])
    assert np.allclose(rmsnorm(x, np.ones(4), 0.0), x / np.sqrt(169 / 4))
    assert np.allclose(rmsnorm(x, 2 * np.ones(4), 1e-5), 2 * x / np.sqrt(169 / 4 + 1e-5))
    # RoPE: position 0 is the identity; norm-preserving; pairs (i, i+hd/2) rotate by pos*theta^(-2i/hd)
    v = np.arange(1.0, 9.0).reshape(1, 8)
    assert np.array_equal(rope(v, 0, 1e4), v)
    r = rope(v, 3, 1e4)
    assert np.isclose(np.linalg.norm(r), np.linalg.norm(v))
    for i in range(4):
        a = 3 * 1e4 ** (-2 * i / 8)
        assert np.isclose(r[0, i], v[0, i] * np.cos(a) - v[0, i + 4] * np.sin(a))
        assert np.isclose(r[0, i + 4], v[0, i + 4] * np.cos(a) + v[0, i] * np.sin(a))
    # relative-position property: <rope(q,m), rope(k,n)> depends on m-n only
    q, k = np.random.default_rng(0).normal(size=(2, 1, 8))
    assert np.isclose((rope(q, 5, 1e4) * rope(k, 2, 1e4)).sum(), (rope(q, 13, 1e4) * rope(k, 10, 1e4)).sum())
    # bf16 rounding: ties to even on the 16 dropped bits; matches torch
    torch = pytest.importorskip("torch")
    z = np.random.default_rng(1).normal(size=4096).astype(np.float32)
    z[:4] = np.array([1.00390625, 1.01171875, -1.00390625, 3.0e-39], dtype=np.float32)   # two exact ties, a denormal
    assert np.array_equal(bf16_round(z), torch.from_numpy(z).bfloat16().float().numpy())
    assert np.array_equal(dex_synth.bf16_round_f32(z), bf16_round(z))


def test_prefill_matches_ar_state(c1, c1_model):
    wl, _, p = c1
    ck, cv = prefill(c1_model, p)
    assert len(ck) == wl.shape.n_layers and all(len(c) == len(p) - 1 for c in ck)


@pytest.mark.parametrize("kv_round", [None, "bf16"])
def test_prefill_matrix_equals_positionwise(c1, kv_round):
    """oracle.ar.prefill_matrix (whole-sequence causal form, used for the long-context GPU parity cases) gives the
    K/V of the position-at-a-time prefill: c1 (MHA) and a GQA shape with non-unit norm weights."""
    from oracle.ar import prefill_matrix
    wl, w, p = c1
    shp = dex_synth.ModelShape("gqa-mini", 3, 64, 8, 2, 8, 96, 50, rope_theta=5e5)
    cases = [(wl.shape, w, dex_synth.make_prompt(wl.shape.vocab, 70, 5)),
             (shp, dex_synth.make_weights(shp, 7, norm_jitter=0.2), dex_synth.make_prompt(shp.vocab, 33, 3))]
    for shape, ww, pp in cases:
        m = OracleModel(shape, ww, kv_round=kv_round)
        ck, cv = prefill(m, pp)
        mk, mv = prefill_matrix(m, pp)
        assert len(mk) == len(ck) == shape.n_layers
        tol = 1e-11 if kv_round is None else 1e-2 * 2.0 ** -7     # bf16 cache: a last-place flip of a rounded value
        n_flip = 0
        for l in range(shape.n_layers):
            assert len(mk[l]) == len(ck[l]) == len(pp) - 1
            a, b = np.stack(ck[l]), np.stack(mk[l])
            va, vb = np.stack(cv[l]), np.stack(mv[l])
            assert np.abs(a - b).max() <= tol * max(1.0, np.abs(a).max())
            assert np.abs(va - vb).max() <= tol * max(1.0, np.abs(va).max())
            n_flip += int((a != b).sum() + (va != vb).sum())
        if kv_round == "bf16":
            assert n_flip <= 2                     # rounded values are bit-equal up to rare last-place ties
        # and the decode that continues from either state is the same stream
        t1 = ar_greedy(m, pp, 6, state=(ck, cv))["tokens"]
        t2 = ar_greedy(m, pp, 6, state=(mk, mv))["tokens"]
        assert np.array_equal(t1, t2)
    ck0, cv0 = prefill_matrix(OracleModel(wl.shape, w), p[:1])   # one-token prompt: nothing to prefill
    assert all(len(c) == 0 for c in ck0)
