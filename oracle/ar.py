"""O2 + O3: greedy autoregressive decoding with every-depth exits (Sec. 2.1).

init per reading R3: K/V of prompt[0..P-2] are prefilled at all layers and prompt[P-1] is the
first input, so all T tokens come out of the same one-token loop (as they do for DEX).
"""
import numpy as np

from .gumbel import gumbel_row, perturbed
from .model import argmax_lowest


def prefill(model, prompt):
    """K/V of prompt[0..P-2] at every layer, one position at a time."""
    ck = [[] for _ in range(model.L)]
    cv = [[] for _ in range(model.L)]
    for pos, tok in enumerate(prompt[:-1]):
        x = model.embed_tok(tok)
        for l in range(model.L):
            x, k, v = model.layer(l, x, pos, ck[l], cv[l])
            ck[l].append(k)
            cv[l].append(v)
    return ck, cv


def prefill_matrix(model, prompt):
    """The same K/V as prefill(), written as the whole-sequence causal form of O1 (every position of
    prompt[0..P-2] at once, explicit lower-triangular mask) instead of one position at a time.  Same definition,
    same dtype, K/V rounded the same way when the cache is bf16; only the summation order inside the library
    matmuls differs.  Exists because the position-at-a-time GEMVs make a 600-token prompt at d = 4096 take
    minutes; pinned against prefill() in tests/test_oracle_model.py."""
    from .model import bf16_round, rmsnorm, silu
    toks = np.asarray([int(t) for t in prompt[:-1]], dtype=np.int64)
    n = len(toks)
    ck = [[] for _ in range(model.L)]
    cv = [[] for _ in range(model.L)]
    if n == 0:
        return ck, cv
    dt = model.dtype
    nh, nkv, hd = model.nh, model.nkv, model.hd
    half = hd // 2
    ang = np.arange(n, dtype=np.float64)[:, None] * model.theta ** (-2.0 * np.arange(half, dtype=np.float64) / hd)[None, :]
    c, s = np.cos(ang).astype(dt)[:, None, :], np.sin(ang).astype(dt)[:, None, :]      # [n, 1, hd/2]

    def rope_all(A):                                   # A [n, heads, hd], rotate-half pairing (R13)
        x1, x2 = A[..., :half], A[..., half:]
        return np.concatenate([x1 * c - x2 * s, x2 * c + x1 * s], axis=-1)

    X = model.embed[toks].astype(dt)
    mask = np.tril(np.ones((n, n), dtype=bool))
    g = nh // nkv
    for l in range(model.L):
        A = rmsnorm(X, model.norm_attn[l], model.eps).astype(dt)
        Y = A @ model.wqkv[l].T
        Q = rope_all(Y[:, :nh * hd].reshape(n, nh, hd))
        K = rope_all(Y[:, nh * hd:(nh + nkv) * hd].reshape(n, nkv, hd))
        V = Y[:, (nh + nkv) * hd:].reshape(n, nkv, hd)
        if model.kv_round == "bf16":
            K, V = bf16_round(K), bf16_round(V)
        O = np.empty((n, nh, hd), dtype=dt)
        for h in range(nh):
            S = Q[:, h, :] @ K[:, h // g, :].T / np.sqrt(dt(hd))
            S = np.where(mask, S, -np.inf)
            P = np.exp(S - S.max(-1, keepdims=True))
            P = P / P.sum(-1, keepdims=True)
            O[:, h, :] = P @ V[:, h // g, :]
        X = X + O.reshape(n, nh * hd) @ model.wo[l].T
        Bn = rmsnorm(X, model.norm_ffn[l], model.eps).astype(dt)
        X = X + (silu(Bn @ model.wgu[l, 0].T) * (Bn @ model.wgu[l, 1].T)) @ model.wdn[l].T
        ck[l] = [K[i].copy() for i in range(n)]
        cv[l] = [V[i].copy() for i in range(n)]
    return ck, cv


def ar_greedy(model, prompt, T, keep_hidden=False, keep_logits=False, state=None):
    """Returns dict: tokens [T]; exit_tokens [T, L] (greedy token decoded at every depth l,
    for Def. 1); top1/top2 final-depth logit values [T]; optionally hidden [T, L, d] and
    final-depth logits [T, V]."""
    prompt = list(int(t) for t in prompt)
    ck, cv = state if state is not None else prefill(model, prompt)
    toks = list(prompt)
    out = dict(tokens=[], exit_tokens=[], top1=[], top2=[], hidden=[], logits=[])
    for _ in range(T):
        pos = len(toks) - 1
        x = model.embed_tok(toks[-1])
        exits, hid = [], []
        for l in range(model.L):
            x, k, v = model.layer(l, x, pos, ck[l], cv[l])
            ck[l].append(k)
            cv[l].append(v)
            logits = model.exit_logits(x)
            exits.append(argmax_lowest(logits))
            if keep_hidden:
                hid.append(x.copy())
        y = exits[-1]                      # y_t = argmax logits_L
        srt = np.sort(logits)
        out["tokens"].append(y)
        out["exit_tokens"].append(exits)
        out["top1"].append(float(srt[-1]))
        out["top2"].append(float(srt[-2]))
        if keep_hidden:
            out["hidden"].append(np.stack(hid))
        if keep_logits:
            out["logits"].append(logits.copy())
        toks.append(y)
    out["tokens"] = np.array(out["tokens"], dtype=np.int64)
    out["exit_tokens"] = np.array(out["exit_tokens"], dtype=np.int64)
    out["state"] = (ck, cv)
    return out


def ar_sample(model, prompt, T, tau, seed, seq=0, state=None):
    """Autoregressive SAMPLING with the Gumbel-Max rule and the shared counter-based noise of oracle/gumbel.py:
    y_t = argmax_v (logits_L / tau + G[pos of y_t]).  Returns tokens [T] and the top-2 of the perturbed logits."""
    prompt = list(int(t) for t in prompt)
    ck, cv = state if state is not None else prefill(model, prompt)
    toks = list(prompt)
    out = dict(tokens=[], top1=[], top2=[])
    V = model.lm_head.shape[0]
    for _ in range(T):
        pos = len(toks) - 1
        x = model.embed_tok(toks[-1])
        for l in range(model.L):
            x, k, v = model.layer(l, x, pos, ck[l], cv[l])
            ck[l].append(k)
            cv[l].append(v)
        z = perturbed(model.exit_logits(x), tau, gumbel_row(seed, seq, pos + 1, V))
        y = argmax_lowest(z)
        srt = np.sort(z)
        out["tokens"].append(y)
        out["top1"].append(float(srt[-1]))
        out["top2"].append(float(srt[-2]))
        toks.append(y)
    out["tokens"] = np.array(out["tokens"], dtype=np.int64)
    return out
