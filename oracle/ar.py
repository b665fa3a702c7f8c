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
