"""Cache-free brute force used ONLY to pin oracle/model.py, ar.py and dex.py.

Whole-sequence matrix form with an explicit causal mask: a different code path from the
one-position-at-a-time cached forward (no KV lists, no per-position loop, RoPE built from
complex rotation), so an indexing / masking / cache bug in either shows up as a mismatch.
"""
import numpy as np


def forward_nocache(model, tokens):
    """tokens [n] -> hidden [L+1, n, d] (hidden[0] = embeddings, hidden[l] = residual after
    layer l).  Always float64, no KV rounding."""
    tokens = np.asarray(tokens, dtype=np.int64)
    n = len(tokens)
    nh, nkv, hd, d = model.nh, model.nkv, model.hd, model.d
    f64 = np.float64
    X = model.embed[tokens].astype(f64)
    hidden = [X.copy()]
    pos = np.arange(n)[:, None]
    freqs = model.theta ** (-np.arange(0, hd, 2, dtype=f64) / hd)[None, :]
    rot = np.exp(1j * pos * freqs)                            # [n, hd/2]
    mask = np.tril(np.ones((n, n), dtype=bool))

    def norm(A, w):
        return A * (1.0 / np.sqrt((A ** 2).mean(-1, keepdims=True) + model.eps)) * w.astype(f64)

    def rope_c(A):                                            # A [n, heads, hd]
        z = (A[..., : hd // 2] + 1j * A[..., hd // 2:]) * rot[:, None, :]
        return np.concatenate([z.real, z.imag], -1)

    for l in range(model.L):
        A = norm(X, model.norm_attn[l])
        QKV = A @ model.wqkv[l].astype(f64).T
        Q = rope_c(QKV[:, : nh * hd].reshape(n, nh, hd))
        K = rope_c(QKV[:, nh * hd: (nh + nkv) * hd].reshape(n, nkv, hd))
        V = QKV[:, (nh + nkv) * hd:].reshape(n, nkv, hd)
        K = np.repeat(K, nh // nkv, axis=1)
        V = np.repeat(V, nh // nkv, axis=1)
        S = np.einsum("ihd,jhd->hij", Q, K) / np.sqrt(hd)
        S = np.where(mask[None], S, -np.inf)
        P = np.exp(S - S.max(-1, keepdims=True))
        P /= P.sum(-1, keepdims=True)
        O = np.einsum("hij,jhd->ihd", P, V).reshape(n, nh * hd)
        X = X + O @ model.wo[l].astype(f64).T
        Bn = norm(X, model.norm_ffn[l])
        G = Bn @ model.wgu[l, 0].astype(f64).T
        U = Bn @ model.wgu[l, 1].astype(f64).T
        X = X + (G / (1 + np.exp(-G)) * U) @ model.wdn[l].astype(f64).T
        hidden.append(X.copy())
    return np.stack(hidden)


def logits_nocache(model, h):
    f64 = np.float64
    hn = h * (1.0 / np.sqrt((h ** 2).mean(-1, keepdims=True) + model.eps)) * model.norm_final.astype(f64)
    return hn @ model.lm_head.astype(f64).T
