"""O1: Llama-style pre-norm decoder forward (BASELINE.json:configs).

The paper inherits the backbone from Hugging Face Llama and only states that every
exit depth is "decoded by the same final normalization and LM head as the backbone"
(App. C.2).  Model details per reading R13: rms_eps 1e-5,
RoPE "rotate-half" pairing (i, i+hd/2), untied embed / LM head, no biases.

Everything here is one position at a time with an explicit KV list: no blocking, no fusion.
"""
import numpy as np


def bf16_round(x):
    """fp -> (fp32 RNE) -> bf16 RNE -> back to x.dtype.  Models "K/V are stored in a bf16
    cache" (BASELINE.json:north_star (b)) when kv_round='bf16'."""
    x = np.asarray(x)
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = ((u >> 16) & 1) + np.uint32(0x7FFF)
    y = ((u + r) & np.uint32(0xFFFF0000)).view(np.float32)
    return y.astype(x.dtype)


def rmsnorm(x, w, eps):
    """RMSNorm(x) = x / sqrt(mean(x^2) + eps) * w   (Llama; R13)."""
    ms = np.mean(x * x, axis=-1, keepdims=True)
    return x / np.sqrt(ms + eps) * w


def rope(x, pos, theta):
    """Rotary embedding, rotate-half convention (R13).  x: [heads, hd]; absolute position pos."""
    hd = x.shape[-1]
    half = hd // 2
    i = np.arange(half, dtype=np.float64)
    ang = float(pos) * theta ** (-2.0 * i / hd)
    c, s = np.cos(ang).astype(x.dtype), np.sin(ang).astype(x.dtype)
    x1, x2 = x[..., :half], x[..., half:]
    return np.concatenate([x1 * c - x2 * s, x2 * c + x1 * s], axis=-1)


def silu(x):
    return x / (1.0 + np.exp(-x))


class OracleModel:
    """Holds the tensors of dex_synth.make_weights upcast to `dtype` (exact for bf16)."""

    def __init__(self, shape, weights, dtype=np.float64, kv_round=None, adapters=None):
        self.shape = shape
        self.dtype = dtype
        self.kv_round = kv_round
        self.L, self.d = shape.n_layers, shape.d_model
        self.nh, self.nkv, self.hd = shape.n_heads, shape.n_kv_heads, shape.head_dim
        self.eps, self.theta = shape.rms_eps, shape.rope_theta

        def cv(t):
            return t.float().numpy().astype(dtype) if hasattr(t, "numpy") else np.asarray(t, dtype=dtype)

        self.embed = cv(weights["embed"])
        self.lm_head = cv(weights["lm_head"])
        self.wqkv = cv(weights["wqkv"])
        self.wo = cv(weights["wo"])
        self.wgu = cv(weights["wgu"])
        self.wdn = cv(weights["wdn"])
        self.norm_attn = cv(weights["norm_attn"])
        self.norm_ffn = cv(weights["norm_ffn"])
        self.norm_final = cv(weights["norm_final"])
        # inducing adapters of the non-final exit depths (App. C.2), optional:
        # dict of w1 [n,m,h], b1 [n,m], w2 [n,h,m], b2 [n,h], norm [n,h], alpha [n]
        self.adapters = None if adapters is None else {k: cv(v) for k, v in adapters.items()}

    # ---- one layer, one position -------------------------------------------------------
    def qkv(self, l, x, pos):
        """Layer l (0-based) projections of residual x at absolute position pos -> q,k,v [heads, hd];
        q,k rotated.  k,v bf16-rounded when the cache is bf16."""
        a = rmsnorm(x, self.norm_attn[l], self.eps)
        y = self.wqkv[l] @ a
        nq = self.nh * self.hd
        nk = self.nkv * self.hd
        q = rope(y[:nq].reshape(self.nh, self.hd), pos, self.theta)
        k = rope(y[nq:nq + nk].reshape(self.nkv, self.hd), pos, self.theta)
        v = y[nq + nk:].reshape(self.nkv, self.hd)
        if self.kv_round == "bf16":
            k, v = bf16_round(k), bf16_round(v)
        return q, k, v

    def attend(self, q, keys, vals):
        """softmax(q.k/sqrt(hd)).v over the listed positions; GQA: query head h uses kv head
        h // (nh/nkv).  keys/vals: lists of [nkv, hd] (the visible context incl. self)."""
        K = np.stack(keys, axis=0)            # [n, nkv, hd]
        V = np.stack(vals, axis=0)
        g = self.nh // self.nkv
        out = np.empty((self.nh, self.hd), dtype=self.dtype)
        for h in range(self.nh):
            s = K[:, h // g, :] @ q[h] / np.sqrt(self.dtype(self.hd))
            s = s - s.max()
            p = np.exp(s)
            p = p / p.sum()
            out[h] = p @ V[:, h // g, :]
        return out.reshape(-1)

    def layer(self, l, x, pos, ctx_k, ctx_v):
        """Run layer l on residual x.  ctx_k/ctx_v: K/V (this layer) of every earlier visible
        position, in position order.  Returns (x_out, k, v) with k,v of this position."""
        q, k, v = self.qkv(l, x, pos)
        o = self.attend(q, list(ctx_k) + [k], list(ctx_v) + [v])
        x = x + self.wo[l] @ o
        b = rmsnorm(x, self.norm_ffn[l], self.eps)
        x = x + self.wdn[l] @ (silu(self.wgu[l, 0] @ b) * (self.wgu[l, 1] @ b))
        return x, k, v

    def exit_logits(self, h):
        """Shared exit: final RMSNorm + LM head at any depth."""
        return self.lm_head @ rmsnorm(h, self.norm_final, self.eps)

    def adapter_delta(self, h, k):
        """Delta h = alpha_k W2_k sigma(W1_k RMSNorm(h) + b1_k) + b2_k scaled by alpha_k (the parameter
        count P_ad = hm + mh + m + 2h + 1 fixes two biased linears, an RMSNorm scale and the scalar gate,
        PAPER.md:498-500); sigma = the backbone activation (SiLU)."""
        A = self.adapters
        a = rmsnorm(h, A["norm"][k], self.eps)
        z = silu(A["w1"][k] @ a + A["b1"][k])
        return A["alpha"][k] * (A["w2"][k] @ z + A["b2"][k])

    def exit_logits_at(self, h, k, n_depths):
        """Exit at candidate depth index k of n_depths: non-final depths decode the induced representation
        h~ = h + Delta h "by the same final normalization and LM head as the backbone"; the
        final depth uses the original hidden state without an adapter."""
        if self.adapters is not None and k < n_depths - 1:
            h = h + self.adapter_delta(h, k)
        return self.exit_logits(h)

    def embed_tok(self, tok):
        return self.embed[int(tok)].copy()


def argmax_lowest(logits, masked=()):
    """Greedy decode, ties -> lowest token id (R11); `masked` ids set to -inf (Alg. 2 l.5-7)."""
    if len(masked):
        logits = logits.copy()
        logits[list(masked)] = -np.inf
    return int(np.argmax(logits))
