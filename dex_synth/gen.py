"""Seeded tensor / prompt generators.  No model arithmetic lives here.

Packed tensor layout (all row-major, "out x in" like nn.Linear):
  embed   [V, d]                      bf16-representable
  lm_head [V, d]
  wqkv    [L, (nh+2*nkv)*hd, d]       rows: all q heads, then k heads, then v heads
  wo      [L, d, nh*hd]               * exp(-decay*l/L), l = 1..L
  wgu     [L, 2, ffn, d]              [.,0]=gate, [.,1]=up
  wdn     [L, d, ffn]                 * exp(-decay*l/L)
  norm_attn [L, d], norm_ffn [L, d], norm_final [d]   fp32 (ones unless norm_jitter>0)

Every tensor is N(0, 0.02) from its own sub-seed (seed, tensor name, layer) and is
rounded to bf16 ("bf16-rounded weights shared", BASELINE.json:north_star), returned
as torch.bfloat16 so both sides upcast the same bits exactly.  ``exact_fp32=True``
returns the unrounded fp32 draws instead (config c1's "fp32" invariant runs, R15).
"""
import hashlib
import math
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import torch

from .configs import ModelShape


def _subseed(seed: int, name: str, layer: int) -> int:
    h = hashlib.sha256(f"{seed}/{name}/{layer}".encode()).digest()
    return int.from_bytes(h[:8], "little") & 0x7FFFFFFFFFFFFFFF


def _normal(shape, seed, name, layer, std, scale=1.0):
    g = torch.Generator(device="cpu").manual_seed(_subseed(seed, name, layer))
    t = torch.empty(shape, dtype=torch.float32)
    t.normal_(0.0, std, generator=g)
    if scale != 1.0:
        t.mul_(scale)
    return t


def bf16_round_f32(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even fp32 -> bf16 -> fp32, pure bit arithmetic (no torch)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = ((u >> 16) & 1) + np.uint32(0x7FFF)
    return ((u + r) & np.uint32(0xFFFF0000)).view(np.float32)


def make_weights(shape: ModelShape, seed: int = 1234, exact_fp32: bool = False,
                 norm_jitter: float = 0.0, threads: int = 8, std: float = 0.02):
    """Returns dict name -> torch tensor (bf16 for matrices unless exact_fp32; fp32 norms)."""
    L, d, f = shape.n_layers, shape.d_model, shape.d_ffn
    qkv, ao = shape.qkv_out, shape.n_heads * shape.head_dim
    mdt = torch.float32 if exact_fp32 else torch.bfloat16
    out = {
        "wqkv": torch.empty((L, qkv, d), dtype=mdt),
        "wo": torch.empty((L, d, ao), dtype=mdt),
        "wgu": torch.empty((L, 2, f, d), dtype=mdt),
        "wdn": torch.empty((L, d, f), dtype=mdt),
    }

    def one_layer(l):
        decay = math.exp(-shape.resid_decay * (l + 1) / L)      # l+1: paper indexes layers from 1 (R14)
        out["wqkv"][l] = _normal((qkv, d), seed, "wqkv", l, std).to(mdt)
        out["wo"][l] = _normal((d, ao), seed, "wo", l, std, decay).to(mdt)
        out["wgu"][l] = _normal((2, f, d), seed, "wgu", l, std).to(mdt)
        out["wdn"][l] = _normal((d, f), seed, "wdn", l, std, decay).to(mdt)

    with ThreadPoolExecutor(max_workers=max(1, threads)) as ex:
        list(ex.map(one_layer, range(L)))
    out["embed"] = _normal((shape.vocab, d), seed, "embed", 0, std).to(mdt)
    out["lm_head"] = _normal((shape.vocab, d), seed, "lm_head", 0, std).to(mdt)
    for nm, shp in (("norm_attn", (L, d)), ("norm_ffn", (L, d)), ("norm_final", (d,))):
        w = torch.ones(shp, dtype=torch.float32)
        if norm_jitter > 0.0:
            w += _normal(shp, seed, nm, 0, norm_jitter)
        out[nm] = w
    return out


def make_prompt(vocab: int, n: int, seed: int = 4321, seq: int = 0) -> np.ndarray:
    """n tokens ~ U[0, vocab) (BASELINE.json:configs "uniform over vocab")."""
    rg = np.random.Generator(np.random.Philox(key=_subseed(seed, "prompt", seq)))
    return rg.integers(0, vocab, size=n, dtype=np.int64).astype(np.int32)


def make_adapters(shape: ModelShape, n_ad: int, seed: int = 1234, alpha: float = 1e-3, m: int = 0, std: float = 0.02):
    """Random-init inducing adapters for the n_ad non-final exit depths: w1 [n,m,h] and
    w2 [n,h,m] bf16-representable N(0, std); biases N(0, std) fp32; RMSNorm scale ones; gate alpha (the paper
    initialises it to 1e-3; tests use larger values so that the adapter changes proposals).  m = 2h by default."""
    h = shape.d_model
    m = m or 2 * h
    out = {
        "w1": torch.stack([_normal((m, h), seed, "ad_w1", k, std) for k in range(n_ad)]).to(torch.bfloat16),
        "w2": torch.stack([_normal((h, m), seed, "ad_w2", k, std) for k in range(n_ad)]).to(torch.bfloat16),
        "b1": torch.stack([_normal((m,), seed, "ad_b1", k, std) for k in range(n_ad)]),
        "b2": torch.stack([_normal((h,), seed, "ad_b2", k, std) for k in range(n_ad)]),
        "norm": torch.ones((n_ad, h), dtype=torch.float32),
        "alpha": torch.full((n_ad,), float(alpha), dtype=torch.float32),
    }
    return out
