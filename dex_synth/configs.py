"""Workload shapes of BASELINE.json:configs[0..4] (c1..c5 in SURVEY.md 8(a))."""
from dataclasses import dataclass, field
from typing import Tuple


@dataclass(frozen=True)
class ModelShape:
    name: str
    n_layers: int          # L
    d_model: int           # d
    n_heads: int
    n_kv_heads: int
    head_dim: int
    d_ffn: int
    vocab: int
    rms_eps: float = 1e-5          # reading R13
    rope_theta: float = 1e4        # reading R13
    resid_decay: float = 4.0       # o_proj/down_proj of layer l scaled by exp(-decay*l/L), l=1..L (R14)

    @property
    def qkv_out(self) -> int:
        return (self.n_heads + 2 * self.n_kv_heads) * self.head_dim

    def bytes_per_layer(self) -> int:
        """bf16 weight bytes of one decoder layer."""
        d, f = self.d_model, self.d_ffn
        return 2 * (self.qkv_out * d + d * self.n_heads * self.head_dim + 3 * f * d)

    def lm_head_bytes(self) -> int:
        return 2 * self.vocab * self.d_model

    def kv_bytes_per_pos(self) -> int:
        """bf16 K+V bytes per position, all layers."""
        return 2 * 2 * self.n_kv_heads * self.head_dim * self.n_layers


@dataclass(frozen=True)
class Workload:
    key: str
    shape: ModelShape
    depths: Tuple[int, ...]        # exploration set X, last == L (Def. 4)
    prompt_len: int
    gen_len: int
    n_seqs: int = 1
    weight_seed: int = 1234
    prompt_seed: int = 4321


TINY = ModelShape("tiny", 8, 256, 4, 4, 64, 688, 1024)
L7B = ModelShape("llama2-7b-shape", 32, 4096, 32, 32, 128, 11008, 32000)
L8B = ModelShape("llama3-8b-shape", 32, 4096, 32, 8, 128, 14336, 128256, rope_theta=5e5)
L13B = ModelShape("llama2-13b-shape", 40, 5120, 40, 40, 128, 13824, 32000, resid_decay=3.0)

WORKLOADS = {
    "c1": Workload("c1", TINY, (2, 4, 6, 8), 16, 64),
    "c2": Workload("c2", L7B, (8, 16, 24, 32), 512, 256),
    "c3": Workload("c3", L7B, tuple(range(4, 33, 4)), 512, 256),
    "c4": Workload("c4", L8B, tuple(range(4, 33, 4)), 2048, 512),
    "c5": Workload("c5", L13B, tuple(range(5, 41, 5)), 1024, 256, n_seqs=4),
}


def workload(key: str) -> Workload:
    return WORKLOADS[key]
