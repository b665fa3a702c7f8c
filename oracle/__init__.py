"""CPU oracle for Depth Exploration Decoding (DEX, arxiv/paper_2606_29223).

TEST INFRASTRUCTURE ONLY.  A plain, slow, obviously-correct NumPy implementation of
(i) standard greedy autoregressive decoding and (ii) DEX exactly as PAPER.md defines it,
written from the paper before any CUDA kernel and sharing no code with the CUDA path
(``paper_2606_29223_b200/``).  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import it.  The only
module it shares with the product is ``dex_synth`` (seeded input generators, no arithmetic).

Precision: float64 by default (``dtype=np.float32`` for the 7B-class shapes, where
BASELINE.json:north_star fixes "a plain, slow fp32 ... CPU implementation").

Parity pins (tests/test_oracle_*.py, all ``-m "not gpu"``):
  model.py   forward       cache-free brute force == cached path; Hugging Face
                           LlamaForCausalLM on the same tensors; zero-Wo/Wd closed form
  ead.py     Defs 1,4,5    the paper's worked numbers, bounds
                           Eq. 11 / Eq. 14, monotonicity, X=[L] equality
  lattice.py tree          2^q-1 nodes, ETK_0/1/2, 2^K-1 and 128,
                           brute-force path enumeration
  dex.py     Alg. 1, 2     node hidden == from-scratch forward of its own prefix;
                           losslessness; y == final-depth argmax
                           (PAPER.md:204); closed-form round / layer-eval counts
  ar.py      prefill_matrix  whole-sequence causal form == the position-wise prefill (K/V, continued decode)
  dex.py     force_u hook  forcing the oracle's own decisions changes nothing; a forced decision records the logit gap
  model.py   adapter_delta a torch.nn module assembled from the paper's description, parameter count
                           4h^2+4h+1; fails when b2 leaves the gate, sigma != SiLU, the RMSNorm is dropped
  gumbel.py  Alg. 2 l.10-15  Gumbel-Max frequencies == softmax(l/tau) (chi-square), moments of the rows,
                           sampled DEX stream == sampled AR stream for every X
Nothing is "parity unpinned".
"""
from .model import OracleModel, rmsnorm, bf16_round  # noqa: F401
from .ar import ar_greedy, ar_sample  # noqa: F401
from .dex import dex_decode  # noqa: F401
from . import ead, gumbel, lattice  # noqa: F401
