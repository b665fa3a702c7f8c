"""Seeded synthetic inputs (model tensors, prompts, workload shapes) for DEX.

This module is the ONLY code shared by the CPU oracle (``oracle/``) and the CUDA
path (``paper_2606_29223_b200/``).  It holds none of the method's arithmetic: it
draws seeded random tensors in the shapes ``BASELINE.json:configs`` names and
packs them in the layout ``DESIGN.md`` ("Data layout") describes.  The inputs
stand in for the paper's checkpoints and GSM8K / HumanEval / XSum prompts
(Sec. 4), none of which exist in this environment.
"""
from .configs import ModelShape, Workload, WORKLOADS, workload  # noqa: F401
from .gen import make_weights, make_adapters, make_prompt, bf16_round_f32  # noqa: F401
