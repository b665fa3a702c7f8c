"""Boundary checks that need no GPU: the C-ABI library builds, loads and exports every symbol
include/dex.h declares; host-side argument validation; loud failure without a CUDA device."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def P():
    from paper_2606_29223_b200 import build
    build.build()
    import paper_2606_29223_b200 as P
    return P


def _declared():
    src = open(os.path.join(ROOT, "include", "dex.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dex_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(P):
    names = _declared()
    assert {"dex_init", "dex_prefill", "dex_step", "dex_collapse", "dex_workspace_bytes", "dex_destroy"} <= set(names)
    lib = P.lib()
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/dex.h but not exported"
    assert sorted(P.exported_symbols) == names


def test_struct_layout_matches_header(P):
    assert ctypes.sizeof(P.DexStepResult) == 128
    assert ctypes.sizeof(P.DexConfig) == 23 * 4
    assert ctypes.sizeof(P.DexWeights) == 15 * ctypes.sizeof(ctypes.c_void_p)
    assert P.DexStepResult.layer_evals.offset == 32


def _cfg(P, **kw):
    base = dict(n_layers=8, d_model=256, n_heads=4, n_kv_heads=4, head_dim=64, d_ffn=688, vocab=1024, rms_eps=1e-5,
                rope_theta=1e4, max_seqs=1, max_ctx=256, page_size=128, decs=1, eos_id=-1, debug_taps=0, act_planes=2,
                use_graph=1, round_kernel=1, sample=0, temperature=1.0, sample_seed=0, adapter_dim=0, lookahead=0)
    base.update(kw)
    return P.DexConfig(*[base[n] for n, _ in P.DexConfig._fields_])


def test_exploration_set_validation(P):
    """Def. 4: strictly increasing, within [1,L], last == L, |X| <= 8."""
    cfg = _cfg(P)
    assert P.dex_workspace_bytes(cfg, (2, 4, 6, 8)) > 0
    assert P.dex_workspace_bytes(cfg, (8,)) > 0
    for bad in [(2, 4, 6), (4, 2, 8), (2, 2, 8), (0, 8), (2, 9), (), tuple(range(0, 9))]:
        with pytest.raises(P.DexError) as e:
            P.dex_workspace_bytes(cfg, bad)
        assert e.value.code == P.DEX_EINVAL
    for kw in [dict(head_dim=96), dict(n_kv_heads=3), dict(page_size=100), dict(max_seqs=0), dict(act_planes=3),
               dict(d_model=250), dict(adapter_dim=96), dict(adapter_dim=704), dict(adapter_dim=512, round_kernel=0)]:
        with pytest.raises(P.DexError):
            P.dex_workspace_bytes(_cfg(P, **kw), (2, 4, 6, 8))
    with pytest.raises(P.DexError):           # adapters need a non-final depth
        P.dex_workspace_bytes(_cfg(P, adapter_dim=512), (8,))
    assert P.dex_workspace_bytes(_cfg(P, adapter_dim=512), (2, 4, 6, 8)) >= P.dex_workspace_bytes(cfg, (2, 4, 6, 8))
    with pytest.raises(P.DexError) as e:      # 8 seqs x 64 stage-0 rows > 256
        P.dex_workspace_bytes(_cfg(P, max_seqs=8), tuple(range(1, 9)))
    assert e.value.code == P.DEX_ECAPACITY


def test_workspace_grows_with_lattice(P):
    cfg = _cfg(P)
    assert P.dex_workspace_bytes(cfg, tuple(range(1, 9))) > P.dex_workspace_bytes(cfg, (2, 4, 6, 8)) \
        >= P.dex_workspace_bytes(cfg, (8,))


def test_no_cpu_fallback(P):
    """Without a CUDA device dex_init must fail loudly (DEX_ECUDA), never fall back."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    cfg = _cfg(P)
    w = P.DexWeights(*([1 << 20] * 9))
    with pytest.raises(P.DexError) as e:
        P.dex_init(cfg, w, (2, 4, 6, 8), 1 << 20, P.dex_workspace_bytes(cfg, (2, 4, 6, 8)), None)
    assert e.value.code == P.DEX_ECUDA
    with pytest.raises(RuntimeError):
        import dex_synth
        P.Dex(dex_synth.workload("c1").shape, {}, (8,))


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_29223_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("oracle's", ""), f"{f} mentions the oracle"
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_2606_29223_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "``paper_2606_29223_b200/``", "")
