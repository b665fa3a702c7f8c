import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def c1():
    """Config c1 (BASELINE.json:configs[0]): shape, bf16-rounded weights, prompt."""
    import dex_synth
    wl = dex_synth.workload("c1")
    w = dex_synth.make_weights(wl.shape, wl.weight_seed)
    p = dex_synth.make_prompt(wl.shape.vocab, wl.prompt_len, wl.prompt_seed)
    return wl, w, p


@pytest.fixture(scope="session")
def c1_model(c1):
    from oracle import OracleModel
    wl, w, _ = c1
    return OracleModel(wl.shape, w)


@pytest.fixture(scope="session")
def c1_ar(c1, c1_model):
    from oracle import ar_greedy
    wl, _, p = c1
    return ar_greedy(c1_model, p, wl.gen_len, keep_hidden=True, keep_logits=True)
