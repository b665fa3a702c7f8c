"""dex_gemm_noalloc: the weight-streaming GEMM through the entry point that allocates nothing (its scratch is one static
device array, include/dex.h) against the EXISTING path for the same kernel, dex_debug_gemm (scratch in the context's
caller-allocated workspace), and against the definition Y = X W^T in float64.  Tolerance: the 2e-5 relative error the GEMM
parity tests use (tests/test_gpu_parity.py::test_gemm_matches_definition).  Several calls in a row share the static array,
so a later, smaller call must not see what an earlier one left behind.

This file sorts last on purpose (pytest --collect-only): the suite runs with pytest -x, and a failure here must not hide
the tests of the hot path.  It passes alone in a fresh process and after the other tests (it touches no shared state but
the static array, which every call re-initialises)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 2e-5


@pytest.fixture(scope="module")
def P():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2606_29223_b200 import build
    build.build()
    import paper_2606_29223_b200 as P
    return P


def _rel(g, o):
    return float(np.abs(g - o).max() / np.abs(o).max())


def _noalloc(P, torch, W_dev, x_host, planes=2):
    """One call of the new entry point: device weights [out, k] bf16, host x -> host y."""
    x_dev = torch.from_numpy(x_host).cuda()
    y_dev = torch.full((x_host.shape[0], W_dev.shape[0]), float("nan"), dtype=torch.float32, device="cuda")
    st = torch.cuda.current_stream()
    P.dex_gemm_noalloc(W_dev.data_ptr(), x_dev.data_ptr(), x_host.shape[0], W_dev.shape[0], W_dev.shape[1], planes,
                       y_dev.data_ptr(), st.cuda_stream)
    st.synchronize()
    return y_dev.cpu().numpy()


def test_noalloc_gemm_matches_context_path_two_calls_in_a_row(P, c1):
    import torch
    wl, w, _ = c1
    d = P.Dex(wl.shape, w, (wl.shape.n_layers,), max_ctx=256, debug_taps=1, use_graph=0)      # the existing path
    rng = np.random.default_rng(11)
    # (weight kind, layer, rows): QKV [768 x 256]; down [256 x 688] (ragged K tail); gate/up [1376 x 256] (ragged out
    # tile); 19 rows = two 16-row boxes with a ragged tail, then SMALLER calls that reuse the array
    calls = [(0, 3, 19), (3, 5, 3), (2, 1, 32), (0, 3, 19), (1, 7, 1)]
    names = ("wqkv", "wo", "wgu", "wdn")
    first = {}
    for which, layer, rows in calls:
        W = w[names[which]][layer].reshape(-1, w[names[which]].shape[-1])
        W_dev = W.cuda().contiguous()
        x = rng.standard_normal((rows, W.shape[1])).astype(np.float32) if (which, layer, rows) not in first else first[(which, layer, rows)][0]
        y_new = _noalloc(P, torch, W_dev, x)
        y_old = d.gemm(which, layer, x)                                                      # dex_debug_gemm
        ref = x.astype(np.float64) @ W.float().numpy().astype(np.float64).T
        assert np.isfinite(y_new).all()
        assert _rel(y_new, y_old) < TOL, (which, layer, rows, _rel(y_new, y_old))
        assert _rel(y_new, ref) < TOL, (which, layer, rows)
        if (which, layer, rows) in first:                                                    # same call again: same bits
            assert np.array_equal(y_new, first[(which, layer, rows)][1])
        else:
            first[(which, layer, rows)] = (x, y_new)
    d.close()


def test_noalloc_single_plane_and_limits(P, c1):
    import torch
    import dex_synth
    wl, w, _ = c1
    W = w["wqkv"][2]
    W_dev = W.cuda().contiguous()
    rng = np.random.default_rng(12)
    x = rng.standard_normal((7, 256)).astype(np.float32)
    y = _noalloc(P, torch, W_dev, x, planes=1)                # plain bf16 activations: the definition on the rounded input
    ref = dex_synth.bf16_round_f32(x).astype(np.float64) @ W.float().numpy().astype(np.float64).T
    assert _rel(y, ref) < TOL
    xd = torch.zeros((40, 256), dtype=torch.float32, device="cuda")
    yd = torch.zeros((40, 768), dtype=torch.float32, device="cuda")
    s = torch.cuda.current_stream().cuda_stream
    with pytest.raises(P.DexError) as e:                      # beyond the static scratch's maximum: a clear error
        P.dex_gemm_noalloc(W_dev.data_ptr(), xd.data_ptr(), 33, 768, 256, 2, yd.data_ptr(), s)
    assert e.value.code == P.DEX_ECAPACITY and "exceed" in str(e.value)
    with pytest.raises(P.DexError) as e:
        P.dex_gemm_noalloc(W_dev.data_ptr(), xd.data_ptr(), 4, 768, 252, 2, yd.data_ptr(), s)   # k not a multiple of 8
    assert e.value.code == P.DEX_EINVAL
    with pytest.raises(P.DexError) as e:
        P.dex_gemm_noalloc(0, xd.data_ptr(), 4, 768, 256, 2, yd.data_ptr(), s)
    assert e.value.code == P.DEX_EINVAL
    y2 = _noalloc(P, torch, W_dev, x, planes=1)               # a rejected call leaves the array usable
    assert np.array_equal(y, y2)
