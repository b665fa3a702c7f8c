"""Inducing-adapter exits in the oracle (App. C.2).  Pins: the paper's parameter counts, the
gate at zero, a closed form that does not go through the oracle's own routine, the final depth left untouched,
and losslessness of DEX with adapters at the non-final depths."""
import numpy as np
import pytest

from oracle import ead


def test_paper_parameter_counts():
    """P_ad = 4h^2 + 4h + 1 at m = 2h; 536.9 M (34B, DEX-1/3), 805.4 M (70B, DEX-1/4), 1.88 B (70B, DEX-1/8): h = 8192
    (PAPER.md:498-502)."""
    h = 8192
    assert ead.adapter_params(h) == 4 * h * h + 4 * h + 1 == h * 2 * h + 2 * h * h + 2 * h + 2 * h + 1
    assert round(2 * ead.adapter_params(h) / 1e6, 1) == 536.9
    assert round(3 * ead.adapter_params(h) / 1e6, 1) == 805.4
    assert round(7 * ead.adapter_params(h) / 1e9, 2) == 1.88


@pytest.fixture(scope="module")
def c1_ad(c1):
    import dex_synth
    from oracle import OracleModel
    wl, w, p = c1
    ad = dex_synth.make_adapters(wl.shape, 3, seed=99, alpha=0.5)
    return wl, w, p, ad, OracleModel(wl.shape, w, adapters=ad)


def test_gate_zero_and_final_depth_untouched(c1, c1_model, c1_ad):
    import dex_synth
    from oracle import OracleModel
    wl, w, p, ad, om = c1_ad
    h = np.random.default_rng(0).standard_normal(wl.shape.d_model)
    assert np.array_equal(om.exit_logits_at(h, 3, 4), c1_model.exit_logits(h))          # final depth: no adapter
    assert not np.allclose(om.exit_logits_at(h, 1, 4), c1_model.exit_logits(h))          # non-final: induced
    ad0 = dict(ad)
    ad0["alpha"] = ad["alpha"] * 0
    om0 = OracleModel(wl.shape, w, adapters=ad0)
    assert np.array_equal(om0.exit_logits_at(h, 1, 4), c1_model.exit_logits(h))          # alpha = 0: identity


def test_delta_closed_form(c1_ad):
    """Delta h recomputed with plain NumPy from the tensors (not through the oracle's routine)."""
    wl, w, p, ad, om = c1_ad
    k = 2
    h = np.random.default_rng(1).standard_normal(wl.shape.d_model)
    W1, W2 = ad["w1"][k].float().numpy().astype(np.float64), ad["w2"][k].float().numpy().astype(np.float64)
    b1, b2 = ad["b1"][k].numpy().astype(np.float64), ad["b2"][k].numpy().astype(np.float64)
    a = h / np.sqrt((h * h).mean() + wl.shape.rms_eps) * ad["norm"][k].numpy()
    t = W1 @ a + b1
    ref = float(ad["alpha"][k]) * (W2 @ (t / (1.0 + np.exp(-t))) + b2)
    assert np.allclose(om.adapter_delta(h, k), ref, rtol=1e-12, atol=1e-14)
    assert W1.shape == (2 * wl.shape.d_model, wl.shape.d_model)                          # m = 2h by default


@pytest.mark.parametrize("X", [(2, 4, 6, 8), (4, 8)])
def test_lossless_with_adapters_and_proposals_change(c1, c1_ar, c1_ad, X):
    from oracle import dex_decode
    wl, w, p, ad, om = c1_ad
    T = 24
    od = dex_decode(om, p, T, X, trace=True)
    assert np.array_equal(od["tokens"], c1_ar["tokens"][:T])
    from oracle import OracleModel
    plain = dex_decode(OracleModel(wl.shape, w), p, T, X, trace=True)
    differs = any(a["u"] != b["u"] for a, b in zip(od["rounds"], plain["rounds"]) if a["nodes"] == b["nodes"])
    assert differs or od["n_rounds"] != plain["n_rounds"]                                 # the adapters do act


def test_delta_against_torch_module_built_from_the_paper(c1_ad):
    """A pin that is not the oracle's own formula: the adapter as a torch.nn module assembled from the paper's
    description - input RMSNorm, two biased linears h -> m -> h with the backbone activation between them, a scalar
    gate on the whole branch - whose parameter count must be the paper's
    P_ad = hm + mh + m + 2h + 1 = 4h^2 + 4h + 1 at m = 2h.  Evaluated by torch's own layers on the same tensors.
    Fails if b2 sits outside the gate, if the activation is not SiLU, if the RMSNorm is dropped or if W1/W2 are
    transposed (variants checked below)."""
    torch = pytest.importorskip("torch")
    nn = torch.nn
    wl, w, p, ad, om = c1_ad
    hdim, k = wl.shape.d_model, 1
    m = ad["w1"].shape[1]

    class Adapter(nn.Module):
        def __init__(self):
            super().__init__()
            self.norm = nn.RMSNorm(hdim, eps=wl.shape.rms_eps)
            self.w1 = nn.Linear(hdim, m, bias=True)
            self.w2 = nn.Linear(m, hdim, bias=True)
            self.alpha = nn.Parameter(torch.zeros(()))

        def forward(self, h):
            return self.alpha * self.w2(nn.functional.silu(self.w1(self.norm(h))))

    mod = Adapter().double()
    assert sum(q.numel() for q in mod.parameters()) == ead.adapter_params(hdim) == 4 * hdim * hdim + 4 * hdim + 1
    with torch.no_grad():
        mod.norm.weight.copy_(ad["norm"][k].double())
        mod.w1.weight.copy_(ad["w1"][k].double()); mod.w1.bias.copy_(ad["b1"][k].double())
        mod.w2.weight.copy_(ad["w2"][k].double()); mod.w2.bias.copy_(ad["b2"][k].double())
        mod.alpha.copy_(ad["alpha"][k].double())
    rng = np.random.default_rng(4)
    for _ in range(3):
        h = rng.standard_normal(hdim) * 3.0
        with torch.no_grad():
            ref = mod(torch.from_numpy(h)).numpy()
        got = om.adapter_delta(h, k)
        assert np.allclose(got, ref, rtol=1e-10, atol=1e-12)
        # the plausible mistakes are far outside that tolerance on these tensors
        with torch.no_grad():
            t = torch.from_numpy(h)
            z = mod.w1(mod.norm(t))
            b2_outside = (mod.alpha * nn.functional.linear(nn.functional.silu(z), mod.w2.weight) + mod.w2.bias).numpy()
            gelu = (mod.alpha * mod.w2(nn.functional.gelu(z))).numpy()
            no_norm = (mod.alpha * mod.w2(nn.functional.silu(mod.w1(t)))).numpy()
        for wrong in (b2_outside, gelu, no_norm):
            assert np.abs(wrong - ref).max() > 1e-4 * np.abs(ref).max()
            assert not np.allclose(got, wrong, rtol=1e-6, atol=1e-9)
