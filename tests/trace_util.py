"""Trace harness shared by the GPU parity tests (reading R17 / R17b in DESIGN.md).

The GPU runs FREE (its own exit decisions, commits through dex_collapse).  The oracle then replays Alg. 1 with
every exit decision teacher-forced to the GPU's candidate (`dex_decode(force_u=...)`), which keeps the two
lattices identical for the whole run, so EVERY round and EVERY node is compared - nothing is skipped after a
near-tie flip.  A forced decision that differs from the oracle's own arg-max must be a near-tie of the oracle's
(masked) logits of that node: gap < 1e-2 (the tolerance BASELINE.json:north_star gives for token mismatches).
"""
import numpy as np

HID_TOL, LOGIT_TOL, MARGIN = 2e-2, 5e-2, 1e-2


def rel_err(g, o):
    return float(np.abs(g - o).max() / np.abs(o).max())


def gpu_trace(g, T, seq=0):
    """Run rounds until T tokens are committed for `seq`; every commit goes through dex_collapse with the GPU's own
    (token, branch).  Returns per-round records with the integer results, B of the new nodes and their
    stage-boundary hidden states (debug taps)."""
    N = len(g.depths)
    recs, n = [], 0
    while n < T:
        r = g.step(0)[seq]
        q = r.q_before
        B = g.tap_B(seq)
        nodes = [i for i in range((1 << q) - 1, (2 << q) - 1) if B[i] >= 0]
        rec = dict(q=q, rows=list(r.rows_per_stage)[:N], evals=int(r.layer_evals), crit=int(r.critical_layers),
                   exit_rows=int(r.exit_rows), nodes=nodes, u={i: int(B[i]) for i in nodes},
                   h={i: g.tap_hidden(i, seq)[-1].copy() for i in nodes}, committed=0,
                   anchor=list(r.anchor_tokens)[:N], mask=int(r.branch_mask))
        if r.match_k >= 0:
            rec.update(committed=1, token=int(r.token), k=int(r.match_k), top1=float(r.ref_top1), top2=float(r.ref_top2))
            g.collapse(seq, r.match_k, r.token)
            fsm = g.tap_fsm(seq).tolist()
            rec["fsm_after"] = fsm
            n += 1
        else:
            rec["q_after"] = int(r.q_after)
        recs.append(rec)
    return recs


def compare_with_oracle(recs, model, prompt, X, T, decs=True, lookahead=0, sample=None, hid_tol=HID_TOL,
                        max_forced_frac=0.10):
    """Replays the oracle with the GPU's exit decisions forced and compares every round.  Returns a summary dict
    (rounds, nodes, forced, worst hidden error); asserts on any violation."""
    from oracle import dex_decode
    force_u = {(ri, i): t for ri, rec in enumerate(recs) for i, t in rec["u"].items()}
    od = dex_decode(model, prompt, T, X, decs=decs, trace=True, force_u=force_u, lookahead=lookahead, sample=sample)
    assert len(od["rounds"]) == len(recs), (len(od["rounds"]), len(recs))
    N = len(X)
    n_nodes = n_forced = n_commit = 0
    worst_h = worst_gap = 0.0
    for ri, (g, o) in enumerate(zip(recs, od["rounds"])):
        assert g["q"] == o["q"], ri
        assert g["nodes"] == sorted(o["nodes"]), (ri, g["nodes"], o["nodes"])          # exactly the oracle's nodes
        assert g["rows"] == o["rows_per_stage"], ri
        assert g["evals"] == o["layer_evals"] and g["crit"] == o["critical_layers"] and g["exit_rows"] == o["exit_rows"], ri
        for i in g["nodes"]:
            n_nodes += 1
            worst_h = max(worst_h, rel_err(g["h"][i], o["h_out"][i]))
            assert o["u"][i] == g["u"][i]                                                # forced or equal
        for i, (own, tok, gap) in o.get("u_forced", {}).items():
            n_forced += 1
            worst_gap = max(worst_gap, gap)
            assert gap < MARGIN, f"round {ri} node {i}: gpu {tok} vs oracle {own}, oracle logit gap {gap:.4f} >= {MARGIN}"
        assert g["committed"] == o["committed"], ri
        if o["committed"]:
            n_commit += 1
            assert g["token"] == o["token"] and g["k"] == o["match_k"], (ri, g["token"], o["token"], g["k"], o["match_k"])
            # reported top-2 of the final-depth anchor: the fused exit's own reduction (tcgen05 accumulators)
            assert abs(g["top1"] - o["ref_top1"]) < LOGIT_TOL and abs(g["top2"] - o["ref_top2"]) < LOGIT_TOL, ri
            assert g["fsm_after"][0] == o["q_after"], ri
            if lookahead:
                assert [(g["mask"] >> k) & 1 for k in range(N - 1)] == [int(e) for e in o["explored"]], ri
        else:
            assert g["q_after"] == o["q_after"], ri
    assert worst_h < hid_tol, worst_h
    assert n_commit == T
    assert n_forced <= max(2, int(max_forced_frac * n_nodes)), (n_forced, n_nodes)
    return dict(rounds=len(recs), nodes=n_nodes, forced=n_forced, worst_h=worst_h, worst_gap=worst_gap,
                tokens=od["tokens"], oracle=od)


def check_ref_blocks(blocks, logits, tol=LOGIT_TOL):
    """`blocks` [n_blocks, 2] from Dex.tap_ref_blocks(): top-1 / top-2 of every 32 consecutive vocabulary ids as the
    fused exit epilogue reduced them; `logits` [V]: the oracle's final-depth logits of the same position."""
    V = len(logits)
    nb = (V + 31) // 32
    pad = np.full(nb * 32, -np.inf, dtype=np.float64)
    pad[:V] = logits
    srt = np.sort(pad.reshape(nb, 32), axis=1)
    want1, want2 = srt[:, -1], srt[:, -2]
    got = np.asarray(blocks, dtype=np.float64)[:nb]
    assert np.abs(got[:, 0] - want1).max() < tol, float(np.abs(got[:, 0] - want1).max())
    fin = np.isfinite(want2)
    assert np.abs(got[fin, 1] - want2[fin]).max() < tol
    return float(np.abs(got[:, 0] - want1).max())
