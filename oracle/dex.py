"""O4: Depth Exploration Decoding, step by step (Alg. 1; Sec. 3.2
lines 196-208; Alg. 2 lines 454-482 greedy branch).  Notation follows the paper:
X = {d_0<...<d_{N-1}=L}, stage Pi_k = Layers(d_{k-1}, d_k], explore buffer B (here `u`),
FSM state q, anchor branches b_k with candidates u_k.

Loop body (reading R1 for the scrambled lines 13-16):
    H_q <- expand;  Z_q <- DECS;  B <- insert
    if ReachFinalDepth(q): (b,y) <- validate_and_commit; Y <- Y||y; stop?; collapse
    else: q <- advance(q)
"""
import numpy as np

from . import lattice as lt
from .ar import prefill
from .ead import check_X
from .gumbel import gumbel_row, perturbed
from .model import argmax_lowest


def dex_decode(model, prompt, T, X, decs=True, trace=False, state=None, force_tokens=None, sample=None, lookahead=0,
               force_u=None):
    """Returns dict with tokens [T], match_k [T] (anchor index b_k selected at each commit),
    rounds (list of per-round records) and totals.  `force_tokens` (optional [T]) replaces the
    committed token y (teacher forcing used by the GPU parity harness, R17) - never set when
    checking losslessness.  `sample` = (tau, seed, seq): sampling-mode DECS (Alg. 2 lines 10-15) with the
    shared Gumbel rows of oracle/gumbel.py (reading R24); None: greedy.  `lookahead` = P > 0: the sparse lattice of
    reading R26 ("prune low-value branches or construct sparse exploration lattices while preserving
    the final-depth commit invariant"): a node is expanded only if it lies at most P token positions ahead of the
    commit position and its parent was expanded; 0: the full lattice of Sec. 3.2.
    `force_u` (optional dict {(round index, node): token}) replaces the candidate token DECS decodes for that node
    (teacher forcing of EVERY exit decision, used by the GPU parity harness: reading R17b in DESIGN.md); the gap
    between the oracle's own arg-max and the forced token among the node's unmasked logits is recorded in
    rec["u_forced"][node] so that the harness can require it to be a near-tie.  Never set when checking
    losslessness or any other pin."""
    X = check_X(X, model.L)
    N = len(X)
    lo = [0] + X[:-1]                          # d_{k-1}, with d_{-1}=0
    prompt = [int(t) for t in prompt]
    ck, cv = state if state is not None else prefill(model, prompt)    # S <- init(x,{E_k})
    x = list(prompt)                           # committed tokens; x[n-1] is the next root input
    Y, match_k, rounds = [], [], []
    q = 0
    u = {}                                     # B: node -> candidate token
    h_out = {}                                 # node -> hidden at its stage boundary
    slot_kv = {}                               # slot root -> {layer: (k, v)}

    while len(Y) < T:
        n = len(x)
        new_nodes = lt.level_nodes(q)
        if lookahead > 0:                      # R26: position look-ahead cap; the anchor chain (offset 0) always survives
            new_nodes = [i for i in new_nodes
                         if lt.pos_offset(i) <= lookahead and (i == 0 or lt.parent(i) in u)]
        assert lt.anchor(q) in new_nodes
        rec = dict(q=q, n=n, nodes=new_nodes, rows_per_stage=[0] * N, layer_evals=0,
                   exit_rows=len(new_nodes), critical_layers=0)
        new_h, new_u, new_margin = {}, {}, {}
        # ---- expand (Alg. 1 line 5): every new node through its stage -------------------
        for i in new_nodes:
            m = lt.stage(i)
            pos = n - 1 + lt.pos_offset(i)
            if i == 0:
                h = model.embed_tok(x[n - 1])
            elif i % 2 == 1:                   # depth expansion
                h = h_out[lt.parent(i)].copy()
            else:                              # position expansion: parent's candidate is the prefix
                h = model.embed_tok(u[lt.parent(i)])
            anc = lt.ancestor_slots(i)
            sr = lt.slot_root(i)
            for l in range(lo[m], X[m]):
                ctx_k = list(ck[l]) + [slot_kv[a][l][0] for a in anc]
                ctx_v = list(cv[l]) + [slot_kv[a][l][1] for a in anc]
                assert len(ck[l]) == n - 1
                h, k, v = model.layer(l, h, pos, ctx_k, ctx_v)
                slot_kv.setdefault(sr, {})[l] = (k, v)
            new_h[i] = h
            rec["rows_per_stage"][m] += 1
            rec["layer_evals"] += X[m] - lo[m]
            rec["critical_layers"] = max(rec["critical_layers"], X[m] - lo[m])
        # ---- DECS (line 6, Alg. 2 greedy) + insert (line 7) -----------------------------
        ref_node = lt.anchor(N - 1)
        logits_ref = None
        for i in new_nodes:
            logits = model.exit_logits_at(new_h[i], lt.stage(i), N)   # adapters (if any) at non-final depths
            if sample is not None:             # Alg. 2 line 13: l / tau + G of the slot (position being decoded)
                tau, seed, sseq = sample
                logits = perturbed(logits, tau, gumbel_row(seed, sseq, n + lt.pos_offset(i), logits.shape[0]))
            masked = set()
            if decs and i != ref_node:         # Alg. 2 lines 1-4: reference node never masked
                masked = {u[a] if a in u else new_u[a] for a in lt.slot_chain_prior(i)}
            new_u[i] = argmax_lowest(logits, sorted(masked))
            if force_u is not None and (len(rounds), i) in force_u and int(force_u[(len(rounds), i)]) != new_u[i]:
                tok = int(force_u[(len(rounds), i)])
                gap = np.inf if tok in masked else float(logits[new_u[i]] - logits[tok])
                rec.setdefault("u_forced", {})[i] = (new_u[i], tok, gap)
                new_u[i] = tok
            if trace:                          # trace only: top-2 gap among the unmasked logits of node i
                lm = logits.copy()
                lm[sorted(masked)] = -np.inf
                top2 = np.sort(lm)[-2:]
                new_margin[i] = float(top2[1] - top2[0])
            if i == ref_node:
                logits_ref = logits
        u.update(new_u)
        h_out = new_h                          # only the frontier level has children
        if trace:
            rec["h_out"] = {i: new_h[i].copy() for i in new_nodes}
            rec["u"] = dict(new_u)
            rec["u_margin"] = dict(new_margin)
        # ---- commit / collapse or advance ------------------------------------------------
        if q == N - 1:                         # ReachFinalDepth(q)
            cand = [u[lt.anchor(k)] for k in range(N)]
            ref = cand[N - 1]
            srt = np.sort(logits_ref)
            rec["ref_top1"], rec["ref_top2"] = float(srt[-1]), float(srt[-2])
            if trace:
                rec["ref_logits"] = logits_ref.copy()
            y = ref if force_tokens is None else int(force_tokens[len(Y)])
            k_sel = N - 1                      # fallback b_{N-1}
            for k in range(N - 1):             # shallowest matching branch (R6) whose continuation was explored
                if cand[k] == y and (2 * lt.anchor(k) + 2) in u:      # (R26; always true on the full lattice)
                    k_sel = k
                    break
            Y.append(y)
            match_k.append(k_sel)
            x.append(y)
            for l in range(model.L):           # root slot joins the committed context C
                ck[l].append(slot_kv[0][l][0])
                cv[l].append(slot_kv[0][l][1])
            q_new, mp = lt.collapse_map(k_sel, N)
            u_before = u
            u = {j: u[o] for j, o in mp.items() if o in u}
            h_out = {j: h_out[o] for j, o in mp.items() if o in h_out}
            slot_kv = {j: slot_kv[o] for j, o in mp.items() if lt.slot_root(j) == j and o in slot_kv}
            rec.update(committed=1, token=y, match_k=k_sel, ref=ref, q_after=q_new,
                       explored=[(2 * lt.anchor(k) + 2) in u_before for k in range(N - 1)])
            q = q_new
        else:
            rec.update(committed=0, q_after=q + 1)
            q += 1                             # advance
        rounds.append(rec)

    return dict(tokens=np.array(Y, dtype=np.int64), match_k=np.array(match_k, dtype=np.int64),
                rounds=rounds, n_rounds=len(rounds),
                layer_evals=sum(r["layer_evals"] for r in rounds),
                critical_layers=sum(r["critical_layers"] for r in rounds),
                state=(ck, cv))
