"""The binary expansion tree of PAPER.md Sec. 3.2 (lines 196-206), heap reading R2.

Node i >= 0; depth child 2i+1 ("keeps the same token position and forwards its hidden state
to the next explorer"), position child 2i+2 ("uses the current candidate token as the prefix
for the next token position and starts that position from E_0").  ETK_0 -> ETK_1 (depth),
ETK_2 (position) as in PAPER.md:198-200.  All helpers walk the path explicitly.
"""


def path(i):
    """Moves from the root to node i: list of 'D' / 'P'."""
    mv = []
    while i > 0:
        mv.append('D' if i % 2 == 1 else 'P')
        i = (i - 1) // 2
    return mv[::-1]


def parent(i):
    return (i - 1) // 2


def level(i):
    return len(path(i))


def stage(i):
    """Explorer index of node i = number of trailing depth moves."""
    m = 0
    for mv in reversed(path(i)):
        if mv != 'D':
            break
        m += 1
    return m


def pos_offset(i):
    """Token position of node i relative to the commit position p_c."""
    return path(i).count('P')


def slot_root(i):
    """First node of i's slot chain: strip the trailing depth moves."""
    while i > 0 and i % 2 == 1:
        i = (i - 1) // 2
    return i


def slot_chain_prior(i):
    """Prior(i): shallower nodes of the same slot chain (Alg. 2 line 1)."""
    r, out, j = slot_root(i), [], slot_root(i)
    while j != i:
        out.append(j)
        j = 2 * j + 1
    return out


def ancestor_slots(i):
    """Slot roots whose K/V node i attends to besides the committed context and itself:
    the slot of the node at which each position move on i's root path was taken."""
    out, j = [], 0
    for mv in path(i):
        if mv == 'P':
            out.append(slot_root(j))
        j = 2 * j + (1 if mv == 'D' else 2)
    return out


def prefix_tokens_nodes(i):
    """Nodes whose candidate tokens form i's branch prefix after the committed context
    (one per position move), in position order."""
    out, j = [], 0
    for mv in path(i):
        if mv == 'P':
            out.append(j)
        j = 2 * j + (1 if mv == 'D' else 2)
    return out


def level_nodes(q):
    """Nodes created by the round at FSM state q (tree level q)."""
    return list(range(2 ** q - 1, 2 ** (q + 1) - 1))


def anchor(k):
    """Anchor-path node at stage k: 2^k - 1."""
    return 2 ** k - 1


def rows_per_stage(q, N):
    out = [0] * N
    for i in level_nodes(q):
        out[stage(i)] += 1
    return out


def collapse_map(k, N):
    """Survivors after a commit that matched anchor index k:
    the sub-tree hanging off the position child of anchor node 2^k-1, re-rooted at 0.
    Returns (q_new, {new_index: old_index}).  Written as a sub-tree walk, not the closed form."""
    if k >= N - 1:
        return 0, {}                         # fallback b_{N-1}: nothing reusable (R4)
    root_old = 2 * anchor(k) + 2
    q_new = N - 1 - k
    mp, frontier = {0: root_old}, [0]
    while frontier:
        nxt = []
        for j in frontier:
            for c_new, c_old in ((2 * j + 1, 2 * mp[j] + 1), (2 * j + 2, 2 * mp[j] + 2)):
                if c_new < 2 ** q_new - 1:
                    mp[c_new] = c_old
                    nxt.append(c_new)
        frontier = nxt
    return q_new, mp
