"""Definitions 1-5, Props 3, 6, 7 of PAPER.md Sec. 2 (integer helpers; O3 in SURVEY.md 8(c))."""
import numpy as np


def acceptance(exit_tokens):
    """Omega(t, l) = [e_l(t) == e_L(t)]  (Def. 1).  exit_tokens: [T, L] int,
    column l-1 = greedy token decoded at depth l."""
    e = np.asarray(exit_tokens)
    return (e == e[:, -1:]).astype(np.int8)


def ead(omega):
    """EAD(t) = min{l in [L]: Omega(t,l)=1}  (Eq. 1), 1-based depth."""
    return np.argmax(np.asarray(omega) == 1, axis=1) + 1


def stable_acceptance(omega):
    """Omega_stab(t,l)=1 iff Omega(t,n)=1 for all n in {l..L}  (Eq. 2)."""
    om = np.asarray(omega)
    return np.flip(np.cumprod(np.flip(om, axis=1), axis=1), axis=1).astype(np.int8)


def stable_ead(omega):
    """Eq. 3."""
    return ead(stable_acceptance(omega))


def check_X(X, L):
    X = list(X)
    if not X or X[-1] != L or any(b <= a for a, b in zip(X, X[1:])) or X[0] < 1:
        raise ValueError("exploration set must be strictly increasing in [1,L] and end at L (Def. 4)")
    return X


def ceil_X(l, X):
    """Depth ceiling: min{d in X: d >= l}  (Eq. 6)."""
    return min(d for d in X if d >= l)


def resolution(X, L):
    """Delta(X) = max_l (ceil_X(l) - l)  (Eq. 7)."""
    return max(ceil_X(l, X) - l for l in range(1, L + 1))


def workload_X(stab_omega_row, X):
    """W_X(t) = min{d in X: Omega_stab(t,d)=1}  (Eq. 8)."""
    return min(d for d in X if stab_omega_row[d - 1] == 1)


def speedup(L, W):
    """S = L*T / sum_t W(t)  (Eq. 12)."""
    W = np.asarray(W, dtype=np.float64)
    return L * len(W) / W.sum()


def speedup_X(L, ead_t, X):
    """Eq. 13."""
    return speedup(L, [ceil_X(int(e), X) for e in ead_t])


def speedup_lower(L, ead_t, X):
    """Leftmost-but-one term of Eq. 14."""
    D = resolution(X, L)
    return speedup(L, [min(int(e) + D, L) for e in ead_t])


def selection_cost(p_acc, s, L, discarded):
    """W_sel (Eq. 4): p*s_t + (1-p)*(L + sum of the v_t discarded selected exits, s_t first)."""
    return p_acc * s + (1.0 - p_acc) * (L + sum(discarded))


def first_match_depth(omega_row, X):
    """Vanilla DEX commit rule (reading R7): shallowest explored depth whose
    candidate equals the final-depth token (plain equality, not stable)."""
    return min(d for d in X if omega_row[d - 1] == 1)


def adapter_params(h, m=None):
    """P_ad = hm + mh + m + 2h + 1; m = 2h by default -> 4h^2 + 4h + 1."""
    m = 2 * h if m is None else m
    return h * m + m * h + m + 2 * h + 1
