"""Sampling-mode DECS (Sec. 3.3; Alg. 2 lines 10-15; App. C.1):
y = argmax_v (l_v / tau + G_v) with a Gumbel(0,1) row shared by every depth of a slot chain, so the
final-depth reference is the exact Gumbel-Max sample of the unmasked final-depth logits.

Reading R24: the paper indexes the shared buffer by the slot root r(i); here the row is a
function of (seed, sequence, ABSOLUTE position of the token being decoded) only, drawn by a counter-based
generator that the CUDA side implements independently.  All slots that decode the same position share the
row (whatever their prefix); the committed token at position p is then argmax(l_final / tau + G_p), exactly
what AR sampling with the same generator produces, and G_p is independent of the committed prefix.
"""
import numpy as np

_M = np.uint64(0xFFFFFFFFFFFFFFFF)


def uniform_row(seed, seq, pos, V):
    """u_v in (0,1), 24 significant bits: splitmix64 finaliser of a counter built from (seed, seq, pos, v)."""
    v = np.arange(V, dtype=np.uint64)
    key = np.uint64(seed & 0xFFFFFFFF) ^ (np.uint64(seq) << np.uint64(56))
    ctr = (np.uint64(pos) << np.uint64(32)) + v + np.uint64(1)
    with np.errstate(over="ignore"):
        z = key + np.uint64(0x9E3779B97F4A7C15) * ctr
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return ((z >> np.uint64(41)).astype(np.float64) + 0.5) * 2.0 ** -23


def gumbel_row(seed, seq, pos, V):
    """G_v = -log(-log(u_v))  (Gumbel(0,1))."""
    return -np.log(-np.log(uniform_row(seed, seq, pos, V)))


def perturbed(logits, tau, g):
    """l / tau + G  (Alg. 2 line 13), in the dtype of the logits' accumulation (float64 here)."""
    return np.asarray(logits, dtype=np.float64) / float(tau) + g
