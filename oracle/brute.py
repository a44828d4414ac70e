"""Brute-force enumeration used to pin the nucleus rule (oracle; test infrastructure).

PAPER.md:92: S_nuc "is the smallest prefix of B_res, sorted by p~ descending,
whose cumulative mass reaches p".  Independent characterisation, checked by
exhaustive enumeration on tiny inputs: among ALL subsets of B_res with mass
>= p the nucleus has minimum cardinality, and among all subsets of that
cardinality it has maximum mass.  Pure-Python loops, exact rationals optional.
"""
from itertools import combinations


def min_cardinality_max_mass(probs, p):
    """probs: dict {block: mass}.  Returns (k, best_mass, argbest sets) where k
    is the smallest subset size reaching mass >= p and best_mass the largest
    mass any k-subset reaches."""
    items = sorted(probs)
    for k in range(0, len(items) + 1):
        best, arg = -1.0, []
        for sub in combinations(items, k):
            m = sum(probs[b] for b in sub)
            if m > best + 1e-15:
                best, arg = m, [set(sub)]
            elif abs(m - best) <= 1e-15:
                arg.append(set(sub))
        if best >= p:
            return k, best, arg
    return len(items), sum(probs.values()), [set(items)]


def topk_by_enumeration(scores, k):
    """Eq. 6 by exhaustion: the k-subset with the largest score sum, ties broken
    towards lexicographically smaller index tuples (== lower index first)."""
    items = list(range(len(scores)))
    best, arg = None, None
    for sub in combinations(items, k):
        key = (sum(scores[b] for b in sub), tuple(-b for b in sub))
        if best is None or key > best:
            best, arg = key, sub
    return set(arg) if arg is not None else set()
