"""Fold assignment (test infrastructure).  Integer-only so that it is bit-exact in any
language (reading G13; PAPER.md:110, 283 say only "same
cross-validation folds").

SplitMix64(seed) -> Fisher-Yates permutation pi (j = next() mod (i+1), i = n-1..1)
-> foldid[pi[i]] = i mod V.
"""
import numpy as np

_MASK = (1 << 64) - 1


def splitmix64_stream(seed):
    """Generator of SplitMix64 outputs (Steele, Lea & Flood 2014), Python ints mod 2^64."""
    x = seed & _MASK
    while True:
        x = (x + 0x9E3779B97F4A7C15) & _MASK
        z = x
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK
        z = z ^ (z >> 31)
        yield z


def make_folds(n, V, seed):
    """int32 foldid[n] with values 0..V-1; fold sizes differ by at most one."""
    if V < 2 or V > n:
        raise ValueError("need 2 <= V <= n")
    g = splitmix64_stream(seed)
    pi = list(range(n))
    for i in range(n - 1, 0, -1):
        j = next(g) % (i + 1)
        pi[i], pi[j] = pi[j], pi[i]
    foldid = np.empty(n, dtype=np.int32)
    for i in range(n):
        foldid[pi[i]] = i % V
    return foldid
