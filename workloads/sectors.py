"""Sector-size recipe of the synthetic workloads (SURVEY.md §8(c) reading r14/r16).

BASELINE.json config 2: "total dim 1024 split into 33 sectors q=0..32 with sizes
∝ exp(-(q-16)²/32), rounded, min 1".  Plain rounding does not sum to 1024, so
the sizes are fixed by the largest-remainder rule below; configs 3-5 use the
same law with the width scaled to the lattice.
"""
import math
import numpy as np


def binom(n, k):
    return math.comb(n, k) if 0 <= k <= n else 0


def gaussian_sectors(total, weights, caps=None):
    """Integer sector sizes ∝ ``weights`` summing to ``total``.

    x_q = total*w_q/Σw ; s_q = max(1, floor(x_q)) capped at caps[q]; the units
    still missing are handed out one each in decreasing order of frac(x_q)
    (ties → lower q, repeated passes if needed, never above the cap); if the
    minimum-1 rule overshot, units are taken one at a time from the currently
    largest sector (ties → lower q).
    """
    w = np.asarray(weights, dtype=np.float64)
    n = len(w)
    caps = [total] * n if caps is None else [int(c) for c in caps]
    x = total * w / w.sum()
    s = [min(max(1, int(math.floor(v))), caps[i]) for i, v in enumerate(x)]
    frac = [v - math.floor(v) for v in x]
    order = sorted(range(n), key=lambda i: (-frac[i], i))
    guard = 0
    while sum(s) < total:
        progressed = False
        for i in order:
            if sum(s) >= total:
                break
            if s[i] < caps[i]:
                s[i] += 1
                progressed = True
        guard += 1
        if not progressed or guard > total:
            raise ValueError("caps too small for requested total")
    while sum(s) > total:
        i = max(range(n), key=lambda j: (s[j], -j))
        if s[i] <= 1:
            raise ValueError("cannot reduce below one state per sector")
        s[i] -= 1
    return s
