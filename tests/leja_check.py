"""Independent check of the Leja-point sequence on [-2, 2] ("Leja points (see [11])"; reading c2):
    l_k = argmax_{x in [-2,2]} prod_{j<k} |x - l_j|.

Neither the oracle's bisection nor the library's safeguarded Newton is used here.  Between two neighbouring nodes
log prod |x - l_j| is strictly concave (a sum of concave logs), so the maximum over [-2,2] is the largest of the
per-gap maxima; each of those is bracketed by a vectorised golden-section search in float64 and polished in mpmath.
"""
from __future__ import annotations

import mpmath
import numpy as np


def gap_maxima(prev: np.ndarray):
    """Per-gap maximiser and maximum of sum_j log|x - prev_j| for the gaps of sort(prev) (float64 golden section)."""
    s = np.sort(np.asarray(prev, dtype=np.float64))
    a, b = s[:-1].copy(), s[1:].copy()
    gr = (np.sqrt(5.0) - 1.0) / 2.0

    def logp(x):
        return np.sum(np.log(np.abs(x[:, None] - s[None, :])), axis=1)

    c, d = b - gr * (b - a), a + gr * (b - a)
    fc, fd = logp(c), logp(d)
    for _ in range(90):
        left = fc > fd
        b = np.where(left, d, b)
        a = np.where(left, a, c)
        c, d = b - gr * (b - a), a + gr * (b - a)
        fc, fd = logp(c), logp(d)
    x = 0.5 * (a + b)
    return x, logp(x)


def check_sequence(l: np.ndarray, first: int = 4, margin: float = 1e-7):
    """Asserts that every l[k], k >= first, is the global maximiser given l[:k]; returns the smallest
    log-gap between the winning gap and the runner-up (how unambiguous the choices are)."""
    mpmath.mp.dps = 40
    worst = np.inf
    for k in range(first, len(l)):
        prev = l[:k]
        x, fx = gap_maxima(prev)
        best = int(np.argmax(fx))
        mine = float(np.sum(np.log(np.abs(l[k] - prev))))
        # (1) the point sits in the winning gap and reaches its maximum
        s = np.sort(prev)
        assert s[best] < l[k] < s[best + 1], (k, l[k], s[best], s[best + 1])
        assert mine >= fx[best] - 1e-10, (k, mine, fx[best])
        # (2) the stationary point of the winning gap, polished in 40-digit arithmetic, is l[k] to double precision
        nodes = [mpmath.mpf(float(t)) for t in prev]
        root = mpmath.findroot(lambda t: mpmath.fsum(1 / (t - u) for u in nodes), mpmath.mpf(float(x[best])),
                               tol=1e-30, maxsteps=50)
        assert abs(float(root) - l[k]) <= 4e-15, (k, float(root), l[k])
        # (3) no other gap comes close: the choice is unambiguous in double precision
        others = np.delete(fx, best)
        gap = fx[best] - others.max()
        assert gap > margin, (k, gap)
        worst = min(worst, gap)
    return worst
