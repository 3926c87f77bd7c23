"""Ranked-zeta (fast subset convolution) logarithm of the all-diagram sums -- the strictly O(n^2 2^n) route to the
connected value that SURVEY.md 8(f4) names as an alternative to the subset recursion of the paper's Ref. [9].

TEST INFRASTRUCTURE / EXPERIMENT ONLY (numpy, FP64): used by tests/test_ranked_zeta.py to decide whether a CUDA kernel
of this shape is worth building.  It is NOT part of the oracle's parity path and nothing in the product imports it.

With S' a subset of the vertices 1..n-1 (m = n - 1 bits), D0[S'] = D[S' + {0}], D1[S'] = D[S'], the connected values
solve C' * D1 = D0 in the subset-convolution algebra.  Ranked zeta transform: f^[k][S] = sum_{T subset S, |T| = k} f[T]
turns the subset convolution into a product of polynomials in a rank variable z at every S, so
  c^(S, z) = D0^(S, z) / D1^(S, z)   (power series division, D1^(S, 0) = D[empty] = 1), and
  C'[full] = sum_S (-1)^{m - |S|} [z^m] c^(S, z)                      (Moebius inversion at the full set, rank m).
Cost: 2 (m+1) m 2^(m-1) additions for the transforms + about m^2 2^m / 2 FMAs for the divisions.
The coefficients [z^m] c^(S, z) of the strict subsets S are "garbage" (products of D's on OVERLAPPING vertex sets)
that cancels only in the signed sum; `amplification` returns sum_S |[z^m] c^(S, z)| / |C'[full]|, the factor by which
rounding errors are magnified.
"""
import numpy as np


def connected_ranked_zeta(D, n):
    """D: [2^n] all-diagram sums D[S] (oracle.DC).  Returns (connected, amplification)."""
    m = n - 1
    N = 1 << m
    idx = np.arange(N)
    pc = np.array([bin(i).count("1") for i in range(N)])
    f0 = np.zeros((m + 1, N))
    f1 = np.zeros((m + 1, N))
    f0[pc, idx] = D[2 * idx + 1]
    f1[pc, idx] = D[2 * idx]
    for b in range(m):                                   # zeta transform, one vertex at a time
        hi = idx[(idx >> b) & 1 == 1]
        f0[:, hi] += f0[:, hi ^ (1 << b)]
        f1[:, hi] += f1[:, hi ^ (1 << b)]
    c = np.zeros((m + 1, N))
    for k in range(m + 1):                               # power-series division at every S (f1[0] = D[empty] = 1)
        acc = f0[k].copy()
        for j in range(1, k + 1):
            acc -= f1[j] * c[k - j]
        c[k] = acc
    sign = np.where((m - pc) % 2 == 0, 1.0, -1.0)
    value = float((sign * c[m]).sum())
    return value, float(np.abs(c[m]).sum() / abs(value)) if value != 0.0 else float("inf")
