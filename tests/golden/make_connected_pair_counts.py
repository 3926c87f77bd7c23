"""Writes connected_pair_counts.txt from the integer recursion alone (no oracle, no CUDA)."""
from math import comb, factorial
import os

c = {}
for n in range(1, 8):
    c[n] = factorial(n) ** 2 - sum(comb(n - 1, k - 1) * c[k] * factorial(n - k) ** 2
                                   for k in range(1, n))
with open(os.path.join(os.path.dirname(__file__), "connected_pair_counts.txt"), "w") as f:
    f.write("# n  connected pairs (sigma_up, sigma_dn); see README.md\n")
    for n in range(1, 8):
        f.write(f"{n} {c[n]}\n")
