"""Writes halfvertex_connected_counts.txt from the integer recursion alone (no oracle, no CUDA).

Half-vertex formulation (reading R18): n' interaction lines, m = 2n' half-vertices, one species.  Every
permutation of the half-vertices of a set of k lines is a diagram on that set, so D(k) = (2k)!; the number c(n') of
permutations whose interaction-line graph is connected follows from the same subset recursion the method uses
(component of line 0 has k lines): c(n') = (2n')! - sum_{k=1}^{n'-1} C(n'-1, k-1) c(k) (2(n'-k))!.
"""
from math import comb, factorial
import os

c = {}
for n in range(1, 7):
    c[n] = factorial(2 * n) - sum(comb(n - 1, k - 1) * c[k] * factorial(2 * (n - k)) for k in range(1, n))
with open(os.path.join(os.path.dirname(__file__), "halfvertex_connected_counts.txt"), "w") as f:
    f.write("# n'  permutations of the 2n' half-vertices whose interaction-line graph is connected\n")
    for n in range(1, 7):
        f.write(f"{n} {c[n]}\n")
