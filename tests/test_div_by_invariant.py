"""The division by the invariant beta in the G assembly kernel (div_by_beta, csrc/cos_kernels_generic.cuh).

The kernel replaces u = x / beta by the sequence  y = RN(1 / beta) (taken once on the host);  q = RN(x y);
r = RN(x - beta q);  q = RN(q + r y);  r = RN(x - beta q);  u = RN(q + r y)  -- every step one IEEE operation (a product
or a fused multiply-add).  G must be bit-identical to the oracle's, which divides, so the sequence has to round like
the division for every operand the kernel feeds it (1e-200 < x < 1e200; the all-ones significand of beta is excluded
on the host).  Here the sequence is restated in exact rational arithmetic (Fraction -> float conversion rounds to
nearest even, like the hardware) and compared with Python's correctly rounded division on random and structured
operands: significands next to powers of two, sparse and dense bit patterns, quotients next to rounding boundaries.
The GPU side of the same claim is tests/test_gpu_parity.py::test_build_G_division_by_beta_bit_exact."""
import math
import random
from fractions import Fraction as F


def rn(x: F) -> float:
    return float(x)            # CPython converts a Fraction by a correctly rounded integer division


def div_by_invariant(x: float, beta: float) -> float:
    y = 1.0 / beta
    q = rn(F(x) * F(y))
    r = rn(F(x) - F(beta) * F(q))
    q = rn(F(q) + F(r) * F(y))
    r = rn(F(x) - F(beta) * F(q))
    return rn(F(q) + F(r) * F(y))


def all_ones(b: float) -> bool:
    m, _ = math.frexp(b)
    return int(m * 2 ** 53) == 2 ** 53 - 1


def structured_significands(rng):
    out = [1.0, math.nextafter(1.0, 2.0), math.nextafter(2.0, 0.0), math.nextafter(math.nextafter(2.0, 0.0), 0.0), 1.5, 1.25,
           4.0 / 3.0, 5.0 / 3.0, math.sqrt(2.0), 1.0 + 2.0 ** -26, 1.0 + 2.0 ** -27, 2.0 - 2.0 ** -26, 1.0 + 2.0 ** -51]
    for _ in range(40):
        k = rng.randrange(1, 52)
        out.append(1.0 + 2.0 ** -k)
        out.append(2.0 - 2.0 ** -k)
        out.append(1.0 + rng.randrange(1, 1 << 12) * 2.0 ** -52)          # just above a power of two
        out.append(2.0 - rng.randrange(2, 1 << 12) * 2.0 ** -52)          # just below
    return out


def test_sequence_rounds_like_the_division():
    rng = random.Random(20250107)
    sig = structured_significands(rng)
    cases = []
    for b in sig:                                  # structured divisor x structured dividend
        for a in sig:
            cases.append((a * 2.0 ** rng.randrange(-40, 40), b * 2.0 ** rng.randrange(-40, 40)))
    for _ in range(60000):                         # random significands, exponents inside the kernel's guard
        a = rng.uniform(1.0, 2.0) * 2.0 ** rng.randrange(-600, 600)
        b = rng.uniform(1.0, 2.0) * 2.0 ** rng.randrange(-60, 60)
        cases.append((a, b))
    for _ in range(20000):                         # quotients next to a rounding boundary: x = RN(q beta) for q near midpoints
        b = rng.choice(sig) * 2.0 ** rng.randrange(-8, 8)
        qq = rng.uniform(1.0, 2.0)
        cases.append((qq * b, b))
        cases.append((math.nextafter(qq * b, math.inf), b))
    checked = 0
    for x, b in cases:
        if all_ones(b) or not (1e-200 < x < 1e200):
            continue                               # the kernel takes the generic division there
        assert div_by_invariant(x, b) == x / b, (x.hex(), b.hex())
        checked += 1
    assert checked > 80000


def test_kernel_grid_values():
    """Operands of the shape the kernel sees: x = dtau (ntau - 1) with dtau in (0, beta], u = x / beta in (0, ntau - 1]."""
    rng = random.Random(7)
    for beta in (1.0 / 3.0, math.pi, 0.1, 7.0, 1e-3, 123.456, 8.0, 5.0, 2.0, 1.7e12, 2.0 ** -74):
        for ntau in (2, 33, 257, 512, 513):
            for _ in range(300):
                dtau = rng.uniform(0.0, beta) if rng.random() < 0.8 else beta * 2.0 ** -rng.randrange(1, 60)
                if dtau <= 0.0:
                    continue
                x = dtau * float(ntau - 1)
                assert div_by_invariant(x, beta) == x / beta, (x.hex(), beta.hex())
