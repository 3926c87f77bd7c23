"""Pins of the oracle's Monte Carlo driver (reading R19); no GPU.

 * the generator against published known-answer vectors (tests/golden/philox4x32_10_kat.txt);
 * the 53-bit uniform map against its closed form;
 * the Metropolis rule against what it must sample: for order 2 on a 2 x 2 lattice the stationary distribution of the
   relative site is proportional to the time integral of |connected|, computed here by plain quadrature of the
   oracle's own integrand (a wrong acceptance ratio, a biased proposal or a stale weight all shift it);
 * order 1 with an equal-time diagonal: the weight is constant, so every proposal must be accepted."""
import os

import numpy as np
import pytest

from harness import workloads as wl

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_philox_known_answers(oracle_mod):
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) if not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert oracle_mod.philox4x32_10(v[0:4], v[4:6]) == tuple(v[6:10])


def test_u53_closed_form_and_uniformity(oracle_mod):
    assert oracle_mod.u53(0, 0) == 0.0
    assert oracle_mod.u53(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0 ** -53
    assert oracle_mod.u53(0x80000000, 0) == 0.5
    assert oracle_mod.u53(0, 1 << 11) == 2.0 ** -53
    x = np.array([oracle_mod.u53(*oracle_mod.philox4x32_10((i, 0, 0, 0), (7, 0))[:2]) for i in range(20000)])
    assert abs(x.mean() - 0.5) < 5 * np.sqrt(1 / 12 / x.size)
    assert abs((x < 0.25).mean() - 0.25) < 5 * np.sqrt(0.25 * 0.75 / x.size)


def test_constant_weight_accepts_everything(oracle_mod):
    """Order 1, g_diag != 0: connected = -U g_diag^2 whatever the vertex does."""
    table = wl.g0_table(4, 2.0, 0.0, 9)
    W = 50
    xy = np.zeros((W, 1, 2), dtype=np.int32)
    tau = np.full((W, 1), 0.3)
    r = oracle_mod.mc_run(xy, tau, table, 2.0, steps=20, seed=5, U=1.5, g_diag=0.4)
    assert r["accept"].all() and (r["accepted"] == 20).all()
    np.testing.assert_allclose(r["weight"], -1.5 * 0.4 * 0.4, rtol=1e-15)
    assert (r["sign_sum"] == -20).all()
    assert (r["xy"] != 0).any() and (r["tau"] != 0.3).all()


def test_metropolis_samples_the_integrand(oracle_mod):
    L, beta, ntau, U = 2, 1.5, 5, 2.0
    table = wl.g0_table(L, beta, -0.3, ntau)
    # exact marginal of the relative site d = x_0 - x_1: p(d) ~ int int dtau_0 dtau_1 |connected| (midpoint rule; the
    # integrand is piecewise polynomial in the times because the table is interpolated linearly)
    M = 240
    t = (np.arange(M) + 0.5) * beta / M
    t0, t1 = np.meshgrid(t, t, indexing="ij")
    p = np.zeros((L, L))
    for dx in range(L):
        for dy in range(L):
            xy = np.zeros((M * M, 2, 2), dtype=np.int32)
            xy[:, 0] = (dx, dy)
            tau = np.stack([t0.ravel(), t1.ravel()], axis=1)
            G, _ = oracle_mod.build_G(xy, tau, table, None, beta, 0.0)
            p[dx, dy] = np.abs(oracle_mod.eval_all_connected(G, None, U=U)[1]).sum()
    p /= p.sum()
    assert p.min() > 0.02                              # every relative site has visible weight in this set-up
    # chains: all walkers start from the same configuration, 80 single-vertex updates, the final states are used
    W, steps = 24000, 80
    xy0 = np.zeros((W, 2, 2), dtype=np.int32)
    tau0 = np.tile(np.array([[0.2, 1.1]]), (W, 1))
    r = oracle_mod.mc_run(xy0, tau0, table, beta, steps=steps, seed=2024, U=U)
    d = (r["xy"][:, 0] - r["xy"][:, 1]) % L
    for dx in range(L):
        for dy in range(L):
            f = np.mean((d[:, 0] == dx) & (d[:, 1] == dy))
            sigma = np.sqrt(p[dx, dy] * (1 - p[dx, dy]) / W)
            assert abs(f - p[dx, dy]) < 4.5 * sigma, (dx, dy, f, p[dx, dy], sigma)
    acc = r["accepted"].mean() / steps
    assert 0.05 < acc < 0.95                           # the rule is exercised both ways
    # the recorded weight is the connected value of the recorded state
    G, _ = oracle_mod.build_G(r["xy"][:64], r["tau"][:64], table, None, beta, 0.0)
    np.testing.assert_array_equal(r["weight"][:64], oracle_mod.eval_all_connected(G, None, U=U)[1])
