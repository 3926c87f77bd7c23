"""Pins for the G-assembly oracle (oracle_build_G) and for the G0 table generator (workloads.g0_table).
None of these re-types the interpolation formula: they check grid-point exactness, exact reproduction
of tables that are linear in tau, antiperiodicity, translation invariance, the interpolation error
bound against a direct k-sum, and the table's closed-form end points.  No GPU.
"""
import os

import numpy as np
import pytest

from harness import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _direct_g0(L, beta, mu, x, y, tau):
    """G0(x, tau) for 0 < tau < beta by a direct sum over the k grid (no FFT, no table)."""
    k = 2.0 * np.pi * np.arange(L) / L
    eps = -2.0 * (np.cos(k)[:, None] + np.cos(k)[None, :]) - mu
    phase = np.cos(k[:, None] * x + k[None, :] * y)             # imaginary parts cancel
    f = np.where(eps >= 0, np.exp(-np.abs(eps) * tau) / (1 + np.exp(-beta * np.abs(eps))),
                 np.exp(-np.abs(eps) * (beta - tau)) / (1 + np.exp(-beta * np.abs(eps))))
    return -(phase * f).sum() / L ** 2


def test_table_end_points_and_density():
    for line in open(os.path.join(GOLD, "half_filling.txt")):
        if line.startswith("#"):
            continue
        L, beta, mu, n0_gold = line.split()
        L, beta, mu, n0_gold = int(L), float(beta), float(mu), float(n0_gold)
        ntau = 64
        T = wl.g0_table(L, beta, mu, ntau)
        k = 2.0 * np.pi * np.arange(L) / L
        eps = -2.0 * (np.cos(k)[:, None] + np.cos(k)[None, :]) - mu
        n0 = (1.0 / (np.exp(beta * eps) + 1.0)).mean()           # direct Fermi-function sum
        assert n0 == pytest.approx(n0_gold, abs=2e-14)
        assert T[0, 0, ntau - 1] == pytest.approx(-n0, abs=1e-14)            # G0(0, beta-) = -n0
        assert T[0, 0, 0] == pytest.approx(-(1.0 - n0), abs=1e-14)          # G0(0, 0+)  = -(1-n0)
        # sum over sites projects on k = 0: sum_x G0(x,tau) = G0(k=0,tau)
        e0 = -4.0 - mu
        tau = np.arange(ntau) * beta / (ntau - 1)
        ref = -np.exp(-e0 * tau) / (1 + np.exp(-beta * e0)) if e0 >= 0 else \
            -np.exp(e0 * (beta - tau)) / (np.exp(beta * e0) + 1)
        np.testing.assert_allclose(T.sum(axis=(0, 1)), ref, rtol=1e-11, atol=1e-13)


def test_table_matches_direct_k_sum():
    L, beta, mu, ntau = 8, 3.0, -0.3, 33
    T = wl.g0_table(L, beta, mu, ntau)
    for (x, y, k) in [(0, 0, 0), (1, 0, 5), (3, 7, 16), (4, 4, 32), (7, 1, 31)]:
        tau = k * beta / (ntau - 1)
        assert T[x, y, k] == pytest.approx(_direct_g0(L, beta, mu, x, y, tau), abs=1e-13)
    # inversion symmetry of the band: G0(x,y) = G0(-x,-y) = G0(y,x)
    np.testing.assert_allclose(T[1, 3], T[7, 5], atol=1e-14)
    np.testing.assert_allclose(T[1, 3], T[3, 1], atol=1e-14)


def test_grid_point_exactness_and_antiperiodicity(oracle_mod):
    """Vertices whose time differences fall exactly on table points must return table entries
    bit-for-bit (positive branch) and their negatives shifted by beta (negative branch)."""
    L, ntau, beta = 4, 9, 2.0                       # grid step 0.25: exactly representable
    rng = np.random.default_rng(0)
    T = rng.normal(size=(L, L, ntau))
    Td = rng.normal(size=(L, L, ntau))
    xy = np.array([[[0, 0], [1, 3], [2, 2]]], dtype=np.int32)
    tau = np.array([[0.25, 1.0, 1.75]])
    Gup, Gdn = oracle_mod.build_G(xy, tau, T, Td, beta, g_diag=0.125)
    h = beta / (ntau - 1)
    for i in range(3):
        for j in range(3):
            if i == j:
                assert Gup[0, i, j] == 0.125 and Gdn[0, i, j] == 0.125
                continue
            dx = (xy[0, i, 0] - xy[0, j, 0]) % L
            dy = (xy[0, i, 1] - xy[0, j, 1]) % L
            d = tau[0, i] - tau[0, j]
            if d > 0:
                k = int(round(d / h))
                assert Gup[0, i, j] == T[dx, dy, k] and Gdn[0, i, j] == Td[dx, dy, k]
            else:
                k = int(round((d + beta) / h))
                assert Gup[0, i, j] == -T[dx, dy, k] and Gdn[0, i, j] == -Td[dx, dy, k]


def test_equal_times_take_the_negative_branch(oracle_mod):
    """R9: tau_i == tau_j (i != j) is dtau = 0-, i.e. -T[beta-] (last table point)."""
    L, ntau, beta = 3, 5, 1.0
    T = np.arange(L * L * ntau, dtype=np.float64).reshape(L, L, ntau) + 1.0
    xy = np.array([[[0, 0], [1, 2]]], dtype=np.int32)
    tau = np.array([[0.5, 0.5]])
    Gup, _ = oracle_mod.build_G(xy, tau, T, None, beta)
    assert Gup[0, 0, 1] == -T[(0 - 1) % L, (0 - 2) % L, ntau - 1]
    assert Gup[0, 1, 0] == -T[1, 2, ntau - 1]


def test_linear_tables_are_reproduced(oracle_mod):
    """For a table that is linear in tau the 2-point interpolation is exact up to rounding."""
    L, ntau, beta = 5, 17, 4.0
    rng = np.random.default_rng(1)
    a, b = rng.normal(size=(L, L)), rng.normal(size=(L, L))
    tk = np.arange(ntau) * beta / (ntau - 1)
    T = a[:, :, None] + b[:, :, None] * tk[None, None, :]
    B, n = 16, 6
    xy = rng.integers(0, L, size=(B, n, 2)).astype(np.int32)
    tau = rng.uniform(0, beta, size=(B, n))
    Gup, Gdn = oracle_mod.build_G(xy, tau, T, None, beta)
    np.testing.assert_array_equal(Gup, Gdn)
    for bb in range(B):
        for i in range(n):
            for j in range(n):
                if i == j:
                    assert Gup[bb, i, j] == 0.0
                    continue
                dx, dy = (xy[bb, i] - xy[bb, j]) % L
                d = tau[bb, i] - tau[bb, j]
                ref = a[dx, dy] + b[dx, dy] * d if d > 0 else -(a[dx, dy] + b[dx, dy] * (d + beta))
                assert Gup[bb, i, j] == pytest.approx(ref, abs=1e-13)


def test_translation_invariance_and_interpolation_error(oracle_mod):
    L, beta, mu, ntau = 16, 5.0, 0.0, 512
    T = wl.g0_table(L, beta, mu, ntau)
    rng = np.random.default_rng(2)
    B, n = 8, 5
    xy = rng.integers(0, L, size=(B, n, 2)).astype(np.int32)
    tau = rng.uniform(0, beta, size=(B, n))
    G0, _ = oracle_mod.build_G(xy, tau, T, None, beta)
    shift = np.array([3, 11], dtype=np.int32)
    G1, _ = oracle_mod.build_G((xy + shift) % L, tau, T, None, beta)
    np.testing.assert_array_equal(G0, G1)                       # lattice translation: bit-exact
    # against the direct k-sum at the vertex's own tau: error <= h^2/8 * max|d2G/dtau2| <= h^2/8 * 16 * 1
    h = beta / (ntau - 1)
    for bb in range(2):
        for i in range(n):
            for j in range(n):
                if i == j:
                    continue
                dx, dy = (xy[bb, i] - xy[bb, j]) % L
                d = tau[bb, i] - tau[bb, j]
                ref = _direct_g0(L, beta, mu, dx, dy, d) if d > 0 else -_direct_g0(L, beta, mu, dx, dy, d + beta)
                assert abs(G0[bb, i, j] - ref) <= 2.0 * h * h + 1e-14


def test_workload_recipes_are_seeded_and_shaped():
    w = wl.baseline_config(1)
    assert (w.n, w.batch, w.L, w.ntau) == (4, 64, 16, 512) and w.xy.shape == (64, 4, 2)
    assert w.xy.dtype == np.int32 and w.tau.dtype == np.float64 and w.table.shape == (16, 16, 512)
    assert 0 <= w.xy.min() and w.xy.max() < 16 and 0 <= w.tau.min() and w.tau.max() < 5.0
    w2 = wl.baseline_config(1)
    np.testing.assert_array_equal(w.xy, w2.xy)
    np.testing.assert_array_equal(w.tau, w2.tau)
    w4 = wl.baseline_config(4, batch=256)
    assert w4.n == 12 and 0 <= w4.tau.min() and w4.tau.max() < 10.0
    # clustered: many near-coincident time pairs (sigma = 0.1) compared with a uniform draw
    d = np.abs(w4.tau[:, :, None] - w4.tau[:, None, :])[:, np.triu_indices(12, 1)[0], np.triu_indices(12, 1)[1]]
    assert (d < 0.2).mean() > 3 * (0.2 * 2 / 10.0) * 0.5
    w5 = wl.baseline_config(5, batch=8)
    assert w5.G.shape == (8, 15, 15) and w5.u.shape == (8, 15)
    assert abs(np.diagonal(w5.G, axis1=1, axis2=2).mean() - 0.5) < 0.2
    assert wl.sweep_batch(8) == 4096 and wl.sweep_batch(13) == 1024 and wl.sweep_batch(16) == 256
