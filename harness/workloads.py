"""Seeded synthetic inputs for the CoS hot path (numpy only).

This module holds NONE of the method's arithmetic: it tabulates the free propagator that is an
INPUT of the boundary (`cos_set_g0_table` takes the table as given), draws vertex configurations
and dense test matrices, and names the BASELINE.json configurations.  Both the CUDA path's callers
(tests, bench.py, smoke) and the oracle's callers use it, so that the two sides always see the
same bytes.  Recipe: DESIGN.md "Inputs" (readings R8 and R15).

The paper measures on no public dataset (PAPER.md P:91 only says "function-calls of the graph");
everything here is synthetic with the shapes BASELINE.json `configs` names.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np


def g0_table(L: int, beta: float, mu: float, ntau: int, t: float = 1.0) -> np.ndarray:
    """Free lattice propagator G0(x, tau_k) of the 2D square-lattice tight-binding band.

    G0(k,tau) = -exp(-eps_k tau) / (1 + exp(-beta eps_k)),  eps_k = -2t(cos kx + cos ky) - mu,
    on tau_k = k*beta/(ntau-1), k = 0..ntau-1 (the end points stand for 0+ and beta-), and
    G0(x,tau) = L^-2 sum_k exp(i k.x) G0(k,tau) (real by inversion symmetry).
    Returns float64 [L][L][ntau], tau fastest (layout of SURVEY §8(a) a0).
    """
    k = 2.0 * np.pi * np.arange(L) / L
    eps = -2.0 * t * (np.cos(k)[:, None] + np.cos(k)[None, :]) - mu          # [L, L]
    tau = np.arange(ntau, dtype=np.float64) * (beta / (ntau - 1))              # [ntau]
    e = eps[:, :, None]
    tt = tau[None, None, :]
    # overflow-safe: eps >= 0: exp(-eps tau)/(1+exp(-beta eps)); eps < 0: exp(eps (beta-tau))/(exp(beta eps)+1)
    pos = np.exp(-np.abs(e) * tt) / (1.0 + np.exp(-beta * np.abs(e)))
    neg = np.exp(-np.abs(e) * (beta - tt)) / (1.0 + np.exp(-beta * np.abs(e)))
    gk = -np.where(e >= 0, pos, neg)                                           # [L, L, ntau]
    gx = np.fft.ifft2(gk, axes=(0, 1)).real
    return np.ascontiguousarray(gx, dtype=np.float64)


@dataclass
class Workload:
    name: str
    n: int
    batch: int
    kind: str                      # "hubbard" (vertices + table) or "dense" (matrices given)
    U: float
    seed: int
    # hubbard
    L: int = 0
    beta: float = 0.0
    mu: float = 0.0
    ntau: int = 0
    g_diag: float = 0.0
    xy: Optional[np.ndarray] = None        # int32 [B, n, 2]
    tau: Optional[np.ndarray] = None       # float64 [B, n]
    _table: Optional[np.ndarray] = field(default=None, repr=False)
    # dense
    G: Optional[np.ndarray] = None         # float64 [B, n, n]
    u: Optional[np.ndarray] = None         # float64 [B, n] per-vertex couplings (R10: diag of V)

    @property
    def table(self) -> np.ndarray:
        if self._table is None:
            self._table = _cached_table(self.L, self.beta, self.mu, self.ntau)
        return self._table


_TABLES: dict = {}


def _cached_table(L, beta, mu, ntau):
    key = (L, float(beta), float(mu), ntau)
    if key not in _TABLES:
        _TABLES[key] = g0_table(L, beta, mu, ntau)
    return _TABLES[key]


def hubbard_workload(name, n, batch, L, beta, U, mu, ntau, seed, clustered=False) -> Workload:
    """Uniform (or R15-clustered) vertices.  Draw order: all sites, all times, then mixture draws."""
    rng = np.random.default_rng(seed)
    xy = rng.integers(0, L, size=(batch, n, 2), dtype=np.int64).astype(np.int32)
    tau = rng.uniform(0.0, beta, size=(batch, n))
    if clustered:
        # R15: per configuration 4 centres ~ U[0,beta); each vertex keeps its uniform time with
        # probability 1/2, else centre (uniform among 4) + N(0, 0.1^2), wrapped into [0, beta).
        centres = rng.uniform(0.0, beta, size=(batch, 4))
        use_cluster = rng.random(size=(batch, n)) < 0.5
        which = rng.integers(0, 4, size=(batch, n))
        jitter = rng.normal(0.0, 0.1, size=(batch, n))
        clustered_tau = np.mod(np.take_along_axis(centres, which, axis=1) + jitter, beta)
        tau = np.where(use_cluster, clustered_tau, tau)
    tau = np.ascontiguousarray(tau, dtype=np.float64)
    return Workload(name=name, n=n, batch=batch, kind="hubbard", U=U, seed=seed, L=L, beta=beta,
                    mu=mu, ntau=ntau, g_diag=0.0, xy=np.ascontiguousarray(xy), tau=tau)


def dense_workload(name, n, batch, U, seed) -> Workload:
    """BASELINE config 5: G = N(0, 1/n) + 0.5 I, V = U (1 + 0.1 N(0,1)) symmetrised; u = diag V (R10)."""
    rng = np.random.default_rng(seed)
    G = rng.normal(0.0, 1.0 / np.sqrt(n), size=(batch, n, n)) + 0.5 * np.eye(n)[None]
    V = U * (1.0 + 0.1 * rng.normal(0.0, 1.0, size=(batch, n, n)))
    V = 0.5 * (V + np.transpose(V, (0, 2, 1)))
    u = np.ascontiguousarray(np.diagonal(V, axis1=1, axis2=2), dtype=np.float64)
    return Workload(name=name, n=n, batch=batch, kind="dense", U=U, seed=seed,
                    G=np.ascontiguousarray(G, dtype=np.float64), u=u)


# BASELINE.json `configs`, in order.  batch=None -> the configuration's own batch.
_BASELINE = {
    1: dict(n=4, batch=64, L=16, beta=5.0, U=2.0, mu=0.0, ntau=512, seed=0),
    2: dict(n=8, batch=4096, L=16, beta=5.0, U=2.0, mu=0.0, ntau=512, seed=1),
    3: dict(n=10, batch=16384, L=32, beta=8.0, U=4.0, mu=-0.5, ntau=1024, seed=2),
    4: dict(n=12, batch=4096, L=32, beta=10.0, U=4.0, mu=0.0, ntau=1024, seed=3, clustered=True),
    5: dict(n=15, batch=512, U=4.0, seed=4),
}


def baseline_config(idx: int, batch: Optional[int] = None) -> Workload:
    """BASELINE.json configs[idx-1] (idx = 1..5); `batch` overrides the size, same recipe and seed."""
    p = dict(_BASELINE[idx])
    if batch is not None:
        p["batch"] = int(batch)
    name = f"cfg{idx}_n{p['n']}_b{p['batch']}"
    if idx == 5:
        return dense_workload(name, p["n"], p["batch"], p["U"], p["seed"])
    return hubbard_workload(name, **p)


def sweep_batch(n: int) -> int:
    """SURVEY §8(d) sweep sizes: 4096 (n<=12), 1024 (13-14), 512 (15), 256 (16)."""
    if n <= 12:
        return 4096
    if n <= 14:
        return 1024
    return 512 if n == 15 else 256


def sweep_workload(n: int, kind: str = "hubbard", batch: Optional[int] = None) -> Workload:
    """One point of the n = 8..16 sweep: cfg-3-style Hubbard or cfg-5-style dense inputs, seed 100+n."""
    b = sweep_batch(n) if batch is None else int(batch)
    if kind == "dense":
        return dense_workload(f"sweep_dense_n{n}_b{b}", n, b, 4.0, 100 + n)
    return hubbard_workload(f"sweep_hubbard_n{n}_b{b}", n, b, L=32, beta=8.0, U=4.0, mu=-0.5,
                            ntau=1024, seed=100 + n)
