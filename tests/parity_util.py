"""The parity rule of DESIGN.md §4 ("Tolerance and the exception rule"), in one place.

north_star: "GPU results must match the oracle on the same seeded inputs to a relative error of
<= 1e-10 in FP64".  `connected` is obtained by subtracting disconnected parts (reading R5), so for a
small fraction of configurations (near-singular G, clustered times) NO FP64 evaluation of the exact
sum is reproducible to 1e-10: the oracle's own FP64 result moves by more than that when the vertices
are merely relabelled (an exact symmetry of the sum).  The rule therefore is

  (1) |gpu - oracle64| <= 1e-10 * |oracle64|                         for every configuration, EXCEPT
  (2) configurations failing (1) must satisfy |gpu - truth| <= 6 * sigma, where truth is the same
      oracle run with long-double accumulators and sigma is the RMS deviation from truth of the FP64
      oracle over K = 16 random relabellings of the vertices (i.e. the GPU is no less accurate than
      FP64 arithmetic is for that configuration), and
  (3) the number of such exceptions is at most max(1, ceil(f * batch)) with f = 0.2 % by default and f = 1 % for
      the clustered-time workload cfg4, whose FP64 oracle itself misses the bar against its long-double mode on
      5 of 1024 configurations (DESIGN.md §4 lists the measured counts).

Every call appends its statistics to STATS; tests/conftest.py prints them in the terminal summary, so the number of
exceptions each test used is on record even under `pytest -q`.
"""
import math

import numpy as np

REL_TOL = 1e-10
K_RELABEL = 16
MAX_EXCEPTION_FRACTION = 0.002
CLUSTERED_EXCEPTION_FRACTION = 0.01
STATS = []          # one dict per check_parity call (label, batch, exceptions, ...)


def oracle_reference(oracle_mod, Gup, Gdn, U, u, loop_weight=1.0):
    a64, c64 = oracle_mod.eval_all_connected_lw(Gup, Gdn, U=U, u=u, loop_weight=loop_weight)
    return {"all": a64, "connected": c64}


def check_parity(oracle_mod, gpu, Gup, Gdn, U, u, which, ref64=None, max_fraction=MAX_EXCEPTION_FRACTION, label="",
                 loop_weight=1.0):
    """gpu: float64 [B] from the CUDA path.  Returns a dict of statistics; raises AssertionError."""
    gpu = np.asarray(gpu, dtype=np.float64)
    B = gpu.shape[0]
    assert np.all(np.isfinite(gpu)), "non-finite GPU result"
    if ref64 is None:
        ref64 = oracle_reference(oracle_mod, Gup, Gdn, U, u, loop_weight)[which]
    scale = np.abs(ref64)
    diff = np.abs(gpu - ref64)
    ok = diff <= REL_TOL * scale
    bad = np.nonzero(~ok)[0]
    stats = {"label": label, "which": which, "n": int(Gup.shape[1]), "batch": B, "max_rel_strict": float((diff[ok] / np.maximum(scale[ok], 1e-300)).max()) if ok.any() else 0.0,
             "exceptions": int(bad.size), "worst_exception_sigmas": 0.0}
    if not label.startswith("("):          # "(...)": a check that is expected to raise (tests of the rule itself)
        STATS.append(stats)
    if bad.size == 0:
        return stats
    assert bad.size <= max(1, math.ceil(max_fraction * B)), \
        f"{which}: {bad.size}/{B} configurations miss the 1e-10 bar (max rel {float((diff / scale).max()):.3e})"
    # conditioning of the exceptions: relabelling scatter of the FP64 oracle around the long-double truth
    Gu = Gup[bad]
    Gd = Gu if Gdn is None else Gdn[bad]
    uu = None if u is None else u[bad]
    pick = 0 if which == "all" else 1
    truth = oracle_mod.eval_all_connected_lw(Gu, None if Gdn is None else Gd, U=U, u=uu, loop_weight=loop_weight,
                                             f80=True)[pick]
    n = Gup.shape[1]
    rng = np.random.default_rng(12345)
    dev2 = np.zeros(bad.size)
    for _ in range(K_RELABEL):
        p = rng.permutation(n)
        Gu_p = np.ascontiguousarray(Gu[:, p][:, :, p])
        Gd_p = None if Gdn is None else np.ascontiguousarray(Gd[:, p][:, :, p])
        uu_p = None if uu is None else np.ascontiguousarray(uu[:, p])
        v = oracle_mod.eval_all_connected_lw(Gu_p, Gd_p, U=U, u=uu_p, loop_weight=loop_weight)[pick]
        dev2 += (v - truth) ** 2
    sigma = np.sqrt(dev2 / K_RELABEL)
    err = np.abs(gpu[bad] - truth)
    ratio = err / np.maximum(sigma, 1e-300)
    stats["worst_exception_sigmas"] = float(ratio.max())
    assert np.all(err <= 6.0 * sigma + REL_TOL * np.abs(truth)), \
        f"{which}: exception beyond 6 sigma of the FP64 relabelling scatter (worst {ratio.max():.2f} sigma)"
    return stats
