"""GPU test of the on-device Monte Carlo driver (cos_mc_run) against the oracle's driver on the same
seed: the accept / reject history and the final configurations must agree bit for bit, except where the oracle's own
margin shows a tie within the FP64 parity tolerance (then that walker's later history is not comparable and it is
only required to hold a valid state)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TIE = 1e-9          # |margin| below this: a decision another FP64 summation order may take the other way


@pytest.mark.parametrize("n,walkers,steps", [(1, 64, 10), (2, 777, 40), (5, 600, 30), (8, 333, 25), (10, 300, 20),
                                             (11, 40, 8), (14, 6, 4)])
def test_mc_matches_oracle(oracle_mod, n, walkers, steps):
    import torch
    from paper_2501_00675_b200 import api, build
    from harness import workloads as wl
    build.build()
    L, beta, ntau, U, seed = 8, 4.0, 65, 2.5, 1234567 + n
    table = wl.g0_table(L, beta, -0.4, ntau)
    rng = np.random.default_rng(n)
    xy0 = rng.integers(0, L, size=(walkers, n, 2)).astype(np.int32)
    tau0 = rng.uniform(0, beta, size=(walkers, n))
    g_diag = 0.3 if n == 1 else 0.0
    ref = oracle_mod.mc_run(xy0, tau0, table, beta, steps=steps, seed=seed, U=U, g_diag=g_diag)
    with api.Context() as c:
        c.set_g0_table(torch.from_numpy(table).cuda(), beta)
        xy = torch.from_numpy(xy0.copy()).cuda()
        tau = torch.from_numpy(tau0.copy()).cuda()
        weight = torch.empty(walkers, dtype=torch.float64, device="cuda")
        hist = torch.zeros((steps, walkers), dtype=torch.uint8, device="cuda")
        accepted = torch.empty(walkers, dtype=torch.int64, device="cuda")
        sign_sum = torch.empty(walkers, dtype=torch.float64, device="cuda")
        c.mc_run(xy, tau, weight, steps, seed, U=U, g_diag=g_diag, d_accept_hist=hist, d_accepted=accepted,
                 d_sign_sum=sign_sum)
        torch.cuda.synchronize()
        assert c.last_launch_count() >= 4 * steps
    h = hist.cpu().numpy()
    same = (h == ref["accept"])
    first_bad = np.where(same.all(axis=0), steps, np.argmin(same, axis=0))      # first differing step per walker
    diverged = np.nonzero(first_bad < steps)[0]
    for w in diverged:                                   # a difference must start at a tie of the oracle's own decision
        assert abs(ref["margin"][first_bad[w], w]) < TIE, (w, first_bad[w], ref["margin"][first_bad[w], w])
    assert len(diverged) <= max(1, walkers // 100)
    good = np.setdiff1d(np.arange(walkers), diverged)
    np.testing.assert_array_equal(xy.cpu().numpy()[good], ref["xy"][good])
    np.testing.assert_array_equal(tau.cpu().numpy()[good], ref["tau"][good])
    np.testing.assert_array_equal(accepted.cpu().numpy()[good], ref["accepted"][good])
    np.testing.assert_array_equal(sign_sum.cpu().numpy()[good], ref["sign_sum"][good])
    np.testing.assert_allclose(weight.cpu().numpy()[good], ref["weight"][good], rtol=1e-9)
    assert 0 < h.mean() <= 1.0
    # whatever the history, every walker ends in a state whose recorded weight is its connected value
    G, _ = oracle_mod.build_G(xy.cpu().numpy(), tau.cpu().numpy(), table, None, beta, g_diag)
    np.testing.assert_allclose(weight.cpu().numpy(), oracle_mod.eval_all_connected(G, None, U=U)[1], rtol=1e-9)
