"""GPU parity tests: the CUDA path, called through the C-ABI binding, against the CPU oracle element by
element on the same seeded inputs.  Every test here needs a B200 (`-m gpu`).  Tolerances: G assembly
bit-exact (same FP64 operations in the same order, one explicit fma); evaluation by the rule in
tests/parity_util.py (1e-10 relative, conditioning-aware exceptions)."""
import numpy as np
import pytest

from parity_util import CLUSTERED_EXCEPTION_FRACTION, MAX_EXCEPTION_FRACTION, check_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_mod():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device: the CUDA path has no CPU fallback")
    from paper_2501_00675_b200 import build
    build.build()          # compiles the in-tree library only when it is missing or older than its sources
    return torch


@pytest.fixture(scope="module")
def ctx(torch_mod):
    from paper_2501_00675_b200 import api
    c = api.Context()
    yield c
    c.close()


def _dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _gpu_eval(torch, ctx, Gup, Gdn, U, u, which):
    dGup = _dev(torch, Gup)
    dGdn = dGup if Gdn is None else _dev(torch, Gdn)
    du = None if u is None else _dev(torch, u)
    out = torch.empty(Gup.shape[0], dtype=torch.float64, device="cuda")
    fn = ctx.eval_all if which == "all" else ctx.eval_connected
    fn(dGup, dGdn, out, U=U, d_u=du)
    torch.cuda.synchronize()
    assert ctx.last_launch_count() >= 1
    return out.cpu().numpy()


def _workload_mats(oracle_mod, w):
    if w.kind == "hubbard":
        Gup, _ = oracle_mod.build_G(w.xy, w.tau, w.table, None, w.beta, w.g_diag)
        return Gup, None, w.U, None
    return w.G, None, w.U, w.u


# ------------------------------------------------------------------------------------------ a1
@pytest.mark.parametrize("cfg,batch", [(1, 64), (2, 4096), (3, 2048), (4, 1024)])
def test_build_G_bit_exact(torch_mod, ctx, oracle_mod, cfg, batch):
    from harness import workloads as wl
    torch = torch_mod
    w = wl.baseline_config(cfg, batch=batch)
    ref_up, ref_dn = oracle_mod.build_G(w.xy, w.tau, w.table, None, w.beta, 0.0)
    ctx.set_g0_table(_dev(torch, w.table), w.beta)
    Gup = torch.empty((batch, w.n, w.n), dtype=torch.float64, device="cuda")
    ctx.build_G(_dev(torch, w.xy), _dev(torch, w.tau), Gup, None, g_diag=0.0)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(Gup.cpu().numpy(), ref_up)


def test_build_G_two_tables_diag_and_ragged(torch_mod, ctx, oracle_mod):
    torch = torch_mod
    rng = np.random.default_rng(0)
    L, ntau, beta, B, n = 7, 33, 3.7, 37, 5          # odd sizes: ragged tail of the thread grid
    Tu, Td = rng.normal(size=(L, L, ntau)), rng.normal(size=(L, L, ntau))
    xy = rng.integers(0, L, size=(B, n, 2)).astype(np.int32)
    tau = rng.uniform(0, beta, size=(B, n))
    tau[3, 1] = tau[3, 4]                            # equal times: R9 negative branch
    ref_up, ref_dn = oracle_mod.build_G(xy, tau, Tu, Td, beta, 0.25)
    from paper_2501_00675_b200 import api
    with api.Context() as c2:
        c2.set_g0_table(_dev(torch, Tu), beta, spin=0)
        c2.set_g0_table(_dev(torch, Td), beta, spin=1)
        Gup = torch.empty((B, n, n), dtype=torch.float64, device="cuda")
        Gdn = torch.empty((B, n, n), dtype=torch.float64, device="cuda")
        c2.build_G(_dev(torch, xy), _dev(torch, tau), Gup, Gdn, g_diag=0.25)
        torch.cuda.synchronize()
        np.testing.assert_array_equal(Gup.cpu().numpy(), ref_up)
        np.testing.assert_array_equal(Gdn.cpu().numpy(), ref_dn)


@pytest.mark.parametrize("n", [1, 2, 3, 6, 7, 9, 11, 13, 14, 15, 16])
def test_build_G_every_thread_shape(torch_mod, oracle_mod, n):
    """build_G_kernel keeps one entry (i, j) per thread and as many whole configurations per pass as fit in 256 threads
    (256, 64, 28, 7, 5, 3, 2, 1, 1, 1, 1 for these orders): every shape, with a batch that leaves a ragged last pass and
    makes the grid loop more than once, bit for bit against the oracle, both tables."""
    torch = torch_mod
    rng = np.random.default_rng(600 + n)
    L, ntau, beta = 6, 65, 2.5
    B = 148 * 8 * 8 + 8 * 3 + 5                     # more than one pass of the capped grid, then a ragged tail
    if n >= 13:
        B = 148 * 8 * 8 // 4 + 13
    Tu, Td = rng.normal(size=(L, L, ntau)), rng.normal(size=(L, L, ntau))
    xy = rng.integers(0, L, size=(B, n, 2)).astype(np.int32)
    tau = rng.uniform(0, beta, size=(B, n))
    ref_up, ref_dn = oracle_mod.build_G(xy, tau, Tu, Td, beta, 0.75)
    from paper_2501_00675_b200 import api
    with api.Context() as c2:
        c2.set_g0_table(_dev(torch, Tu), beta, spin=0)
        c2.set_g0_table(_dev(torch, Td), beta, spin=1)
        Gup = torch.full((B, n, n), float("nan"), dtype=torch.float64, device="cuda")
        Gdn = torch.full((B, n, n), float("nan"), dtype=torch.float64, device="cuda")
        c2.build_G(_dev(torch, xy), _dev(torch, tau), Gup, Gdn, g_diag=0.75)
        torch.cuda.synchronize()
        np.testing.assert_array_equal(Gup.cpu().numpy(), ref_up)
        np.testing.assert_array_equal(Gdn.cpu().numpy(), ref_dn)


@pytest.mark.parametrize("beta", [1.0 / 3.0, np.pi, 0.1, 7.0, 1e-3, 123.456, 0.125, 8.0, float(np.nextafter(2.0, 0.0)),
                                  float(np.nextafter(1.0, 2.0)), 5e-324 * 2 ** 1000, 1.7e12])
def test_build_G_division_by_beta_bit_exact(torch_mod, oracle_mod, beta):
    """u = dtau (ntau - 1) / beta is taken with the reciprocal of beta and two FMA refinements (div_by_beta in
    cos_kernels_generic.cuh); it must round like the division the oracle performs.  A quotient off by one ulp moves the
    interpolation weight and with it the last bits of G, so every entry is compared bit for bit.  The values of beta
    cover non-terminating binary fractions, powers of two, the all-ones significand (the generic division is used
    there), the successor of 1, and magnitudes far from 1; times include equal pairs, pairs one ulp apart and the
    ends of [0, beta); sites lie outside [0, L) as well (the modulo path)."""
    torch = torch_mod
    rng = np.random.default_rng(int(abs(np.log2(beta)) * 1000) % 100000)
    L, ntau, B, n = 5, 257, 777, 8
    T = rng.normal(size=(L, L, ntau))
    xy = rng.integers(-2 * L, 3 * L, size=(B, n, 2)).astype(np.int32)
    tau = rng.uniform(0, beta, size=(B, n))
    tau[0, 1] = tau[0, 2]
    tau[1, 3] = np.nextafter(tau[1, 4], 0.0)
    tau[2, 0] = 0.0
    tau[2, 5] = np.nextafter(beta, 0.0)
    tau[3, :] = tau[3, 0] + np.arange(n) * (beta * 2.0 ** -40)        # clustered times (reading R15)
    ref_up, _ = oracle_mod.build_G(xy, tau, T, None, beta, -0.5)
    from paper_2501_00675_b200 import api
    with api.Context() as c2:
        c2.set_g0_table(_dev(torch, T), beta)
        Gup = torch.empty((B, n, n), dtype=torch.float64, device="cuda")
        c2.build_G(_dev(torch, xy), _dev(torch, tau), Gup, None, g_diag=-0.5)
        torch.cuda.synchronize()
        np.testing.assert_array_equal(Gup.cpu().numpy(), ref_up)


# ------------------------------------------------------------------------------------------ a2..a5
@pytest.mark.parametrize("n", list(range(1, 17)))
def test_eval_every_order_dense(torch_mod, ctx, oracle_mod, n):
    """Every order 1..16, two distinct species with per-vertex couplings, and the aliased form."""
    rng = np.random.default_rng(1000 + n)
    B = 37 if n <= 12 else (9 if n <= 14 else 3)     # ragged, spans several CTAs
    Gup = rng.normal(size=(B, n, n)) / np.sqrt(n) + 0.5 * np.eye(n)
    Gdn = rng.normal(size=(B, n, n)) / np.sqrt(n) + 0.5 * np.eye(n)
    u = rng.uniform(0.5, 2.0, size=(B, n))
    for which in ("all", "connected"):
        got = _gpu_eval(torch_mod, ctx, Gup, Gdn, 1.0, u, which)
        check_parity(oracle_mod, got, Gup, Gdn, 1.0, u, which, label="every_order two species")
        got = _gpu_eval(torch_mod, ctx, Gup, None, 1.7, None, which)
        check_parity(oracle_mod, got, Gup, None, 1.7, None, which, label="every_order aliased")


# Batches large enough that every persistent CTA loops over at least three teams (or three grid strides of the
# generic kernel): this drives the prefetch of the next team's matrices, the re-use of the shared-memory / scratch
# areas between teams and the ragged last team, for EVERY order, one and two species.
_MANY = {1: 4741, 2: 4741, 3: 4741, 4: 4741, 5: 28417, 6: 28417, 7: 28417, 8: 14209, 9: 7105, 10: 3553,
         11: 1777, 12: 2400, 13: 1200, 14: 450, 15: 450, 16: 450}


@pytest.mark.parametrize("nsp", [1, 2])
@pytest.mark.parametrize("n", list(range(1, 17)))
def test_eval_many_teams_per_cta(torch_mod, ctx, oracle_mod, n, nsp):
    rng = np.random.default_rng(5000 + 17 * n + nsp)
    B = _MANY[n]
    Gup = rng.normal(size=(B, n, n)) / np.sqrt(n) + 0.5 * np.eye(n)
    Gdn = rng.normal(size=(B, n, n)) / np.sqrt(n) + 0.5 * np.eye(n) if nsp == 2 else None
    u = rng.uniform(0.5, 2.0, size=(B, n)) if nsp == 2 else None
    U = 1.0 if nsp == 2 else 1.7
    # the oracle checks every output up to order 12 and a seeded sample (first and last included) above
    if n <= 12:
        idx = np.arange(B)
    else:
        idx = np.sort(rng.choice(B, size=8, replace=False))
        idx[0], idx[-1] = 0, B - 1
    sub = lambda a: None if a is None else np.ascontiguousarray(a[idx])
    for which in ("connected", "all"):
        got = _gpu_eval(torch_mod, ctx, Gup, Gdn, U, u, which)
        assert np.all(np.isfinite(got))
        st = check_parity(oracle_mod, got[idx], sub(Gup), sub(Gdn), U, sub(u), which, label=f"many_teams nsp={nsp}")
        # random dense matrices: a few of several thousand draws are near-cancelling (exception rule)
        assert st["exceptions"] <= max(1, int(np.ceil(1e-3 * len(idx)))), st


@pytest.mark.parametrize("cfg,batch", [(1, 64), (2, 4096), (3, 1024), (4, 256), (5, 16)])
def test_eval_baseline_configs(torch_mod, ctx, oracle_mod, cfg, batch):
    """BASELINE.json configs (sizes the oracle finishes in seconds), element by element."""
    from harness import workloads as wl
    w = wl.baseline_config(cfg, batch=batch)
    Gup, Gdn, U, u = _workload_mats(oracle_mod, w)
    for which in ("all", "connected"):
        got = _gpu_eval(torch_mod, ctx, Gup, Gdn, U, u, which)
        st = check_parity(oracle_mod, got, Gup, Gdn, U, u, which, label=f"cfg{cfg}",
                          max_fraction=CLUSTERED_EXCEPTION_FRACTION if cfg == 4 else MAX_EXCEPTION_FRACTION)
        if cfg in (1, 5):
            assert st["exceptions"] == 0, st
    # two-propagation form of the same Hubbard input (separate copy of G_down) gives the same numbers
    if w.kind == "hubbard":
        got2 = _gpu_eval(torch_mod, ctx, Gup, Gup.copy(), U, None, "connected")
        check_parity(oracle_mod, got2, Gup, Gup.copy(), U, None, "connected", label=f"cfg{cfg} two propagations",
                     max_fraction=CLUSTERED_EXCEPTION_FRACTION if cfg == 4 else MAX_EXCEPTION_FRACTION)


def test_fused_xt_and_host_paths(torch_mod, ctx, oracle_mod):
    from harness import workloads as wl
    torch = torch_mod
    w = wl.baseline_config(3, batch=300)
    Gup, _ = oracle_mod.build_G(w.xy, w.tau, w.table, None, w.beta, 0.0)
    ctx.set_g0_table(_dev(torch, w.table), w.beta)
    out = torch.empty(w.batch, dtype=torch.float64, device="cuda")
    ctx.eval_connected_xt(_dev(torch, w.xy), _dev(torch, w.tau), out, U=w.U)
    torch.cuda.synchronize()
    assert ctx.last_launch_count() >= 1
    check_parity(oracle_mod, out.cpu().numpy(), Gup, None, w.U, None, "connected", label="xt cfg3")
    h_out = np.empty(w.batch)
    ctx.eval_connected_xt_host(w.xy, w.tau, h_out, U=w.U)
    np.testing.assert_array_equal(h_out, out.cpu().numpy())
    # the fused entry assembles exactly the matrices cos_build_G writes: same value as the two-call route
    G = torch.empty((w.batch, w.n, w.n), dtype=torch.float64, device="cuda")
    ctx.build_G(_dev(torch, w.xy), _dev(torch, w.tau), G, None, g_diag=0.0)
    out2 = torch.empty_like(out)
    ctx.eval_connected(G, G, out2, U=w.U)
    torch.cuda.synchronize()
    np.testing.assert_array_equal(out2.cpu().numpy(), out.cpu().numpy())


@pytest.mark.parametrize("n,B", [(5, 77), (8, 130), (10, 45), (12, 21)])
def test_fused_xt_two_tables(torch_mod, oracle_mod, n, B):
    """Fused entry with distinct spin-up / spin-down tables (two propagation instances per configuration),
    per-vertex couplings and a non-zero equal-time diagonal; ragged batch sizes."""
    torch = torch_mod
    from paper_2501_00675_b200 import api
    rng = np.random.default_rng(77 + n)
    L, ntau, beta = 6, 41, 2.9
    Tu = rng.normal(size=(L, L, ntau)) * 0.6
    Td = rng.normal(size=(L, L, ntau)) * 0.6
    xy = rng.integers(0, L, size=(B, n, 2)).astype(np.int32)
    tau = rng.uniform(0, beta, size=(B, n))
    u = rng.uniform(0.5, 1.5, size=(B, n))
    Gup, Gdn = oracle_mod.build_G(xy, tau, Tu, Td, beta, 0.3)
    with api.Context() as c2:
        c2.set_g0_table(_dev(torch, Tu), beta, spin=0)
        c2.set_g0_table(_dev(torch, Td), beta, spin=1)
        out = torch.empty(B, dtype=torch.float64, device="cuda")
        c2.eval_connected_xt(_dev(torch, xy), _dev(torch, tau), out, U=1.0, d_u=_dev(torch, u), g_diag=0.3)
        torch.cuda.synchronize()
        check_parity(oracle_mod, out.cpu().numpy(), Gup, Gdn, 1.0, u, "connected", label="xt two tables")


def test_degenerate_inputs(torch_mod, ctx, oracle_mod):
    torch = torch_mod
    # empty batch: legal, no work
    e = torch.empty((0, 6, 6), dtype=torch.float64, device="cuda")
    o = torch.empty(0, dtype=torch.float64, device="cuda")
    ctx.eval_connected(e, e, o, U=1.0)
    # zero matrix, identity, singular (rank-1) and block-diagonal (disconnected => 0) inputs
    n = 8
    Z = np.zeros((1, n, n))
    I = np.eye(n)[None]
    x = np.linspace(0.5, 1.5, n)
    R1 = np.outer(x, x[::-1])[None]
    blk = np.zeros((1, n, n)); blk[0, :3, :3] = 0.3 + np.eye(3); blk[0, 3:, 3:] = 0.2 + np.eye(5)
    G = np.concatenate([Z, I, R1, blk])
    ref_all, ref_conn = oracle_mod.eval_all_connected(G, None, U=2.0)
    got_all = _gpu_eval(torch, ctx, G, None, 2.0, None, "all")
    got_conn = _gpu_eval(torch, ctx, G, None, 2.0, None, "connected")
    np.testing.assert_allclose(got_all, ref_all, rtol=1e-10, atol=1e-12 * np.abs(ref_all).max())
    np.testing.assert_allclose(got_conn, ref_conn, rtol=1e-10, atol=1e-12 * np.abs(ref_all).max())
    assert got_all[0] == 0.0 and got_conn[0] == 0.0                  # zero matrix
    assert got_conn[1] == 0.0                                        # identity: only sigma = id, disconnected
    assert abs(got_conn[3]) <= 1e-12 * abs(got_all[3])               # two blocks: no connected diagram
    # bad arguments fail loudly
    from paper_2501_00675_b200 import api
    with pytest.raises(api.CosError):
        big = torch.empty((1, 17, 17), dtype=torch.float64, device="cuda")
        ctx.eval_connected(big, big, torch.empty(1, dtype=torch.float64, device="cuda"))
    with api.Context() as fresh:
        with pytest.raises(api.CosError):
            fresh.build_G(torch.zeros((1, 2, 2), dtype=torch.int32, device="cuda"),
                          torch.zeros((1, 2), dtype=torch.float64, device="cuda"),
                          torch.empty((1, 2, 2), dtype=torch.float64, device="cuda"))


def test_probes_report_plausible_peaks(ctx):
    tf = ctx.probe_dfma_tflops()
    bw = ctx.probe_smem_gbs()
    print(f"DFMA probe {tf:.2f} TFLOP/s, shared-memory probe {bw:.0f} GB/s")
    assert 10.0 < tf < 80.0
    assert 5e3 < bw < 1e5


# ------------------------------------------------------------------------------------------ full sizes
@pytest.mark.parametrize("cfg,nsample", [(2, 512), (3, 512), (4, 128), (5, 8)])
def test_full_size_sampled_outputs(torch_mod, oracle_mod, cfg, nsample):
    """BASELINE.json configs at their FULL batch, through the entry point and launch configuration bench.py
    times (cos_eval_connected_xt for the Hubbard configs: build_G + evaluation over the whole batch;
    cos_eval_connected for config 5), checked on a seeded sample of outputs the oracle computes one by one."""
    from paper_2501_00675_b200 import api
    from harness import workloads as wl
    torch = torch_mod
    w = wl.baseline_config(cfg)                       # full batch: 4096 / 16384 / 4096 / 512
    out = torch.empty(w.batch, dtype=torch.float64, device="cuda")
    with api.Context() as c:
        if w.kind == "hubbard":
            c.set_g0_table(_dev(torch, w.table), w.beta)
            c.eval_connected_xt(_dev(torch, w.xy), _dev(torch, w.tau), out, U=w.U, g_diag=w.g_diag)
        else:
            dG = _dev(torch, w.G)
            c.eval_connected(dG, dG, out, U=w.U, d_u=_dev(torch, w.u))
        torch.cuda.synchronize()
        assert c.last_launch_count() >= 1
    got = out.cpu().numpy()
    assert np.all(np.isfinite(got))
    idx = np.sort(np.random.default_rng(77 + cfg).choice(w.batch, size=min(nsample, w.batch), replace=False))
    idx[0], idx[-1] = 0, w.batch - 1                  # first and last configuration of the batch (ragged last team)
    if w.kind == "hubbard":
        Gup, _ = oracle_mod.build_G(w.xy[idx], w.tau[idx], w.table, None, w.beta, w.g_diag)
        check_parity(oracle_mod, got[idx], Gup, None, w.U, None, "connected", label=f"full size cfg{cfg}",
                     max_fraction=CLUSTERED_EXCEPTION_FRACTION if cfg == 4 else MAX_EXCEPTION_FRACTION)
    else:
        check_parity(oracle_mod, got[idx], np.ascontiguousarray(w.G[idx]), None, w.U,
                     np.ascontiguousarray(w.u[idx]), "connected", label=f"full size cfg{cfg}")


@pytest.mark.parametrize("n", [5, 8, 10, 11, 12, 13, 14])
def test_generic_kernel_cross_check(torch_mod, oracle_mod, n):
    """cos_debug_force_generic: the plain one-thread-per-node kernel at orders the tuned kernels normally serve,
    against the oracle (so the switch itself is verified) and against the tuned kernel."""
    from paper_2501_00675_b200 import api
    rng = np.random.default_rng(900 + n)
    B = 301 if n <= 10 else (37 if n <= 12 else 5)      # more configurations than persistent CTAs at n <= 10
    Gup = rng.normal(size=(B, n, n)) / np.sqrt(n) + 0.5 * np.eye(n)
    Gdn = rng.normal(size=(B, n, n)) / np.sqrt(n) + 0.5 * np.eye(n)
    u = rng.uniform(0.5, 2.0, size=(B, n))
    with api.Context() as c:
        tuned = _gpu_eval(torch_mod, c, Gup, Gdn, 1.0, u, "connected")
        assert c.last_kernel_name() != "eval_generic_kernel"
        c.force_generic(True)
        for which in ("all", "connected"):
            got = _gpu_eval(torch_mod, c, Gup, Gdn, 1.0, u, which)
            assert c.last_kernel_name() == "eval_generic_kernel"
            check_parity(oracle_mod, got, Gup, Gdn, 1.0, u, which, label="forced generic kernel")
        np.testing.assert_allclose(got, tuned, rtol=1e-9)
        got1 = _gpu_eval(torch_mod, c, Gup, None, 1.3, None, "connected")
        check_parity(oracle_mod, got1, Gup, None, 1.3, None, "connected", label="forced generic kernel aliased")


# ------------------------------------------------------------------------------------------ f3: loop weight
@pytest.mark.parametrize("n", [2, 4, 6, 9, 10, 11, 12, 13, 14])
def test_loop_weight(torch_mod, oracle_mod, n):
    """cos_set_loop_weight: -N_f per closed fermion loop (reading R17) through every kernel family, one and two
    species, against the oracle's loop-weight mode; N_f = 1 restores the default."""
    from paper_2501_00675_b200 import api
    rng = np.random.default_rng(4000 + n)
    B = 45 if n <= 12 else 5
    Gup = rng.normal(size=(B, n, n)) / np.sqrt(n) + 0.5 * np.eye(n)
    Gdn = rng.normal(size=(B, n, n)) / np.sqrt(n) + 0.5 * np.eye(n)
    u = rng.uniform(0.5, 2.0, size=(B, n))
    with api.Context() as c:
        for nf in (2.0, -1.0, 0.5):
            c.set_loop_weight(nf)
            for which in ("all", "connected"):
                got = _gpu_eval(torch_mod, c, Gup, Gdn, 1.0, u, which)
                check_parity(oracle_mod, got, Gup, Gdn, 1.0, u, which, loop_weight=nf, label=f"loop weight {nf}")
            got = _gpu_eval(torch_mod, c, Gup, None, 1.3, None, "connected")
            check_parity(oracle_mod, got, Gup, None, 1.3, None, "connected", loop_weight=nf,
                         label=f"loop weight {nf} aliased")
        c.set_loop_weight(1.0)
        got = _gpu_eval(torch_mod, c, Gup, Gdn, 1.0, u, "connected")
        check_parity(oracle_mod, got, Gup, Gdn, 1.0, u, "connected", label="loop weight reset")


@pytest.mark.parametrize("nl", [1, 2, 3, 4, 5, 6, 7])
def test_halfvertex(torch_mod, oracle_mod, nl):
    """cos_eval_halfvertex (reading R18) against the oracle's half-vertex mode, N_f = 1 and 2."""
    from paper_2501_00675_b200 import api
    torch = torch_mod
    m = 2 * nl
    rng = np.random.default_rng(6000 + nl)
    B = 333 if nl <= 5 else 19                        # more configurations than persistent CTAs at small sizes
    W = rng.normal(size=(B, m, m)) / np.sqrt(m) + 0.5 * np.eye(m)
    V = rng.uniform(0.5, 2.0, size=(B, nl))
    with api.Context() as c:
        for nf in (1.0, 2.0):
            c.set_loop_weight(nf)
            ref_all, ref_conn = oracle_mod.eval_halfvertex(W, V, loop_weight=nf)
            for connected, ref in ((False, ref_all), (True, ref_conn)):
                out = torch.empty(B, dtype=torch.float64, device="cuda")
                c.eval_halfvertex(_dev(torch, W), _dev(torch, V), out, connected=connected)
                torch.cuda.synchronize()
                assert c.last_kernel_name() == "eval_generic_kernel" and c.last_launch_count() >= 1
                got = out.cpu().numpy()
                bad = np.abs(got - ref) > 1e-10 * np.abs(ref)
                assert bad.sum() <= max(1, int(np.ceil(2e-3 * B))), (nl, nf, connected, np.abs(got / ref - 1).max())
                assert np.all(np.abs(got - ref) <= 1e-7 * np.abs(ref))


# ------------------------------------------------------------------------------------------ races / stale state
@pytest.mark.parametrize("n,nsp", [(3, 1), (6, 2), (8, 1), (9, 2), (10, 1), (10, 2), (11, 1), (12, 2), (13, 1), (13, 2),
                                   (14, 1), (15, 1)])
def test_result_independent_of_batch_position_and_repeatable(torch_mod, ctx, n, nsp):
    """compute-sanitizer is closed on this GPU pool, so data races and stale shared-memory / scratch state are hunted
    with properties they would break: (1) the value of a configuration does not depend on where it sits in the batch
    (other team mates, another lane group, another W replica, another persistent CTA, first or last team of the
    loop) -- bit for bit; (2) repeated launches give identical bits.  Batches give every persistent CTA several teams."""
    torch = torch_mod
    rng = np.random.default_rng(8000 + 10 * n + nsp)
    B = _MANY[n] // (2 if n >= 13 else 1)
    # orders 12..16: whole rounds of the persistent grid (148 CTAs x team size), so that every configuration is evaluated
    # with the same team size wherever it sits (a partial last round is launched with smaller teams: pair_tail_split)
    B = {(12, 1): 2368, (12, 2): 1184, (13, 1): 592, (13, 2): 592, (15, 1): 296}.get((n, nsp), B)
    Gup = rng.normal(size=(B, n, n)) / np.sqrt(n) + 0.5 * np.eye(n)
    Gdn = rng.normal(size=(B, n, n)) / np.sqrt(n) + 0.5 * np.eye(n) if nsp == 2 else None
    u = rng.uniform(0.5, 2.0, size=(B, n))
    perm = rng.permutation(B)
    a = _gpu_eval(torch, ctx, Gup, Gdn, 1.0, u, "connected")
    b = _gpu_eval(torch, ctx, Gup[perm], None if Gdn is None else Gdn[perm], 1.0, u[perm], "connected")
    np.testing.assert_array_equal(a[perm], b)
    for _ in range(3):
        np.testing.assert_array_equal(_gpu_eval(torch, ctx, Gup, Gdn, 1.0, u, "connected"), a)
    # a ragged sub-batch (different team boundaries, fewer CTAs) reproduces the same bits for the configurations it holds
    k = max(1, B // 3 + 1)
    c = _gpu_eval(torch, ctx, Gup[:k], None if Gdn is None else Gdn[:k], 1.0, u[:k], "connected")
    if n <= 10:
        np.testing.assert_array_equal(c, a[:k])
    else:       # from order 11 the team size follows the batch (cos_dispatch.cuh: pair_plan), and with it the order in
        np.testing.assert_allclose(c, a[:k], rtol=1e-10)      # which the reduction sums its partial blocks


@pytest.mark.parametrize("n,nsp", [(11, 1), (11, 2), (13, 1), (13, 2), (14, 1), (16, 1), (16, 2)])
def test_sweep_shapes_sampled_outputs(torch_mod, ctx, oracle_mod, n, nsp):
    """The team plans of orders 11..16 (cos_dispatch.cuh: pair_plan) at the batch sizes of the bench sweep -- two CTAs of
    256 threads at n = 11, teams of 4 at n = 13, one instance with its reduction arrays in shared memory at n = 14,
    teams of 2 / 4 at n = 16 -- checked against the oracle on a seeded sample that includes the first and the last
    configuration."""
    from harness import workloads as wl
    B = wl.sweep_batch(n)
    rng = np.random.default_rng(9000 + 10 * n + nsp)
    Gup = rng.normal(size=(B, n, n)) / np.sqrt(n) + 0.5 * np.eye(n)
    Gdn = rng.normal(size=(B, n, n)) / np.sqrt(n) + 0.5 * np.eye(n) if nsp == 2 else None
    u = rng.uniform(0.5, 2.0, size=(B, n))
    got = _gpu_eval(torch_mod, ctx, Gup, Gdn, 1.0, u, "connected")
    assert np.all(np.isfinite(got))
    idx = np.sort(rng.choice(B, size=64 if n <= 13 else 8, replace=False))
    idx[0], idx[-1] = 0, B - 1
    sub = lambda a: None if a is None else np.ascontiguousarray(a[idx])
    st = check_parity(oracle_mod, got[idx], sub(Gup), sub(Gdn), 1.0, sub(u), "connected", label=f"sweep shape nsp={nsp}")
    assert st["exceptions"] == 0, st
