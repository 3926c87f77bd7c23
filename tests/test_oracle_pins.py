"""Pins for the CPU oracle (oracle/cos_oracle.c): every check here compares the oracle with something
OTHER than itself -- the plain definition enumerated in pure Python, numpy.linalg determinants,
closed forms, invariances and integer combinatorics -- chosen so that a dropped term, a wrong sign,
a wrong index or a transposed operand anywhere in propagate / combine / reduce_connected fails one.
Runs without a GPU.  Citations: SURVEY.md §8(c) "What pins each part"; DESIGN.md §3.
"""
import itertools
import math
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rand(rng, n):
    return rng.normal(size=(n, n)), rng.normal(size=(n, n)), rng.uniform(0.5, 2.0, size=n)


# ------------------------------------------------------------------ plain definition in pure Python
def _cycles(p):
    seen, c = [False] * len(p), 0
    for i in range(len(p)):
        if not seen[i]:
            c += 1
            j = i
            while not seen[j]:
                seen[j] = True
                j = p[j]
    return c


def _connected(n, pa, pb):
    adj = [set() for _ in range(n)]
    for i in range(n):
        for j in (pa[i], pb[i]):
            adj[i].add(j)
            adj[j].add(i)
    stack, seen = [0], {0}
    while stack:
        v = stack.pop()
        for w in adj[v]:
            if w not in seen:
                seen.add(w)
                stack.append(w)
    return len(seen) == n


def python_bruteforce(Gup, Gdn, u):
    """sum over all (sigma_up, sigma_dn), depth-first-search connectivity (not union-find)."""
    n = Gup.shape[0]
    w = math.prod(-x for x in u)
    tot = conn = 0.0
    cnt = 0
    perms = list(itertools.permutations(range(n)))
    tu = [(-1) ** _cycles(p) * math.prod(Gup[i, p[i]] for i in range(n)) for p in perms]
    td = [(-1) ** _cycles(p) * math.prod(Gdn[i, p[i]] for i in range(n)) for p in perms]
    for a, pa in enumerate(perms):
        for b, pb in enumerate(perms):
            t = tu[a] * td[b]
            tot += t
            if _connected(n, pa, pb):
                conn += t
                cnt += 1
    return w * tot, w * conn, cnt


@pytest.mark.parametrize("n", [1, 2, 3, 4])
def test_oracle_vs_pure_python_enumeration(oracle_mod, n):
    rng = np.random.default_rng(10 + n)
    for _ in range(3):
        Gup, Gdn, u = _rand(rng, n)
        a_ref, c_ref, _ = python_bruteforce(Gup, Gdn, u)
        a, c = oracle_mod.eval_all_connected(Gup[None], Gdn[None], u=u[None])
        assert a[0] == pytest.approx(a_ref, rel=1e-12, abs=1e-13)
        assert c[0] == pytest.approx(c_ref, rel=1e-12, abs=1e-13)


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6])
def test_oracle_vs_c_bruteforce_and_pair_counts(oracle_mod, n):
    gold = dict(tuple(map(int, l.split())) for l in open(os.path.join(GOLD, "connected_pair_counts.txt"))
                if not l.startswith("#"))
    rng = np.random.default_rng(20 + n)
    for _ in range(2):
        Gup, Gdn, u = _rand(rng, n)
        a_ref, c_ref, cnt = oracle_mod.bruteforce(Gup, Gdn, u)
        assert cnt == gold[n]
        a, c = oracle_mod.eval_all_connected(Gup[None], Gdn[None], u=u[None])
        scale = abs(a_ref) + abs(c_ref)
        assert abs(a[0] - a_ref) <= 1e-11 * scale
        assert abs(c[0] - c_ref) <= 1e-11 * scale


def test_c_bruteforce_agrees_with_python_bruteforce(oracle_mod):
    rng = np.random.default_rng(5)
    for n in (2, 3, 4):
        Gup, Gdn, u = _rand(rng, n)
        a1, c1, k1 = python_bruteforce(Gup, Gdn, u)
        a2, c2, k2 = oracle_mod.bruteforce(Gup, Gdn, u)
        assert k1 == k2
        assert a2 == pytest.approx(a1, rel=1e-12)
        assert c2 == pytest.approx(c1, rel=1e-12)


# ------------------------------------------------------------------ determinant invariant
@pytest.mark.parametrize("n", [1, 2, 3, 5, 8, 10, 12])
def test_all_equals_det_product(oracle_mod, n):
    """all = prod_a(-u_a) det Gup det Gdn  (north_star: "the all-diagrams sum equals det Gup det Gdn
    times the order's U and sign factors"; (-1)^cyc = (-1)^n sgn, the two (-1)^n cancel)."""
    rng = np.random.default_rng(30 + n)
    B = 4
    Gup = rng.normal(size=(B, n, n))
    Gdn = rng.normal(size=(B, n, n))
    u = rng.uniform(0.5, 2.0, size=(B, n))
    a, _ = oracle_mod.eval_all_connected(Gup, Gdn, u=u)
    ref = np.prod(-u, axis=1) * np.linalg.det(Gup) * np.linalg.det(Gdn)
    np.testing.assert_allclose(a, ref, rtol=1e-10)
    # Hubbard form: scalar U
    a2, _ = oracle_mod.eval_all_connected(Gup, Gdn, U=1.7)
    np.testing.assert_allclose(a2, (-1.7) ** n * np.linalg.det(Gup) * np.linalg.det(Gdn), rtol=1e-10)


@pytest.mark.parametrize("n", [3, 6, 9, 10])
def test_every_minor_matches_lu(oracle_mod, n):
    """Z[S] = (-1)^{|S|} det W[S,S] for EVERY subset S, from numpy's LU.  Absolute error scaled by the
    product of row norms (odd minors vanish by particle-hole symmetry at mu=0, so not relative)."""
    rng = np.random.default_rng(40 + n)
    W = rng.normal(size=(n, n))
    Z = oracle_mod.minors(W)
    assert Z[0] == 1.0
    rown = np.linalg.norm(W, axis=1)
    for S in range(1, 1 << n):
        idx = [v for v in range(n) if S >> v & 1]
        ref = (-1) ** len(idx) * np.linalg.det(W[np.ix_(idx, idx)])
        assert abs(Z[S] - ref) <= 1e-12 * np.prod(rown[idx]) * math.factorial(min(len(idx), 6))


def test_minors_not_transposed(oracle_mod):
    """A strictly upper-triangular perturbation distinguishes W from W^T only in products along
    cycles; check a 3-cycle weight directly: Z[{0,1,2}] contains -(W01 W12 W20 + W02 W21 W10)."""
    W = np.zeros((3, 3))
    W[0, 1], W[1, 2], W[2, 0] = 2.0, 3.0, 5.0          # one directed 3-cycle 0->1->2->0, weight 30
    Z = oracle_mod.minors(W)
    assert Z[7] == pytest.approx(-30.0)
    assert Z[3] == 0.0 and Z[5] == 0.0 and Z[6] == 0.0


# ------------------------------------------------------------------ closed forms
def test_closed_form_n1(oracle_mod):
    a, c = oracle_mod.eval_all_connected(np.array([[[0.3]]]), np.array([[[-0.7]]]), U=2.0)
    assert a[0] == pytest.approx(-2.0 * 0.3 * -0.7)
    assert c[0] == pytest.approx(-2.0 * 0.3 * -0.7)


def test_closed_form_n2(oracle_mod):
    """n=2: connected = U^2 [b_up b_dn - a_up b_dn - b_up a_dn], a = G00 G11, b = G01 G10."""
    rng = np.random.default_rng(7)
    Gup, Gdn = rng.normal(size=(2, 2)), rng.normal(size=(2, 2))
    U = 1.3
    au, bu = Gup[0, 0] * Gup[1, 1], Gup[0, 1] * Gup[1, 0]
    ad, bd = Gdn[0, 0] * Gdn[1, 1], Gdn[0, 1] * Gdn[1, 0]
    a, c = oracle_mod.eval_all_connected(Gup[None], Gdn[None], U=U)
    assert c[0] == pytest.approx(U * U * (bu * bd - au * bd - bu * ad), rel=1e-13)
    assert a[0] == pytest.approx(U * U * (au - bu) * (ad - bd), rel=1e-13)


@pytest.mark.parametrize("n", [3, 5, 7, 9])
def test_rank_one_up_species(oracle_mod, n):
    """Gup = x y^T (rank 1), Gdn arbitrary: connected = (-1)^{n-1} (n-1)! prod_i D({i})."""
    rng = np.random.default_rng(50 + n)
    x, y = rng.normal(size=n), rng.normal(size=n)
    Gup = np.outer(x, y)
    Gdn = rng.normal(size=(n, n))
    u = rng.uniform(0.5, 2.0, size=n)
    _, c = oracle_mod.eval_all_connected(Gup[None], Gdn[None], u=u[None])
    D1 = -u * np.diag(Gup) * np.diag(Gdn)              # D({i}) = (-u_i)(-Gup_ii)(-Gdn_ii)
    ref = (-1) ** (n - 1) * math.factorial(n - 1) * np.prod(D1)
    # rank-1 minors of size >= 2 vanish, so only sigma_up with ... see DESIGN.md §3; check value
    assert c[0] == pytest.approx(ref, rel=1e-9)


@pytest.mark.parametrize("n", [3, 4, 5, 6])
def test_identity_down_species(oracle_mod, n):
    """Gdn = I: sigma_dn must be the identity (n loops), so connectivity rests on sigma_up alone:
    connected = (-U)^n (-1)^n * (-1) * sum over the (n-1)! cyclic orders of prod Gup."""
    rng = np.random.default_rng(60 + n)
    Gup = rng.normal(size=(n, n))
    U = 0.9
    _, c = oracle_mod.eval_all_connected(Gup[None], np.eye(n)[None], U=U)
    s = 0.0
    for rest in itertools.permutations(range(1, n)):
        cyc = (0,) + rest
        s += math.prod(Gup[cyc[i], cyc[(i + 1) % n]] for i in range(n))
    ref = (-U) ** n * (-1) ** n * (-1) * s
    assert c[0] == pytest.approx(ref, rel=1e-11)


def test_block_diagonal_is_disconnected(oracle_mod):
    rng = np.random.default_rng(8)
    for n, k in ((4, 2), (6, 2), (7, 3)):
        def blk():
            G = np.zeros((n, n))
            G[:k, :k] = rng.normal(size=(k, k))
            G[k:, k:] = rng.normal(size=(n - k, n - k))
            return G
        Gup, Gdn = blk(), blk()
        a, c = oracle_mod.eval_all_connected(Gup[None], Gdn[None], U=1.1)
        assert abs(c[0]) <= 1e-12 * abs(a[0])
        # and with the blocks interleaved by a relabelling (exercises the max-head asymmetry)
        p = rng.permutation(n)
        a2, c2 = oracle_mod.eval_all_connected(Gup[np.ix_(p, p)][None], Gdn[np.ix_(p, p)][None], U=1.1)
        assert abs(c2[0]) <= 1e-12 * abs(a2[0])


# ------------------------------------------------------------------ invariances
@pytest.mark.parametrize("n", [4, 7, 9])
def test_invariances(oracle_mod, n):
    rng = np.random.default_rng(70 + n)
    Gup, Gdn, u = _rand(rng, n)
    _, c0 = oracle_mod.eval_all_connected(Gup[None], Gdn[None], u=u[None])
    c0 = c0[0]
    # simultaneous relabelling of the vertices
    for _ in range(3):
        p = rng.permutation(n)
        _, c = oracle_mod.eval_all_connected(Gup[np.ix_(p, p)][None], Gdn[np.ix_(p, p)][None], u=u[p][None])
        assert c[0] == pytest.approx(c0, rel=1e-9)
    # transpose both species
    _, c = oracle_mod.eval_all_connected(Gup.T.copy()[None], Gdn.T.copy()[None], u=u[None])
    assert c[0] == pytest.approx(c0, rel=1e-9)
    # transposing ONE species is also a symmetry: sigma -> sigma^-1 keeps the cycle count and the
    # undirected edges {i, sigma(i)}, hence the connectivity
    _, c = oracle_mod.eval_all_connected(Gup.T.copy()[None], Gdn[None], u=u[None])
    assert c[0] == pytest.approx(c0, rel=1e-9)
    # diagonal similarity G -> L G L^-1
    lam = rng.uniform(0.5, 2.0, size=n)
    _, c = oracle_mod.eval_all_connected((lam[:, None] * Gup / lam[None, :])[None], Gdn[None], u=u[None])
    assert c[0] == pytest.approx(c0, rel=1e-9)
    # Gup -> s Gup scales by s^n ; u -> s u scales by s^n ; swapping the species is a symmetry
    _, c = oracle_mod.eval_all_connected((1.5 * Gup)[None], Gdn[None], u=u[None])
    assert c[0] == pytest.approx(1.5 ** n * c0, rel=1e-9)
    _, c = oracle_mod.eval_all_connected(Gup[None], Gdn[None], u=(0.5 * u)[None])
    assert c[0] == pytest.approx(0.5 ** n * c0, rel=1e-9)
    _, c = oracle_mod.eval_all_connected(Gdn[None], Gup[None], u=u[None])
    assert c[0] == pytest.approx(c0, rel=1e-9)
    # overall sign of G is immaterial when applied to both species? No: (-G)^(n) per species -> (+1) overall
    _, c = oracle_mod.eval_all_connected((-Gup)[None], (-Gdn)[None], u=u[None])
    assert c[0] == pytest.approx(c0, rel=1e-9)


# ------------------------------------------------------------------ exp/log consistency
def _set_partitions(elems):
    if not elems:
        yield []
        return
    first, rest = elems[0], elems[1:]
    for k in range(len(rest) + 1):
        for others in itertools.combinations(rest, k):
            block = [first] + list(others)
            remaining = [e for e in rest if e not in others]
            for p in _set_partitions(remaining):
                yield [block] + p


@pytest.mark.parametrize("n", [3, 4, 5, 6])
def test_exp_log_consistency(oracle_mod, n):
    """sum over set partitions of prod_blocks connected(block) = all(full): the connected values of
    every sub-configuration, computed by separate oracle calls, must re-exponentiate to D[full]."""
    rng = np.random.default_rng(80 + n)
    Gup, Gdn, u = _rand(rng, n)
    conn = {}
    for S in range(1, 1 << n):
        idx = [v for v in range(n) if S >> v & 1]
        _, c = oracle_mod.eval_all_connected(Gup[np.ix_(idx, idx)][None], Gdn[np.ix_(idx, idx)][None],
                                             u=u[idx][None])
        conn[tuple(idx)] = c[0]
    total = sum(math.prod(conn[tuple(b)] for b in part) for part in _set_partitions(list(range(n))))
    a, _ = oracle_mod.eval_all_connected(Gup[None], Gdn[None], u=u[None])
    assert total == pytest.approx(a[0], rel=1e-9)
    # and the D/C tables are consistent with the per-subset calls
    D, C = oracle_mod.DC(Gup, Gdn, u)
    for S in range(1, 1 << n, 2):
        idx = tuple(v for v in range(n) if S >> v & 1)
        assert C[S] == pytest.approx(conn[idx], rel=1e-9, abs=1e-12)


# ------------------------------------------------------------------ independent fast route
@pytest.mark.parametrize("n", [6, 8, 10, 12])
def test_independent_lu_minor_route(oracle_mod, n):
    """D(S) from numpy LU determinants of principal submatrices (no CoS code), then the subset
    recursion written separately here in the 'sum over the complement' form."""
    rng = np.random.default_rng(90 + n)
    Gup, Gdn, u = _rand(rng, n)
    N = 1 << n
    D = np.ones(N)
    for S in range(1, N):
        idx = [v for v in range(n) if S >> v & 1]
        D[S] = np.prod(-u[idx]) * np.linalg.det(Gup[np.ix_(idx, idx)]) * np.linalg.det(Gdn[np.ix_(idx, idx)])
    C = np.zeros(N)
    for S in sorted(range(1, N, 2), key=lambda s: bin(s).count("1")):
        acc = D[S]
        rest = S & ~1
        R = rest                                   # R = S \ T runs over the non-empty subsets of rest
        while R:
            acc -= C[S & ~R] * D[R]
            R = (R - 1) & rest
        C[S] = acc
    a, c = oracle_mod.eval_all_connected(Gup[None], Gdn[None], u=u[None])
    assert a[0] == pytest.approx(D[N - 1], rel=1e-10)
    assert c[0] == pytest.approx(C[N - 1], rel=1e-8)


def test_aliased_species_and_batching(oracle_mod):
    """Gdn omitted == Gdn equal to Gup; batch entries are independent."""
    rng = np.random.default_rng(3)
    G = rng.normal(size=(5, 6, 6))
    a1, c1 = oracle_mod.eval_all_connected(G, None, U=2.0)
    a2, c2 = oracle_mod.eval_all_connected(G, G.copy(), U=2.0)
    np.testing.assert_array_equal(a1, a2)
    np.testing.assert_array_equal(c1, c2)
    for b in range(5):
        a, c = oracle_mod.eval_all_connected(G[b:b + 1], None, U=2.0, threads=1)
        assert a[0] == a1[b] and c[0] == c1[b]


def test_long_double_mode_close_to_double(oracle_mod):
    rng = np.random.default_rng(4)
    G = rng.normal(size=(3, 8, 8)) / np.sqrt(8) + 0.5 * np.eye(8)
    a, c = oracle_mod.eval_all_connected(G, None, U=4.0)
    a80, c80 = oracle_mod.eval_all_connected_f80(G, None, U=4.0)
    np.testing.assert_allclose(a, a80, rtol=1e-12)
    np.testing.assert_allclose(c, c80, rtol=1e-10)
    kappa = np.array([oracle_mod.abs_sum(G[b], G[b], np.full(8, 4.0)) for b in range(3)]) / np.abs(c80)
    assert np.all(kappa >= 1.0)
    assert np.all(np.abs(c - c80) <= 64 * kappa * np.finfo(float).eps * np.abs(c80))
