"""Pins of the oracle's extensions (no GPU): the loop-weight generalisation (reading R17),
the half-vertex formulation (reading R18), and the conditioning sums oracle_abs_sum(s).

Each pin is something other than the oracle's own recursion: plain enumeration written here in Python, the
permanent by Ryser's textbook formula, integer counts from tests/golden, closed forms, and the reduction of the
half-vertex sum to the two-species sum when the two half-vertex classes do not mix."""
import itertools
import os

import numpy as np
import pytest

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


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


def _ryser_permanent(M):
    """perm(M) = (-1)^n sum_{S subset of columns} (-1)^{|S|} prod_i sum_{j in S} M[i][j]  (Ryser 1963)."""
    n = M.shape[0]
    if n == 0:
        return 1.0
    tot = 0.0
    for S in range(1, 1 << n):
        cols = [j for j in range(n) if S >> j & 1]
        tot += (-1) ** len(cols) * np.prod(M[:, cols].sum(axis=1))
    return (-1) ** n * tot


# ------------------------------------------------------------------------------------------ loop weight (R17)
@pytest.mark.parametrize("n", [1, 2, 3, 4, 5])
@pytest.mark.parametrize("nf", [2.0, 3.0, 0.5, -1.0])
def test_loop_weight_matches_plain_enumeration(oracle_mod, n, nf):
    """Every pair of permutations, (-N_f)^(closed loops), connectivity by a DFS written here."""
    rng = np.random.default_rng(10 * n + int(4 * nf) + 50)
    Gup, Gdn, u = rng.normal(size=(n, n)), rng.normal(size=(n, n)), rng.uniform(0.5, 2.0, size=n)
    perms = list(itertools.permutations(range(n)))
    all_sum = conn_sum = 0.0
    for pu in perms:
        tu = (-nf) ** _cycles(pu) * np.prod([Gup[i, pu[i]] for i in range(n)])
        for pd in perms:
            term = tu * (-nf) ** _cycles(pd) * np.prod([Gdn[i, pd[i]] for i in range(n)])
            all_sum += term
            adj = {i: {pu[i], pd[i]} for i in range(n)}
            for i in range(n):
                adj[pu[i]].add(i)
                adj[pd[i]].add(i)
            seen, stack = {0}, [0]
            while stack:
                for w in adj[stack.pop()]:
                    if w not in seen:
                        seen.add(w)
                        stack.append(w)
            if len(seen) == n:
                conn_sum += term
    w = np.prod(-u)
    a, c = oracle_mod.eval_all_connected_lw(Gup[None], Gdn[None], u=u[None], loop_weight=nf)
    assert a[0] == pytest.approx(w * all_sum, rel=1e-10, abs=1e-12)
    assert c[0] == pytest.approx(w * conn_sum, rel=1e-9, abs=1e-12)
    ab, cb, _ = oracle_mod.bruteforce_lw(Gup, Gdn, u, nf)          # the C enumerator agrees with the Python one
    assert ab == pytest.approx(w * all_sum, rel=1e-10, abs=1e-12)
    assert cb == pytest.approx(w * conn_sum, rel=1e-10, abs=1e-12)


@pytest.mark.parametrize("n", [1, 2, 4, 6, 8])
def test_loop_weight_minus_one_gives_permanents(oracle_mod, n):
    """N_f = -1 drops every sign: Z[S] = perm(W[S,S]) for every S (Ryser's formula, independent of the graph)."""
    rng = np.random.default_rng(n)
    W = rng.normal(size=(n, n))
    Z = oracle_mod.minors_lw(W, -1.0)
    for S in range(1 << n):
        idx = [v for v in range(n) if S >> v & 1]
        assert Z[S] == pytest.approx(_ryser_permanent(W[np.ix_(idx, idx)]), rel=1e-9, abs=1e-10)


def test_loop_weight_one_is_the_papers_sign(oracle_mod):
    rng = np.random.default_rng(5)
    G = rng.normal(size=(4, 7, 7))
    a0, c0 = oracle_mod.eval_all_connected(G, None, U=1.3)
    a1, c1 = oracle_mod.eval_all_connected_lw(G, None, U=1.3, loop_weight=1.0)
    np.testing.assert_array_equal(a0, a1)
    np.testing.assert_array_equal(c0, c1)


def test_loop_weight_closed_forms(oracle_mod):
    """n = 1: -U (N_f g_up)(N_f g_dn).  n = 2: Z = N_f^2 W00 W11 - N_f W01 W10 per species;
    connected = U^2 [Zu Zd - (N_f^2 a_up)(N_f^2 a_dn)], a = W00 W11 (the disconnected part is the two tadpole pairs)."""
    rng = np.random.default_rng(6)
    nf, U = 2.5, 1.7
    Gu, Gd = rng.normal(size=(2, 2)), rng.normal(size=(2, 2))
    a, c = oracle_mod.eval_all_connected_lw(Gu[None, :1, :1], Gd[None, :1, :1], U=U, loop_weight=nf)
    assert a[0] == pytest.approx(-U * nf * Gu[0, 0] * nf * Gd[0, 0], rel=1e-14)
    assert c[0] == pytest.approx(a[0], rel=1e-14)
    zu = nf ** 2 * Gu[0, 0] * Gu[1, 1] - nf * Gu[0, 1] * Gu[1, 0]
    zd = nf ** 2 * Gd[0, 0] * Gd[1, 1] - nf * Gd[0, 1] * Gd[1, 0]
    a, c = oracle_mod.eval_all_connected_lw(Gu[None], Gd[None], U=U, loop_weight=nf)
    assert a[0] == pytest.approx(U ** 2 * zu * zd, rel=1e-13)
    disc = (nf ** 2 * Gu[0, 0] * Gu[1, 1]) * (nf ** 2 * Gd[0, 0] * Gd[1, 1])
    assert c[0] == pytest.approx(U ** 2 * (zu * zd - disc), rel=1e-12)


# ------------------------------------------------------------------------------------------ half-vertex (R18)
def _golden_counts(name):
    out = {}
    for line in open(os.path.join(GOLDEN, name)):
        if not line.startswith("#"):
            k, v = line.split()
            out[int(k)] = int(v)
    return out


@pytest.mark.parametrize("np_", [1, 2, 3])
@pytest.mark.parametrize("nf", [1.0, 2.0])
def test_halfvertex_matches_plain_enumeration(oracle_mod, np_, nf):
    """Every permutation of the 2n' half-vertices, connectivity of the interaction-line graph by union-find here."""
    m = 2 * np_
    rng = np.random.default_rng(100 + np_)
    W, V = rng.normal(size=(m, m)), rng.uniform(0.5, 2.0, size=np_)
    all_sum = conn_sum = 0.0
    count = 0
    for p in itertools.permutations(range(m)):
        term = (-nf) ** _cycles(p) * np.prod([W[i, p[i]] for i in range(m)])
        all_sum += term
        parent = list(range(np_))

        def find(x):
            while parent[x] != x:
                x = parent[x]
            return x
        for i in range(m):
            a, b = find(i // 2), find(p[i] // 2)
            if a != b:
                parent[a] = b
        if len({find(k) for k in range(np_)}) == 1:
            conn_sum += term
            count += 1
    w = np.prod(-V)
    assert count == _golden_counts("halfvertex_connected_counts.txt")[np_]
    a, c = oracle_mod.eval_halfvertex(W[None], V[None], loop_weight=nf)
    assert a[0] == pytest.approx(w * all_sum, rel=1e-10, abs=1e-12)
    assert c[0] == pytest.approx(w * conn_sum, rel=1e-9, abs=1e-12)


def test_halfvertex_c_enumerator_counts_and_value(oracle_mod):
    counts = _golden_counts("halfvertex_connected_counts.txt")
    rng = np.random.default_rng(7)
    for np_ in (1, 2, 3, 4):
        m = 2 * np_
        W, V = rng.normal(size=(m, m)), rng.uniform(0.5, 2.0, size=np_)
        ab, cb, k = oracle_mod.bruteforce_halfvertex(W, V, 1.0)
        assert k == counts[np_]
        a, c = oracle_mod.eval_halfvertex(W[None], V[None])
        assert a[0] == pytest.approx(ab, rel=1e-10, abs=1e-12)
        assert c[0] == pytest.approx(cb, rel=1e-9, abs=1e-12)


@pytest.mark.parametrize("np_", [2, 4, 6])
def test_halfvertex_reduces_to_two_species_when_classes_do_not_mix(oracle_mod, np_):
    """If no fermion line joins an even half-vertex to an odd one, every permutation factorises into one of the even
    and one of the odd half-vertices: the two species of the Hubbard form, G_up = W[even, even], G_dn = W[odd, odd],
    u_k = V_k.  The two sides run different code (one 2n'-point propagation + reduction over lines against two
    n'-point propagations + reduction over vertices)."""
    m = 2 * np_
    rng = np.random.default_rng(200 + np_)
    B = 3
    Gup = rng.normal(size=(B, np_, np_)) / np.sqrt(np_) + 0.5 * np.eye(np_)
    Gdn = rng.normal(size=(B, np_, np_)) / np.sqrt(np_) + 0.5 * np.eye(np_)
    V = rng.uniform(0.5, 2.0, size=(B, np_))
    W = np.zeros((B, m, m))
    W[:, 0::2, 0::2] = Gup
    W[:, 1::2, 1::2] = Gdn
    for nf in (1.0, 2.0):
        a, c = oracle_mod.eval_halfvertex(W, V, loop_weight=nf)
        a2, c2 = oracle_mod.eval_all_connected_lw(Gup, Gdn, u=V, loop_weight=nf)
        np.testing.assert_allclose(a, a2, rtol=1e-11)
        np.testing.assert_allclose(c, c2, rtol=1e-9)


def test_halfvertex_all_is_a_determinant(oracle_mod):
    """loop_weight = 1: sum over all permutations of the 2n' points = prod(-V) det W (library routine)."""
    rng = np.random.default_rng(8)
    W = rng.normal(size=(4, 10, 10)) / 3.0
    V = rng.uniform(0.5, 2.0, size=(4, 5))
    a, _ = oracle_mod.eval_halfvertex(W, V)
    ref = np.prod(-V, axis=1) * np.linalg.det(W)          # (-1)^cyc = sgn for an even number of points
    np.testing.assert_allclose(a, ref, rtol=1e-10)


# ------------------------------------------------------------------------------------------ conditioning sums
def _ordered_partitions(items):
    """Every ordered tuple of disjoint non-empty blocks whose union is `items` (the empty tuple for no items)."""
    items = list(items)
    if not items:
        yield ()
        return
    for r in range(1, len(items) + 1):
        for first in itertools.combinations(items, r):
            rest = [x for x in items if x not in first]
            for tail in _ordered_partitions(rest):
                yield (first,) + tail


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5])
def test_abs_sum_is_the_majorant_of_the_recursion(oracle_mod, n):
    """What oracle_abs_sum(s) returns, written out: with |D|[S] = prod|u| perm|Gup[S,S]| perm|Gdn[S,S]| (Ryser),
    abs_all = |D|[full] and abs_conn = the sum of |every product the subset recursion forms| when it is unrolled,
    i.e. sum over T1 containing vertex 0 of |D|[T1] times the sum over ORDERED partitions (B1..Bk) of the remaining
    vertices of prod |D|[Bi]  (each subtraction C[T] D[S minus T] of the recursion, expanded down to D's)."""
    rng = np.random.default_rng(300 + n)
    Gup, Gdn, u = rng.normal(size=(n, n)), rng.normal(size=(n, n)), rng.uniform(0.5, 2.0, size=n)

    def absD(block):
        idx = list(block)
        return (np.prod(np.abs(u[idx])) * _ryser_permanent(np.abs(Gup[np.ix_(idx, idx)])) *
                _ryser_permanent(np.abs(Gdn[np.ix_(idx, idx)])))
    others = list(range(1, n))
    total = 0.0
    for r in range(len(others) + 1):
        for extra in itertools.combinations(others, r):
            rest = [x for x in others if x not in extra]
            total += absD((0,) + extra) * sum(np.prod([absD(b) for b in part]) for part in _ordered_partitions(rest))
    ac, aa = oracle_mod.abs_sums(Gup[None], Gdn[None], u=u[None])
    assert aa[0] == pytest.approx(absD(range(n)), rel=1e-12)
    assert ac[0] == pytest.approx(total, rel=1e-12)
    assert oracle_mod.abs_sum(Gup, Gdn, u) == pytest.approx(total, rel=1e-12)
    # it bounds the exact connected value, which is what the conditioning number kappa = abs_conn / |connected| uses
    assert total >= abs(oracle_mod.bruteforce(Gup, Gdn, u)[1])
