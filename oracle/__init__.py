"""ctypes loader for the CPU oracle (oracle/cos_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product package paper_2501_00675_b200 never imports
this module and this module never imports the product package.

Every wrapper only marshals numpy arrays into the C functions; the arithmetic is all in
cos_oracle.c / cos_oracle_core.inc, where each function cites the passage of the paper
 or the DESIGN.md reading it follows.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# COS_ORACLE_SANITIZE=1: a second build with AddressSanitizer + UndefinedBehaviorSanitizer, used as
#   COS_ORACLE_SANITIZE=1 LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 \
#       python -m pytest tests -m "not gpu" -k oracle
_SANITIZE = os.environ.get("COS_ORACLE_SANITIZE", "") not in ("", "0")
_SO = os.path.join(_HERE, "liboracle_san.so" if _SANITIZE else "liboracle.so")
_SRC = [os.path.join(_HERE, "cos_oracle.c"), os.path.join(_HERE, "cos_oracle_core.inc")]
_lib = None

_c_double_p = ctypes.POINTER(ctypes.c_double)
_c_int_p = ctypes.POINTER(ctypes.c_int)


def build(force: bool = False) -> str:
    """Compile liboracle.so with gcc if it is missing or older than its sources."""
    stale = force or not os.path.exists(_SO) or any(
        os.path.getmtime(s) > os.path.getmtime(_SO) for s in _SRC)
    if stale:
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               _SRC[0], "-o", _SO, "-lm"]
        if _SANITIZE:
            cmd[1:1] = ["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        lib.oracle_build_G.restype = None
        lib.oracle_build_G.argtypes = [ctypes.c_int, ctypes.c_longlong, _c_int_p, _c_double_p,
                                       _c_double_p, _c_double_p, ctypes.c_int, ctypes.c_int,
                                       ctypes.c_int, ctypes.c_double, ctypes.c_double,
                                       _c_double_p, _c_double_p]
        for name in ("oracle_eval", "oracle_eval_f80"):
            f = getattr(lib, name)
            f.restype = ctypes.c_int
            f.argtypes = [ctypes.c_int, ctypes.c_longlong, _c_double_p, _c_double_p, _c_double_p,
                          ctypes.c_double, _c_double_p, _c_double_p, ctypes.c_int]
        for name in ("oracle_eval_lw", "oracle_eval_lw_f80"):
            f = getattr(lib, name)
            f.restype = ctypes.c_int
            f.argtypes = [ctypes.c_int, ctypes.c_longlong, _c_double_p, _c_double_p, _c_double_p,
                          ctypes.c_double, ctypes.c_double, _c_double_p, _c_double_p, ctypes.c_int]
        lib.oracle_eval_halfvertex.restype = ctypes.c_int
        lib.oracle_eval_halfvertex.argtypes = [ctypes.c_int, ctypes.c_longlong, _c_double_p, _c_double_p,
                                               ctypes.c_double, _c_double_p, _c_double_p, ctypes.c_int]
        lib.oracle_bruteforce_lw.restype = ctypes.c_int
        lib.oracle_bruteforce_lw.argtypes = [ctypes.c_int, _c_double_p, _c_double_p, _c_double_p, ctypes.c_double,
                                             _c_double_p, _c_double_p, ctypes.POINTER(ctypes.c_longlong)]
        lib.oracle_bruteforce_halfvertex.restype = ctypes.c_int
        lib.oracle_bruteforce_halfvertex.argtypes = [ctypes.c_int, _c_double_p, _c_double_p, ctypes.c_double,
                                                     _c_double_p, _c_double_p, ctypes.POINTER(ctypes.c_longlong)]
        lib.oracle_minors_lw.restype = None
        lib.oracle_minors_lw.argtypes = [ctypes.c_int, _c_double_p, ctypes.c_double, _c_double_p]
        lib.oracle_minors.restype = None
        lib.oracle_minors.argtypes = [ctypes.c_int, _c_double_p, _c_double_p]
        lib.oracle_DC.restype = None
        lib.oracle_DC.argtypes = [ctypes.c_int, _c_double_p, _c_double_p, _c_double_p,
                                  _c_double_p, _c_double_p]
        lib.oracle_abs_sum.restype = ctypes.c_double
        lib.oracle_abs_sum.argtypes = [ctypes.c_int, _c_double_p, _c_double_p, _c_double_p, _c_double_p]
        lib.oracle_abs_sums.restype = None
        lib.oracle_abs_sums.argtypes = [ctypes.c_int, ctypes.c_longlong, _c_double_p, _c_double_p,
                                        _c_double_p, ctypes.c_double, _c_double_p, _c_double_p,
                                        ctypes.c_int]
        lib.oracle_bruteforce.restype = ctypes.c_int
        lib.oracle_bruteforce.argtypes = [ctypes.c_int, _c_double_p, _c_double_p, _c_double_p,
                                          _c_double_p, _c_double_p,
                                          ctypes.POINTER(ctypes.c_longlong)]
        lib.oracle_philox4x32_10.restype = None
        lib.oracle_philox4x32_10.argtypes = [ctypes.POINTER(ctypes.c_uint32)] * 3
        lib.oracle_u53.restype = ctypes.c_double
        lib.oracle_u53.argtypes = [ctypes.c_uint32, ctypes.c_uint32]
        lib.oracle_mc_run.restype = None
        lib.oracle_mc_run.argtypes = [ctypes.c_int, ctypes.c_longlong, ctypes.c_int, ctypes.c_ulonglong, _c_int_p,
                                      _c_double_p, _c_double_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                      ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_double, _c_double_p,
                                      ctypes.POINTER(ctypes.c_ubyte), _c_double_p,
                                      ctypes.POINTER(ctypes.c_longlong), _c_double_p, ctypes.c_int]
        lib.oracle_max_threads.restype = ctypes.c_int
        lib.oracle_max_threads.argtypes = []
        _lib = lib
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(_c_double_p)


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def build_G(xy, tau, table_up, table_dn, beta, g_diag=0.0):
    """G assembly.  xy [B,n,2] int32, tau [B,n]; tables [Lx,Ly,ntau].  Returns (Gup, Gdn) [B,n,n]."""
    lib = _load()
    xy = np.ascontiguousarray(xy, dtype=np.int32)
    tau = _f64(tau)
    table_up = _f64(table_up)
    table_dn = table_up if table_dn is None else _f64(table_dn)
    B, n = tau.shape
    Lx, Ly, ntau = table_up.shape
    assert xy.shape == (B, n, 2) and table_dn.shape == table_up.shape
    Gup = np.empty((B, n, n), dtype=np.float64)
    Gdn = np.empty((B, n, n), dtype=np.float64)
    lib.oracle_build_G(n, B, xy.ctypes.data_as(_c_int_p), _p(tau), _p(table_up), _p(table_dn),
                       Lx, Ly, ntau, float(beta), float(g_diag), _p(Gup), _p(Gdn))
    return Gup, Gdn


def _eval(fname, Gup, Gdn, U, u, threads, loop_weight=None):
    lib = _load()
    Gup = _f64(Gup)
    Gdn = Gup if Gdn is None else _f64(Gdn)
    B, n, n2 = Gup.shape
    assert n == n2 and Gdn.shape == Gup.shape and 1 <= n <= 20
    up = None
    if u is not None:
        u = _f64(u)
        assert u.shape == (B, n)
        up = _p(u)
    out_all = np.empty(B, dtype=np.float64)
    out_conn = np.empty(B, dtype=np.float64)
    if loop_weight is None:
        used = getattr(lib, fname)(n, B, _p(Gup), _p(Gdn), up, float(U), _p(out_all), _p(out_conn), int(threads))
    else:
        used = getattr(lib, fname)(n, B, _p(Gup), _p(Gdn), up, float(U), float(loop_weight), _p(out_all),
                                   _p(out_conn), int(threads))
    return out_all, out_conn, used


def eval_all_connected(Gup, Gdn=None, U=1.0, u=None, threads=0):
    """Returns (all[B], connected[B]) in FP64.  threads<=0: every OpenMP thread."""
    a, c, _ = _eval("oracle_eval", Gup, Gdn, U, u, threads)
    return a, c


def eval_all_connected_timed(Gup, Gdn=None, U=1.0, u=None, threads=0):
    """Like eval_all_connected but also returns the thread count the C code used."""
    return _eval("oracle_eval", Gup, Gdn, U, u, threads)


def eval_all_connected_f80(Gup, Gdn=None, U=1.0, u=None, threads=0):
    """Long-double accumulators ("truth" for conditioning reports)."""
    a, c, _ = _eval("oracle_eval_f80", Gup, Gdn, U, u, threads)
    return a, c


def eval_all_connected_lw(Gup, Gdn=None, U=1.0, u=None, loop_weight=1.0, threads=0, f80=False):
    """Loop-weight generalisation (reading R17): every closed fermion loop contributes -loop_weight."""
    a, c, _ = _eval("oracle_eval_lw_f80" if f80 else "oracle_eval_lw", Gup, Gdn, U, u, threads, loop_weight)
    return a, c


def eval_halfvertex(W, V, loop_weight=1.0, threads=0):
    """Half-vertex formulation (reading R18).  W [B, 2n', 2n'], V [B, n'].  Returns (all[B], connected[B])."""
    lib = _load()
    W, V = _f64(W), _f64(V)
    B, m, m2 = W.shape
    assert m == m2 and m % 2 == 0 and V.shape == (B, m // 2) and m <= 20
    out_all = np.empty(B, dtype=np.float64)
    out_conn = np.empty(B, dtype=np.float64)
    lib.oracle_eval_halfvertex(m // 2, B, _p(W), _p(V), float(loop_weight), _p(out_all), _p(out_conn), int(threads))
    return out_all, out_conn


def bruteforce_lw(Gup, Gdn, u, loop_weight):
    """Plain definition with (-loop_weight)^(closed loops), n <= 8.  Returns (all, connected, count)."""
    lib = _load()
    Gup, Gdn, u = _f64(Gup), _f64(Gdn), _f64(u)
    a, c, k = ctypes.c_double(), ctypes.c_double(), ctypes.c_longlong()
    rc = lib.oracle_bruteforce_lw(Gup.shape[0], _p(Gup), _p(Gdn), _p(u), float(loop_weight), ctypes.byref(a),
                                  ctypes.byref(c), ctypes.byref(k))
    if rc != 0:
        raise ValueError("bruteforce_lw: n out of range")
    return a.value, c.value, k.value


def bruteforce_halfvertex(W, V, loop_weight=1.0):
    """Plain definition of the half-vertex formulation, n' <= 4.  Returns (all, connected, count)."""
    lib = _load()
    W, V = _f64(W), _f64(V)
    a, c, k = ctypes.c_double(), ctypes.c_double(), ctypes.c_longlong()
    rc = lib.oracle_bruteforce_halfvertex(V.shape[0], _p(W), _p(V), float(loop_weight), ctypes.byref(a),
                                          ctypes.byref(c), ctypes.byref(k))
    if rc != 0:
        raise ValueError("bruteforce_halfvertex: n' out of range")
    return a.value, c.value, k.value


def minors_lw(W, loop_weight):
    """Z[S] = sum over permutations of S of (-loop_weight)^cyc prod W, for every subset S."""
    lib = _load()
    W = _f64(W)
    n = W.shape[0]
    Z = np.empty(1 << n, dtype=np.float64)
    lib.oracle_minors_lw(n, _p(W), float(loop_weight), _p(Z))
    return Z


def minors(W):
    """Z[S] = sum over permutations of S of (-1)^cyc prod W, for every subset S.  W [n,n] -> [2^n]."""
    lib = _load()
    W = _f64(W)
    n = W.shape[0]
    Z = np.empty(1 << n, dtype=np.float64)
    lib.oracle_minors(n, _p(W), _p(Z))
    return Z


def DC(Gup, Gdn, u):
    """D[S], C[S] for every subset S of one configuration."""
    lib = _load()
    Gup, Gdn, u = _f64(Gup), _f64(Gdn), _f64(u)
    n = Gup.shape[0]
    D = np.empty(1 << n, dtype=np.float64)
    C = np.empty(1 << n, dtype=np.float64)
    lib.oracle_DC(n, _p(Gup), _p(Gdn), _p(u), _p(D), _p(C))
    return D, C


def abs_sum(Gup, Gdn, u):
    """Sum of |term| over the connected recursion with every sign dropped (one configuration)."""
    lib = _load()
    Gup, Gdn, u = _f64(Gup), _f64(Gdn), _f64(u)
    return float(lib.oracle_abs_sum(Gup.shape[0], _p(Gup), _p(Gdn), _p(u), None))


def abs_sums(Gup, Gdn=None, U=1.0, u=None, threads=0):
    """Rounding-error scales for a batch: (abs_connected[B], abs_all[B]); see DESIGN.md §3 tolerance."""
    lib = _load()
    Gup = _f64(Gup)
    Gdn = Gup if Gdn is None else _f64(Gdn)
    B, n, _ = Gup.shape
    up = None
    if u is not None:
        u = _f64(u)
        up = _p(u)
    ac = np.empty(B, dtype=np.float64)
    aa = np.empty(B, dtype=np.float64)
    lib.oracle_abs_sums(n, B, _p(Gup), _p(Gdn), up, float(U), _p(ac), _p(aa), int(threads))
    return ac, aa


def bruteforce(Gup, Gdn, u):
    """Plain definition over all (n!)^2 permutation pairs, n <= 8.  Returns (all, connected, count)."""
    lib = _load()
    Gup, Gdn, u = _f64(Gup), _f64(Gdn), _f64(u)
    n = Gup.shape[0]
    a = ctypes.c_double()
    c = ctypes.c_double()
    k = ctypes.c_longlong()
    rc = lib.oracle_bruteforce(n, _p(Gup), _p(Gdn), _p(u), ctypes.byref(a), ctypes.byref(c),
                               ctypes.byref(k))
    if rc != 0:
        raise ValueError("bruteforce: n out of range")
    return a.value, c.value, k.value


def philox4x32_10(counter, key):
    """Counter-based generator of reading R19: counter (4 x uint32), key (2 x uint32) -> 4 x uint32."""
    lib = _load()
    c = (ctypes.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in counter])
    k = (ctypes.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (ctypes.c_uint32 * 4)()
    lib.oracle_philox4x32_10(c, k, o)
    return tuple(int(x) for x in o)


def u53(a, b):
    return float(_load().oracle_u53(int(a) & 0xFFFFFFFF, int(b) & 0xFFFFFFFF))


def mc_run(xy, tau, table, beta, steps, seed, U=1.0, g_diag=0.0, loop_weight=1.0, threads=0):
    """Metropolis walkers of reading R19.  xy [W,n,2] int32, tau [W,n] (copied, not modified).  Returns a dict:
    xy, tau (final state), weight [W], accept [steps,W] uint8, margin [steps,W], accepted [W], sign_sum [W]."""
    lib = _load()
    xy = np.array(xy, dtype=np.int32, order="C", copy=True)
    tau = np.array(tau, dtype=np.float64, order="C", copy=True)
    table = _f64(table)
    W, n = tau.shape
    Lx, Ly, ntau = table.shape
    weight = np.empty(W)
    hist = np.empty((steps, W), dtype=np.uint8)
    margin = np.empty((steps, W))
    accepted = np.empty(W, dtype=np.int64)
    sign_sum = np.empty(W)
    lib.oracle_mc_run(n, W, int(steps), int(seed), xy.ctypes.data_as(_c_int_p), _p(tau), _p(table), Lx, Ly, ntau,
                      float(beta), float(g_diag), float(U), float(loop_weight), _p(weight),
                      hist.ctypes.data_as(ctypes.POINTER(ctypes.c_ubyte)), _p(margin),
                      accepted.ctypes.data_as(ctypes.POINTER(ctypes.c_longlong)), _p(sign_sum), int(threads))
    return {"xy": xy, "tau": tau, "weight": weight, "accept": hist, "margin": margin, "accepted": accepted,
            "sign_sum": sign_sum}
