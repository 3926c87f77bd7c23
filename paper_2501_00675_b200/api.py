"""Thin ctypes binding over the C-ABI of libcos_b200.so (include/cos.h).

Argument marshalling only: every step of the hot path runs in the CUDA kernels of the library.
PyTorch appears here solely as the owner of device memory and streams (`tensor.data_ptr()`,
`torch.cuda.current_stream()`).  There is no CPU fallback: if the library is missing or no
sm_100 device is present, the calls raise.

    ctx = Context()                         # cos_create on the current device / stream
    ctx.set_g0_table(table_dev, beta)       # cos_set_g0_table
    ctx.build_G(xy, tau, Gup, Gdn)          # cos_build_G
    ctx.eval_connected(Gup, Gdn, out, U=4.0)  # cos_eval_connected
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcos_b200.so")

COS_OK, COS_EINVAL, COS_ECUDA, COS_ENOMEM, COS_ENOTABLE, COS_ETOOBIG = 0, -1, -2, -3, -4, -5
COS_NOALLOC_MIN_ORDER, COS_NOALLOC_MAX_ORDER, COS_NOALLOC_MAX_BATCH = 11, 12, 1 << 20
COS_MAX_ORDER = 16

_lib = None
_vp = ctypes.c_void_p
_ll = ctypes.c_longlong
_dbl = ctypes.c_double
_int = ctypes.c_int

# name -> (restype, argtypes); mirrors include/cos.h one to one
SIGNATURES = {
    "cos_create": (_int, [ctypes.POINTER(_vp), _int, _vp]),
    "cos_destroy": (_int, [_vp]),
    "cos_set_g0_table": (_int, [_vp, _int, _vp, _int, _int, _int, _dbl]),
    "cos_build_G": (_int, [_vp, _int, _ll, _vp, _vp, _dbl, _vp, _vp]),
    "cos_eval_all": (_int, [_vp, _int, _ll, _vp, _vp, _vp, _dbl, _vp]),
    "cos_eval_connected": (_int, [_vp, _int, _ll, _vp, _vp, _vp, _dbl, _vp]),
    "cos_eval_all_f32": (_int, [_vp, _int, _ll, _vp, _vp, _vp, _dbl, _vp]),
    "cos_eval_connected_noalloc": (_int, [_vp, _int, _ll, _vp, _vp, _vp, _dbl, _vp]),
    "cos_eval_connected_f32": (_int, [_vp, _int, _ll, _vp, _vp, _vp, _dbl, _vp]),
    "cos_eval_connected_xt": (_int, [_vp, _int, _ll, _vp, _vp, _dbl, _vp, _dbl, _vp]),
    "cos_eval_connected_xt_host": (_int, [_vp, _int, _ll, _vp, _vp, _dbl, _vp, _dbl, _vp]),
    "cos_mc_run": (_int, [_vp, _int, _ll, _int, ctypes.c_ulonglong, _vp, _vp, _dbl, _dbl, _vp, _vp, _vp, _vp]),
    "cos_set_loop_weight": (_int, [_vp, _dbl]),
    "cos_eval_halfvertex": (_int, [_vp, _int, _ll, _vp, _vp, _int, _vp]),
    "cos_debug_force_generic": (_int, [_vp, _int]),
    "cos_last_launch_count": (_int, [_vp]),
    "cos_last_kernel_name": (ctypes.c_char_p, [_vp]),
    "cos_enable_kernel_timer": (_int, [_vp, _int]),
    "cos_reset_kernel_timer": (_int, [_vp]),
    "cos_kernel_time_ms": (_int, [_vp, ctypes.POINTER(_dbl), ctypes.POINTER(_ll)]),
    "cos_flop_count": (_ll, [_int, _int, _int]),
    "cos_probe_dfma": (_int, [_vp, ctypes.POINTER(_dbl)]),
    "cos_probe_smem": (_int, [_vp, ctypes.POINTER(_dbl)]),
    "cos_strerror": (ctypes.c_char_p, [_int]),
    "cos_last_cuda_error": (ctypes.c_char_p, [_vp]),
    "cos_abi_version": (_int, []),
}


class CosError(RuntimeError):
    def __init__(self, code, text):
        super().__init__(f"libcos_b200: {text} (status {code})")
        self.code = code


def load_library():
    """dlopen the in-tree library; raises if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} is missing: build it with `python -m paper_2501_00675_b200.build` "
                "(or __graft_entry__.build()); there is no CPU fallback")
        lib = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def strerror(code: int) -> str:
    return load_library().cos_strerror(int(code)).decode()


def flop_count(n: int, n_species: int, connected: bool) -> int:
    """Algorithmic FLOP per configuration (include/cos.h: cos_flop_count)."""
    v = int(load_library().cos_flop_count(int(n), int(n_species), 1 if connected else 0))
    if v < 0:
        raise CosError(COS_EINVAL, "invalid argument")
    return v


def _ptr(t):
    """Device/host address of a torch tensor or numpy array, or None."""
    if t is None:
        return None
    if hasattr(t, "data_ptr"):
        return ctypes.c_void_p(t.data_ptr())
    return ctypes.c_void_p(t.ctypes.data)


def _kind(t):
    """('f64' | 'i32' | other, shape tuple) of a torch tensor or numpy array."""
    name = str(t.dtype).replace("torch.", "")
    return {"float64": "f64", "int32": "i32"}.get(name, name), tuple(int(x) for x in t.shape)


class Context:
    """Owner of one cos_ctx.  All tensors passed to the d_* arguments must live on `device`.

    The ctx launches on the stream given at construction (default: torch's current stream of the device at that
    moment); work the caller enqueues on another stream must be ordered with it by the caller.  Every call leaves
    `device` as the current CUDA device of the calling thread."""

    def __init__(self, device: int | None = None, stream=None):
        import torch  # device memory and streams only

        lib = load_library()
        if not torch.cuda.is_available():
            raise CosError(COS_ECUDA, "no CUDA device: libcos_b200 has no CPU fallback")
        self.device = torch.cuda.current_device() if device is None else int(device)
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        self.stream = stream
        handle = _vp()
        rc = lib.cos_create(ctypes.byref(handle), self.device, _vp(stream.cuda_stream))
        if rc != COS_OK:
            raise CosError(rc, strerror(rc))
        self._h = handle
        self._lib = lib
        self._table_refs = {}

    # -- lifetime -------------------------------------------------------------------------
    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._lib.cos_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def _check(self, rc):
        if rc != COS_OK:
            text = strerror(rc)
            if rc == COS_ECUDA:
                text += ": " + self._lib.cos_last_cuda_error(self._h).decode()
            raise CosError(rc, text)

    def _dev(self, t, kind, shape, name, optional=False):
        """Marshalling guard: dtype, shape, contiguity and residency of a d_* argument (no arithmetic)."""
        if t is None:
            if optional:
                return None
            raise CosError(COS_EINVAL, f"{name} is required")
        k, shp = _kind(t)
        if k != kind:
            raise CosError(COS_EINVAL, f"{name}: dtype {t.dtype}, expected {'float64' if kind == 'f64' else 'int32'}")
        if shape is not None and shp != tuple(shape):
            raise CosError(COS_EINVAL, f"{name}: shape {shp}, expected {tuple(shape)}")
        if not getattr(t, "is_cuda", False) or t.device.index != self.device:
            raise CosError(COS_EINVAL, f"{name}: must be a CUDA tensor on device {self.device}")
        if not t.is_contiguous():
            raise CosError(COS_EINVAL, f"{name}: must be contiguous")
        return _ptr(t)

    @staticmethod
    def _host(t, kind, shape, name, optional=False):
        if t is None:
            if optional:
                return None
            raise CosError(COS_EINVAL, f"{name} is required")
        k, shp = _kind(t)
        if k != kind or shp != tuple(shape):
            raise CosError(COS_EINVAL, f"{name}: {t.dtype} {shp}, expected {kind} {tuple(shape)}")
        if getattr(t, "is_cuda", False):
            raise CosError(COS_EINVAL, f"{name}: must be a host buffer")
        contiguous = t.is_contiguous() if hasattr(t, "is_contiguous") else t.flags["C_CONTIGUOUS"]
        if not contiguous:
            raise CosError(COS_EINVAL, f"{name}: must be contiguous")
        return _ptr(t)

    # -- the boundary ---------------------------------------------------------------------
    def set_g0_table(self, d_table, beta: float, spin: int = -1):
        """d_table: CUDA float64 tensor [Lx, Ly, ntau] (tau fastest); kept alive by this object."""
        Lx, Ly, ntau = (int(s) for s in d_table.shape)
        p = self._dev(d_table, "f64", (Lx, Ly, ntau), "d_table")
        self._check(self._lib.cos_set_g0_table(self._h, int(spin), p, Lx, Ly, ntau, float(beta)))
        self._table_refs[spin] = d_table

    def build_G(self, d_xy, d_tau, d_Gup, d_Gdn=None, g_diag: float = 0.0):
        batch, n = (int(s) for s in d_tau.shape)
        self._check(self._lib.cos_build_G(self._h, n, batch, self._dev(d_xy, "i32", (batch, n, 2), "d_xy"),
                                          self._dev(d_tau, "f64", (batch, n), "d_tau"), float(g_diag),
                                          self._dev(d_Gup, "f64", (batch, n, n), "d_Gup"),
                                          self._dev(d_Gdn, "f64", (batch, n, n), "d_Gdn", optional=True)))

    def _eval_ptrs(self, d_Gup, d_Gdn, d_out, d_u):
        batch, n = int(d_Gup.shape[0]), int(d_Gup.shape[1])
        return (n, batch, self._dev(d_Gup, "f64", (batch, n, n), "d_Gup"), self._dev(d_Gdn, "f64", (batch, n, n), "d_Gdn"),
                self._dev(d_u, "f64", (batch, n), "d_u", optional=True), self._dev(d_out, "f64", (batch,), "d_out"))

    def eval_all(self, d_Gup, d_Gdn, d_out, U: float = 1.0, d_u=None):
        n, batch, gu, gd, u, out = self._eval_ptrs(d_Gup, d_Gdn, d_out, d_u)
        self._check(self._lib.cos_eval_all(self._h, n, batch, gu, gd, u, float(U), out))

    def eval_connected(self, d_Gup, d_Gdn, d_out, U: float = 1.0, d_u=None):
        n, batch, gu, gd, u, out = self._eval_ptrs(d_Gup, d_Gdn, d_out, d_u)
        self._check(self._lib.cos_eval_connected(self._h, n, batch, gu, gd, u, float(U), out))

    def eval_connected_noalloc(self, d_Gup, d_Gdn, d_out, U: float = 1.0, d_u=None):
        """Allocation-free variant (include/cos.h: cos_eval_connected_noalloc): orders 11..12, scratch in a static
        device array shared by every call on the GPU; CosError(COS_ETOOBIG) beyond the stated maximum."""
        n, batch, gu, gd, u, out = self._eval_ptrs(d_Gup, d_Gdn, d_out, d_u)
        self._check(self._lib.cos_eval_connected_noalloc(self._h, n, batch, gu, gd, u, float(U), out))

    def eval_all_f32(self, d_Gup, d_Gdn, d_out, U: float = 1.0, d_u=None):
        """FP32 variant (include/cos.h: cos_eval_all_f32); FP64 tensors in and out."""
        n, batch, gu, gd, u, out = self._eval_ptrs(d_Gup, d_Gdn, d_out, d_u)
        self._check(self._lib.cos_eval_all_f32(self._h, n, batch, gu, gd, u, float(U), out))

    def eval_connected_f32(self, d_Gup, d_Gdn, d_out, U: float = 1.0, d_u=None):
        n, batch, gu, gd, u, out = self._eval_ptrs(d_Gup, d_Gdn, d_out, d_u)
        self._check(self._lib.cos_eval_connected_f32(self._h, n, batch, gu, gd, u, float(U), out))

    def eval_connected_xt(self, d_xy, d_tau, d_out, U: float = 1.0, d_u=None, g_diag: float = 0.0):
        batch, n = (int(s) for s in d_tau.shape)
        self._check(self._lib.cos_eval_connected_xt(
            self._h, n, batch, self._dev(d_xy, "i32", (batch, n, 2), "d_xy"), self._dev(d_tau, "f64", (batch, n), "d_tau"),
            float(g_diag), self._dev(d_u, "f64", (batch, n), "d_u", optional=True), float(U),
            self._dev(d_out, "f64", (batch,), "d_out")))

    def eval_connected_xt_host(self, h_xy, h_tau, h_out, U: float = 1.0, h_u=None, g_diag: float = 0.0):
        """Host buffers (numpy arrays or pinned CPU tensors); synchronises before returning."""
        batch, n = (int(s) for s in h_tau.shape)
        self._check(self._lib.cos_eval_connected_xt_host(
            self._h, n, batch, self._host(h_xy, "i32", (batch, n, 2), "h_xy"), self._host(h_tau, "f64", (batch, n), "h_tau"),
            float(g_diag), self._host(h_u, "f64", (batch, n), "h_u", optional=True), float(U),
            self._host(h_out, "f64", (batch,), "h_out")))

    def mc_run(self, d_xy, d_tau, d_weight, steps: int, seed: int, U: float = 1.0, g_diag: float = 0.0,
               d_accept_hist=None, d_accepted=None, d_sign_sum=None):
        """Metropolis walkers on the device (include/cos.h: cos_mc_run); d_xy / d_tau are updated in place."""
        walkers, n = (int(s) for s in d_tau.shape)
        hist = None
        if d_accept_hist is not None:
            k, shp = _kind(d_accept_hist)
            if k != "uint8" or shp != (int(steps), walkers) or not d_accept_hist.is_cuda or not d_accept_hist.is_contiguous():
                raise CosError(COS_EINVAL, "d_accept_hist: expected a contiguous CUDA uint8 tensor [steps, walkers]")
            hist = _ptr(d_accept_hist)
        acc = None
        if d_accepted is not None:
            k, shp = _kind(d_accepted)
            if k != "int64" or shp != (walkers,) or not d_accepted.is_cuda or not d_accepted.is_contiguous():
                raise CosError(COS_EINVAL, "d_accepted: expected a contiguous CUDA int64 tensor [walkers]")
            acc = _ptr(d_accepted)
        self._check(self._lib.cos_mc_run(
            self._h, n, walkers, int(steps), int(seed), self._dev(d_xy, "i32", (walkers, n, 2), "d_xy"),
            self._dev(d_tau, "f64", (walkers, n), "d_tau"), float(g_diag), float(U),
            self._dev(d_weight, "f64", (walkers,), "d_weight"), hist, acc,
            self._dev(d_sign_sum, "f64", (walkers,), "d_sign_sum", optional=True)))

    def eval_halfvertex(self, d_W, d_V, d_out, connected: bool = True):
        """Half-vertex formulation (include/cos.h: cos_eval_halfvertex).  d_W [B, 2n', 2n'], d_V [B, n']."""
        batch, m = int(d_W.shape[0]), int(d_W.shape[1])
        self._check(self._lib.cos_eval_halfvertex(
            self._h, m // 2, batch, self._dev(d_W, "f64", (batch, m, m), "d_W"),
            self._dev(d_V, "f64", (batch, m // 2), "d_V"), 1 if connected else 0, self._dev(d_out, "f64", (batch,), "d_out")))

    def set_loop_weight(self, n_f: float = 1.0):
        """-n_f per closed fermion loop (include/cos.h: cos_set_loop_weight); 1 is the paper's rule."""
        self._check(self._lib.cos_set_loop_weight(self._h, float(n_f)))

    def force_generic(self, on: bool = True):
        """Cross-check switch (include/cos.h: cos_debug_force_generic)."""
        self._check(self._lib.cos_debug_force_generic(self._h, 1 if on else 0))

    # -- bookkeeping and probes -------------------------------------------------------------
    def last_launch_count(self) -> int:
        return int(self._lib.cos_last_launch_count(self._h))

    def last_kernel_name(self) -> str:
        return self._lib.cos_last_kernel_name(self._h).decode()

    def enable_kernel_timer(self, on: bool = True):
        self._check(self._lib.cos_enable_kernel_timer(self._h, 1 if on else 0))

    def reset_kernel_timer(self):
        self._check(self._lib.cos_reset_kernel_timer(self._h))

    def kernel_time_ms(self):
        avg, cnt = _dbl(), _ll()
        self._check(self._lib.cos_kernel_time_ms(self._h, ctypes.byref(avg), ctypes.byref(cnt)))
        return avg.value, cnt.value

    def probe_dfma_tflops(self) -> float:
        v = _dbl()
        self._check(self._lib.cos_probe_dfma(self._h, ctypes.byref(v)))
        return v.value

    def probe_smem_gbs(self) -> float:
        v = _dbl()
        self._check(self._lib.cos_probe_smem(self._h, ctypes.byref(v)))
        return v.value
