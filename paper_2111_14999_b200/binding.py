"""Thin ctypes binding of include/phoebe_elph.h -- argument marshalling only.

Every step of the path runs in the CUDA kernels of libphoebe_elph.so; PyTorch is
used for device memory and streams only.  There is no CPU fallback: if the
shared library is missing or no CUDA device is present, the calls raise.
This module never imports ``oracle``.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, byref, c_char_p, c_double, c_int32, c_int64, c_size_t, c_void_p

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libphoebe_elph.so")

KERNEL_KINDS = ["setk_stream", "setk_rotate", "qphase", "contract", "rotate_epilogue", "setk_gemm", "rate_reduce", "polar", "pack", "qfold"]

#: every symbol declared in include/phoebe_elph.h
EXPORTS = [
    "phoebe_elph_workspace_bytes", "phoebe_elph_setup", "phoebe_elph_set_k", "phoebe_elph_set_k_host",
    "phoebe_elph_set_k_batch", "phoebe_elph_set_k_batch_host", "phoebe_elph_select_k",
    "phoebe_elph_q_batch", "phoebe_elph_q_batch_multi", "phoebe_elph_q_batch_host", "phoebe_elph_q_batch_host_async", "phoebe_elph_wait",
    "phoebe_elph_q_batch_rates", "phoebe_elph_q_batch_rates_host", "phoebe_elph_q_batch_rates_host_async",
    "phoebe_elph_q_batch_rates_multi", "phoebe_elph_q_batch_multi_host_async", "phoebe_elph_q_batch_rates_multi_host_async",
    "phoebe_elph_copy_g1", "phoebe_elph_g1_buffer", "phoebe_elph_set_polar", "phoebe_elph_set_conventions", "phoebe_elph_launch_counts",
    "phoebe_elph_profile", "phoebe_elph_profile_read", "phoebe_elph_set_tuning", "phoebe_elph_get_tuning",
    "phoebe_elph_destroy", "phoebe_elph_last_error",
    "phoebe_elph_version",
    "phoebe_elph_noalloc_setup", "phoebe_elph_set_k_noalloc", "phoebe_elph_noalloc_last_error",
]

ERRORS = {0: "OK", -1: "E_NULL", -2: "E_DIMS", -3: "E_ALIGN", -4: "E_NO_K", -5: "E_WORKSPACE", -6: "E_CUDA"}


class Dims(ctypes.Structure):
    _fields_ = [(n, c_int32) for n in ("nRe", "nRp", "nw", "nmodes", "nb1_max", "nb2_max", "nq_max", "nk_max")]

    def __init__(self, nRe=0, nRp=0, nw=0, nmodes=0, nb1_max=0, nb2_max=0, nq_max=0, nk_max=0):
        super().__init__(nRe, nRp, nw, nmodes, nb1_max, nb2_max, nq_max, nk_max)


class RateParams(ctypes.Structure):
    """phoebe_elph_rate_params: k_B T, chemical potential, Gaussian sigma (Eq. 61), prefactor of Eq. 29."""
    _fields_ = [(n, c_double) for n in ("kT", "mu", "sigma", "pref")]


class PhoebeElphError(RuntimeError):
    def __init__(self, code, where, text=""):
        self.code = code
        super().__init__(f"{where}: {ERRORS.get(code, code)} {text}".strip())


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen the in-tree C-ABI library; raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(f"{LIB_PATH} not built; run `python -m paper_2111_14999_b200.build` "
                                "(there is no CPU fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    lib.phoebe_elph_workspace_bytes.argtypes = [POINTER(Dims), c_size_t, POINTER(c_size_t), POINTER(c_int32)]
    lib.phoebe_elph_setup.argtypes = [POINTER(c_void_p), c_void_p, c_void_p, c_void_p, c_void_p, c_void_p,
                                      POINTER(Dims), c_void_p, c_size_t, c_void_p]
    lib.phoebe_elph_set_k.argtypes = [c_void_p, c_void_p, c_void_p, c_int32]
    lib.phoebe_elph_set_k_host.argtypes = [c_void_p, c_void_p, c_void_p, c_int32]
    lib.phoebe_elph_set_k_batch.argtypes = [c_void_p, c_int32, c_void_p, c_void_p, c_int32]
    lib.phoebe_elph_set_k_batch_host.argtypes = [c_void_p, c_int32, c_void_p, c_void_p, c_int32]
    lib.phoebe_elph_select_k.argtypes = [c_void_p, c_int32]
    lib.phoebe_elph_q_batch.argtypes = [c_void_p, c_int32, c_int32] + [c_void_p] * 5
    lib.phoebe_elph_q_batch_multi.argtypes = [c_void_p, c_int32, c_int32, c_int32] + [c_void_p] * 5
    lib.phoebe_elph_q_batch_host.argtypes = [c_void_p, c_int32, c_int32] + [c_void_p] * 5
    lib.phoebe_elph_q_batch_host_async.argtypes = [c_void_p, c_int32, c_int32] + [c_void_p] * 5
    lib.phoebe_elph_q_batch_multi_host_async.argtypes = [c_void_p, c_int32, c_int32, c_int32] + [c_void_p] * 5
    lib.phoebe_elph_q_batch_rates_multi_host_async.argtypes = ([c_void_p, c_int32, c_int32, c_int32] + [c_void_p] * 6 +
                                                               [POINTER(RateParams), c_void_p, c_void_p])
    lib.phoebe_elph_wait.argtypes = [c_void_p]
    lib.phoebe_elph_q_batch_rates.argtypes = [c_void_p, c_int32, c_int32] + [c_void_p] * 6 + [POINTER(RateParams), c_void_p, c_void_p]
    lib.phoebe_elph_q_batch_rates_multi.argtypes = [c_void_p, c_int32, c_int32, c_int32] + [c_void_p] * 6 + [POINTER(RateParams), c_void_p, c_void_p]
    lib.phoebe_elph_q_batch_rates_host.argtypes = [c_void_p, c_int32, c_int32] + [c_void_p] * 6 + [POINTER(RateParams), c_void_p, c_void_p]
    lib.phoebe_elph_q_batch_rates_host_async.argtypes = [c_void_p, c_int32, c_int32] + [c_void_p] * 6 + [POINTER(RateParams), c_void_p, c_void_p]
    lib.phoebe_elph_copy_g1.argtypes = [c_void_p, c_void_p, c_size_t]
    lib.phoebe_elph_set_polar.argtypes = [c_void_p, c_void_p, c_int32, c_void_p, c_void_p, c_void_p, c_double]
    lib.phoebe_elph_set_conventions.argtypes = [c_void_p, c_int32, c_int32, c_int32, c_int32]
    lib.phoebe_elph_g1_buffer.argtypes = [c_void_p, c_int32, POINTER(c_void_p), POINTER(c_size_t), POINTER(c_size_t)]
    lib.phoebe_elph_launch_counts.argtypes = [c_void_p, POINTER(c_int64)]
    lib.phoebe_elph_profile.argtypes = [c_void_p, c_int32]
    lib.phoebe_elph_profile_read.argtypes = [c_void_p, POINTER(c_double), POINTER(c_int64)]
    lib.phoebe_elph_set_tuning.argtypes = [c_void_p, c_char_p, c_int64]
    lib.phoebe_elph_get_tuning.argtypes = [c_void_p, c_char_p, POINTER(c_int64)]
    lib.phoebe_elph_destroy.argtypes = [c_void_p]
    lib.phoebe_elph_last_error.argtypes = [c_void_p]
    lib.phoebe_elph_last_error.restype = c_char_p
    lib.phoebe_elph_version.restype = c_char_p
    lib.phoebe_elph_noalloc_setup.argtypes = []
    lib.phoebe_elph_set_k_noalloc.argtypes = [c_void_p, c_void_p, c_void_p] + [c_int32] * 5 + [c_void_p] * 4
    lib.phoebe_elph_noalloc_last_error.restype = c_char_p
    _lib = lib
    return lib


def version() -> str:
    return load_library().phoebe_elph_version().decode()


NOALLOC_MAX_BYTES = 4 << 20       # PHOEBE_ELPH_NOALLOC_MAX_BYTES of include/phoebe_elph.h


def noalloc_setup():
    """phoebe_elph_noalloc_setup: resolve the fixed scratch array's address on the current device (once per device)."""
    lib = load_library()
    rc = lib.phoebe_elph_noalloc_setup()
    if rc:
        raise PhoebeElphError(rc, "phoebe_elph_noalloc_setup", lib.phoebe_elph_noalloc_last_error().decode())


def set_k_noalloc(gW, Re, deg_e, k, Uk, g1_out, stream=None):
    """phoebe_elph_set_k_noalloc (a1 + a2 without context, workspace or allocation): gW [nRp][nRe][nw][nw][nm] complex128,
    Re [nRe][3] float64, deg_e [nRe] float64 or None, Uk [nw][nb1] complex128, g1_out [nRp][nb1][nw][nm] complex128 -- all
    CUDA tensors; k: three host floats.  Marshalling only; raises PhoebeElphError."""
    import numpy as np
    import torch
    lib = load_library()
    for name, t, dt in (("gW", gW, torch.complex128), ("Re", Re, torch.float64), ("Uk", Uk, torch.complex128),
                        ("g1_out", g1_out, torch.complex128)) + ((("deg_e", deg_e, torch.float64),) if deg_e is not None else ()):
        if not (t.is_cuda and t.dtype == dt and t.is_contiguous()):
            raise TypeError(f"set_k_noalloc: {name} must be a contiguous CUDA tensor of dtype {dt}")
    nRp, nRe, nw, _, nm = gW.shape
    nb1 = Uk.shape[1]
    if tuple(Re.shape) != (nRe, 3) or Uk.shape[0] != nw or tuple(g1_out.shape) != (nRp, nb1, nw, nm):
        raise ValueError("set_k_noalloc: inconsistent shapes")
    k_arr = np.ascontiguousarray(k, dtype=np.float64)
    if k_arr.shape != (3,):
        raise ValueError("set_k_noalloc: k must be three numbers")
    s = stream if stream is not None else torch.cuda.current_stream().cuda_stream
    rc = lib.phoebe_elph_set_k_noalloc(gW.data_ptr(), Re.data_ptr(), deg_e.data_ptr() if deg_e is not None else None, nRe, nRp,
                                       nw, nm, nb1, k_arr.ctypes.data, Uk.data_ptr(), g1_out.data_ptr(), s)
    if rc:
        raise PhoebeElphError(rc, "phoebe_elph_set_k_noalloc", lib.phoebe_elph_noalloc_last_error().decode())


def workspace_bytes(dims: Dims, hbm_budget_bytes: int):
    """-> (bytes, nq_batch).  Raises PhoebeElphError."""
    nbytes, nqb = c_size_t(0), c_int32(0)
    rc = load_library().phoebe_elph_workspace_bytes(byref(dims), hbm_budget_bytes, byref(nbytes), byref(nqb))
    if rc:
        raise PhoebeElphError(rc, "phoebe_elph_workspace_bytes")
    return int(nbytes.value), int(nqb.value)


def _chk_host(**arrays):
    """The host entry points read raw memory: every array must be C-contiguous with the dtype the C ABI expects
    (complex128 for Ukq / ev, float64 otherwise)."""
    import numpy as np
    for name, a in arrays.items():
        if a is None:
            continue
        want = np.complex128 if name in ("Ukq", "ev") else np.float64
        if a.dtype != want or not a.flags.c_contiguous:
            raise TypeError(f"{name}: expected a C-contiguous {np.dtype(want).name} array, got {a.dtype}"
                            f"{'' if a.flags.c_contiguous else ' (not contiguous)'}")


def _host_ptr(a):
    """pointer of a C-contiguous numpy array (or None)."""
    if a is None:
        return None
    assert a.flags.c_contiguous
    return a.ctypes.data


class ElphContext:
    """phoebe_elph_ctx with the same method names as the C ABI (set_k, q_batch, ...).

    ``gW`` is a CUDA torch tensor (complex128 [nRp][nRe][nw][nw][nm]) that is
    BORROWED; the workspace is allocated here with torch and kept alive with the
    context.  Array arguments of the device entry points are CUDA torch tensors,
    those of the ``*_host`` entry points are NumPy arrays (or pinned CPU tensors).
    """

    def __init__(self, gW, Re, Rp, deg_e=None, deg_p=None, *, nb1_max=None, nb2_max=None, nq_max, nk_max=0,
                 hbm_budget_bytes=None, stream=None, poison_workspace=False):
        import numpy as np
        import torch

        self._lib = load_library()
        if not torch.cuda.is_available():
            raise PhoebeElphError(-6, "ElphContext", "no CUDA device (there is no CPU fallback)")
        assert gW.is_cuda and gW.dtype == torch.complex128 and gW.is_contiguous() and gW.dim() == 5
        nRp, nRe, nw, nw2, nm = gW.shape
        assert nw == nw2
        self.dims = Dims(nRe, nRp, nw, nm, nb1_max or nw, nb2_max or nw, nq_max, nk_max)
        self._gW = gW
        self._torch = torch
        self.device = gW.device
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        if hbm_budget_bytes is None:
            free, _total = torch.cuda.mem_get_info(self.device)
            hbm_budget_bytes = int(free * 0.9)
        nbytes, nqb = workspace_bytes(self.dims, hbm_budget_bytes)
        if nqb < nq_max:
            import warnings
            warnings.warn(f"workspace budget {hbm_budget_bytes} B fits only {nqb} of the requested {nq_max} q-points per "
                          "batch: dims.nq_max lowered, larger q_batch calls will fail with E_DIMS", RuntimeWarning)
            self.dims.nq_max = nqb
        self.nq_batch = nqb
        self.workspace_nbytes = nbytes
        self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        if poison_workspace:      # test aid: every double of the workspace starts as a NaN (tests/test_gpu_guards.py)
            self._ws.fill_(0xFF)
        ws_ptr = (self._ws.data_ptr() + 255) // 256 * 256
        Re = np.ascontiguousarray(Re, dtype=np.float64); Rp = np.ascontiguousarray(Rp, dtype=np.float64)
        assert Re.shape == (nRe, 3) and Rp.shape == (nRp, 3)
        deg_e = None if deg_e is None else np.ascontiguousarray(deg_e, dtype=np.float64)
        deg_p = None if deg_p is None else np.ascontiguousarray(deg_p, dtype=np.float64)
        ctx = c_void_p(0)
        rc = self._lib.phoebe_elph_setup(byref(ctx), gW.data_ptr(), _host_ptr(Re), _host_ptr(Rp), _host_ptr(deg_e),
                                         _host_ptr(deg_p), byref(self.dims), ws_ptr, nbytes, self.stream.cuda_stream)
        if rc:
            raise PhoebeElphError(rc, "phoebe_elph_setup")
        self._ctx = ctx
        self.nb1 = 0

    # -- helpers -----------------------------------------------------------
    def _check(self, rc, where):
        if rc:
            raise PhoebeElphError(rc, where, self._lib.phoebe_elph_last_error(self._ctx).decode())

    def close(self):
        if getattr(self, "_ctx", None):
            self._lib.phoebe_elph_destroy(self._ctx)
            self._ctx = None

    def __del__(self):  # pragma: no cover
        try:
            self.close()
        except Exception:
            pass

    # -- the C ABI, same names ----------------------------------------------
    def set_k(self, k, Uk):
        """k: 3 floats (host); Uk: CUDA complex128 tensor [nw][nb1]."""
        import numpy as np
        k = np.ascontiguousarray(k, dtype=np.float64)
        assert k.shape == (3,) and Uk.is_cuda and Uk.is_contiguous() and Uk.dim() == 2
        nb1 = Uk.shape[1]
        self._check(self._lib.phoebe_elph_set_k(self._ctx, k.ctypes.data, Uk.data_ptr(), nb1), "phoebe_elph_set_k")
        self.nb1 = nb1

    def set_k_host(self, k, Uk):
        import numpy as np
        k = np.ascontiguousarray(k, dtype=np.float64)
        Uk = np.ascontiguousarray(Uk, dtype=np.complex128)
        nb1 = Uk.shape[1]
        self._check(self._lib.phoebe_elph_set_k_host(self._ctx, k.ctypes.data, Uk.ctypes.data, nb1),
                    "phoebe_elph_set_k_host")
        self.nb1 = nb1

    def set_k_batch(self, k, Uk):
        """k: [nk][3] floats (host); Uk: CUDA complex128 tensor [nk][nw][nb1].  One pass over g_W."""
        import numpy as np
        k = np.ascontiguousarray(k, dtype=np.float64)
        assert k.ndim == 2 and k.shape[1] == 3 and Uk.is_cuda and Uk.is_contiguous() and Uk.dim() == 3
        assert Uk.shape[0] == k.shape[0]
        nb1 = Uk.shape[2]
        self._check(self._lib.phoebe_elph_set_k_batch(self._ctx, k.shape[0], k.ctypes.data, Uk.data_ptr(), nb1),
                    "phoebe_elph_set_k_batch")
        self.nb1 = nb1

    def set_k_batch_host(self, k, Uk):
        import numpy as np
        k = np.ascontiguousarray(k, dtype=np.float64)
        Uk = np.ascontiguousarray(Uk, dtype=np.complex128)
        assert k.ndim == 2 and k.shape[1] == 3 and Uk.ndim == 3 and Uk.shape[0] == k.shape[0]
        nb1 = Uk.shape[2]
        self._check(self._lib.phoebe_elph_set_k_batch_host(self._ctx, k.shape[0], k.ctypes.data, Uk.ctypes.data, nb1),
                    "phoebe_elph_set_k_batch_host")
        self.nb1 = nb1

    def select_k(self, i: int):
        self._check(self._lib.phoebe_elph_select_k(self._ctx, int(i)), "phoebe_elph_select_k")

    def q_batch(self, q, Ukq, ev, omega, out=None):
        """All CUDA tensors: q [nq][3] f64, Ukq [nq][nw][nb2] c128, ev [nq][nm][nm] c128, omega [nq][nm] f64.
        Returns out [nq][nb1][nb2][nm] f64 (CUDA)."""
        torch = self._torch
        nq, nw, nb2 = Ukq.shape
        nm = self.dims.nmodes
        for t in (q, Ukq, ev, omega):
            assert t.is_cuda and t.is_contiguous()
        assert q.shape == (nq, 3) and ev.shape == (nq, nm, nm) and omega.shape == (nq, nm)
        if out is None:
            out = torch.empty((nq, self.nb1, nb2, nm), dtype=torch.float64, device=self.device)
        else:
            assert out.is_cuda and out.is_contiguous() and out.numel() == nq * self.nb1 * nb2 * nm
        self._check(self._lib.phoebe_elph_q_batch(self._ctx, nq, nb2, q.data_ptr(), Ukq.data_ptr(), ev.data_ptr(),
                                                  omega.data_ptr(), out.data_ptr()), "phoebe_elph_q_batch")
        return out

    def q_batch_multi(self, q, Ukq, ev, omega, out=None):
        """q_batch for the first nk k slots of the last set_k_batch in one pass.  CUDA tensors stacked over k:
        q [nk][nq][3], Ukq [nk][nq][nw][nb2], ev [nk][nq][nm][nm], omega [nk][nq][nm] -> out [nk][nq][nb1][nb2][nm]."""
        torch = self._torch
        nk, nq, nw, nb2 = Ukq.shape
        nm = self.dims.nmodes
        for t in (q, Ukq, ev, omega):
            assert t.is_cuda and t.is_contiguous()
        assert q.shape == (nk, nq, 3) and ev.shape == (nk, nq, nm, nm) and omega.shape == (nk, nq, nm)
        if out is None:
            out = torch.empty((nk, nq, self.nb1, nb2, nm), dtype=torch.float64, device=self.device)
        else:
            assert out.is_cuda and out.is_contiguous() and out.numel() == nk * nq * self.nb1 * nb2 * nm
        self._check(self._lib.phoebe_elph_q_batch_multi(self._ctx, nk, nq, nb2, q.data_ptr(), Ukq.data_ptr(),
                                                        ev.data_ptr(), omega.data_ptr(), out.data_ptr()),
                    "phoebe_elph_q_batch_multi")
        return out

    def q_batch_host(self, q, Ukq, ev, omega, out):
        """NumPy arrays (or pinned CPU tensors via .numpy()); synchronises before returning."""
        _chk_host(q=q, Ukq=Ukq, ev=ev, omega=omega, out=out)
        nq, nw, nb2 = Ukq.shape
        self._check(self._lib.phoebe_elph_q_batch_host(self._ctx, nq, nb2, q.ctypes.data, Ukq.ctypes.data,
                                                       ev.ctypes.data, omega.ctypes.data, out.ctypes.data),
                    "phoebe_elph_q_batch_host")
        return out

    def q_batch_host_async(self, q, Ukq, ev, omega, out):
        """Pipelined q_batch_host: NumPy views of PINNED memory; returns at once -- call wait() before reading out."""
        _chk_host(q=q, Ukq=Ukq, ev=ev, omega=omega, out=out)
        nq, nw, nb2 = Ukq.shape
        self._check(self._lib.phoebe_elph_q_batch_host_async(self._ctx, nq, nb2, q.ctypes.data, Ukq.ctypes.data,
                                                             ev.ctypes.data, omega.ctypes.data, out.ctypes.data),
                    "phoebe_elph_q_batch_host_async")
        return out

    def q_batch_multi_host_async(self, q, Ukq, ev, omega, out):
        """Pipelined q_batch_multi over PINNED host arrays stacked over k (q [nk][nq][3], ...); call wait() before
        reading out [nk][nq][nb1][nb2][nm]."""
        _chk_host(q=q, Ukq=Ukq, ev=ev, omega=omega, out=out)
        nk, nq, nw, nb2 = Ukq.shape
        self._check(self._lib.phoebe_elph_q_batch_multi_host_async(self._ctx, nk, nq, nb2, q.ctypes.data, Ukq.ctypes.data,
                                                                   ev.ctypes.data, omega.ctypes.data, out.ctypes.data),
                    "phoebe_elph_q_batch_multi_host_async")
        return out

    def q_batch_rates_multi_host_async(self, q, Ukq, ev, omega, eps_k, eps_kq, rate, *, kT, mu, sigma, pref, out=None):
        """Pipelined q_batch_rates_multi over PINNED host arrays stacked over k; rate [nk][nb1] is accumulated into;
        call wait() before reading rate / out."""
        _chk_host(q=q, Ukq=Ukq, ev=ev, omega=omega, eps_k=eps_k, eps_kq=eps_kq, rate=rate, out=out)
        nk, nq, nw, nb2 = Ukq.shape
        prm = RateParams(kT, mu, sigma, pref)
        self._check(self._lib.phoebe_elph_q_batch_rates_multi_host_async(
            self._ctx, nk, nq, nb2, q.ctypes.data, Ukq.ctypes.data, ev.ctypes.data, omega.ctypes.data, eps_k.ctypes.data,
            eps_kq.ctypes.data, byref(prm), rate.ctypes.data, None if out is None else out.ctypes.data),
            "phoebe_elph_q_batch_rates_multi_host_async")
        return rate, out

    def wait(self):
        self._check(self._lib.phoebe_elph_wait(self._ctx), "phoebe_elph_wait")

    def q_batch_rates(self, q, Ukq, ev, omega, eps_k, eps_kq, rate, *, kT, mu, sigma, pref, out=None, store_out=False):
        """q_batch with the linewidth sum of Eq. 29 fused in.  All CUDA tensors; eps_k [nb1],
        eps_kq [nq][nb2], rate [nb1] f64 is ACCUMULATED INTO.  |g|^2 is stored only if `out` is given or
        store_out=True.  Returns (rate, out-or-None)."""
        torch = self._torch
        nq, nw, nb2 = Ukq.shape
        nm = self.dims.nmodes
        for t in (q, Ukq, ev, omega, eps_k, eps_kq, rate):
            assert t.is_cuda and t.is_contiguous()
        assert q.shape == (nq, 3) and ev.shape == (nq, nm, nm) and omega.shape == (nq, nm)
        assert eps_k.shape == (self.nb1,) and eps_kq.shape == (nq, nb2) and rate.shape == (self.nb1,)
        assert eps_k.dtype == eps_kq.dtype == rate.dtype == torch.float64
        if out is None and store_out:
            out = torch.empty((nq, self.nb1, nb2, nm), dtype=torch.float64, device=self.device)
        prm = RateParams(kT, mu, sigma, pref)
        self._check(self._lib.phoebe_elph_q_batch_rates(
            self._ctx, nq, nb2, q.data_ptr(), Ukq.data_ptr(), ev.data_ptr(), omega.data_ptr(), eps_k.data_ptr(),
            eps_kq.data_ptr(), byref(prm), rate.data_ptr(), None if out is None else out.data_ptr()),
            "phoebe_elph_q_batch_rates")
        return rate, out

    def q_batch_rates_multi(self, q, Ukq, ev, omega, eps_k, eps_kq, rate, *, kT, mu, sigma, pref, out=None, store_out=False):
        """q_batch_rates for the first nk k slots of the last set_k_batch in one pass.  CUDA tensors stacked over k:
        q [nk][nq][3], Ukq [nk][nq][nw][nb2], ev [nk][nq][nm][nm], omega [nk][nq][nm], eps_k [nk][nb1], eps_kq [nk][nq][nb2],
        rate [nk][nb1] (ACCUMULATED INTO).  Returns (rate, out-or-None)."""
        torch = self._torch
        nk, nq, nw, nb2 = Ukq.shape
        nm = self.dims.nmodes
        for t in (q, Ukq, ev, omega, eps_k, eps_kq, rate):
            assert t.is_cuda and t.is_contiguous()
        assert q.shape == (nk, nq, 3) and ev.shape == (nk, nq, nm, nm) and omega.shape == (nk, nq, nm)
        assert eps_k.shape == (nk, self.nb1) and eps_kq.shape == (nk, nq, nb2) and rate.shape == (nk, self.nb1)
        assert eps_k.dtype == eps_kq.dtype == rate.dtype == torch.float64
        if out is None and store_out:
            out = torch.empty((nk, nq, self.nb1, nb2, nm), dtype=torch.float64, device=self.device)
        prm = RateParams(kT, mu, sigma, pref)
        self._check(self._lib.phoebe_elph_q_batch_rates_multi(
            self._ctx, nk, nq, nb2, q.data_ptr(), Ukq.data_ptr(), ev.data_ptr(), omega.data_ptr(), eps_k.data_ptr(),
            eps_kq.data_ptr(), byref(prm), rate.data_ptr(), None if out is None else out.data_ptr()),
            "phoebe_elph_q_batch_rates_multi")
        return rate, out

    def q_batch_rates_host(self, q, Ukq, ev, omega, eps_k, eps_kq, rate, *, kT, mu, sigma, pref, out=None):
        """NumPy arrays; rate [nb1] is accumulated into in place; synchronises before returning."""
        _chk_host(q=q, Ukq=Ukq, ev=ev, omega=omega, eps_k=eps_k, eps_kq=eps_kq, rate=rate, out=out)
        nq, nw, nb2 = Ukq.shape
        prm = RateParams(kT, mu, sigma, pref)
        self._check(self._lib.phoebe_elph_q_batch_rates_host(
            self._ctx, nq, nb2, q.ctypes.data, Ukq.ctypes.data, ev.ctypes.data, omega.ctypes.data, eps_k.ctypes.data,
            eps_kq.ctypes.data, byref(prm), rate.ctypes.data, None if out is None else out.ctypes.data),
            "phoebe_elph_q_batch_rates_host")
        return rate, out

    def q_batch_rates_host_async(self, q, Ukq, ev, omega, eps_k, eps_kq, rate, *, kT, mu, sigma, pref, out=None):
        """Pipelined q_batch_rates_host (NumPy views of PINNED memory; one rate array per call in flight); returns at
        once -- call wait() before reading rate / out."""
        _chk_host(q=q, Ukq=Ukq, ev=ev, omega=omega, eps_k=eps_k, eps_kq=eps_kq, rate=rate, out=out)
        nq, nw, nb2 = Ukq.shape
        prm = RateParams(kT, mu, sigma, pref)
        self._check(self._lib.phoebe_elph_q_batch_rates_host_async(
            self._ctx, nq, nb2, q.ctypes.data, Ukq.ctypes.data, ev.ctypes.data, omega.ctypes.data, eps_k.ctypes.data,
            eps_kq.ctypes.data, byref(prm), rate.ctypes.data, None if out is None else out.ctypes.data),
            "phoebe_elph_q_batch_rates_host_async")
        return rate, out

    def copy_g1(self):
        torch = self._torch
        d = self.dims
        g1 = torch.empty((d.nRp, self.nb1, d.nw, d.nmodes), dtype=torch.complex128, device=self.device)
        self._check(self._lib.phoebe_elph_copy_g1(self._ctx, g1.data_ptr(), g1.numel() * 16), "phoebe_elph_copy_g1")
        return g1

    def set_polar(self, recip=None, G=None, Zstar=None, eps_inf=None, coeff=0.0):
        """Switch the polar long-range term (Eq. 14-15) on (NumPy arrays: recip [3][3], G [nG][3] crystal coords,
        Zstar [nm/3][3][3], eps_inf [3][3]) or, with G=None, off."""
        import numpy as np
        if G is None:
            self._check(self._lib.phoebe_elph_set_polar(self._ctx, None, 0, None, None, None, 0.0), "phoebe_elph_set_polar")
            return
        recip, G, Zstar, eps_inf = [np.ascontiguousarray(a, dtype=np.float64) for a in (recip, G, Zstar, eps_inf)]
        assert recip.shape == (3, 3) and eps_inf.shape == (3, 3) and G.ndim == 2 and G.shape[1] == 3
        assert Zstar.shape == (self.dims.nmodes // 3, 3, 3)
        self._check(self._lib.phoebe_elph_set_polar(self._ctx, recip.ctypes.data, len(G), G.ctypes.data, Zstar.ctypes.data,
                                                    eps_inf.ctypes.data, float(coeff)), "phoebe_elph_set_polar")

    def set_conventions(self, phase_sign=1, conj_Uk=False, conj_Ukq=True, conj_ev=False):
        """Sign of the Fourier phases and conjugation of the three rotation matrices of Eq. 70 (defaults: el-ph,
        Eq. 13; three-phonon coupling of Eq. 5: phase_sign=-1, all three conjugated)."""
        self._check(self._lib.phoebe_elph_set_conventions(self._ctx, int(phase_sign), int(bool(conj_Uk)),
                                                          int(bool(conj_Ukq)), int(bool(conj_ev))),
                    "phoebe_elph_set_conventions")

    def g1_view(self, slot: int = -1):
        """float64 view (no copy) of the g1' storage inside the workspace: slot >= 0 -> that k slot's
        [nRp][nb1][nw][nm][2]; slot = -1 -> every filled slot as one flat range (for an in-place all_reduce of the
        Re-pool)."""
        ptr, nbytes, stride = c_void_p(0), c_size_t(0), c_size_t(0)
        self._check(self._lib.phoebe_elph_g1_buffer(self._ctx, int(slot), byref(ptr), byref(nbytes), byref(stride)),
                    "phoebe_elph_g1_buffer")
        off = ptr.value - self._ws.data_ptr()
        assert 0 <= off and off + nbytes.value <= self._ws.numel()
        flat = self._ws[off:off + nbytes.value].view(self._torch.float64)
        if slot >= 0:
            d = self.dims
            return flat.view(d.nRp, self.nb1, d.nw, d.nmodes, 2)
        return flat

    def launch_counts(self):
        arr = (c_int64 * len(KERNEL_KINDS))()
        self._check(self._lib.phoebe_elph_launch_counts(self._ctx, arr), "phoebe_elph_launch_counts")
        return dict(zip(KERNEL_KINDS, [int(x) for x in arr]))

    def profile(self, enable: bool):
        self._check(self._lib.phoebe_elph_profile(self._ctx, 1 if enable else 0), "phoebe_elph_profile")

    def profile_read(self):
        """-> {kind: (ms, launches)} since the last read."""
        ms = (c_double * len(KERNEL_KINDS))()
        n = (c_int64 * len(KERNEL_KINDS))()
        self._check(self._lib.phoebe_elph_profile_read(self._ctx, ms, n), "phoebe_elph_profile_read")
        return {k: (float(ms[i]), int(n[i])) for i, k in enumerate(KERNEL_KINDS)}

    def set_tuning(self, key: str, value: int):
        self._check(self._lib.phoebe_elph_set_tuning(self._ctx, key.encode(), int(value)), "phoebe_elph_set_tuning")

    def get_tuning(self, key: str) -> int:
        v = c_int64(0)
        self._check(self._lib.phoebe_elph_get_tuning(self._ctx, key.encode(), byref(v)), "phoebe_elph_get_tuning")
        return int(v.value)


#: every symbol declared in include/phoebe_elph_probes.h (libphoebe_elph_probes.so: measurement aids, not the product)
PROBE_EXPORTS = ["phoebe_elph_probe_fp64", "phoebe_elph_probe_hbm_read"]
PROBES_LIB_PATH = os.path.join(HERE, "libphoebe_elph_probes.so")
_probes = None


def load_probes() -> ctypes.CDLL:
    global _probes
    if _probes is None:
        if not os.path.exists(PROBES_LIB_PATH):
            raise FileNotFoundError(f"{PROBES_LIB_PATH} not built; run `python -m paper_2111_14999_b200.build`")
        lib = ctypes.CDLL(PROBES_LIB_PATH)
        lib.phoebe_elph_probe_fp64.argtypes = [c_int32, c_int32, c_void_p, POINTER(c_double)]
        lib.phoebe_elph_probe_hbm_read.argtypes = [c_void_p, c_size_t, c_void_p, POINTER(c_double)]
        _probes = lib
    return _probes


def probe_fp64(kind: str = "dmma", iters: int = 20000, stream=None) -> float:
    """FP64 ceiling in TFLOP/s measured on this device (kind: 'dfma' | 'dmma')."""
    t = c_double(0.0)
    st = None if stream is None else stream.cuda_stream
    rc = load_probes().phoebe_elph_probe_fp64({"dfma": 0, "dmma": 1}[kind], iters, st, byref(t))
    if rc:
        raise PhoebeElphError(rc, "phoebe_elph_probe_fp64")
    return float(t.value)


def probe_hbm_read(buf, stream=None) -> float:
    """HBM read-stream bandwidth in GB/s over a CUDA tensor."""
    t = c_double(0.0)
    st = None if stream is None else stream.cuda_stream
    rc = load_probes().phoebe_elph_probe_hbm_read(buf.data_ptr(), buf.numel() * buf.element_size(), st, byref(t))
    if rc:
        raise PhoebeElphError(rc, "phoebe_elph_probe_hbm_read")
    return float(t.value)
