"""Thin ctypes binding of include/snk.h (argument marshalling only -- every step of the path runs in the
CUDA kernels of libsnk.so).  Same names as the C ABI.  PyTorch appears only as the owner of device memory
and streams.  There is NO CPU fallback: ``load()`` raises if the library is missing or does not export a symbol.

Never imports ``oracle/``.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsnk.so")
HEADER_PATH = os.path.join(os.path.dirname(_HERE), "include", "snk.h")

SNK_OK, SNK_EINVAL, SNK_ENOMEM, SNK_ECUDA, SNK_ESTATE = 0, -1, -2, -3, -4

EXPORTS = ["snk_create", "snk_set_option", "snk_set_grid", "snk_build_K", "snk_build_K_host", "snk_screen", "snk_batch_costs", "snk_nbf", "snk_get_stats",
           "snk_export_lists", "snk_debug_boys", "snk_debug_A_pair", "snk_A_pair_noalloc", "snk_measure_fp64_peak", "snk_last_error", "snk_destroy",
           "snk_version"]

CLASS_NAMES = ["ss", "ps", "pp", "ds", "dp", "dd", "fs", "fp", "fd", "ff"]


class SnkStats(C.Structure):
    _fields_ = [("npts", C.c_int64), ("npts_kept", C.c_int64), ("nbatch", C.c_int64), ("sum_B", C.c_int64), ("sum_B_fn", C.c_int64),
                ("npair_sig", C.c_int64), ("sum_V", C.c_int64), ("nprimpair", C.c_int64), ("nsuper", C.c_int64),
                ("n_pairpoints", C.c_double), ("n_int_contracted", C.c_double), ("n_int_primitive", C.c_double),
                ("flops_integral", C.c_double), ("flops_gemm", C.c_double), ("ms_set_grid", C.c_double), ("ms_screen", C.c_double),
                ("ms_colloc", C.c_double), ("ms_F", C.c_double), ("ms_G", C.c_double), ("ms_Kt", C.c_double), ("ms_sym", C.c_double),
                ("ms_build", C.c_double), ("ms_G_class", C.c_double * 10), ("n_int_class", C.c_double * 10),
                ("flops_class", C.c_double * 10), ("n_launches", C.c_int64), ("flops_gemm_alg", C.c_double)]

    def asdict(self):
        d = {}
        for name, _ in self._fields_:
            v = getattr(self, name)
            d[name] = list(v) if hasattr(v, "__len__") else v
        return d


class SnkError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("snk error %d: %s" % (code, msg))
        self.code = code


_lib = None


def load():
    """dlopen libsnk.so; fail loudly when it is missing (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libsnk.so not built: run `python -m paper_2303_14280_b200.build` (there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    for name in EXPORTS:
        if not hasattr(lib, name):
            raise ImportError("libsnk.so does not export %s" % name)
    vp, dp, ip, lp = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_int64)
    lib.snk_create.argtypes = [C.POINTER(vp), C.c_int32, dp, C.c_int32, ip, ip, ip, dp, dp]
    lib.snk_set_option.argtypes = [vp, C.c_char_p, C.c_double]
    lib.snk_set_grid.argtypes = [vp, C.c_int64, vp, vp, vp]
    lib.snk_build_K.argtypes = [vp, vp, vp, vp]
    lib.snk_build_K_host.argtypes = [vp, vp, vp, vp]
    lib.snk_screen.argtypes = [vp, vp, vp]
    lib.snk_batch_costs.argtypes = [vp, dp]
    lib.snk_nbf.argtypes = [vp]
    lib.snk_get_stats.argtypes = [vp, C.POINTER(SnkStats)]
    lib.snk_export_lists.argtypes = [vp, lp, lp, lp, lp, ip, lp, ip]
    lib.snk_debug_boys.argtypes = [C.c_int32, C.c_int64, vp, vp, vp]
    lib.snk_debug_A_pair.argtypes = [vp, C.c_int32, C.c_int32, C.c_int64, vp, vp, vp]
    lib.snk_A_pair_noalloc.argtypes = [vp, C.c_int32, C.c_int32, C.c_int64, vp, vp, vp]
    lib.snk_measure_fp64_peak.argtypes = [dp, dp, C.c_int32]
    lib.snk_last_error.argtypes = [vp]
    lib.snk_last_error.restype = C.c_char_p
    lib.snk_destroy.argtypes = [vp]
    lib.snk_destroy.restype = None
    lib.snk_version.restype = C.c_char_p
    _lib = lib
    return lib


def _np(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def _ptr(t):
    """device pointer of a torch tensor (or a raw int)"""
    return C.c_void_p(int(t) if isinstance(t, int) else t.data_ptr())


def _stream(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    return C.c_void_p(int(stream) if isinstance(stream, int) else stream.cuda_stream)


class Snk:
    """One basis set on one GPU.  Methods mirror the C ABI one to one."""

    def __init__(self, basis):
        lib = load()
        self._lib = lib
        self.h = C.c_void_p()
        xyz = _np(basis.atom_xyz, np.float64)
        sa, sl, sn = _np(basis.shell_atom, np.int32), _np(basis.shell_l, np.int32), _np(basis.shell_nprim, np.int32)
        pe, pc = _np(basis.prim_exp, np.float64), _np(basis.prim_coef, np.float64)
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int32)
        rc = lib.snk_create(C.byref(self.h), int(xyz.shape[0]), xyz.ctypes.data_as(dp), int(sl.shape[0]), sa.ctypes.data_as(ip),
                            sl.ctypes.data_as(ip), sn.ctypes.data_as(ip), pe.ctypes.data_as(dp), pc.ctypes.data_as(dp))
        if rc != SNK_OK:
            raise SnkError(rc, (lib.snk_last_error(None) or b"").decode())
        self.nbf = lib.snk_nbf(self.h)
        self.nsh = int(sl.shape[0])
        self._sl = [int(l) for l in sl]

    def _check(self, rc):
        if rc != SNK_OK:
            raise SnkError(rc, (self._lib.snk_last_error(self.h) or b"").decode())

    def close(self):
        if getattr(self, "h", None) and self.h.value:
            self._lib.snk_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, key: str, value: float):
        self._check(self._lib.snk_set_option(self.h, key.encode(), float(value)))

    def set_grid(self, points, weights, stream=None):
        """points: CUDA float64 tensor [npts,3] contiguous; weights: CUDA float64 [npts]."""
        assert points.is_cuda and weights.is_cuda and points.is_contiguous() and weights.is_contiguous()
        assert points.dtype.is_floating_point and points.element_size() == 8 and weights.element_size() == 8
        n = int(weights.shape[0])
        assert points.numel() == 3 * n
        self._check(self._lib.snk_set_grid(self.h, n, _ptr(points), _ptr(weights), _stream(stream)))

    def build_K(self, P, K=None, stream=None):
        """P: CUDA float64 [nbf,nbf]; returns K (CUDA float64 [nbf,nbf]); asynchronous on the stream."""
        import torch
        assert P.is_cuda and P.is_contiguous() and P.element_size() == 8 and tuple(P.shape) == (self.nbf, self.nbf)
        if K is None:
            K = torch.empty_like(P)
        assert K.is_cuda and K.is_contiguous() and tuple(K.shape) == (self.nbf, self.nbf)
        self._check(self._lib.snk_build_K(self.h, _ptr(P), _ptr(K), _stream(stream)))
        return K

    def screen(self, P, stream=None):
        """Row a3 only (V_j for this P); then batch_costs()."""
        assert P.is_cuda and P.is_contiguous() and P.element_size() == 8 and tuple(P.shape) == (self.nbf, self.nbf)
        self._check(self._lib.snk_screen(self.h, _ptr(P), _stream(stream)))

    def batch_costs(self) -> np.ndarray:
        """Primitive pair-points per batch (batch order) after screen() or build_K()."""
        nb = int(self.stats()["nbatch"])
        out = np.zeros(max(nb, 1), dtype=np.float64)
        self._check(self._lib.snk_batch_costs(self.h, out.ctypes.data_as(C.POINTER(C.c_double))))
        return out[:nb]

    def build_K_host(self, P_host: np.ndarray, K_host: np.ndarray = None, stream=None):
        """End-to-end call with HOST buffers (numpy or pinned torch CPU tensors exposing data_ptr)."""
        if isinstance(P_host, np.ndarray):
            assert P_host.dtype == np.float64 and P_host.flags.c_contiguous and P_host.shape == (self.nbf, self.nbf)
            if K_host is None:
                K_host = np.empty_like(P_host)
            pp, kp = C.c_void_p(P_host.ctypes.data), C.c_void_p(K_host.ctypes.data)
        else:
            import torch
            assert not P_host.is_cuda and P_host.is_contiguous()
            if K_host is None:
                K_host = torch.empty_like(P_host, pin_memory=True)
            pp, kp = C.c_void_p(P_host.data_ptr()), C.c_void_p(K_host.data_ptr())
        self._check(self._lib.snk_build_K_host(self.h, pp, kp, _stream(stream)))
        return K_host

    def stats(self) -> dict:
        st = SnkStats()
        self._check(self._lib.snk_get_stats(self.h, C.byref(st)))
        return st.asdict()

    def export_lists(self, want_V=True):
        lp, ip = C.POINTER(C.c_int64), C.POINTER(C.c_int32)
        sizes = np.zeros(4, dtype=np.int64)
        self._check(self._lib.snk_export_lists(self.h, sizes.ctypes.data_as(lp), None, None, None, None, None, None))
        nb, nk, sB, sV = (int(x) for x in sizes)
        boff = np.zeros(nb + 1, dtype=np.int64); perm = np.zeros(max(nk, 1), dtype=np.int64)
        Boff = np.zeros(nb + 1, dtype=np.int64); Bids = np.zeros(max(sB, 1), dtype=np.int32)
        Voff = np.zeros(nb + 1, dtype=np.int64); Vp = np.zeros((max(sV, 1), 2), dtype=np.int32)
        self._check(self._lib.snk_export_lists(self.h, sizes.ctypes.data_as(lp), boff.ctypes.data_as(lp), perm.ctypes.data_as(lp),
                                               Boff.ctypes.data_as(lp), Bids.ctypes.data_as(ip),
                                               Voff.ctypes.data_as(lp) if want_V and sV else None,
                                               Vp.ctypes.data_as(ip) if want_V and sV else None))
        return dict(batch_off=boff, perm=perm[:nk], B_off=Boff, B_ids=Bids[:sB], V_off=Voff, V_pairs=Vp[:sV])

    def debug_A_pair(self, a: int, b: int, pts, stream=None):
        import torch
        assert pts.is_cuda and pts.is_contiguous() and pts.element_size() == 8
        n = pts.shape[0]
        out = torch.empty((n, self._nc(a), self._nc(b)), dtype=torch.float64, device=pts.device)
        self._check(self._lib.snk_debug_A_pair(self.h, int(a), int(b), int(n), _ptr(pts), _ptr(out), _stream(stream)))
        return out

    def A_pair_noalloc(self, a: int, b: int, pts, out, stream=None):
        """snk_A_pair_noalloc: like debug_A_pair, but the caller passes ``out`` (CUDA float64 [n, ncart(l_a), ncart(l_b)]) and
        the library allocates nothing; asynchronous on the stream."""
        assert pts.is_cuda and pts.is_contiguous() and pts.element_size() == 8
        n = pts.shape[0]
        assert out.is_cuda and out.is_contiguous() and out.element_size() == 8 and out.numel() == n * self._nc(a) * self._nc(b)
        self._check(self._lib.snk_A_pair_noalloc(self.h, int(a), int(b), int(n), _ptr(pts), _ptr(out), _stream(stream)))
        return out

    def _nc(self, s):
        l = self._sl[s]
        return (l + 1) * (l + 2) // 2


def debug_boys(mmax: int, x, stream=None):
    """F_0..F_mmax through the device Boys routine; x: CUDA float64 tensor [n] -> [n, mmax+1]."""
    import torch
    lib = load()
    assert x.is_cuda and x.is_contiguous() and x.element_size() == 8
    out = torch.empty((x.shape[0], mmax + 1), dtype=torch.float64, device=x.device)
    rc = lib.snk_debug_boys(int(mmax), int(x.shape[0]), _ptr(x), _ptr(out), _stream(stream))
    if rc != SNK_OK:
        raise SnkError(rc, "snk_debug_boys")
    return out


def measure_fp64_peak(reps: int = 5):
    lib = load()
    a, b = C.c_double(), C.c_double()
    rc = lib.snk_measure_fp64_peak(C.byref(a), C.byref(b), int(reps))
    if rc != SNK_OK:
        raise SnkError(rc, "snk_measure_fp64_peak")
    return a.value, b.value


def version() -> str:
    return load().snk_version().decode()


def build_K(basis, points, weights, P, *, eps=0.0, batch_cell=6.0, batch_max=2048, workspace_gb=None, device="cuda:0", return_ctx=False):
    """Convenience: numpy inputs -> numpy K through the three C-ABI calls (create / set_grid / build_K)."""
    import torch
    dev = torch.device(device)
    with torch.cuda.device(dev):
        s = Snk(basis)
        s.set_option("eps", eps); s.set_option("batch_cell", batch_cell); s.set_option("batch_max", batch_max)
        if workspace_gb is not None:
            s.set_option("workspace_gb", workspace_gb)
        pts = torch.as_tensor(np.ascontiguousarray(points, dtype=np.float64).reshape(-1, 3), device=dev)
        w = torch.as_tensor(np.ascontiguousarray(weights, dtype=np.float64).reshape(-1), device=dev)
        Pd = torch.as_tensor(np.ascontiguousarray(P, dtype=np.float64), device=dev)
        s.set_grid(pts, w)
        K = s.build_K(Pd)
        torch.cuda.synchronize(dev)
        Kh = K.cpu().numpy()
    return (Kh, s) if return_ctx else Kh
