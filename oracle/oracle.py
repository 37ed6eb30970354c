"""ctypes wrapper around oracle/snk_oracle.cpp -- the CPU ORACLE.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It does not import, read or call anything of the CUDA path
(paper_2303_14280_b200/csrc, paper_2303_14280_b200/snk.py); the only module it shares with the
product is the input generator (paper_2303_14280_b200/inputs.py), whose Basis dataclass it accepts.

Every function cites the passage of /root/reference/PAPER.md it follows in snk_oracle.cpp.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "snk_oracle.cpp")
_LIB = os.path.join(_HERE, "libsnk_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """g++ -O2 -fopenmp (plain build, never tuned)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(build())
    dp, ip, lp = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_int64)
    lib.orc_boys.argtypes = [C.c_int, C.c_double, dp]
    lib.orc_create.restype = C.c_void_p
    lib.orc_create.argtypes = [C.c_int, dp, C.c_int, ip, ip, ip, dp, dp]
    lib.orc_destroy.argtypes = [C.c_void_p]
    lib.orc_nbf.argtypes = [C.c_void_p]
    lib.orc_A_pair.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int64, dp, dp]
    lib.orc_collocation.argtypes = [C.c_void_p, C.c_int64, dp, dp]
    lib.orc_A_bound.restype = C.c_double
    lib.orc_A_bound.argtypes = [C.c_void_p, C.c_int, C.c_int]
    lib.orc_rcut.restype = C.c_double
    lib.orc_rcut.argtypes = [C.c_void_p, C.c_int, C.c_double]
    lib.orc_set_grid.argtypes = [C.c_void_p, C.c_int64, dp, dp, C.c_double, C.c_double, C.c_int]
    lib.orc_nbatch.restype = C.c_int64
    lib.orc_nbatch.argtypes = [C.c_void_p]
    lib.orc_get_batches.argtypes = [C.c_void_p, lp, lp, dp]
    lib.orc_get_B.restype = C.c_int64
    lib.orc_get_B.argtypes = [C.c_void_p, lp, ip]
    lib.orc_get_V.restype = C.c_int64
    lib.orc_get_V.argtypes = [C.c_void_p, lp, ip]
    lib.orc_get_maxima.argtypes = [C.c_void_p, dp, dp]
    lib.orc_screen.argtypes = [C.c_void_p, dp]
    lib.orc_build_K.argtypes = [C.c_void_p, dp, dp, C.c_int, ip]
    lib.orc_get_stats.argtypes = [C.c_void_p, dp]
    lib.orc_set_extended.argtypes = [C.c_void_p, C.c_int]
    _lib = lib
    return lib


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _i(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


def _l(a):
    return a.ctypes.data_as(C.POINTER(C.c_int64))


def boys(mmax: int, x: float) -> np.ndarray:
    """F_0..F_mmax(x), Eq. 22."""
    out = np.zeros(mmax + 1)
    if _load().orc_boys(int(mmax), float(x), _d(out)) != 0:
        raise ValueError("orc_boys: bad argument")
    return out


class Oracle:
    """One basis (+ optionally one grid).  Mirrors the three calls of the product
    (create / set_grid / build_K) so tests can drive both with the same inputs."""

    def __init__(self, basis):
        lib = _load()
        self._keep = [np.ascontiguousarray(basis.atom_xyz, dtype=np.float64),
                      np.ascontiguousarray(basis.shell_atom, dtype=np.int32),
                      np.ascontiguousarray(basis.shell_l, dtype=np.int32),
                      np.ascontiguousarray(basis.shell_nprim, dtype=np.int32),
                      np.ascontiguousarray(basis.prim_exp, dtype=np.float64),
                      np.ascontiguousarray(basis.prim_coef, dtype=np.float64)]
        k = self._keep
        self.h = lib.orc_create(int(k[0].shape[0]), _d(k[0]), int(k[1].shape[0]), _i(k[1]), _i(k[2]), _i(k[3]), _d(k[4]), _d(k[5]))
        if not self.h:
            raise ValueError("orc_create: invalid basis")
        self.nbf = lib.orc_nbf(self.h)
        self.nsh = int(k[1].shape[0])
        self.shell_l = k[2]
        self._grid = False

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            _lib.orc_destroy(self.h)
            self.h = None

    # ---- pieces (pins) ----
    def A_pair(self, a: int, b: int, pts: np.ndarray) -> np.ndarray:
        """A[g, ia, ib] for shell pair (a,b) at points pts, Eq. 37."""
        pts = np.ascontiguousarray(pts, dtype=np.float64).reshape(-1, 3)
        na = (self.shell_l[a] + 1) * (self.shell_l[a] + 2) // 2
        nb = (self.shell_l[b] + 1) * (self.shell_l[b] + 2) // 2
        out = np.zeros((pts.shape[0], na, nb))
        if _lib.orc_A_pair(self.h, int(a), int(b), pts.shape[0], _d(pts), _d(out)) != 0:
            raise ValueError("orc_A_pair")
        return out

    def collocation(self, pts: np.ndarray) -> np.ndarray:
        """Phi[g, mu], Eq. 31."""
        pts = np.ascontiguousarray(pts, dtype=np.float64).reshape(-1, 3)
        out = np.zeros((pts.shape[0], self.nbf))
        _lib.orc_collocation(self.h, pts.shape[0], _d(pts), _d(out))
        return out

    def A_bound(self, a: int, b: int) -> float:
        return _lib.orc_A_bound(self.h, int(a), int(b))

    def rcut(self, a: int, eps: float) -> float:
        return _lib.orc_rcut(self.h, int(a), float(eps))

    # ---- the path ----
    def set_grid(self, points, weights, *, eps=0.0, batch_cell=6.0, batch_max=2048):
        pts = np.ascontiguousarray(points, dtype=np.float64).reshape(-1, 3)
        w = np.ascontiguousarray(weights, dtype=np.float64).reshape(-1)
        assert pts.shape[0] == w.shape[0]
        rc = _lib.orc_set_grid(self.h, pts.shape[0], _d(pts), _d(w), float(eps), float(batch_cell), int(batch_max))
        if rc != 0:
            raise ValueError("orc_set_grid: bad argument (negative weight?)")
        self._grid = True
        self.npts = pts.shape[0]

    def build_K(self, P, sel_shells=None, extended=False) -> np.ndarray:
        """Eqs. 31-40.  ``extended``: the sums over sigma, lambda and g in long double (same terms, same order): a
        rounding-order check of the fp64 result, not a different method."""
        assert self._grid
        _lib.orc_set_extended(self.h, 1 if extended else 0)
        P = np.ascontiguousarray(P, dtype=np.float64)
        assert P.shape == (self.nbf, self.nbf)
        K = np.zeros((self.nbf, self.nbf))
        if sel_shells is None:
            rc = _lib.orc_build_K(self.h, _d(P), _d(K), 0, None)
        else:
            s = np.ascontiguousarray(sel_shells, dtype=np.int32)
            rc = _lib.orc_build_K(self.h, _d(P), _d(K), int(s.shape[0]), _i(s))
        if rc != 0:
            raise ValueError("orc_build_K failed (%d): P not symmetric?" % rc)
        return K

    def screen(self, P):
        P = np.ascontiguousarray(P, dtype=np.float64)
        _lib.orc_screen(self.h, _d(P))

    def stats(self) -> dict:
        o = np.zeros(5)
        _lib.orc_get_stats(self.h, _d(o))
        return dict(n_int_contracted=o[0], n_int_primitive=o[1], n_pairpoints=o[2], seconds=o[3], threads=int(o[4]))

    # ---- lists (audit) ----
    def batches(self):
        nb = _lib.orc_nbatch(self.h)
        off = np.zeros(nb + 1, dtype=np.int64)
        perm = np.zeros(self.npts, dtype=np.int64)
        bbox = np.zeros((nb, 6))
        _lib.orc_get_batches(self.h, _l(off), _l(perm), _d(bbox))
        return off, perm[:off[-1]], bbox

    def B_lists(self):
        nb = _lib.orc_nbatch(self.h)
        off = np.zeros(nb + 1, dtype=np.int64)
        n = _lib.orc_get_B(self.h, _l(off), None)
        ids = np.zeros(max(n, 1), dtype=np.int32)
        _lib.orc_get_B(self.h, _l(off), _i(ids))
        return off, ids[:n]

    def V_lists(self):
        nb = _lib.orc_nbatch(self.h)
        off = np.zeros(nb + 1, dtype=np.int64)
        n = _lib.orc_get_V(self.h, _l(off), None)
        pairs = np.zeros((max(n, 1), 2), dtype=np.int32)
        _lib.orc_get_V(self.h, _l(off), _i(pairs))
        return off, pairs[:n]

    def maxima(self):
        nb = _lib.orc_nbatch(self.h)
        Pt = np.zeros((nb, self.nsh))
        pt = np.zeros(nb)
        _lib.orc_get_maxima(self.h, _d(Pt), _d(pt))
        return Pt, pt
