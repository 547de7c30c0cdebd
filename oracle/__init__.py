"""ctypes front-end of the CPU oracle (oracle/lqcd_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  Nothing here touches the CUDA path.  All arrays are numpy, fp64, in the paper's
public cb2 layouts.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liblqcd_oracle.so")
_SRC = os.path.join(_HERE, "lqcd_oracle.cpp")


def build(force=False):
    """g++ -O2 -fopenmp, no fast-math."""
    if not force and os.path.exists(_SO) and os.path.getmtime(_SO) >= os.path.getmtime(_SRC):
        return _SO
    subprocess.check_call(
        ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-o", _SO, _SRC])
    return _SO


class Result(ctypes.Structure):
    _fields_ = [("status", ctypes.c_int), ("iterations", ctypes.c_int),
                ("iter_resid", ctypes.c_double), ("true_resid", ctypes.c_double),
                ("seconds", ctypes.c_double), ("hops", ctypes.c_long)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_SO)
        vp, ci, cd, cl = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_long
        L.orc_threads.restype = ci
        L.orc_gamma.argtypes = [ci, vp]
        L.orc_sigma.argtypes = [ci, ci, vp]
        L.orc_create.restype = vp
        L.orc_create.argtypes = [ctypes.POINTER(ci), ci, vp]
        L.orc_destroy.argtypes = [vp]
        L.orc_set_clover.argtypes = [vp, cd, cd]
        L.orc_set_anisotropy.argtypes = [vp, cd]
        L.orc_set_clover_aniso.argtypes = [vp, cd, cd, cd]
        L.orc_clover_defect.restype = cd
        L.orc_clover_defect.argtypes = [vp]
        L.orc_get_clover.argtypes = [vp, vp, vp]
        L.orc_clover_dense.argtypes = [vp, cd, cd, vp]
        L.orc_fmunu.argtypes = [vp, ci, ci, vp]
        L.orc_dslash.argtypes = [vp, vp, vp, ci, ci]
        L.orc_dslash_site.argtypes = [vp, vp, cl, ci, vp]
        L.orc_clover_apply.argtypes = [vp, vp, vp, ci, ci]
        L.orc_mat.argtypes = [vp, vp, vp, ci]
        L.orc_mpc.argtypes = [vp, vp, vp, ci, ci]
        L.orc_invert.argtypes = [vp, vp, vp, cd, ci, ci, ci, ctypes.POINTER(Result)]
        L.orc_true_residual.restype = cd
        L.orc_true_residual.argtypes = [vp, vp, vp]
        _lib = L
    return _lib


def threads():
    return lib().orc_threads()


def gamma(mu):
    """mu = 0..3: gamma_x..gamma_t; 4: gamma_5.  4x4 complex128."""
    out = np.empty((4, 4), dtype=np.complex128)
    lib().orc_gamma(mu, out.ctypes.data)
    return out


def sigma(mu, nu):
    out = np.empty((4, 4), dtype=np.complex128)
    lib().orc_sigma(mu, nu, out.ctypes.data)
    return out


SOLVERS = {"cgne": 0, "cgnr": 1, "bicgstab": 2}


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a


class Oracle:
    """Holds links (and, after set_clover, A and A^-1 and kappa) for one lattice."""

    def __init__(self, dims, U_public, t_boundary=-1):
        self.dims = tuple(int(d) for d in dims)
        Lx, Ly, Lz, Lt = self.dims
        self.site_shape = (2, Lt, Lz, Ly, Lx // 2)
        self.V = Lx * Ly * Lz * Lt
        U = _c(U_public)
        assert U.shape == (4,) + self.site_shape + (3, 3), U.shape
        d = (ctypes.c_int * 4)(*self.dims)
        self._h = lib().orc_create(d, int(t_boundary), U.ctypes.data)
        if not self._h:
            raise ValueError("orc_create failed for dims %r" % (self.dims,))

    def __del__(self):
        if getattr(self, "_h", None):
            lib().orc_destroy(self._h)
            self._h = None

    def _spinor(self):
        return np.empty(self.site_shape + (4, 3), dtype=np.complex128)

    def set_clover(self, kappa, csw):
        rc = lib().orc_set_clover(self._h, float(kappa), float(csw))
        if rc != 0:
            raise ArithmeticError("singular clover block")
        return self

    def set_anisotropy(self, nu_over_xi0):
        """Spatial hop weight nu/xi_0 of Eq. 5; the temporal weight is 1."""
        lib().orc_set_anisotropy(self._h, float(nu_over_xi0))
        return self

    def set_clover_aniso(self, kappa, csw_s, csw_t):
        """A with csw_s = c_SW^r/xi_0 on the spatial planes and csw_t = c_SW^t on the temporal ones."""
        rc = lib().orc_set_clover_aniso(self._h, float(kappa), float(csw_s), float(csw_t))
        if rc != 0:
            raise ArithmeticError("singular clover block")
        return self

    def clover_defect(self):
        return lib().orc_clover_defect(self._h)

    def clover(self):
        """(A, Ainv) packed, float64 [2,Lt,Lz,Ly,Lx/2,2,36]."""
        A = np.empty(self.site_shape + (2, 36), dtype=np.float64)
        Ai = np.empty_like(A)
        lib().orc_get_clover(self._h, A.ctypes.data, Ai.ctypes.data)
        return A, Ai

    def clover_dense(self, kappa, csw):
        out = np.empty(self.site_shape + (12, 12), dtype=np.complex128)
        lib().orc_clover_dense(self._h, float(kappa), float(csw), out.ctypes.data)
        return out

    def fmunu(self, mu, nu):
        out = np.empty(self.site_shape + (3, 3), dtype=np.complex128)
        lib().orc_fmunu(self._h, mu, nu, out.ctypes.data)
        return out

    def dslash(self, psi, dagger=False, only_parity=-1):
        psi = _c(psi)
        out = self._spinor()
        lib().orc_dslash(self._h, psi.ctypes.data, out.ctypes.data, int(dagger), int(only_parity))
        return out

    def dslash_site(self, psi, public_index, dagger=False):
        psi = _c(psi)
        out = np.empty((4, 3), dtype=np.complex128)
        lib().orc_dslash_site(self._h, psi.ctypes.data, int(public_index), int(dagger),
                              out.ctypes.data)
        return out

    def clover_apply(self, psi, inverse=False, only_parity=-1):
        psi = _c(psi)
        out = self._spinor()
        lib().orc_clover_apply(self._h, psi.ctypes.data, out.ctypes.data, int(inverse),
                               int(only_parity))
        return out

    def mat(self, psi, dagger=False):
        psi = _c(psi)
        out = self._spinor()
        lib().orc_mat(self._h, psi.ctypes.data, out.ctypes.data, int(dagger))
        return out

    def mpc(self, psi, matpc=0, dagger=False):
        psi = _c(psi)
        out = self._spinor()
        lib().orc_mpc(self._h, psi.ctypes.data, out.ctypes.data, int(matpc), int(dagger))
        return out

    def invert(self, b, tol=1e-10, maxiter=1000, solver="cgne", matpc=0):
        b = _c(b)
        x = self._spinor()
        res = Result()
        lib().orc_invert(self._h, b.ctypes.data, x.ctypes.data, float(tol), int(maxiter),
                         SOLVERS[solver], int(matpc), ctypes.byref(res))
        return x, res

    def true_residual(self, b, x):
        b, x = _c(b), _c(x)
        return lib().orc_true_residual(self._h, b.ctypes.data, x.ctypes.data)
