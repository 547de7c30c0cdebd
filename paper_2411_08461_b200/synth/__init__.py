"""Seeded synthetic inputs (SU(3) links, sources) in the paper's public cb2 layout.

PAPER.md:54 (§II.A Convention) fixes the layouts; SURVEY.md §8(c) O10/O11 and DESIGN.md
"Input recipe" fix the distributions.  This module only makes inputs: it holds none of the
method's arithmetic and is the one module the oracle's tests and the CUDA path's tests share.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libsynth.so")
_SRC = os.path.join(_HERE, "synth.cpp")


def build(force=False):
    """Compile libsynth.so in-tree (g++ -O2 -fopenmp, no fast-math)."""
    if not force and os.path.exists(_SO) and os.path.getmtime(_SO) >= os.path.getmtime(_SRC):
        return _SO
    subprocess.check_call(
        ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-o", _SO, _SRC])
    return _SO


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        ip = ctypes.POINTER(ctypes.c_int)
        dp = ctypes.c_void_p
        lib.synth_gauge.argtypes = [ip, ctypes.c_double, ctypes.c_uint64, dp]
        lib.synth_colour_rotation.argtypes = [ip, ctypes.c_double, ctypes.c_uint64, dp]
        lib.synth_source.argtypes = [ip, ctypes.c_int, ctypes.c_uint64, ctypes.c_int,
                                     ctypes.c_int, dp]
        _lib = lib
    return _lib


def _dims(dims):
    return (ctypes.c_int * 4)(*[int(d) for d in dims])


def gauge(dims, eps, seed):
    """Links U_mu(x) = exp(i*eps*H), reunitarised. complex128 [4,2,Lt,Lz,Ly,Lx/2,3,3]."""
    Lx, Ly, Lz, Lt = dims
    U = np.empty((4, 2, Lt, Lz, Ly, Lx // 2, 3, 3), dtype=np.complex128)
    rc = _load().synth_gauge(_dims(dims), float(eps), int(seed), U.ctypes.data)
    if rc != 0:
        raise ValueError("synth_gauge: bad dims %r" % (dims,))
    return U


def unit_gauge(dims):
    Lx, Ly, Lz, Lt = dims
    U = np.zeros((4, 2, Lt, Lz, Ly, Lx // 2, 3, 3), dtype=np.complex128)
    for c in range(3):
        U[..., c, c] = 1.0
    return U


def colour_rotation(dims, seed, eps=1.0):
    """One random SU(3) matrix per site. complex128 [2,Lt,Lz,Ly,Lx/2,3,3]."""
    Lx, Ly, Lz, Lt = dims
    g = np.empty((2, Lt, Lz, Ly, Lx // 2, 3, 3), dtype=np.complex128)
    rc = _load().synth_colour_rotation(_dims(dims), float(eps), int(seed), g.ctypes.data)
    if rc != 0:
        raise ValueError("synth_colour_rotation: bad dims %r" % (dims,))
    return g


_KINDS = {"point": 0, "z2": 1, "gaussian": 2}


def source(dims, kind, seed=0, spin=0, colour=0):
    """Source vector. complex128 [2,Lt,Lz,Ly,Lx/2,4,3]. kind: point | z2 | gaussian."""
    Lx, Ly, Lz, Lt = dims
    b = np.empty((2, Lt, Lz, Ly, Lx // 2, 4, 3), dtype=np.complex128)
    rc = _load().synth_source(_dims(dims), _KINDS[kind], int(seed), int(spin), int(colour),
                              b.ctypes.data)
    if rc != 0:
        raise ValueError("synth_source: bad arguments")
    return b


def round_fp32(a):
    """Round a complex128/float64 array to fp32 precision, kept in the 64-bit dtype (A16)."""
    if np.iscomplexobj(a):
        return a.astype(np.complex64).astype(np.complex128)
    return a.astype(np.float32).astype(np.float64)


# BASELINE.json configs: dims (Lx,Ly,Lz,Lt), eps, gauge seed, kappa, csw,
# source kind, source seed
CONFIGS = {
    1: dict(dims=(4, 4, 4, 8), eps=0.3, seed=1, kappa=0.12, csw=1.0, source="point", src_seed=101),
    2: dict(dims=(8, 8, 8, 16), eps=0.5, seed=2, kappa=0.124, csw=1.2, source="z2", src_seed=102),
    3: dict(dims=(16, 16, 16, 32), eps=0.7, seed=3, kappa=0.1245, csw=1.5, source="gaussian",
            src_seed=103),
    4: dict(dims=(32, 32, 32, 64), eps=0.8, seed=4, kappa=0.1248, csw=1.8, source="gaussian",
            src_seed=104),
    5: dict(dims=(48, 48, 48, 96), eps=0.8, seed=5, kappa=0.12485, csw=1.9, source="gaussian",
            src_seed=105),
}
