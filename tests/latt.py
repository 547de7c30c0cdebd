"""Index helpers for the paper's cb2 layout [2, Lt, Lz, Ly, Lx/2].  Test-side host
logic only: index permutations, no operator arithmetic."""
import numpy as np


def coords(dims):
    """x, y, z, t integer arrays of shape (2, Lt, Lz, Ly, Lx/2) for every cb2 slot."""
    Lx, Ly, Lz, Lt = dims
    par, t, z, y, xh = np.meshgrid(np.arange(2), np.arange(Lt), np.arange(Lz), np.arange(Ly),
                                   np.arange(Lx // 2), indexing="ij")
    x = 2 * xh + ((par + y + z + t) & 1)
    return x, y, z, t


def cb_to_lex(f, dims):
    """[2,Lt,Lz,Ly,Lx/2,...] -> [Lt,Lz,Ly,Lx,...]"""
    Lx, Ly, Lz, Lt = dims
    t, z, y, x = np.meshgrid(np.arange(Lt), np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    par = (x + y + z + t) & 1
    return f[par, t, z, y, x // 2]


def lex_to_cb(f, dims):
    """[Lt,Lz,Ly,Lx,...] -> [2,Lt,Lz,Ly,Lx/2,...]"""
    x, y, z, t = coords(dims)
    return f[t, z, y, x]


def gauge_cb_to_lex(U, dims):
    return np.stack([cb_to_lex(U[mu], dims) for mu in range(4)])


def gauge_lex_to_cb(U, dims):
    return np.stack([lex_to_cb(U[mu], dims) for mu in range(4)])


# axis of direction mu (0..3 = x,y,z,t) in a lexicographic [Lt,Lz,Ly,Lx,...] array
AXIS = {0: 3, 1: 2, 2: 1, 3: 0}


def shift(f, mu, s):
    """g(x) = f(x + s*mu_hat), periodic, on a lexicographic array."""
    return np.roll(f, -s, axis=AXIS[mu])


def dagger(m):
    return np.conj(np.swapaxes(m, -1, -2))


def rel_err(a, b):
    return np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300)
