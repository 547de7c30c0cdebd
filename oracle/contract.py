"""CPU ORACLE (TEST INFRASTRUCTURE) for the source / contraction steps of the paper's Listing 1
(Eqs. 6-8).  Plain numpy in complex128;
the einsum subscripts are the paper's own.  Only tests/, smoke() and bench.py's cpu legs may import this.

Layouts: site axes [2, Lt, Lz, Ly, Lx/2] ("wtzyx"); a propagator is
[2, Lt, Lz, Ly, Lx/2, Ns_sink, Ns_src, Nc_sink, Nc_src] ("wtzyxjiba" reads sink spin j, source spin i,
sink colour b, source colour a); a solution column for source (spin i, colour a) is a spinor
[2, Lt, Lz, Ly, Lx/2, 4, 3]."""
import numpy as np


def coordinates(dims):
    """x, y, z, t of every cb2 slot, shape [2, Lt, Lz, Ly, Lx/2] (x = 2*xh + ((w+y+z+t) mod 2))."""
    Lx, Ly, Lz, Lt = dims
    w, t, z, y, xh = np.meshgrid(np.arange(2), np.arange(Lt), np.arange(Lz), np.arange(Ly),
                                 np.arange(Lx // 2), indexing="ij")
    return 2 * xh + ((w + y + z + t) & 1), y, z, t


def momentum_phase(dims, mom):
    """exp(i p.x), p_i = 2 pi n_i / L_i, n = mom = [nx, ny, nz] (PAPER.md:163 MomentumPhase.getPhase)."""
    x, y, z, _ = coordinates(dims)
    arg = 2 * np.pi * (mom[0] * x / dims[0] + mom[1] * y / dims[1] + mom[2] * z / dims[2])
    return np.exp(1j * arg)


def wall_source(dims, t0, spin, colour, phase=None):
    """Wall source at time-slice t0 for one (spin, colour) column: 1 (or phase(x)) on every site of the
    slice in that spin-colour component, 0 elsewhere."""
    Lx, Ly, Lz, Lt = dims
    b = np.zeros((2, Lt, Lz, Ly, Lx // 2, 4, 3), dtype=np.complex128)
    b[:, t0, :, :, :, spin, colour] = 1.0 if phase is None else phase[:, t0]
    return b


def assemble(columns):
    """12 solution columns (index 3*spin_src + colour_src) -> propagator [.., j, i, b, a]."""
    cols = np.asarray(columns)
    prop = np.zeros(cols.shape[1:6] + (4, 4, 3, 3), dtype=np.complex128)
    for i in range(4):
        for a in range(3):
            prop[..., :, i, :, a] = cols[3 * i + a]
    return prop


def twopt(phase, S_0, S_p):
    """Eq. 6 (listing lines 33-38): sum_{w,x,y,z,i,j,a,b} e^{-ipx} S_0^* S_p per time-slice."""
    return np.einsum("wtzyx,wtzyxjiba,wtzyxjiba->t", phase.conj(), S_0.conj(), S_p, optimize=True)


def threept(S_p0, gamma, S_p):
    """Eq. 7 (listing lines 40-46): sum S_p0^*_{ji}^{ba} Gamma_{jk} S_p_{ki}^{ba} per time-slice."""
    return np.einsum("wtzyxjiba,jk,wtzyxkiba->t", S_p0.conj(), gamma, S_p, optimize=True)


def sequential_source(phase, gamma, S_0, t):
    """Eq. 8 (listing lines 21-28): X = e^{-ipx} Gamma_{ij} S_0(x,t)_{jk}^{ab} on slice t, 0 elsewhere."""
    X = np.zeros_like(S_0)
    X[:, t] = np.einsum("wzyx,ij,wzyxjkab->wzyxikab", phase[:, t].conj(), gamma, S_0[:, t], optimize=True)
    return X
