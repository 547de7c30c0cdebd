"""The 16-bit storage format of include/lqcd.h ("16-bit storage"), restated in numpy for the tests: a spinor site is 24
int16 q and one fp32 norm n = max |component| with value = q * n / 32767; a link entry is rint(32767 u).  In memory the
integers are offset binary (q + 32768 as uint16)."""
import numpy as np

QMAX = np.float32(32767.0)


def quantise_spinor(psi):
    """psi: [..., 4, 3] complex -> (q int16 [..., 24], norm float32 [...]) exactly as the kernels do (fp32, round to nearest even)."""
    r = np.ascontiguousarray(psi.astype(np.complex64)).view(np.float32).reshape(psi.shape[:-2] + (24,))
    n = np.abs(r).max(axis=-1).astype(np.float32)
    inv = np.where(n > 0, QMAX / np.where(n > 0, n, 1), 0).astype(np.float32)
    q = np.rint(r.astype(np.float64) * inv[..., None].astype(np.float64)).astype(np.int16)  # one rounding (an fma in the kernel)
    return q, n


def dequantise_spinor(q, n):
    s = (n * (np.float32(1.0) / QMAX)).astype(np.float32)
    r = (q.astype(np.float32) * s[..., None]).astype(np.float32)
    return r.view(np.complex64).reshape(q.shape[:-1] + (4, 3))


def round_spinor(psi):
    """What a 16-bit context holds after packing psi."""
    return dequantise_spinor(*quantise_spinor(psi)).astype(np.complex128)


def round_links(U, recon=18):
    """What a 16-bit context multiplies by: entries rint(32767 u)/32767 in fp32; with 12 stored reals per link the
    third row is conj(row0 x row1) of the ROUNDED rows (rebuilt in fp32 in the kernel; here in fp64: 1e-7 apart)."""
    r = np.ascontiguousarray(U.astype(np.complex64)).view(np.float32)
    q = (np.rint(r.astype(np.float64) * 32767.0).astype(np.float32) * (np.float32(1.0) / QMAX)).astype(np.float32)
    V = q.view(np.complex64).reshape(U.shape).astype(np.complex128)
    if recon == 12:
        a, b = V[..., 0, :], V[..., 1, :]
        V[..., 2, :] = np.conj(np.cross(a, b))
    return V
