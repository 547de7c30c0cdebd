"""CPU test of the 16-bit storage format (include/lqcd.h "16-bit storage"): the round trip
error of a packed spinor is within the format's bound, norm / 65534 per component (half a quantisation step), and a
link entry within 1 / 65534."""
import numpy as np

from halfmodel import quantise_spinor, dequantise_spinor, round_links


def test_spinor_round_trip_within_half_a_step():
    rng = np.random.default_rng(7)
    for scale in (1e-6, 1.0, 3e4):
        psi = scale * (rng.normal(size=(500, 4, 3)) + 1j * rng.normal(size=(500, 4, 3)))
        psi[3] = 0                       # a zero site stays zero (norm 0)
        psi[4] = 0
        psi[4, 2, 1] = scale             # a point source: one component, exactly representable
        q, n = quantise_spinor(psi)
        back = dequantise_spinor(q, n).astype(np.complex128)
        p32 = psi.astype(np.complex64).astype(np.complex128)
        err = np.abs((back - p32).view(np.float64)).reshape(500, 24).max(axis=1)
        assert np.all(err <= n.astype(np.float64) / 65534 * (1 + 2e-2) + 1e-30)   # half a step + the fp32 rounding of the two scalings
        assert np.all(np.abs(q.astype(np.int32)).max(axis=1)[n > 0] == 32767)   # the largest component uses the full range
        assert not back[3].any() and back[4, 2, 1] == np.complex64(scale) and np.count_nonzero(back[4]) == 1


def test_link_rounding_bound_and_reconstruction():
    rng = np.random.default_rng(3)
    g = rng.normal(size=(200, 3, 3)) + 1j * rng.normal(size=(200, 3, 3))
    U = np.linalg.qr(g)[0]
    U = U / np.linalg.det(U)[:, None, None] ** (1 / 3)   # SU(3)
    for recon in (18, 12):
        V = round_links(U, recon)
        assert np.abs((V - U).view(np.float64)).max() <= (1 / 65534 * (1 + 1e-3) if recon == 18 else 2e-4)
