"""Error budget of the block fixed-point operand slices (precision BIP_PREC_FP16X4: 2^-21 of the ROW maximum; BF16X6:
2^-24), emulated on the CPU with the oracle's own arrays -- the evidence behind DESIGN.md section 6 "FP16X4 is block fixed
point, and where that shows".  No GPU and no library code: the quantiser below is the format's definition
(paper_2607_00756_b200/csrc/bip_sliced.cuh, restated), applied to the fp64 operands of one site."""
import numpy as np
import pytest

from bip_inputs.specimen import make_workload
from helpers import OracleSetup
from oracle import bip as obip
from oracle import multislice as oms


def _quantise_rows(M, bits):
    """Every row against its own power-of-two scale > max(|re|, |im|): values rounded to 2^-bits of that scale."""
    m = np.maximum(np.abs(M.real).max(axis=1), np.abs(M.imag).max(axis=1))
    s = 2.0 ** (np.floor(np.log2(np.maximum(m, 1e-300))) + 1.0)
    q = (s * 2.0 ** -bits)[:, None]
    return (np.round(M.real / q) + 1j * np.round(M.imag / q)) * q


@pytest.mark.slow
def test_one_channel_cube_is_where_fp16x4_reaches_the_pixel_bound():
    """The O edge (ONE channel) of the configs[2] clone, one site: quantising only Phi = H psi to 2^-21 of its row maxima
    gives ~1e-4 of the floored cube denominator (c15) -- what the GPU measures with FP16X4 (1.0-1.1e-4) -- at a weak beam
    of the scan position that sits on the atom; 2^-24 (BF16X6) gives ~2e-5; R2, A and R1 contribute 10x less."""
    wl = make_workload("cfg3", scale=4, nz=8, scan=(8, 16))
    e = wl.edges[0].take(np.array([0]))
    assert e.n_ch == 1
    orc = OracleSetup(wl, e)
    T = wl.T.astype(np.complex128)
    plane = int(e.slice[0])
    S1 = oms.build_S1(orc.ap[orc.p1_pos], wl.ny, wl.nx)
    for i in range(plane):
        S1 = oms.advance_S1(S1, T[i], orc.P)
    S2 = oms.build_S2_at(orc.det[orc.p2_pos], T, orc.P, plane)
    R1 = obip.reconstruct_window(S1, orc.ap[orc.p1_pos], orc.ap, orc.w1, e.centre[0], e.W, wl.ny, wl.nx, +1, "linear")
    R2 = obip.reconstruct_window(S2, orc.det[orc.p2_pos], orc.det, orc.w2, e.centre[0], e.W, wl.ny, wl.nx, -1, "linear")
    A = obip.illumination(orc.c, orc.ap, wl.scan, wl.ny, wl.nx)
    H = e.H.astype(np.complex128)[0].reshape(1, -1)
    G = wl.ny * wl.nx
    Phi = (A @ R1) * H
    exact = np.abs(Phi @ R2.T) ** 2 / G

    def floored(c):
        err = np.abs(c - exact) / np.maximum(exact, 1e-3 * exact.max())
        i = np.unravel_index(np.argmax(err), err.shape)
        return float(err.max()), int(i[0])

    e21, row21 = floored(np.abs(_quantise_rows(Phi, 21) @ R2.T) ** 2 / G)
    e24, _ = floored(np.abs(_quantise_rows(Phi, 24) @ R2.T) ** 2 / G)
    r21, _ = floored(np.abs(Phi @ _quantise_rows(R2, 21).T) ** 2 / G)
    bright = int(np.argmax(exact.max(axis=1)))
    assert 5e-5 < e21 < 2e-4 and row21 == bright           # at the bound, in the brightest row (the scan on the atom)
    assert e24 < 3e-5 and r21 < 0.2 * e21
