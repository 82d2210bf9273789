"""Pins of the two oracle functions whose sign / scale no other pin fixes: the Fresnel transfer function
(eq. 2) and the lens phase of the probe coefficients (reading c4).

Every other test that involves ``P`` uses the oracle's own ``P`` on both sides (Parseval holds for any unimodular
``P``; Alg. 1 vs Alg. 5 share it; reciprocity and peel are identities in ``P``), so a wrong sign, a missing pi, lambda
in the wrong unit or q in pixels instead of 1/Angstrom would pass them all.  The pins here compare
``oracle.multislice.propagate`` with closed forms of free-space paraxial propagation that are written out
independently of eq. 2:

  * the Gaussian beam (complex field, so the SIGN of the exponent is pinned too): with the paper's carrier
    convention -- plane waves exp(+2 pi i q.r), eq. 1 -- a forward-going beam is
        psi(r, z) = q0 / q(z) . exp(+i pi r^2 / (lambda q(z))),  q(z) = z - i z_R,  z_R = pi w0^2 / lambda,
    i.e. width w0 sqrt(1 + (z / z_R)^2) and a DIVERGING wavefront exp(+i pi r^2 / (lambda R)) behind the waist;
  * Talbot self-imaging: a grating of period a returns to itself after z_T = 2 a^2 / lambda and to its half-period
    shift after z_T / 2, on both axes of a non-square cell (pins pi, lambda, the 1/Angstrom unit of q and ly vs lx);
  * the focus of the probe: with defocus df < 0 the on-axis intensity of the vacuum-propagated probe peaks at depth
    |df| (one slice tolerance), with df > 0 it only falls from the entrance surface (pins the sign and the scale of
    the lens phase relative to the propagator).
"""
import numpy as np

from bip_inputs import electron_wavelength
from oracle import beams as ob
from oracle import multislice as ms
from oracle import sibson as osb


def test_fresnel_propagator_gaussian_beam_closed_form():
    lam = electron_wavelength(200.0)
    ny, nx, ly, lx = 192, 256, 30.0, 40.0                   # non-square cell and grid
    w0, dz, n = 1.5, 5.0, 40
    y = (np.arange(ny) - ny // 2) * (ly / ny)
    x = (np.arange(nx) - nx // 2) * (lx / nx)
    r2 = y[:, None] ** 2 + x[None, :] ** 2
    zR = np.pi * w0 * w0 / lam

    def beam(z):
        q = z - 1j * zR
        return (-1j * zR / q) * np.exp(1j * np.pi * r2 / (lam * q))

    P = ms.fresnel_propagator(ny, nx, ly, lx, lam, dz)
    psi = beam(0.0)
    assert np.allclose(psi, np.exp(-r2 / (w0 * w0)))        # the waist is the plain Gaussian
    for _ in range(n):
        psi = ms.propagate(psi, P)
    want = beam(n * dz)
    assert np.abs(psi - want).max() < 1e-9
    # the textbook width law on the intensity, and the conjugate (wrong-sign) field is NOT what comes out
    wz = w0 * np.sqrt(1.0 + (n * dz / zR) ** 2)
    I = np.abs(psi) ** 2
    assert abs(np.sqrt(2.0 * (I * r2).sum() / I.sum()) - wz) < 1e-8 * wz      # <r^2> = w^2 / 2 for exp(-2 r^2 / w^2)
    assert np.abs(psi - np.conj(want)).max() > 0.1


def test_fresnel_propagator_talbot_self_imaging():
    lam = electron_wavelength(300.0)
    ny, nx, ly, lx = 48, 64, 12.0, 20.0
    y = np.arange(ny) * (ly / ny)
    x = np.arange(nx) * (lx / nx)
    for axis, a in ((0, ly / 3.0), (1, lx / 4.0)):          # an integer number of periods in the cell
        coord = y[:, None] + 0 * x[None, :] if axis == 0 else 0 * y[:, None] + x[None, :]
        grating = 1.0 + 0.3 * np.cos(2 * np.pi * coord / a) + 0.1 * np.sin(4 * np.pi * coord / a)
        shifted = 1.0 + 0.3 * np.cos(2 * np.pi * (coord + a / 2) / a) + 0.1 * np.sin(4 * np.pi * (coord + a / 2) / a)
        zT = 2.0 * a * a / lam
        n = 32
        P = ms.fresnel_propagator(ny, nx, ly, lx, lam, zT / n)
        psi = grating.astype(np.complex128)
        for k in range(n):
            psi = ms.propagate(psi, P)
            if k + 1 == n // 2:
                assert np.abs(psi - shifted).max() < 1e-10   # half the Talbot length: shifted by half a period
                assert np.abs(psi - grating).max() > 0.1
            if k + 1 == n // 4:
                assert np.abs(np.abs(psi) ** 2 - grating ** 2).max() > 0.05    # no self-image at a quarter
        assert np.abs(psi - grating).max() < 1e-10           # the Talbot length: the grating itself


def _on_axis_depth_profile(defocus, n_steps):
    lam = electron_wavelength(300.0)
    ny = nx = 128
    ly = lx = 19.5
    dz = 1.95
    beams = ob.beams_in_disc(ny, nx, ly, lx, 25e-3 / lam)
    c = ob.aperture_coefficients(beams, ny, nx, ly, lx, lam, defocus)
    rho = np.array([40.0, 72.0])
    psi = ms.probe(c, beams, rho, ny, nx)
    P = ms.fresnel_propagator(ny, nx, ly, lx, lam, dz)
    prof = [abs(psi[40, 72]) ** 2]
    for _ in range(n_steps):
        psi = ms.propagate(psi, P)                            # vacuum slices
        prof.append(abs(psi[40, 72]) ** 2)
    return np.array(prof), dz


def test_defocus_sign_and_scale_reading_c4():
    """df = -50 A focuses 50 A below the entrance surface (configs[1] and [4] run there); df = +50 A does not."""
    prof, dz = _on_axis_depth_profile(-50.0, 52)
    k = int(np.argmax(prof))
    assert abs(k * dz - 50.0) <= dz                          # focus at depth |df|, to one slice
    assert prof[k] > 3.0 * prof[0]                           # and it IS a focus: far brighter than at the surface
    # the in-focus probe (df = 0) at the surface has the same on-axis intensity as the defocused one at its focus
    prof0, _ = _on_axis_depth_profile(0.0, 1)
    assert abs(prof.max() - prof0[0]) < 0.02 * prof0[0]
    over, _ = _on_axis_depth_profile(+50.0, 52)
    # overfocus: the crossover lies above the surface -- brightest at depth 0, no focus anywhere in the slab
    assert int(np.argmax(over)) == 0 and over[1:].max() < over[0] and over.max() < 0.1 * prof.max()
    # half the defocus, half the depth (scale of the lens phase)
    half, dz = _on_axis_depth_profile(-25.0, 30)
    assert abs(int(np.argmax(half)) * dz - 25.0) <= dz


def test_pruned_sibson_equals_unpruned_on_cfg2_tables():
    """The pruned path of sibson_row (an optimisation inside the oracle, used alone on the 1951 / 4921-parent tables
    of BASELINE.json configs[1]) against the unpruned definition on a sample of rows of those very tables,
    interior, rim and hull-exterior beams."""
    lam = electron_wavelength(300.0)
    ny = nx = 512
    L = 78.1
    for mrad, nr in ((25.0, 25), (40.0, 40)):
        qmax = mrad * 1e-3 / lam
        beams = ob.beams_in_disc(ny, nx, L, L, qmax)
        pos = ob.hexring_parents(beams, ny, nx, L, L, qmax, nr)
        q = np.stack([beams[:, 0] / L, beams[:, 1] / L], axis=1)
        r = np.hypot(q[:, 0], q[:, 1])
        rows = list(range(7, len(beams), len(beams) // 12)) + list(np.argsort(r)[-6:]) + list(np.argsort(r)[:3])
        for b in rows:
            i0, w0 = osb.sibson_row(q[b], q[pos], qmax, prune=False)
            i1, w1 = osb.sibson_row(q[b], q[pos], qmax, prune=True)
            assert np.array_equal(i0, i1) and np.abs(w0 - w1).max() < 1e-12
