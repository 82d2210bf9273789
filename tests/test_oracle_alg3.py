"""Pins of the oracle's Algorithm 3 (oracle/alg3.py): the S1-partitioned 4D cube with a per-scan exit
multislice.  None of them re-types its formulas: brute force (Algorithm 1), the regrouping identity between the two
forms of the partitioned probe, Parseval, and Algorithm 5 with an exact detector matrix."""
import numpy as np

from bip_inputs.specimen import tiny_random_workload
from oracle import alg3
from oracle import beams as ob
from oracle import bip
from oracle import multislice as ms
from oracle import sibson as osb


def _setup(seed, **kw):
    wl = tiny_random_workload(seed, **kw)
    e = wl.edges[0]
    qa = wl.alpha_mrad * 1e-3 / wl.lam
    ap = ob.beams_in_disc(wl.ny, wl.nx, wl.ly, wl.lx, qa)
    c = ob.aperture_coefficients(ap, wl.ny, wl.nx, wl.ly, wl.lx, wl.lam, wl.defocus)
    P = ms.fresnel_propagator(wl.ny, wl.nx, wl.ly, wl.lx, wl.lam, wl.dz)
    T = np.exp(1j * np.angle(wl.T.astype(np.complex128)))
    return wl, e, qa, ap, c, P, T


def _all_beams(ny, nx):
    """Every pixel of the corner-origin DFT grid as a signed beam (the Nyquist row / column as -N/2), flat order."""
    hy = np.fft.fftfreq(ny, 1.0 / ny).astype(np.int64)
    hx = np.fft.fftfreq(nx, 1.0 / nx).astype(np.int64)
    return np.stack(np.meshgrid(hy, hx, indexing="ij"), axis=-1).reshape(-1, 2)


def test_alg3_full_parent_limit_equals_conventional_multislice():
    """Parents = all aperture beams, w = I: Algorithm 3 is exact PRISM-EELS (eq. 20) and must equal Algorithm 1 -- per scan
    conventional transition-potential multislice -- on EVERY exit beam, wrapped windows and a sub-pixel scan included."""
    wl, e, qa, ap, c, P, T = _setup(41, W=6, n_atoms=4, n_scan=3)
    I3 = alg3.alg3_cube(T, P, ap, c, np.arange(len(ap)), np.eye(len(ap)), wl.scan, e.slice, e.centre, e.H, "linear")
    I1 = ms.conventional_cube(c, ap, T, P, wl.scan, e.slice, e.centre, e.H.astype(complex), _all_beams(wl.ny, wl.nx))
    assert I3.shape == (3, wl.ny, wl.nx)
    assert np.abs(I3.reshape(3, -1) - I1).max() <= 1e-12 * I1.max()
    I3m = alg3.alg3_cube(T, P, ap, c, np.arange(len(ap)), np.eye(len(ap)), wl.scan, e.slice, e.centre, e.H, "magphase")
    assert np.abs(I3m - I3).max() <= 1e-12 * I3.max()                     # eq. 11 is exact at the parents


def test_beamlet_form_equals_reconstruct_then_sum():
    """eq. 9-10 only regroups the double sum of eq. 7 + eq. 15: for fewer parents than beams the beamlet-basis probe (the
    form Algorithm 3 prints) equals the reconstruct-then-sum probe, integer and sub-pixel scan positions alike; and the
    integer-scan beamlet is the roll of the rho = 0 beamlet."""
    wl, e, qa, ap, c, P, T = _setup(42, ny=16, nx=12)
    par = ob.hexring_parents(ap, wl.ny, wl.nx, wl.ly, wl.lx, qa, 2)
    assert len(par) < len(ap)
    w = osb.to_dense(osb.natural_neighbour_weights(ap, par, wl.ly, wl.lx, qa), len(par))
    S = ms.advance_S1(ms.build_S1(ap[par], wl.ny, wl.nx), T[0], P)
    spec = alg3.beamlet_spectra(w, c, ap, wl.ny, wl.nx)
    for rho in (np.array([0.0, 0.0]), np.array([5.0, 3.0]), np.array([2.5, 7.25])):
        a = alg3.beamlet_probe(S, ap[par], spec, rho, wl.ny, wl.nx)
        b = alg3.reconstructed_probe(S, ap[par], ap, w, c, rho, wl.ny, wl.nx, "linear")
        assert np.abs(a - b).max() <= 1e-13 * np.abs(b).max()
    hy = np.fft.fftfreq(wl.ny, 1.0 / wl.ny)[:, None]
    hx = np.fft.fftfreq(wl.nx, 1.0 / wl.nx)[None, :]
    b0 = np.fft.ifft2(spec[1])
    b53 = np.fft.ifft2(spec[1] * np.exp(-2j * np.pi * (hy * 5 / wl.ny + hx * 3 / wl.nx)))
    assert np.abs(b53 - np.roll(b0, (5, 3), axis=(0, 1))).max() <= 1e-15


def test_alg3_parseval_and_agreement_with_alg5_on_the_detector():
    """With fewer parents (a real approximation): (i) summing the cube over all exit beams gives sum_n ||H_n psi||^2 on the
    window, per scan (unitary exit operator and F); (ii) on the detector beams it equals Algorithm 5's cube
    when S2 is exact (parents = all detector beams): the two algorithms differ only in how the exit leg is carried."""
    wl, e, qa, ap, c, P, T = _setup(43, ny=16, nx=16, W=6, n_atoms=3, n_scan=3)
    par = ob.hexring_parents(ap, wl.ny, wl.nx, wl.ly, wl.lx, qa, 2)
    w = osb.to_dense(osb.natural_neighbour_weights(ap, par, wl.ly, wl.lx, qa), len(par))
    for recon in ("linear", "magphase"):
        I3 = alg3.alg3_cube(T, P, ap, c, par, w, wl.scan, e.slice, e.centre, e.H, recon)
        det = ob.beams_in_disc(wl.ny, wl.nx, wl.ly, wl.lx, e.det_mrad * 1e-3 / wl.lam)
        r5 = bip.bip_run(T, P, ap, c, ap[par], w, det, det, np.eye(len(det)), wl.scan, e.slice, e.centre, e.H, recon=recon,
                         want_psi=True)
        got = I3[:, det[:, 0] % wl.ny, det[:, 1] % wl.nx]
        assert np.abs(got - r5["cube"]).max() <= 1e-12 * r5["cube"].max()
        # Parseval per scan: the probe on the window is what Algorithm 5 hands out as Psi
        want = np.zeros(wl.n_rho)
        for Psi in r5["psi"]:
            for n in range(e.n_ch):
                want += (np.abs(Psi * e.H[n].reshape(1, -1)) ** 2).sum(axis=1)
        assert np.abs(I3.sum(axis=(1, 2)) - want).max() <= 1e-12 * want.max()
