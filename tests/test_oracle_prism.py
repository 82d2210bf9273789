"""Pins of the PRISM beam subsampling, coefficient rescale and crop mask in the oracle."""
import numpy as np
import scipy.sparse as sp

from oracle import beams as ob
from oracle import bip as obip
from oracle import multislice as oms


def test_subsampled_probe_is_the_periodic_replica_of_the_exact_probe():
    """with every f-th beam kept and the coefficients rescaled by f_y f_x the synthesised probe "becomes
    periodic with period (N_y / f_y, N_x / f_x), matching the exact probe inside this window" -- exactly, the sum of
    the shifted copies of the exact probe (DFT decimation <-> periodic summation).  The exact probe comes from
    numpy.fft here, not from the oracle's plane-wave sum."""
    ny, nx, ly, lx, lam = 48, 36, 20.0, 15.0, 0.02
    fy, fx = 4, 3
    qa = 0.6
    beams = ob.beams_in_disc(ny, nx, ly, lx, qa)
    c = ob.aperture_coefficients(beams, ny, nx, ly, lx, lam, -30.0)
    rho = np.array([[13.0, 7.5]])
    # exact probe by library FFT: psi(r) = sum_h C[h] exp(2 pi i h.r/N) = G * ifft2(C)
    Cg = np.zeros((ny, nx), dtype=complex)
    Cg[beams[:, 0] % ny, beams[:, 1] % nx] = c * np.exp(-2j * np.pi * (beams[:, 0] * rho[0, 0] / ny + beams[:, 1] * rho[0, 1] / nx))
    psi1 = np.fft.ifft2(Cg) * (ny * nx)
    replica = sum(np.roll(psi1, (-my * ny // fy, -mx * nx // fx), axis=(0, 1)) for my in range(fy) for mx in range(fx))
    # oracle: subsampled beams, rescaled coefficients, eq. 7 with plane-wave columns (plane 0)
    keep = ob.prism_subsample(beams, fy, fx)
    assert 0 < len(keep) < len(beams) and np.all(beams[keep, 0] % fy == 0) and np.all(beams[keep, 1] % fx == 0)
    assert np.array_equal(keep, np.sort(keep))
    cf = ob.prism_coefficients(c, keep, fy, fx)
    S = oms.build_S1(beams[keep], ny, nx)
    A = obip.illumination(cf, beams[keep], rho, ny, nx)
    psif = np.tensordot(A[0], S, axes=(0, 0))
    assert np.abs(psif - replica).max() < 1e-12 * np.abs(psi1).max()
    assert np.abs(psif - np.roll(psif, ny // fy, axis=0)).max() < 1e-12 * np.abs(psi1).max()      # period N_y / f_y
    assert np.abs(psif - np.roll(psif, nx // fx, axis=1)).max() < 1e-12 * np.abs(psi1).max()


def _run(T, ly, lx, lam, dz, qa, qd, f, scan, sl, centre, H, crop_f=None, full_counts=None):
    nz, ny, nx = T.shape
    ap = ob.beams_in_disc(ny, nx, ly, lx, qa)
    det = ob.beams_in_disc(ny, nx, ly, lx, qd)
    c = ob.aperture_coefficients(ap, ny, nx, ly, lx, lam, -8.0)
    if f != (1, 1):
        keep = ob.prism_subsample(ap, *f)
        ap, c = ap[keep], ob.prism_coefficients(c, keep, *f)
        det = det[ob.prism_subsample(det, *f)]
    P = oms.fresnel_propagator(ny, nx, ly, lx, lam, dz)
    I1, I2 = sp.identity(len(ap), format="csr"), sp.identity(len(det), format="csr")
    out = obip.bip_run(T, P, ap, c, ap, I1, det, det, I2, scan, sl, centre, H, crop_f=crop_f)
    return out, ap, det


def test_prism_on_a_tiled_cell_equals_the_small_cell():
    """A specimen that is itself periodic with period N / f: the f-subsampled calculation on the big grid is the
    all-beam calculation on one tile (the retained beams ARE the tile's beams, the columns are the tile's columns
    repeated).  With the probe normalisations of c3 the maps differ by the ratio of beam counts only:
    I_big = I_small * B_small / B_full.  Pins the subsampling rule and the f_y f_x rescale through the whole Alg. 5."""
    rng = np.random.default_rng(11)
    n_y, n_x, fy, fx, nz = 12, 10, 2, 3, 3
    ly, lx, lam, dz = 6.0, 5.0, 0.025, 2.0
    Ts = np.exp(1j * rng.normal(size=(nz, n_y, n_x)))
    Tb = np.tile(Ts, (1, fy, fx))
    W = 6
    H = rng.normal(size=(2, W, W)) + 1j * rng.normal(size=(2, W, W))
    sl = np.array([0, 1, 2])
    centre_b = np.array([[3, 4], [17, 22], [23, 29]])
    scan_b = np.array([[2.0, 3.0], [15.5, 21.25], [20.0, 28.0], [8.0, 11.0]])
    qa, qd = 0.45, 0.8
    big, ap_b, det_b = _run(Tb, ly * fy, lx * fx, lam, dz, qa, qd, (fy, fx), scan_b, sl, centre_b, H)
    small, ap_s, det_s = _run(Ts, ly, lx, lam, dz, qa, qd, (1, 1), scan_b % np.array([n_y, n_x]), sl, centre_b % np.array([n_y, n_x]), H)
    assert np.array_equal(ap_b // np.array([fy, fx]), ap_s) and np.array_equal(det_b // np.array([fy, fx]), det_s)
    B_full = len(ob.beams_in_disc(n_y * fy, n_x * fx, ly * fy, lx * fx, qa))
    ratio = len(ap_s) / B_full
    assert np.abs(big["map"] - small["map"] * ratio).max() < 1e-12 * small["map"].max()
    assert np.abs(big["cube"] - small["cube"] * ratio).max() < 1e-12 * small["cube"].max()


def test_crop_mask_geometry_and_definition():
    """"a PRISM crop mask restricts each atom's contribution to the scans inside its 1/f window"."""
    ny, nx = 32, 24
    yy, xx = np.meshgrid(np.arange(0, ny, 2.0), np.arange(0, nx, 2.0), indexing="ij")
    scan = np.stack([yy.ravel(), xx.ravel()], axis=1)
    m = ob.crop_mask(scan, (1, 23), ny, nx, 4, 2)                      # window wraps both axes
    # |dy| < 4 -> y in {30, 0, 2, 4} (dy = -3, -1, 1, 3); |dx| < 6 -> x in {18, 20, 22, 0, 2, 4} (dx = -5 .. 5)
    inside = {(y, x) for y in (30, 0, 2, 4) for x in (18, 20, 22, 0, 2, 4)}
    assert {(int(a), int(b)) for a, b in scan[m]} == inside
    assert ob.crop_mask(scan, (1, 23), ny, nx, 1, 1).sum() == len(scan)    # f = 1: |d| < N/2 excludes only d = -N/2 (none here)
    # definition: masked run == sum over sites of (single-site run) * mask
    rng = np.random.default_rng(3)
    T = np.exp(1j * rng.normal(size=(2, ny, nx)))
    H = rng.normal(size=(1, 6, 6)) + 1j * rng.normal(size=(1, 6, 6))
    sl, centre = np.array([0, 1]), np.array([[1, 23], [20, 10]])
    sc = scan[::7]
    args = (16.0, 12.0, 0.025, 2.0, 0.4, 0.7, (1, 1), sc)
    both, _, _ = _run(T, *args, sl, centre, H, crop_f=(4, 2))
    want = 0.0
    for a in range(2):
        one, _, _ = _run(T, *args, sl[a:a + 1], centre[a:a + 1], H)
        want = want + one["map"] * ob.crop_mask(sc, centre[a], ny, nx, 4, 2)
    assert np.abs(both["map"] - want).max() < 1e-14 * want.max()
    assert both["map"].min() >= 0 and (both["map"] == 0).any() and (both["map"] > 0).any()
