"""Pins of the oracle's forward model against what the paper and the mathematics fix (SURVEY.md §8(c) "pins").

None of these tests retypes an oracle formula: each compares an oracle routine with brute force (Alg. 1), a
library FFT closed form, an exact identity (reciprocity, Parseval) or an invariant.
"""
import os

import numpy as np
import pytest

from bip_inputs import electron_wavelength, interaction_constant
from bip_inputs.specimen import tiny_random_workload
from oracle import beams as ob
from oracle import bip
from oracle import multislice as ms

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _setup(seed=1, unitary=True, **kw):
    wl = tiny_random_workload(seed, **kw)
    e = wl.edges[0]
    qa = wl.alpha_mrad * 1e-3 / wl.lam
    qd = e.det_mrad * 1e-3 / wl.lam
    ap = ob.beams_in_disc(wl.ny, wl.nx, wl.ly, wl.lx, qa)
    det = ob.beams_in_disc(wl.ny, wl.nx, wl.ly, wl.lx, qd)
    c = ob.aperture_coefficients(ap, wl.ny, wl.nx, wl.ly, wl.lx, wl.lam, wl.defocus)
    P = ms.fresnel_propagator(wl.ny, wl.nx, wl.ly, wl.lx, wl.lam, wl.dz)
    T = wl.T.astype(np.complex128)
    if unitary:                                   # exact |T| = 1 (the complex64 rounding is ~6e-8 off)
        T = np.exp(1j * np.angle(T))
    return wl, e, ap, det, c, P, T


def test_constants_golden():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "constants.txt")) if l.strip() and not l.startswith("#")]
    for kv, lam, sig in rows:
        assert abs(electron_wavelength(float(kv)) - float(lam)) < 5e-7
        assert abs(interaction_constant(float(kv)) - float(sig)) < 5e-8


def test_beam_order_and_membership():
    b = ob.beams_in_disc(16, 12, 8.0, 6.0, 0.6)
    flat = ob.flat_index(b, 16, 12)
    assert np.all(np.diff(flat) > 0)
    # brute force membership over the whole signed grid, boundary included (<=)
    n = 0
    for hy in range(-7, 8):
        for hx in range(-5, 6):
            n += (hy / 8.0) ** 2 + (hx / 6.0) ** 2 <= 0.36
    assert n == b.shape[0]
    assert any((h == (0, 0)).all() for h in b)


def test_probe_unit_norm_and_position():
    wl, e, ap, det, c, P, T = _setup()
    for rho in wl.scan:
        psi = ms.probe(c, ap, rho, wl.ny, wl.nx)
        assert abs(np.sum(np.abs(psi) ** 2) - 1.0) < 1e-12
    # zero defocus: the probe peaks on the scan pixel (eq. 1 phase-ramp sign)
    c0 = ob.aperture_coefficients(ap, wl.ny, wl.nx, wl.ly, wl.lx, wl.lam, 0.0)
    psi = ms.probe(c0, ap, np.array([5.0, 7.0]), wl.ny, wl.nx)
    assert np.unravel_index(np.argmax(np.abs(psi)), psi.shape) == (5, 7)
    # eq. 1 is the inverse DFT of the aperture with a ramp: library check
    spec = np.zeros((wl.ny, wl.nx), complex)
    spec[ap[:, 0] % wl.ny, ap[:, 1] % wl.nx] = c0 * np.exp(-2j * np.pi * (ap[:, 0] * 5.0 / wl.ny + ap[:, 1] * 7.0 / wl.nx))
    assert np.abs(psi - np.fft.ifft2(spec) * wl.ny * wl.nx).max() < 1e-12


def test_parseval_unitary_steps():
    wl, e, ap, det, c, P, T = _setup()
    rng = np.random.default_rng(0)
    psi = rng.normal(size=(wl.ny, wl.nx)) + 1j * rng.normal(size=(wl.ny, wl.nx))
    n0 = np.linalg.norm(psi)
    assert abs(np.linalg.norm(ms.propagate(psi, P)) - n0) < 1e-12 * n0            # vacuum slice
    assert abs(np.linalg.norm(ms.exit_operator(psi, 0, T, P)) - n0) < 1e-12 * n0   # |T| = 1


def test_reciprocity_eq12_every_plane():
    """sum_r S2^d(r) w(r) = [F M_{i->exit} w]_{h_d} for random w (eq. 12)."""
    wl, e, ap, det, c, P, T = _setup()
    rng = np.random.default_rng(3)
    hs = det[[0, 5, len(det) // 2, -1]]
    for i in range(wl.nz + 1):
        S2 = ms.build_S2_at(hs, T, P, i)
        w = rng.normal(size=(wl.ny, wl.nx)) + 1j * rng.normal(size=(wl.ny, wl.nx))
        rhs = np.fft.fft2(ms.exit_operator(w, i, T, P))
        for k, h in enumerate(hs):
            lhs = np.sum(S2[k] * w)
            assert abs(lhs - rhs[h[0] % wl.ny, h[1] % wl.nx]) < 1e-11 * abs(lhs)


def test_peel_equals_rebuild():
    wl, e, ap, det, c, P, T = _setup()
    hs = det[[1, 7, -2]]
    S2 = ms.build_S2(hs, T, P)
    assert np.abs(S2 - ms.build_S2_at(hs, T, P, 0)).max() < 1e-13
    for i in range(wl.nz):
        S2 = ms.peel_S2(S2, T[i], P)
        assert np.abs(S2 - ms.build_S2_at(hs, T, P, i + 1)).max() < 1e-12
    # fully peeled = the bare conjugate plane wave
    assert np.abs(S2[0] - ms.plane_wave(hs[0], wl.ny, wl.nx, -1)).max() < 1e-12


@pytest.mark.parametrize("recon", ["linear", "magphase"])
@pytest.mark.parametrize("seed", [1, 2])
def test_full_parent_limit_equals_conventional(seed, recon):
    """BiP with parents = all aperture beams and all detector beams equals Alg. 1 per scan.
    Tiny non-square cell, wrapped windows, one sub-pixel scan position."""
    wl, e, ap, det, c, P, T = _setup(seed)
    I1 = ms.conventional_cube(c, ap, T, P, wl.scan, e.slice, e.centre, e.H.astype(complex), det)
    r = bip.bip_run(T, P, ap, c, ap, np.eye(len(ap)), det, det, np.eye(len(det)), wl.scan, e.slice, e.centre, e.H,
                    recon=recon)
    assert np.abs(I1 - r["cube"]).max() <= 1e-12 * I1.max()
    assert np.abs(I1.sum(1) - r["map"]).max() <= 1e-12 * I1.sum(1).max()


def test_complex64_T_peel_error_is_small():
    """With the complex64-rounded T (|T| = 1 +- 6e-8) the conjugate peel is exact only to that level."""
    wl, e, ap, det, c, P, T = _setup(1, unitary=False)
    I1 = ms.conventional_cube(c, ap, T, P, wl.scan, e.slice, e.centre, e.H.astype(complex), det)
    r = bip.bip_run(T, P, ap, c, ap, np.eye(len(ap)), det, det, np.eye(len(det)), wl.scan, e.slice, e.centre, e.H)
    assert np.abs(I1 - r["cube"]).max() <= 1e-6 * I1.max()


def test_vacuum_closed_form_library_fft():
    """Vacuum: S1_b stays a plane wave times P(q_b)^i, so a_d = P(q_d)^(nz-i) FFT[H psi_i](h_d) / sqrt(G)."""
    wl, e, ap, det, c, P, T = _setup(4)
    Tv = np.ones_like(T)
    r = bip.bip_run(Tv, P, ap, c, ap, np.eye(len(ap)), det, det, np.eye(len(det)), wl.scan, e.slice, e.centre, e.H)
    G = wl.ny * wl.nx
    cube = np.zeros((wl.scan.shape[0], len(det)))
    for si, rho in enumerate(wl.scan):
        spec = np.zeros((wl.ny, wl.nx), complex)
        spec[ap[:, 0] % wl.ny, ap[:, 1] % wl.nx] = c * np.exp(-2j * np.pi * (ap[:, 0] * rho[0] / wl.ny + ap[:, 1] * rho[1] / wl.nx))
        for a in range(e.n_atoms):
            i = int(e.slice[a])
            psi_i = np.fft.ifft2(spec * P ** i) * G
            for n in range(e.n_ch):
                src = ms.embed_window(e.H[n].astype(complex), e.centre[a], wl.ny, wl.nx) * psi_i
                amp = (P ** (wl.nz - i) * np.fft.fft2(src))[det[:, 0] % wl.ny, det[:, 1] % wl.nx] / np.sqrt(G)
                cube[si] += np.abs(amp) ** 2
    assert np.abs(cube - r["cube"]).max() <= 1e-12 * cube.max()


def test_all_G_detector_collects_everything():
    """Detector = every beam of the grid => I(rho) = sum_n sum_r |H_n(r - tau)|^2 |psi(r, rho)|^2 (unitary exit)."""
    wl, e, ap, det, c, P, T = _setup(5, ny=8, nx=8, W=4)
    allb = np.array([(ky if ky < 4 else ky - 8, kx if kx < 4 else kx - 8) for ky in range(8) for kx in range(8)])
    # (the Nyquist beams |h| = N/2 are outside the ABI's beam range but harmless for the oracle)
    r = bip.bip_run(T, P, ap, c, ap, np.eye(len(ap)), allb, allb, np.eye(64), wl.scan, e.slice, e.centre, e.H)
    want = np.zeros(wl.scan.shape[0])
    for si, rho in enumerate(wl.scan):
        psi = ms.probe(c, ap, rho, 8, 8)
        for i in range(wl.nz):
            for a in np.nonzero(e.slice == i)[0]:
                for n in range(e.n_ch):
                    want[si] += np.sum(np.abs(ms.embed_window(e.H[n].astype(complex), e.centre[a], 8, 8) * psi) ** 2)
            psi = ms.slice_step(psi, T[i], P)
    assert np.abs(want - r["map"]).max() <= 1e-12 * want.max()


def test_reducer_invariants_and_metamorphic():
    wl, e, ap, det, c, P, T = _setup(6)
    args = (T, P, ap, c, ap, np.eye(len(ap)), det, det, np.eye(len(det)), wl.scan)
    r = bip.bip_run(*args, e.slice, e.centre, e.H)
    m = r["map"]
    assert np.all(m >= 0) and np.all(r["cube"] >= 0)
    assert np.abs(r["qeels_x"].sum(1) - m).max() <= 4e-16 * m.max()
    assert np.abs(r["qeels_y"].sum(1) - m).max() <= 4e-16 * m.max()
    assert np.abs(r["cube"].sum(1) - m).max() <= 4e-16 * m.max()
    assert r["qeels_x"].shape[1] == len(np.unique(det[:, 1]))
    # H -> 2H  =>  I -> 4I
    r2 = bip.bip_run(*args, e.slice, e.centre, 2 * e.H)
    assert np.abs(r2["map"] - 4 * m).max() <= 1e-13 * m.max()
    # sites are additive (incoherent sum, eq. 4 / 14)
    parts = sum(bip.bip_run(*args, e.slice[k:k + 1], e.centre[k:k + 1], e.H)["map"] for k in range(e.n_atoms))
    assert np.abs(parts - m).max() <= 1e-13 * m.max()
    # channels are additive
    parts = sum(bip.bip_run(*args, e.slice, e.centre, e.H[n:n + 1])["map"] for n in range(e.n_ch))
    assert np.abs(parts - m).max() <= 1e-13 * m.max()


def test_translation_covariance():
    """Integer-pixel translation of (potential, atoms, scans) leaves every I(rho) unchanged."""
    wl, e, ap, det, c, P, T = _setup(7)
    args = (P, ap, c, ap, np.eye(len(ap)), det, det, np.eye(len(det)))
    r = bip.bip_run(T, *args, wl.scan, e.slice, e.centre, e.H)
    dy, dx = 3, 5
    T2 = np.roll(T, (dy, dx), axis=(1, 2))
    cen2 = (e.centre + np.array([dy, dx])) % np.array([wl.ny, wl.nx])
    r2 = bip.bip_run(T2, *args, wl.scan + np.array([dy, dx]), e.slice, cen2.astype(np.int32), e.H)
    assert np.abs(r["cube"] - r2["cube"]).max() <= 1e-12 * r["cube"].max()


def test_coupling_matrix_association_equals_conventional():
    """Eq. 13 as printed (coupling matrix M first, then all scans; Alg. 4 lines 6-8) with parents = all beams against
    Alg. 1 brute force, and against the probe-first association of the same triple product (BiP, f > 1)."""
    from bip_inputs.specimen import make_workload
    from helpers import OracleSetup
    wl, e, ap, det, c, P, T = _setup(5, W=8, n_atoms=3, n_scan=4)
    I1 = ms.conventional_cube(c, ap, T, P, wl.scan, e.slice, e.centre, e.H.astype(complex), det)
    r = bip.bip_run(T, P, ap, c, ap, np.eye(len(ap)), det, det, np.eye(len(det)), wl.scan, e.slice, e.centre, e.H,
                    association="coupling")
    assert np.abs(r["cube"] - I1).max() <= 1e-12 * I1.max()
    wl2 = make_workload("cfg1", scale=2, nz=3, scan=(3, 3))
    e2 = wl2.edges[0].take([0, 1])
    orc2 = OracleSetup(wl2, e2)
    for recon in ("linear", "magphase"):
        a, b = orc2.run(wl2, e2, recon), orc2.run(wl2, e2, recon, association="coupling")
        assert np.abs(a["cube"] - b["cube"]).max() <= 1e-12 * a["cube"].max()
