"""The locality result (eq. 16-19) and the soft convergence trend on small cells."""
import numpy as np
import pytest

from bip_inputs.specimen import make_workload, tiny_random_workload
from oracle import beams as ob
from oracle import bip
from oracle import multislice as ms
from oracle import sibson as osb


def test_locality_equalities_alg3_vs_alg2():
    """Alg. 3 (partitioned S1 + exact exit multislice) against Alg. 2 (exact S1):
    the error of the complex exit wavefield equals the error of its source (eq. 18), which is the on-window
    probe error weighted by H (eq. 16) and bounded by max|H| * ||dpsi||_Omega (eq. 17)."""
    wl = tiny_random_workload(21, ny=16, nx=16, nz=3, n_ch=2, W=6)
    e = wl.edges[0]
    ny = nx = 16
    qa = 0.62
    ap = ob.beams_in_disc(ny, nx, wl.ly, wl.lx, qa)
    c = ob.aperture_coefficients(ap, ny, nx, wl.ly, wl.lx, wl.lam, wl.defocus)
    P = ms.fresnel_propagator(ny, nx, wl.ly, wl.lx, wl.lam, wl.dz)
    T = np.exp(1j * np.angle(wl.T.astype(np.complex128)))
    par = ob.hexring_parents(ap, ny, nx, wl.ly, wl.lx, qa, 2)
    assert len(par) < len(ap)
    w1 = osb.to_dense(osb.natural_neighbour_weights(ap, par, wl.ly, wl.lx, qa), len(par))
    S_exact = ms.build_S1(ap, ny, nx)
    S_par = ms.build_S1(ap[par], ny, nx)
    G = ny * nx
    checked = 0
    for i in range(wl.nz):
        for a in np.nonzero(e.slice == i)[0]:
            for rho in wl.scan:
                A = bip.illumination(c, ap, rho[None, :], ny, nx)
                psi = (A @ S_exact.reshape(len(ap), -1)).reshape(ny, nx)                   # eq. 7
                psi_p = bip.partitioned_probe_full(S_par, ap[par], ap, w1, c, rho, ny, nx)  # eq. 9
                dpsi = psi_p - psi
                assert np.linalg.norm(dpsi) > 1e-6                                          # a real approximation
                ys, xs = bip.window_pixels(e.centre[a], e.W, ny, nx)
                for n in range(e.n_ch):
                    Hfull = ms.embed_window(e.H[n].astype(complex), e.centre[a], ny, nx)
                    lhs = np.linalg.norm(np.fft.fft2(ms.exit_operator(Hfull * dpsi, i, T, P))) / np.sqrt(G)
                    src = np.linalg.norm(e.H[n] * dpsi[np.ix_(ys, xs)])                     # ||H dpsi||_Omega
                    assert abs(lhs - src) <= 1e-12 * src                                    # eq. 16 + 18
                    assert src <= np.abs(e.H[n]).max() * np.linalg.norm(dpsi[np.ix_(ys, xs)]) * (1 + 1e-12)  # eq. 17
                    checked += 1
        S_exact = ms.advance_S1(S_exact, T[i], P)
        S_par = ms.advance_S1(S_par, T[i], P)
    assert checked >= 6


def test_partitioned_probe_full_parent_limit():
    """eq. 20: with every beam its own parent the partitioned probe is the exact PRISM probe term by term."""
    wl = tiny_random_workload(22, ny=16, nx=16)
    ap = ob.beams_in_disc(16, 16, wl.ly, wl.lx, 0.62)
    c = ob.aperture_coefficients(ap, 16, 16, wl.ly, wl.lx, wl.lam, wl.defocus)
    S = ms.build_S1(ap, 16, 16)
    P = ms.fresnel_propagator(16, 16, wl.ly, wl.lx, wl.lam, wl.dz)
    S = ms.advance_S1(S, np.exp(1j * np.angle(wl.T[0].astype(complex))), P)
    rho = np.array([3.5, 9.25])
    psi_p = bip.partitioned_probe_full(S, ap, ap, np.eye(len(ap)), c, rho, 16, 16)
    psi = (bip.illumination(c, ap, rho[None, :], 16, 16) @ S.reshape(len(ap), -1)).reshape(16, 16)
    assert np.abs(psi - psi_p).max() < 1e-13
    # and at plane 0 both are the probe of eq. 1
    S0 = ms.build_S1(ap, 16, 16)
    psi0 = bip.partitioned_probe_full(S0, ap, ap, np.eye(len(ap)), c, rho, 16, 16)
    assert np.abs(psi0 - ms.probe(c, ap, rho, 16, 16)).max() < 1e-13


@pytest.mark.slow
def test_error_falls_with_parent_count():
    """Soft trend: with the magnitude-preserving reconstruction the map error against the
    full-parent (exact) map falls as parents are added, and vanishes in the full-parent limit."""
    wl = make_workload("cfg1", scale=2, nz=6, scan=(4, 4), window=16)
    e = wl.edges[0].take([0, 1, 5, 6])
    ny, nx = wl.ny, wl.nx
    qa, qd = wl.alpha_mrad * 1e-3 / wl.lam, e.det_mrad * 1e-3 / wl.lam
    ap = ob.beams_in_disc(ny, nx, wl.ly, wl.lx, qa)
    det = ob.beams_in_disc(ny, nx, wl.ly, wl.lx, qd)
    c = ob.aperture_coefficients(ap, ny, nx, wl.ly, wl.lx, wl.lam, wl.defocus)
    P = ms.fresnel_propagator(ny, nx, wl.ly, wl.lx, wl.lam, wl.dz)
    T = wl.T.astype(np.complex128)

    def run(n1, n2, recon):
        p1 = ob.hexring_parents(ap, ny, nx, wl.ly, wl.lx, qa, n1) if n1 else np.arange(len(ap))
        p2 = ob.hexring_parents(det, ny, nx, wl.ly, wl.lx, qd, n2) if n2 else np.arange(len(det))
        w1 = osb.to_dense(osb.natural_neighbour_weights(ap, p1, wl.ly, wl.lx, qa), len(p1))
        w2 = osb.to_dense(osb.natural_neighbour_weights(det, p2, wl.ly, wl.lx, qd), len(p2))
        return bip.bip_run(T, P, ap, c, ap[p1], w1, det, det[p2], w2, wl.scan, e.slice, e.centre, e.H, recon=recon)["map"]

    exact = run(0, 0, "linear")
    errs = [np.linalg.norm(run(n, n + 1, "magphase") - exact) / np.linalg.norm(exact) for n in (1, 2, 4)]
    assert errs[0] > errs[1] > errs[2] > 0
    assert errs[2] < 0.1
    lin = np.linalg.norm(run(2, 3, "linear") - exact) / np.linalg.norm(exact)
    assert lin > 0 and np.sum(run(2, 3, "linear")) <= np.sum(run(2, 3, "magphase")) * (1 + 1e-9)   # decoherence loses amplitude
