"""Algorithm 3 of the paper: partitioned PRISM-EELS, S1 only, per-scan exit multislice -- the energy-filtered 4D cube on ALL
exit beams (oracle; see oracle/__init__.py).  PAPER.md:188-201 (Algorithm 3), 159-169 (eq. 9-10), Table 1.

Steps, in the paper's order and notation:

  build        {h_p} hex-ring parents, w natural-neighbour weights, S_p <- F^-1[delta_{h_p}]            (lines 1-3)
  per plane i  ADVANCETO(i): eq. 6 on the B_p parent columns                                             (line 4)
               S_p^dt <- S_p exp(-2 pi i h_p.r/N);  spectrum_p[h_b] <- w_{p,b} Psi(h_b)                  (line 5)
               psi(., rho) <- sum_p F^-1[spectrum_p exp(-2 pi i q.rho/N)] S_p^dt   (general, sub-pixel path;
               for integer rho this is the roll of psi^_p(., 0), the same numbers)                      (lines 6-10)
               for every site of the plane and channel n:  psi_n = H_n0(r - tau) psi  (eq. 3),
               carried to the exit surface by conventional multislice, |F psi_n|^2 accumulated          (line 11 = Alg. 1 l. 5-8)

With recon="magphase" the probe is instead the sum over beams of the eq. 11 columns (magnitude-preserving
reconstruction, "applied to both S1 and S2"); eq. 11 is not linear in the parents, so it has no
beamlet-basis form and is evaluated beam by beam (oracle.bip.reconstruct_window on the whole grid).

Output: I[rho, ky, kx] on the corner-origin DFT grid, every one of the G exit beams (unitary F: sum over (ky, kx) of
I[rho] = sum_n ||H_n psi||^2).

Pins (tests/test_oracle_alg3.py): equals Algorithm 1 with parents = all beams (brute force); the beamlet form equals
reconstruct-then-sum (eq. 9-10 vs eq. 15 + eq. 7); summed over exit beams it equals sum |H_n psi|^2 on the window;
restricted to the detector beams and with an exact S2 it equals Algorithm 5's cube.
"""
import numpy as np
import scipy.sparse as sp

from . import bip
from . import multislice as ms


def beamlet_spectra(w, c, ap_beams, ny, nx):
    """spectrum_p[h_b] <- w_{p,b} Psi(h_b) on the beam grid (Alg. 3 line 5; eq. 10): [B_p, ny, nx].
    ``w`` is [B, B_p] (row b = beam, as everywhere in the oracle: w[b, p] = w_{p,b} of eq. 8)."""
    w = sp.csr_matrix(w).toarray()
    spec = np.zeros((w.shape[1], ny, nx), dtype=np.complex128)
    ky, kx = ap_beams[:, 0] % ny, ap_beams[:, 1] % nx
    for p in range(w.shape[1]):
        spec[p, ky, kx] = w[:, p] * c
    return spec


def beamlet_probe(S_par, parent_h, spec, rho, ny, nx):
    """psi(., rho) = sum_p F^-1[spectrum_p exp(-2 pi i q.rho/N)] S_p^dt (eq. 9-10; Alg. 3 line 9).
    F^-1 here is the plain synthesis sum_h spectrum[h] exp(+2 pi i h.r/N) (no 1/G: eq. 1 / eq. 10 are sums over beams)."""
    hy = np.fft.fftfreq(ny, 1.0 / ny)[:, None]
    hx = np.fft.fftfreq(nx, 1.0 / nx)[None, :]
    ramp = np.exp(-2j * np.pi * (hy * rho[0] / ny + hx * rho[1] / nx))
    psi = np.zeros((ny, nx), dtype=np.complex128)
    for p in range(S_par.shape[0]):
        beamlet = np.fft.ifft2(spec[p] * ramp) * (ny * nx)                     # psi^_p(r, rho)
        S_dt = S_par[p] * ms.plane_wave(parent_h[p], ny, nx, -1)                # de-tilt (eq. 10)
        psi += beamlet * S_dt
    return psi


def reconstructed_probe(S_par, parent_h, ap_beams, w, c, rho, ny, nx, recon):
    """The partitioned probe on the whole grid as reconstruct-then-sum: every aperture beam's column from the de-tilted
    parents (eq. 15, or eq. 11 for recon="magphase"), re-tilted, then eq. 7.  For recon="linear" this is the same number
    as beamlet_probe (eq. 9-10 only regroups the double sum)."""
    ys, xs = np.arange(ny), np.arange(nx)
    D = S_par.reshape(S_par.shape[0], -1) * bip.tilt_phases(parent_h, ys, xs, ny, nx, -1)        # S_p^dt
    w = sp.csr_matrix(w)
    z = w @ D
    if recon == "magphase":
        mag = w @ np.abs(D)
        az = np.abs(z)
        ok = az >= 1e-30
        z = np.where(ok, mag * z / np.where(ok, az, 1.0), 0.0)                                   # eq. 11
    R = z * bip.tilt_phases(ap_beams, ys, xs, ny, nx, +1)                                        # re-tilt
    A = bip.illumination(c, ap_beams, np.asarray([rho], dtype=np.float64), ny, nx)
    return (A @ R).reshape(ny, nx)


def alg3_cube(T, P, ap_beams, c, parent_pos, w, scan, sites_slice, sites_centre, H, recon="linear"):
    """Algorithm 3 end to end.  T [nz, ny, nx] complex; w [B, B_p] dense or sparse; returns I[n_rho, ny, nx] float64."""
    nz, ny, nx = T.shape
    G = ny * nx
    T = T.astype(np.complex128)
    parent_h = ap_beams[parent_pos]
    spec = beamlet_spectra(w, c, ap_beams, ny, nx) if recon == "linear" else None
    S = ms.build_S1(parent_h, ny, nx)                                          # line 3
    I = np.zeros((scan.shape[0], ny, nx))
    for i in range(nz):
        here = np.nonzero(sites_slice == i)[0]
        if here.size:
            for si in range(scan.shape[0]):
                if recon == "linear":
                    psi = beamlet_probe(S, parent_h, spec, scan[si], ny, nx)   # lines 5-10
                else:
                    psi = reconstructed_probe(S, parent_h, ap_beams, w, c, scan[si], ny, nx, recon)
                for a in here:
                    for n in range(H.shape[0]):
                        psi_n = ms.embed_window(H[n].astype(np.complex128), sites_centre[a], ny, nx) * psi     # eq. 3
                        ex = np.fft.fft2(ms.exit_operator(psi_n, i, T, P)) / np.sqrt(G)                        # Alg. 1 l. 6-7
                        I[si] += np.abs(ex) ** 2
        if i + 1 < nz and np.any(sites_slice > i):
            S = ms.advance_S1(S, T[i], P)                                      # line 4 for the next plane
    return I
