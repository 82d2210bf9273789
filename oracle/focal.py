"""S1 focal back-propagation to the scattering-centroid plane (section 2.2.3.1) and frozen-phonon averaging
 -- oracle; see oracle/__init__.py.  NEXT-4 of SURVEY.md 8(f).

The paper gives one sentence: "We therefore back-propagate S1 to this centroid plane via a padded-window Fresnel step,
interpolate, and then propagate to the target plane", the plane being "the scattering centroid of the entrance-to-
ionization path".  Neither the centroid nor the padding is defined; the reading taken (DESIGN.md c20) is

  centroid   z_c(i) = sum_{j<i} m_j z_j / sum_{j<i} m_j,  z_j = (j + 1/2) dz the depth of slice j's centre,
             m_j = sum_r |T_j(r) - 1|^2 the scattering strength of the slice (the power a unit plane wave loses from the
             forward beam at that slice); the ionisation plane i is the entrance face of slice i, depth i dz, so the
             back-propagation distance is d_i = i dz - z_c(i) >= 0 (0 when nothing scatters above the site);
  window     the padded window Omega+ of side W_p = 2^ceil(log2(W + 16)) pixels around the atom (at least 8 pixels of
             margin on every side), periodic on itself for the Fresnel step;
  step       the de-tilted parent envelope E_p = S_p exp(-2 pi i h_p.r/N) on Omega+ is carried by the free-space
             transfer function of its own carrier, E_p <- F_w^-1[ exp(+i pi lambda d |q_w + q_p|^2) F_w E_p ]
             (eq. 2 conjugated and shifted by the carrier q_p = (h_y / L_y, h_x / L_x): de-tilting commutes with free
             propagation up to that shift); the envelopes are interpolated there (eq. 15 or eq. 11); every interpolated
             beam envelope is carried forward the same distance with ITS carrier, exp(-i pi lambda d |q_w + q_b|^2),
             re-tilted and cropped to the W x W window.

Properties this reading has by construction (pins in tests/test_oracle_focal.py): with parents = all beams, or with d = 0,
or in vacuum it reproduces the plain reconstruction exactly; the tilted transfer function equals full-grid propagation
(oracle.multislice.propagate) of the tilted column.  PARITY UNPINNED against the paper: its centroid and padding are not
stated and its "2-3x lower on-atom error" was measured on structures that are not available.
"""
import numpy as np
import scipy.sparse as sp

from . import bip


def padded_window(W):
    """Side W_p of the padded window Omega+: the power of two >= W + 16."""
    return 1 << int(np.ceil(np.log2(W + 16)))


def scattering_centroid_distance(T, i, dz):
    """d_i = i dz - z_c(i): distance from the ionisation plane i (entrance face of slice i) back to the scattering centroid
    of slices 0 .. i-1; 0.0 when there is no slice above or none of them scatters."""
    if i <= 0:
        return 0.0
    m = np.array([np.sum(np.abs(T[j].astype(np.complex128) - 1.0) ** 2) for j in range(i)])
    if not np.any(m > 0):
        return 0.0
    z = (np.arange(i) + 0.5) * dz
    return float(i * dz - np.sum(m * z) / np.sum(m))


def propagate_envelopes(E, h, ny, nx, ly, lx, lam, d):
    """Free-space propagation over distance d (d < 0: backwards) of de-tilted envelopes E [n, W_p, W_p] whose carriers are
    the beams h [n, 2]: E <- F_w^-1[ exp(-i pi lam d |q_w + q_h|^2) F_w E ], q_w the frequencies of the window's own DFT."""
    Wp = E.shape[-1]
    qwy = np.fft.fftfreq(Wp, ly / ny)                       # cycles / Angstrom
    qwx = np.fft.fftfreq(Wp, lx / nx)
    out = np.empty_like(E)
    for k in range(E.shape[0]):
        qy = qwy[:, None] + h[k, 0] / ly
        qx = qwx[None, :] + h[k, 1] / lx
        out[k] = np.fft.ifft2(np.exp(-1j * np.pi * lam * d * (qy * qy + qx * qx)) * np.fft.fft2(E[k]))
    return out


def reconstruct_window_focal(S_par, parent_h, beam_h, w, centre, W, ny, nx, ly, lx, lam, d, recon):
    """Windowed reconstruction of the S1 columns with focal back-propagation over distance d: [n_beams, W*W]."""
    Wp = padded_window(W)
    if Wp > min(ny, nx):
        raise ValueError("padded window larger than the grid")
    ys, xs = bip.window_pixels(centre, Wp, ny, nx)                                  # Omega+
    crop = S_par[:, ys][:, :, xs].reshape(S_par.shape[0], -1)
    E = (crop * bip.tilt_phases(parent_h, ys, xs, ny, nx, -1)).reshape(-1, Wp, Wp)  # de-tilted parent envelopes
    E = propagate_envelopes(E, parent_h, ny, nx, ly, lx, lam, -d).reshape(E.shape[0], -1)        # back to the centroid
    w = sp.csr_matrix(w)
    z = w @ E                                                                         # interpolate there (eq. 15)
    if recon == "magphase":
        mag = w @ np.abs(E)
        az = np.abs(z)
        ok = az >= 1e-30
        z = np.where(ok, mag * z / np.where(ok, az, 1.0), 0.0)                       # eq. 11
    elif recon != "linear":
        raise ValueError(recon)
    z = propagate_envelopes(z.reshape(-1, Wp, Wp), beam_h, ny, nx, ly, lx, lam, +d).reshape(z.shape[0], -1)   # forward again
    R = (z * bip.tilt_phases(beam_h, ys, xs, ny, nx, +1)).reshape(-1, Wp, Wp)        # re-tilt
    o = (Wp - W) // 2
    return R[:, o:o + W, o:o + W].reshape(R.shape[0], -1)                            # crop Omega+ -> Omega


def bip_run_focal(T, P, ap_beams, c, p1_h, w1, det_beams, p2_h, w2, scan, sites_slice, sites_centre, H, ly, lx, lam, dz,
                  recon="linear"):
    """Algorithm 5 with the S1 side reconstructed through the scattering-centroid plane; S2 as in bip.bip_run ("focal
    back-propagation is applied to S1 alone")."""
    from . import multislice as ms
    nz, ny, nx = T.shape
    T = T.astype(np.complex128)
    w1 = sp.csr_matrix(w1)
    w2 = sp.csr_matrix(w2)
    A = bip.illumination(c, ap_beams, scan, ny, nx)
    S1 = ms.build_S1(p1_h, ny, nx)
    S2 = ms.build_S2(p2_h, T, P)
    acc = None
    for i in range(nz):
        d = scattering_centroid_distance(T, i, dz)
        for a in np.nonzero(sites_slice == i)[0]:
            R1 = reconstruct_window_focal(S1, p1_h, ap_beams, w1, sites_centre[a], H.shape[1], ny, nx, ly, lx, lam, d, recon)
            amp, _ = bip.atom_amplitudes(S1, S2, p1_h, p2_h, ap_beams, det_beams, w1, w2, A, H.astype(np.complex128),
                                         sites_centre[a], ny, nx, recon, R1=R1)
            r = bip.reduce_modes(amp, det_beams)
            acc = r if acc is None else {k: acc[k] + r[k] for k in acc}
        if i + 1 < nz and np.any(sites_slice > i):
            S1 = ms.advance_S1(S1, T[i], P)
            S2 = ms.peel_S2(S2, T[i], P)
    if acc is None:
        acc = bip.reduce_modes(np.zeros((1, scan.shape[0], det_beams.shape[0]), dtype=np.complex128), det_beams)
    return acc


def frozen_phonon_average(run, T_configs):
    """Frozen-phonon averaging ("thermal diffuse scattering enters only through the frozen-phonon average over
    T_j"): the incoherent mean of the outputs of ``run(T)`` over the displaced configurations."""
    acc = None
    for T in T_configs:
        r = run(T)
        acc = r if acc is None else {k: acc[k] + r[k] for k in acc}
    return {k: v / len(T_configs) for k, v in acc.items()}
