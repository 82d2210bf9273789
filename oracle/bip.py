"""The on-atom contraction of BiP-PRISM, Algorithm 5, step by step (oracle; see oracle/__init__.py).

Notation as in the paper: S1 probe-forming parent columns, S2 adjoint detector parent columns, w^(1), w^(2)
natural-neighbour weights, Omega_tau the W x W window, a_d(rho) detector amplitudes.

Carrier convention (reading c18).  "De-tilt" removes the parent's carrier frequency.
S1 rows carry exp(+2 pi i h.r/N).  With the bilinear S2 of eq. 12 / SURVEY c1 (S2^d = M^T chi*_d, no conjugate
in the pairing) the columns carry exp(-2 pi i h.r/N), i.e. this S2 is the complex conjugate of the Hermitian-
convention column M^dagger chi_d for which eq. 15 is printed; conjugating eq. 15 (the weights are real) gives the
same operation with the conjugate phases.  ``carrier`` = +1 for S1, -1 for S2.
"""
import numpy as np
import scipy.sparse as sp


def window_pixels(centre, W, ny, nx):
    """Global pixel rows / columns of the window: centre - W/2 ... centre + W/2 - 1, periodic."""
    ys = (centre[0] - W // 2 + np.arange(W)) % ny
    xs = (centre[1] - W // 2 + np.arange(W)) % nx
    return ys, xs


def tilt_phases(h, ys, xs, ny, nx, sign):
    """exp(sign 2 pi i h.r/N) on the window for every beam in h: [n, W*W].  Integer products reduced mod N first."""
    fy = ((h[:, 0:1] * ys[None, :]) % ny) / ny            # [n, W]
    fx = ((h[:, 1:2] * xs[None, :]) % nx) / nx            # [n, W]
    ph = fy[:, :, None] + fx[:, None, :]
    return np.exp(sign * 2j * np.pi * ph).reshape(h.shape[0], -1)


def crop_window(S_par, centre, W, ny, nx):
    """S_p | Omega_tau for every parent column: [Bp, W*W]."""
    ys, xs = window_pixels(centre, W, ny, nx)
    return S_par[:, ys][:, :, xs].reshape(S_par.shape[0], -1)


def reconstruct_window(S_par, parent_h, beam_h, w, centre, W, ny, nx, carrier, recon, crop=None):
    """Windowed column reconstruction (eq. 15; eq. 11, PAPER.md:183 for recon="magphase").

    crop the parent columns on Omega_tau -> de-tilt -> NNW-combine to the full beam set -> re-tilt.
    S_par [Bp, ny, nx]; w sparse/dense [n_beams, Bp]; returns R [n_beams, W*W].
    ``crop`` may hand in the already cropped columns [Bp, W*W] (then S_par is not read): large configs keep
    only the windows of the sampled atoms in memory (SURVEY 8(d) "Parity protocol")."""
    ys, xs = window_pixels(centre, W, ny, nx)
    if crop is None:
        crop = crop_window(S_par, centre, W, ny, nx)                          # S_p | Omega
    D = crop * tilt_phases(parent_h, ys, xs, ny, nx, -carrier)                # S_p^dt  (eq. 10)
    z = w @ D                                                                 # sum_p w_{b,p} S_p^dt
    if recon == "linear":
        R = z
    elif recon == "magphase":
        mag = w @ np.abs(D)                                                   # sum_p w |S_p^dt|
        az = np.abs(z)
        ok = az >= 1e-30
        R = np.where(ok, mag * z / np.where(ok, az, 1.0), 0.0)                # eq. 11
    else:
        raise ValueError(recon)
    return R * tilt_phases(beam_h, ys, xs, ny, nx, +carrier)                  # re-tilt


def illumination(c, beams, scan, ny, nx):
    """c_b(rho) = Psi(h_b) exp(-2 pi i h_b.rho/N): [n_rho, B]."""
    ph = scan[:, 0:1] * beams[None, :, 0] / ny + scan[:, 1:2] * beams[None, :, 1] / nx
    return c[None, :] * np.exp(-2j * np.pi * ph)


def atom_amplitudes(S1, S2, p1_h, p2_h, ap_beams, det_beams, w1, w2, A, H, centre, ny, nx, recon, crops=None, R1=None):
    """Steps a1-a7 for one ionised atom: amplitudes a[n, rho, d] (eq. 13 in the probe-first association).
    ``R1`` may hand in the reconstructed S1 window [B, W*W] (oracle.focal reconstructs it through the scattering-centroid
    plane); everything after the reconstruction is unchanged.

    Psi[rho, s] = sum_b c_b(rho) S1^b|Omega (eq. 7 on the window);  Phi_n = H_n . Psi (eq. 3);
    a_d = G^-1/2 sum_s S2^d|Omega[s] Phi_n[s]  (eq. 12-13, unitary F: SURVEY c3)."""
    W = H.shape[1]
    c1, c2 = crops if crops is not None else (None, None)
    if R1 is None:
        R1 = reconstruct_window(S1, p1_h, ap_beams, w1, centre, W, ny, nx, +1, recon, c1)     # [B, W^2]
    R2 = reconstruct_window(S2, p2_h, det_beams, w2, centre, W, ny, nx, -1, recon, c2)    # [K, W^2]
    Psi = A @ R1                                                                       # [n_rho, W^2]
    a = np.empty((H.shape[0], A.shape[0], det_beams.shape[0]), dtype=np.complex128)
    for n in range(H.shape[0]):
        Phi = Psi * H[n].reshape(1, -1)
        a[n] = (Phi @ R2.T) / np.sqrt(float(ny * nx))
    return a, Psi


def atom_amplitudes_coupling(S1, S2, p1_h, p2_h, ap_beams, det_beams, w1, w2, A, H, centre, ny, nx, recon, crops=None):
    """The other association of the same triple product (eq. 13; Alg. 4 lines 6-8):
    first the scan-independent transition coupling matrix of the site and channel,

        M^{(n,tau)}_{d,b} = sum_{r in Omega_tau} S2^d(r) H_n(r - tau) S1^b(r)        [K, B]

    then a_d(rho) = G^-1/2 sum_b M_{d,b} c_b(rho) for all scan positions at once.  Returns a[n, rho, d]."""
    W = H.shape[1]
    c1, c2 = crops if crops is not None else (None, None)
    R1 = reconstruct_window(S1, p1_h, ap_beams, w1, centre, W, ny, nx, +1, recon, c1)     # S1^b | Omega   [B, W^2]
    R2 = reconstruct_window(S2, p2_h, det_beams, w2, centre, W, ny, nx, -1, recon, c2)    # S2^d | Omega   [K, W^2]
    a = np.empty((H.shape[0], A.shape[0], det_beams.shape[0]), dtype=np.complex128)
    for n in range(H.shape[0]):
        M = (R2 * H[n].reshape(1, -1)) @ R1.T                                             # [K, B]
        a[n] = (A @ M.T) / np.sqrt(float(ny * nx))
    return a


def qeels_bins(det_beams, axis):
    """Distinct signed beam indices along the resolved axis, ascending. axis 1 = x, 0 = y."""
    return np.unique(det_beams[:, axis])


def reduce_modes(a, det_beams):
    """Output modes as reductions of |a_d|^2 over d (section 2.2.6), summed over channels.
    Returns dict(map [n_rho], qeels_x [n_rho, nbx], qeels_y [n_rho, nby], cube [n_rho, K])."""
    cube = np.sum(np.abs(a) ** 2, axis=0)                                 # sum over channels n
    out = {"cube": cube, "map": cube.sum(axis=1)}
    for name, axis in (("qeels_x", 1), ("qeels_y", 0)):
        bins = qeels_bins(det_beams, axis)
        q = np.zeros((cube.shape[0], bins.shape[0]))
        for j, hv in enumerate(bins):
            q[:, j] = cube[:, det_beams[:, axis] == hv].sum(axis=1)
        out[name] = q
    return out


def bip_run(T, P, ap_beams, c, p1_h, w1, det_beams, p2_h, w2, scan, sites_slice, sites_centre, H,
            recon="linear", want_psi=False, crop_f=None, association="probe"):
    """Algorithm 5: build S1 / S2 on the parents, then for every ionisation plane with >= 1
    site ADVANCETO / PEELTO and run the on-atom contraction for every site and channel, accumulating the outputs.
    T complex [nz, ny, nx]; weights w1 [B, Bp1], w2 [K, Bp2] (dense or scipy.sparse).  Returns the dict of
    reduce_modes() summed over sites (eq. 14).  ``crop_f`` = (f_y, f_x) applies the PRISM crop mask:
    a site contributes only to the scans of beams.crop_mask()."""
    from . import multislice as ms
    from . import beams as ob
    nz, ny, nx = T.shape
    T = T.astype(np.complex128)
    w1 = sp.csr_matrix(w1)
    w2 = sp.csr_matrix(w2)
    A = illumination(c, ap_beams, scan, ny, nx)
    S1 = ms.build_S1(p1_h, ny, nx)                    # plane 0
    S2 = ms.build_S2(p2_h, T, P)                      # plane 0 (all slices still inside)
    K = det_beams.shape[0]
    acc = None
    psis = []
    for i in range(nz):
        for a_idx in np.nonzero(sites_slice == i)[0]:
            if association == "coupling":                # eq. 13 as printed: M first, then all scans (NEXT-2)
                a, Psi = atom_amplitudes_coupling(S1, S2, p1_h, p2_h, ap_beams, det_beams, w1, w2, A,
                                                  H.astype(np.complex128), sites_centre[a_idx], ny, nx, recon), None
            else:
                a, Psi = atom_amplitudes(S1, S2, p1_h, p2_h, ap_beams, det_beams, w1, w2, A,
                                         H.astype(np.complex128), sites_centre[a_idx], ny, nx, recon)
            r = reduce_modes(a, det_beams)
            if crop_f is not None:
                inside = ob.crop_mask(scan, sites_centre[a_idx], ny, nx, crop_f[0], crop_f[1])
                r = {k: v * (inside[:, None] if v.ndim == 2 else inside) for k, v in r.items()}
            acc = r if acc is None else {k: acc[k] + r[k] for k in acc}
            if want_psi:
                psis.append(Psi)
        if i + 1 < nz and np.any(sites_slice > i):
            S1 = ms.advance_S1(S1, T[i], P)           # wave entering slice i+1
            S2 = ms.peel_S2(S2, T[i], P)              # slices i+1 .. nz-1 remain
    if acc is None:
        acc = reduce_modes(np.zeros((1, scan.shape[0], K), dtype=np.complex128), det_beams)
    if want_psi:
        acc["psi"] = psis
    return acc


def partitioned_probe_full(S1, p1_h, ap_beams, w1, c, rho, ny, nx, recon="linear"):
    """The partitioned probe on the FULL grid (Alg. 3 probe synthesis, eq. 9-10 written as reconstruct-then-sum):
    psi^p(r, rho) = sum_b c_b(rho) [re-tilt_b sum_p w_{b,p} S_p^dt](r).  Used only by the locality pin."""
    R1 = reconstruct_window(S1, p1_h, ap_beams, sp.csr_matrix(w1), (ny // 2, nx // 2), ny, ny, nx, +1, recon) \
        if ny == nx else None
    if R1 is None:
        raise ValueError("locality pin uses square grids")
    # reconstruct_window returns rows over the window starting at centre - W/2 = 0: identity pixel order
    A = illumination(c, ap_beams, np.asarray([rho], dtype=np.float64), ny, nx)
    return (A @ R1).reshape(ny, nx)
