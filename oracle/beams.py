"""Beam sets, probe coefficients and hex-ring parent selection (oracle; see oracle/__init__.py)."""
import math

import numpy as np


def flat_index(h, ny, nx):
    """Corner-origin flat DFT index of signed beam h = (hy, hx): (hy mod ny) * nx + (hx mod nx)."""
    h = np.asarray(h)
    return (h[..., 0] % ny) * nx + (h[..., 1] % nx)


def beams_in_disc(ny, nx, ly, lx, qmax):
    """All integer beams with |h| < N/2 and q_y^2 + q_x^2 <= qmax^2, q = (hy/ly, hx/lx), in ascending flat
    corner-origin index (eq. 5 / Alg. 4 line 1; inclusion and order: SURVEY c5).
    Returns int64 [n, 2] signed (hy, hx)."""
    out = []
    for ky in range(ny):
        hy = ky if ky < (ny + 1) // 2 else ky - ny
        if 2 * abs(hy) >= ny:
            continue
        for kx in range(nx):
            hx = kx if kx < (nx + 1) // 2 else kx - nx
            if 2 * abs(hx) >= nx:
                continue
            qy = hy / ly
            qx = hx / lx
            if qy * qy + qx * qx <= qmax * qmax:
                out.append((hy, hx))
    return np.asarray(out, dtype=np.int64).reshape(-1, 2)


def prism_subsample(beams, fy, fx):
    """PRISM beam subsampling (Alg. 2 line 1): keep h with h_y = 0 (mod f_y) and
    h_x = 0 (mod f_x).  Returns the positions into ``beams`` (ascending, so the flat-index order is kept)."""
    keep = (beams[:, 0] % fy == 0) & (beams[:, 1] % fx == 0)
    return np.nonzero(keep)[0]


def prism_coefficients(c_full, keep, fy, fx):
    """Coefficients of the retained beams, rescaled by f_y f_x, "the DFT decimation factor": the
    synthesised probe is then the exact probe replicated with period (N_y / f_y, N_x / f_x)."""
    return c_full[keep] * float(fy * fx)


def crop_mask(scan, centre, ny, nx, fy, fx):
    """PRISM crop mask: the scans inside the atom's 1/f window, i.e. whose periodic distance from the
    atom's pixel is below half the alias-free period, |rho - tau| < N / (2 f) on both axes (reading c19).
    scan [n_rho, 2] in pixels; returns bool [n_rho]."""
    dy = (scan[:, 0] - centre[0] + ny / 2.0) % ny - ny / 2.0
    dx = (scan[:, 1] - centre[1] + nx / 2.0) % nx - nx / 2.0
    return (np.abs(dy) < ny / (2.0 * fy)) & (np.abs(dx) < nx / (2.0 * fx))


def aperture_coefficients(beams, ny, nx, ly, lx, lam, defocus):
    """c_b = Psi(h_b) = exp(-i pi lam df |q_b|^2) / sqrt(G B): pure-defocus lens phase inside the aperture,
    probe normalised to sum_r |psi_0|^2 = 1 (eq. 1)."""
    qy = beams[:, 0] / ly
    qx = beams[:, 1] / lx
    q2 = qy * qy + qx * qx
    return np.exp(-1j * np.pi * lam * defocus * q2) / np.sqrt(float(ny * nx) * beams.shape[0])


def n_radial_from_factor(n_beams, factor):
    """parent spacing f in beam pixels -> n_radial = max(1, round(sqrt(B / pi) / f))."""
    return max(1, int(np.floor(np.sqrt(n_beams / np.pi) / factor + 0.5)))


def hexring_parents(beams, ny, nx, ly, lx, qmax, n_radial, n_angular=6):
    """Hex-ring parent selection (geometry: SURVEY c6).

    DC beam plus rings k = 1..n_radial at |q| = k qmax / n_radial with n_angular * k samples at angles
    2 pi j / (n_angular k) from +x; each sample snapped to the nearest member of ``beams`` in physical q
    distance (ties -> lowest flat index); deduplicated; returned as ascending positions into ``beams``
    (``beams`` is in ascending flat index, so this is also ascending flat index)."""
    qy = beams[:, 0] / ly
    qx = beams[:, 1] / lx
    flat = flat_index(beams, ny, nx)

    def snap(sy, sx):
        d2 = (qy - sy) * (qy - sy) + (qx - sx) * (qx - sx)
        best = np.nonzero(d2 == d2.min())[0]
        return int(best[np.argmin(flat[best])])

    chosen = {snap(0.0, 0.0)}
    for k in range(1, n_radial + 1):
        r = k * qmax / n_radial
        m = n_angular * k
        for j in range(m):
            ang = 2.0 * math.pi * j / m
            chosen.add(snap(r * math.sin(ang), r * math.cos(ang)))
    return np.asarray(sorted(chosen), dtype=np.int64)
