"""Multislice, scattering-matrix builds and the ground-truth Algorithm 1 (oracle; see oracle/__init__.py).

Conventions: ``F`` is NumPy's unnormalised forward DFT on the corner-origin grid;
the *unitary* transform of PAPER.md:312 is F / sqrt(G) (c3).  No band-limit (c13).  Beam h = (hy, hx)
signed; pixel r = (ry, rx); h.r/N = hy ry / ny + hx rx / nx.
"""
import numpy as np
from scipy import fft as _fft


def fresnel_propagator(ny, nx, ly, lx, lam, dz):
    """P(q) = exp(-i pi lam dz |q|^2) on the corner-origin grid (eq. 2)."""
    hy = np.fft.fftfreq(ny, 1.0 / ny)
    hx = np.fft.fftfreq(nx, 1.0 / nx)
    qy = hy / ly
    qx = hx / lx
    q2 = qy[:, None] ** 2 + qx[None, :] ** 2
    return np.exp(-1j * np.pi * lam * dz * q2)


def propagate(psi, P):
    """Fresnel operator: F^-1[P . F psi] (eq. 2) on the last two axes (library FFT; stacks of columns are
    transformed together, one thread per column)."""
    return _fft.ifft2(P * _fft.fft2(psi, workers=-1), workers=-1)


def slice_step(psi, T_j, P):
    """One multislice step through slice j: transmit then propagate, psi -> P(T_j psi) (eq. 6)."""
    return propagate(T_j * psi, P)


def plane_wave(h, ny, nx, sign=+1):
    """exp(sign 2 pi i h.r/N), amplitude exactly 1 (unit plane wave F^-1[delta_h])."""
    ry = np.arange(ny)[:, None]
    rx = np.arange(nx)[None, :]
    # reduce the integer products mod N before dividing: exact phases
    ph = ((h[0] * ry) % ny) / ny + ((h[1] * rx) % nx) / nx
    return np.exp(sign * 2j * np.pi * ph)


def exit_operator(psi, i, T, P):
    """M_{i->exit}: transmit-and-propagate through slices i .. nz-1."""
    for j in range(i, T.shape[0]):
        psi = slice_step(psi, T[j], P)
    return psi


def probe(c, beams, rho, ny, nx):
    """psi_0(r, rho) = sum_b c_b exp(-2 pi i h_b.rho/N) exp(2 pi i h_b.r/N) (eq. 1)."""
    psi = np.zeros((ny, nx), dtype=np.complex128)
    for b in range(beams.shape[0]):
        ramp = np.exp(-2j * np.pi * (beams[b, 0] * rho[0] / ny + beams[b, 1] * rho[1] / nx))
        psi += c[b] * ramp * plane_wave(beams[b], ny, nx, +1)
    return psi


def build_S1(parent_h, ny, nx):
    """S1 rows at plane 0: unit plane waves exp(+2 pi i h_p.r/N) (Alg. 2 line 2 / Alg. 3 line 3)."""
    return np.stack([plane_wave(h, ny, nx, +1) for h in parent_h])


def advance_S1(S1, T_i, P):
    """ADVANCETO by one slice: S_b <- P(T_i S_b) on every row (eq. 6).
    After advancing through slices 0..i-1 the rows are the waves entering slice i."""
    return slice_step(S1, T_i, P)


def build_S2(parent_h, T, P):
    """S2 columns at plane 0 (eq. 12; reading SURVEY c1).

    S2^d := M^T chi*_d so that sum_r S2^d(r) w(r) = [F M_{i->exit} w]_{h_d} with NO conjugation in the pairing:
    start from the conjugate detector plane wave exp(-2 pi i h_d.r/N) at the exit surface and apply
    u <- T_j . P[u] for j = nz-1 .. 0 (transpose of transmit-then-propagate; P^T = P since P(q) is even)."""
    return build_S2_at(parent_h, T, P, 0)


def build_S2_at(parent_h, T, P, i):
    """S2 at plane i built directly from the exit surface (contains slices i .. nz-1)."""
    ny, nx = T.shape[1:]
    u = np.stack([plane_wave(h, ny, nx, -1) for h in parent_h])
    for j in range(T.shape[0] - 1, i - 1, -1):
        u = T[j] * propagate(u, P)
    return u


def peel_S2(S2, T_i, P):
    """PEELTO by one slice: S2^(i+1) = P*[T_i* . S2^(i)], exact because |T| = 1."""
    Pc = np.conj(P)
    return propagate(np.conj(T_i) * S2, Pc)


def embed_window(Hwin, centre, ny, nx):
    """H_n0(r - tau) on the full grid: the W x W window placed with Hwin[W/2, W/2] on the atom's pixel,
    periodic wrap, zero elsewhere (eq. 3)."""
    W = Hwin.shape[0]
    full = np.zeros((ny, nx), dtype=np.complex128)
    for sy in range(W):
        for sx in range(W):
            full[(centre[0] - W // 2 + sy) % ny, (centre[1] - W // 2 + sx) % nx] = Hwin[sy, sx]
    return full


def conventional_cube(c, beams, T, P, scan, sites_slice, sites_centre, H, det_beams):
    """Algorithm 1, the ground truth: per scan position form the probe (eq. 1), walk the slices,
    at every site/channel spawn H psi (eq. 3), carry it to the exit (M_{i->exit}), unitary-Fourier-transform it
    and accumulate |.|^2 on the detector beams (eq. 4).  Returns I[rho, d] float64."""
    nz, ny, nx = T.shape
    G = ny * nx
    ky = det_beams[:, 0] % ny
    kx = det_beams[:, 1] % nx
    I = np.zeros((scan.shape[0], det_beams.shape[0]))
    for si in range(scan.shape[0]):
        psi = probe(c, beams, scan[si], ny, nx)
        for i in range(nz):
            for a in range(sites_slice.shape[0]):
                if sites_slice[a] != i:
                    continue
                for n in range(H.shape[0]):
                    psi_n = embed_window(H[n], sites_centre[a], ny, nx) * psi
                    ex = np.fft.fft2(exit_operator(psi_n, i, T, P)) / np.sqrt(G)
                    I[si] += np.abs(ex[ky, kx]) ** 2
            psi = slice_step(psi, T[i], P)
    return I
