"""Synthetic specimens shaped like the paper's workloads (BASELINE.json ``configs``).

The paper's own structures (FePt nanoparticle of Brown et al. 2019, LaAlO3/SrTiO3
film, SrTiO3 slabs) and its hydrogenic / GPAW transition potentials
 are not available here; these seeded stand-ins take their
shapes.  Everything returned is *data*: complex64 transmission
functions, complex64 ``H_n`` windows, int32 sites, float64 scan positions.

Recipe (one PCG64 stream per config, ``default_rng(75600 + k)``, draws in this order):
  1. in-plane jitter of every atom, if the config has jitter (atom order = slice, row, column);
  2. for each edge in order: ``A_n ~ U(0.5,1)``, ``sigma_n ~ U(W/12, W/8)`` px,
     ``phi_n ~ U(0, 2 pi)`` (three vectors of length N_ch), then, for the
     ``h_kind="iid"`` parity variant only, a ``W x W`` field of phases per channel.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

from .physics import electron_wavelength, interaction_constant

GAUSS_SIGMA_A = 0.3       # width of the projected atomic potential / Angstrom
GAUSS_AMP_PER_Z = 0.5     # peak of the projected potential per unit Z / (V Angstrom)


@dataclasses.dataclass
class Edge:
    name: str
    slice: np.ndarray      # int32 [n_atoms], ascending
    centre: np.ndarray     # int32 [n_atoms, 2]  (py, px) pixel the atom sits on
    H: np.ndarray          # complex64 [n_ch, W, W]; H[n, W/2, W/2] is on the atom's pixel
    det_mrad: float

    @property
    def n_atoms(self) -> int:
        return int(self.slice.shape[0])

    @property
    def n_ch(self) -> int:
        return int(self.H.shape[0])

    @property
    def W(self) -> int:
        return int(self.H.shape[1])

    def take(self, idx: Sequence[int]) -> "Edge":
        idx = np.asarray(idx, dtype=np.int64)
        order = np.argsort(self.slice[idx], kind="stable")
        idx = idx[order]
        return dataclasses.replace(self, slice=self.slice[idx].copy(), centre=self.centre[idx].copy())

    def first_planes(self, n_atoms: int) -> "Edge":
        """The first ``n_atoms`` sites in depth order (used for sampled bench / parity steps)."""
        return self.take(np.arange(min(n_atoms, self.n_atoms)))


@dataclasses.dataclass
class Workload:
    name: str
    ny: int
    nx: int
    ly: float              # Angstrom
    lx: float
    nz: int
    dz: float              # Angstrom
    kv: float
    lam: float             # Angstrom
    sigma: float           # rad / (V Angstrom)
    alpha_mrad: float
    defocus: float         # Angstrom; <0 focuses |df| below the entrance surface
    parent_factor: Tuple[float, float]   # (S1, S2) parent spacing in beam pixels
    T: np.ndarray          # complex64 [nz, ny, nx]
    scan: np.ndarray       # float64 [n_rho, 2] (py, px) in pixels
    scan_shape: Tuple[int, int]
    edges: List[Edge]
    prism: Tuple[int, int] = (1, 1)      # PRISM beam subsampling (f_y, f_x) of aperture and detector sets
    crop: Tuple[int, int] = (1, 1)       # PRISM crop mask factors; (1, 1) = no mask

    @property
    def n_rho(self) -> int:
        return int(self.scan.shape[0])


def _gauss_1d(n: int, length: float, centres: np.ndarray) -> np.ndarray:
    """Minimum-image periodic Gaussian profiles, [n_atoms, n]."""
    coords = np.arange(n, dtype=np.float64) * (length / n)
    d = coords[None, :] - centres[:, None]
    d = (d + 0.5 * length) % length - 0.5 * length
    return np.exp(-(d * d) / (2.0 * GAUSS_SIGMA_A ** 2))


def transmission_functions(ny, nx, ly, lx, nz, sigma, atoms_z, atoms_y, atoms_x, atoms_slice) -> np.ndarray:
    """T_j = exp(i sigma V_j), V_j = sum of Gaussian projected potentials of the slice's atoms,
    rounded to complex64 (SURVEY §8(d) "Common")."""
    T = np.empty((nz, ny, nx), dtype=np.complex64)
    for j in range(nz):
        sel = np.nonzero(atoms_slice == j)[0]
        if sel.size == 0:
            T[j] = 1.0
            continue
        gy = _gauss_1d(ny, ly, atoms_y[sel]) * (GAUSS_AMP_PER_Z * atoms_z[sel])[:, None]
        gx = _gauss_1d(nx, lx, atoms_x[sel])
        V = gy.T @ gx
        T[j] = np.exp(1j * sigma * V).astype(np.complex64)
    return T


def transition_windows(rng: np.random.Generator, n_ch: int, W: int, h_kind: str = "vortex") -> np.ndarray:
    """Synthetic H_n[s] = A_n exp(-|s-c|^2/(2 sigma_n^2)) exp(i (phi_n + m_n atan2(y, x))), c = (W/2, W/2)."""
    A = rng.uniform(0.5, 1.0, n_ch)
    sg = rng.uniform(W / 12.0, W / 8.0, n_ch)
    phi = rng.uniform(0.0, 2.0 * math.pi, n_ch)
    y = np.arange(W, dtype=np.float64)[:, None] - W / 2
    x = np.arange(W, dtype=np.float64)[None, :] - W / 2
    H = np.empty((n_ch, W, W), dtype=np.complex128)
    for n in range(n_ch):
        m = n - n_ch // 2
        phase = phi[n] + m * np.arctan2(y, x)
        if h_kind == "iid":
            phase = rng.uniform(0.0, 2.0 * math.pi, (W, W))
        H[n] = A[n] * np.exp(-(y * y + x * x) / (2.0 * sg[n] ** 2)) * np.exp(1j * phase)
    return H.astype(np.complex64)


def snap_sites(y_a, x_a, z_a, ny, nx, ly, lx, nz, dz):
    """centre = floor(tau / pixel + 0.5) mod N ; slice = min(nz-1, floor(z / dz))."""
    py = np.floor(y_a / (ly / ny) + 0.5).astype(np.int64) % ny
    px = np.floor(x_a / (lx / nx) + 0.5).astype(np.int64) % nx
    sl = np.minimum(nz - 1, np.floor(z_a / dz).astype(np.int64))
    return sl.astype(np.int32), np.stack([py, px], axis=1).astype(np.int32)


def _perovskite(cells_y, cells_x, cells_z, a, ZA_of_col, ZB_of_col, ZO):
    """ABO3 on a cubic lattice, two slices per cell: AO plane (A at (0,0), O at (1/2,1/2)) then BO2 plane
    (B at (1/2,1/2), O at (1/2,0) and (0,1/2)); planes sit at slice centres.
    Returns arrays Z, y, x, z(Angstrom), slice, tag ('A'/'B'/'O' as 0/1/2), column index ix."""
    Z, Y, X, S, TAG, COL = [], [], [], [], [], []
    for kz in range(cells_z):
        for plane in (0, 1):
            sl = 2 * kz + plane
            for iy in range(cells_y):
                for ix in range(cells_x):
                    if plane == 0:
                        sites = ((ZA_of_col(ix), 0.0, 0.0, 0), (ZO, 0.5, 0.5, 2))
                    else:
                        sites = ((ZB_of_col(ix), 0.5, 0.5, 1), (ZO, 0.5, 0.0, 2), (ZO, 0.0, 0.5, 2))
                    for z_, fy, fx, tag in sites:
                        Z.append(z_); Y.append((iy + fy) * a); X.append((ix + fx) * a)
                        S.append(sl); TAG.append(tag); COL.append(ix)
    f = lambda v, t: np.asarray(v, dtype=t)
    return f(Z, np.float64), f(Y, np.float64), f(X, np.float64), f(S, np.int32), f(TAG, np.int32), f(COL, np.int32)


def _fept_sphere(cell_y, cell_x, cell_z, radius, a, c):
    """FePt L1_0 (Fe at (0,0,0), (1/2,1/2,0); Pt at (1/2,0,1/2), (0,1/2,1/2); a = b, c along the beam), the lattice
    sites within ``radius`` of the cell centre.  The lattice is placed so that no atomic plane sits on a slice
    boundary: planes are c/2 = 1.855 A apart against 2 A slices, and with the centre plane 1.505 A above the cell's
    mid-height every plane within the sphere stays >= 0.04 A away from a boundary (c11 then assigns slices safely).
    Returns Z, y, x, z (Angstrom) and tag (0 = Fe, 1 = Pt)."""
    cy, cx, cz = 0.5 * cell_y, 0.5 * cell_x, 0.5 * cell_z + 1.505
    n = int(math.ceil(radius / min(a, c))) + 1
    Z, Y, X, Zc, TAG = [], [], [], [], []
    basis = ((26, 0.0, 0.0, 0.0, 0), (26, 0.5, 0.5, 0.0, 0), (78, 0.5, 0.0, 0.5, 1), (78, 0.0, 0.5, 0.5, 1))
    for kz in range(-n, n + 1):
        for ky in range(-n, n + 1):
            for kx in range(-n, n + 1):
                for z_, fy, fx, fz, tag in basis:
                    dy, dx, dz_ = (ky + fy) * a, (kx + fx) * a, (kz + fz) * c
                    if dy * dy + dx * dx + dz_ * dz_ <= radius * radius:
                        Z.append(z_); Y.append(cy + dy); X.append(cx + dx); Zc.append(cz + dz_); TAG.append(tag)
    f = lambda v, t: np.asarray(v, dtype=t)
    return f(Z, np.float64), f(Y, np.float64), f(X, np.float64), f(Zc, np.float64), f(TAG, np.int32)


def _make_fept(name, rc, scale, nz, scan, parent_factor, h_kind, window) -> Workload:
    """BASELINE.json configs[3] in the paper's own regime (PRISM f, crop mask: "4-prism" of SURVEY 8(d))."""
    gy, gx = rc["grid"]
    if gy % scale or gx % scale:
        raise ValueError("scale must divide the grid")
    gy, gx = gy // scale, gx // scale
    ly, lx, lz = rc["cell"][0] / scale, rc["cell"][1] / scale, rc["cell"][2]
    dz = rc["dz"]
    nz_full = int(round(lz / dz))
    nz_use = nz_full if nz is None else int(nz)
    if not 1 <= nz_use <= nz_full:
        raise ValueError("nz out of range")
    kv = rc["kv"]
    lam, sigma = electron_wavelength(kv), interaction_constant(kv)
    rng = np.random.default_rng(rc["seed"])
    Z, Y, X, Zc, TAG = _fept_sphere(ly, lx, lz, rc["radius"] / scale, rc["a"], rc["c"])
    S = np.minimum(nz_full - 1, np.floor(Zc / dz).astype(np.int64)).astype(np.int32)     # c11
    keep = S < nz_use
    Z, Y, X, Zc, TAG, S = Z[keep], Y[keep], X[keep], Zc[keep], TAG[keep], S[keep]
    T = transmission_functions(gy, gx, ly, lx, nz_use, sigma, Z, Y, X, S)
    edges = []
    for e in rc["edges"]:
        idx = np.nonzero(TAG == e["tag"])[0]
        sl, centre = snap_sites(Y[idx], X[idx], Zc[idx], gy, gx, ly, lx, nz_use, dz)
        W = int(window) if window is not None else e["W"]
        H = transition_windows(rng, e["n_ch"], W, h_kind)
        order = np.argsort(sl, kind="stable")
        edges.append(Edge(e["name"], sl[order], centre[order], H, e["det"]))
    sy, sx = scan if scan is not None else (max(1, rc["scan"][0] // scale), max(1, rc["scan"][1] // scale))
    pf = tuple(parent_factor) if parent_factor is not None else tuple(rc["parent_factor"])
    return Workload(name=f"{name}/s{scale}", ny=gy, nx=gx, ly=ly, lx=lx, nz=nz_use, dz=dz, kv=kv, lam=lam, sigma=sigma,
                    alpha_mrad=rc["alpha"], defocus=rc["defocus"], parent_factor=pf, T=T, scan=_scan_grid(gy, gx, sy, sx),
                    scan_shape=(sy, sx), edges=edges, prism=tuple(rc["prism"]), crop=tuple(rc["crop"]))


def _scan_grid(ny, nx, sy, sx):
    """rho_ij = (i N_y / S_y, j N_x / S_x) px, row-major."""
    iy, ix = np.meshgrid(np.arange(sy), np.arange(sx), indexing="ij")
    return np.stack([iy.ravel() * (ny / sy), ix.ravel() * (nx / sx)], axis=1).astype(np.float64)


# name -> recipe. ``scale`` divides the cell count and the grid (keeps the pixel size): the
# "quarter-size clones" of SURVEY §8(d) are scale=4.
CONFIGS: Dict[str, dict] = {
    # BASELINE.json configs[0]
    "cfg1": dict(seed=75601, kind="perovskite", cells=(4, 4, 5), a=3.905, grid=(128, 128), kv=200.0, alpha=20.0,
                 defocus=0.0, jitter=0.02, ZA=(38, 38), ZB=(22, 22), ZO=8, parent_factor=(2.0, 2.0),
                 scan=(16, 16), edges=[dict(name="B", tag=1, n_ch=5, W=32, det=30.0)]),
    # BASELINE.json configs[1] -- the headline workload
    "cfg2": dict(seed=75602, kind="perovskite", cells=(20, 20, 20), a=3.905, grid=(512, 512), kv=300.0, alpha=25.0,
                 defocus=-50.0, jitter=0.0, ZA=(38, 38), ZB=(22, 22), ZO=8, parent_factor=(4.0, 4.0),
                 scan=(64, 64), edges=[dict(name="B", tag=1, n_ch=9, W=48, det=40.0)]),
    # BASELINE.json configs[2]: 160x80 A is not a multiple of 3.905 A -> common a = 4.0 A
    "cfg3": dict(seed=75603, kind="perovskite", cells=(20, 40, 30), a=4.0, grid=(512, 1024), kv=300.0, alpha=25.0,
                 defocus=0.0, jitter=0.0, ZA=(57, 38), ZB=(25, 22), ZO=8, parent_factor=(4.0, 4.0),
                 scan=(64, 128),
                 edges=[dict(name="O", tag=2, n_ch=1, W=48, det=40.0),
                        dict(name="B_left", tag=1, side=0, n_ch=9, W=48, det=40.0),
                        dict(name="B_right", tag=1, side=1, n_ch=9, W=48, det=40.0),
                        dict(name="A_left", tag=0, side=0, n_ch=9, W=48, det=40.0),
                        dict(name="A_right", tag=0, side=1, n_ch=9, W=48, det=40.0)]),
    # BASELINE.json configs[3]: FePt L1_0 nanoparticle in vacuum, in the regime the paper ran it (PRISM f = 8 beam lists,
    # n_radial = 8 -> 217 + 217 parents, crop mask f = 8 -> 32 x 32 scans per atom; SURVEY §8(d) "4-prism")
    "cfg4": dict(seed=75604, kind="fept", cell=(120.0, 120.0, 90.0), dz=2.0, radius=42.0, a=3.85, c=3.71, grid=(2048, 2048),
                 kv=300.0, alpha=25.0, defocus=0.0, parent_factor=(2.4, 2.4), prism=(8, 8), crop=(8, 8), scan=(256, 256),
                 edges=[dict(name="Fe", tag=0, n_ch=9, W=64, det=25.0)]),
    # BASELINE.json configs[4]: config-2 pixel size on 10x10x20 cells (SURVEY §8(d) cfg 5)
    "cfg5": dict(seed=75605, kind="perovskite", cells=(10, 10, 20), a=3.905, grid=(256, 256), kv=300.0, alpha=25.0,
                 defocus=-50.0, jitter=0.0, ZA=(38, 38), ZB=(22, 22), ZO=8, parent_factor=(4.0, 4.0),
                 scan=(64, 64), edges=[dict(name="B", tag=1, n_ch=9, W=48, det=40.0)]),
}


def make_workload(name: str, scale: int = 1, nz: Optional[int] = None, scan: Optional[Tuple[int, int]] = None,
                  parent_factor: Optional[Tuple[float, float]] = None, h_kind: str = "vortex",
                  window: Optional[int] = None) -> Workload:
    """Instantiate a config.  ``scale`` shrinks cells and grid together (pixel size kept), ``nz`` truncates
    the slab to its first ``nz`` slices, ``scan`` overrides the scan raster, ``window`` overrides W."""
    rc = CONFIGS[name]
    if rc["kind"] == "fept":
        return _make_fept(name, rc, scale, nz, scan, parent_factor, h_kind, window)
    cy, cx, cz = rc["cells"]
    gy, gx = rc["grid"]
    if cy % scale or cx % scale or gy % scale or gx % scale:
        raise ValueError("scale must divide cells and grid")
    cy, cx, gy, gx = cy // scale, cx // scale, gy // scale, gx // scale
    a = rc["a"]
    ly, lx = cy * a, cx * a
    dz = a / 2.0
    nz_full = 2 * cz
    nz_use = nz_full if nz is None else int(nz)
    if not 1 <= nz_use <= nz_full:
        raise ValueError("nz out of range")
    kv = rc["kv"]
    lam, sigma = electron_wavelength(kv), interaction_constant(kv)
    rng = np.random.default_rng(rc["seed"])

    half = cx // 2
    ZA = lambda ix: rc["ZA"][0] if ix < half else rc["ZA"][1]
    ZB = lambda ix: rc["ZB"][0] if ix < half else rc["ZB"][1]
    Z, Y, X, S, TAG, COL = _perovskite(cy, cx, cz, a, ZA, ZB, rc["ZO"])
    keep = S < nz_use
    Z, Y, X, S, TAG, COL = Z[keep], Y[keep], X[keep], S[keep], TAG[keep], COL[keep]
    Yj, Xj = Y, X
    if rc["jitter"] > 0.0:
        jit = rng.uniform(-rc["jitter"], rc["jitter"], (Z.shape[0], 2))
        Yj, Xj = Y + jit[:, 0], X + jit[:, 1]
    T = transmission_functions(gy, gx, ly, lx, nz_use, sigma, Z, Yj, Xj, S)

    edges = []
    for e in rc["edges"]:
        sel = TAG == e["tag"]
        if "side" in e:
            sel &= (COL < half) if e["side"] == 0 else (COL >= half)
        idx = np.nonzero(sel)[0]
        zc = (S[idx].astype(np.float64) + 0.5) * dz          # plane at the slice centre
        sl, centre = snap_sites(Y[idx], X[idx], zc, gy, gx, ly, lx, nz_use, dz)   # ideal (un-jittered) position
        W = int(window) if window is not None else e["W"]
        H = transition_windows(rng, e["n_ch"], W, h_kind)
        order = np.argsort(sl, kind="stable")
        edges.append(Edge(e["name"], sl[order], centre[order], H, e["det"]))

    sy, sx = scan if scan is not None else (max(1, rc["scan"][0] // scale), max(1, rc["scan"][1] // scale))
    pf = tuple(parent_factor) if parent_factor is not None else tuple(rc["parent_factor"])
    return Workload(name=f"{name}/s{scale}", ny=gy, nx=gx, ly=ly, lx=lx, nz=nz_use, dz=dz, kv=kv, lam=lam,
                    sigma=sigma, alpha_mrad=rc["alpha"], defocus=rc["defocus"], parent_factor=pf, T=T,
                    scan=_scan_grid(gy, gx, sy, sx), scan_shape=(sy, sx), edges=edges)


def tiny_random_workload(seed: int, ny: int = 16, nx: int = 12, nz: int = 3, n_ch: int = 2, W: int = 6,
                         n_atoms: int = 3, n_scan: int = 3) -> Workload:
    """A tiny random-phase cell for brute-force pins (non-square grid, wrapped windows, a non-integer scan)."""
    rng = np.random.default_rng(seed)
    ly, lx, lam, dz = 8.0 * ny / 16, 6.0 * nx / 12, 0.025, 2.0
    T = np.exp(1j * rng.normal(size=(nz, ny, nx))).astype(np.complex64)
    sl = np.sort(rng.integers(0, nz, n_atoms)).astype(np.int32)
    centre = np.stack([rng.integers(0, ny, n_atoms), rng.integers(0, nx, n_atoms)], axis=1).astype(np.int32)
    centre[0] = (0, 0)                                       # a window that wraps both axes
    H = (rng.normal(size=(n_ch, W, W)) + 1j * rng.normal(size=(n_ch, W, W))).astype(np.complex64)
    scan = np.stack([rng.integers(0, ny, n_scan).astype(np.float64), rng.integers(0, nx, n_scan).astype(np.float64)], axis=1)
    scan[-1] += (0.5, 0.25)                                  # one sub-pixel position
    return Workload(name=f"tiny{seed}", ny=ny, nx=nx, ly=ly, lx=lx, nz=nz, dz=dz, kv=0.0, lam=lam, sigma=0.0,
                    alpha_mrad=0.6 * lam * 1e3, defocus=-5.0, parent_factor=(1.0, 1.0), T=T, scan=scan,
                    scan_shape=(n_scan, 1), edges=[Edge("rand", sl, centre, H, 0.9 * lam * 1e3)])
