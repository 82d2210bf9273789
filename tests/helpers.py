"""Shared test plumbing: run the oracle and the CUDA library on the same seeded workload."""
import numpy as np

from oracle import beams as ob
from oracle import bip as obip
from oracle import multislice as oms
from oracle import sibson as osb


class OracleSetup:
    """Everything the oracle derives from a workload edge: beams, parents, weights, coefficients, propagator."""

    def __init__(self, wl, edge, parent_factor=None, n_jobs=1):
        f1, f2 = parent_factor if parent_factor is not None else wl.parent_factor
        ny, nx, ly, lx = wl.ny, wl.nx, wl.ly, wl.lx
        self.qa = wl.alpha_mrad * 1e-3 / wl.lam
        self.qd = edge.det_mrad * 1e-3 / wl.lam
        self.ap = ob.beams_in_disc(ny, nx, ly, lx, self.qa)
        self.det = ob.beams_in_disc(ny, nx, ly, lx, self.qd)
        self.c = ob.aperture_coefficients(self.ap, ny, nx, ly, lx, wl.lam, wl.defocus)
        self.P = oms.fresnel_propagator(ny, nx, ly, lx, wl.lam, wl.dz)

        def part(beams, q, f):
            if f == 1:
                import scipy.sparse as sp
                return np.arange(len(beams)), sp.identity(len(beams), format="csr")
            pos = ob.hexring_parents(beams, ny, nx, ly, lx, q, ob.n_radial_from_factor(len(beams), f))
            if n_jobs == 1:
                tab = osb.natural_neighbour_weights(beams, pos, ly, lx, q)
            else:                                     # harness-level parallelism over rows; the oracle is unchanged
                from joblib import Parallel, delayed
                chunks = np.array_split(np.arange(len(beams)), 8 * n_jobs)
                parts = Parallel(n_jobs=n_jobs)(delayed(osb.natural_neighbour_weights)(beams, pos, ly, lx, q, rows=c) for c in chunks)
                tab = [r for part in parts for r in part]
            import scipy.sparse as sp
            rows = np.concatenate([np.full(len(i), b) for b, (i, _) in enumerate(tab)])
            cols = np.concatenate([i for i, _ in tab])
            vals = np.concatenate([w for _, w in tab])
            return pos, sp.csr_matrix((vals, (rows, cols)), shape=(len(beams), len(pos)))

        self.p1_pos, self.w1 = part(self.ap, self.qa, f1)
        self.p2_pos, self.w2 = part(self.det, self.qd, f2)

    def run(self, wl, edge, recon="linear", scan=None):
        return obip.bip_run(wl.T.astype(np.complex128), self.P, self.ap, self.c, self.ap[self.p1_pos], self.w1, self.det,
                            self.det[self.p2_pos], self.w2, wl.scan if scan is None else scan, edge.slice, edge.centre,
                            edge.H, recon=recon)


def gpu_context(wl, edges, parent_factor=None, max_nn=8, T_on_device=True):
    """Create a library context for a workload; geometry comes from the library's own helpers.
    All edges must share the detector angle of edges[0] for the S2 parent set (as in every config here)."""
    import torch
    import paper_2607_00756_b200 as B
    g = B.Grid(wl.ny, wl.nx, wl.ly, wl.lx, wl.nz, wl.dz, wl.lam)
    pf = parent_factor if parent_factor is not None else wl.parent_factor
    geo = B.plan_geometry(g, wl.alpha_mrad, edges[0].det_mrad, wl.defocus, pf, max_nn)
    T = torch.from_numpy(wl.T).cuda() if T_on_device else wl.T
    ctx = B.Context(g, T, geo.ap_h, geo.ap_c, geo.p1_h, geo.w1, geo.p2_h)
    ctx.build_S1()
    ctx.build_S2()
    ctx.set_scan(wl.scan)
    ids = [ctx.add_edge(e.slice, e.centre, e.H, geo.det_h, geo.w2) for e in edges]
    return ctx, geo, ids


def rel_err_map(got, want, floor=0.0):
    """max |got - want| / max(want, floor * max(want)); floor = 0 is the plain per-pixel form."""
    den = np.maximum(np.abs(want), floor * np.abs(want).max()) if floor > 0 else np.abs(want)
    return float(np.max(np.abs(got - want) / den))
