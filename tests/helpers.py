"""Shared test plumbing: run the oracle and the CUDA library on the same seeded workload."""
import numpy as np

from oracle import beams as ob
from oracle import bip as obip
from oracle import multislice as oms
from oracle import sibson as osb


class OracleSetup:
    """Everything the oracle derives from a workload edge: beams, parents, weights, coefficients, propagator."""

    def __init__(self, wl, edge, parent_factor=None, n_jobs=1, prism=None):
        f1, f2 = parent_factor if parent_factor is not None else wl.parent_factor
        ny, nx, ly, lx = wl.ny, wl.nx, wl.ly, wl.lx
        self.qa = wl.alpha_mrad * 1e-3 / wl.lam
        self.qd = edge.det_mrad * 1e-3 / wl.lam
        self.ap = ob.beams_in_disc(ny, nx, ly, lx, self.qa)
        self.det = ob.beams_in_disc(ny, nx, ly, lx, self.qd)
        self.c = ob.aperture_coefficients(self.ap, ny, nx, ly, lx, wl.lam, wl.defocus)
        self.P = oms.fresnel_propagator(ny, nx, ly, lx, wl.lam, wl.dz)
        prism = tuple(prism) if prism is not None else tuple(getattr(wl, 'prism', (1, 1)))
        if prism != (1, 1):                           # PRISM beam subsampling of both sets
            keep = ob.prism_subsample(self.ap, *prism)
            self.ap, self.c = self.ap[keep], ob.prism_coefficients(self.c, keep, *prism)
            self.det = self.det[ob.prism_subsample(self.det, *prism)]

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

    def run(self, wl, edge, recon="linear", scan=None, crop_f=None, association="probe"):
        return obip.bip_run(wl.T.astype(np.complex128), self.P, self.ap, self.c, self.ap[self.p1_pos], self.w1, self.det,
                            self.det[self.p2_pos], self.w2, wl.scan if scan is None else scan, edge.slice, edge.centre,
                            edge.H, recon=recon, crop_f=crop_f, association=association)


def gpu_context(wl, edges, parent_factor=None, max_nn=8, T_on_device=True, prism=None, crop=None, allow_tf32x3=True, stream=None):
    """Create a library context for a workload; geometry comes from the library's own helpers.
    All edges must share the detector angle of edges[0] for the S2 parent set (as in every config here)."""
    import torch
    import paper_2607_00756_b200 as B
    g = B.Grid(wl.ny, wl.nx, wl.ly, wl.lx, wl.nz, wl.dz, wl.lam)
    pf = parent_factor if parent_factor is not None else wl.parent_factor
    prism = tuple(prism) if prism is not None else tuple(getattr(wl, 'prism', (1, 1)))
    crop = tuple(crop) if crop is not None else tuple(getattr(wl, 'crop', (1, 1)))
    geo = B.plan_geometry(g, wl.alpha_mrad, edges[0].det_mrad, wl.defocus, pf, max_nn, prism=prism)
    T = torch.from_numpy(wl.T).cuda() if T_on_device else wl.T
    ctx = B.Context(g, T, geo.ap_h, geo.ap_c, geo.p1_h, geo.w1, geo.p2_h, stream=stream)
    ctx.allow_tf32x3(allow_tf32x3)                    # the parity tests run TF32X3 as the measured A/B case (include/bip.h)
    ctx.build_S1()
    ctx.build_S2()
    ctx.set_scan(wl.scan)
    ctx.set_crop(*crop)
    ids = [ctx.add_edge(e.slice, e.centre, e.H, geo.det_h, geo.w2) for e in edges]
    return ctx, geo, ids


def rel_err_map(got, want, floor=0.0):
    """max |got - want| / max(want, floor * max(want)); floor = 0 is the plain per-pixel form."""
    den = np.maximum(np.abs(want), floor * np.abs(want).max()) if floor > 0 else np.abs(want)
    return float(np.max(np.abs(got - want) / den))


class OracleSample:
    """A bounded sample of a full-size workload for the oracle (SURVEY 8(d) "Parity protocol"): the first ``n_atoms``
    sites of the edge, a regular subset of ``n_scan`` scan positions, every channel and every detector beam.  The
    slab is truncated to ``nz`` slices so that the fp64 parent columns are cheap to build; parents are processed in
    chunks and only their W x W windows at the sampled sites are kept.  Contraction shapes per (scan, channel,
    beam) are those of the full workload.  Used by the full-size parity test and by bench.py's oracle legs."""

    def __init__(self, workload="cfg2", scale=1, nz=2, n_atoms=1, n_scan=256, n_jobs=None, edge=0, atom_idx=None):
        import os
        from bip_inputs.specimen import make_workload
        self.wl = wl = make_workload(workload, scale=scale, nz=nz)
        if atom_idx is not None:                          # explicit sites (e.g. one deep inside the slab)
            atom_idx = np.asarray(atom_idx)
            n_atoms = len(atom_idx)
        self.e = e = wl.edges[edge].take(np.arange(n_atoms) if atom_idx is None else atom_idx)
        self.orc = orc = OracleSetup(wl, e, n_jobs=n_jobs or os.cpu_count())
        T = wl.T.astype(np.complex128)
        planes = sorted(set(int(s) for s in e.slice))
        self.crops = [[None, None] for _ in range(n_atoms)]
        for which, par_h in ((0, orc.ap[orc.p1_pos]), (1, orc.det[orc.p2_pos])):
            parts = [[] for _ in range(n_atoms)]
            for c0 in range(0, len(par_h), 256):          # parents in chunks: only the windows are kept
                hs = par_h[c0:c0 + 256]
                for plane in planes:
                    if which == 0:
                        S = oms.build_S1(hs, wl.ny, wl.nx)
                        for i in range(plane):
                            S = oms.advance_S1(S, T[i], orc.P)
                    else:
                        S = oms.build_S2_at(hs, T, orc.P, plane)
                    for a in np.nonzero(e.slice == plane)[0]:
                        parts[a].append(obip.crop_window(S, e.centre[a], e.W, wl.ny, wl.nx))
            for a in range(n_atoms):
                self.crops[a][which] = np.concatenate(parts[a])
        sy, sx = wl.scan_shape
        side = max(1, int(round(np.sqrt(n_scan))))
        sub = [iy * sx + ix for iy in range(0, sy, max(1, sy // side)) for ix in range(0, sx, max(1, sx // side))]
        self.scan_idx = np.array(sub[:n_scan])
        self.A = obip.illumination(orc.c, orc.ap, wl.scan[self.scan_idx], wl.ny, wl.nx)

    def run(self, recon, atoms=None):
        """Steps a1-a8 of the oracle on the sample: dict of reduce_modes() summed over the sampled atoms."""
        o, e, wl, acc = self.orc, self.e, self.wl, None
        for a in (range(e.n_atoms) if atoms is None else atoms):
            amp, _ = obip.atom_amplitudes(None, None, o.ap[o.p1_pos], o.det[o.p2_pos], o.ap, o.det, o.w1, o.w2, self.A,
                                          e.H.astype(np.complex128), e.centre[a], wl.ny, wl.nx, recon, crops=tuple(self.crops[a]))
            r = obip.reduce_modes(amp, o.det)
            acc = r if acc is None else {k: acc[k] + r[k] for k in acc}
        return acc
