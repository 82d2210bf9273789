"""NEXT-4 on the GPU: S1 focal back-propagation to the scattering-centroid plane (bip_set_focal, reading c20)
and frozen-phonon averaging (bip_set_transmission + bip_set_accumulate) against oracle/focal.py."""
import numpy as np
import pytest

from bip_inputs.specimen import make_workload
from helpers import OracleSetup, gpu_context, rel_err_map
from oracle import focal

pytestmark = pytest.mark.gpu

TOL_PIXEL = 1e-4
TOL_SUM = 1e-6


def _focal_oracle(wl, e, orc, recon):
    return focal.bip_run_focal(wl.T.astype(np.complex128), orc.P, orc.ap, orc.c, orc.ap[orc.p1_pos], orc.w1, orc.det, orc.det[orc.p2_pos],
                               orc.w2, wl.scan, e.slice, e.centre, e.H, wl.ly, wl.lx, wl.lam, wl.dz, recon)


@pytest.mark.parametrize("recon", ["linear", "magphase"])
def test_focal_back_propagation_matches_oracle(recon):
    """configs[0] geometry at half size (64 x 64 grid, W = 16 -> padded window 32), parent factor 2, sites in the 2nd, 4th
    and 6th slice (so the centroid distances differ), 9 scan positions, 3 of them sub-pixel."""
    import torch
    import paper_2607_00756_b200 as B
    wl = make_workload("cfg1", scale=2, nz=6, scan=(3, 3), window=16)
    wl.scan = wl.scan + np.array([[0, 0]] * 6 + [[0.37, 0.21]] * 3)
    e = wl.edges[0]
    e = e.take(np.concatenate([np.nonzero(e.slice == p)[0][:2] for p in np.unique(e.slice)]))
    assert len(np.unique(e.slice)) == 3
    orc = OracleSetup(wl, e)
    want = _focal_oracle(wl, e, orc, recon)
    plain = orc.run(wl, e, recon)
    ctx, geo, ids = gpu_context(wl, [e])
    for plane in range(wl.nz + 1):                                              # the centroid distances, reading c20
        assert abs(ctx.get_focal_distance(plane) - focal.scattering_centroid_distance(wl.T, plane, wl.dz)) < 1e-6
    rc = B.RECON_LINEAR if recon == "linear" else B.RECON_MAGPHASE
    ctx.set_focal(True)
    m = ctx.map(0, B.MODE_MAP, rc, B.PREC_FP16X4)
    cube = ctx.map(0, B.MODE_CUBE, rc, B.PREC_FP16X4)
    torch.cuda.synchronize()
    m, cube = m.cpu().numpy(), cube.cpu().numpy()
    assert rel_err_map(m, want["map"]) <= TOL_PIXEL, rel_err_map(m, want["map"])
    assert abs(m.sum() - want["map"].sum()) <= TOL_SUM * want["map"].sum(), abs(m.sum() - want["map"].sum()) / want["map"].sum()
    assert rel_err_map(cube, want["cube"], 1e-3) <= TOL_PIXEL
    assert rel_err_map(m, plain["map"]) > 10 * TOL_PIXEL                        # it IS a different estimate from the plain one
    ctx.set_focal(False)
    m0 = ctx.map(0, B.MODE_MAP, rc, B.PREC_FP16X4)
    torch.cuda.synchronize()
    assert rel_err_map(m0.cpu().numpy(), plain["map"]) <= TOL_PIXEL
    ctx.set_focal(True)
    ctx.set_association(B.ASSOC_COUPLING)
    with pytest.raises(B.BipError) as ei:
        ctx.map(0, B.MODE_MAP, rc, B.PREC_FP16X4)
    assert ei.value.status == 5
    ctx.close()


def test_focal_full_parent_limit_is_exact():
    """Parents = all beams: the back and forward Fresnel steps cancel beam by beam (to fp32 round-off), whatever the
    distance -- the map equals the plain exact-PRISM map."""
    import torch
    import paper_2607_00756_b200 as B
    wl = make_workload("cfg1", scale=2, nz=6, scan=(3, 3), window=16)
    e = wl.edges[0].take(np.nonzero(wl.edges[0].slice == 5)[0][:3])
    orc = OracleSetup(wl, e, parent_factor=(1, 1))
    want = orc.run(wl, e, "magphase")
    ctx, geo, ids = gpu_context(wl, [e], parent_factor=(1, 1))
    ctx.set_focal(True)
    assert ctx.get_focal_distance(5) > 1.0
    m = ctx.map(0, B.MODE_MAP, B.RECON_MAGPHASE, B.PREC_FP16X4)
    torch.cuda.synchronize()
    assert rel_err_map(m.cpu().numpy(), want["map"]) <= TOL_PIXEL
    ctx.close()


def test_frozen_phonon_average_over_two_configurations():
    """Two displaced configurations (two seeds of the jittered configs[0] cell): set_transmission, rebuild, accumulate;
    the mean of the two maps against the oracle's frozen_phonon_average."""
    import torch
    import paper_2607_00756_b200 as B
    wl = make_workload("cfg1", scale=2, nz=4, scan=(4, 4))
    e = wl.edges[0].take(np.arange(6))
    rng = np.random.default_rng(7)
    T2 = (wl.T * np.exp(1j * 0.05 * rng.standard_normal(wl.T.shape))).astype(np.complex64)
    T2 = (T2 / np.abs(T2)).astype(np.complex64)                                   # still a pure phase object
    orc = OracleSetup(wl, e)

    def run(T):
        wl_t = type(wl)(**{**wl.__dict__, "T": T})
        return orc.run(wl_t, e, "magphase")

    want = focal.frozen_phonon_average(run, [wl.T, T2])
    ctx, geo, ids = gpu_context(wl, [e])
    out = torch.zeros(wl.n_rho, dtype=torch.float64, device="cuda")
    ctx.set_accumulate(True)
    for T in (wl.T, T2):
        ctx.set_transmission(torch.from_numpy(T).cuda())
        with pytest.raises(B.BipError):
            ctx.map(0, B.MODE_MAP, B.RECON_MAGPHASE, B.PREC_FP16X4, out=out)     # the matrices belong to the old configuration
        ctx.build_S1(); ctx.build_S2()
        ctx.map(0, B.MODE_MAP, B.RECON_MAGPHASE, B.PREC_FP16X4, out=out)
    torch.cuda.synchronize()
    m = out.cpu().numpy() / 2
    assert rel_err_map(m, want["map"]) <= TOL_PIXEL
    assert abs(m.sum() - want["map"].sum()) <= TOL_SUM * want["map"].sum()
    ctx.close()
