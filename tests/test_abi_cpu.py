"""CPU-side checks of the C ABI: the library loads, exports every declared symbol, validates arguments, refuses to
run without a device, and its host geometry (beam sets, hex-ring parents, Sibson tables, probe coefficients) equals
the oracle's -- index lists bit-exact, weights to 1e-6 (BASELINE.json north_star)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2607_00756_b200 as B
from paper_2607_00756_b200 import api
from bip_inputs import electron_wavelength
from oracle import beams as ob
from oracle import sibson as osb

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "bip.h")).read()
    declared = set(re.findall(r"BIP_API[^;(]*?\b(bip_\w+)\s*\(", hdr))
    assert declared == set(api.ABI_SYMBOLS) and len(declared) >= 20
    lib = B.load_library()
    for name in declared:
        assert getattr(lib, name) is not None
    assert "libbip" in B.bip_version()


def test_struct_layouts_match_header():
    assert C.sizeof(api._Grid) == 48 and C.sizeof(api._Weights) == 24 and C.sizeof(api._Timing) == 48


def _dense(idx, w, n_par):
    W = np.zeros((idx.shape[0], n_par))
    for b in range(idx.shape[0]):
        m = idx[b] >= 0
        W[b, idx[b][m]] = w[b][m]
    return W


@pytest.mark.parametrize("ny,nx,ly,lx,kv,mrad,nr", [(128, 128, 15.62, 15.62, 200.0, 20.0, 6), (128, 128, 15.62, 15.62, 200.0, 30.0, 9),
                                                   (64, 128, 20.0, 40.0, 300.0, 25.0, 4)])
def test_geometry_matches_oracle(ny, nx, ly, lx, kv, mrad, nr):
    lam = electron_wavelength(kv)
    g = B.Grid(ny, nx, ly, lx, 4, 2.0, lam)
    q = mrad * 1e-3 / lam
    h = B.bip_beams_in_disc(g, q)
    ho = ob.beams_in_disc(ny, nx, ly, lx, q)
    assert h.dtype == np.int32 and np.array_equal(h, ho)                       # bit-exact beam list and order
    pos = B.bip_hexring(g, h, q, nr)
    poso = ob.hexring_parents(ho, ny, nx, ly, lx, q, nr)
    assert np.array_equal(pos, poso)                                           # bit-exact parent list
    idx, w = B.bip_sibson(g, h, h[pos], q, 8)
    tab = osb.natural_neighbour_weights(ho, poso, ly, lx, q)
    assert np.abs(_dense(idx, w, len(pos)) - osb.to_dense(tab, len(poso))).max() < 1e-6
    for b, (io, wo) in enumerate(tab):                                         # same neighbour sets above the noise floor
        assert set(io[wo > 1e-6].tolist()) <= set(idx[b][idx[b] >= 0].tolist())
        m = idx[b] >= 0
        assert np.all(np.diff(idx[b][m]) > 0) and np.all(idx[b][~m] == -1) and abs(w[b][m].sum() - 1) < 1e-6
    c = B.bip_aperture_coeffs(g, h, -50.0)
    co = ob.aperture_coefficients(ho, ny, nx, ly, lx, lam, -50.0)
    assert np.abs((c[:, 0] + 1j * c[:, 1]) - co).max() < 1e-7 * np.abs(co).max()
    assert B.bip_n_radial_from_factor(len(h), 2.0) == ob.n_radial_from_factor(len(ho), 2.0)


@pytest.mark.slow
def test_geometry_full_size_cfg2_sampled_rows():
    """BASELINE.json configs[1] sizes: B = 30 909, K = 79 105, parents 1 951 / 4 921 (SURVEY section 8 size table);
    index lists bit-exact in full, weight rows compared on a sample the oracle computes one by one."""
    lam = electron_wavelength(300.0)
    g = B.Grid(512, 512, 78.1, 78.1, 40, 1.9525, lam)
    geo = B.plan_geometry(g, 25.0, 40.0, -50.0, (4, 4))
    assert geo.ap_h.shape[0] == 30909 and geo.det_h.shape[0] == 79105
    assert geo.p1_pos.shape[0] == 1951 and geo.p2_pos.shape[0] == 4921
    for h, pos, (idx, w), q, nr in ((geo.ap_h, geo.p1_pos, geo.w1, geo.qa, 25), (geo.det_h, geo.p2_pos, geo.w2, geo.qd, 40)):
        ho = ob.beams_in_disc(512, 512, 78.1, 78.1, q)
        assert np.array_equal(h, ho)
        assert np.array_equal(pos, ob.hexring_parents(ho, 512, 512, 78.1, 78.1, q, nr))
        rows = list(range(0, len(ho), 1999)) + [0, 1, len(ho) - 2, len(ho) - 1]
        tab = osb.natural_neighbour_weights(ho, pos, 78.1, 78.1, q, rows=rows)
        for (io, wo), b in zip(tab, rows):
            d = np.zeros(len(pos)); d[io] = wo
            l = np.zeros(len(pos)); m = idx[b] >= 0; l[idx[b][m]] = w[b][m]
            assert np.abs(d - l).max() < 1e-6


def test_identity_partition_for_factor_one():
    g = B.Grid(32, 32, 8.0, 8.0, 2, 2.0, 0.025)
    geo = B.plan_geometry(g, 12.0, 16.0, 0.0, (1, 1))
    assert np.array_equal(geo.p1_pos, np.arange(len(geo.ap_h)))
    assert np.array_equal(geo.w1[0][:, 0], np.arange(len(geo.ap_h))) and np.all(geo.w1[1][:, 0] == 1.0)
    assert np.all(geo.w1[0][:, 1:] == -1) and np.all(geo.w1[1][:, 1:] == 0.0)


def test_argument_validation_and_no_cpu_fallback():
    lib = B.load_library()
    g = B.Grid(32, 32, 8.0, 8.0, 2, 2.0, 0.025)
    with pytest.raises(B.BipError) as ei:
        B.bip_hexring(g, np.array([[1, 0], [0, 0]], dtype=np.int32), 1.0, 2)       # not in ascending flat index
    assert ei.value.status == 1
    with pytest.raises(B.BipError):
        B.bip_sibson(g, np.zeros((0, 2), np.int32), np.zeros((1, 2), np.int32), 1.0)
    # more neighbours than max_nn is an error, not a truncation
    h = B.bip_beams_in_disc(g, 1.0)
    pos = B.bip_hexring(g, h, 1.0, 3)
    with pytest.raises(B.BipError) as ei:
        B.bip_sibson(g, h, h[pos], 1.0, 2)
    assert "max_nn" in str(ei.value)
    # bad grid / NULL arguments are rejected before anything touches a device
    ctx = C.c_void_p(None)
    assert lib.bip_create(C.byref(ctx), None, None, 0, 0, None, None, 0, None, None, 0, None, None) == 1
    assert lib.bip_map(None, 0, 0, 0, 0, None, 0) == 1
    assert lib.bip_destroy(None) == 0
    import torch
    if not torch.cuda.is_available():
        geo = B.plan_geometry(g, 12.0, 16.0, 0.0, (2, 2))
        T = np.ones((2, 32, 32), np.complex64)
        with pytest.raises(B.BipError) as ei:
            B.Context(g, T, geo.ap_h, geo.ap_c, geo.p1_h, geo.w1, geo.p2_h, stream=0)
        assert ei.value.status == 4 and "no CPU path" in str(ei.value)           # fails loudly: no fallback


def test_prism_subsample_matches_oracle():
    """bip_prism_subsample against the oracle's rule, bit-exact, incl. negative indices."""
    import paper_2607_00756_b200 as B
    from oracle import beams as ob
    beams = ob.beams_in_disc(64, 48, 20.0, 15.0, 0.9)
    for fy, fx in ((1, 1), (2, 2), (4, 3), (5, 1)):
        assert np.array_equal(B.bip_prism_subsample(beams, fy, fx), ob.prism_subsample(beams, fy, fx))


def test_partition_and_prism_coeffs_match_oracle():
    """bip_partition (hex-ring + Sibson by parent factor, reading c7) and bip_prism_coeffs (f_y f_x rescale)
    are C entry points, so that no method arithmetic is left in the Python binding: both against the oracle."""
    lam = electron_wavelength(200.0)
    g = B.Grid(64, 96, 12.0, 18.0, 2, 2.0, lam)
    q = 18e-3 / lam
    h = B.bip_beams_in_disc(g, q)
    ho = ob.beams_in_disc(64, 96, 12.0, 18.0, q)
    pos, (idx, w) = B.bip_partition(g, h, q, 2.0)
    poso = ob.hexring_parents(ho, 64, 96, 12.0, 18.0, q, ob.n_radial_from_factor(len(ho), 2.0))
    assert np.array_equal(pos, poso)
    tab = osb.natural_neighbour_weights(ho, poso, 12.0, 18.0, q)
    assert np.abs(_dense(idx, w, len(pos)) - osb.to_dense(tab, len(poso))).max() < 1e-6
    c = B.bip_aperture_coeffs(g, h, -30.0)
    co = ob.aperture_coefficients(ho, 64, 96, 12.0, 18.0, lam, -30.0)
    for fy, fx in ((2, 2), (3, 2)):
        keep = B.bip_prism_subsample(h, fy, fx)
        got = B.bip_prism_coeffs(keep, c, fy, fx)
        want = ob.prism_coefficients(co, ob.prism_subsample(ho, fy, fx), fy, fx)
        assert np.abs((got[:, 0] + 1j * got[:, 1]) - want).max() < 1e-6 * np.abs(want).max()
    with pytest.raises(B.BipError):
        B.bip_prism_coeffs(np.array([len(h)], np.int32), c, 2, 2)                  # position outside the full list
    with pytest.raises(B.BipError):
        B.bip_partition(g, h, q, 0.5)                                               # factor < 1
