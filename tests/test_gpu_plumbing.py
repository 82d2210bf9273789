"""The slice-step plumbing (bip_build_S2, ADVANCETO, PEELTO; eq. 6, eq. 12): the native fused fp32 slice step against the
oracle and against the cuFFT fp64 route, and the measurement that decides between them -- the drift of the column norms
over a 40-slice slab (every step is unitary for |T| = 1, so ||S_p||^2 / G must stay 1; a systematic loss shows directly
in the summed intensity, which north_star bounds by 1e-6).  `pytest -s` prints the measured drifts
(summarised in profiles/r02_fft_norm_drift.md)."""
import numpy as np
import pytest

from bip_inputs.specimen import make_workload
from helpers import OracleSetup, gpu_context
from oracle import multislice as oms

pytestmark = pytest.mark.gpu


def _column_norm_drift(S):
    G = S.shape[1] * S.shape[2]
    n2 = (np.abs(S.astype(np.complex128)) ** 2).sum(axis=(1, 2)) / G
    return n2 - 1.0


@pytest.mark.parametrize("name,scale,nz", [("cfg1", 2, 6), ("cfg3", 4, 5)])
def test_native_slice_step_matches_oracle(name, scale, nz):
    """Power-of-two grids (64 x 64 and the anisotropic 128 x 256) take the native route: S1 and S2 at several planes,
    forwards and backwards, against the oracle's fp64 multislice."""
    import paper_2607_00756_b200 as B
    wl = make_workload(name, scale=scale, nz=nz)
    e = wl.edges[0]
    ctx, geo, ids = gpu_context(wl, [e])
    orc = OracleSetup(wl, e)
    T = wl.T.astype(np.complex128)
    n1, n2 = min(ctx.n_p1, 24), min(ctx.n_p2, 24)
    S1 = oms.build_S1(orc.ap[orc.p1_pos][:n1], wl.ny, wl.nx)
    S2 = oms.build_S2(orc.det[orc.p2_pos][:n2], T, orc.P)
    want = {0: (S1, S2)}
    for i in range(wl.nz):
        S1 = oms.advance_S1(S1, T[i], orc.P)
        S2 = oms.peel_S2(S2, T[i], orc.P)
        want[i + 1] = (S1, S2)
    for backend in (B.FFT_NATIVE, B.FFT_CUFFT_F64):
        ctx.set_fft_backend(backend)
        ctx.build_S1(); ctx.build_S2()
        for plane in (0, 2, nz, 1, 3):
            ctx.seek_plane(plane)
            assert np.abs(ctx.copy_S(1, 0, n1) - want[plane][0]).max() < 1e-5, (backend, plane)
            assert np.abs(ctx.copy_S(2, 0, n2) - want[plane][1]).max() < 1e-5, (backend, plane)
    ctx.close()


@pytest.mark.parametrize("ny,nx", [(8, 8), (16, 64), (32, 8), (64, 256), (128, 32), (256, 1024), (1024, 64), (2048, 16), (16, 4096)])
def test_native_slice_step_on_every_transform_length(ny, nx):
    """Every compile-time transform length of the native route (8 ... 4096 along either axis, all three radix tails, row
    tiles that span several columns, column tiles wider than a block) on a random-phase slab: S1 and S2 parents at two
    planes against the oracle's fp64 multislice (eq. 6, eq. 12)."""
    import paper_2607_00756_b200 as B
    from bip_inputs.specimen import tiny_random_workload
    wl = tiny_random_workload(11, ny=ny, nx=nx, nz=3, W=8, n_atoms=2, n_scan=2)
    # a few dozen beams whatever the shape of the grid, all of them below the Nyquist index of both axes
    q = min(np.sqrt(40.0 / (np.pi * wl.ly * wl.lx)), 0.9 * (ny / 2 - 1) / wl.ly, 0.9 * (nx / 2 - 1) / wl.lx)
    wl.alpha_mrad = 1e3 * wl.lam * q
    e = wl.edges[0]
    e.det_mrad = 1.2 * wl.alpha_mrad
    ctx, geo, ids = gpu_context(wl, [e], parent_factor=(1, 1))
    ctx.set_fft_backend(B.FFT_NATIVE)
    ctx.build_S1(); ctx.build_S2()
    orc = OracleSetup(wl, e, parent_factor=(1, 1))
    T = wl.T.astype(np.complex128)
    S1 = oms.build_S1(orc.ap[orc.p1_pos], ny, nx)
    S2 = oms.build_S2(orc.det[orc.p2_pos], T, orc.P)
    want = {0: (S1, S2)}
    for i in range(wl.nz):
        S1 = oms.advance_S1(S1, T[i], orc.P)
        S2 = oms.peel_S2(S2, T[i], orc.P)
        want[i + 1] = (S1, S2)
    for plane in (0, 3, 1):
        ctx.seek_plane(plane)
        assert np.abs(ctx.copy_S(1, 0, ctx.n_p1) - want[plane][0]).max() < 2e-5, plane
        assert np.abs(ctx.copy_S(2, 0, ctx.n_p2) - want[plane][1]).max() < 2e-5, plane
    ctx.close()


def test_native_route_is_refused_on_a_grid_that_is_not_a_power_of_two():
    import paper_2607_00756_b200 as B
    from bip_inputs.specimen import tiny_random_workload
    wl = tiny_random_workload(3, W=8)                              # 16 x 12
    ctx, geo, ids = gpu_context(wl, [wl.edges[0]], parent_factor=(1, 1))
    with pytest.raises(B.BipError) as ei:
        ctx.set_fft_backend(B.FFT_NATIVE)
    assert ei.value.status == 5
    ctx.close()


def test_column_norm_drift_over_a_forty_slice_slab(capsys):
    """40 unitary slice steps on 271 S2 parent columns of the configs[0] geometry repeated to 40 slices: drift of
    ||S_p||^2 / G for the native fp32 route, the cuFFT fp64 route and, for reference, plain single-precision cuFFT C2C
    (through torch.fft, the same library) on the same columns."""
    import torch
    import paper_2607_00756_b200 as B
    wl = make_workload("cfg1", nz=10)
    wl.T = np.concatenate([wl.T] * 4)                              # 40 slices
    wl.nz = 40
    e = wl.edges[0]
    ctx, geo, ids = gpu_context(wl, [e])
    drift = {}
    for name, backend in (("native fp32", B.FFT_NATIVE), ("cuFFT fp64 workspace", B.FFT_CUFFT_F64)):
        ctx.set_fft_backend(backend)
        ctx.build_S2()                                             # 40 steps u <- T_j P[u] from the exit surface
        d = _column_norm_drift(ctx.copy_S(2, 0, ctx.n_p2))
        drift[name] = (float(d.mean()), float(np.abs(d).max()))
    # plain cuFFT C2C in single precision on the same problem
    g = B.Grid(wl.ny, wl.nx, wl.ly, wl.lx, wl.nz, wl.dz, wl.lam)
    hy = np.fft.fftfreq(wl.ny, 1.0 / wl.ny) / wl.ly
    hx = np.fft.fftfreq(wl.nx, 1.0 / wl.nx) / wl.lx
    P = torch.from_numpy(np.exp(-1j * np.pi * wl.lam * wl.dz * (hy[:, None] ** 2 + hx[None, :] ** 2)).astype(np.complex64)).cuda()
    ry, rx = np.arange(wl.ny)[:, None], np.arange(wl.nx)[None, :]
    u = np.stack([np.exp(-2j * np.pi * (((h[0] * ry) % wl.ny) / wl.ny + ((h[1] * rx) % wl.nx) / wl.nx)) for h in geo.p2_h]).astype(np.complex64)
    u = torch.from_numpy(u).cuda()
    Td = torch.from_numpy(wl.T).cuda()
    for j in range(wl.nz - 1, -1, -1):
        u = Td[j] * torch.fft.ifft2(P * torch.fft.fft2(u))
    d = _column_norm_drift(u.cpu().numpy())
    drift["cuFFT C2C fp32 (torch.fft)"] = (float(d.mean()), float(np.abs(d).max()))
    with capsys.disabled():
        print("\ncolumn-norm drift ||S_p||^2/G - 1 after 40 slices (mean over 271 columns, max |.|):")
        for k, v in drift.items():
            print(f"  {k:32s} mean {v[0]:+.3e}   max {v[1]:.3e}")
    # |T| = 1 only to c64 rounding (6e-8 per element, unbiased): what is asserted is the absence of a SYSTEMATIC drift
    assert abs(drift["native fp32"][0]) < 5e-7 and drift["native fp32"][1] < 2e-6
    assert abs(drift["cuFFT fp64 workspace"][0]) < 5e-7
    ctx.close()
