"""bip_reconstruct_noalloc (include/bip.h): the one entry point of the library that allocates nothing -- the windowed
reconstruction of one site (steps a1-a2 / a6; eq. 15; eq. 11) with its intermediate de-tilted
parent windows in a static device array of BIP_NOALLOC_SCRATCH_BYTES (4 MiB) inside the library -- against the existing,
allocating path bip_debug_reconstruct (itself compared with the oracle in test_gpu_parity.py), on two calls in a row that share
the static scratch, and its refusal of a request beyond the maximum.

The file name makes pytest collect it last: the suite runs with `pytest -x`, and a failure here must not hide the other tests.
Each test builds its own context and passes alone in a fresh process as well as after the rest of the suite."""
import numpy as np
import pytest

from bip_inputs.specimen import make_workload
from helpers import gpu_context

pytestmark = pytest.mark.gpu

TOL = 2e-5                      # the absolute tolerance test_windowed_reconstruction_matches_oracle holds these windows to
SCRATCH_BYTES = 4 << 20         # BIP_NOALLOC_SCRATCH_BYTES of include/bip.h


def test_no_alloc_reconstruction_matches_the_allocating_path_on_two_calls_in_a_row():
    """BASELINE.json configs[0] at full size (128 x 128, 127 / 271 parents, 32 x 32 windows: 1.0 / 2.2 MB of scratch).  Two calls
    back to back on the context's stream without a synchronisation between them -- S1 side of one site, then S2 side of another,
    the second overwriting the scratch the first used -- and a second pair in the other order and reconstruction mode."""
    import torch
    import paper_2607_00756_b200 as B
    wl = make_workload("cfg1", nz=3, scan=(4, 4))
    e = wl.edges[0]
    ctx, geo, ids = gpu_context(wl, [e])
    assert ctx.n_p1 * e.W * e.W * 8 <= SCRATCH_BYTES and ctx.n_p2 * e.W * e.W * 8 <= SCRATCH_BYTES
    ctx.seek_plane(int(e.slice[0]))
    a0, a1 = 0, e.n_atoms - 1                                   # a1's window wraps around the cell
    for first, second, rc in (((a0, 1), (a1, 2), B.RECON_MAGPHASE), ((a1, 2), (a0, 1), B.RECON_LINEAR)):
        out_a = ctx.reconstruct_noalloc(0, first[0], first[1], rc)
        out_b = ctx.reconstruct_noalloc(0, second[0], second[1], rc)          # in a row: no synchronisation in between
        torch.cuda.synchronize()
        got_a, got_b = out_a.cpu().numpy(), out_b.cpu().numpy()
        want_a = ctx.debug_reconstruct(0, first[0], first[1], rc)
        want_b = ctx.debug_reconstruct(0, second[0], second[1], rc)
        assert got_a.shape == want_a.shape and got_b.shape == want_b.shape
        assert np.abs(want_a).max() > 0.1 and np.abs(want_b).max() > 0.1       # the comparison is not between two empty buffers
        assert np.abs(got_a - want_a).max() <= TOL, np.abs(got_a - want_a).max()
        assert np.abs(got_b - want_b).max() <= TOL, np.abs(got_b - want_b).max()
    # into a buffer the caller made beforehand, twice: the second call must not depend on what the first left in the scratch
    out = torch.full((geo.det_h.shape[0], e.W * e.W), float("nan"), dtype=torch.complex64, device="cuda")
    want = ctx.debug_reconstruct(0, a0, 2, B.RECON_MAGPHASE)
    for _ in range(2):
        free_before = torch.cuda.mem_get_info()[0]
        ctx.reconstruct_noalloc(0, a0, 2, B.RECON_MAGPHASE, out=out)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before          # the (warm) call took no device memory
        assert np.abs(out.cpu().numpy() - want).max() <= TOL
    ctx.close()


def test_no_alloc_reconstruction_rejects_a_request_beyond_the_static_scratch():
    """Parents = all beams (parent factor 1): the S2 side needs 1101 x 32 x 32 x 8 = 9.0 MB of scratch, beyond the 4 MiB array ->
    BIP_ERR_UNSUPPORTED, output untouched; the S1 side (489 parents: 4.0 MB) still fits and still matches.  A wrong output size
    is BIP_ERR_INVALID."""
    import torch
    import paper_2607_00756_b200 as B
    wl = make_workload("cfg1", nz=3, scan=(4, 4))
    e = wl.edges[0]
    ctx, geo, ids = gpu_context(wl, [e], parent_factor=(1, 1))
    w2 = e.W * e.W
    assert ctx.n_p2 * w2 * 8 > SCRATCH_BYTES >= ctx.n_p1 * w2 * 8
    ctx.seek_plane(int(e.slice[0]))
    out = torch.full((geo.det_h.shape[0], w2), 7.0, dtype=torch.complex64, device="cuda")
    with pytest.raises(B.BipError) as ei:
        ctx.reconstruct_noalloc(0, 0, 2, B.RECON_LINEAR, out=out)
    assert ei.value.status == 5 and "BIP_NOALLOC_SCRATCH_BYTES" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())                             # refused before anything was launched
    with pytest.raises(B.BipError) as ei:
        ctx.reconstruct_noalloc(0, 0, 1, B.RECON_LINEAR, out=out)               # [n_det][w2] is not the S1 side's shape
    assert ei.value.status == 1
    got = ctx.reconstruct_noalloc(0, 0, 1, B.RECON_LINEAR)
    torch.cuda.synchronize()
    assert np.abs(got.cpu().numpy() - ctx.debug_reconstruct(0, 0, 1, B.RECON_LINEAR)).max() <= TOL
    ctx.close()
