"""Host-side check of the shared-memory layout of the native slice step (paper_2607_00756_b200/csrc/bip_fft.cu): the XOR swizzle
slot(i) = i ^ g(bits 4-6 of i) with the masks the kernel uses must (a) be a permutation of every line, (b) put the 16 lanes of a
half-warp on 16 different 8-byte bank pairs in every access pattern of every stage of every transform length (the claim in the
kernel's header comment: "found by exhaustive search"), and (c) together with the stage offsets (XOR part + ADD part) reproduce a
DFT in the digit-reversed order the propagator tables are stored in.  Pure Python / NumPy; no GPU, no library call."""
import numpy as np
import pytest

NT = 256


def masks(ln):
    return (3 if ln % 3 == 1 else 1), (2 if ln % 3 == 0 else 4 if ln % 3 == 1 else 6), (12 if ln % 3 == 0 else 8)


def swz_g(ln, i):
    m4, m5, m6 = masks(ln)
    g = 0
    if ln > 4: g ^= ((i >> 4) & 1) * m4
    if ln > 5: g ^= ((i >> 5) & 1) * m5
    if ln > 6: g ^= ((i >> 6) & 1) * m6
    return g


def slot(ln, i):
    return i ^ swz_g(ln, i)


def stages(ln):
    out, l = [], ln
    while l >= 3:
        out.append((8, l)); l -= 3
    if l:
        out.append((1 << l, l))
    return out


def stage_offsets(ln, r, ll, v):
    """byte offsets of the r elements of butterfly v, as the kernel forms them: (p0 ^ XK) + AK"""
    lr = {8: 3, 4: 2, 2: 1}[r]
    lsub = ll - lr
    blk, j = v >> lsub, v & ((1 << lsub) - 1)
    p0 = 8 * slot(ln, (blk << ll) + j)
    xk = [8 * swz_g(ln, k << lsub) if lsub >= 4 else 8 * slot(ln, k << lsub) for k in range(r)]
    ak = [8 * (k << lsub) if lsub >= 4 else 0 for k in range(r)]
    return [(p0 ^ x) + a for x, a in zip(xk, ak)]


@pytest.mark.parametrize("ln", range(3, 13))
def test_swizzle_is_a_permutation_and_conflict_free(ln):
    n = 1 << ln
    assert sorted(slot(ln, i) for i in range(n)) == list(range(n))
    worst = 1
    for s in range(0, min(n, 512), 16):                                  # contiguous runs (copies, long-stride stages)
        worst = max(worst, 17 - len({slot(ln, s + t) % 16 for t in range(16)}))
    for r, ll in stages(ln):
        nv = n // r
        for v0 in range(0, min(nv, 256), 16):
            lanes = [stage_offsets(ln, r, ll, v) for v in range(v0, min(v0 + 16, nv))]
            for k in range(r):
                banks = [(o[k] // 8) % 16 for o in lanes]
                worst = max(worst, len(banks) - len(set(banks)) + 1)
    assert worst == 1, f"bank conflict of degree {worst} at N = {n}"


def dif_frequency(pos, n):
    if n == 1:
        return 0
    r = 8 if n >= 8 else n
    sub = n // r
    return r * dif_frequency(pos % sub, sub) + pos // sub


@pytest.mark.parametrize("ln", [3, 4, 5, 7, 9])
def test_stage_offsets_give_the_dft_in_digit_reversed_order(ln):
    n = 1 << ln
    rng = np.random.default_rng(ln)
    x = rng.normal(size=n) + 1j * rng.normal(size=n)
    sm = np.zeros(n, complex)
    for i in range(n):
        sm[slot(ln, i)] = x[i]
    for r, ll in stages(ln):                                            # forward (DIF): butterfly, then twiddle w_L^(j m)
        lsub = ll - {8: 3, 4: 2, 2: 1}[r]
        k = np.arange(r)
        W = np.exp(-2j * np.pi * np.outer(k, k) / r)
        for v in range(n // r):
            offs = [o // 8 for o in stage_offsets(ln, r, ll, v)]
            y = W @ sm[offs]
            if r == 8 and lsub > 0:
                y = y * np.exp(-2j * np.pi * (v & ((1 << lsub) - 1)) * k / (1 << ll))
            sm[offs] = y
    got = np.zeros(n, complex)
    for p in range(n):
        got[dif_frequency(p, n)] = sm[slot(ln, p)]
    assert np.abs(got - np.fft.fft(x)).max() < 1e-9 * n
