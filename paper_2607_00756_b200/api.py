"""ctypes binding of libbip (include/bip.h): argument marshalling only.

Every function here has the name of the C entry point it calls.  PyTorch is used for device memory and the
CUDA stream, nothing else.  A missing ``libbip.so`` raises: there is no fallback path.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbip.so")

MODE_MAP, MODE_QEELS_X, MODE_QEELS_Y, MODE_CUBE = 0, 1, 2, 3
RECON_LINEAR, RECON_MAGPHASE = 0, 1
ASSOC_PROBE, ASSOC_COUPLING, ASSOC_AUTO = 0, 1, 2
PREC_TF32X3, PREC_FP32_SIMT, PREC_BF16X6, PREC_FP16X4, PREC_FP16X3 = 0, 1, 2, 3, 4
FFT_NATIVE, FFT_CUFFT_F64 = 0, 1
MAX_NN = 16
_STATUS = {1: "BIP_ERR_INVALID", 2: "BIP_ERR_STATE", 3: "BIP_ERR_OOM", 4: "BIP_ERR_CUDA", 5: "BIP_ERR_UNSUPPORTED"}


class BipError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


class _Grid(C.Structure):
    _fields_ = [("ny", C.c_int32), ("nx", C.c_int32), ("ly", C.c_double), ("lx", C.c_double), ("nz", C.c_int32),
                ("dz", C.c_double), ("lam", C.c_double)]


class _Weights(C.Structure):
    _fields_ = [("n_rows", C.c_int32), ("max_nn", C.c_int32), ("nn_idx", C.POINTER(C.c_int32)), ("nn_w", C.POINTER(C.c_float))]


class _Timing(C.Structure):
    _fields_ = [("build_s1_ms", C.c_float), ("build_s2_ms", C.c_float), ("advance_peel_ms", C.c_float),
                ("contract_ms", C.c_float), ("gemm2_ms", C.c_float), ("gemm2_launches", C.c_int32),
                ("kernel_launches", C.c_int32), ("amplitudes", C.c_double), ("flops", C.c_double)]


@dataclass(frozen=True)
class Grid:
    ny: int
    nx: int
    ly: float
    lx: float
    nz: int
    dz: float
    lam: float

    def c(self) -> _Grid:
        return _Grid(self.ny, self.nx, self.ly, self.lx, self.nz, self.dz, self.lam)


# every symbol include/bip.h declares (tests check that the library exports each of them)
ABI_SYMBOLS = (
    "bip_beams_in_disc", "bip_aperture_coeffs", "bip_hexring", "bip_n_radial_from_factor", "bip_sibson", "bip_create",
    "bip_destroy", "bip_last_error", "bip_build_S1", "bip_build_S2", "bip_set_scan", "bip_add_edge", "bip_clear_edges",
    "bip_output_size", "bip_map", "bip_map_host", "bip_map_all", "bip_get_windows", "bip_get_qeels_bins",
    "bip_seek_plane", "bip_copy_S", "bip_debug_reconstruct", "bip_get_timing", "bip_version", "bip_prism_subsample",
    "bip_set_crop", "bip_set_association", "bip_prism_coeffs", "bip_partition", "bip_set_scratch_budget", "bip_allow_tf32x3",
    "bip_get_parents", "bip_get_weights", "bip_set_fft_backend", "bip_cube_alg3", "bip_set_focal", "bip_get_focal_distance",
    "bip_set_transmission", "bip_set_accumulate", "bip_reconstruct_noalloc",
)

_lib: Optional[C.CDLL] = None


def load_library() -> C.CDLL:
    """dlopen libbip.so (built by ``python -m paper_2607_00756_b200.build``); raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2607_00756_b200.build` (there is no fallback path)")
    lib = C.CDLL(LIB_PATH)
    for name in ABI_SYMBOLS:
        getattr(lib, name).restype = C.c_int32
    lib.bip_version.restype = C.c_char_p
    lib.bip_last_error.restype = C.c_char_p
    lib.bip_last_error.argtypes = [C.c_void_p]
    _lib = lib
    return lib


def _check(status: int, ctx=None):
    if status != 0:
        raise BipError(status, load_library().bip_last_error(ctx).decode(errors="replace"))


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


def _p(a: np.ndarray, t):
    return a.ctypes.data_as(C.POINTER(t))


def bip_version() -> str:
    return load_library().bip_version().decode()


def bip_beams_in_disc(g: Grid, qmax: float) -> np.ndarray:
    lib = load_library()
    n = C.c_int32(0)
    gc = g.c()
    _check(lib.bip_beams_in_disc(C.byref(gc), C.c_double(qmax), None, 0, C.byref(n)))
    h = np.empty((n.value, 2), dtype=np.int32)
    _check(lib.bip_beams_in_disc(C.byref(gc), C.c_double(qmax), _p(h, C.c_int32), n.value, C.byref(n)))
    return h


def bip_aperture_coeffs(g: Grid, h: np.ndarray, defocus: float) -> np.ndarray:
    h = _i32(h)
    c = np.empty((h.shape[0], 2), dtype=np.float32)
    gc = g.c()
    _check(load_library().bip_aperture_coeffs(C.byref(gc), h.shape[0], _p(h, C.c_int32), C.c_double(defocus), _p(c, C.c_float)))
    return c


def bip_n_radial_from_factor(n_beams: int, factor: float) -> int:
    return int(load_library().bip_n_radial_from_factor(int(n_beams), C.c_double(factor)))


def bip_hexring(g: Grid, h: np.ndarray, qmax: float, n_radial: int, n_angular: int = 6) -> np.ndarray:
    h = _i32(h)
    n = C.c_int32(0)
    pos = np.empty(h.shape[0], dtype=np.int32)
    gc = g.c()
    _check(load_library().bip_hexring(C.byref(gc), h.shape[0], _p(h, C.c_int32), C.c_double(qmax), int(n_radial), int(n_angular),
                                      _p(pos, C.c_int32), pos.shape[0], C.byref(n)))
    return pos[: n.value].copy()


def bip_prism_subsample(h: np.ndarray, fy: int, fx: int) -> np.ndarray:
    """Positions of the beams kept by PRISM subsampling (h_y = 0 mod fy, h_x = 0 mod fx)."""
    h = _i32(h)
    keep = np.empty(h.shape[0], dtype=np.int32)
    n = C.c_int32(0)
    _check(load_library().bip_prism_subsample(h.shape[0], _p(h, C.c_int32), int(fy), int(fx), _p(keep, C.c_int32), keep.shape[0], C.byref(n)))
    return keep[: n.value].copy()


def bip_sibson(g: Grid, h: np.ndarray, parent_h: np.ndarray, qmax: float, max_nn: int = 8) -> Tuple[np.ndarray, np.ndarray]:
    h, parent_h = _i32(h), _i32(parent_h)
    idx = np.empty((h.shape[0], max_nn), dtype=np.int32)
    w = np.empty((h.shape[0], max_nn), dtype=np.float32)
    gc = g.c()
    _check(load_library().bip_sibson(C.byref(gc), h.shape[0], _p(h, C.c_int32), parent_h.shape[0], _p(parent_h, C.c_int32),
                                     C.c_double(qmax), int(max_nn), _p(idx, C.c_int32), _p(w, C.c_float)))
    return idx, w


def bip_prism_coeffs(keep: np.ndarray, c_full: np.ndarray, fy: int, fx: int) -> np.ndarray:
    """Coefficients of the retained beams rescaled by fy * fx."""
    keep = _i32(keep)
    c_full = np.ascontiguousarray(c_full, dtype=np.float32)
    out = np.empty((keep.shape[0], 2), dtype=np.float32)
    _check(load_library().bip_prism_coeffs(keep.shape[0], _p(keep, C.c_int32), c_full.shape[0], _p(c_full, C.c_float), int(fy), int(fx),
                                           _p(out, C.c_float)))
    return out


def bip_partition(g: Grid, h: np.ndarray, qmax: float, factor: float, max_nn: int = 8):
    """Parents (positions into h) and ELL weight table of a beam set for a parent factor (f = 1: identity)."""
    h = _i32(h)
    pos = np.empty(h.shape[0], dtype=np.int32)
    n = C.c_int32(0)
    idx = np.empty((h.shape[0], max_nn), dtype=np.int32)
    w = np.empty((h.shape[0], max_nn), dtype=np.float32)
    gc = g.c()
    _check(load_library().bip_partition(C.byref(gc), h.shape[0], _p(h, C.c_int32), C.c_double(qmax), C.c_double(factor), int(max_nn),
                                        _p(pos, C.c_int32), pos.shape[0], C.byref(n), _p(idx, C.c_int32), _p(w, C.c_float)))
    return pos[: n.value].copy(), (idx, w)


def _weights(idx: np.ndarray, w: np.ndarray):
    idx = _i32(idx)
    w = np.ascontiguousarray(w, dtype=np.float32)
    st = _Weights(idx.shape[0], idx.shape[1], _p(idx, C.c_int32), _p(w, C.c_float))
    return st, (idx, w)


@dataclass
class Geometry:
    """Beam sets, parents and weight tables of one (aperture, detector) pair, all produced by the library's helpers."""
    ap_h: np.ndarray
    ap_c: np.ndarray
    p1_pos: np.ndarray
    w1: Tuple[np.ndarray, np.ndarray]
    det_h: np.ndarray
    p2_pos: np.ndarray
    w2: Tuple[np.ndarray, np.ndarray]
    qa: float
    qd: float

    @property
    def p1_h(self):
        return self.ap_h[self.p1_pos]

    @property
    def p2_h(self):
        return self.det_h[self.p2_pos]


def plan_geometry(g: Grid, alpha_mrad: float, det_mrad: float, defocus: float, parent_factor: Sequence[float],
                  max_nn: int = 8, prism: Sequence[int] = (1, 1)) -> Geometry:
    """Aperture / detector beams (eq. 5), hex-ring parents and Sibson tables (eq. 8): a sequence of calls
    into the library (bip_beams_in_disc, bip_aperture_coeffs, bip_prism_subsample, bip_prism_coeffs, bip_partition) --
    no arithmetic here.  ``prism`` = (f_y, f_x) keeps every f-th beam of both sets."""
    qa, qd = alpha_mrad * 1e-3 / g.lam, det_mrad * 1e-3 / g.lam
    ap_h = bip_beams_in_disc(g, qa)
    det_h = bip_beams_in_disc(g, qd)
    ap_c = bip_aperture_coeffs(g, ap_h, defocus)
    if tuple(prism) != (1, 1):
        keep = bip_prism_subsample(ap_h, prism[0], prism[1])
        ap_h, ap_c = ap_h[keep], bip_prism_coeffs(keep, ap_c, prism[0], prism[1])
        det_h = det_h[bip_prism_subsample(det_h, prism[0], prism[1])]
    p1_pos, w1 = bip_partition(g, ap_h, qa, parent_factor[0], max_nn)
    p2_pos, w2 = bip_partition(g, det_h, qd, parent_factor[1], max_nn)
    return Geometry(ap_h, ap_c, p1_pos, w1, det_h, p2_pos, w2, qa, qd)


class Context:
    """Owner of a ``bip_ctx*``.  Methods are the C calls of the same name (``bip_`` prefix dropped)."""

    def __init__(self, g: Grid, T, ap_h, ap_c, p1_h, w1, p2_h, stream: Optional[int] = None):
        import torch
        self._lib = load_library()
        self.g = g
        self._ctx = C.c_void_p(None)
        ap_h, p1_h, p2_h = _i32(ap_h), _i32(p1_h), _i32(p2_h)
        ap_c = np.ascontiguousarray(ap_c, dtype=np.float32)
        w1s, keep = _weights(*w1) if w1 is not None else (None, None)     # None: the library computes the Sibson table
        if isinstance(T, np.ndarray):
            T = np.ascontiguousarray(T, dtype=np.complex64)
            assert T.shape == (g.nz, g.ny, g.nx)
            t_ptr, on_dev = T.ctypes.data, 0
        else:
            assert T.is_cuda and T.dtype == torch.complex64 and T.is_contiguous() and tuple(T.shape) == (g.nz, g.ny, g.nx)
            t_ptr, on_dev = T.data_ptr(), 1
        self._T = T                    # borrowed by the library: keep it alive
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0
        gc = g.c()
        _check(self._lib.bip_create(C.byref(self._ctx), C.byref(gc), C.c_void_p(t_ptr), on_dev, ap_h.shape[0],
                                    _p(ap_h, C.c_int32), _p(ap_c, C.c_float), p1_h.shape[0], _p(p1_h, C.c_int32),
                                    C.byref(w1s) if w1s is not None else None, p2_h.shape[0], _p(p2_h, C.c_int32), C.c_void_p(stream)))
        self.n_ap, self.n_p1, self.n_p2 = ap_h.shape[0], p1_h.shape[0], p2_h.shape[0]
        self.n_rho = 0
        self._edges = []

    def _ck(self, st):
        _check(st, self._ctx)

    def close(self):
        if self._ctx:
            self._lib.bip_destroy(self._ctx)
            self._ctx = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def build_S1(self):
        self._ck(self._lib.bip_build_S1(self._ctx))

    def build_S2(self):
        self._ck(self._lib.bip_build_S2(self._ctx))

    def set_scan(self, rho_px: np.ndarray):
        rho = np.ascontiguousarray(rho_px, dtype=np.float64)
        self._ck(self._lib.bip_set_scan(self._ctx, rho.shape[0], _p(rho, C.c_double)))
        self.n_rho = rho.shape[0]

    def set_association(self, assoc: int):
        """Probe-first (default), coupling-matrix (eq. 13 as printed) or automatic association of the contraction."""
        self._ck(self._lib.bip_set_association(self._ctx, int(assoc)))

    def set_crop(self, fy: int, fx: int):
        """PRISM crop mask: sites contribute only to the scans within N / (2 f) of them; (1, 1) = off."""
        self._ck(self._lib.bip_set_crop(self._ctx, int(fy), int(fx)))

    def set_scratch_budget(self, n_bytes: int):
        self._ck(self._lib.bip_set_scratch_budget(self._ctx, C.c_size_t(int(n_bytes))))

    def set_fft_backend(self, backend: int):
        """Slice-step route: FFT_NATIVE (fused fp32 kernels, power-of-two grids) or FFT_CUFFT_F64."""
        self._ck(self._lib.bip_set_fft_backend(self._ctx, int(backend)))

    def set_focal(self, on: bool = True):
        """S1 focal back-propagation to the scattering-centroid plane (NEXT-4; include/bip.h)."""
        self._ck(self._lib.bip_set_focal(self._ctx, int(bool(on))))

    def get_focal_distance(self, plane: int) -> float:
        d = C.c_double(0.0)
        self._ck(self._lib.bip_get_focal_distance(self._ctx, int(plane), C.byref(d)))
        return d.value

    def set_accumulate(self, on: bool = True):
        self._ck(self._lib.bip_set_accumulate(self._ctx, int(bool(on))))

    def set_transmission(self, T):
        """Replace the transmission functions (frozen-phonon configurations); S1 / S2 must be rebuilt afterwards."""
        import torch
        g = self.g
        if isinstance(T, np.ndarray):
            T = np.ascontiguousarray(T, dtype=np.complex64)
            assert T.shape == (g.nz, g.ny, g.nx)
            self._ck(self._lib.bip_set_transmission(self._ctx, C.c_void_p(T.ctypes.data), 0))
        else:
            assert T.is_cuda and T.dtype == torch.complex64 and T.is_contiguous() and tuple(T.shape) == (g.nz, g.ny, g.nx)
            self._ck(self._lib.bip_set_transmission(self._ctx, C.c_void_p(T.data_ptr()), 1))
        self._T = T

    def allow_tf32x3(self, allow: bool = True):
        self._ck(self._lib.bip_allow_tf32x3(self._ctx, int(bool(allow))))

    def add_edge(self, slice_, centre_px, H, det_h, w2=None) -> int:
        slice_, centre_px, det_h = _i32(slice_), _i32(centre_px), _i32(det_h)
        H = np.ascontiguousarray(H, dtype=np.complex64)
        w2s, keep = _weights(*w2) if w2 is not None else (None, None)     # None: the library computes the Sibson table
        eid = C.c_int32(-1)
        self._ck(self._lib.bip_add_edge(self._ctx, slice_.shape[0], _p(slice_, C.c_int32), _p(centre_px, C.c_int32), H.shape[0],
                                        H.shape[1], C.c_void_p(H.ctypes.data), det_h.shape[0], _p(det_h, C.c_int32),
                                        C.byref(w2s) if w2s is not None else None, C.byref(eid)))
        self._edges.append((slice_.shape[0], H.shape[0], H.shape[1], det_h.shape[0]))
        return eid.value

    def clear_edges(self):
        self._ck(self._lib.bip_clear_edges(self._ctx))
        self._edges = []

    def output_size(self, edge_id: int, mode: int) -> Tuple[int, int]:
        n, nb = C.c_int64(0), C.c_int32(0)
        self._ck(self._lib.bip_output_size(self._ctx, edge_id, mode, C.byref(n), C.byref(nb)))
        return n.value, nb.value

    def _shape(self, edge_id, mode):
        n, nb = self.output_size(edge_id, mode)
        if mode == MODE_MAP:
            return (self.n_rho,), np.float64
        return (self.n_rho, n // self.n_rho), np.float32

    def map(self, edge_id: int, mode: int = MODE_MAP, recon: int = RECON_LINEAR, precision: int = PREC_FP16X4, out=None):
        """bip_map into a torch CUDA tensor (allocated here unless given); returns it without synchronising."""
        import torch
        shape, dt = self._shape(edge_id, mode)
        tdt = torch.float64 if dt == np.float64 else torch.float32
        if out is None:
            out = torch.empty(shape, dtype=tdt, device="cuda")
        assert out.is_cuda and out.is_contiguous() and out.dtype == tdt and tuple(out.shape) == shape
        self._ck(self._lib.bip_map(self._ctx, edge_id, mode, recon, precision, C.c_void_p(out.data_ptr()),
                                   C.c_size_t(out.numel() * out.element_size())))
        return out

    def cube_alg3(self, edge_id: int, recon: int = RECON_LINEAR, precision: int = PREC_FP16X4, out=None):
        """bip_cube_alg3: the S1-partitioned 4D cube on all exit beams, float32 [n_rho, ny, nx] (torch CUDA tensor)."""
        import torch
        shape = (self.n_rho, self.g.ny, self.g.nx)
        if out is None:
            out = torch.empty(shape, dtype=torch.float32, device="cuda")
        assert out.is_cuda and out.is_contiguous() and out.dtype == torch.float32 and tuple(out.shape) == shape
        self._ck(self._lib.bip_cube_alg3(self._ctx, int(edge_id), int(recon), int(precision), C.c_void_p(out.data_ptr()),
                                         C.c_size_t(out.numel() * 4)))
        return out

    def map_all(self, mode: int = MODE_MAP, recon: int = RECON_LINEAR, precision: int = PREC_FP16X4):
        import torch
        outs = []
        for e in range(len(self._edges)):
            shape, dt = self._shape(e, mode)
            outs.append(torch.empty(shape, dtype=torch.float64 if dt == np.float64 else torch.float32, device="cuda"))
        ptrs = (C.c_void_p * len(outs))(*[o.data_ptr() for o in outs])
        sizes = (C.c_size_t * len(outs))(*[o.numel() * o.element_size() for o in outs])
        self._ck(self._lib.bip_map_all(self._ctx, mode, recon, precision, ptrs, sizes, len(outs)))
        return outs

    def map_host(self, edge_id: int, mode: int = MODE_MAP, recon: int = RECON_LINEAR, precision: int = PREC_FP16X4) -> np.ndarray:
        shape, dt = self._shape(edge_id, mode)
        out = np.empty(shape, dtype=dt)
        self._ck(self._lib.bip_map_host(self._ctx, edge_id, mode, recon, precision, C.c_void_p(out.ctypes.data), C.c_size_t(out.nbytes)))
        return out

    def get_parents(self, which: int) -> np.ndarray:
        n = C.c_int32(0)
        self._ck(self._lib.bip_get_parents(self._ctx, int(which), None, 0, C.byref(n)))
        h = np.empty((n.value, 2), dtype=np.int32)
        self._ck(self._lib.bip_get_parents(self._ctx, int(which), _p(h, C.c_int32), n.value, C.byref(n)))
        return h

    def get_weights(self, edge_id: int = -1) -> Tuple[np.ndarray, np.ndarray]:
        """ELL table in use: edge_id < 0: w1; else the edge's w2."""
        rows, nn = C.c_int32(0), C.c_int32(0)
        self._ck(self._lib.bip_get_weights(self._ctx, int(edge_id), C.byref(rows), C.byref(nn), None, None))
        idx = np.empty((rows.value, nn.value), dtype=np.int32)
        w = np.empty((rows.value, nn.value), dtype=np.float32)
        self._ck(self._lib.bip_get_weights(self._ctx, int(edge_id), C.byref(rows), C.byref(nn), _p(idx, C.c_int32), _p(w, C.c_float)))
        return idx, w

    def get_windows(self, edge_id: int) -> np.ndarray:
        o = np.empty((self._edges[edge_id][0], 2), dtype=np.int32)
        self._ck(self._lib.bip_get_windows(self._ctx, edge_id, _p(o, C.c_int32)))
        return o

    def get_qeels_bins(self, edge_id: int, mode: int) -> np.ndarray:
        _, nb = self.output_size(edge_id, mode)
        b = np.empty(nb, dtype=np.int32)
        self._ck(self._lib.bip_get_qeels_bins(self._ctx, edge_id, mode, _p(b, C.c_int32)))
        return b

    def seek_plane(self, plane: int):
        self._ck(self._lib.bip_seek_plane(self._ctx, int(plane)))

    def copy_S(self, which: int, p0: int, n: int) -> np.ndarray:
        out = np.empty((n, self.g.ny, self.g.nx), dtype=np.complex64)
        self._ck(self._lib.bip_copy_S(self._ctx, which, p0, n, C.c_void_p(out.ctypes.data)))
        return out

    def debug_reconstruct(self, edge_id: int, atom: int, which: int, recon: int = RECON_LINEAR) -> np.ndarray:
        n_at, n_ch, w, n_det = self._edges[edge_id]
        rows = self.n_ap if which == 1 else n_det
        out = np.empty((rows, w * w), dtype=np.complex64)
        self._ck(self._lib.bip_debug_reconstruct(self._ctx, edge_id, atom, which, recon, C.c_void_p(out.ctypes.data)))
        return out

    def reconstruct_noalloc(self, edge_id: int, atom: int, which: int, recon: int = RECON_LINEAR, out=None):
        """bip_reconstruct_noalloc: as debug_reconstruct, into the caller's DEVICE tensor ``out`` (complex64 [rows][w*w]; made
        here when None -- the library itself allocates nothing), enqueued on the context's stream without synchronising."""
        import torch
        n_at, n_ch, w, n_det = self._edges[edge_id]
        rows = self.n_ap if which == 1 else n_det
        if out is None:
            out = torch.empty((rows, w * w), dtype=torch.complex64, device="cuda")
        assert out.is_cuda and out.is_contiguous() and out.dtype == torch.complex64
        self._ck(self._lib.bip_reconstruct_noalloc(self._ctx, edge_id, atom, which, recon, C.c_void_p(out.data_ptr()),
                                                   C.c_size_t(out.numel() * out.element_size())))
        return out

    def get_timing(self) -> dict:
        t = _Timing()
        self._ck(self._lib.bip_get_timing(self._ctx, C.byref(t)))
        return {k: getattr(t, k) for k, _ in _Timing._fields_}
