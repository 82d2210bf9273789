"""B200-native BiP-PRISM on-atom contraction (arxiv/paper_2607_00756).

``libbip.so`` (hand-written CUDA for sm_100a behind the C ABI of ``include/bip.h``) does all of the work; this
package is a thin ctypes binding with the same names.  There is no CPU fallback: importing works anywhere,
but every call that touches a scattering matrix needs the built library and a B200.
"""
from .api import (  # noqa: F401
    ASSOC_PROBE, ASSOC_COUPLING, ASSOC_AUTO, FFT_NATIVE, FFT_CUFFT_F64, BipError, Context, Grid, MODE_MAP, MODE_QEELS_X, MODE_QEELS_Y, MODE_CUBE, RECON_LINEAR, RECON_MAGPHASE,
    PREC_TF32X3, PREC_FP32_SIMT, PREC_BF16X6, PREC_FP16X4, PREC_FP16X3, bip_aperture_coeffs, bip_beams_in_disc, bip_hexring, bip_prism_subsample, bip_n_radial_from_factor,
    bip_partition, bip_prism_coeffs, bip_sibson, bip_version, load_library, plan_geometry,
)
