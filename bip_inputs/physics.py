"""Textbook relativistic electron constants (inputs, not method arithmetic).

SURVEY.md §8(c) "constants": lambda(200 kV)=0.025079 A, lambda(300 kV)=0.019687 A,
sigma = 7.288e-4 / 6.526e-4 rad V^-1 A^-1.
"""
import math

M0C2_EV = 510998.95      # electron rest energy / eV
HC_EV_A = 12398.4198     # h c / (eV Angstrom)


def electron_wavelength(kv: float) -> float:
    """Relativistic de Broglie wavelength in Angstrom for an acceleration voltage in kV."""
    e = kv * 1e3
    return HC_EV_A / math.sqrt(e * (2.0 * M0C2_EV + e))


def interaction_constant(kv: float) -> float:
    """sigma in rad / (V Angstrom): 2 pi / (lambda E) * (m0c2 + E) / (2 m0c2 + E)."""
    e = kv * 1e3
    lam = electron_wavelength(kv)
    return 2.0 * math.pi / (lam * e) * (M0C2_EV + e) / (2.0 * M0C2_EV + e)
