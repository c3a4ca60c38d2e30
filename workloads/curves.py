"""Smooth synthetic stand-ins for the tabulated curves the paper takes as input.

The paper uses a Boone-Seibert spectrum, NIST-like mass-attenuation tables and a
measured detector response (Fig. 2); none is in the
container.  These analytic curves have the same general shape (photo-electric
~E^-3 plus a Klein-Nishina Compton term; Kramers bremsstrahlung filtered by Al)
and no K-edges.  They are inputs, not part of the projector's arithmetic.
All energies in keV, lengths in mm, mu in mm^-1 (per g/cm^3 for mu_hat).
"""
import numpy as np

M_E_C2_KEV = 510.99895


def klein_nishina(E):
    """Klein-Nishina total cross-section per electron, up to a constant factor
    (SURVEY.md section 8(d) 'Fixed synthetic curves')."""
    k = np.asarray(E, dtype=np.float64) / M_E_C2_KEV
    l = np.log1p(2.0 * k)
    return ((1.0 + k) / k**2 * (2.0 * (1.0 + k) / (1.0 + 2.0 * k) - l / k)
            + l / (2.0 * k) - (1.0 + 3.0 * k) / (1.0 + 2.0 * k) ** 2)


def _pe_kn(E, a, b):
    """a*(E/60)^-3 + b*KN(E)/KN(60): a, b are the photo-electric and Compton
    parts at 60 keV."""
    E = np.asarray(E, dtype=np.float64)
    return a * (E / 60.0) ** -3 + b * klein_nishina(E) / klein_nishina(60.0)


def mu_al(E):
    """Linear attenuation of the Al stand-in, mm^-1 (0.075 at 60 keV)."""
    return _pe_kn(E, 0.034, 0.041)


def mu_csi(E):
    """Linear attenuation of the CsI stand-in, mm^-1."""
    return _pe_kn(E, 3.1, 0.06)


def mu_hat_curve(E, a, b):
    """Mass-attenuation curve of a material, mm^-1 per g/cm^3."""
    return _pe_kn(E, a, b)


def kramers_spectrum(E, e_max, al_mm=2.5):
    """Per-bin probabilities phi_E ~ max(Emax-E,0)/E * exp(-mu_Al(E)*al_mm),
    normalised to sum 1 (the spectrum is normalised)."""
    E = np.asarray(E, dtype=np.float64)
    w = np.maximum(e_max - E, 0.0) / E * np.exp(-mu_al(E) * al_mm)
    return w / w.sum()


def response_linear(E):
    """Energy-integrating ideal detector: R(E) = E."""
    return np.asarray(E, dtype=np.float64).copy()


def response_csi(E, thickness_mm=0.6):
    """R(E) = E * (1 - exp(-mu_CsI(E) * thickness))."""
    E = np.asarray(E, dtype=np.float64)
    return E * (1.0 - np.exp(-mu_csi(E) * thickness_mm))


def bowtie_thickness(nu, du_mm):
    """Al thickness seen by detector column i: t = min(30, 2 + 28*(u_i/u_max)^2)
    mm, u_i the column centre, u_max = nu*du/2."""
    u = (np.arange(nu, dtype=np.float64) - 0.5 * (nu - 1)) * du_mm
    u_max = 0.5 * nu * du_mm
    return np.minimum(30.0, 2.0 + 28.0 * (u / u_max) ** 2)
