"""Physical units of the paper's water model <-> reduced Lennard-Jones units.

sigma = 3.17 Angstrom, epsilon = 6.74e-3 eV, m = 18.015 u (one water molecule).  Reduced time unit
tau = sigma sqrt(m / epsilon) = 1.668 ps, so the paper's dt = 0.016 ps is 0.00959 tau and its Berendsen rise times
tau_B in [0.1, 2] ps are 0.06-1.2 tau; T* = k_B T / epsilon = 3.94 at 35 C, 3.81 at 25 C.
"""
import math

SIGMA_M = 3.17e-10
EPSILON_J = 6.74e-3 * 1.602176634e-19
MASS_KG = 18.015 * 1.66053906660e-27
K_B = 1.380649e-23
TAU_S = SIGMA_M * math.sqrt(MASS_KG / EPSILON_J)


def length_reduced(metres: float) -> float:
    return metres / SIGMA_M


def time_reduced(seconds: float) -> float:
    return seconds / TAU_S


def temperature_reduced(celsius: float) -> float:
    return K_B * (celsius + 273.15) / EPSILON_J


PAPER_DT = time_reduced(0.016e-12)
