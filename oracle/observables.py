"""Oracle side of the host-derived observables (R10) -- TEST INFRASTRUCTURE ONLY.

Everything is computed in exact rational arithmetic (Python ints / Fraction) from the integer
energy series and histograms and converted to double once, so each value is the correctly
rounded double of its definition:

  e    = E / N                                               (energy per spin)
  m    = (q N_max / N - 1) / (q - 1)                          (Eq. 7; the extracted
                                                               text prints q(N_max/N - 1), which would
                                                               give m = 0 for the ordered state --
                                                               DESIGN.md reading G4)
  C_v  = (<E^2> - <E>^2) / (N T^2)                            (fluctuation formula, k_B = 1;
                                                               Binder's criterion)
  V_L  = 1 - <E^4> / (3 <E^2>^2)                              (Eq. 9)

<.> is the plain mean over the series handed in.  T enters as the exact rational value of the
double that was passed.
"""
from __future__ import annotations

from fractions import Fraction


def energy_per_spin(E: int, N: int) -> float:
    return float(Fraction(int(E), int(N)))


def magnetisation(hist, q: int) -> float:
    counts = [int(c) for c in hist]
    N = sum(counts)
    return float((Fraction(q * max(counts), N) - 1) / (q - 1))


def specific_heat(E_series, N: int, T: float) -> float:
    Es = [int(e) for e in E_series]
    n = len(Es)
    s1 = sum(Es)
    s2 = sum(e * e for e in Es)
    Tq = Fraction(float(T))
    return float(Fraction(n * s2 - s1 * s1, n * n) / (N * Tq * Tq))


def binder_cumulant(E_series) -> float:
    Es = [int(e) for e in E_series]
    n = len(Es)
    s2 = sum(e * e for e in Es)
    s4 = sum(e ** 4 for e in Es)
    return float(1 - Fraction(n * s4, 3 * s2 * s2))


def mean_energy_per_spin(E_series, N: int) -> float:
    Es = [int(e) for e in E_series]
    return float(Fraction(sum(Es), len(Es) * N))


def magnetisation_moments(hist_series, q: int):
    """(<m>, <m^2>) of the order parameter m (Eq. 7, reading G4) over a series of q-bin histograms,
    in exact rational arithmetic: m_k = (q Nmax_k - N) / ((q - 1) N)."""
    ms = []
    for hist in hist_series:
        counts = [int(c) for c in hist]
        N = sum(counts)
        ms.append((Fraction(q * max(counts), N) - 1) / (q - 1))
    n = len(ms)
    m1 = sum(ms, Fraction(0)) / n
    m2 = sum((m * m for m in ms), Fraction(0)) / n
    return float(m1), float(m2)


def susceptibility(hist_series, q: int, T: float) -> float:
    """chi = N / T (<m^2> - <m>^2) (Eq. 11), exact rationals, one conversion at the end."""
    ms, N = [], None
    for hist in hist_series:
        counts = [int(c) for c in hist]
        N = sum(counts)
        ms.append((Fraction(q * max(counts), N) - 1) / (q - 1))
    n = len(ms)
    m1 = sum(ms, Fraction(0)) / n
    m2 = sum((m * m for m in ms), Fraction(0)) / n
    return float(N * (m2 - m1 * m1) / Fraction(float(T)))
