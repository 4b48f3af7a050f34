"""Physical units -> the library's dimensionless parameters (host-side front end; Eqs. (1)-(11)).

The library integrates  phi'' + alpha phi' + sin phi = gamma(t) + sqrt(2 alpha T) xi(t)  with time in units of the inverse
plasma frequency 1/omega_p, omega_p = sqrt(2 e I0 / (hbar C)), and temperature in units of the Josephson energy
E_J = hbar I0 / (2 e).  The paper's own normalisation (time hbar/E_C, Eq. (5); beta, theta, V0 = E_J/E_C, Eqs. (6)-(9)) is the
same equation with time stretched by sqrt(V0):  alpha = beta / sqrt(V0),  T = theta / V0,  nu = d gamma / d(omega_p t').
"""
from __future__ import annotations

import math

HBAR = 1.054571817e-34          # J s      (CODATA 2018, exact SI)
E_CHARGE = 1.602176634e-19      # C
K_B = 1.380649e-23              # J / K


def junction_params(resistance_ohm: float, capacitance_f: float, critical_current_a: float, temperature_k: float,
                    ramp_time_s: float | None = None, gamma_start: float = 0.0, gamma_end: float = 1.0) -> dict:
    """Dimensionless (alpha, temperature, nu) of a junction; ramp_time_s is the time the bias takes from gamma_start to
    gamma_end (None: constant bias, nu = 0).  Also returns omega_p [1/s], E_J [J] and the paper's (beta, theta, V0)."""
    if min(resistance_ohm, capacitance_f, critical_current_a) <= 0 or temperature_k < 0:
        raise ValueError("R, C, I0 must be positive and T non-negative")
    omega_p = math.sqrt(2.0 * E_CHARGE * critical_current_a / (HBAR * capacitance_f))
    e_j = HBAR * critical_current_a / (2.0 * E_CHARGE)
    alpha = 1.0 / (resistance_ohm * capacitance_f * omega_p)
    temperature = K_B * temperature_k / e_j
    nu = 0.0 if ramp_time_s is None else (gamma_end - gamma_start) / (ramp_time_s * omega_p)
    e_c = (2.0 * E_CHARGE) ** 2 / capacitance_f
    return dict(alpha=alpha, temperature=temperature, nu=nu, omega_p=omega_p, e_j=e_j,
                beta=HBAR / (resistance_ohm * (2.0 * E_CHARGE) ** 2), theta=K_B * temperature_k / e_c, v0=e_j / e_c)
