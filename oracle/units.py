"""ORACLE (test infrastructure, not product code) -- the paper's normalisation, Eqs. (4)-(9), step by step.

E_C = (2e)^2 / C; time unit hbar / E_C (5); beta = hbar / (R (2e)^2) (6); theta = k_B T / E_C (8); V0 = E_J / E_C with
E_J = I0 hbar / (2e) (9).  Eq. (9) is  phi'' + beta phi' = V0 (-sin phi + gamma + gamma_N),  <gamma_N gamma_N> = 2 beta theta delta.
Rescaling time by s = sqrt(V0) (tau = s t) gives the library's form  phi'' + (beta/s) phi' + sin phi = gamma + noise  whose noise
correlator is 2 (beta/s) (theta/V0) delta(tau): alpha = beta / sqrt(V0), T = theta / V0 (for V0 = 1 the two forms coincide, R2).
"""
import math

HBAR = 1.054571817e-34
QE = 1.602176634e-19
KB = 1.380649e-23


def paper_normalisation(R, C, I0, T):
    EC = (2 * QE) ** 2 / C
    beta = (1.0 / R) * HBAR / (2 * QE) ** 2
    theta = KB * T / EC
    EJ = I0 * HBAR / (2 * QE)
    V0 = EJ / EC
    time_unit = HBAR / EC
    return dict(beta=beta, theta=theta, V0=V0, time_unit=time_unit, D=beta * theta)


def library_parameters(R, C, I0, T, ramp_time=None):
    n = paper_normalisation(R, C, I0, T)
    s = math.sqrt(n["V0"])
    out = dict(alpha=n["beta"] / s, temperature=n["theta"] / n["V0"], omega_p=s / n["time_unit"])
    out["nu"] = 0.0 if ramp_time is None else 1.0 / (ramp_time / n["time_unit"] * s)
    return out
