"""Temperature moments of PAPER.md sec. 6.1 (lines 238-252), shared by the oracle pins (P10, P11) and the GPU relaxation
tests.  In the units of this repo (v in v0, T in T0 = m0 v0^2 / 2, theta = T/m, reading A8) and with
`mf` = M f the mass-matrix-weighted nodal vector of one species (so that psi^T mf = int psi f r dr dz):

    n        = 2 pi  1^T mf
    T_perp   = m <r^2>             (paper: m v0^2 int f v_perp v_perp^2 / (2 int f v_perp))
    T_par    = 2 m <(z - u)^2>     (paper: m v0^2 int f v_perp (v_par - u)^2 / int f v_perp)
    T        = (2 T_perp + T_par) / 3

The same weights applied to rhs = J[f] f give the time derivatives (M df/dt = rhs), no solve needed."""
import math

import numpy as np


def temperatures(mf, r, z, mass, u=0.0):
    """(n, T_perp, T_par) from mf = M f."""
    n = mf.sum()
    return 2.0 * math.pi * n, mass * ((r ** 2) @ mf) / n, 2.0 * mass * (((z - u) ** 2) @ mf) / n


def temperature_rates(mf, rhs, r, z, mass, u=0.0):
    """(dT_perp/dt, dT_par/dt) from rhs = J[f] f (density is conserved, so n is constant)."""
    n = mf.sum()
    return mass * ((r ** 2) @ rhs) / n, 2.0 * mass * (((z - u) ** 2) @ rhs) / n


def nrl_isotropization_rate(c_iso, n, mass, t_perp, t_par):
    """nu_T t0 of PAPER.md App. B (lines 427-431) in the units of eq. (2.2); c_iso from tests/golden/nrl_rates.txt."""
    A = t_perp / t_par - 1.0
    return c_iso * n * mass ** -0.5 * t_par ** -1.5 * (-3.0 + (A + 3.0) * math.atan(math.sqrt(A)) / math.sqrt(A)) / A ** 2


def nrl_equilibration_rate(c_eq, za, zb, n_b, m_a, m_b, t_a, t_b):
    """nu_bar t0 of PAPER.md App. B (lines 435-439); c_eq from tests/golden/nrl_rates.txt."""
    return c_eq * za ** 2 * zb ** 2 * n_b * math.sqrt(m_a * m_b) / (m_a * t_b + m_b * t_a) ** 1.5


def golden_rates(path):
    vals = {}
    for line in open(path):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()[:2]
            vals[k] = float(v)
    return vals


def rk4(rate, y, dt, nsteps):
    out = [np.array(y, dtype=float)]
    y = out[0].copy()
    for _ in range(nsteps):
        k1 = rate(y)
        k2 = rate(y + 0.5 * dt * k1)
        k3 = rate(y + 0.5 * dt * k2)
        k4 = rate(y + dt * k3)
        y = y + dt * (k1 + 2 * k2 + 2 * k3 + k4) / 6
        out.append(y.copy())
    return np.array(out)
