"""CPU ORACLE of the sub-grid star-formation / energy-injection step (section 2.4, :226-283) and its transpose.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's CPU legs may import this
module; it never imports the CUDA package and shares no code with it.  Plain numpy, fp64, in the paper's order:

  class probability (Eq. 25, :279):   pi0 = Pi0 sigma((delta - delta_c)/a) sigma((T_c - T)/b),   sigma(x) = 1/(1 + e^-x)
  relaxed Bernoulli (Eq. 24, :265):   z = e^{(log pi0 + g0)/tau} / (e^{(log pi0 + g0)/tau} + e^{(log(1 - pi0) + g1)/tau})
  with g0, g1 ~ Gumbel(0, 1) supplied as INPUTS (Eq. 22-23, :253-263), tau = 0.1 in the paper (:273);
  energy injection (:236): the feedback energy heats the gas of the cell, eps += e_inject * rho * z.
Readings (R29-R32): delta = rho/rho_mean_gas - 1 is the gas overdensity; T = t_per_e * e~ with
e~ = eps/rho - |m|^2/(2 rho^2) (reading R27; the caller folds (gamma-1) mu m_p/(k_B a^2) into t_per_e); E_0 is an energy
per unit star-forming gas mass and the caller folds a^2 and units into e_inject; Eq. 24 is evaluated as the logistic
function of its log-odds (identical in exact arithmetic, no overflow at tau = 0.1).
Pins (tests/test_oracle_subgrid.py): Eq. 24 retyped literally; tau -> 0 gives the Gumbel-max indicator whose mean over
draws is pi0; a, b -> 0 gives the sharp thresholds of :232; the transpose against central finite differences.
"""
from __future__ import annotations

import numpy as np


def _log_sigmoid(x):
    return -(np.maximum(-x, 0.0) + np.log1p(np.exp(-np.abs(x))))


def _sigmoid(x):
    return np.exp(_log_sigmoid(x))


def class_probability(rho, T, rho_mean, T_c, delta_c, Pi0, a_w, b_w):
    """Eq. 25."""
    delta = np.asarray(rho, dtype=np.float64) / rho_mean - 1.0
    return Pi0 * _sigmoid((delta - delta_c) / a_w) * _sigmoid((T_c - np.asarray(T, dtype=np.float64)) / b_w)


def relaxed_bernoulli(pi0, g0, g1, tau):
    """Eq. 24 as sigma(((log pi0 + g0) - (log(1 - pi0) + g1)) / tau)."""
    return _sigmoid((np.log(pi0) - np.log1p(-pi0) + g0 - g1) / tau)


def temperature(gas, t_per_e):
    g = np.asarray(gas, dtype=np.float64)
    return t_per_e * (g[4] / g[0] - 0.5 * np.sum(g[1:4] ** 2, axis=0) / g[0] ** 2)


def step(gas, g0, g1, rho_mean, t_per_e, T_c, delta_c, Pi0, e_inject, a_w, b_w, tau):
    """gas (5,N,N,N) -> (gas_out, z): eps_out = eps + e_inject rho z; the other fields unchanged."""
    g = np.array(gas, dtype=np.float64)
    pi0 = class_probability(g[0], temperature(g, t_per_e), rho_mean, T_c, delta_c, Pi0, a_w, b_w)
    z = relaxed_bernoulli(pi0, np.asarray(g0, dtype=np.float64), np.asarray(g1, dtype=np.float64), tau)
    g[4] = g[4] + e_inject * g[0] * z
    return g, z


def step_vjp(gas, g0, g1, rho_mean, t_per_e, T_c, delta_c, Pi0, e_inject, a_w, b_w, tau, cot_gas, cot_z=None):
    """Transpose of `step` at `gas` (the state BEFORE the injection): returns (cot_gas_in, dparams) with
    dparams = (dT_c, ddelta_c, dPi0, de_inject)."""
    g = np.asarray(gas, dtype=np.float64)
    cg = np.array(cot_gas, dtype=np.float64)
    rho, m, eps = g[0], g[1:4], g[4]
    m2 = np.sum(m * m, axis=0)
    T = t_per_e * (eps / rho - 0.5 * m2 / rho ** 2)
    x = (rho / rho_mean - 1.0 - delta_c) / a_w
    y = (T_c - T) / b_w
    ell = np.log(Pi0) + _log_sigmoid(x) + _log_sigmoid(y)
    pi0 = np.exp(ell)
    z = _sigmoid((ell - np.log1p(-pi0) + np.asarray(g0, dtype=np.float64) - np.asarray(g1, dtype=np.float64)) / tau)
    z_b = cg[4] * e_inject * rho + (0.0 if cot_z is None else np.asarray(cot_z, dtype=np.float64))
    de = np.sum(cg[4] * rho * z)
    out = cg.copy()
    out[0] += cg[4] * e_inject * z
    ell_b = z_b * z * (1.0 - z) / (tau * (1.0 - pi0))
    x_b = ell_b * _sigmoid(-x)
    y_b = ell_b * _sigmoid(-y)
    dPi0 = np.sum(ell_b) / Pi0
    ddc = -np.sum(x_b) / a_w
    dTc = np.sum(y_b) / b_w
    out[0] += x_b / (a_w * rho_mean)
    e_b = -y_b / b_w * t_per_e                      # cotangent of e~
    out[4] += e_b / rho
    out[1:4] += -e_b[None] * m / rho[None] ** 2
    out[0] += e_b * (-eps / rho ** 2 + m2 / rho ** 3)
    return out, np.array([dTc, ddc, dPi0, de])
