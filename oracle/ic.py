"""CPU ORACLE of the two ends of the path: the initial-condition map  delta_init -> (gas, particles)  with its
transpose, and (at the bottom) the data term of Eq. 27 with its cotangent.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module; it never imports the CUDA package and shares no code with it.

What it follows.  PAPER.md:49 (section 2.1): "initial conditions ... evolved with Lagrangian perturbation theory"; the
paper's Eisenstein-Hu spectrum and its LPT code are not available, so reading R19 of DESIGN.md takes first-order LPT
(the Zel'dovich map) of a given density contrast delta at scale factor a0, in plain numpy fp64 with numpy's FFT as the
library step:
    psi^_d(k) = i k~_d delta^(k) / k^2          (div psi = -delta; k~_d = 0 on the axis-d Nyquist plane, 0 at k = 0)
    particles  x = q + psi / dx  (q = cell centres, grid units, wrapped to [0, N)),   w = a u = vel_factor * psi
    gas        rho = f_b (1 + delta),   m = rho w(q),   eps = rho (e~_0 + |w|^2 / 2)
with vel_factor = a^2 H(a) f(a) (Einstein-de Sitter: H0 sqrt(a)) and e~_0 = a0^2 k_B T0 / ((gamma - 1) mu m_p) (R18, R27).
Pins (tests/test_oracle_pm.py, -m "not gpu"): div psi = -delta in Fourier space, a single Fourier mode against its
analytic displacement, <J v, w> against central finite differences of the map, and the Zel'dovich pancake / linear-growth
tests that start from this state.
"""
from __future__ import annotations

import numpy as np


def _psi_operator(N, L):
    """Fourier multipliers i k~_d / k^2 (d = x, y, z) on numpy's rfftn layout [z][y][kx]."""
    kf = 2.0 * np.pi / L
    n1 = np.fft.fftfreq(N, d=1.0 / N)
    nz = n1[:, None, None]; ny = n1[None, :, None]; nx = np.arange(N // 2 + 1)[None, None, :]
    k2 = kf * kf * (nx * nx + ny * ny + nz * nz) + 0.0 * (nx + ny + nz)
    inv = np.zeros_like(k2)
    inv[k2 > 0] = 1.0 / k2[k2 > 0]
    comps = []
    for n in (nx, ny, nz):
        nt = np.where(np.abs(n) == N // 2, 0.0, n) + 0.0 * k2
        comps.append(1j * kf * nt * inv)
    return comps


def displacement(delta: np.ndarray, L: float) -> np.ndarray:
    """Zel'dovich displacement psi (3,N,N,N), same length unit as L, with div psi = -delta."""
    N = delta.shape[0]
    dh = np.fft.rfftn(delta)
    return np.stack([np.fft.irfftn(op * dh, s=(N, N, N), axes=(0, 1, 2)) for op in _psi_operator(N, L)])


def displacement_T(psib: np.ndarray, L: float) -> np.ndarray:
    """Transpose of `displacement` (each multiplier is odd and imaginary, hence antisymmetric)."""
    N = psib.shape[1]
    acc = 0.0
    for d, op in enumerate(_psi_operator(N, L)):
        acc = acc - np.fft.irfftn(op * np.fft.rfftn(psib[d]), s=(N, N, N), axes=(0, 1, 2))
    return acc


def zeldovich_state(delta: np.ndarray, N: int, L: float, f_b: float, vel_factor: float, e_tilde0: float):
    """delta (N^3, fp64) -> gas (5,N,N,N), part (6,N^3), fp64; one particle per cell."""
    dx = L / N
    psi = displacement(delta, L)
    q = np.arange(N) + 0.5
    Q = np.stack(np.meshgrid(q, q, q, indexing="ij")[::-1])     # (x, y, z) components on the [z][y][x] grid
    pos = (Q + psi / dx).reshape(3, -1)
    pos = pos - N * np.floor(pos / N)
    v = vel_factor * psi
    part = np.concatenate([pos, v.reshape(3, -1)], axis=0)
    rho = f_b * (1.0 + delta)
    gas = np.empty((5, N, N, N))
    gas[0] = rho
    gas[1:4] = rho[None] * v
    gas[4] = rho * (e_tilde0 + 0.5 * np.sum(v * v, axis=0))
    return gas, part


def zeldovich_state_vjp(delta: np.ndarray, N: int, L: float, f_b: float, vel_factor: float, e_tilde0: float,
                        cot_gas: np.ndarray, cot_part: np.ndarray) -> np.ndarray:
    """Transpose of d(zeldovich_state)/d(delta) applied to (cot_gas, cot_part) -> cotangent of delta (the wrap of
    the positions has derivative 1, reading R26)."""
    dx = L / N
    psi = displacement(delta, L)
    rho = f_b * (1.0 + delta)
    v = vel_factor * psi
    cg = np.asarray(cot_gas, dtype=np.float64).reshape(5, N, N, N)
    cp = np.asarray(cot_part, dtype=np.float64).reshape(6, N, N, N)
    rho_b = cg[0] + np.sum(cg[1:4] * v, axis=0) + cg[4] * (e_tilde0 + 0.5 * np.sum(v * v, axis=0))
    v_b = cg[1:4] * rho[None] + cg[4][None] * rho[None] * v
    psi_b = vel_factor * v_b + cp[0:3] / dx + vel_factor * cp[3:6]
    return f_b * rho_b + displacement_T(psi_b, L)


# ---- the two factors of the map (readings R18, R19, R27).  The oracle's own statement of them: the CUDA library has its
# own (dh_ic_factors); the two are compared in tests/, never shared.
K_BOLTZMANN = 1.380649e-23          # J / K (SI definition)
M_PROTON = 1.67262192369e-27        # kg (CODATA 2018)
MU_IONISED = 0.59                   # mean molecular weight of fully ionised primordial gas (R18)


def thermal_energy_tilde(a0: float, T0: float, gamma: float, mu: float = MU_IONISED) -> float:
    """e~_0 = a0^2 e(T0),  e(T) = k_B T / ((gamma - 1) mu m_p)  in (km/s)^2  (R18, R27)."""
    e_si = K_BOLTZMANN * T0 / ((gamma - 1.0) * mu * M_PROTON)      # m^2 / s^2
    return a0 * a0 * e_si * 1e-6


def velocity_factor_eds(H0: float, a: float) -> float:
    """w = a^2 H(a) f(a) psi.  Einstein-de Sitter: H = H0 a^-3/2, D = a so f = 1:  a^2 H f = H0 sqrt(a)  (R19)."""
    return H0 * np.sqrt(a)


def ic_factors(cfg):
    """(vel_factor, e_tilde0) of a workloads.Config (EdS only, like the configs of BASELINE.json)."""
    assert cfg.Omega_L == 0.0 and abs(cfg.Omega_m - 1.0) < 1e-15, "the oracle states the EdS factor only"
    return velocity_factor_eds(cfg.H0, cfg.a0), thermal_energy_tilde(cfg.a0, cfg.T0, cfg.gamma)


# ---- the same for a workloads.Config (tests and the CPU-baseline legs); W supplies the seeded field only
def state_of(delta, cfg, W=None):
    vf, e0 = ic_factors(cfg)
    return zeldovich_state(delta, cfg.N, cfg.box, cfg.f_b, vf, e0)


def state_vjp_of(delta, cfg, W, cot_gas, cot_part):
    vf, e0 = ic_factors(cfg)
    return zeldovich_state_vjp(delta, cfg.N, cfg.box, cfg.f_b, vf, e0, cot_gas, cot_part)


def coupled_ic(W, cfg, seed=None):
    """Seeded IC of a coupled config: (delta f64, gas f32, part f32).  The fp32 arrays are THE inputs both the step
    oracle (promoted to fp64) and the CUDA path receive in the step / run parity tests (reading R24)."""
    assert cfg.n_side == cfg.N, "one particle per cell"
    delta = W.gaussian_field(cfg.N, cfg.box, cfg.seed if seed is None else seed, cfg.rms_delta)
    gas, part = state_of(delta, cfg, W)
    return delta, gas.astype(np.float32), part.astype(np.float32)


# ------------------------------------------------------------------ output end: the data term of Eq. 27 ------
def data_term(gas, data, noise_var=None, scale=1.0, weight=0.5, observable=0):
    """PAPER.md:341, Eq. 27, first term:  L = weight sum_i (scale O_i - d_i)^2 / N_i  (Eq. 27: weight = 1/2) and
    dL/d(gas) (5,N,N,N), fp64.  observable 0: O = rho (reading R21, the configs' loss); 1: O = eps - |m|^2/(2 rho), the
    internal energy density the mock observable delta_b T is proportional to.
    Pins (tests/test_oracle_pm.py): closed form on constant fields, central finite differences of L."""
    g = np.asarray(gas, dtype=np.float64)
    d = np.asarray(data, dtype=np.float64)
    iv = 1.0 if noise_var is None else 1.0 / np.asarray(noise_var, dtype=np.float64)
    rho, m, eps = g[0], g[1:4], g[4]
    m2 = np.sum(m * m, axis=0)
    obs = rho if observable == 0 else eps - 0.5 * m2 / rho
    r = scale * obs - d
    L = weight * np.sum(r * r * iv)
    ob = 2.0 * weight * scale * r * iv
    cot = np.zeros_like(g)
    if observable == 0:
        cot[0] = ob
    else:
        cot[0] = ob * 0.5 * m2 / rho ** 2
        cot[1:4] = -ob[None] * m / rho[None]
        cot[4] = ob
    return L, cot


# ------------------------------------------------------------------ output end: binned power spectrum ------
def _ps_bins(N):
    n1 = np.fft.fftfreq(N, d=1.0 / N)
    nz = n1[:, None, None]; ny = n1[None, :, None]; nx = n1[None, None, :]
    return np.rint(np.sqrt(nx * nx + ny * ny + nz * nz)).astype(np.int64)      # full spectrum, [z][y][x]


def power_spectrum(field, L):
    """PAPER.md:310 ("power spectra of the baryon density"): with F = FFT3(field) over the FULL spectrum and bins
    b = round(|n|), b = 1 .. N/2:  P_b = (L^3 / N^6) sum_{k in b} |F_k|^2 / count_b.  Returns (P, count), index b - 1.
    Pins (tests/test_oracle_pm.py): a single cosine puts (amplitude^2 L^3 / 4) * 2 / count_b into exactly its own bin;
    sum_b count_b P_b + the dropped modes = Parseval; central finite differences of the transpose."""
    f = np.asarray(field, dtype=np.float64)
    N = f.shape[0]
    F2 = np.abs(np.fft.fftn(f)) ** 2
    b = _ps_bins(N).ravel()
    nb = N // 2
    s = np.bincount(b, weights=F2.ravel(), minlength=nb + 1)[1:nb + 1]
    cnt = np.bincount(b, minlength=nb + 1)[1:nb + 1].astype(np.float64)
    return (L ** 3 / float(N) ** 6) * s / cnt, cnt


def power_spectrum_vjp(field, L, power_bar):
    """sum_b power_bar_b dP_b/dfield:  d/df(x) sum_k g_k |F_k|^2 = 2 N^3 IFFT3(g F)(x),  g_k = (L^3/N^6) power_bar_b / count_b."""
    f = np.asarray(field, dtype=np.float64)
    N = f.shape[0]
    nb = N // 2
    b = _ps_bins(N)
    cnt = np.bincount(b.ravel(), minlength=nb + 1).astype(np.float64)
    g = np.zeros(b.max() + 1)
    g[1:nb + 1] = (L ** 3 / float(N) ** 6) * np.asarray(power_bar, dtype=np.float64) / cnt[1:nb + 1]
    return 2.0 * N ** 3 * np.real(np.fft.ifftn(g[b] * np.fft.fftn(f)))
