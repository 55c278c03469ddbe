"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs 0-4).

This module is the ONE thing the CPU oracle's tests and the CUDA path's tests share.  It holds input
recipes only (numpy on the host) -- none of the method's arithmetic (the factors of the Zel'dovich map, a^2 H f and
e~(T0), are computed by each side on its own: dh_ic_factors in the library, oracle/ic.py in the oracle), no CUDA, no
oracle import:
  * a seeded Gaussian random field with P(k) = A k^-2 exp(-(k/k_c)^2), k_c = k_Nyq/2, rescaled to the stated rms
    (stand-in for the paper's Eisenstein-Hu + LPT initial conditions; reading R19 in DESIGN.md);
    -- the field is the input; the Zel'dovich map  delta -> (gas, particles)  is part of the method: the CUDA path does
    it on the device (dh_ic_zeldovich), the oracle in oracle/ic.py;
  * the spherical Sod-type Riemann problem of config 1, a 1-D Sod tube and the paper's Sedov blast;
  * the config table and the (a, dt) schedule in ln a for an EdS cosmology.
Units (reading R18): length h^-1 Mpc, velocity km/s, H0 = 100, density in units of the mean comoving total
matter density, positions in grid units [0, N).
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np


@dataclass
class Config:
    name: str
    N: int
    box: float
    gamma: float
    static_mode: int = 0
    gravity_on: int = 1
    n_part_side: int = -1          # -1: N
    H0: float = 100.0
    Omega_m: float = 1.0
    Omega_b: float = 0.16
    Omega_L: float = 0.0
    a0: float = 0.01
    a1: float = 0.1
    n_steps: int = 20
    rms_delta: float = 0.02
    seed: int = 1000
    target_seed: int = 0
    T0: float = 1.0e4
    checkpoint_stride: int = 0
    lim_eps: float = 1e-20
    e_floor_cosmo: float = 2.1e-5  # option dh_options.e_floor of the cosmological configs, (km/s)^2: about 1e-3 of the
                                   # initial e~ (R17); a stated input, given identically to both sides
    extra: dict = field(default_factory=dict)

    @property
    def n_side(self):
        return self.N if self.n_part_side < 0 else self.n_part_side

    @property
    def f_b(self):
        return self.Omega_b / self.Omega_m

    def e_floor(self):
        return 1e-12 if self.static_mode else self.e_floor_cosmo


CONFIGS = {
    0: Config("cfg0_32_coupled", 32, 20.0, 5.0 / 3.0, a1=0.1, n_steps=20, rms_delta=0.02, seed=1000),
    1: Config("cfg1_128_hydro", 128, 1.0, 1.4, static_mode=1, gravity_on=0, n_part_side=0, n_steps=0),
    2: Config("cfg2_64_coupled", 64, 50.0, 5.0 / 3.0, a1=0.33, n_steps=100, rms_delta=0.01, seed=1002,
              target_seed=2002),
    3: Config("cfg3_256_coupled", 256, 100.0, 5.0 / 3.0, a1=0.33, n_steps=200, rms_delta=0.01, seed=1003,
              target_seed=2003, checkpoint_stride=10),
    4: Config("cfg4_512_coupled", 512, 200.0, 5.0 / 3.0, a1=0.33, n_steps=50, rms_delta=0.01, seed=1004,
              checkpoint_stride=5),
}


def scaled_config(base: int, N: int, **kw) -> Config:
    """A config with the recipe of `base` on an N^3 grid (same cell size), for small parity cases."""
    import copy
    c = copy.deepcopy(CONFIGS[base])
    c.box = c.box * N / c.N
    c.N = N
    c.name = f"{c.name}_at{N}"
    for k, v in kw.items():
        setattr(c, k, v)
    return c


# ------------------------------------------------------------------ schedule -------
def eds_schedule(cfg: Config):
    """a_k = a0 exp(k r) (k = 0..n), dt_k = t(a_{k+1}) - t(a_k) with the EdS closed form t = 2/(3 H0) a^{3/2}."""
    n = cfg.n_steps
    r = np.log(cfg.a1 / cfg.a0) / n
    a = cfg.a0 * np.exp(r * np.arange(n + 1))
    a[-1] = cfg.a1
    t = 2.0 / (3.0 * cfg.H0) * a ** 1.5
    return a, np.diff(t)


# ------------------------------------------------------------ Gaussian field -------
def _kgrid(N, L):
    kf = 2.0 * np.pi / L
    n1 = np.fft.fftfreq(N, d=1.0 / N)             # integers, Nyquist = -N/2
    nz = n1[:, None, None]; ny = n1[None, :, None]; nx = np.arange(N // 2 + 1)[None, None, :]
    return kf, nx, ny, nz


def gaussian_field(N: int, L: float, seed: int, rms: float) -> np.ndarray:
    """Real N^3 field, zero mean, P(k) ~ k^-2 exp(-(k/k_c)^2) with k_c = pi N / (2 L), rms exactly `rms`."""
    rng = np.random.default_rng(seed)
    white = rng.standard_normal((N, N, N))
    kf, nx, ny, nz = _kgrid(N, L)
    k2 = kf * kf * (nx * nx + ny * ny + nz * nz)
    kc = np.pi * N / (2.0 * L)
    with np.errstate(divide="ignore", invalid="ignore"):
        P = np.where(k2 > 0, np.exp(-k2 / kc ** 2) / k2, 0.0)
    d = np.fft.irfftn(np.fft.rfftn(white) * np.sqrt(P), s=(N, N, N), axes=(0, 1, 2))
    d -= d.mean()
    d *= rms / np.sqrt(np.mean(d * d))
    return d


# ------------------------------------------------------------------ hydro ICs ------
def sod_sphere(N: int, gamma: float = 1.4, r0: float = 0.2):
    """Config 1: rho, p = 1, 1 inside r < r0 L about the box centre, else 0.125, 0.1; v = 0.  gas (5,N,N,N) f32."""
    c = (np.arange(N) + 0.5) / N - 0.5
    z, y, x = np.meshgrid(c, c, c, indexing="ij")
    inside = (x * x + y * y + z * z) < r0 * r0
    rho = np.where(inside, 1.0, 0.125)
    p = np.where(inside, 1.0, 0.1)
    gas = np.zeros((5, N, N, N))
    gas[0] = rho
    gas[4] = p / (gamma - 1.0)
    return gas.astype(np.float32)


def sedov_ic(N: int, gamma: float = 5.0 / 3.0, E0: float = 1.0, rho1: float = 1.0, p0: float = 1e-5):
    """Sedov-Taylor blast: uniform density rho1, negligible pressure p0, energy E0 in the central cell
    (cell units: dx = 1, box = N).  gas (5,N,N,N) f32."""
    gas = np.zeros((5, N, N, N))
    gas[0] = rho1
    gas[4] = p0 / (gamma - 1.0)
    c = N // 2
    gas[4, c, c, c] += E0
    return gas.astype(np.float32)


def sedov_time(r_sh: float, E0: float = 1.0, rho1: float = 1.0, phi0: float = 1.15) -> float:
    """Time at which Eq. 21, r_sh = phi0 (E0 t^2 / rho1)^(1/5), reaches r_sh."""
    return float(np.sqrt((r_sh / phi0) ** 5 * rho1 / E0))


def sod_tube(nx: int, gamma: float = 1.4, axis: int = 0, ny: int = 1, nz: int = 1, mirror: bool = False):
    """Two back-to-back Sod tubes on a periodic line: left state (1, 1) on the middle half, right state
    (0.125, 0.1) outside, so each discontinuity is a Sod problem until the waves meet.  f64."""
    shape = [nz, ny, nx]
    n = shape[2 - axis]
    i = (np.arange(n) + 0.5) / n
    hi = (i > 0.25) & (i < 0.75)
    if mirror:
        hi = ~hi
    prof_rho = np.where(hi, 1.0, 0.125)
    prof_p = np.where(hi, 1.0, 0.1)
    sh = [1, 1, 1]; sh[2 - axis] = n
    gas = np.zeros((5, nz, ny, nx))
    gas[0] = prof_rho.reshape(sh)
    gas[4] = prof_p.reshape(sh) / (gamma - 1.0)
    return gas


def smooth_random_state(N: int, seed: int, amp: float = 0.1, n_part_side=None, mach: float = 0.5):
    """Smooth, kink-free random gas + particle state on an N^3 grid for derivative tests (low modes only)."""
    rng = np.random.default_rng(seed)
    c = (np.arange(N) + 0.5) / N
    z, y, x = np.meshgrid(c, c, c, indexing="ij")

    def field():
        f = np.zeros((N, N, N))
        for _ in range(4):
            kx, ky, kz = rng.integers(-2, 3, size=3)
            f += rng.standard_normal() * np.cos(2 * np.pi * (kx * x + ky * y + kz * z) + rng.uniform(0, 2 * np.pi))
        return f / 2.0
    rho = 1.0 + amp * field()
    v = np.stack([mach * (0.3 + amp * field()) for _ in range(3)])   # offset keeps v away from the |v| kink
    e = 1.0 + amp * field()
    gas = np.empty((5, N, N, N))
    gas[0] = rho; gas[1:4] = rho * v; gas[4] = rho * (e + 0.5 * np.sum(v * v, axis=0))
    ns = N if n_part_side is None else n_part_side
    q = (np.arange(ns) + 0.5) * N / ns
    Q = np.stack(np.meshgrid(q, q, q, indexing="ij")[::-1]).reshape(3, -1)
    pos = Q + 0.2 * rng.uniform(-1, 1, size=Q.shape) + 0.013
    pos = pos - N * np.floor(pos / N)
    w = 0.1 * rng.standard_normal(Q.shape)
    return gas, np.concatenate([pos, w], axis=0)
