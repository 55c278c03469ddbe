"""Pins of the oracle's particle-mesh pieces, step factors and cosmological limits: CPU only."""
import numpy as np
import pytest


# ------------------------------------------------------------------------- FFT / Poisson
def test_own_fft_matches_numpy(O):
    rng = np.random.default_rng(0)
    a = rng.standard_normal((16, 16, 16)) + 1j * rng.standard_normal((16, 16, 16))
    f = O.fft3(a, -1)
    assert np.max(np.abs(f - np.fft.fftn(a))) < 1e-11
    b = O.fft3(a, +1)
    assert np.max(np.abs(b - np.fft.ifftn(a) * a.size)) < 1e-11


@pytest.mark.parametrize("mode", [(1, 0, 0), (0, 2, 0), (0, 0, 3), (1, 2, 3), (-2, 1, 5), (7, -7, 7)])
def test_poisson_single_mode_analytic(O, mode):
    """delta = cos(k0.x + 0.3), lap phi' = A delta => phi' = -A cos/k0^2, g' = -grad phi' = -A k0 sin(k0.x + 0.3)/k0^2
    (the force points towards the density maximum)."""
    N, L, A = 16, 20.0, 1.5 * 100.0 ** 2
    c = (np.arange(N) + 0.5) * L / N
    z, y, x = np.meshgrid(c, c, c, indexing="ij")
    k0 = 2 * np.pi / L * np.array(mode, dtype=float)
    ph = k0[0] * x + k0[1] * y + k0[2] * z + 0.3
    g = O.poisson(N, L, A, np.cos(ph))
    k2 = np.sum(k0 * k0)
    for d in range(3):
        expect = -A * k0[d] / k2 * np.sin(ph)
        assert np.max(np.abs(g[d] - expect)) < 1e-9 * A / np.sqrt(k2)
        assert abs(g[d].mean()) < 1e-9


def test_poisson_nyquist_and_zero_mode(O):
    N, L, A = 8, 8.0, 2.0
    g = O.poisson(N, L, A, np.full((N, N, N), 3.7))          # pure k = 0
    assert np.all(g == 0.0)
    x = np.arange(N)
    d = np.broadcast_to(np.cos(np.pi * x)[None, None, :], (N, N, N)).copy()   # x-Nyquist: odd factor zeroed
    g = O.poisson(N, L, A, d)
    assert np.max(np.abs(g)) < 1e-13


def test_poisson_operator_is_antisymmetric_and_vjp_is_its_transpose(O):
    rng = np.random.default_rng(1)
    N, L, A = 8, 5.0, 3.0
    d = rng.standard_normal((N, N, N)); gb = rng.standard_normal((3, N, N, N))
    g = O.poisson(N, L, A, d)
    db = O.poisson_vjp(N, L, A, gb)
    assert abs(np.sum(g * gb) - np.sum(d * db)) < 1e-11 * np.abs(g * gb).sum()
    # G_d^T = -G_d
    for k in range(3):
        e = np.zeros((3, N, N, N)); e[k] = gb[k]
        assert np.max(np.abs(O.poisson_vjp(N, L, A, e) + O.poisson(N, L, A, gb[k])[k])) < 1e-12


# ------------------------------------------------------------------------------------ CIC
def _rand_pos(rng, n, N):
    return rng.uniform(0, N, size=(3, n))


def test_cic_mass_conservation_and_single_cell(O):
    rng = np.random.default_rng(2)
    N = 8
    pos = _rand_pos(rng, 500, N)
    mesh = O.deposit(N, pos, 0.37)
    assert abs(mesh.sum() - 0.37 * 500) < 1e-11
    assert mesh.min() >= 0.0
    # a particle at a cell centre hits exactly one cell (R13: mesh values at i + 1/2)
    p = np.array([[2.5], [0.5], [7.5]])
    m = O.deposit(N, p, 1.0)
    assert m[7, 0, 2] == 1.0 and np.count_nonzero(m) == 1
    # a particle on a cell corner hits 8 cells equally, with periodic wrap
    p = np.array([[0.0], [0.0], [0.0]])
    m = O.deposit(N, p, 8.0)
    assert np.count_nonzero(m) == 8 and np.all(m[m > 0] == 1.0)
    assert m[0, 0, 0] == 1 and m[N - 1, N - 1, N - 1] == 1 and m[0, N - 1, 0] == 1


def test_cic_brute_force_tiny(O):
    """Brute force over all cells with the tent function W(r) = max(0, 1 - |r|) per axis (periodic)."""
    rng = np.random.default_rng(3)
    N = 4
    pos = _rand_pos(rng, 7, N)
    m = O.deposit(N, pos, 1.0)
    centres = np.arange(N) + 0.5
    ref = np.zeros((N, N, N))
    for p in range(pos.shape[1]):
        def tent(xp):
            r = np.abs(centres - xp)
            r = np.minimum(r, N - r)
            return np.maximum(0.0, 1.0 - r)
        ref += tent(pos[2, p])[:, None, None] * tent(pos[1, p])[None, :, None] * tent(pos[0, p])[None, None, :]
    assert np.max(np.abs(m - ref)) < 1e-14


def test_lattice_gives_uniform_density_and_zero_force(O):
    N = 8
    q = np.arange(N) + 0.5
    Q = np.stack(np.meshgrid(q, q, q, indexing="ij")[::-1]).reshape(3, -1)
    m = O.deposit(N, Q, 1.0)
    assert np.all(m == 1.0)
    g = O.poisson(N, 10.0, 1.5e4, m - 1.0)
    assert np.all(g == 0.0)


def test_gather_reproduces_affine_field(O):
    rng = np.random.default_rng(4)
    N = 8
    c = np.arange(N) + 0.5
    z, y, x = np.meshgrid(c, c, c, indexing="ij")
    mesh = 1.0 + 0.3 * x - 0.2 * y + 0.7 * z
    pos = rng.uniform(1.0, N - 1.0, size=(3, 200))            # away from the periodic wrap
    got = O.gather(N, pos, mesh)
    assert np.max(np.abs(got - (1.0 + 0.3 * pos[0] - 0.2 * pos[1] + 0.7 * pos[2]))) < 1e-13


def test_deposit_gather_adjoint_pair(O):
    rng = np.random.default_rng(5)
    N = 8
    pos = _rand_pos(rng, 300, N)
    f = rng.standard_normal((N, N, N))
    lhs = np.sum(O.gather(N, pos, f))                          # <gather(f), 1>
    rhs = np.sum(f * O.deposit(N, pos, 1.0))                   # <f, deposit(1)>
    assert abs(lhs - rhs) < 1e-11


def test_no_net_self_force(O):
    """Same weights for deposit and gather + antisymmetric Green's operator => sum_p m_p g'_p = 0."""
    rng = np.random.default_rng(6)
    N, L, A = 8, 10.0, 1.5e4
    pos = _rand_pos(rng, 100, N)
    delta = O.deposit(N, pos, 1.0)
    g = O.poisson(N, L, A, delta - delta.mean())
    for d in range(3):
        gp = O.gather(N, pos, g[d])
        assert abs(gp.sum()) < 1e-9 * np.abs(gp).sum()


def test_cell_index_bit_exact_cases(O):
    x = np.array([0.0, 0.25, 0.49999997, 0.5, 0.50000006, 1.4999999, 1.5, 7.5, 7.9999995, 31.5, 31.999998],
                 dtype=np.float32)
    i0, i1 = O.cell_index(x, 32)
    assert list(i0) == [31, 31, 31, 0, 0, 0, 1, 7, 7, 31, 31]
    assert list(i1) == [0, 0, 0, 1, 1, 1, 2, 8, 8, 0, 0]


# ------------------------------------------------------------------------- step factors
def test_eds_step_factors_closed_form(O, W):
    """R15: midpoint factors vs the exact EdS integrals; ratio = sinh(3r/4) / (3 sinh(r/4))."""
    P = O.make_params(8, 10.0, 5.0 / 3.0)
    H0 = 100.0
    for r in (0.01, 0.05, 0.1151):
        a0 = 0.02
        a1 = a0 * np.exp(r)
        a_s, dt_s = O.schedule_lna(P, a0, a1, 1)
        dt = dt_s[0]
        assert abs(dt - 2.0 / (3 * H0) * (a1 ** 1.5 - a0 ** 1.5)) < 1e-15
        sc = O.step_scalars(P, a0, a1, dt, dt)
        drift_exact = (2.0 / H0) * (a0 ** -0.5 - a1 ** -0.5)       # int dt / a^2
        kick_exact = (2.0 / H0) * (np.sqrt(a1) - np.sqrt(a0))      # int dt / a
        ratio = np.sinh(0.75 * r) / (3.0 * np.sinh(0.25 * r))
        assert abs(sc["dtau"] / drift_exact - ratio) < 1e-12
        assert abs(sc["kappa"] / kick_exact - ratio) < 1e-12
        assert abs(ratio - (1 + r * r / 12)) < r ** 4
        assert abs(sc["K"] - dt / a0) < 1e-15                       # (dt_prev + dt)/(2 a_i) with dt_prev = dt
        assert sc["A"] == 1.5 * H0 ** 2
    # first step: opening half kick
    assert abs(O.step_scalars(P, 0.02, 0.03, 0.4, 0.0)["K"] - 0.4 / (2 * 0.02)) < 1e-15
    # static mode
    Ps = O.make_params(8, 1.0, 1.4, static_mode=1)
    sc = O.step_scalars(Ps, 1.0, 1.0, 0.3, 0.1)
    assert sc["dtau"] == 0.3 and sc["kappa"] == 0.3 and abs(sc["K"] - 0.2) < 1e-16


def test_schedule_matches_workloads_and_quadrature(O, W):
    cfg = W.CONFIGS[0]
    P = O.make_params(cfg.N, cfg.box, cfg.gamma)
    a, dt = O.schedule_lna(P, cfg.a0, cfg.a1, cfg.n_steps)
    a2, dt2 = W.eds_schedule(cfg)
    assert np.max(np.abs(a - a2)) < 1e-15 and np.max(np.abs(dt / dt2 - 1)) < 1e-13
    # the quadrature branch reduces to the closed form when Omega_m -> 1
    Pq = O.make_params(cfg.N, cfg.box, cfg.gamma, Omega_m=1.0 - 1e-12, Omega_L=1e-12)
    _, dtq = O.schedule_lna(Pq, cfg.a0, cfg.a1, cfg.n_steps)
    assert np.max(np.abs(dtq / dt - 1)) < 1e-9


# ---------------------------------------------------------------------- dynamics pins
def _pancake(O, N, n, a0=0.05, a1=0.4):
    """1-D sinusoidal perturbation, DM only, crossing at a_c = 1.  Returns (x_final - x_exact in grid units, amplitude)."""
    L, H0 = float(N), 100.0
    dx = L / N
    q = np.arange(N) + 0.5
    Q = np.stack(np.meshgrid(q, q, q, indexing="ij")[::-1]).reshape(3, -1)
    k = 2 * np.pi / N

    def exact(a):
        psi = -np.sin(k * Q[0]) / k                              # displacement at a_c = 1, grid units
        x = Q.copy(); x[0] = Q[0] + a * psi
        w = np.zeros_like(Q); w[0] = H0 * np.sqrt(a) * a * psi * dx
        return x, w
    P = O.make_params(N, L, 5.0 / 3.0, hydro_on=0, gas_sources_gravity=0, Omega_b=0.0)
    a_s, dt_s = O.schedule_lna(P, a0, a1, n)
    x0, w0 = exact(a0)
    # staggered leapfrog (R15): the opening half kick K = dt/(2 a_0) takes w(a_0) to the first mid-time, so the
    # run starts from the synchronised exact state
    gas = np.zeros((5, N, N, N)); gas[0] = 1e-30; gas[4] = 1e-30
    _, part, _, _ = O.run(P, gas, np.concatenate([x0, w0]), a0, a_s[1:], dt_s)
    xe, _ = exact(a1)
    assert np.max(np.abs(part[1] - xe[1])) < 1e-12 and np.max(np.abs(part[2] - xe[2])) < 1e-12
    d = part[0] - xe[0]
    d -= N * np.round(d / N)
    return d, a1 / k, part[0], xe[0] - Q[0]


def test_zeldovich_pancake_before_shell_crossing(O):
    """Zel'dovich is exact in 1-D before shell crossing: x(q,a) = q + (a/a_c) psi_c(q), w = H0 sqrt(a) (a/a_c) psi_c.
    The leapfrog is second order in time (Richardson); in space the agreement is limited to O(dx) by the kink of the
    CIC kernel at zero lag for a lattice that starts on cell centres (R13), so the error halves with N."""
    d8, amp, x8, psi = _pancake(O, 32, 8)
    d16, _, x16, _ = _pancake(O, 32, 16)
    d32, _, x32, _ = _pancake(O, 32, 32)
    r = np.max(np.abs(x8 - x16)) / np.max(np.abs(x16 - x32))
    assert 3.3 < r < 4.7, r                                       # second order in time
    e32 = np.max(np.abs(d32)) / amp
    e16 = np.max(np.abs(_pancake(O, 16, 32)[0])) / (amp / 2)
    assert e32 < 0.07 and 1.6 < e16 / e32 < 2.4, (e16, e32)
    # amplitude of the final displacement against the exact one: CIC window sinc^4(pi/N) ~ 0.99 lowers the growth a bit
    disp = psi + d32
    coeff = np.sum(disp * psi) / np.sum(psi * psi)
    assert 0.975 < coeff < 1.0, coeff


def test_linear_growth_of_3d_field_in_eds(O, W, IC):
    """Small 3-D perturbation, DM only: the fundamental modes grow ~ a (growing mode, EdS).  Only |n| <= 1 modes are
    compared: the CIC window sinc^4 lowers the growth of shorter waves (at N = 32 the fundamental loses < 1 %)."""
    cfg = W.scaled_config(0, 32, n_steps=24, a1=0.08, rms_delta=1e-3, Omega_b=0.0)
    delta = W.gaussian_field(cfg.N, cfg.box, 7, cfg.rms_delta)
    gas, part = IC.state_of(delta, cfg, W)
    P = O.make_params(cfg.N, cfg.box, cfg.gamma, hydro_on=0, gas_sources_gravity=0, Omega_b=0.0)
    a_s, dt_s = O.schedule_lna(P, cfg.a0, cfg.a1, cfg.n_steps)
    _, part1, _, _ = O.run(P, gas, part, cfg.a0, a_s[1:], dt_s)
    d0 = np.fft.fftn(O.deposit(cfg.N, part[:3], 1.0) - 1.0)
    d1 = np.fft.fftn(O.deposit(cfg.N, part1[:3], 1.0) - 1.0)
    n = np.fft.fftfreq(cfg.N, 1.0 / cfg.N)
    low = (np.abs(n)[:, None, None] <= 1) & (np.abs(n)[None, :, None] <= 1) & (np.abs(n)[None, None, :] <= 1)
    low[0, 0, 0] = False
    growth = np.real(np.sum(d1[low] * np.conj(d0[low])) / np.sum(np.abs(d0[low]) ** 2))
    assert abs(growth / (cfg.a1 / cfg.a0) - 1.0) < 0.03, growth
    phase = np.abs(np.angle(d1[low] / d0[low]))
    assert phase.max() < 0.05


def test_uniform_gas_hubble_drag_and_adiabatic_cooling_bitwise(O):
    """Uniform gas at rest w.r.t. a uniform flow: conserved tilde variables stay constant bitwise, i.e.
    U = m/(a rho) ~ 1/a (Hubble drag) and e = e~/a^2 ~ a^-2 (adiabatic gamma = 5/3 expansion)."""
    N = 8
    P = O.make_params(N, 10.0, 5.0 / 3.0, n_part_side=0, gravity_on=0)
    gas = np.zeros((5, N, N, N)); gas[0] = 0.16; gas[1] = 0.16 * 3.0; gas[2] = -0.16; gas[4] = 0.16 * (0.02 + 5.0)
    a_s, dt_s = O.schedule_lna(P, 0.01, 0.1, 10)
    g1, _, cm, _ = O.run(P, gas, np.zeros((6, 0)), 0.01, a_s[1:], dt_s)
    assert np.array_equal(g1, gas)


def test_cold_gas_tracks_dark_matter_in_linear_regime(O, W, IC):
    """Pressureless gas obeys the same linear growth as the DM: on the fundamental modes delta_gas = delta_dm and both
    have grown by a1/a0 (shorter waves differ: CIC window for the DM, numerical diffusion for the gas)."""
    N = 16
    cfg = W.scaled_config(0, N, n_steps=16, a1=0.04, rms_delta=2e-3)
    cfg.T0 = 1.0     # cold: negligible pressure
    cfg.e_floor_cosmo = 2.1e-9
    delta, gas, part = IC.coupled_ic(W, cfg, seed=21)
    P = O.make_params(cfg.N, cfg.box, cfg.gamma, e_floor=cfg.e_floor())
    a_s, dt_s = O.schedule_lna(P, cfg.a0, cfg.a1, cfg.n_steps)
    g1, p1, _, _ = O.run(P, gas, part, cfg.a0, a_s[1:], dt_s)
    d_dm = np.fft.fftn(O.deposit(N, p1[:3], 1.0) - 1.0)
    d_gas = np.fft.fftn(g1[0] / cfg.f_b - 1.0)
    d0 = np.fft.fftn(delta)
    n = np.abs(np.fft.fftfreq(N, 1.0 / N))
    low = (n[:, None, None] <= 1) & (n[None, :, None] <= 1) & (n[None, None, :] <= 1)
    low[0, 0, 0] = False

    def proj(a, b):
        return np.real(np.sum(a[low] * np.conj(b[low])) / np.sum(np.abs(b[low]) ** 2))
    assert abs(proj(d_gas, d_dm) - 1.0) < 0.03
    assert abs(proj(d_dm, d0) / 4.0 - 1.0) < 0.06 and abs(proj(d_gas, d0) / 4.0 - 1.0) < 0.06
    # gas mass is conserved to round-off also with gravity on (the source term does not touch rho)
    assert abs(g1[0].sum() / gas[0].astype(np.float64).sum() - 1.0) < 1e-13


def test_workload_generators(W, IC):
    d = W.gaussian_field(16, 20.0, 1000, 0.02)
    assert abs(np.sqrt(np.mean(d * d)) - 0.02) < 1e-15 and abs(d.mean()) < 1e-15
    assert np.array_equal(d, W.gaussian_field(16, 20.0, 1000, 0.02))            # seeded
    psi = IC.displacement(d, 20.0)
    # div psi = -delta (spectral, away from the zeroed Nyquist planes): check in Fourier space
    dh = np.fft.fftn(d); k = 2 * np.pi / 20.0 * np.fft.fftfreq(16, 1 / 16.0)
    div = 1j * (k[None, None, :] * np.fft.fftn(psi[0]) + k[None, :, None] * np.fft.fftn(psi[1])
                + k[:, None, None] * np.fft.fftn(psi[2]))
    mask = (np.abs(np.fft.fftfreq(16, 1 / 16.0)) < 8)
    m3 = mask[:, None, None] & mask[None, :, None] & mask[None, None, :]
    assert np.max(np.abs((div + dh)[m3])) < 1e-9 * np.abs(dh).max()
    # transpose of the IC map
    cfg = W.scaled_config(0, 8)
    rng = np.random.default_rng(0)
    d = W.gaussian_field(8, cfg.box, 3, 0.05)
    v = rng.standard_normal((8, 8, 8)); h = 1e-6
    gp, pp = IC.state_of(d + h * v, cfg, W); gm, pm = IC.state_of(d - h * v, cfg, W)
    cg = rng.standard_normal(gp.shape); cp = rng.standard_normal(pp.shape)
    lhs = (np.sum(cg * (gp - gm)) + np.sum(cp * (pp - pm))) / (2 * h)
    rhs = np.sum(v * IC.state_vjp_of(d, cfg, W, cg, cp))
    assert abs(lhs - rhs) < 1e-6 * abs(lhs)


@pytest.mark.parametrize("mode", [(1, 0, 0), (0, 2, 0), (2, -1, 3)])
def test_ic_oracle_single_mode_analytic(IC, mode):
    """Pin of oracle/ic.py against the closed form: delta = eps cos(k.x) gives psi = -eps (k / k^2) sin(k.x) (div psi =
    -delta), positions q + psi/dx, w = vf psi, rho = f_b (1 + delta)."""
    N, L, eps, f_b, vf, e0 = 16, 20.0, 0.03, 0.16, 7.0, 1e-3
    c = (np.arange(N) + 0.5) * L / N
    z, y, x = np.meshgrid(c, c, c, indexing="ij")
    k = 2 * np.pi / L * np.array(mode, dtype=float)
    ph = k[0] * x + k[1] * y + k[2] * z
    delta = eps * np.cos(ph)
    gas, part = IC.zeldovich_state(delta, N, L, f_b, vf, e0)
    psi = [-eps * k[d] / np.dot(k, k) * np.sin(ph) for d in range(3)]
    q = [x / (L / N), y / (L / N), z / (L / N)]
    for d in range(3):
        want = (q[d] + psi[d] / (L / N)).ravel()
        diff = part[d] - want
        diff -= N * np.round(diff / N)
        assert np.max(np.abs(diff)) < 1e-12
        assert np.max(np.abs(part[3 + d] - vf * psi[d].ravel())) < 1e-12
        assert np.max(np.abs(gas[1 + d] - f_b * (1 + delta) * vf * psi[d])) < 1e-12
    assert np.max(np.abs(gas[0] - f_b * (1 + delta))) < 1e-15
    v2 = vf * vf * sum(p * p for p in psi)
    assert np.max(np.abs(gas[4] - f_b * (1 + delta) * (e0 + 0.5 * v2))) < 1e-12


@pytest.mark.parametrize("observable", [0, 1])
def test_data_term_oracle_closed_form_and_finite_differences(IC, observable):
    """Pins of oracle/ic.py data_term (Eq. 27): constant fields give weight n (scale O - d)^2 / N in closed
    form; the cotangent equals the central finite difference of L along a random direction."""
    n = 6
    gas = np.zeros((5, n, n, n)); gas[0] = 2.0; gas[1] = 1.0; gas[2] = -2.0; gas[3] = 0.5; gas[4] = 7.0
    O = 2.0 if observable == 0 else 7.0 - 0.5 * (1 + 4 + 0.25) / 2.0
    L, cot = IC.data_term(gas, np.full((n, n, n), 1.5), np.full((n, n, n), 4.0), scale=3.0, weight=0.5, observable=observable)
    assert abs(L - 0.5 * n ** 3 * (3.0 * O - 1.5) ** 2 / 4.0) < 1e-10
    rng = np.random.default_rng(3)
    gas = gas + 0.1 * rng.standard_normal(gas.shape)
    d = rng.standard_normal((n, n, n)); nv = 1.0 + rng.uniform(size=(n, n, n))
    v = rng.standard_normal(gas.shape); h = 1e-6
    Lp, _ = IC.data_term(gas + h * v, d, nv, 1.3, 0.5, observable); Lm, _ = IC.data_term(gas - h * v, d, nv, 1.3, 0.5, observable)
    _, cot = IC.data_term(gas, d, nv, 1.3, 0.5, observable)
    assert abs((Lp - Lm) / (2 * h) - np.sum(cot * v)) < 1e-7 * abs(np.sum(cot * v))


def test_power_spectrum_oracle_single_mode_parseval_and_transpose(IC):
    """Pins of oracle/ic.py power_spectrum: f = A cos(k.x) with |n| = 3 has |F|^2 = (A N^3 / 2)^2 at +-k only, so
    P_3 = 2 (A/2)^2 L^3 / count_3 and every other bin is empty; Parseval over all bins of a random field (the corner
    modes beyond N/2 and the mean are added back); the transpose against central finite differences."""
    N, L, A = 16, 20.0, 0.7
    c = (np.arange(N) + 0.5) / N
    z, y, x = np.meshgrid(c, c, c, indexing="ij")
    f = A * np.cos(2 * np.pi * (2 * x + 2 * y - 1 * z))                         # |n| = 3 exactly
    P, cnt = IC.power_spectrum(f, L)
    assert abs(P[2] - 2 * (A / 2) ** 2 * L ** 3 / cnt[2]) < 1e-12 * P[2]
    assert np.max(np.abs(np.delete(P, 2))) < 1e-20
    assert cnt[0] == 18 and cnt[1] == 62                                         # |n| rounds to 1: 6 + 12 modes; to 2: 62
    rng = np.random.default_rng(0)
    f = rng.standard_normal((N, N, N))
    P, cnt = IC.power_spectrum(f, L)
    F2 = np.abs(np.fft.fftn(f)) ** 2
    b = IC._ps_bins(N)
    rest = F2[(b == 0) | (b > N // 2)].sum()
    assert abs((np.sum(P * cnt) * N ** 6 / L ** 3 + rest) / (N ** 3 * np.sum(f * f)) - 1) < 1e-12
    pb = rng.standard_normal(N // 2); v = rng.standard_normal(f.shape); h = 1e-6
    lhs = np.sum(pb * (IC.power_spectrum(f + h * v, L)[0] - IC.power_spectrum(f - h * v, L)[0])) / (2 * h)
    rhs = np.sum(v * IC.power_spectrum_vjp(f, L, pb))
    assert abs(lhs - rhs) < 1e-7 * abs(lhs)
