"""Pins of the dual-energy oracle (oracle/dual_energy.py; readings R33-R36 of DESIGN.md).  CPU only.

What fixes it other than itself:
  * eta = 0 reduces it to the single-energy sweep, which the C++ oracle states independently and which is pinned to the
    exact Riemann solution (tests/test_oracle_hydro.py) -- every shared term (flux split, stages, limiter, source, CFL);
  * the internal-energy equation alone (eta > 1: the total energy is never trusted) must carry a sound wave at the
    analytic speed sqrt(gamma p / rho): the coefficient and sign of the source -p dv/dx (without it the speed would be
    sqrt(p / rho), with the wrong sign imaginary), and must keep q = rho e_T to second order in smooth flow;
  * uniform states are preserved bit for bit, the five conserved sums to round-off whatever eta;
  * the purpose of the formalism: in single precision a density wave advected at Mach 1000 with uniform
    pressure keeps its temperature to 1e-5 with dual energy and loses it without;
  * the transpose: <J v, w> against central differences of the forward, all three axes, both branches of the selection
    active, with and without gravity, and the three scalar cotangents;
  * the coupled step composed in Python (deposit, Poisson, gather of the C++ oracle + the particle update written out)
    equals the C++ oracle's own coupled step when eta = 0.
"""
import numpy as np
import pytest

from oracle import dual_energy as DE


def _state6(W, N, seed, mach=0.5, amp=0.1):
    gas, _ = W.smooth_random_state(N, seed, amp=amp, n_part_side=2, mach=mach)
    rho = gas[0]
    eT = gas[4] / rho - 0.5 * np.sum(gas[1:4] ** 2, axis=0) / rho ** 2
    rng = np.random.default_rng(seed + 1)
    q = rho * eT * (1.0 + 0.05 * rng.standard_normal(rho.shape))      # an internal energy that has drifted from rho e_T
    return np.concatenate([gas, q[None]], axis=0)


@pytest.mark.parametrize("d", [0, 1, 2])
def test_eta_zero_is_the_single_energy_sweep(O, W, d):
    N = 16
    g6 = _state6(W, N, 11 + d)
    rng = np.random.default_rng(5)
    g = 0.3 * rng.standard_normal((N, N, N))
    out, cm = DE.sweep(g6, d, 0.07, 0.05, 1.4, g, e_floor=1e-9, lim_eps=1e-20, eta=0.0)
    ref, cm_ref = O.sweep(g6[:5], d, 0.07, 0.05, 1.4, g, e_floor=1e-9, lim_eps=1e-20)
    assert np.max(np.abs(out[:5] - ref)) < 1e-13 * np.max(np.abs(ref))
    assert abs(cm - cm_ref) < 1e-13 * cm_ref
    # and with the default eta on a subsonic state (thermal fraction ~ 0.9 everywhere): still the same five fields
    out2, _ = DE.sweep(g6, d, 0.07, 0.05, 1.4, g, e_floor=1e-9, lim_eps=1e-20, eta=1e-3)
    assert np.max(np.abs(out2[:5] - ref)) < 1e-13 * np.max(np.abs(ref))


def test_uniform_state_is_preserved_and_sums_are_conserved(W):
    N = 8
    u = np.zeros((6, N, N, N))
    u[0], u[1], u[2], u[3] = 1.3, 0.4, -0.2, 0.9
    u[4] = 1.3 * (2.0 + 0.5 * (0.4 ** 2 + 0.2 ** 2 + 0.9 ** 2) / 1.3 ** 2)
    u[5] = 1.3 * 1.7                                                  # deliberately not rho e_T
    for eta in (0.0, 1e-3, 2.0):
        for d in range(3):
            out, _ = DE.sweep(u, d, 0.1, 0.0, 5.0 / 3.0, None, eta=eta)
            assert np.array_equal(out[:5], u[:5])
            assert np.max(np.abs(out[5] - (u[5] if eta > 1 else 1.3 * 2.0))) < 1e-15 * 3
    g6 = _state6(W, 12, 3, mach=3.0, amp=0.3)
    for eta in (1e-3, 0.3, 2.0):
        cur = g6
        for d in (0, 1, 2):
            cur, _ = DE.sweep(cur, d, 0.05, 0.0, 5.0 / 3.0, None, eta=eta)
        for k in range(5):
            s0, s1 = g6[k].sum(), cur[k].sum()
            assert abs(s1 - s0) < 1e-12 * np.abs(g6[k]).sum(), (eta, k)


def _sound_wave(n, amp, gamma=5.0 / 3.0, rho0=1.0, p0=0.6, mode=1):
    x = (np.arange(n) + 0.5) / n
    cs = np.sqrt(gamma * p0 / rho0)
    s = amp * np.sin(2 * np.pi * mode * x)
    rho = rho0 * (1 + s)
    v = cs * s
    p = p0 * (1 + gamma * s)
    u = np.zeros((6, 1, 1, n))
    u[0, 0, 0] = rho
    u[1, 0, 0] = rho * v
    u[4, 0, 0] = p / (gamma - 1) + 0.5 * rho * v * v
    u[5, 0, 0] = p / (gamma - 1)
    return u, cs


def _phase_speed(n, eta, t_end=0.25, amp=1e-5, gamma=5.0 / 3.0):
    u, cs = _sound_wave(n, amp, gamma)
    dx = 1.0 / n
    nsteps = int(np.ceil(t_end / (0.4 * dx / (1.01 * cs))))
    dt = t_end / nsteps
    for _ in range(nsteps):
        u, _ = DE.sweep(u, 0, dt / dx, 0.0, gamma, None, eta=eta)
    x = (np.arange(n) + 0.5) / n
    f = u[0, 0, 0] - u[0, 0, 0].mean()
    ph = np.angle(np.sum(f * np.exp(-2j * np.pi * x)))                 # sin(2 pi (x - s)) has phase -pi/2 - 2 pi s
    shift = (-np.pi / 2 - ph) / (2 * np.pi)
    shift = shift - np.round(shift - cs * t_end)
    return shift / t_end, cs, u


def test_internal_energy_equation_alone_carries_sound_at_the_analytic_speed():
    """eta = 2: the pressure always comes from q, so the wave speed is set by the q equation's source term."""
    speed, cs, u = _phase_speed(128, eta=2.0)
    assert abs(speed / cs - 1) < 2e-3, (speed, cs)
    iso = np.sqrt(0.6 / 1.0)                                            # what a missing source term would give
    assert abs(speed / iso - 1) > 0.2
    # the total-energy path gives the same speed
    speed_T, _, _ = _phase_speed(128, eta=0.0)
    assert abs(speed_T / cs - 1) < 2e-3
    # q stays rho e_T of the evolved state to second order in L1 (the two energy equations agree in smooth flow; the
    # TVD limiter clips the extrema, so the maximum norm is first order like everywhere else in the scheme)
    errs = []
    for n in (64, 128):
        _, _, u = _phase_speed(n, eta=2.0, amp=1e-3)
        eT = u[4] - 0.5 * u[1] ** 2 / u[0]
        errs.append(np.mean(np.abs(u[5] - eT)) / 1e-3)
    assert errs[1] < 0.35 * errs[0] and errs[1] < 1e-3, errs


def _advect(n, mach, steps, eta, dtype):
    """A 30 % density wave carried at the given Mach number with uniform pressure and velocity (exact solution: the
    pressure stays uniform); returns p / p0 after `steps` sweeps in the given arithmetic."""
    gamma = 5.0 / 3.0
    x = (np.arange(n) + 0.5) / n
    rho = 1.0 + 0.3 * np.sin(2 * np.pi * x)
    p0 = 1.0
    cs = np.sqrt(gamma * p0 / 0.7)
    v = mach * np.sqrt(gamma * p0)
    u = np.zeros((6, 1, 1, n))
    u[0, 0, 0] = rho; u[1, 0, 0] = rho * v
    u[4, 0, 0] = p0 / (gamma - 1) + 0.5 * rho * v * v
    u[5, 0, 0] = p0 / (gamma - 1)
    lam = 0.4 / (v + cs)
    u = u.astype(dtype)
    for _ in range(steps):
        u, _ = DE.sweep(u, 0, lam, 0.0, gamma, None, e_floor=1e-6, eta=eta, dtype=dtype)
    u = u.astype(np.float64)
    return (gamma - 1) * u[0] * DE.thermal_energy(u, eta) / p0


def test_cold_supersonic_advection_keeps_its_temperature_only_with_dual_energy():
    """"more accurate solutions in low-density, high-velocity regions".  At Mach 1000 the thermal energy is
    2e-6 of the total: in single precision e_T = eps/rho - |m|^2/(2 rho^2) is rounding noise (relative 6e-8 x 5e5 per
    operation) and the temperature is lost within 200 sweeps; the separately advanced q keeps it to 1e-5.  In fp64 both
    are fine, so this is a statement about the arithmetic the CUDA path uses (eta = 0 IS the single-energy scheme, see
    test_eta_zero_is_the_single_energy_sweep)."""
    p_single32 = _advect(64, 1000.0, 200, 0.0, np.float32)
    p_dual32 = _advect(64, 1000.0, 200, 1e-3, np.float32)
    assert np.max(np.abs(p_single32 - 1)) > 0.3, np.max(np.abs(p_single32 - 1))
    assert np.max(np.abs(p_dual32 - 1)) < 1e-3, np.max(np.abs(p_dual32 - 1))
    for eta in (0.0, 1e-3):
        assert np.max(np.abs(_advect(64, 1000.0, 200, eta, np.float64) - 1)) < 1e-3
    # at Mach 0.3 the thermal fraction is far above eta: the two schemes are the same scheme
    a = _advect(64, 0.3, 50, 1e-3, np.float64)
    b = _advect(64, 0.3, 50, 0.0, np.float64)
    assert np.max(np.abs(a - b)) < 1e-12


@pytest.mark.parametrize("d", [0, 1, 2])
@pytest.mark.parametrize("with_g", [True, False])
def test_sweep_vjp_against_central_differences(W, d, with_g):
    N = 10
    gamma, lam, kap = 1.5, 0.06, 0.04 if with_g else 0.0
    # eta at the median thermal fraction of the state splits the cells between the two branches of the selection
    g6 = _state6(W, N, 40 + d, mach=2.5, amp=0.3)
    eT = g6[4] / g6[0] - 0.5 * np.sum(g6[1:4] ** 2, axis=0) / g6[0] ** 2
    eta = float(np.median(eT * g6[0] / g6[4]))
    frac = np.mean(eT > eta * g6[4] / g6[0])
    assert 0.3 < frac < 0.7, frac
    rng = np.random.default_rng(77 + d)
    g = 0.5 * rng.standard_normal((N, N, N)) if with_g else None
    e_floor = float(np.quantile(eT, 0.1))                               # the floor is active in a tenth of the cells
    w = rng.standard_normal(g6.shape)
    cin, gb, sc = DE.sweep_vjp(g6, d, lam, kap, gamma, w, g, e_floor=e_floor, eta=eta)

    def f(g6_, g_, lam_, kap_, gamma_):
        return np.sum(w * DE.sweep(g6_, d, lam_, kap_, gamma_, g_, e_floor=e_floor, eta=eta)[0])
    h = 1e-7
    for trial in range(3):
        v = rng.standard_normal(g6.shape) * np.abs(g6).mean(axis=(1, 2, 3), keepdims=True)
        fd = (f(g6 + h * v, g, lam, kap, gamma) - f(g6 - h * v, g, lam, kap, gamma)) / (2 * h)
        an = np.sum(cin * v)
        assert abs(fd - an) < 2e-6 * max(abs(an), np.linalg.norm(cin) * np.linalg.norm(v) * 1e-2), (trial, fd, an)
    if with_g:
        vg = rng.standard_normal(g.shape)
        fd = (f(g6, g + h * vg, lam, kap, gamma) - f(g6, g - h * vg, lam, kap, gamma)) / (2 * h)
        assert abs(fd - np.sum(gb * vg)) < 1e-6 * abs(fd)
        fd = (f(g6, g, lam, kap + h, gamma) - f(g6, g, lam, kap - h, gamma)) / (2 * h)
        assert abs(fd - sc["kap"]) < 1e-6 * abs(fd)
    fd = (f(g6, g, lam + h, kap, gamma) - f(g6, g, lam - h, kap, gamma)) / (2 * h)
    assert abs(fd - sc["lam"]) < 1e-6 * abs(fd), (fd, sc["lam"])
    fd = (f(g6, g, lam, kap, gamma + h) - f(g6, g, lam, kap, gamma - h)) / (2 * h)
    assert abs(fd - sc["gamma"]) < 1e-6 * abs(fd), (fd, sc["gamma"])


def test_hydro_run_vjp_is_the_gradient_of_the_run(W):
    N = 8
    g6 = _state6(W, N, 90, mach=2.5, amp=0.3)
    lams = [0.05, 0.06, 0.04]
    eta = float(np.median((g6[4] - 0.5 * np.sum(g6[1:4] ** 2, axis=0) / g6[0]) / g6[4]))

    def loss(x, gamma=1.5):
        out, _ = DE.hydro_run(x, gamma, lams, eta=eta)
        return 0.5 * np.sum(out[0] ** 2) + np.sum(out[5])
    out, _ = DE.hydro_run(g6, 1.5, lams, eta=eta)
    cot = np.zeros_like(out); cot[0] = out[0]; cot[5] = 1.0
    grad, dgamma = DE.hydro_run_vjp(g6, 1.5, lams, cot, eta=eta)
    rng = np.random.default_rng(1)
    v = rng.standard_normal(g6.shape) * np.abs(g6).mean(axis=(1, 2, 3), keepdims=True)
    h = 1e-7
    fd = (loss(g6 + h * v) - loss(g6 - h * v)) / (2 * h)
    assert abs(fd - np.sum(grad * v)) < 5e-6 * abs(fd)
    fd = (loss(g6, 1.5 + h) - loss(g6, 1.5 - h)) / (2 * h)
    assert abs(fd - dgamma) < 5e-6 * abs(fd)


def test_coupled_step_with_eta_zero_is_the_cpp_oracle_step(O, W, IC):
    cfg = W.scaled_config(0, 16, n_steps=3, a1=0.02)
    _, gas, part = IC.coupled_ic(W, cfg)
    P = O.make_params(cfg.N, cfg.box, cfg.gamma, e_floor=cfg.e_floor(), lim_eps=cfg.lim_eps)
    a_s, dt_s = O.schedule_lna(P, cfg.a0, cfg.a1, cfg.n_steps)
    g_ref, p_ref, cm_ref, _ = O.run(P, gas, part, cfg.a0, a_s[1:], dt_s)
    rho = gas[0].astype(np.float64)
    q0 = gas[4] - 0.5 * np.sum(gas[1:4].astype(np.float64) ** 2, axis=0) / rho
    g6 = np.concatenate([gas.astype(np.float64), q0[None]], axis=0)
    g6o, po, cm = DE.coupled_run(O, P, g6, part, cfg.a0, a_s[1:], dt_s, eta=0.0)
    assert np.max(np.abs(g6o[:5] - g_ref)) < 1e-11 * np.max(np.abs(g_ref))
    d = po[:3] - p_ref[:3]
    d -= cfg.N * np.round(d / cfg.N)
    assert np.max(np.abs(d)) < 1e-10 and np.max(np.abs(po[3:] - p_ref[3:])) < 1e-11 * np.max(np.abs(p_ref[3:]))
    assert np.max(np.abs(cm - cm_ref)) < 1e-11 * np.max(cm_ref)


def test_coupled_step_vjp_with_the_selection_off_is_the_cpp_oracle_step_vjp(O, W, IC):
    """The transpose of the coupled step composed in numpy (sweep transposes, particle update, Poisson transpose, deposit
    transpose written out) against the C++ oracle's hand-written step VJP -- itself pinned by <Jv,w> = <v,J^T w> and finite
    differences -- with the total energy always trusted (eta = -inf), and against finite differences of its own forward
    with the selection on."""
    cfg = W.scaled_config(0, 16, n_steps=4, a1=0.02)
    _, gas, part = IC.coupled_ic(W, cfg)
    gas = gas.astype(np.float64); part = part.astype(np.float64)
    P = O.make_params(cfg.N, cfg.box, cfg.gamma, e_floor=cfg.e_floor(), lim_eps=cfg.lim_eps)
    a_s, dt_s = O.schedule_lna(P, cfg.a0, cfg.a1, cfg.n_steps)
    k = 2
    g, p, _, _ = O.run(P, gas, part, cfg.a0, a_s[1:k + 1], dt_s[:k])
    rng = np.random.default_rng(4)
    cg = rng.standard_normal(g.shape); cp = rng.standard_normal(p.shape)
    s_in = O.State(g, p, a_s[k], dt_prev=dt_s[k - 1], step=k)
    rg, rp, rdp = O.step_vjp(P, s_in, dt_s[k], a_s[k + 1], cg, cp)
    g6 = np.concatenate([g, np.zeros((1,) + g.shape[1:])], axis=0)
    c6 = np.concatenate([cg, np.zeros((1,) + g.shape[1:])], axis=0)
    got_g, got_p, dgam = DE.coupled_step_vjp(O, P, g6, p, a_s[k], a_s[k + 1], dt_s[k], dt_s[k - 1], k, c6, cp, eta=-1e30)
    assert np.max(np.abs(got_g[:5] - rg)) < 1e-10 * np.max(np.abs(rg))
    assert np.max(np.abs(got_p - rp)) < 1e-10 * np.max(np.abs(rp))
    assert abs(dgam - rdp[0]) < 1e-10 * abs(rdp[0])
    # selection on, q carrying the pressure in half of the cells: <J^T w, v> against central differences
    eT = g[4] / g[0] - 0.5 * np.sum(g[1:4] ** 2, axis=0) / g[0] ** 2
    eta = float(np.median(eT * g[0] / g[4]))
    g6[5] = g[0] * eT * (1.0 + 0.05 * rng.standard_normal(eT.shape))
    c6[5] = rng.standard_normal(eT.shape)
    got_g, got_p, _ = DE.coupled_step_vjp(O, P, g6, p, a_s[k], a_s[k + 1], dt_s[k], dt_s[k - 1], k, c6, cp, eta=eta)

    def f(g6_, p_):
        a, b, _ = DE.coupled_step(O, P, g6_, p_, a_s[k], a_s[k + 1], dt_s[k], dt_s[k - 1], k, eta=eta)
        d = b[:3] - p[:3]
        d -= cfg.N * np.round(d / cfg.N)                      # positions are compared unwrapped
        return np.sum(c6 * a) + np.sum(cp[:3] * d) + np.sum(cp[3:] * b[3:])
    vg = rng.standard_normal(g6.shape) * np.abs(g6).mean(axis=(1, 2, 3), keepdims=True)
    vp = rng.standard_normal(p.shape) * np.array([1e-3] * 3 + [np.abs(p[3:]).mean()] * 3)[:, None]
    an = np.sum(got_g * vg) + np.sum(got_p * vp)
    errs = []
    for h in (1e-6, 1e-7):
        fd = (f(g6 + h * vg, p + h * vp) - f(g6 - h * vg, p - h * vp)) / (2 * h)
        errs.append(abs(fd / an - 1))
    # a handful of the 4096 cells sit within h of a limiter gate or of the selection threshold: 2e-5 at h = 1e-6
    assert min(errs) < 1e-4, (errs, an)
