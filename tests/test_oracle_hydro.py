"""Pins of the oracle's hydro sweep (SURVEY.md 8(c) "What pins each part"): CPU only."""
import os

import numpy as np
import pytest

import exact_riemann as ER

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _evolve_1d(O, gas, axis, t_end, cfl=0.4, gamma=1.4):
    n = gas.shape[3 - axis]
    dx = 1.0 / n
    t = 0.0
    _, cm = O.sweep(gas, axis, 0.0, 0.0, gamma)
    while t < t_end - 1e-14:
        dt = min(cfl * dx / cm, t_end - t)
        gas, cm_in = O.sweep(gas, axis, dt / dx, dt, gamma)
        _, cm = O.sweep(gas, axis, 0.0, 0.0, gamma)
        t += dt
    return gas


def test_exact_riemann_solver_matches_textbook_star_values():
    vals = {}
    for line in open(os.path.join(GOLD, "sod_star_values.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, v, tol = line.split()
        vals[k] = (float(v), float(tol))
    g = 1.4
    ps, us = ER.star_state(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, g)
    rho, u, p = ER.sample(np.array([0.5 * us, us + 0.5 * (ER.shock_speed_right(0.125, 0.0, 0.1, ps, g) - us)]),
                          1.0, 0.0, 1.0, 0.125, 0.0, 0.1, g)
    got = dict(p_star=ps, u_star=us, rho_star_L=rho[0], rho_star_R=rho[1],
               shock_speed=ER.shock_speed_right(0.125, 0.0, 0.1, ps, g))
    for k, (v, tol) in vals.items():
        assert abs(got[k] - v) <= tol, (k, got[k], v)


def _sod_l1(O, W, nx, t_end=0.1):
    g = 1.4
    gas = W.sod_tube(nx, g)
    out = _evolve_1d(O, gas, 0, t_end, gamma=g)
    x = (np.arange(nx) + 0.5) / nx
    sel = x >= 0.5                              # the standard-orientation Sod problem sits at x = 0.75
    rho_e, u_e, p_e = ER.sample((x[sel] - 0.75) / t_end, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, g)
    rho = out[0, 0, 0, sel]
    u = out[1, 0, 0, sel] / rho
    p = (g - 1.0) * (out[4, 0, 0, sel] - 0.5 * rho * u * u)
    return np.mean(np.abs(rho - rho_e)), np.mean(np.abs(u - u_e)), np.mean(np.abs(p - p_e)), out


def test_sod_tube_converges_to_exact_riemann_solution(O, W):
    e200 = _sod_l1(O, W, 200)
    e400 = _sod_l1(O, W, 400)
    e800 = _sod_l1(O, W, 800)
    # absolute accuracy at 800 cells and ~first-order convergence (discontinuities limit the L1 rate to ~1)
    assert e800[0] < 2.5e-3 and e800[1] < 5e-3 and e800[2] < 2.5e-3, e800[:3]
    for k in range(3):
        r1 = e200[k] / e400[k]
        r2 = e400[k] / e800[k]
        assert 1.5 < r1 < 2.6 and 1.5 < r2 < 2.6, (k, r1, r2)


def test_sod_star_plateau_and_shock_position(O, W):
    nx, t_end, g = 800, 0.1, 1.4
    out = _sod_l1(O, W, nx, t_end)[3]
    x = (np.arange(nx) + 0.5) / nx
    rho = out[0, 0, 0]; u = out[1, 0, 0] / rho; p = (g - 1) * (out[4, 0, 0] - 0.5 * rho * u * u)
    # plateau between contact (0.75 + 0.0927) and shock (0.75 + 0.1752)
    i = np.argmin(np.abs(x - (0.75 + 0.135)))
    assert abs(p[i] - 0.30313) < 2e-3 and abs(u[i] - 0.92745) < 3e-3 and abs(rho[i] - 0.26557) < 2e-3
    # shock position: where rho crosses the mean of pre/post shock density
    right = x > 0.85
    cross = x[right][np.argmin(np.abs(rho[right] - 0.5 * (0.26557 + 0.125)))]
    assert abs(cross - (0.75 + 1.75216 * t_end)) < 2.5 / nx


def test_sod_no_new_extrema(O, W):
    """TVD: density stays within the initial bounds, velocity within [-(u*), u*] up to a small overshoot."""
    out = _sod_l1(O, W, 400)[3]
    rho = out[0, 0, 0]
    assert rho.min() >= 0.125 - 1e-3 and rho.max() <= 1.0 + 1e-3
    u = out[1, 0, 0] / rho
    assert np.abs(u).max() <= 0.92745 * 1.02


def test_mirror_symmetry(O, W):
    """Mirror-image data gives the mirror-image solution to round-off (pins the sign handling of R8)."""
    nx, g = 128, 1.4
    rng = np.random.default_rng(5)
    gas = W.sod_tube(nx, g)
    gas[0] += 0.05 * rng.random(gas[0].shape)
    gas[1] = gas[0] * 0.3 * rng.standard_normal(gas[0].shape)
    gas[2] = gas[0] * 0.2
    gas[4] += 0.5 * (gas[1] ** 2 + gas[2] ** 2) / gas[0]
    grav = 0.1 * rng.standard_normal(gas[0].shape)
    out, _ = O.sweep(gas, 0, 0.2, 0.05, g, g=grav)
    gm = gas[..., ::-1].copy(); gm[1] *= -1.0
    outm, _ = O.sweep(gm, 0, 0.2, 0.05, g, g=-grav[..., ::-1].copy())
    back = outm[..., ::-1].copy(); back[1] *= -1.0
    assert np.max(np.abs(back - out)) < 1e-14


def test_uniform_state_preserved_bitwise(O):
    gas = np.zeros((5, 4, 6, 8))
    gas[0] = 1.3; gas[1] = 0.4; gas[2] = -0.7; gas[3] = 0.2; gas[4] = 2.9
    for d in range(3):
        out, cm = O.sweep(gas, d, 0.37, 0.0, 5.0 / 3.0)
        assert np.array_equal(out, gas)
        out, _ = O.sweep(gas, d, 0.37, 0.11, 5.0 / 3.0, g=np.zeros(gas.shape[1:]))
        assert np.array_equal(out, gas)


def test_conservation_to_roundoff(O, W):
    gas, _ = W.smooth_random_state(12, 3, amp=0.3)
    tot0 = gas.reshape(5, -1).sum(axis=1)
    scale = np.abs(gas).reshape(5, -1).sum(axis=1)
    for step in range(6):
        for d in O.strang_order(step):
            gas, _ = O.sweep(gas, d, 0.25, 0.25 * 0.1, 5.0 / 3.0)
    tot = gas.reshape(5, -1).sum(axis=1)
    assert np.all(np.abs(tot - tot0) <= 1e-13 * scale), (tot - tot0) / scale


def test_floor_does_not_touch_conserved_state(O):
    """R17: with the floor active everywhere the update is still conservative."""
    rng = np.random.default_rng(0)
    gas = np.zeros((5, 1, 1, 64))
    gas[0] = 1 + 0.1 * rng.random(64); gas[1] = gas[0] * (1.0 + 0.1 * rng.random(64))
    gas[4] = 0.5 * gas[1] ** 2 / gas[0] * (1 + 1e-9)        # e ~ 0  => floored
    out, _ = O.sweep(gas, 0, 0.1, 0.0, 5.0 / 3.0, e_floor=1e-3)
    assert np.all(np.abs(out.reshape(5, -1).sum(1) - gas.reshape(5, -1).sum(1)) < 1e-12)


def test_axis_symmetry(O, W):
    gas, _ = W.smooth_random_state(8, 11, amp=0.3)
    grav = np.random.default_rng(1).standard_normal((8, 8, 8))
    ox, cx = O.sweep(gas, 0, 0.3, 0.02, 1.4, g=grav)
    # y-sweep of the x<->y transposed state
    gt = gas.transpose(0, 1, 3, 2).copy()
    gt[[1, 2]] = gt[[2, 1]]
    oy, cy = O.sweep(gt, 1, 0.3, 0.02, 1.4, g=grav.transpose(0, 2, 1).copy())
    back = oy.transpose(0, 1, 3, 2).copy(); back[[1, 2]] = back[[2, 1]]
    # transverse components are carried in cyclic order (d+1, d+2), so |m|^2 is summed in a different order:
    # equal to round-off, not bitwise
    assert np.max(np.abs(back - ox)) < 5e-15 and abs(cx - cy) < 1e-15
    gt = gas.transpose(0, 3, 2, 1).copy()
    gt[[1, 3]] = gt[[3, 1]]
    oz, cz = O.sweep(gt, 2, 0.3, 0.02, 1.4, g=grav.transpose(2, 1, 0).copy())
    back = oz.transpose(0, 3, 2, 1).copy(); back[[1, 3]] = back[[3, 1]]
    assert np.max(np.abs(back - ox)) < 5e-15 and abs(cx - cz) < 1e-15


def test_strang_table_period_six_and_balanced(O):
    orders = [O.strang_order(n) for n in range(12)]
    assert orders[:6] == orders[6:]
    assert orders[:6] == [(0, 1, 2), (2, 1, 0), (2, 0, 1), (1, 0, 2), (1, 2, 0), (0, 2, 1)]
    # "XYZZYX, ZXYYXZ, YZXXZY": consecutive pairs are mirror images
    for k in (0, 2, 4):
        assert orders[k] == orders[k + 1][::-1]
    for o in orders:
        assert sorted(o) == [0, 1, 2]


def test_sound_wave_speed_and_second_order(O):
    """Small-amplitude sound wave moves at c_s; L1 error falls faster than first order (limiter active)."""
    g, amp = 5.0 / 3.0, 1e-6
    cs = np.sqrt(g * 1.0 / 1.0)
    errs = []
    for nx in (32, 64, 128):
        x = (np.arange(nx) + 0.5) / nx
        d = amp * np.sin(2 * np.pi * x)
        rho = 1.0 + d; v = cs * d; p = 1.0 + g * d
        gas = np.zeros((5, 1, 1, nx))
        gas[0, 0, 0] = rho; gas[1, 0, 0] = rho * v; gas[4, 0, 0] = p / (g - 1) + 0.5 * rho * v * v
        t_end, dx = 0.25 / cs, 1.0 / nx                 # quarter period
        nsteps = int(np.ceil(t_end / (0.4 * dx / cs)))
        dt = t_end / nsteps
        for _ in range(nsteps):
            gas, _ = O.sweep(gas, 0, dt / dx, dt, g)
        exact = 1.0 + amp * np.sin(2 * np.pi * (x - 0.25))
        errs.append(np.mean(np.abs(gas[0, 0, 0] - exact)) / amp)
    # L1 error: better than first order (ratio 2) -- the harmonic-mean limiter clips the two smooth extrema to
    # first order, which caps the observed L1 rate of a TVD scheme near 2^1.6 ~ 3 per doubling
    assert errs[2] < 2.5e-3
    assert errs[0] / errs[1] > 2.6 and errs[1] / errs[2] > 2.6, errs


def test_limiter_identities(O):
    rng = np.random.default_rng(2)
    for _ in range(200):
        a, b = rng.standard_normal(2)
        f = O.limiter(a, b)
        assert f == O.limiter(b, a) or abs(f - O.limiter(b, a)) < 1e-15
        if a * b <= 0:
            assert f == 0.0
        else:
            assert abs(f) <= 2 * min(abs(a), abs(b)) + 1e-15
            assert abs(f - 2 * a * b / (a + b)) < 1e-15          # Van Leer harmonic mean as eps -> 0
        assert O.limiter(-a, -b) == -f                           # odd symmetry (R8)
    assert abs(O.limiter(0.7, 0.7) - 0.7) < 1e-15                # phi(a,a) = a
    assert O.limiter(0.0, 0.0) == 0.0 and O.limiter(1e-30, 1e-30, 1e-20) < 1e-30
    assert O.limiter(1.0, -1.0) == 0.0                            # extremum: gated, no division by a+b=0


def test_cfl_maximum_is_max_freezing_speed(O):
    g = 1.4
    gas = np.zeros((5, 2, 3, 4))
    gas[0] = 1.0; gas[4] = 1.0 / (g - 1)
    gas[0, 1, 2, 3] = 0.5; gas[2, 1, 2, 3] = 0.5 * (-3.0); gas[4, 1, 2, 3] = 1.0 / (g - 1) + 0.5 * 0.5 * 9.0
    cs_bg = np.sqrt(g)
    cs_hot = np.sqrt(g * 1.0 / 0.5)
    for d, expect in ((0, max(cs_bg, cs_hot)), (1, 3.0 + cs_hot), (2, max(cs_bg, cs_hot))):
        _, cm = O.sweep(gas, d, 0.0, 0.0, g)
        assert abs(cm - expect) < 1e-14


def test_sedov_blast_radius_matches_eq21(O, W):
    """The paper's own closed-form anchor for the hydro solver (Eq. 21): r_sh = 1.15 (E0 t^2 / rho1)^(1/5);
    "shock-front well resolved within roughly 2 pixels, and angular variation of the shock profile of less than 1 pixel"
    (PAPER.md:196).  48^3 cells, gamma = 5/3, energy in the central cell, CFL 0.4 steps up to the time Eq. 21 gives
    r_sh = 8 cells."""
    import parity as PT
    N, g, target = 48, 5.0 / 3.0, 8.0
    gas0 = W.sedov_ic(N, g)
    P = O.make_params(N, float(N), g, n_part_side=0, static_mode=1, gravity_on=0, e_floor=1e-12)
    so = O.State(gas0, np.zeros((6, 0)), 1.0)
    ref = PT.golden("sedov_eq21.txt")
    tf, t = W.sedov_time(target, phi0=ref["phi0"]), 0.0
    while t < tf * (1 - 1e-12):
        cm = max(O.sweep(so.gas, d, 0.0, 0.0, g)[1] for d in range(3))
        dt = min(0.4 / cm, tf - t)
        O.step(P, so, dt, 1.0)
        t += dt
    peak, rmin, rmax = PT.shock_radii(so.gas[0])
    assert abs(peak - target) <= 0.5 * ref["shock_width_cells"], peak
    assert rmax - rmin <= ref["angular_variation_cells"] + 0.5 and abs(0.5 * (rmin + rmax) - target) <= 1.0, (rmin, rmax)
    assert abs(so.gas[0].sum() / gas0[0].astype(np.float64).sum() - 1) < 1e-13      # conservative scheme
    assert abs(so.gas[4].sum() / gas0[4].astype(np.float64).sum() - 1) < 1e-13
    assert 1.5 < so.gas[0].max() < 4.0                           # compression below the strong-shock limit (gamma+1)/(gamma-1)
