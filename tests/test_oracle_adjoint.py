"""Pins of the oracle's derivatives (SURVEY.md 8(c) "Adjoint"): the dual-number JVP against central finite
differences, and the hand-written VJP against the JVP by <Jv, w> = <v, J^T w>.  CPU only, 8^3..16^3."""
import numpy as np
import pytest

GAMMA = 5.0 / 3.0


def _rel(a, b):
    return abs(a - b) / max(abs(a), abs(b), 1e-300)


def _fd_check(f0, fp, fm, jv, h, tol, max_kink_frac=0.03):
    """Central difference vs JVP, element by element.  The scheme is only piecewise smooth (limiter gate ab > 0, |v|,
    floor: R26), and any smooth field has extrema where a limiter argument changes sign, so a few elements straddle
    a kink within +-h: those are recognised by their one-sided differences disagreeing and are left out (bounded
    fraction); every other element must match to `tol`."""
    fwd = (fp - f0) / h
    bwd = (f0 - fm) / h
    cen = (fp - fm) / (2 * h)
    scale = np.max(np.abs(jv))
    kink = np.abs(fwd - bwd) > 1e-4 * scale
    assert kink.mean() <= max_kink_frac, kink.mean()
    assert np.max(np.abs(cen - jv)[~kink]) < tol * scale
    # at a kink the JVP (branch taken at the point itself) must lie between / at the one-sided slopes
    lo = np.minimum(fwd, bwd) - 1e-4 * scale
    hi = np.maximum(fwd, bwd) + 1e-4 * scale
    assert np.all((jv[kink] >= lo[kink]) & (jv[kink] <= hi[kink]))


# ------------------------------------------------------------------------------ sweep
@pytest.mark.parametrize("d", [0, 1, 2])
def test_sweep_jvp_matches_central_differences(O, W, d):
    gas, _ = W.smooth_random_state(8, 100 + d, amp=0.2)
    rng = np.random.default_rng(d)
    g = 0.3 * rng.standard_normal((8, 8, 8))
    v = rng.standard_normal(gas.shape); vg = rng.standard_normal(g.shape)
    lam, kap = 0.21, 0.13
    dl, dk, dgm = 0.7, -0.4, 0.3
    _, jv = O.sweep_jvp(gas, d, lam, kap, GAMMA, g=g, dgas=v, dg=vg, dlam=dl, dkap=dk, dgamma=dgm)
    h = 1e-6
    u0, _ = O.sweep(gas, d, lam, kap, GAMMA, g=g)
    up, _ = O.sweep(gas + h * v, d, lam + h * dl, kap + h * dk, GAMMA + h * dgm, g=g + h * vg)
    um, _ = O.sweep(gas - h * v, d, lam - h * dl, kap - h * dk, GAMMA - h * dgm, g=g - h * vg)
    _fd_check(u0, up, um, jv, h, 2e-7)


@pytest.mark.parametrize("d", [0, 1, 2])
@pytest.mark.parametrize("with_g", [True, False])
def test_sweep_vjp_dot_product(O, W, d, with_g):
    gas, _ = W.smooth_random_state(8, 200 + d, amp=0.3)
    rng = np.random.default_rng(10 + d)
    g = 0.3 * rng.standard_normal((8, 8, 8)) if with_g else None
    v = rng.standard_normal(gas.shape)
    vg = rng.standard_normal((8, 8, 8)) if with_g else None
    w = rng.standard_normal(gas.shape)
    lam, kap = 0.21, 0.13
    dl, dk, dgm = 0.7, -0.4, 0.3
    _, jv = O.sweep_jvp(gas, d, lam, kap, GAMMA, g=g, dgas=v, dg=vg, dlam=dl, dkap=dk, dgamma=dgm)
    cin, gb, sc = O.sweep_vjp(gas, d, lam, kap, GAMMA, w, g=g)
    lhs = np.sum(jv * w)
    rhs = np.sum(v * cin) + dl * sc["lam"] + dk * sc["kap"] + dgm * sc["gamma"]
    if with_g:
        rhs += np.sum(vg * gb)
    assert _rel(lhs, rhs) < 1e-12


def test_sweep_vjp_through_shocks_floor_and_extrema(O, W):
    """Dot-product identity also holds with the limiter gates, |v| kinks and the energy floor in play (the JVP and the
    VJP take the same branch: R26)."""
    nx = 64
    gas = W.sod_tube(nx, 1.4)
    for _ in range(20):
        gas, _ = O.sweep(gas, 0, 0.15, 0.0, 1.4)
    gas[4, 0, 0, 10:14] = 0.5 * gas[1, 0, 0, 10:14] ** 2 / gas[0, 0, 0, 10:14] + 1e-9   # floored cells
    rng = np.random.default_rng(3)
    v = rng.standard_normal(gas.shape); w = rng.standard_normal(gas.shape)
    _, jv = O.sweep_jvp(gas, 0, 0.15, 0.02, 1.4, dgas=v, dgamma=1.0, e_floor=1e-3)
    cin, _, sc = O.sweep_vjp(gas, 0, 0.15, 0.02, 1.4, w, e_floor=1e-3)
    assert _rel(np.sum(jv * w), np.sum(v * cin) + sc["gamma"]) < 1e-12


# --------------------------------------------------------------------------- whole step
def _step_setup(O, W, N=8, seed=0, gravity=True, hydro=True, gas_src=True):
    gas, part = W.smooth_random_state(N, seed, amp=0.2)
    part[3:] *= 5.0
    P = O.make_params(N, 10.0, GAMMA, gravity_on=int(gravity), hydro_on=int(hydro),
                      gas_sources_gravity=int(gas_src), e_floor=1e-6)
    sc = dict(dtau=0.02, kappa=0.015, K=0.011, A=40.0)
    return P, gas, part, sc


@pytest.mark.parametrize("step_idx", [0, 3])
def test_step_jvp_matches_central_differences(O, W, step_idx):
    P, gas, part, sc = _step_setup(O, W, seed=step_idx)
    rng = np.random.default_rng(1)
    vg = rng.standard_normal(gas.shape); vp = rng.standard_normal(part.shape)
    ds = np.array([0.3, 0.01, -0.02, 0.015, 5.0])          # (gamma, dtau, kappa, K, A)
    g1, p1, dg, dp = O.step_jvp(P, gas, part, sc, GAMMA, step_idx, dgas=vg, dpart=vp, dscal=ds)
    # the value part of the dual run is the plain step
    g1b, p1b = O.step_explicit(P, gas, part, sc, GAMMA, step_idx)
    assert np.array_equal(g1, g1b) and np.array_equal(p1, p1b)
    h = 1e-6

    def pert(s):
        scp = dict(dtau=sc["dtau"] + s * h * ds[1], kappa=sc["kappa"] + s * h * ds[2], K=sc["K"] + s * h * ds[3],
                   A=sc["A"] + s * h * ds[4])
        return O.step_explicit(P, gas + s * h * vg, part + s * h * vp, scp, GAMMA + s * h * ds[0], step_idx)
    gp, pp = pert(+1); gm, pm = pert(-1)
    for q in (pp, pm):                                    # undo periodic wraps relative to the base point
        q[:3] -= P.N * np.round((q[:3] - p1[:3]) / P.N)
    _fd_check(g1, gp, gm, dg, h, 2e-7, max_kink_frac=0.08)
    _fd_check(p1, pp, pm, dp, h, 2e-7)


@pytest.mark.parametrize("case", ["coupled", "dm_only", "hydro_only", "gas_not_sourcing", "step4"])
def test_step_vjp_dot_product(O, W, case):
    kw = dict(coupled={}, dm_only=dict(hydro=False, gas_src=False), hydro_only=dict(gravity=False),
              gas_not_sourcing=dict(gas_src=False), step4={})[case]
    step_idx = 4 if case == "step4" else 1
    P, gas, part, sc = _step_setup(O, W, seed=7, **kw)
    rng = np.random.default_rng(2)
    vg = rng.standard_normal(gas.shape); vp = rng.standard_normal(part.shape)
    wg = rng.standard_normal(gas.shape); wp = rng.standard_normal(part.shape)
    ds = np.array([0.3, 0.01, -0.02, 0.015, 5.0])
    _, _, dg, dp = O.step_jvp(P, gas, part, sc, GAMMA, step_idx, dgas=vg, dpart=vp, dscal=ds)
    cg, cp, dpar = O.step_vjp_explicit(P, gas, part, sc, GAMMA, step_idx, wg, wp)
    lhs = np.sum(dg * wg) + np.sum(dp * wp)
    rhs = np.sum(vg * cg) + np.sum(vp * cp) + np.sum(ds * dpar)
    assert _rel(lhs, rhs) < 1e-11


def test_run_vjp_equals_chained_step_vjps_and_fd_of_loss(O, W, IC):
    """Reverse sweep over a 6-step run (one full Strang cycle) with the cosmological scalars: the gradient of
    L = sum(rho_final^2)/2 w.r.t. the initial state agrees with central differences along a random direction, and
    dgamma with a central difference in gamma."""
    cfg = W.scaled_config(0, 8, n_steps=6, a1=0.02, rms_delta=0.05)
    delta, gas, part = IC.coupled_ic(W, cfg, seed=5)
    gas = gas.astype(np.float64); part = part.astype(np.float64)

    def params(gamma):
        return O.make_params(cfg.N, cfg.box, gamma, e_floor=cfg.e_floor())
    a_s, dt_s = O.schedule_lna(params(GAMMA), cfg.a0, cfg.a1, cfg.n_steps)

    def loss(g, p, gamma=GAMMA):
        g1, _, _, _ = O.run(params(gamma), g, p, cfg.a0, a_s[1:], dt_s)
        return 0.5 * np.sum(g1[0] ** 2), g1
    L0, g1 = loss(gas, part)
    cot_g = np.zeros_like(gas); cot_g[0] = g1[0]
    cg, cp, dpar = O.run_vjp(params(GAMMA), gas, part, cfg.a0, a_s[1:], dt_s, cot_g, np.zeros_like(part))
    rng = np.random.default_rng(9)
    vg = rng.standard_normal(gas.shape) * np.abs(gas).mean(axis=(1, 2, 3), keepdims=True)
    vp = rng.standard_normal(part.shape) * 0.01
    h = 1e-6
    fd = (loss(gas + h * vg, part + h * vp)[0] - loss(gas - h * vg, part - h * vp)[0]) / (2 * h)
    assert _rel(fd, np.sum(vg * cg) + np.sum(vp * cp)) < 1e-6
    fdg = (loss(gas, part, GAMMA + h)[0] - loss(gas, part, GAMMA - h)[0]) / (2 * h)
    assert _rel(fdg, dpar[0]) < 1e-6
