"""The paper's own gradient check on the CUDA path (PAPER.md:294 Fig. 6, :312: "automatic derivatives ... compared with
those calculated with finite differences"), i.e. evidence for the GPU gradient that does not come from the oracle
(VERDICT r01 missing #5, weak #2), and the per-step late-time checks of ADVICE r01.

Directional derivatives <dL/d delta_init, v> of the whole chain delta_init -> state -> n steps -> loss along smooth
low-k directions v against central differences of the loss the LIBRARY returns (fp64 sum over fp32 fields), at three
step sizes.  The loss is continuous and piecewise smooth (reading R28): finite differences average over the gate flips
the pointwise gradient comparison is sensitive to, so this is the check that says whether the gradient is USEFUL.
"""
import numpy as np
import pytest

import parity as PT

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def api():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2502_02294_b200 import api
    return api


@pytest.fixture(scope="module")
def torch_():
    import torch
    return torch


def _gpu(torch, a):
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float32)).cuda()


class Chain:
    """delta_init -> loss and dL/d delta_init, d/d gamma through the library's device calls."""

    def __init__(self, api, torch, W, cfg, target, stride, gamma=None):
        self.api, self.torch, self.cfg, self.stride = api, torch, cfg, stride
        self.ctx = api.context_for(cfg, **({} if gamma is None else {"gamma": gamma}))
        self.vf, self.e0 = api.ic_factors_for(cfg)            # reading R20: the initial state does not move with gamma
        self.a_s, self.dt_s = api.dh_schedule_lna(cfg.a0, cfg.a1, cfg.n_steps)
        self.target = _gpu(torch, target)

    def loss(self, delta, want_grad=False):
        torch, ctx = self.torch, self.ctx
        dd = _gpu(torch, delta)
        st = ctx.dh_ic_zeldovich(dd, self.cfg.a0, self.vf, self.e0)
        ctx.dh_run(st, self.a_s[1:], self.dt_s, self.stride if want_grad else 0)
        if not want_grad:
            return ctx.dh_data_term(0, st.gas, self.target, None, 1.0, 1.0, None)
        cg = torch.empty_like(st.gas)
        L = ctx.dh_data_term(0, st.gas, self.target, None, 1.0, 1.0, cg)
        ct = self.api.Cot(cg, torch.zeros_like(st.part))
        dp = ctx.dh_run_vjp(ct, ct)
        g = ctx.dh_ic_zeldovich_vjp(dd, self.vf, self.e0, ct)
        return L, g.double().cpu().numpy(), dp

    def close(self):
        self.ctx.close()


def fd_table(chain, delta, dirs, hs):
    """[(direction index, h, central difference of the loss)]"""
    out = []
    for j, v in enumerate(dirs):
        for h in hs:
            lp = chain.loss((delta + h * v).astype(np.float32))
            lm = chain.loss((delta - h * v).astype(np.float32))
            out.append((j, h, (lp - lm) / (2 * h)))
    return out


@pytest.mark.parametrize("which", [0, 2])
def test_gpu_gradient_against_finite_differences_of_the_gpu_loss(api, torch_, O, W, IC, which):
    """Configs 0 and 2 in full (20 steps to a = 0.1 at 32^3; 100 steps to a = 0.33 at 64^3), loss sum (rho - rho_t)^2.
    <grad, v> from dh_run_vjp + dh_ic_zeldovich_vjp against central differences of the GPU loss for h = 0.03 ... 0.001
    (v has the rms of delta_init itself), and d/d gamma against a central difference over two more
    contexts."""
    cfg = W.CONFIGS[which]
    delta = W.gaussian_field(cfg.N, cfg.box, cfg.seed, cfg.rms_delta)
    target = cfg.f_b * (1.0 + W.gaussian_field(cfg.N, cfg.box, cfg.target_seed or cfg.seed + 1000, cfg.rms_delta))
    dirs = [W.gaussian_field(cfg.N, cfg.box, 9000 + j, cfg.rms_delta) for j in range(2)]
    ch = Chain(api, torch_, W, cfg, target, 10)
    L, g, dp = ch.loss(delta.astype(np.float32), want_grad=True)
    assert np.isfinite(L) and np.all(np.isfinite(g))
    # the same chain is deterministic up to the deposit's atomic order: the loss repeats to ~1e-7
    L2 = ch.loss(delta.astype(np.float32))
    assert abs(L2 / L - 1) < 1e-5
    hs = (0.03, 0.01, 0.003, 0.001)
    best = [np.inf] * len(dirs)
    for j, h, fd in fd_table(ch, delta, dirs, hs):
        ad = float(np.sum(g * dirs[j]))
        print(f"config{which} dir {j} h {h}: <grad,v> {ad:.6e}  FD {fd:.6e}  ratio-1 {ad / fd - 1:+.2e}")
        best[j] = min(best[j], abs(ad / fd - 1))
    ch.close()
    # The loss is piecewise smooth and, after many steps, rough at small scales (gates, floor): large h sees curvature,
    # small h sees the roughness and the run-to-run noise of the deposit's atomics, so the difference quotients scatter
    # around the derivative instead of converging monotonically; the closest of the four must agree
    assert max(best) < FD_TOL[which], best
    # d/d gamma
    hg = 1e-3
    lp = Chain(api, torch_, W, cfg, target, 10, gamma=cfg.gamma + hg)
    lm = Chain(api, torch_, W, cfg, target, 10, gamma=cfg.gamma - hg)
    fdg = (lp.loss(delta.astype(np.float32)) - lm.loss(delta.astype(np.float32))) / (2 * hg)
    lp.close(); lm.close()
    print(f"config{which} dgamma {dp.dgamma:.6e}  FD {fdg:.6e}  ratio-1 {dp.dgamma / fdg - 1:+.2e}")
    assert abs(dp.dgamma / fdg - 1) < FD_TOL_GAMMA[which]


# Measured on B200 (reading R28): the closest difference quotient agrees to 7e-4 / 2e-3 (config 0) and
# 1.2e-2 / 3.9e-2 (config 2: 100 steps, overdensities ~7, a quarter of the cells on the energy floor).
FD_TOL = {0: 6e-3, 2: 8e-2}
FD_TOL_GAMMA = {0: 1e-2, 2: 5e-2}


def test_config0_directional_derivative_matches_the_oracle(api, torch_, O, W, IC):
    """<grad, v> of config 0's chain: GPU against the fp64 oracle (run VJP + Zel'dovich transpose) -- the gate flips that
    move individual entries by O(1) (R28) average out in a projection on a smooth direction."""
    cfg = W.CONFIGS[0]
    delta, gas, part = IC.coupled_ic(W, cfg)
    target = cfg.f_b * (1.0 + W.gaussian_field(cfg.N, cfg.box, cfg.seed + 1000, cfg.rms_delta))
    P = PT.oracle_params(O, cfg)
    a_s, dt_s = O.schedule_lna(P, cfg.a0, cfg.a1, cfg.n_steps)
    g_ref, p_ref, _, _ = O.run(P, gas, part, cfg.a0, a_s[1:], dt_s)
    cot = np.zeros_like(g_ref); cot[0] = 2.0 * (g_ref[0] - target)
    rg, rp, rdp = O.run_vjp(P, gas, part, cfg.a0, a_s[1:], dt_s, cot, np.zeros_like(p_ref))
    gd_ref = IC.state_vjp_of(delta, cfg, W, rg, rp)
    ch = Chain(api, torch_, W, cfg, target, 10)
    L, g, dp = ch.loss(delta.astype(np.float32), want_grad=True)
    ch.close()
    L_ref = float(np.sum((g_ref[0] - target) ** 2))
    assert abs(L / L_ref - 1) < 1e-4
    for j in range(3):
        v = W.gaussian_field(cfg.N, cfg.box, 9000 + j, cfg.rms_delta)
        a, b = float(np.sum(g * v)), float(np.sum(gd_ref * v))
        print(f"config0 dir {j}: GPU {a:.6e} oracle {b:.6e} ratio-1 {a / b - 1:+.2e}")
        assert abs(a / b - 1) < 5e-3          # the oracle's own projections move by up to 3.3e-3 under one fp32 rounding
    assert abs(dp.dgamma / rdp[0] - 1) < 1e-3


@pytest.mark.parametrize("k", [50, 90, 99])
def test_config2_late_step_vjp_matches_oracle(api, torch_, O, W, IC, k):
    """chaos-independent late-time checks.  Config 2's GPU state after k steps (a up to 0.33, gas
    overdensities ~7, particles displaced by several cells) goes to BOTH sides; one step and its VJP with a random
    cotangent: fields <= 1e-5; cotangents <= 1e-3 on all but the worst 0.1 % of entries (see the comment at the bounds)."""
    cfg = W.CONFIGS[2]
    delta, gas, part = IC.coupled_ic(W, cfg)
    P = PT.oracle_params(O, cfg)
    a_s, dt_s = O.schedule_lna(P, cfg.a0, cfg.a1, cfg.n_steps)
    ctx = api.context_for(cfg)
    sg = api.State(gas, part, cfg.a0)
    ctx.dh_run(sg, a_s[1:k + 1], dt_s[:k], 0)
    gas_k, part_k = sg.gas.cpu().numpy(), sg.part.cpu().numpy()
    so = O.State(gas_k, part_k, a_s[k], dt_prev=dt_s[k - 1], step=k)
    s_in = so.copy()
    cm_ref, _ = O.step(P, so, dt_s[k], a_s[k + 1])
    cm = torch_.zeros(3, device="cuda")
    s1 = sg.clone()
    ctx.dh_step(s1, dt_s[k], a_s[k + 1], cm)
    e = PT.field_err(s1.gas.cpu().numpy(), so.gas)
    e.update(PT.part_err(s1.part.cpu().numpy(), so.part, cfg.N))
    assert max(e.values()) < 1e-5, e
    assert np.max(np.abs(cm.cpu().numpy() / cm_ref - 1)) < 1e-5
    rng = np.random.default_rng(k)
    cg = rng.standard_normal(gas.shape).astype(np.float32)
    cp = rng.standard_normal(part.shape).astype(np.float32)
    rg, rp, rdp = O.step_vjp(P, s_in, dt_s[k], a_s[k + 1], cg, cp)
    co = api.Cot(cg, cp)
    dp = ctx.dh_step_vjp(sg, dt_s[k], a_s[k + 1], co, co)
    eg, ep = PT.rel_l2(co.gas.cpu().numpy(), rg), PT.rel_l2(co.part.cpu().numpy(), rp)
    et = PT.rel_l2_trimmed(co.gas.cpu().numpy(), rg, frac=1e-3)
    rho = gas_k[0] / cfg.f_b
    print(f"config2 step {k} (max gas overdensity {rho.max():.2f}): fields {max(e.values()):.1e}; VJP gas {eg:.2e} "
          f"(trimmed {et:.2e}), particles {ep:.2e}, dgamma {dp.dgamma:.6g} vs {rdp[0]:.6g}")
    # Late in the run the total-energy formulation has lost the thermal energy of the cold supersonic gas (PAPER.md:85:
    # the case for a dual energy formalism): e~ = eps/rho - |m|^2/(2 rho^2) sits below e_floor in about a quarter of the
    # cells and within its own fp32 evaluation error (6e-8 x kinetic energy >> e_floor) of the floor in a few per cent, so
    # the floor switch (R17, R26) falls on either side there and those entries -- and d gamma, which sums rho e+ terms --
    # move by O(1).  North-star bound on all but the worst 0.1 % of entries; everything finite; particles (no floor) tight.
    assert np.all(np.isfinite(co.gas.cpu().numpy())) and np.all(np.isfinite(co.part.cpu().numpy()))
    assert et < 1e-3 and ep < 1e-2
    got = np.array([dp.dgamma, dp.dDtau, dp.dkappa, dp.dK, dp.dA])
    scale = np.abs(rdp) + 1e-3 * np.max(np.abs(rdp))
    # the scalar cotangents are sums over all cells, the switched entries included: the same oracle VJP with its input
    # moved by one fp32 rounding says how far they are defined (reading R28)
    prng = np.random.default_rng(1000 + k)
    s_pert = O.State(gas_k.astype(np.float64) * (1.0 + 6e-8 * prng.standard_normal(gas_k.shape)), part_k, a_s[k],
                     dt_prev=dt_s[k - 1], step=k)
    rg2, rp2, rdp2 = O.step_vjp(P, s_pert, dt_s[k], a_s[k + 1], cg, cp)
    sens_g = PT.rel_l2(rg2, rg)
    print(f"   the oracle's gas cotangent under one fp32 rounding of its input moves by {sens_g:.2e}")
    # (over all entries: printed, not asserted -- heavy-tailed at these epochs, 0.13 ... 0.32 on the GPU where one perturbed
    # copy of the oracle moves by 5e-3 (k = 50) ... 0.35 (k = 90); the bound on all but the worst 0.1 % is the claim)
    print("   dparams", got, "oracle", rdp, "oracle under one fp32 rounding of its input", rdp2)
    # d K and d A come from the particle / Poisson side (smooth sums): tight.  d gamma, d Dtau, d kappa sum the switched
    # entries of a RANDOM cotangent: at k = 90 d gamma is a difference of O(1e3) terms that lands anywhere in +-7 from run to
    # run (-7.9, 2.9, -6.7, -1.5 on the GPU against -7.9, -6.4, -5.3, 0.7 in the oracle), so these three get the larger of a
    # 10 % / absolute floor and five times what the oracle's own perturbed copy does
    assert np.all(np.abs(got - rdp)[3:] < 5e-3 * scale[3:]), (got, rdp)
    floor_abs = np.array([20.0, 0.1 * abs(rdp[1]), 0.1 * abs(rdp[2])])
    assert np.all(np.abs(got - rdp)[:3] < np.maximum(floor_abs, 5.0 * np.abs(rdp2 - rdp)[:3])), (got, rdp, rdp2)
    ctx.close()


@pytest.mark.parametrize("d", [0, 1, 2])
def test_sweep_and_its_vjp_with_a_large_limiter_epsilon(api, torch_, O, W, d):
    """Eq. 18's epsilon at the scale of the limiter's arguments (lim_eps = 1e-2 on O(1) fluxes): the kernels' epsilon
    branches (denominator and numerators of the partials) against the oracle, free of any multi-step amplification."""
    N, eps = 64, 1e-2
    gas, _ = W.smooth_random_state(N, 31 + d, amp=0.1, n_part_side=2)
    gas = gas.astype(np.float32)
    rng = np.random.default_rng(3 + d)
    g = (0.2 * rng.standard_normal((N, N, N))).astype(np.float32)
    cot = rng.standard_normal(gas.shape).astype(np.float32)
    lam, kap, gamma = 0.11, 0.07, 5.0 / 3.0
    ctx = api.Context(N, float(N), gamma, n_part_side=0, static_mode=1, gravity_on=0, e_floor=1e-6, lim_eps=eps)
    out = ctx.dh_sweep(d, _gpu(torch_, gas), _gpu(torch_, g), lam, kap).cpu().numpy()
    ref, _ = O.sweep(gas.astype(np.float64), d, lam, kap, gamma, g.astype(np.float64), e_floor=1e-6, lim_eps=eps)
    ref0, _ = O.sweep(gas.astype(np.float64), d, lam, kap, gamma, g.astype(np.float64), e_floor=1e-6, lim_eps=1e-20)
    assert max(PT.field_err(out, ref).values()) < 1e-5
    assert max(PT.field_err(ref0, ref).values()) > 1e-4          # the epsilon matters at this size
    cin, gb, sc = ctx.dh_sweep_vjp(d, _gpu(torch_, gas), _gpu(torch_, g), lam, kap, _gpu(torch_, cot))
    rin, rgb, rsc = O.sweep_vjp(gas.astype(np.float64), d, lam, kap, gamma, cot.astype(np.float64), g.astype(np.float64),
                                e_floor=1e-6, lim_eps=eps)
    e_all, e_trim = PT.rel_l2(cin.cpu().numpy(), rin), PT.rel_l2_trimmed(cin.cpu().numpy(), rin, frac=2e-4)
    print(f"sweep vjp with lim_eps 1e-2, d={d}: rel L2 {e_all:.2e} (trimmed {e_trim:.2e}), g_bar {PT.rel_l2(gb.cpu().numpy(), rgb):.2e}")
    assert e_all < 1e-3 and e_trim < 2e-5 and PT.rel_l2(gb.cpu().numpy(), rgb) < 1e-3
    sc = sc.cpu().numpy()
    for k, key in ((0, "lam"), (1, "kap"), (2, "gamma")):
        assert abs(sc[k] - rsc[key]) < 1e-3 * max(abs(rsc[key]), np.sqrt(gas[0].size)), (key, sc[k], rsc[key])
    ctx.close()


@pytest.mark.parametrize("which", [0, 2])
def test_gradient_conditioning_against_the_limiter_epsilon(api, torch_, O, W, IC, which):
    """VERDICT r01 weak #2 (iv), the experiment of DESIGN.md reading R28: the same gradient (configs 0 and 2, the configs'
    own losses) with the epsilon of Eq. 18 ("regular near a = b = 0") raised from 1e-20 to the scale of
    the limiter's arguments.  For each value: how far the fp64 oracle's gradient moves under one fp32 rounding of its
    input, and how far the GPU is from it.  With |a + b| << eps the jump of d phi / d a at the gate, 2 b / (b + eps), closes, so
    both numbers must fall together; the bound on the GPU is the conditioning rule of R28 at every epsilon."""
    cfg = W.CONFIGS[which]
    delta, gas, part = IC.coupled_ic(W, cfg)
    target = None
    if which == 2:
        target = cfg.f_b * (1.0 + W.gaussian_field(cfg.N, cfg.box, cfg.target_seed, cfg.rms_delta))
    rows = []
    for eps in (1e-20, 1e-4, 1e-2, 1.0):
        P = PT.oracle_params(O, cfg, lim_eps=eps)
        a_s, dt_s = O.schedule_lna(P, cfg.a0, cfg.a1, cfg.n_steps)

        def oracle_grad(g_, p_):
            gf, pf, _, _ = O.run(P, g_, p_, cfg.a0, a_s[1:], dt_s)
            cot = np.zeros_like(gf)
            cot[0] = gf[0] / np.linalg.norm(gf[0]) if target is None else 2.0 * (gf[0] - target)
            return O.run_vjp(P, g_, p_, cfg.a0, a_s[1:], dt_s, cot, np.zeros_like(pf))[0], gf
        rg, gf = oracle_grad(gas, part)
        prng = np.random.default_rng(7)
        rg2, _ = oracle_grad(gas.astype(np.float64) * (1.0 + 6e-8 * prng.standard_normal(gas.shape)),
                             part.astype(np.float64) * (1.0 + 6e-8 * prng.standard_normal(part.shape)))
        sens = PT.rel_l2(rg2, rg)
        ctx = api.context_for(cfg, lim_eps=eps)
        sg = api.State(gas, part, cfg.a0)
        ctx.dh_run(sg, a_s[1:], dt_s, 10)
        e_fwd = max(PT.field_err(sg.gas.cpu().numpy(), gf).values())
        cg = torch_.zeros_like(sg.gas)
        if target is None:
            rho = sg.gas[0].double()
            cg[0] = (rho / rho.norm()).float()
        else:
            cg[0] = 2.0 * (sg.gas[0] - _gpu(torch_, target))
        ct = api.Cot(cg, torch_.zeros_like(sg.part))
        ctx.dh_run_vjp(ct, ct)
        got = ct.gas.cpu().numpy()
        ctx.close()
        err, err_t = PT.rel_l2(got, rg), PT.rel_l2_trimmed(got, rg, frac=1e-2)
        rows.append((eps, sens, err, err_t, e_fwd))
        print(f"config{which} lim_eps {eps:.0e}: oracle moves itself {sens:.2e}; GPU vs oracle {err:.2e} "
              f"(all but the worst 1 %: {err_t:.2e}); forward {e_fwd:.1e}")
        assert np.all(np.isfinite(got))
    # an experiment, so loose assertions: the GPU stays within a few times what the oracle does to itself at every epsilon
    # (one perturbed copy is a noisy estimate of that), and the looseness follows the gate -- it shrinks once epsilon
    # dominates the limiter's arguments (the scheme is first order by then)
    # (config 2 over ALL entries is heavy-tailed on the GPU -- 2.6e-2 ... 1.4e-1 from run to run, see
    # test_config2_full_run_forward_and_gradient -- so it gets that test's stated cap; all but the worst 1 % is the tight one)
    for eps, sens, err, err_t, e_fwd in rows:
        assert err < (0.35 if which == 2 else 5.0 * max(1e-3, sens)), rows
        assert err_t < (1.2e-2 if which == 2 else 1e-3), rows
    assert rows[-1][1] < rows[0][1] / 2.0 and rows[-1][2] < rows[0][2] / 2.0, rows
