"""Cosmological-parameter gradients through the step scalars.

CPU part: the library's host-only dh_chain_cosmology fed with the ORACLE's per-step scalar cotangents must equal the
central finite difference of the oracle's loss w.r.t. Omega_m / H0 with the schedule rebuilt (initial state fixed).
GPU part: the per-step cotangents dh_run_vjp keeps (want_dsched = 1) against the oracle's, step by step."""
import ctypes as C
import os

import numpy as np
import pytest

import parity as PT

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


class Cosmo(C.Structure):
    _fields_ = [("H0", C.c_double), ("Omega_m", C.c_double), ("Omega_b", C.c_double), ("Omega_L", C.c_double),
                ("static_mode", C.c_int32)]


def _oracle_per_step(O, P, gas, part, a0, a_s, dt_s):
    """Forward with every step's input kept, then the step VJPs in reverse: (loss, per-step dparams (n,5), cot_gas0)."""
    s = O.State(gas, part, a0)
    ins = []
    for k in range(len(dt_s)):
        ins.append(s.copy())
        O.step(P, s, dt_s[k], a_s[k + 1])
    loss = 0.5 * np.sum(s.gas[0] ** 2)
    cg = np.zeros_like(s.gas); cg[0] = s.gas[0]
    cp = np.zeros_like(s.part)
    per = np.zeros((len(dt_s), 5))
    for k in reversed(range(len(dt_s))):
        cg, cp, per[k] = O.step_vjp(P, ins[k], dt_s[k], a_s[k + 1], cg, cp)
    return loss, per, cg


def _case(W, IC, N, n_steps):
    cfg = W.scaled_config(0, N, n_steps=n_steps, a1=0.03, rms_delta=0.05)
    _, gas, part = IC.coupled_ic(W, cfg)
    return cfg, gas, part


def test_chain_matches_finite_difference_of_the_oracle_loss(O, W, IC):
    lib = C.CDLL(os.path.join(ROOT, "paper_2502_02294_b200", "libdiffhydro.so"))
    dp = C.POINTER(C.c_double)
    lib.dh_chain_cosmology.argtypes = [C.POINTER(Cosmo), C.c_double, C.c_double, C.c_int, dp, dp, dp]
    cfg, gas, part = _case(W, IC, 16, 5)
    Om, OL, H0 = 0.31, 0.69, 100.0

    def run(Om_, H0_):
        # the baryon FRACTION is held fixed (it sets particle mass and mean densities, not a step scalar)
        P = PT.oracle_params(O, cfg, Omega_m=Om_, Omega_b=0.16 * Om_, Omega_L=OL, H0=H0_)
        a_s, dt_s = O.schedule_lna(P, cfg.a0, cfg.a1, cfg.n_steps)
        return _oracle_per_step(O, P, gas, part, cfg.a0, a_s, dt_s)
    _, per, _ = run(Om, H0)
    co = Cosmo(H0, Om, 0.16 * Om, OL, 0)
    dOm, dH0 = C.c_double(0), C.c_double(0)
    per_c = np.ascontiguousarray(per)
    assert lib.dh_chain_cosmology(C.byref(co), cfg.a0, cfg.a1, cfg.n_steps, per_c.ctypes.data_as(dp), C.byref(dOm),
                                  C.byref(dH0)) == 0
    h = 1e-4
    fd_Om = (run(Om + h, H0)[0] - run(Om - h, H0)[0]) / (2 * h)
    fd_H0 = (run(Om, H0 + 100 * h)[0] - run(Om, H0 - 100 * h)[0]) / (200 * h)
    assert abs(dOm.value - fd_Om) < 1e-4 * abs(fd_Om), (dOm.value, fd_Om)      # FD step 1e-4 on a piecewise-smooth run
    assert abs(dH0.value - fd_H0) < 1e-4 * abs(fd_H0), (dH0.value, fd_H0)


@pytest.mark.gpu
def test_per_step_scalar_cotangents_match_oracle(O, W, IC):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2502_02294_b200 import api
    cfg, gas, part = _case(W, IC, 32, 7)
    Om, OL = 0.31, 0.69
    P = PT.oracle_params(O, cfg, Omega_m=Om, Omega_b=0.16 * Om, Omega_L=OL)
    a_s, dt_s = O.schedule_lna(P, cfg.a0, cfg.a1, cfg.n_steps)
    _, per_ref, cg_ref = _oracle_per_step(O, P, gas, part, cfg.a0, a_s, dt_s)
    ctx = api.context_for(cfg, Omega_m=Om, Omega_L=OL, Omega_b=0.16 * Om)
    a_g, dt_g = api.dh_schedule_lna(cfg.a0, cfg.a1, cfg.n_steps, H0=cfg.H0, Omega_m=Om, Omega_b=0.16 * Om, Omega_L=OL)
    assert np.max(np.abs(dt_g / dt_s - 1)) < 1e-12
    sg = api.State(gas, part, cfg.a0)
    ctx.dh_run(sg, a_g[1:], dt_g, 3)
    cg = torch.zeros_like(sg.gas); cg[0] = sg.gas[0]
    ct = api.Cot(cg, torch.zeros_like(sg.part))
    tot = ctx.dh_run_vjp(ct, ct)
    per = ctx.dh_get_step_dparams(cfg.n_steps)
    # piecewise-differentiable run, deposit atomics: the bounds of reading R28 (all but the worst 1 % of entries within
    # the north-star 1e-3; the whole field within a few gate flips of it); the scalar cotangents are global sums
    eg, egt = PT.rel_l2(ct.gas.cpu().numpy(), cg_ref), PT.rel_l2_trimmed(ct.gas.cpu().numpy(), cg_ref, frac=1e-2)
    scale = np.max(np.abs(per_ref), axis=0)
    es = np.max(np.abs(per - per_ref) / (np.abs(per_ref) + 1e-2 * scale[None, :]))
    print(f"cosmology chain: cot gas {eg:.2e} (trimmed {egt:.2e}), per-step scalars {es:.2e}")
    assert egt < 1e-3 and eg < 5e-3
    assert es < 5e-3, (per, per_ref)
    assert np.allclose(per.sum(axis=0), [tot.dgamma, tot.dDtau, tot.dkappa, tot.dK, tot.dA], rtol=1e-12, atol=0)
    got = ctx.dh_chain_cosmology(cfg.a0, cfg.a1, per)
    ref = ctx.dh_chain_cosmology(cfg.a0, cfg.a1, per_ref)
    assert abs(got[0] / ref[0] - 1) < 5e-3 and abs(got[1] / ref[1] - 1) < 5e-3, (got, ref)
    with pytest.raises(api.DhError):
        ctx.dh_get_step_dparams(cfg.n_steps + 1)
    ctx.close()
