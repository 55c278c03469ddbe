"""Stand-ins for compute-sanitizer, which is closed on this pool.

initcheck: every device buffer the context owns is filled with NaN (dh_debug_poison) before the calls that must not depend
on its old contents; the results have to be the same numbers as without (bit for bit where no atomics are involved) and
finite.  memcheck: every caller-owned array (5 gas fields, 6 particle arrays, and as many cotangents) is carved out of one
buffer with NaN-patterned guard zones between neighbours; after a step and its VJP every guard word must be untouched and
the results must equal those of ordinary tensors."""
import ctypes as C

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


def _run_and_reverse(api, torch, ctx, gas, part, cfg, a_s, dt_s, stride, poison):
    st = api.State(gas, part, cfg.a0)
    if poison:
        ctx.dh_debug_poison(1)
    ctx.dh_run(st, a_s[1:], dt_s, stride)
    cg = torch.zeros_like(st.gas); cg[0] = st.gas[0]
    ct = api.Cot(cg, torch.zeros_like(st.part))
    if poison:
        ctx.dh_debug_poison(0)
    dp = ctx.dh_run_vjp(ct, ct)
    return st.gas.clone(), st.part.clone(), ct.gas.clone(), ct.part.clone(), dp.as_dict()


@pytest.mark.parametrize("case", ["hydro_only", "coupled", "coupled_recompute", "dual_energy", "dual_energy_march"])
def test_poisoned_scratch_changes_nothing(api, torch_, W, IC, case):
    cfg = W.scaled_config(0, 32, n_steps=7, a1=0.03)
    _, gas, part = IC.coupled_ic(W, cfg)
    a_s, dt_s = api.dh_schedule_lna(cfg.a0, cfg.a1, cfg.n_steps)
    kw, tune = {}, {}
    if case == "hydro_only":
        kw = dict(gravity_on=0, n_part_side=0)
        part = np.zeros((6, 0), dtype=np.float32)
    elif case == "coupled_recompute":
        tune = {"tape": 0, "gstore": 0}
    elif case.startswith("dual_energy"):
        kw = dict(dual_energy=1, dual_eta=1e-3, want_dsched=0 if case.endswith("march") else 1)
        vf, e0 = api.ic_factors_for(cfg)
        gas = np.concatenate([gas, (e0 * gas[0].astype(np.float64))[None].astype(np.float32)], axis=0)
    ctx = api.context_for(cfg, **kw)
    for k, v in tune.items():
        ctx.dh_tune(k, v)
    ref = _run_and_reverse(api, torch_, ctx, gas, part, cfg, a_s, dt_s, 3, poison=False)      # also allocates everything
    got = _run_and_reverse(api, torch_, ctx, gas, part, cfg, a_s, dt_s, 3, poison=True)
    for j, (a, b) in enumerate(zip(ref[:4], got[:4])):
        assert bool(torch_.isfinite(b).all())
        if case == "hydro_only":
            assert torch_.equal(a, b)                             # no atomics anywhere: the same bits
        elif a.numel() and j < 2:                                 # forward fields: the order of the deposits' atomics only
            assert float((a - b).abs().max()) <= 2e-5 * float(a.abs().max())
        elif a.numel():                                           # cotangents: the same, amplified at the switches (R28)
            an, bn = a.double().cpu().numpy(), b.double().cpu().numpy()
            assert PT.rel_l2_trimmed(bn, an, frac=1e-2) < 1e-3 and PT.rel_l2(bn, an) < 5e-2
    # want_dsched = 0 leaves the cotangents of Dtau and kappa unset (NaN by contract, include/diffhydro.h)
    assert all(np.isfinite(v) for k, v in got[4].items() if kw.get("want_dsched", 1) or k not in ("dDtau", "dkappa"))
    assert abs(got[4]["dgamma"] - ref[4]["dgamma"]) <= 1e-3 * abs(ref[4]["dgamma"]) + 1e-12
    # the single-step calls and the host-buffer chain after a poisoning of everything
    st = api.State(gas, part, cfg.a0)
    ctx.dh_debug_poison(1)
    ctx.dh_step(st, dt_s[0], a_s[1])
    st_in = api.State(gas, part, cfg.a0)
    co = api.Cot(torch_.ones_like(st.gas), torch_.ones_like(st.part))
    ctx.dh_debug_poison(1)
    dp = ctx.dh_step_vjp(st_in, dt_s[0], a_s[1], co, co)
    assert bool(torch_.isfinite(st.gas).all()) and bool(torch_.isfinite(co.gas).all()) and np.isfinite(dp.dgamma)
    if st.part.numel():
        assert bool(torch_.isfinite(st.part).all()) and bool(torch_.isfinite(co.part).all())
    ctx.close()


def _carve(torch, sizes, guard=4096):
    """One buffer of NaN-patterned words with the requested arrays inside, a guard zone before, between and after them.
    Returns (buffer, [views], guard mask)."""
    total = guard + sum(s + guard for s in sizes)
    buf = torch.full((total,), float("nan"), dtype=torch.float32, device="cuda")
    views, mask = [], torch.ones(total, dtype=torch.bool, device="cuda")
    off = guard
    for s in sizes:
        views.append(buf[off:off + s])
        mask[off:off + s] = False
        off += s + guard
    return buf, views, mask


@pytest.mark.parametrize("nps", [32, 24])
def test_guard_zones_around_caller_arrays_stay_untouched(api, torch_, W, IC, nps):
    """One coupled step and its VJP with every caller-owned array surrounded by guard words (a lattice of 24^3 particles
    on a 32^3 mesh gives the particle kernels a ragged last block)."""
    cfg = W.scaled_config(0, 32, n_steps=2, a1=0.012)
    gas, part = W.smooth_random_state(32, 5, amp=0.05, n_part_side=nps)
    gas = gas.astype(np.float32); part = part.astype(np.float32)
    n3, npart = 32 ** 3, nps ** 3
    a_s, dt_s = api.dh_schedule_lna(cfg.a0, cfg.a1, cfg.n_steps)
    ctx = api.context_for(cfg, n_part_side=nps)
    # ordinary tensors first
    st = api.State(gas, part, cfg.a0)
    ctx.dh_step(st, dt_s[0], a_s[1])
    rng = np.random.default_rng(2)
    cg = rng.standard_normal(gas.shape).astype(np.float32); cp = rng.standard_normal(part.shape).astype(np.float32)
    co = api.Cot(cg, cp)
    ctx.dh_step_vjp(api.State(gas, part, cfg.a0), dt_s[0], a_s[1], co, co)
    # the same through guarded arrays
    buf, v, mask = _carve(torch_, [n3] * 5 + [npart] * 6 + [n3] * 5 + [npart] * 6 + [n3] * 5 + [npart] * 6)
    state, cot, state_in = v[:11], v[11:22], v[22:33]
    for k in range(5):
        state[k].copy_(torch_.from_numpy(gas[k].ravel())); state_in[k].copy_(torch_.from_numpy(gas[k].ravel()))
        cot[k].copy_(torch_.from_numpy(cg[k].ravel()))
    for k in range(6):
        state[5 + k].copy_(torch_.from_numpy(part[k])); state_in[5 + k].copy_(torch_.from_numpy(part[k]))
        cot[5 + k].copy_(torch_.from_numpy(cp[k]))

    def c_state(arrs):
        s = api.dh_state()
        s.gas = (C.c_void_p * 5)(*[a.data_ptr() for a in arrs[:5]])
        s.part = (C.c_void_p * 6)(*[a.data_ptr() for a in arrs[5:11]])
        s.a, s.dt_prev, s.step = cfg.a0, 0.0, 0
        return s
    cs = c_state(state)
    assert api._lib.dh_step(ctx._h, C.byref(cs), float(dt_s[0]), float(a_s[1]), None) == 0
    cc = api.dh_cot()
    cc.gas = (C.c_void_p * 5)(*[a.data_ptr() for a in cot[:5]])
    cc.part = (C.c_void_p * 6)(*[a.data_ptr() for a in cot[5:11]])
    csi = c_state(state_in)
    dp = api.dh_dparams()
    assert api._lib.dh_step_vjp(ctx._h, C.byref(csi), float(dt_s[0]), float(a_s[1]), C.byref(cc), C.byref(cc), C.byref(dp)) == 0
    torch_.cuda.synchronize()
    assert bool(torch_.isnan(buf[mask]).all()), "a guard word was written"
    for k in range(5):
        ref_k, got_k = st.gas[k].ravel(), state[k]
        assert float((ref_k - got_k).abs().max()) <= 1e-5 * float(ref_k.abs().max())
        assert float((co.gas[k].ravel() - cot[k]).abs().max()) <= 2e-3 * float(co.gas.abs().max())
    for k in range(6):
        assert float((st.part[k] - state[5 + k]).abs().max()) <= 1e-4
        assert bool((state_in[5 + k] == torch_.from_numpy(part[k]).cuda()).all())         # the checkpoint is read only
    ctx.close()
