"""Pins of oracle/subgrid.py (section 2.4, Eq. 22-25) against what the paper and the mathematics fix."""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def SG():
    from oracle import subgrid
    return subgrid


def test_eq24_literal_formula(SG):
    """Eq. 24 retyped with its exponentials (moderate values, where they do not overflow) equals the log-odds form."""
    rng = np.random.default_rng(0)
    pi0 = rng.uniform(0.05, 0.9, 1000); g0 = rng.gumbel(size=1000); g1 = rng.gumbel(size=1000); tau = 0.5
    a = np.exp((np.log(pi0) + g0) / tau); b = np.exp((np.log(1 - pi0) + g1) / tau)
    assert np.max(np.abs(SG.relaxed_bernoulli(pi0, g0, g1, tau) - a / (a + b))) < 1e-14


def test_gumbel_max_limit_samples_a_bernoulli_with_probability_pi0(SG):
    """tau -> 0: z is the indicator of log pi0 + g0 > log(1 - pi0) + g1 (the Gumbel-max trick), a Bernoulli(pi0) draw:
    its mean over 2e5 draws is pi0 within 4 sigma (PAPER.md:271 'will exactly match the true discrete random field')."""
    rng = np.random.default_rng(1)
    n = 200000
    for pi0 in (0.03, 0.3, 0.8):
        g0 = rng.gumbel(size=n); g1 = rng.gumbel(size=n)
        z = SG.relaxed_bernoulli(np.full(n, pi0), g0, g1, 1e-4)
        assert np.mean((z > 1e-9) & (z < 1 - 1e-9)) < 0.01          # only draws within ~2e-3 of a tie stay soft
        assert np.array_equal(z > 0.5, np.log(pi0) + g0 > np.log(1 - pi0) + g1)
        assert abs(z.mean() - pi0) < 4 * np.sqrt(pi0 * (1 - pi0) / n)
    # at the paper's tau = 0.1 the relaxed field keeps the right mean to a few per cent and stays in (0, 1)
    z = SG.relaxed_bernoulli(np.full(n, 0.3), rng.gumbel(size=n), rng.gumbel(size=n), 0.1)
    assert np.all((z >= 0) & (z <= 1)) and abs(z.mean() - 0.3) < 0.02


def test_eq25_sharp_threshold_limit(SG):
    """a, b -> 0: star formation is possible below T_c if the density criterion is exceeded, with
    probability Pi0; impossible otherwise."""
    rho = np.array([0.5, 2.0, 2.0, 0.5]) * 0.16; T = np.array([1e3, 1e3, 1e5, 1e5])
    p = SG.class_probability(rho, T, 0.16, T_c=1e4, delta_c=0.5, Pi0=0.2, a_w=1e-6, b_w=1e-3)
    assert np.allclose(p, [0.0, 0.2, 0.0, 0.0], atol=1e-15)
    # on the thresholds both sigmoids are 1/2
    p = SG.class_probability(np.array([1.5 * 0.16]), np.array([1e4]), 0.16, 1e4, 0.5, 0.2, 0.3, 50.0)
    assert abs(p[0] - 0.05) < 1e-15


def test_step_injects_energy_only_and_transpose_matches_finite_differences(SG):
    rng = np.random.default_rng(2)
    n = 5
    gas = np.zeros((5, n, n, n))
    gas[0] = 0.16 * (1 + 0.8 * rng.uniform(-1, 1, (n, n, n))); gas[1:4] = 0.05 * rng.standard_normal((3, n, n, n))
    gas[4] = gas[0] * (0.02 + 0.01 * rng.uniform(size=(n, n, n))) + 0.5 * np.sum(gas[1:4] ** 2, axis=0) / gas[0]
    g0 = rng.gumbel(size=(n, n, n)); g1 = rng.gumbel(size=(n, n, n))
    par = dict(rho_mean=0.16, t_per_e=4e5, T_c=1e4, delta_c=0.1, Pi0=0.3, e_inject=0.03, a_w=0.3, b_w=2e3, tau=0.1)
    out, z = SG.step(gas, g0, g1, **par)
    assert np.array_equal(out[:4], gas[:4]) and np.all(out[4] >= gas[4]) and np.all((z > 0) & (z < 1))
    assert np.allclose(out[4] - gas[4], par["e_inject"] * gas[0] * z, rtol=0, atol=1e-15)
    cg = rng.standard_normal(gas.shape); cz = rng.standard_normal(z.shape)
    cin, dpar = SG.step_vjp(gas, g0, g1, cot_gas=cg, cot_z=cz, **par)

    def loss(gas_, **kw):
        p = dict(par); p.update(kw)
        o, zz = SG.step(gas_, g0, g1, **p)
        return np.sum(cg * o) + np.sum(cz * zz)
    v = rng.standard_normal(gas.shape); h = 1e-7
    fd = (loss(gas + h * v) - loss(gas - h * v)) / (2 * h)
    assert abs(fd - np.sum(cin * v)) < 1e-6 * max(abs(fd), 1.0)
    for i, (name, hh) in enumerate([("T_c", 1e-2), ("delta_c", 1e-7), ("Pi0", 1e-7), ("e_inject", 1e-7)]):
        fd = (loss(gas, **{name: par[name] + hh}) - loss(gas, **{name: par[name] - hh})) / (2 * hh)
        assert abs(fd - dpar[i]) < 1e-5 * max(abs(fd), 1e-3), (name, fd, dpar[i])
