"""CPU ORACLE of the dual-energy variant of the relaxing-TVD sweep, its transpose, and the coupled step built on it.

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module; it never imports the CUDA package and shares no code with it.

What it follows.  PAPER.md:85 (section 2.3): "For now, we use a single energy formalism ... This can straightforwardly be
expanded to a dual energy formalism, bringing more accurate solutions in low-density, high-velocity regions of the flow",
and the internal-energy source the paper prints next to its flux vector, S_e = (0, 0, -a p div U) (Eq. 8) --
the right-hand side of the internal-energy equation, which the total-energy equation (Eq. 7) does not have (reading R2).
The paper gives no further detail; readings R33-R36 of DESIGN.md, stated here in the paper's tilde variables
(rho, m = a rho U, eps = a^2 rho E; dtau = dt / a^2; v~ = m/rho):

  R33  A sixth mesh field q = a^2 rho_b e (internal energy density) obeys  dq/dtau + div(q v~) = -p~ div v~ ; like Eq. 7
       it has no Hubble term (reading R1).  Gravity does no work on it.
  R34  Every evaluation of the primitive variables (both Runge-Kutta stages of every sweep) selects the thermal energy
       e~ = e~_T = eps/rho - |m|^2 / (2 rho^2)   if e~_T > eta * eps/rho   (the total energy resolves it),
       e~ = q / rho                              otherwise,
       with eta = 1e-3 by default; floor, pressure and freezing speed as in the single-energy scheme (R17, R11).  The
       selected value q_s = rho e~ replaces q from then on (the two energies are synchronised wherever eps is trusted).
  R35  In the sweep along d the advective part of the q equation goes through the same flux split, relaxation and limiter
       as the five conserved components (sixth component of F is q_s v~, of the state q_s); the source -p~ d v~_d / dx_d is
       added in both stages with centred differences of the cell velocities:
          stage A:  q*_n = q_s,n - (lam/2)(Phi_q,n+1/2 - Phi_q,n-1/2) - (lam/4) p~_n  (v~_n+1 - v~_n-1)
          stage B:  q'_n = q_s,n -  lam   (Phi*_q,n+1/2 - Phi*_q,n-1/2) - (lam/2) p~*_n (v~*_n+1 - v~*_n-1)
  R36  The five conserved fields are never modified by the dual-energy logic (conservation stays exact, R17); only the
       thermal energy that enters p~ and c changes.  Sub-gradients: the selection has the derivative of the branch taken (R26).

With eta = 0 and e~_T > 0 everywhere the five conserved fields are those of the single-energy sweep (pin), and q' follows
rho e~_T of the input passively.

Everything is plain numpy in fp64: whole-array expressions with numpy.roll for the neighbours along the sweep axis
(periodic), in the order of the formulas above; no blocking, fusion or reordering.  Pins: tests/test_oracle_dual_energy.py.
"""
from __future__ import annotations

import numpy as np

STRANG = ((0, 1, 2), (2, 1, 0), (2, 0, 1), (1, 0, 2), (1, 2, 0), (0, 2, 1))   # PAPER.md:152, reading R9


# ---------------------------------------------------------------------------------------------- limiter (Eq. 18, R8) ----
def limiter(a, b, eps):
    on = a * b > 0.0
    s = np.where(a > 0.0, eps, -eps)
    den = np.where(on, a + b + s, 1.0)
    return np.where(on, 2.0 * a * b / den, 0.0)


def limiter_grad(a, b, eps):
    on = a * b > 0.0
    s = np.where(a > 0.0, eps, -eps)
    den = np.where(on, a + b + s, 1.0)
    da = np.where(on, 2.0 * b * (b + s) / (den * den), 0.0)
    db = np.where(on, 2.0 * a * (a + s) / (den * den), 0.0)
    return da, db


# ----------------------------------------------------------------------------------------- primitive variables (R34) ----
def prim(u, q, gamma, e_floor, eta):
    """u = (rho, m_n, m_t1, m_t2, eps) and q on any array shape.  Returns a dict with FR, FL (6 components each: the five
    conserved ones and the internal energy), c, v, p, q_s, and the branch masks."""
    rho, mn, mt1, mt2, eps = u
    v = mn / rho
    m2 = mn * mn + mt1 * mt1 + mt2 * mt2
    eT = eps / rho - m2 / (2.0 * rho * rho)
    useT = eT > eta * eps / rho                                   # R34
    e = np.where(useT, eT, q / rho)
    qs = rho * e
    active = e > e_floor                                          # R17
    ep = np.where(active, e, e_floor)
    p = (gamma - 1.0) * rho * ep
    cs = np.sqrt(gamma * (gamma - 1.0) * ep)
    c = np.abs(v) + cs                                            # PAPER.md:117, per cell (R11)
    F = [mn, mn * v + p, mt1 * v, mt2 * v, (eps + p) * v, qs * v]
    U6 = [rho, mn, mt1, mt2, eps, qs]
    FR = [(c * U6[k] + F[k]) / 2.0 for k in range(6)]             # R4
    FL = [(c * U6[k] - F[k]) / 2.0 for k in range(6)]
    return dict(FR=FR, FL=FL, c=c, v=v, p=p, qs=qs, useT=useT, active=active, e=e, ep=ep, cs=cs, m2=m2)


def prim_vjp(u, q, gamma, e_floor, eta, P, FRb, FLb, vb0, pb0, qsb0):
    """Transpose of prim at (u, q) (P = its forward result).  Cotangents in: FRb, FLb (6 each) and the extra cotangents
    of v, p and q_s that the internal-energy source and the update hand over.  Returns (ub[5], qb, gamma_b)."""
    rho, mn, mt1, mt2, eps = u
    v, p, qs, c, cs, ep, e, m2 = P["v"], P["p"], P["qs"], P["c"], P["cs"], P["ep"], P["e"], P["m2"]
    U6 = [rho, mn, mt1, mt2, eps, qs]
    cub = [(FRb[k] + FLb[k]) / 2.0 for k in range(6)]
    Fb = [(FRb[k] - FLb[k]) / 2.0 for k in range(6)]
    cb = sum(cub[k] * U6[k] for k in range(6))
    U6b = [c * cub[k] for k in range(6)]
    mnb = Fb[0] + Fb[1] * v
    vb = vb0 + Fb[1] * mn + Fb[2] * mt1 + Fb[3] * mt2 + Fb[4] * (eps + p) + Fb[5] * qs
    pb = pb0 + Fb[1] + Fb[4] * v
    mt1b = Fb[2] * v
    mt2b = Fb[3] * v
    epsb = Fb[4] * v
    qsb = qsb0 + U6b[5] + Fb[5] * v
    vb = vb + np.sign(v) * cb                                     # d|v|/dv = sign(v), sign(0) = 0 (R26)
    epb = cb * gamma * (gamma - 1.0) / (2.0 * cs)
    gamma_b = np.sum(cb * (2.0 * gamma - 1.0) * ep / (2.0 * cs))
    gamma_b += np.sum(pb * rho * ep)
    rhob = pb * (gamma - 1.0) * ep
    epb = epb + pb * (gamma - 1.0) * rho
    eb = np.where(P["active"], epb, 0.0)
    eb = eb + qsb * rho                                           # q_s = rho e
    rhob = rhob + qsb * e
    eTb = np.where(P["useT"], eb, 0.0)                            # e = e_T or q / rho
    qb = np.where(P["useT"], 0.0, eb / rho)
    rhob = rhob + np.where(P["useT"], 0.0, -eb * q / (rho * rho))
    epsb = epsb + eTb / rho
    rhob = rhob + eTb * (-eps / (rho * rho) + m2 / (rho * rho * rho))
    mnb = mnb - eTb * mn / (rho * rho)
    mt1b = mt1b - eTb * mt1 / (rho * rho)
    mt2b = mt2b - eTb * mt2 / (rho * rho)
    mnb = mnb + vb / rho                                          # v = m_n / rho
    rhob = rhob - vb * mn / (rho * rho)
    ub = [U6b[0] + rhob, U6b[1] + mnb, U6b[2] + mt1b, U6b[3] + mt2b, U6b[4] + epsb]
    return ub, qb, float(gamma_b)


# ------------------------------------------------------------------------------------------------- one sweep (R35) ----
def _forward(u, q, g, lam, kap, gamma, e_floor, lim_eps, eta, ax):
    up = lambda x: np.roll(x, -1, ax)                             # x_{n+1}
    dn = lambda x: np.roll(x, 1, ax)                              # x_{n-1}
    g0 = 0.0 if g is None else g
    P = prim(u, q, gamma, e_floor, eta)
    Phi = [P["FR"][k] - up(P["FL"][k]) for k in range(6)]         # stage A: first-order upwind of each family (Eq. 12, 14)
    S = [0.0, u[0] * g0, 0.0, 0.0, u[1] * g0]                     # S_g of Eq. 8 along d (R16)
    us = [u[k] - (lam / 2.0) * (Phi[k] - dn(Phi[k])) + (kap / 2.0) * S[k] for k in range(5)]
    qst = P["qs"] - (lam / 2.0) * (Phi[5] - dn(Phi[5])) - (lam / 4.0) * P["p"] * (up(P["v"]) - dn(P["v"]))
    Ps = prim(us, qst, gamma, e_floor, eta)
    FRs, FLs = Ps["FR"], Ps["FL"]
    aR = [(FRs[k] - dn(FRs[k])) / 2.0 for k in range(6)]          # Eq. 15-17 for the right-moving family
    bR = [(up(FRs[k]) - FRs[k]) / 2.0 for k in range(6)]
    aL = [(up(FLs[k]) - FLs[k]) / 2.0 for k in range(6)]          # mirror image for the left-moving family (R7)
    bL = [(up(up(FLs[k])) - up(FLs[k])) / 2.0 for k in range(6)]
    Phis = [(FRs[k] + limiter(aR[k], bR[k], lim_eps)) - (up(FLs[k]) - limiter(aL[k], bL[k], lim_eps)) for k in range(6)]
    Ss = [0.0, us[0] * g0, 0.0, 0.0, us[1] * g0]
    out = [u[k] - lam * (Phis[k] - dn(Phis[k])) + kap * Ss[k] for k in range(5)]
    qout = P["qs"] - lam * (Phis[5] - dn(Phis[5])) - (lam / 2.0) * Ps["p"] * (up(Ps["v"]) - dn(Ps["v"]))
    return dict(P=P, Phi=Phi, us=us, qst=qst, Ps=Ps, aR=aR, bR=bR, aL=aL, bL=bL, Phis=Phis, out=out, qout=qout)


def _order(d):
    return (0, 1 + d, 1 + (d + 1) % 3, 1 + (d + 2) % 3, 4)


def sweep(gas6, d, lam, kap, gamma, g=None, e_floor=1e-12, lim_eps=1e-20, eta=1e-3, dtype=np.float64):
    """SWEEP_d with dual energy on a (6, nz, ny, nx) state (rho, m_x, m_y, m_z, eps, q).  Returns (new state, c_max of the
    input: Eq. 19-20).  dtype: fp64 is the oracle; numpy.float32 runs the same statements in single precision (only to
    show what the formalism is for: the cancellation in e~_T, tests/test_oracle_dual_energy.py)."""
    gas6 = np.asarray(gas6, dtype=dtype)
    comp = _order(d)
    u = [gas6[k] for k in comp]
    R = _forward(u, gas6[5], None if g is None else np.asarray(g, dtype=dtype), lam, kap, gamma, e_floor, lim_eps, eta,
                 2 - d)
    out = np.empty_like(gas6)
    for k in range(5):
        out[comp[k]] = R["out"][k]
    out[5] = R["qout"]
    return out, float(np.max(R["P"]["c"]))


def sweep_vjp(gas6, d, lam, kap, gamma, cot_out, g=None, e_floor=1e-12, lim_eps=1e-20, eta=1e-3):
    """Transpose of `sweep` at gas6 applied to cot_out (6, nz, ny, nx).  Returns (cot_in (6,...), g_bar or None,
    dict(lam, kap, gamma)).  Statement by statement the reverse of _forward."""
    gas6 = np.asarray(gas6, dtype=np.float64); cot_out = np.asarray(cot_out, dtype=np.float64)
    ax = 2 - d
    up = lambda x: np.roll(x, -1, ax)
    dn = lambda x: np.roll(x, 1, ax)
    comp = _order(d)
    u = [gas6[k] for k in comp]
    q = gas6[5]
    gg = None if g is None else np.asarray(g, dtype=np.float64)
    g0 = 0.0 if gg is None else gg
    R = _forward(u, q, gg, lam, kap, gamma, e_floor, lim_eps, eta, ax)
    P, Ps, us, Phi, Phis = R["P"], R["Ps"], R["us"], R["Phi"], R["Phis"]
    ob = [cot_out[k] for k in comp]
    obq = cot_out[5]
    # ---- stage B update
    ub = [ob[k].copy() for k in range(5)]
    qsb = obq.copy()
    dvs = up(Ps["v"]) - dn(Ps["v"])
    lam_b = -sum(np.sum(ob[k] * (Phis[k] - dn(Phis[k]))) for k in range(5))
    lam_b += -np.sum(obq * (Phis[5] - dn(Phis[5]))) - 0.5 * np.sum(obq * Ps["p"] * dvs)
    Phisb = [-lam * (ob[k] - up(ob[k])) for k in range(5)] + [-lam * (obq - up(obq))]
    psb = -(lam / 2.0) * obq * dvs
    t = Ps["p"] * obq
    vsb = -(lam / 2.0) * (dn(t) - up(t))
    kap_b = np.sum(ob[1] * us[0] * g0 + ob[4] * us[1] * g0)
    usb = [np.zeros_like(q) for _ in range(5)]
    usb[0] = usb[0] + kap * g0 * ob[1]
    usb[1] = usb[1] + kap * g0 * ob[4]
    gb = None if gg is None else kap * (us[0] * ob[1] + us[1] * ob[4])
    # ---- limited fluxes
    FRsb, FLsb = [], []
    for k in range(6):
        daR, dbR = limiter_grad(R["aR"][k], R["bR"][k], lim_eps)
        daL, dbL = limiter_grad(R["aL"][k], R["bL"][k], lim_eps)
        PR = Phisb[k]
        PL = -Phisb[k]
        FRsb.append(PR * (1.0 + 0.5 * daR - 0.5 * dbR) + up(-0.5 * daR * PR) + dn(0.5 * dbR * PR))
        FLsb.append(0.5 * daL * PL + dn((1.0 - 0.5 * daL + 0.5 * dbL) * PL) + dn(dn(-0.5 * dbL * PL)))
    # (PhiR_n = FRs_n + phi(aR, bR):  d/dFRs_{n-1} = -daR/2,  d/dFRs_n = 1 + daR/2 - dbR/2,  d/dFRs_{n+1} = +dbR/2;
    #  PhiL_n = FLs_{n+1} - phi(aL, bL):  d/dFLs_n = +daL/2,  d/dFLs_{n+1} = 1 - daL/2 + dbL/2,  d/dFLs_{n+2} = -dbL/2)
    t5, qstb, gm1 = prim_vjp(us, R["qst"], gamma, e_floor, eta, Ps, FRsb, FLsb, vsb, psb, 0.0)
    for k in range(5):
        usb[k] = usb[k] + t5[k]
    # ---- stage A update
    for k in range(5):
        ub[k] = ub[k] + usb[k]
    qsb = qsb + qstb
    dv = up(P["v"]) - dn(P["v"])
    lam_b += -0.5 * sum(np.sum(usb[k] * (Phi[k] - dn(Phi[k]))) for k in range(5))
    lam_b += -0.5 * np.sum(qstb * (Phi[5] - dn(Phi[5]))) - 0.25 * np.sum(qstb * P["p"] * dv)
    Phib = [-(lam / 2.0) * (usb[k] - up(usb[k])) for k in range(5)] + [-(lam / 2.0) * (qstb - up(qstb))]
    pb = -(lam / 4.0) * qstb * dv
    t = P["p"] * qstb
    vb = -(lam / 4.0) * (dn(t) - up(t))
    kap_b += 0.5 * np.sum(usb[1] * u[0] * g0 + usb[4] * u[1] * g0)
    ub[0] = ub[0] + 0.5 * kap * g0 * usb[1]
    ub[1] = ub[1] + 0.5 * kap * g0 * usb[4]
    if gb is not None:
        gb = gb + 0.5 * kap * (u[0] * usb[1] + u[1] * usb[4])
    FRb = Phib                                                     # Phi_n = FR_n - FL_{n+1}
    FLb = [-dn(Phib[k]) for k in range(6)]
    t5, qb, gm2 = prim_vjp(u, q, gamma, e_floor, eta, P, FRb, FLb, vb, pb, qsb)
    for k in range(5):
        ub[k] = ub[k] + t5[k]
    cin = np.empty_like(gas6)
    for k in range(5):
        cin[comp[k]] = ub[k]
    cin[5] = qb
    return cin, gb, dict(lam=float(lam_b), kap=float(kap_b), gamma=gm1 + gm2)


# ------------------------------------------------------------------------------------ runs built on the sweep ----
def hydro_run(gas6, gamma, lams, e_floor=1e-12, lim_eps=1e-20, eta=1e-3, step0=0):
    """Static hydro-only run (no gravity): step n applies the three sweeps of STRANG[n mod 6] with lam = lams[n]."""
    gas6 = np.asarray(gas6, dtype=np.float64)
    cmax = []
    for n, lam in enumerate(lams):
        cm = []
        for d in STRANG[(step0 + n) % 6]:
            gas6, c = sweep(gas6, d, lam, 0.0, gamma, None, e_floor, lim_eps, eta)
            cm.append(c)
        cmax.append(cm)
    return gas6, np.array(cmax)


def hydro_run_vjp(gas6, gamma, lams, cot, e_floor=1e-12, lim_eps=1e-20, eta=1e-3, step0=0):
    """Reverse pass of hydro_run: (cotangent of the initial state, d gamma)."""
    states = []
    g6 = np.asarray(gas6, dtype=np.float64)
    for n, lam in enumerate(lams):
        for d in STRANG[(step0 + n) % 6]:
            states.append((g6, d, lam))
            g6, _ = sweep(g6, d, lam, 0.0, gamma, None, e_floor, lim_eps, eta)
    cot = np.asarray(cot, dtype=np.float64)
    dgamma = 0.0
    for g6, d, lam in reversed(states):
        cot, _, sc = sweep_vjp(g6, d, lam, 0.0, gamma, cot, None, e_floor, lim_eps, eta)
        dgamma += sc["gamma"]
    return cot, dgamma


def coupled_step(O, P, gas6, part, a_i, a_next, dt, dt_prev, step, eta=1e-3):
    """One coupled step S0-S5 with the dual-energy sweeps; deposit, Poisson solve and gather are the
    pinned routines of the C++ oracle O (oracle/oracle.py), the particle update is Eq. 2-3 written out.
    Returns (gas6', part', c_max[3])."""
    N = P.N
    sc = O.step_scalars(P, a_i, a_next, dt, dt_prev)
    dx = P.box / N
    gas6 = np.asarray(gas6, dtype=np.float64); part = np.asarray(part, dtype=np.float64)
    g = None
    if P.gravity_on:
        f_b = P.Omega_b / P.Omega_m
        npart = part.shape[1]
        m_p = (1.0 - f_b) * N ** 3 / npart if npart else 0.0
        rho_bar = (1.0 - f_b if npart else 0.0) + (f_b if P.gas_sources_gravity else 0.0)
        delta = (gas6[0] if P.gas_sources_gravity else 0.0) - rho_bar + (O.deposit(N, part[:3], m_p) if npart else 0.0)
        g = O.poisson(N, P.box, sc["A"], delta)
    part = part.copy()
    if part.shape[1]:
        if g is not None:
            for d in range(3):
                part[3 + d] += sc["K"] * O.gather(N, part[:3], g[d])          # Eq. 3
        part[:3] = np.mod(part[:3] + part[3:] * (sc["dtau"] / dx), N)         # Eq. 2
    cm = []
    if P.hydro_on:
        lam = sc["dtau"] / dx
        for d in STRANG[step % 6]:
            gas6, c = sweep(gas6, d, lam, sc["kappa"], P.gamma, None if g is None else g[d], P.e_floor, P.lim_eps, eta)
            cm.append(c)
    return gas6, part, cm


def _cic(pos, N):
    """Cloud-in-cell indices and weights (reading R13: s = x - 1/2, i0 = floor(s), f = s - i0), per axis."""
    s_ = pos - 0.5
    i0 = np.floor(s_).astype(np.int64)
    f = s_ - i0
    return i0 % N, (i0 + 1) % N, f


def _gather_grad(mesh, pos, N):
    """d/dx_p of the CIC interpolation of `mesh` at the particles: (3, n_p); the weights' derivatives are -1 | +1."""
    (i0, i1, f) = _cic(pos, N)
    out = np.zeros((3, pos.shape[1]))
    for dz in (0, 1):
        for dy in (0, 1):
            for dx in (0, 1):
                ix = i1[0] if dx else i0[0]; iy = i1[1] if dy else i0[1]; iz = i1[2] if dz else i0[2]
                wx = f[0] if dx else 1 - f[0]; wy = f[1] if dy else 1 - f[1]; wz = f[2] if dz else 1 - f[2]
                v = mesh[iz, iy, ix]
                out[0] += (1.0 if dx else -1.0) * wy * wz * v
                out[1] += (1.0 if dy else -1.0) * wx * wz * v
                out[2] += (1.0 if dz else -1.0) * wx * wy * v
    return out


def coupled_step_vjp(O, P, gas6, part, a_i, a_next, dt, dt_prev, step, cot_gas6, cot_part, eta=1e-3):
    """Transpose of coupled_step at (gas6, part): returns (cot_gas6_in, cot_part_in, d gamma).  Reverse of S4 (the sweeps,
    last first, each handing back the cotangent of g'_d), S3 (w_t_b = w'_b + (dtau/dx) x'_b; x_b = x'_b + K sum_d w_t_b,d
    dg_p,d/dx; g'_b += K W w_t_b), S2 (delta_b = sum_d G_d^T g'_b,d) and S1 (rho_b += delta_b; x_b += m_p sum delta_b dW/dx)."""
    N = P.N
    sc = O.step_scalars(P, a_i, a_next, dt, dt_prev)
    dx = P.box / N
    gas6 = np.asarray(gas6, dtype=np.float64); part = np.asarray(part, dtype=np.float64)
    npart = part.shape[1]
    f_b = P.Omega_b / P.Omega_m
    m_p = (1.0 - f_b) * N ** 3 / npart if npart else 0.0
    g = None
    if P.gravity_on:
        rho_bar = (1.0 - f_b if npart else 0.0) + (f_b if P.gas_sources_gravity else 0.0)
        delta = (gas6[0] if P.gas_sources_gravity else 0.0) - rho_bar + (O.deposit(N, part[:3], m_p) if npart else 0.0)
        g = O.poisson(N, P.box, sc["A"], delta)
    # forward sweeps, keeping every sweep's input
    lam = sc["dtau"] / dx
    ins, cur = [], gas6
    for d in STRANG[step % 6]:
        ins.append((cur, d))
        cur, _ = sweep(cur, d, lam, sc["kappa"], P.gamma, None if g is None else g[d], P.e_floor, P.lim_eps, eta)
    cot = np.asarray(cot_gas6, dtype=np.float64)
    gb = np.zeros((3, N, N, N))
    dgamma = 0.0
    for u_in, d in reversed(ins):
        cot, gbd, scb = sweep_vjp(u_in, d, lam, sc["kappa"], P.gamma, cot, None if g is None else g[d], P.e_floor, P.lim_eps, eta)
        dgamma += scb["gamma"]
        if gbd is not None:
            gb[d] += gbd
    cp = np.asarray(cot_part, dtype=np.float64).copy()
    if npart:
        wt = cp[3:] + (sc["dtau"] / dx) * cp[:3]
        xb = cp[:3].copy()
        if g is not None:
            for d in range(3):
                xb += sc["K"] * wt[d] * _gather_grad(g[d], part[:3], N)
                # vector deposit of K w_t_b with the gather's own weights (adjoint pair of gather / deposit)
                i0, i1, f = _cic(part[:3], N)
                for dz in (0, 1):
                    for dy in (0, 1):
                        for dxx in (0, 1):
                            ix = i1[0] if dxx else i0[0]; iy = i1[1] if dy else i0[1]; iz = i1[2] if dz else i0[2]
                            w_ = (f[0] if dxx else 1 - f[0]) * (f[1] if dy else 1 - f[1]) * (f[2] if dz else 1 - f[2])
                            gb[d] += np.bincount((iz * N + iy) * N + ix, weights=sc["K"] * wt[d] * w_,
                                                 minlength=N ** 3).reshape(N, N, N)
        cp = np.concatenate([xb, wt])
    if g is not None:
        db = O.poisson_vjp(N, P.box, sc["A"], gb)
        if P.gas_sources_gravity:
            cot = cot.copy(); cot[0] += db
        if npart:
            cp[:3] += m_p * _gather_grad(db, part[:3], N)
    return cot, cp, dgamma


def coupled_run(O, P, gas6, part, a0, a_sched, dt_sched, eta=1e-3, step0=0):
    a, dtp = a0, 0.0
    cmax = []
    for k in range(len(dt_sched)):
        gas6, part, cm = coupled_step(O, P, gas6, part, a, a_sched[k], dt_sched[k], dtp, step0 + k, eta)
        a = 1.0 if P.static_mode else a_sched[k]
        dtp = dt_sched[k]
        cmax.append(cm)
    return gas6, part, np.array(cmax)


def coupled_run_vjp(O, P, gas6, part, a0, a_sched, dt_sched, cot_gas6, cot_part, eta=1e-3, step0=0):
    """Reverse pass of coupled_run: every step's input is kept, then coupled_step_vjp last step first.
    Returns (cot_gas6 of the initial state, cot_part, d gamma)."""
    states, a, dtp = [], a0, 0.0
    g6 = np.asarray(gas6, dtype=np.float64); p = np.asarray(part, dtype=np.float64)
    for k in range(len(dt_sched)):
        states.append((g6, p, a, dtp))
        g6, p, _ = coupled_step(O, P, g6, p, a, a_sched[k], dt_sched[k], dtp, step0 + k, eta)
        a = 1.0 if P.static_mode else a_sched[k]
        dtp = dt_sched[k]
    cg = np.asarray(cot_gas6, dtype=np.float64); cp = np.asarray(cot_part, dtype=np.float64)
    dgamma = 0.0
    for k in reversed(range(len(dt_sched))):
        g6, p, a, dtp = states[k]
        cg, cp, dg = coupled_step_vjp(O, P, g6, p, a, a_sched[k], dt_sched[k], dtp, step0 + k, cg, cp, eta)
        dgamma += dg
    return cg, cp, dgamma


def thermal_energy(gas6, eta=1e-3):
    """The selected thermal energy per unit mass e~ of a state (R34) -- what a temperature diagnostic uses."""
    gas6 = np.asarray(gas6, dtype=np.float64)
    rho, eps = gas6[0], gas6[4]
    eT = eps / rho - np.sum(gas6[1:4] ** 2, axis=0) / (2.0 * rho * rho)
    return np.where(eT > eta * eps / rho, eT, gas6[5] / rho)
