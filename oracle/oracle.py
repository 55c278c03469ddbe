"""ctypes front end of the CPU oracle (oracle/dh_oracle.cpp).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It never imports the CUDA package.
All arrays are host numpy float64, C-order [z][y][x]; gas has shape (5, nz, ny, nx) with fields
(rho, m_x, m_y, m_z, eps); particles have shape (6, n_p) = (x, y, z, w_x, w_y, w_z), positions in grid
units [0, N).  See the header of dh_oracle.cpp for citations, readings and pins.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dh_oracle.cpp")
_LIB = os.path.join(_HERE, "libdh_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (-O2 -fopenmp).  Returns the path of the shared library."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off", _SRC, "-o", _LIB]
        subprocess.run(cmd, check=True)
    return _LIB


class Params(C.Structure):
    _fields_ = [
        ("N", C.c_int32), ("n_part_side", C.c_int32),
        ("box", C.c_double), ("gamma", C.c_double),
        ("H0", C.c_double), ("Omega_m", C.c_double), ("Omega_b", C.c_double), ("Omega_L", C.c_double),
        ("static_mode", C.c_int32), ("gravity_on", C.c_int32), ("hydro_on", C.c_int32),
        ("gas_sources_gravity", C.c_int32),
        ("e_floor", C.c_double), ("lim_eps", C.c_double),
    ]


def make_params(N, box, gamma, n_part_side=None, H0=100.0, Omega_m=1.0, Omega_b=0.16, Omega_L=0.0,
                static_mode=0, gravity_on=1, hydro_on=1, gas_sources_gravity=1, e_floor=1e-12,
                lim_eps=1e-20) -> Params:
    if n_part_side is None:
        n_part_side = N
    return Params(int(N), int(n_part_side), float(box), float(gamma), float(H0), float(Omega_m), float(Omega_b),
                  float(Omega_L), int(static_mode), int(gravity_on), int(hydro_on), int(gas_sources_gravity),
                  float(e_floor), float(lim_eps))


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_limiter.restype = C.c_double
        _lib.orc_limiter.argtypes = [C.c_double] * 3
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _p(a):
    if a is None:
        return None
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def limiter(a, b, eps=1e-20) -> float:
    return float(lib().orc_limiter(float(a), float(b), float(eps)))


def strang_order(step: int):
    out = (C.c_int32 * 3)()
    lib().orc_strang_order(C.c_int64(step), out)
    return tuple(out)


def step_scalars(P: Params, a_i, a_next, dt, dt_prev):
    out = (C.c_double * 4)()
    lib().orc_step_scalars(C.byref(P), C.c_double(a_i), C.c_double(a_next), C.c_double(dt), C.c_double(dt_prev), out)
    return dict(dtau=out[0], kappa=out[1], K=out[2], A=out[3])


def schedule_lna(P: Params, a0, a1, n):
    a = np.zeros(n + 1)
    dt = np.zeros(n)
    lib().orc_schedule_lna(C.byref(P), C.c_double(a0), C.c_double(a1), C.c_int(n), _p(a), _p(dt))
    return a, dt


def cell_index(x32: np.ndarray, N: int):
    x32 = np.ascontiguousarray(x32, dtype=np.float32).ravel()
    i0 = np.zeros(x32.size, dtype=np.int32)
    i1 = np.zeros(x32.size, dtype=np.int32)
    lib().orc_cell_index(x32.ctypes.data_as(C.POINTER(C.c_float)), C.c_long(x32.size), C.c_int(N),
                         i0.ctypes.data_as(C.POINTER(C.c_int32)), i1.ctypes.data_as(C.POINTER(C.c_int32)))
    return i0, i1


def fft3(a: np.ndarray, sign: int = -1) -> np.ndarray:
    N = a.shape[0]
    re = _f64(a.real)
    im = _f64(a.imag) if np.iscomplexobj(a) else None
    ro = np.zeros((N, N, N))
    io = np.zeros((N, N, N))
    lib().orc_fft3(C.c_int(N), _p(re), _p(im), C.c_int(sign), _p(ro), _p(io))
    return ro + 1j * io


def _dims(gas):
    assert gas.ndim == 4 and gas.shape[0] == 5
    nz, ny, nx = gas.shape[1:]
    return nx, ny, nz


def sweep(gas, d, lam, kap, gamma, g=None, e_floor=1e-12, lim_eps=1e-20):
    """SWEEP_d on a (5, nz, ny, nx) state.  Returns (new state, c_max of the input)."""
    gas = _f64(gas); g = _f64(g)
    nx, ny, nz = _dims(gas)
    out = np.zeros_like(gas)
    cm = C.c_double(0)
    lib().orc_sweep(nx, ny, nz, int(d), _p(gas), _p(g), C.c_double(lam), C.c_double(kap), C.c_double(gamma),
                    C.c_double(e_floor), C.c_double(lim_eps), _p(out), C.byref(cm))
    return out, cm.value


def sweep_jvp(gas, d, lam, kap, gamma, g=None, dgas=None, dg=None, dlam=0.0, dkap=0.0, dgamma=0.0,
              e_floor=1e-12, lim_eps=1e-20):
    gas = _f64(gas); g = _f64(g); dgas = _f64(dgas); dg = _f64(dg)
    nx, ny, nz = _dims(gas)
    out = np.zeros_like(gas); dout = np.zeros_like(gas)
    lib().orc_sweep_jvp(nx, ny, nz, int(d), _p(gas), _p(g), C.c_double(lam), C.c_double(kap), C.c_double(gamma),
                        C.c_double(e_floor), C.c_double(lim_eps), _p(dgas), _p(dg), C.c_double(dlam),
                        C.c_double(dkap), C.c_double(dgamma), _p(out), _p(dout))
    return out, dout


def sweep_vjp(gas, d, lam, kap, gamma, cot_out, g=None, e_floor=1e-12, lim_eps=1e-20):
    """Returns (cot_in (5,...), g_bar (or None), dict(lam, kap, gamma))."""
    gas = _f64(gas); g = _f64(g); cot_out = _f64(cot_out)
    nx, ny, nz = _dims(gas)
    cin = np.zeros_like(gas)
    gb = np.zeros_like(g) if g is not None else None
    sc = (C.c_double * 3)(0, 0, 0)
    lib().orc_sweep_vjp(nx, ny, nz, int(d), _p(gas), _p(g), C.c_double(lam), C.c_double(kap), C.c_double(gamma),
                        C.c_double(e_floor), C.c_double(lim_eps), _p(cot_out), _p(cin), _p(gb), sc)
    return cin, gb, dict(lam=sc[0], kap=sc[1], gamma=sc[2])


def deposit(N, pos, mp, mesh=None):
    pos = _f64(pos)
    mesh = np.zeros((N, N, N)) if mesh is None else _f64(mesh).copy()
    lib().orc_deposit(C.c_int(N), C.c_long(pos.shape[1]), _p(pos), C.c_double(mp), _p(mesh))
    return mesh


def gather(N, pos, mesh):
    pos = _f64(pos); mesh = _f64(mesh)
    out = np.zeros(pos.shape[1])
    lib().orc_gather(C.c_int(N), C.c_long(pos.shape[1]), _p(pos), _p(mesh), _p(out))
    return out


def poisson(N, L, A, delta):
    delta = _f64(delta)
    g = np.zeros((3, N, N, N))
    lib().orc_poisson(C.c_int(N), C.c_double(L), C.c_double(A), _p(delta), _p(g))
    return g


def poisson_vjp(N, L, A, gb):
    gb = _f64(gb)
    db = np.zeros((N, N, N))
    lib().orc_poisson_vjp(C.c_int(N), C.c_double(L), C.c_double(A), _p(gb), _p(db))
    return db


class State:
    """Mutable oracle state: gas (5,N,N,N) f64, part (6,n_p) f64, scalars a, dt_prev, step."""

    def __init__(self, gas, part, a, dt_prev=0.0, step=0):
        self.gas = np.array(gas, dtype=np.float64, order="C")
        self.part = np.array(part, dtype=np.float64, order="C").reshape(6, -1)
        self.a = float(a)
        self.dt_prev = float(dt_prev)
        self.step = int(step)

    def copy(self):
        return State(self.gas.copy(), self.part.copy(), self.a, self.dt_prev, self.step)


def step(P: Params, s: State, dt, a_next, want_gprime=False):
    """One coupled step in place.  Returns (cmax[3], g' or None)."""
    cm = np.zeros(3)
    gp = np.zeros((3, P.N, P.N, P.N)) if want_gprime else None
    a = C.c_double(s.a); dtp = C.c_double(s.dt_prev); st = C.c_int64(s.step)
    lib().orc_step(C.byref(P), _p(s.gas), _p(s.part), C.byref(a), C.byref(dtp), C.byref(st), C.c_double(dt),
                   C.c_double(a_next), _p(cm), _p(gp))
    s.a, s.dt_prev, s.step = a.value, dtp.value, st.value
    return cm, gp


def step_explicit(P: Params, gas, part, sc, gamma, step_idx):
    gas = np.array(gas, dtype=np.float64, order="C"); part = np.array(part, dtype=np.float64, order="C")
    lib().orc_step_explicit(C.byref(P), _p(gas), _p(part), C.c_double(sc["dtau"]), C.c_double(sc["kappa"]),
                            C.c_double(sc["K"]), C.c_double(sc["A"]), C.c_double(gamma), C.c_int64(step_idx))
    return gas, part


def step_jvp(P: Params, gas, part, sc, gamma, step_idx, dgas=None, dpart=None, dscal=None):
    """dscal = tangents of (gamma, dtau, kappa, K, A).  Returns (gas', part', dgas', dpart')."""
    gas = _f64(gas); part = _f64(part); dgas = _f64(dgas); dpart = _f64(dpart)
    ds = np.zeros(5) if dscal is None else _f64(dscal)
    go = np.zeros_like(gas); po = np.zeros_like(part); dgo = np.zeros_like(gas); dpo = np.zeros_like(part)
    lib().orc_step_jvp(C.byref(P), _p(gas), _p(part), C.c_double(sc["dtau"]), C.c_double(sc["kappa"]),
                       C.c_double(sc["K"]), C.c_double(sc["A"]), C.c_double(gamma), C.c_int64(step_idx),
                       _p(dgas), _p(dpart), _p(ds), _p(go), _p(po), _p(dgo), _p(dpo))
    return go, po, dgo, dpo


def step_vjp_explicit(P: Params, gas_in, part_in, sc, gamma, step_idx, cot_gas, cot_part):
    """Returns (cot_gas_in, cot_part_in, dpar[5] = d(gamma, dtau, kappa, K, A))."""
    gas_in = _f64(gas_in); part_in = _f64(part_in)
    cg = np.array(cot_gas, dtype=np.float64, order="C"); cp = np.array(cot_part, dtype=np.float64, order="C")
    dpar = np.zeros(5)
    lib().orc_step_vjp_explicit(C.byref(P), _p(gas_in), _p(part_in), C.c_double(sc["dtau"]), C.c_double(sc["kappa"]),
                                C.c_double(sc["K"]), C.c_double(sc["A"]), C.c_double(gamma), C.c_int64(step_idx),
                                _p(cg), _p(cp), _p(dpar))
    return cg, cp, dpar


def step_vjp(P: Params, s_in: State, dt, a_next, cot_gas, cot_part):
    cg = np.array(cot_gas, dtype=np.float64, order="C"); cp = np.array(cot_part, dtype=np.float64, order="C")
    dpar = np.zeros(5)
    lib().orc_step_vjp(C.byref(P), _p(s_in.gas), _p(s_in.part), C.c_double(s_in.a), C.c_double(s_in.dt_prev),
                       C.c_int64(s_in.step), C.c_double(dt), C.c_double(a_next), _p(cg), _p(cp), _p(dpar))
    return cg, cp, dpar


def run(P: Params, gas, part, a0, a_sched, dt_sched, step0=0, want_states=False):
    """n steps from (gas, part) (copied).  a_sched[k] = a at the END of step k.
    Returns (gas, part, cmax (n,3), states or None)."""
    gas = np.array(gas, dtype=np.float64, order="C"); part = np.array(part, dtype=np.float64, order="C")
    a_sched = _f64(a_sched); dt_sched = _f64(dt_sched)
    n = len(dt_sched)
    cm = np.zeros((n, 3))
    states = np.zeros((n, gas.size + part.size)) if want_states else None
    lib().orc_run(C.byref(P), _p(gas), _p(part), C.c_double(a0), C.c_int64(step0), _p(a_sched), _p(dt_sched),
                  C.c_int(n), _p(cm), _p(states))
    return gas, part, cm, states


def run_vjp(P: Params, gas0, part0, a0, a_sched, dt_sched, cot_gas, cot_part, step0=0):
    """Returns (cot_gas0, cot_part0, dpar[5])."""
    gas0 = _f64(gas0); part0 = _f64(part0); a_sched = _f64(a_sched); dt_sched = _f64(dt_sched)
    cg = np.array(cot_gas, dtype=np.float64, order="C"); cp = np.array(cot_part, dtype=np.float64, order="C")
    dpar = np.zeros(5)
    lib().orc_run_vjp(C.byref(P), _p(gas0), _p(part0), C.c_double(a0), C.c_int64(step0), _p(a_sched), _p(dt_sched),
                      C.c_int(len(dt_sched)), _p(cg), _p(cp), _p(dpar))
    return cg, cp, dpar
