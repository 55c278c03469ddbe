"""Host-side checks of the C-ABI library that need no GPU: it loads, exports every symbol include/diffhydro.h
declares, refuses to initialise without a device (no CPU fallback), and its host helpers agree with the oracle's."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
LIB = os.path.join(ROOT, "paper_2502_02294_b200", "libdiffhydro.so")


@pytest.fixture(scope="module")
def lib():
    if not os.path.exists(LIB):
        from paper_2502_02294_b200 import build
        build.build()
    return C.CDLL(LIB)


def test_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "diffhydro.h")).read()
    names = sorted(set(re.findall(r"\b(dh_[a-z_0-9]+)\s*\(", hdr)))
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), n
    from importlib import util
    spec = util.find_spec("paper_2502_02294_b200.api")
    src = open(spec.origin).read()
    listed = re.search(r"EXPORTS = \[(.*?)\]", src, re.S).group(1)
    assert sorted(re.findall(r'"(dh_[a-z_0-9]+)"', listed)) == names


class Cosmo(C.Structure):
    _fields_ = [("H0", C.c_double), ("Omega_m", C.c_double), ("Omega_b", C.c_double), ("Omega_L", C.c_double),
                ("static_mode", C.c_int32)]


class Opt(C.Structure):
    _fields_ = [("n_part_side", C.c_int32), ("gravity_on", C.c_int32), ("hydro_on", C.c_int32),
                ("gas_sources_gravity", C.c_int32), ("e_floor", C.c_double), ("lim_eps", C.c_double),
                ("cuda_stream", C.c_void_p), ("want_dA", C.c_int32), ("want_dsched", C.c_int32),
                ("dual_energy", C.c_int32), ("dual_eta", C.c_double)]


def test_init_rejects_bad_arguments_and_missing_device(lib):
    import torch
    lib.dh_last_error.restype = C.c_char_p
    h = C.c_void_p()
    co = Cosmo(100.0, 1.0, 0.16, 0.0, 0)
    op = Opt(32, 1, 1, 1, 1e-6, 1e-20, None, 1, 1, 0, 0.0)
    assert lib.dh_init(C.byref(h), 30, C.c_double(10.0), C.c_double(1.4), C.byref(co), C.byref(op)) == -1   # DH_ERR_INVALID
    assert b"multiple of 32" in lib.dh_last_error()
    bad = Opt(32, 1, 1, 1, 1e-6, 1e-20, None, 1, 1, 1, -1.0)
    assert lib.dh_init(C.byref(h), 32, C.c_double(10.0), C.c_double(1.4), C.byref(co), C.byref(bad)) == -1
    assert b"dual_eta" in lib.dh_last_error()
    assert lib.dh_init(C.byref(h), 32, C.c_double(10.0), C.c_double(1.0), C.byref(co), C.byref(op)) == -1
    if not torch.cuda.is_available():
        rc = lib.dh_init(C.byref(h), 32, C.c_double(10.0), C.c_double(1.4), C.byref(co), C.byref(op))
        assert rc == -2 and h.value is None                                                               # DH_ERR_NO_DEVICE
        assert b"no CPU fallback" in lib.dh_last_error()


def test_host_helpers_match_oracle(lib, O):
    dp = C.POINTER(C.c_double)
    for (Om, OL) in ((1.0, 0.0), (0.3, 0.7)):
        co = Cosmo(100.0, Om, 0.048, OL, 0)
        n = 7
        a = np.zeros(n + 1); dt = np.zeros(n)
        assert lib.dh_schedule_lna(C.byref(co), C.c_double(0.01), C.c_double(0.2), n, a.ctypes.data_as(dp), dt.ctypes.data_as(dp)) == 0
        P = O.make_params(32, 10.0, 1.4, Omega_m=Om, Omega_L=OL, Omega_b=0.048)
        a2, dt2 = O.schedule_lna(P, 0.01, 0.2, n)
        assert np.max(np.abs(a - a2)) < 1e-15 and np.max(np.abs(dt / dt2 - 1)) < 1e-9
        out = np.zeros(4)
        assert lib.dh_step_scalars(C.byref(co), C.c_double(0.02), C.c_double(0.03), C.c_double(dt[0]), C.c_double(0.5 * dt[0]),
                                   out.ctypes.data_as(dp)) == 0
        sc = O.step_scalars(P, 0.02, 0.03, dt[0], 0.5 * dt[0])
        assert np.allclose(out, [sc["dtau"], sc["kappa"], sc["K"], sc["A"]], rtol=1e-15)
    co = Cosmo(100.0, 1.0, 0.16, 0.0, 1)
    out = np.zeros(4)
    lib.dh_step_scalars(C.byref(co), C.c_double(1.0), C.c_double(1.0), C.c_double(0.3), C.c_double(0.1), out.ctypes.data_as(dp))
    assert out[0] == 0.3 and out[1] == 0.3 and abs(out[2] - 0.2) < 1e-16


def test_package_imports_without_cuda_and_has_no_fallback():
    import paper_2502_02294_b200 as pkg
    assert hasattr(pkg, "workloads")
    import torch
    if not torch.cuda.is_available():
        from paper_2502_02294_b200 import api
        with pytest.raises(RuntimeError, match="no CPU fallback"):
            api.Context(32, 10.0, 1.4)


def test_ic_factors_against_textbook_values(lib, IC):
    """dh_ic_factors (the library's own statement of readings R18, R19, R27) and the oracle's (oracle/ic.py), each against
    numbers neither computes: e(10^4 K) = 209.9 (km/s)^2 for gamma = 5/3, mu = 0.59, the sound speed of
    ionised gas at 10^4 K (15.3 km/s), a^2 H f = H0 sqrt(a) in Einstein-de Sitter, and the growth rate of flat LambdaCDM,
    f = dlnD/dlna from the growth ODE integrated in the test (and Omega_m(a)^0.55 to 1 %, Linder's fit), f -> 1 early."""
    dp = C.POINTER(C.c_double)
    vf, e0 = C.c_double(0), C.c_double(0)
    eds = Cosmo(100.0, 1.0, 0.16, 0.0, 0)
    assert lib.dh_ic_factors(C.byref(eds), C.c_double(1.0), C.c_double(1e4), C.c_double(5.0 / 3.0), C.c_double(0.59),
                             C.byref(vf), C.byref(e0)) == 0
    for e in (e0.value, IC.thermal_energy_tilde(1.0, 1e4, 5.0 / 3.0)):
        assert abs(e - 209.9) < 0.05
        assert abs(np.sqrt(5.0 / 3.0 * 2.0 / 3.0 * e) - 15.3) < 0.05
    assert abs(e0.value / IC.thermal_energy_tilde(1.0, 1e4, 5.0 / 3.0) - 1) < 1e-14
    for a in (0.01, 0.1, 0.5):
        lib.dh_ic_factors(C.byref(eds), C.c_double(a), C.c_double(1e4), C.c_double(1.4), C.c_double(0.59), C.byref(vf), C.byref(e0))
        assert abs(vf.value / (100.0 * np.sqrt(a)) - 1) < 1e-12
        assert abs(IC.velocity_factor_eds(100.0, a) / (100.0 * np.sqrt(a)) - 1) < 1e-15
        assert abs(e0.value / (a * a * IC.thermal_energy_tilde(1.0, 1e4, 1.4)) - 1) < 1e-14       # e~ = a^2 e
    # flat LambdaCDM: the growth equation D'' + (2 + dlnH/dlna) D' = 1.5 Omega_m(a) D in x = ln a, integrated here
    from scipy.integrate import solve_ivp
    Om, OL = 0.31, 0.69

    def rhs(x, y):
        a = np.exp(x)
        E2 = Om / a ** 3 + OL
        return [y[1], -(2.0 - 1.5 * Om / a ** 3 / E2) * y[1] + 1.5 * Om / a ** 3 / E2 * y[0]]
    sol = solve_ivp(rhs, [np.log(1e-4), 0.0], [1e-4, 1e-4], rtol=1e-10, atol=1e-14, dense_output=True)
    lcdm = Cosmo(70.0, Om, 0.049, OL, 0)
    for a in (0.01, 0.3, 0.5, 1.0):
        lib.dh_ic_factors(C.byref(lcdm), C.c_double(a), C.c_double(0.0), C.c_double(1.4), C.c_double(0.59), C.byref(vf), None)
        E = np.sqrt(Om / a ** 3 + OL)
        f = vf.value / (a * a * 70.0 * E)
        D, dD = sol.sol(np.log(a))
        assert abs(f / (dD / D) - 1) < 1e-6, (a, f, dD / D)
        assert abs(f / (Om / a ** 3 / E ** 2) ** 0.55 - 1) < 1e-2, (a, f)
        if a == 0.01:
            assert abs(f - 1) < 1e-5
    assert lib.dh_ic_factors(C.byref(eds), C.c_double(-1.0), C.c_double(1e4), C.c_double(1.4), C.c_double(0.59), C.byref(vf), None) == -1
