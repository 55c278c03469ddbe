"""Thin ctypes binding over libdiffhydro.so (include/diffhydro.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; torch is used here for device memory and streams only.
Importing this module fails loudly when the library is missing -- there is no CPU fallback.
Names follow the C ABI: dh_init, dh_step, dh_step_vjp, dh_run, dh_run_vjp, ...
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIBPATH = os.path.join(_HERE, "libdiffhydro.so")

if not os.path.exists(_LIBPATH):
    raise ImportError(f"{_LIBPATH} is missing: build it with `python -m paper_2502_02294_b200.build` "
                      "(nvcc, sm_100a).  This package has no CPU fallback.")
_lib = C.CDLL(_LIBPATH)

DH_OK = 0
ERRORS = {-1: "DH_ERR_INVALID", -2: "DH_ERR_NO_DEVICE", -3: "DH_ERR_CUDA", -4: "DH_ERR_CUFFT", -5: "DH_ERR_NONFINITE",
          -6: "DH_ERR_OOM", -7: "DH_ERR_STATE"}

EXPORTS = ["dh_init", "dh_free", "dh_step", "dh_step_vjp", "dh_run", "dh_run_vjp", "dh_run_host", "dh_run_vjp_host",
           "dh_last_error", "dh_get_cmax", "dh_schedule_lna", "dh_step_scalars", "dh_debug_cell_index",
           "dh_device_bytes", "dh_launch_count", "dh_sync", "dh_sweep", "dh_sweep_vjp", "dh_deposit", "dh_poisson",
           "dh_poisson_vjp", "dh_kick_drift", "dh_profile_enable", "dh_profile_categories", "dh_profile_name",
           "dh_profile_read", "dh_reserve", "dh_tune", "dh_ic_zeldovich", "dh_ic_zeldovich_vjp", "dh_data_term", "dh_power_spectrum",
           "dh_power_spectrum_vjp", "dh_subgrid_step", "dh_subgrid_step_vjp", "dh_get_step_dparams",
           "dh_chain_cosmology", "dh_value_and_grad_host", "dh_ic_factors", "dh_sweep_de", "dh_sweep_de_vjp", "dh_debug_poison", "dh_conserved_sums",
           "dh_conserved_sums_noalloc"]


class DhError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = _lib.dh_last_error().decode(errors="replace")
        super().__init__(f"{where}: {ERRORS.get(code, code)}: {msg}")


class dh_cosmology(C.Structure):
    _fields_ = [("H0", C.c_double), ("Omega_m", C.c_double), ("Omega_b", C.c_double), ("Omega_L", C.c_double),
                ("static_mode", C.c_int32)]


class dh_options(C.Structure):
    _fields_ = [("n_part_side", C.c_int32), ("gravity_on", C.c_int32), ("hydro_on", C.c_int32),
                ("gas_sources_gravity", C.c_int32), ("e_floor", C.c_double), ("lim_eps", C.c_double),
                ("cuda_stream", C.c_void_p), ("want_dA", C.c_int32), ("want_dsched", C.c_int32),
                ("dual_energy", C.c_int32), ("dual_eta", C.c_double)]


class dh_state(C.Structure):
    _fields_ = [("gas", C.c_void_p * 5), ("part", C.c_void_p * 6), ("a", C.c_double), ("dt_prev", C.c_double),
                ("step", C.c_int64), ("eint", C.c_void_p)]


class dh_cot(C.Structure):
    _fields_ = [("gas", C.c_void_p * 5), ("part", C.c_void_p * 6), ("eint", C.c_void_p)]


class dh_subgrid_params(C.Structure):
    _fields_ = [("rho_mean", C.c_double), ("t_per_e", C.c_double), ("T_c", C.c_double), ("delta_c", C.c_double),
                ("Pi0", C.c_double), ("e_inject", C.c_double), ("a_width", C.c_double), ("b_width", C.c_double),
                ("tau", C.c_double)]


class dh_dparams(C.Structure):
    _fields_ = [("dgamma", C.c_double), ("dDtau", C.c_double), ("dkappa", C.c_double), ("dK", C.c_double),
                ("dA", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib.dh_last_error.restype = C.c_char_p
_lib.dh_device_bytes.restype = C.c_int64
_lib.dh_launch_count.restype = C.c_int64
_lib.dh_profile_name.restype = C.c_char_p
_lib.dh_profile_name.argtypes = [C.c_int]
_lib.dh_profile_enable.argtypes = [C.c_void_p, C.c_int]
_lib.dh_profile_read.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
_lib.dh_device_bytes.argtypes = [C.c_void_p]
_lib.dh_launch_count.argtypes = [C.c_void_p]
_dp = C.POINTER(C.c_double)
_lib.dh_init.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_double, C.c_double, C.POINTER(dh_cosmology),
                         C.POINTER(dh_options)]
_lib.dh_free.argtypes = [C.c_void_p]
_lib.dh_sync.argtypes = [C.c_void_p]
_lib.dh_debug_poison.argtypes = [C.c_void_p, C.c_int]
_lib.dh_conserved_sums.argtypes = [C.c_void_p, C.POINTER(dh_state), _dp]
_lib.dh_conserved_sums_noalloc.argtypes = [C.POINTER(C.c_void_p), C.c_int64, C.POINTER(C.c_void_p), C.c_int64, C.c_double,
                                          C.c_void_p, C.c_void_p]
_lib.dh_step.argtypes = [C.c_void_p, C.POINTER(dh_state), C.c_double, C.c_double, C.c_void_p]
_lib.dh_step_vjp.argtypes = [C.c_void_p, C.POINTER(dh_state), C.c_double, C.c_double, C.POINTER(dh_cot),
                             C.POINTER(dh_cot), C.POINTER(dh_dparams)]
_lib.dh_run.argtypes = [C.c_void_p, C.POINTER(dh_state), _dp, _dp, C.c_int, C.c_int]
_lib.dh_run_vjp.argtypes = [C.c_void_p, C.POINTER(dh_cot), C.POINTER(dh_cot), C.POINTER(dh_dparams)]
_lib.dh_run_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, _dp, _dp, C.POINTER(C.c_int64), _dp, _dp, C.c_int,
                             C.c_int]
_lib.dh_run_vjp_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(dh_dparams)]
_lib.dh_reserve.argtypes = [C.c_void_p, C.c_int, C.c_int]
_lib.dh_tune.argtypes = [C.c_void_p, C.c_char_p, C.c_int]
_lib.dh_get_cmax.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
_lib.dh_schedule_lna.argtypes = [C.POINTER(dh_cosmology), C.c_double, C.c_double, C.c_int, _dp, _dp]
_lib.dh_step_scalars.argtypes = [C.POINTER(dh_cosmology), C.c_double, C.c_double, C.c_double, C.c_double, _dp]
_lib.dh_debug_cell_index.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
_P5 = C.c_void_p * 5
_P3 = C.c_void_p * 3
_P6 = C.c_void_p * 6
_lib.dh_sweep.argtypes = [C.c_void_p, C.c_int, _P5, C.c_void_p, C.c_double, C.c_double, _P5, C.c_void_p]
_lib.dh_sweep_vjp.argtypes = [C.c_void_p, C.c_int, _P5, C.c_void_p, C.c_double, C.c_double, _P5, _P5, C.c_void_p,
                              C.c_void_p]
_lib.dh_sweep_de.argtypes = [C.c_void_p, C.c_int, _P6, C.c_void_p, C.c_double, C.c_double, _P6, C.c_void_p]
_lib.dh_sweep_de_vjp.argtypes = [C.c_void_p, C.c_int, _P6, C.c_void_p, C.c_double, C.c_double, _P6, _P6, C.c_void_p,
                                 C.c_void_p]
_lib.dh_deposit.argtypes = [C.c_void_p, C.c_void_p, _P3, C.c_void_p]
_lib.dh_poisson.argtypes = [C.c_void_p, C.c_void_p, C.c_double, _P3]
_lib.dh_poisson_vjp.argtypes = [C.c_void_p, _P3, C.c_double, C.c_void_p]
_lib.dh_kick_drift.argtypes = [C.c_void_p, _P3, _P6, C.c_double, C.c_double]
_lib.dh_ic_zeldovich.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_double, C.POINTER(dh_state)]
_lib.dh_data_term.argtypes = [C.c_void_p, C.c_int, _P5, C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_void_p, _dp]
_lib.dh_subgrid_step.argtypes = [C.c_void_p, _P5, C.c_void_p, C.c_void_p, C.POINTER(dh_subgrid_params), C.c_void_p,
                                 C.c_void_p, C.c_void_p]
_lib.dh_subgrid_step_vjp.argtypes = [C.c_void_p, _P5, C.c_void_p, C.c_void_p, C.POINTER(dh_subgrid_params), _P5,
                                     C.c_void_p, _dp]
_lib.dh_value_and_grad_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_double,
                                        C.c_double, C.c_double, C.c_double, _dp, _dp, C.c_int, C.c_int, C.c_void_p, _dp,
                                        C.POINTER(dh_dparams)]
_lib.dh_get_step_dparams.argtypes = [C.c_void_p, _dp, C.c_int]
_lib.dh_chain_cosmology.argtypes = [C.POINTER(dh_cosmology), C.c_double, C.c_double, C.c_int, _dp, _dp, _dp]
_lib.dh_power_spectrum.argtypes = [C.c_void_p, C.c_void_p, _dp, _dp]
_lib.dh_power_spectrum_vjp.argtypes = [C.c_void_p, C.c_void_p, _dp, C.c_void_p]
_lib.dh_ic_zeldovich_vjp.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.POINTER(dh_cot), C.c_void_p]
_lib.dh_ic_factors.argtypes = [C.POINTER(dh_cosmology), C.c_double, C.c_double, C.c_double, C.c_double, _dp, _dp]


def _check(rc, where):
    if rc != DH_OK:
        raise DhError(rc, where)


def _ptrs(t: torch.Tensor, n: int, arr_type):
    """Pointers to the n leading slices of a contiguous fp32 CUDA tensor of shape (>= n, ...)."""
    assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.shape[0] >= n, (t.shape, t.dtype)
    stride = t[0].numel() * 4
    base = t.data_ptr()
    return arr_type(*[base + i * stride for i in range(n)])


class State:
    """Device state: gas (5,N,N,N) -- (6,N,N,N) with dual energy, the sixth field is q = a^2 rho e (dh_state.eint) -- and
    part (6,N_p) fp32 CUDA tensors (caller-owned) + host scalars."""

    def __init__(self, gas, part, a, dt_prev=0.0, step=0, device="cuda"):
        self.gas = torch.as_tensor(np.asarray(gas, dtype=np.float32) if not torch.is_tensor(gas) else gas,
                                   dtype=torch.float32).to(device).contiguous()
        part = np.asarray(part, dtype=np.float32).reshape(6, -1) if not torch.is_tensor(part) else part
        self.part = torch.as_tensor(part, dtype=torch.float32).to(device).contiguous()
        self.a, self.dt_prev, self.step = float(a), float(dt_prev), int(step)

    def c_struct(self) -> dh_state:
        s = dh_state()
        s.gas = _ptrs(self.gas, 5, _P5)
        if self.gas.shape[0] == 6:
            s.eint = self.gas[5].data_ptr()
        if self.part.shape[1] > 0:
            s.part = _ptrs(self.part, 6, _P6)
        s.a, s.dt_prev, s.step = self.a, self.dt_prev, self.step
        return s

    def clone(self):
        return State(self.gas.clone(), self.part.clone(), self.a, self.dt_prev, self.step)


class Cot:
    def __init__(self, gas, part, device="cuda"):
        self.gas = torch.as_tensor(gas, dtype=torch.float32).to(device).contiguous()
        self.part = torch.as_tensor(part, dtype=torch.float32).to(device).contiguous()

    def c_struct(self) -> dh_cot:
        s = dh_cot()
        s.gas = _ptrs(self.gas, 5, _P5)
        if self.gas.shape[0] == 6:
            s.eint = self.gas[5].data_ptr()
        if self.part.shape[1] > 0:
            s.part = _ptrs(self.part, 6, _P6)
        return s


class Context:
    """Owner of a dh_ctx*.  Methods are the C calls with tensors marshalled to pointers."""

    def __init__(self, N, box, gamma, n_part_side=None, H0=100.0, Omega_m=1.0, Omega_b=0.16, Omega_L=0.0, static_mode=0,
                 gravity_on=1, hydro_on=1, gas_sources_gravity=1, e_floor=1e-12, lim_eps=1e-20, want_dA=1, want_dsched=1,
                 dual_energy=0, dual_eta=1e-3, stream: torch.cuda.Stream | None = None):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2502_02294_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self.N = int(N)
        self.nc = 6 if dual_energy else 5
        self.nps = self.N if n_part_side is None else int(n_part_side)
        self.np = self.nps ** 3
        self.cosmo = dh_cosmology(H0, Omega_m, Omega_b, Omega_L, int(static_mode))
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        self.opt = dh_options(self.nps, int(gravity_on), int(hydro_on), int(gas_sources_gravity), float(e_floor),
                              float(lim_eps), C.c_void_p(self.stream.cuda_stream), int(want_dA), int(want_dsched),
                              int(dual_energy), float(dual_eta))
        self._h = C.c_void_p()
        _check(_lib.dh_init(C.byref(self._h), self.N, float(box), float(gamma), C.byref(self.cosmo), C.byref(self.opt)),
               "dh_init")

    def close(self):
        if self._h:
            _lib.dh_free(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the path
    def dh_step(self, st: State, dt, a, cmax: torch.Tensor | None = None):
        cs = st.c_struct()
        _check(_lib.dh_step(self._h, C.byref(cs), float(dt), float(a), cmax.data_ptr() if cmax is not None else None),
               "dh_step")
        st.a, st.dt_prev, st.step = cs.a, cs.dt_prev, cs.step

    def dh_step_vjp(self, st_in: State, dt, a, cot_out: Cot, cot_in: Cot, dparams: dh_dparams | None = None):
        dparams = dparams if dparams is not None else dh_dparams()
        cs, co, ci = st_in.c_struct(), cot_out.c_struct(), cot_in.c_struct()
        _check(_lib.dh_step_vjp(self._h, C.byref(cs), float(dt), float(a), C.byref(co), C.byref(ci), C.byref(dparams)),
               "dh_step_vjp")
        return dparams

    def dh_run(self, st: State, a_sched, dt_sched, checkpoint_stride=0):
        a_s = np.ascontiguousarray(a_sched, dtype=np.float64)
        d_s = np.ascontiguousarray(dt_sched, dtype=np.float64)
        assert len(a_s) == len(d_s)
        cs = st.c_struct()
        rc = _lib.dh_run(self._h, C.byref(cs), a_s.ctypes.data_as(_dp), d_s.ctypes.data_as(_dp), len(d_s),
                         int(checkpoint_stride))
        st.a, st.dt_prev, st.step = cs.a, cs.dt_prev, cs.step
        _check(rc, "dh_run")

    def dh_reserve(self, n_steps, checkpoint_stride):
        _check(_lib.dh_reserve(self._h, int(n_steps), int(checkpoint_stride)), "dh_reserve")

    def dh_run_vjp(self, cot_final: Cot, cot_initial: Cot, dparams: dh_dparams | None = None):
        dparams = dparams if dparams is not None else dh_dparams()
        cf, ci = cot_final.c_struct(), cot_initial.c_struct()
        _check(_lib.dh_run_vjp(self._h, C.byref(cf), C.byref(ci), C.byref(dparams)), "dh_run_vjp")
        return dparams

    def dh_run_host(self, gas_host: torch.Tensor, part_host: torch.Tensor, a, dt_prev, step, a_sched, dt_sched,
                    checkpoint_stride=0):
        """gas_host (5,N,N,N), part_host (6,N_p): HOST fp32 tensors (pinned or not), updated in place."""
        assert not gas_host.is_cuda and gas_host.dtype == torch.float32 and gas_host.is_contiguous()
        a_s = np.ascontiguousarray(a_sched, dtype=np.float64)
        d_s = np.ascontiguousarray(dt_sched, dtype=np.float64)
        ca, cd, cst = C.c_double(a), C.c_double(dt_prev), C.c_int64(step)
        _check(_lib.dh_run_host(self._h, gas_host.data_ptr(), part_host.data_ptr() if self.np else None, C.byref(ca),
                                C.byref(cd), C.byref(cst), a_s.ctypes.data_as(_dp), d_s.ctypes.data_as(_dp), len(d_s),
                                int(checkpoint_stride)), "dh_run_host")
        return ca.value, cd.value, cst.value

    def dh_run_vjp_host(self, cot_gas_host: torch.Tensor, cot_part_host: torch.Tensor, dparams=None):
        dparams = dparams if dparams is not None else dh_dparams()
        _check(_lib.dh_run_vjp_host(self._h, cot_gas_host.data_ptr(), cot_part_host.data_ptr() if self.np else None,
                                    C.byref(dparams)), "dh_run_vjp_host")
        return dparams

    # ---- helpers
    def dh_conserved_sums(self, st: State):
        """(sum rho, sum m_x, sum m_y, sum m_z, sum eps, m_p sum w_x, m_p sum w_y, m_p sum w_z) as a numpy array (fp64)."""
        out = np.zeros(8)
        cs = st.c_struct()
        _check(_lib.dh_conserved_sums(self._h, C.byref(cs), out.ctypes.data_as(_dp)), "dh_conserved_sums")
        return out

    def dh_debug_poison(self, level=0):
        _check(_lib.dh_debug_poison(self._h, int(level)), "dh_debug_poison")

    def dh_get_cmax(self, n):
        out = np.zeros((n, 3), dtype=np.float32)
        _check(_lib.dh_get_cmax(self._h, out.ctypes.data, n), "dh_get_cmax")
        return out

    def dh_sync(self):
        _check(_lib.dh_sync(self._h), "dh_sync")

    def dh_tune(self, key: str, value: int):
        _check(_lib.dh_tune(self._h, key.encode(), int(value)), "dh_tune")

    def dh_device_bytes(self):
        return int(_lib.dh_device_bytes(self._h))

    def dh_launch_count(self):
        return int(_lib.dh_launch_count(self._h))

    def dh_profile_enable(self, on=True):
        _check(_lib.dh_profile_enable(self._h, int(bool(on))), "dh_profile_enable")

    def dh_profile_read(self):
        """{category: (milliseconds, launches)} since the last read (CUDA events around every launch)."""
        n = _lib.dh_profile_categories()
        ms = (C.c_double * n)()
        cnt = (C.c_int64 * n)()
        _check(_lib.dh_profile_read(self._h, ms, cnt), "dh_profile_read")
        return {_lib.dh_profile_name(i).decode(): (ms[i], cnt[i]) for i in range(n) if cnt[i]}

    def dh_debug_cell_index(self, x: torch.Tensor):
        x = x.contiguous()
        i0 = torch.empty(x.numel(), dtype=torch.int32, device=x.device)
        i1 = torch.empty_like(i0)
        _check(_lib.dh_debug_cell_index(self._h, x.data_ptr(), x.numel(), i0.data_ptr(), i1.data_ptr()),
               "dh_debug_cell_index")
        return i0, i1

    # ---- single kernels
    def dh_sweep(self, d, gas_in: torch.Tensor, g: torch.Tensor | None, lam, kap, cmax: torch.Tensor | None = None):
        out = torch.empty_like(gas_in)
        _check(_lib.dh_sweep(self._h, int(d), _ptrs(gas_in, 5, _P5), g.data_ptr() if g is not None else None, float(lam),
                             float(kap), _ptrs(out, 5, _P5), cmax.data_ptr() if cmax is not None else None), "dh_sweep")
        return out

    def dh_sweep_vjp(self, d, gas_in, g, lam, kap, cot_out):
        cot_in = torch.empty_like(gas_in)
        gb = torch.zeros_like(g) if g is not None else None
        sc = torch.zeros(3, dtype=torch.float64, device=gas_in.device)
        _check(_lib.dh_sweep_vjp(self._h, int(d), _ptrs(gas_in, 5, _P5), g.data_ptr() if g is not None else None,
                                 float(lam), float(kap), _ptrs(cot_out, 5, _P5), _ptrs(cot_in, 5, _P5),
                                 gb.data_ptr() if gb is not None else None, sc.data_ptr()), "dh_sweep_vjp")
        return cot_in, gb, sc

    def dh_sweep_de(self, d, gas_in: torch.Tensor, g: torch.Tensor | None, lam, kap, cmax: torch.Tensor | None = None):
        """The dual-energy sweep on a (6,N,N,N) state (needs a context with dual_energy=1)."""
        out = torch.empty_like(gas_in)
        _check(_lib.dh_sweep_de(self._h, int(d), _ptrs(gas_in, 6, _P6), g.data_ptr() if g is not None else None,
                                float(lam), float(kap), _ptrs(out, 6, _P6),
                                cmax.data_ptr() if cmax is not None else None), "dh_sweep_de")
        return out

    def dh_sweep_de_vjp(self, d, gas_in, g, lam, kap, cot_out):
        cot_in = torch.empty_like(gas_in)
        gb = torch.zeros_like(g) if g is not None else None
        sc = torch.zeros(3, dtype=torch.float64, device=gas_in.device)
        _check(_lib.dh_sweep_de_vjp(self._h, int(d), _ptrs(gas_in, 6, _P6), g.data_ptr() if g is not None else None,
                                    float(lam), float(kap), _ptrs(cot_out, 6, _P6), _ptrs(cot_in, 6, _P6),
                                    gb.data_ptr() if gb is not None else None, sc.data_ptr()), "dh_sweep_de_vjp")
        return cot_in, gb, sc

    def dh_deposit(self, rho_gas: torch.Tensor | None, pos: torch.Tensor):
        out = torch.empty((self.N,) * 3, dtype=torch.float32, device=pos.device)
        _check(_lib.dh_deposit(self._h, rho_gas.data_ptr() if rho_gas is not None else None, _ptrs(pos, 3, _P3),
                               out.data_ptr()), "dh_deposit")
        return out

    def dh_poisson(self, delta: torch.Tensor, A):
        g = torch.empty((3,) + tuple(delta.shape), dtype=torch.float32, device=delta.device)
        _check(_lib.dh_poisson(self._h, delta.data_ptr(), float(A), _ptrs(g, 3, _P3)), "dh_poisson")
        return g

    def dh_poisson_vjp(self, gb: torch.Tensor, A):
        db = torch.empty(tuple(gb.shape[1:]), dtype=torch.float32, device=gb.device)
        _check(_lib.dh_poisson_vjp(self._h, _ptrs(gb, 3, _P3), float(A), db.data_ptr()), "dh_poisson_vjp")
        return db

    def dh_kick_drift(self, g: torch.Tensor | None, part: torch.Tensor, K, dtau_over_dx):
        gp = _ptrs(g, 3, _P3) if g is not None else _P3()
        _check(_lib.dh_kick_drift(self._h, gp, _ptrs(part, 6, _P6), float(K), float(dtau_over_dx)), "dh_kick_drift")

    def dh_ic_zeldovich(self, delta_init: torch.Tensor, a0, vel_factor, e_tilde0) -> State:
        """delta_init (N,N,N) fp32 CUDA tensor -> a new State (tensors allocated here, filled by the library)."""
        assert delta_init.is_cuda and delta_init.dtype == torch.float32 and delta_init.is_contiguous()
        n3 = self.N ** 3
        st = State(torch.empty((self.nc, self.N, self.N, self.N), dtype=torch.float32, device=delta_init.device),
                   torch.empty((6, n3), dtype=torch.float32, device=delta_init.device), a0)
        cs = st.c_struct()
        _check(_lib.dh_ic_zeldovich(self._h, delta_init.data_ptr(), float(a0), float(vel_factor), float(e_tilde0),
                                    C.byref(cs)), "dh_ic_zeldovich")
        st.a, st.dt_prev, st.step = cs.a, cs.dt_prev, cs.step
        return st

    def dh_subgrid_step(self, gas: torch.Tensor, g0: torch.Tensor, g1: torch.Tensor, par: dict, want_z=True,
                        pos: torch.Tensor | None = None, aux: torch.Tensor | None = None):
        """Sub-grid step in place on gas (5,N,N,N); returns z (N,N,N) or None.  par: the fields of dh_subgrid_params."""
        q = dh_subgrid_params(**{k: float(v) for k, v in par.items()})
        z = torch.empty_like(g0) if (want_z or aux is not None) else None
        pp = C.cast(_ptrs(pos, 3, _P3), C.c_void_p) if pos is not None else None
        _check(_lib.dh_subgrid_step(self._h, _ptrs(gas, 5, _P5), g0.data_ptr(), g1.data_ptr(), C.byref(q),
                                    z.data_ptr() if z is not None else None, pp,
                                    aux.data_ptr() if aux is not None else None), "dh_subgrid_step")
        return z

    def dh_subgrid_step_vjp(self, gas_in: torch.Tensor, g0: torch.Tensor, g1: torch.Tensor, par: dict,
                            cot_gas: torch.Tensor, cot_z: torch.Tensor | None = None):
        """cot_gas (5,N,N,N) is transformed in place; returns (dT_c, ddelta_c, dPi0, de_inject) as a float64 array."""
        q = dh_subgrid_params(**{k: float(v) for k, v in par.items()})
        d = np.zeros(4)
        _check(_lib.dh_subgrid_step_vjp(self._h, _ptrs(gas_in, 5, _P5), g0.data_ptr(), g1.data_ptr(), C.byref(q),
                                        _ptrs(cot_gas, 5, _P5), cot_z.data_ptr() if cot_z is not None else None,
                                        d.ctypes.data_as(_dp)), "dh_subgrid_step_vjp")
        return d

    def dh_value_and_grad_host(self, delta_init: torch.Tensor, data: torch.Tensor, noise_var: torch.Tensor | None, observable,
                               scale, weight, a0, vel_factor, e_tilde0, a_sched, dt_sched, checkpoint_stride,
                               grad_out: torch.Tensor, dparams: dh_dparams | None = None):
        """HOST (ideally pinned) fp32 tensors in, grad_out (host) filled; returns (loss, dparams)."""
        for t in (delta_init, data, grad_out) + ((noise_var,) if noise_var is not None else ()):
            assert not t.is_cuda and t.dtype == torch.float32 and t.is_contiguous()
        a_s = np.ascontiguousarray(a_sched, dtype=np.float64); dt_s = np.ascontiguousarray(dt_sched, dtype=np.float64)
        dparams = dparams if dparams is not None else dh_dparams()
        loss = C.c_double(0.0)
        _check(_lib.dh_value_and_grad_host(self._h, delta_init.data_ptr(), data.data_ptr(),
                                           noise_var.data_ptr() if noise_var is not None else None, int(observable),
                                           float(scale), float(weight), float(a0), float(vel_factor), float(e_tilde0),
                                           a_s.ctypes.data_as(_dp), dt_s.ctypes.data_as(_dp), len(dt_s),
                                           int(checkpoint_stride), grad_out.data_ptr(), C.byref(loss), C.byref(dparams)),
               "dh_value_and_grad_host")
        return loss.value, dparams

    def dh_get_step_dparams(self, n_steps: int) -> np.ndarray:
        """(n_steps, 5) = (dgamma, dDtau, dkappa, dK, dA) per step of the last dh_run_vjp (want_dsched = 1)."""
        out = np.zeros((int(n_steps), 5))
        _check(_lib.dh_get_step_dparams(self._h, out.ctypes.data_as(_dp), int(n_steps)), "dh_get_step_dparams")
        return out

    def dh_chain_cosmology(self, a0, a1, step_dparams: np.ndarray):
        """(dL/dOmega_m, dL/dH0) through the step scalars of the ln-a schedule (host arithmetic in the library)."""
        sd = np.ascontiguousarray(step_dparams, dtype=np.float64)
        dom, dh0 = C.c_double(0.0), C.c_double(0.0)
        _check(_lib.dh_chain_cosmology(C.byref(self.cosmo), float(a0), float(a1), int(sd.shape[0]), sd.ctypes.data_as(_dp),
                                       C.byref(dom), C.byref(dh0)), "dh_chain_cosmology")
        return dom.value, dh0.value

    def dh_power_spectrum(self, field: torch.Tensor):
        """(P_b, count_b), b = 1 .. N/2, as host float64 arrays."""
        nb = self.N // 2
        P = np.zeros(nb); cnt = np.zeros(nb)
        _check(_lib.dh_power_spectrum(self._h, field.data_ptr(), P.ctypes.data_as(_dp), cnt.ctypes.data_as(_dp)),
               "dh_power_spectrum")
        return P, cnt

    def dh_power_spectrum_vjp(self, field: torch.Tensor, power_bar) -> torch.Tensor:
        pb = np.ascontiguousarray(power_bar, dtype=np.float64)
        assert pb.shape == (self.N // 2,)
        out = torch.empty_like(field)
        _check(_lib.dh_power_spectrum_vjp(self._h, field.data_ptr(), pb.ctypes.data_as(_dp), out.data_ptr()),
               "dh_power_spectrum_vjp")
        return out

    def dh_data_term(self, observable: int, gas: torch.Tensor, data: torch.Tensor, noise_var: torch.Tensor | None = None,
                     scale=1.0, weight=0.5, cot_gas: torch.Tensor | None = None, want_loss=True):
        """L = weight sum (scale O - data)^2 / noise_var; fills cot_gas (5,N,N,N) if given; returns L (host) or None."""
        loss = C.c_double(0.0)
        cg = C.cast(_ptrs(cot_gas, 5, _P5), C.c_void_p) if cot_gas is not None else None
        _check(_lib.dh_data_term(self._h, int(observable), _ptrs(gas, 5, _P5), data.data_ptr(),
                                 noise_var.data_ptr() if noise_var is not None else None, float(scale), float(weight), cg,
                                 C.byref(loss) if want_loss else None), "dh_data_term")
        return loss.value if want_loss else None

    def dh_ic_zeldovich_vjp(self, delta_init: torch.Tensor, vel_factor, e_tilde0, cot_state: Cot) -> torch.Tensor:
        assert delta_init.is_cuda and delta_init.dtype == torch.float32 and delta_init.is_contiguous()
        grad = torch.empty_like(delta_init)
        cs = cot_state.c_struct()
        _check(_lib.dh_ic_zeldovich_vjp(self._h, delta_init.data_ptr(), float(vel_factor), float(e_tilde0), C.byref(cs),
                                        grad.data_ptr()), "dh_ic_zeldovich_vjp")
        return grad


DH_NOALLOC_MAX_ELEMS = 134217728


def dh_conserved_sums_noalloc(gas: torch.Tensor, w: torch.Tensor | None, m_p: float, out: torch.Tensor, stream=None):
    """include/diffhydro.h: the eight conserved sums without a context and without any allocation.  gas: (>= 5, ...) fp32
    CUDA tensor (fields 0..4 are summed), w: (3, n_part) fp32 CUDA tensor of particle velocities or None, out: 8 fp64 on
    the device, written by the kernel on `stream` (default: torch's current stream).  Marshalling only; asynchronous."""
    assert gas.is_cuda and gas.dtype == torch.float32 and gas.is_contiguous() and gas.shape[0] >= 5
    assert out.is_cuda and out.dtype == torch.float64 and out.is_contiguous() and out.numel() >= 8
    n_cells = gas[0].numel()
    g = (C.c_void_p * 5)(*[gas[k].data_ptr() for k in range(5)])
    n_part = 0 if w is None else int(w.shape[1])
    wp = None
    if n_part:
        assert w.is_cuda and w.dtype == torch.float32 and w.is_contiguous() and w.shape[0] == 3
        wp = (C.c_void_p * 3)(*[w[k].data_ptr() for k in range(3)])
    stream = stream if stream is not None else torch.cuda.current_stream(gas.device)
    with torch.cuda.device(gas.device):
        _check(_lib.dh_conserved_sums_noalloc(g, n_cells, wp, n_part, float(m_p), C.c_void_p(out.data_ptr()),
                                              C.c_void_p(stream.cuda_stream)), "dh_conserved_sums_noalloc")
    return out


def dh_schedule_lna(a0, a1, n, H0=100.0, Omega_m=1.0, Omega_b=0.16, Omega_L=0.0):
    co = dh_cosmology(H0, Omega_m, Omega_b, Omega_L, 0)
    a = np.zeros(n + 1)
    dt = np.zeros(n)
    _check(_lib.dh_schedule_lna(C.byref(co), float(a0), float(a1), int(n), a.ctypes.data_as(_dp), dt.ctypes.data_as(_dp)),
           "dh_schedule_lna")
    return a, dt


def dh_step_scalars(a_i, a_next, dt, dt_prev, H0=100.0, Omega_m=1.0, Omega_b=0.16, Omega_L=0.0, static_mode=0):
    co = dh_cosmology(H0, Omega_m, Omega_b, Omega_L, int(static_mode))
    out = np.zeros(4)
    _check(_lib.dh_step_scalars(C.byref(co), float(a_i), float(a_next), float(dt), float(dt_prev),
                                out.ctypes.data_as(_dp)), "dh_step_scalars")
    return dict(dtau=out[0], kappa=out[1], K=out[2], A=out[3])


def dh_ic_factors(a0, T0, gamma, mu=0.59, H0=100.0, Omega_m=1.0, Omega_b=0.16, Omega_L=0.0):
    """(vel_factor, e_tilde0) = (a0^2 H f, a0^2 e(T0)): the scalar arguments of dh_ic_zeldovich (host call)."""
    co = dh_cosmology(H0, Omega_m, Omega_b, Omega_L, 0)
    vf, e0 = C.c_double(0.0), C.c_double(0.0)
    _check(_lib.dh_ic_factors(C.byref(co), float(a0), float(T0), float(gamma), float(mu), C.byref(vf), C.byref(e0)),
           "dh_ic_factors")
    return vf.value, e0.value


def ic_factors_for(cfg):
    """dh_ic_factors for a workloads.Config."""
    return dh_ic_factors(cfg.a0, cfg.T0, cfg.gamma, H0=cfg.H0, Omega_m=cfg.Omega_m, Omega_b=cfg.Omega_b,
                         Omega_L=cfg.Omega_L)


def context_for(cfg, **kw) -> Context:
    """Context for a workloads.Config."""
    args = dict(N=cfg.N, box=cfg.box, gamma=cfg.gamma, n_part_side=cfg.n_side, H0=cfg.H0, Omega_m=cfg.Omega_m,
                Omega_b=cfg.Omega_b, Omega_L=cfg.Omega_L, static_mode=cfg.static_mode, gravity_on=cfg.gravity_on,
                e_floor=cfg.e_floor(), lim_eps=cfg.lim_eps)
    args.update(kw)
    return Context(**args)
