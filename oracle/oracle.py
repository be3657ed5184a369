"""ctypes binding of the CPU oracle (oracle/libkr_oracle.so).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this.  It never imports the CUDA binding and shares no code with it.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libkr_oracle.so")
_lib = None

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


class _Desc(C.Structure):
    _fields_ = [("n_elem", C.c_int32), ("n_species", C.c_int32), ("n_reac", C.c_int32),
                ("elem_mass", _dp), ("composition", _ip),
                ("reac_idx", _ip), ("reac_nu", _ip), ("prod_idx", _ip), ("prod_nu", _ip),
                ("A", _dp), ("beta", _dp), ("Ea_over_k", _dp),
                ("flags", _ip), ("aux_index", _ip), ("tb_eff", _dp), ("q_ext", _dp),
                ("nasa_lo", _dp), ("nasa_hi", _dp), ("T_mid", _dp),
                ("T_lo", C.c_double), ("T_hi", C.c_double), ("energy_equation", C.c_int32)]


class _Opts(C.Structure):
    _fields_ = [("max_newton", C.c_int32), ("fixed_newton", C.c_int32), ("h0_mode", C.c_int32),
                ("rtol", C.c_double), ("atol_y", C.c_double), ("atol_T", C.c_double), ("neg_tol", C.c_double),
                ("eta", C.c_double), ("y_floor", C.c_double), ("shrink", C.c_double), ("grow_fast", C.c_double),
                ("grow_mid", C.c_double), ("chg_floor", C.c_double), ("chg_max", C.c_double),
                ("it_fast", C.c_int32), ("it_mid", C.c_int32), ("max_substeps", C.c_int32), ("finalize", C.c_int32),
                ("h_min_rel", C.c_double), ("bail_ratio", C.c_double), ("retry", C.c_int32), ("retry_h0", C.c_double),
                ("cons_tol", C.c_double)]


class Stats(C.Structure):
    _fields_ = [("n_substeps", C.c_int64), ("n_rejected", C.c_int64), ("n_newton", C.c_int64),
                ("n_lu", C.c_int64), ("n_rate_evals", C.c_int64), ("n_failed", C.c_int64)]

    def as_dict(self):
        return {k: int(getattr(self, k)) for k, _ in self._fields_}


def load():
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        from . import build as _b  # type: ignore
        _b.build_oracle()
    lib = C.CDLL(_LIB_PATH)
    vp = C.c_void_p
    lib.kr_oracle_network_create.argtypes = [C.POINTER(_Desc), C.POINTER(vp)]
    lib.kr_oracle_network_destroy.argtypes = [vp]
    lib.kr_oracle_network_destroy.restype = None
    lib.kr_oracle_set_options.argtypes = [vp, C.POINTER(_Opts)]
    lib.kr_oracle_thermochem_step_ex.argtypes = [vp, C.c_int64, _dp, _dp, _dp, C.c_double, _dp, C.c_int32, _ip,
                                                 C.POINTER(Stats), _dp, C.c_int32]
    lib.kr_oracle_thermochem_step_diag.argtypes = [vp, C.c_int64, _dp, _dp, _dp, C.c_double, _dp, C.c_int32, _ip,
                                                   C.POINTER(Stats), _dp, _dp, C.c_int32]
    lib.kr_oracle_witness_step_ex.argtypes = [vp, C.c_int64, _dp, _dp, _dp, C.c_double, _dp, C.c_int32, _ip,
                                              C.POINTER(Stats), C.c_int32]
    lib.kr_oracle_rate_constants.argtypes = [vp, C.c_double, _dp, _dp, _dp]
    lib.kr_oracle_eval_rhs.argtypes = [vp, C.c_double, C.c_double, _dp, _dp, _dp]
    lib.kr_oracle_eval_rhs_complex.argtypes = [vp, C.c_double, C.c_double, C.c_double, _dp, _dp, _dp, _dp, _dp]
    lib.kr_oracle_eval_jacobian.argtypes = [vp, C.c_double, C.c_double, _dp, _dp, _dp]
    lib.kr_oracle_lu_solve.argtypes = [C.c_int32, _dp, _dp, _dp, _ip]
    lib.kr_oracle_finalize.argtypes = [vp, _dp, _dp, C.POINTER(C.c_int32)]
    lib.kr_oracle_be_substep.argtypes = [vp, C.c_double, C.c_double, _dp, _dp, C.c_double, _dp, _dp, _ip]
    _lib = lib
    return lib


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _i(a):
    return None if a is None else a.ctypes.data_as(_ip)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.int32)


class OracleNetwork:
    """Owns a kr_oracle_network built from a ``workloads.Network``-shaped object."""

    def __init__(self, net, opts=None):
        lib = load()
        self._keep = dict(
            elem_mass=_f64(net.elem_mass), composition=_i32(net.composition),
            reac_idx=_i32(net.reac_idx), reac_nu=_i32(net.reac_nu), prod_idx=_i32(net.prod_idx),
            prod_nu=_i32(net.prod_nu), A=_f64(net.A), beta=_f64(net.beta), Ea=_f64(net.Ea_over_k),
            flags=_i32(net.flags), aux_index=_i32(net.aux_index), tb_eff=_f64(net.tb_eff), q_ext=_f64(net.q_ext),
            nasa_lo=_f64(net.nasa_lo), nasa_hi=_f64(net.nasa_hi), T_mid=_f64(net.T_mid))
        k = self._keep
        d = _Desc(net.n_elem, net.n_species, net.n_reac, _d(k["elem_mass"]), _i(k["composition"]),
                  _i(k["reac_idx"]), _i(k["reac_nu"]), _i(k["prod_idx"]), _i(k["prod_nu"]),
                  _d(k["A"]), _d(k["beta"]), _d(k["Ea"]), _i(k["flags"]), _i(k["aux_index"]),
                  _d(k["tb_eff"]), _d(k["q_ext"]), _d(k["nasa_lo"]), _d(k["nasa_hi"]), _d(k["T_mid"]),
                  float(net.T_lo), float(net.T_hi), int(net.energy_equation))
        h = C.c_void_p()
        rc = lib.kr_oracle_network_create(C.byref(d), C.byref(h))
        if rc != 0:
            raise ValueError(f"kr_oracle_network_create failed: {rc}")
        self._h = h
        self.S = net.n_species
        self.R = net.n_reac
        self.N = net.n_species + (1 if net.energy_equation else 0)
        self.energy = int(net.energy_equation)
        if opts is not None:
            self.set_options(opts)

    def __del__(self):
        try:
            if getattr(self, "_h", None):
                load().kr_oracle_network_destroy(self._h)
                self._h = None
        except Exception:
            pass

    def set_options(self, o) -> None:
        s = _Opts(o.max_newton, o.fixed_newton, o.h0_mode, o.rtol, o.atol_y, o.atol_T, o.neg_tol, o.eta, o.y_floor,
                  o.shrink, o.grow_fast, o.grow_mid, o.chg_floor, o.chg_max, o.it_fast, o.it_mid, o.max_substeps,
                  getattr(o, "finalize", 1), getattr(o, "h_min_rel", 1e-12), getattr(o, "bail_ratio", 10.0),
                  getattr(o, "retry", 0), getattr(o, "retry_h0", 0.01), getattr(o, "cons_tol", 1e-13))
        rc = load().kr_oracle_set_options(self._h, C.byref(s))
        if rc != 0:
            raise ValueError("kr_oracle_set_options rejected the options")

    # -- the step -------------------------------------------------------------------------
    def step(self, cells, n_threads: int = 1, witness: bool = False, want_margins: bool = False, amps=None):
        """Returns (T, y, status, stats, margins) -- inputs are not modified.  amps: optional float64 [n_cells] array
        that receives the per-cell cancellation diagnostic of kr_oracle_thermochem_step_diag."""
        lib = load()
        n = cells.n_cells
        T = _f64(cells.T).copy()
        y = _f64(cells.y).copy()
        rho = _f64(cells.rho)
        aux = _f64(cells.aux)
        n_aux = 0 if aux is None else int(aux.shape[0])
        status = np.zeros(n, np.int32)
        st = Stats()
        margins = np.full(n, np.inf) if want_margins else None
        if witness:
            rc = lib.kr_oracle_witness_step_ex(self._h, n, _d(rho), _d(T), _d(y), float(cells.dt), _d(aux), n_aux,
                                               _i(status), C.byref(st), int(n_threads))
        elif amps is not None:
            assert amps.dtype == np.float64 and amps.shape == (n,) and amps.flags.c_contiguous
            rc = lib.kr_oracle_thermochem_step_diag(self._h, n, _d(rho), _d(T), _d(y), float(cells.dt), _d(aux), n_aux,
                                                    _i(status), C.byref(st), _d(margins), _d(amps), int(n_threads))
        else:
            rc = lib.kr_oracle_thermochem_step_ex(self._h, n, _d(rho), _d(T), _d(y), float(cells.dt), _d(aux), n_aux,
                                                  _i(status), C.byref(st), _d(margins), int(n_threads))
        if rc != 0:
            raise RuntimeError(f"oracle step failed: {rc}")
        return T, y, status, st.as_dict(), margins

    # -- pieces ---------------------------------------------------------------------------
    def rate_constants(self, T: float, aux_cell=None) -> Tuple[np.ndarray, np.ndarray]:
        kf = np.zeros(self.R); kr = np.zeros(self.R)
        ax = _f64(np.zeros(1) if aux_cell is None else aux_cell)
        load().kr_oracle_rate_constants(self._h, float(T), _d(ax), _d(kf), _d(kr))
        return kf, kr

    def rhs(self, rho: float, T: float, y, aux_cell=None) -> np.ndarray:
        f = np.zeros(self.N)
        ax = _f64(np.zeros(1) if aux_cell is None else aux_cell)
        load().kr_oracle_eval_rhs(self._h, float(rho), float(T), _d(_f64(y)), _d(ax), _d(f))
        return f

    def rhs_complex(self, rho: float, T: complex, y, aux_cell=None) -> np.ndarray:
        y = np.asarray(y, dtype=np.complex128)
        yr = _f64(y.real); yi = _f64(y.imag)
        fr = np.zeros(self.N); fi = np.zeros(self.N)
        ax = _f64(np.zeros(1) if aux_cell is None else aux_cell)
        T = complex(T)
        load().kr_oracle_eval_rhs_complex(self._h, float(rho), T.real, T.imag, _d(yr), _d(yi), _d(ax), _d(fr), _d(fi))
        return fr + 1j * fi

    def jacobian(self, rho: float, T: float, y, aux_cell=None) -> np.ndarray:
        J = np.zeros((self.N, self.N))
        ax = _f64(np.zeros(1) if aux_cell is None else aux_cell)
        load().kr_oracle_eval_jacobian(self._h, float(rho), float(T), _d(_f64(y)), _d(ax), _d(J))
        return J

    def finalize(self, y, y_in=None):
        """Post-processing stages 1-3 on one final state (y_in: the initial state of the step, or None);
        returns (y_out, status bits)."""
        yy = _f64(np.asarray(y, dtype=np.float64)).copy()
        yi = None if y_in is None else _f64(np.asarray(y_in, dtype=np.float64))
        st = C.c_int32(0)
        rc = load().kr_oracle_finalize(self._h, _d(yi), _d(yy), C.byref(st))
        if rc != 0:
            raise RuntimeError("oracle finalize failed")
        return yy, int(st.value)

    def be_substep(self, rho: float, T: float, y, h: float, aux_cell=None):
        u = np.zeros(self.N)
        e = C.c_double(); it = C.c_int32()
        ax = _f64(np.zeros(1) if aux_cell is None else aux_cell)
        rc = load().kr_oracle_be_substep(self._h, float(rho), float(T), _d(_f64(y)), _d(ax), float(h), _d(u),
                                         C.byref(e), C.byref(it))
        return u, e.value, it.value, rc


def lu_solve(M: np.ndarray, b: np.ndarray) -> Tuple[Optional[np.ndarray], np.ndarray, np.ndarray, int]:
    """Oracle LU (step 7).  Returns (x or None when singular, factors, perm, rc)."""
    n = int(M.shape[0])
    a = _f64(M).copy()
    x = np.zeros(n)
    p = np.zeros(n, np.int32)
    rc = load().kr_oracle_lu_solve(n, _d(a), _d(_f64(b)), _d(x), _i(p))
    return (x if rc == 0 else None), a, p, rc
