"""Thin ctypes binding of libkratos_chem.so (include/kratos_chem.h) -- argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  PyTorch appears only as the owner of
device memory (``tensor.data_ptr()``) and streams.  There is no CPU fallback: if the library is
missing it is an ImportError-like RuntimeError, and without a CUDA device ``Network(...)`` raises.
Function names mirror the C ABI (``kr_network_create`` -> ``Network``, ``kr_thermochem_step`` ->
``Network.thermochem_step`` ...).
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libkratos_chem.so")

KR_OK, KR_EINVAL, KR_ENETWORK, KR_ECUDA, KR_EUNSUPPORTED = 0, -1, -2, -3, -4
KR_FP64, KR_MIXED = 0, 1
KR_MAP_AUTO, KR_MAP_THREAD, KR_MAP_WARP, KR_MAP_CTA, KR_MAP_THREAD_TABLE, KR_MAP_GROUP_TABLE = 0, 1, 2, 3, 4, 5
ST_REJECTED_ONCE, ST_CLAMPED_NEG, ST_FP64_FALLBACK, ST_FAILED_REVERTED, ST_T_CLAMPED, ST_NO_RESERVOIR, ST_NEEDS_STAGE3, ST_STAGE3, ST_RETRIED = 1, 2, 4, 8, 16, 32, 64, 128, 256

EXPORTS = [
    "kr_network_create", "kr_network_destroy", "kr_default_opts", "kr_network_set_options",
    "kr_network_get_options", "kr_set_stream", "kr_network_set_mapping", "kr_network_set_tuning", "kr_network_info",
    "kr_network_kernel_desc", "kr_network_spec_source", "kr_network_spec_compile", "kr_network_wpc_compile", "kr_network_row_compile", "kr_last_mixed_stats", "kr_thermochem_step", "kr_thermochem_step_ex", "kr_thermochem_step_host", "kr_last_launch_count",
    "kr_layout_cell_to_soa", "kr_layout_soa_to_cell", "kr_math_probe", "kr_measure_fp64_peak", "kr_last_error", "kr_version",
    "kr_recon_create", "kr_recon_destroy", "kr_recon_projector", "kr_advect_species_1d", "kr_raytrace_cartesian",
    "kr_static_scratch_bytes", "kr_static_setup", "kr_static_max_cells", "kr_thermochem_step_static", "kr_table_rates",
]

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


class KrError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"kratos_chem error {code}: {msg}")
        self.code = code


class NetworkDesc(C.Structure):
    _fields_ = [("n_elem", C.c_int32), ("n_species", C.c_int32), ("n_reac", C.c_int32),
                ("elem_mass", _dp), ("composition", _ip),
                ("reac_idx", _ip), ("reac_nu", _ip), ("prod_idx", _ip), ("prod_nu", _ip),
                ("A", _dp), ("beta", _dp), ("Ea_over_k", _dp),
                ("flags", _ip), ("aux_index", _ip), ("tb_eff", _dp), ("q_ext", _dp),
                ("nasa_lo", _dp), ("nasa_hi", _dp), ("T_mid", _dp),
                ("T_lo", C.c_double), ("T_hi", C.c_double), ("energy_equation", C.c_int32)]


class SolverOpts(C.Structure):
    _fields_ = [("max_newton", C.c_int32), ("fixed_newton", C.c_int32), ("h0_mode", C.c_int32),
                ("rtol", C.c_double), ("atol_y", C.c_double), ("atol_T", C.c_double), ("neg_tol", C.c_double),
                ("eta", C.c_double), ("y_floor", C.c_double), ("shrink", C.c_double),
                ("grow_fast", C.c_double), ("grow_mid", C.c_double), ("chg_floor", C.c_double), ("chg_max", C.c_double),
                ("it_fast", C.c_int32), ("it_mid", C.c_int32), ("max_substeps", C.c_int32), ("finalize", C.c_int32),
                ("h_min_rel", C.c_double), ("bail_ratio", C.c_double), ("retry", C.c_int32), ("retry_h0", C.c_double),
                ("cons_tol", C.c_double)]


class StepStats(C.Structure):
    _fields_ = [("n_substeps", C.c_int64), ("n_rejected", C.c_int64), ("n_newton", C.c_int64),
                ("n_lu", C.c_int64), ("n_rate_evals", C.c_int64), ("n_failed", C.c_int64)]

    def as_dict(self):
        return {k: int(getattr(self, k)) for k, _ in self._fields_}


_lib = None


def load() -> C.CDLL:
    """dlopen the in-tree library.  Raises when it has not been built -- never falls back."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2504_04941_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp = C.c_void_p
    lib.kr_network_create.argtypes = [C.POINTER(NetworkDesc), C.POINTER(vp)]
    lib.kr_network_destroy.argtypes = [vp]
    lib.kr_network_destroy.restype = None
    lib.kr_default_opts.argtypes = [C.POINTER(SolverOpts)]
    lib.kr_default_opts.restype = None
    lib.kr_network_set_options.argtypes = [vp, C.POINTER(SolverOpts)]
    lib.kr_network_get_options.argtypes = [vp, C.POINTER(SolverOpts)]
    lib.kr_set_stream.argtypes = [vp, vp]
    lib.kr_network_set_mapping.argtypes = [vp, C.c_int32, C.c_int32]
    lib.kr_network_info.argtypes = [vp, _ip, _ip, _ip, _ip]
    lib.kr_thermochem_step.argtypes = [vp, C.c_int64, vp, vp, vp, C.c_double, C.c_int]
    lib.kr_thermochem_step_ex.argtypes = [vp, C.c_int64, vp, vp, vp, C.c_double, C.c_int, vp, C.c_int32, vp,
                                          C.POINTER(StepStats), vp]
    lib.kr_thermochem_step_host.argtypes = [vp, C.c_int64, vp, vp, vp, C.c_double, C.c_int, vp, C.c_int32, vp,
                                            C.POINTER(StepStats)]
    lib.kr_static_scratch_bytes.argtypes = []
    lib.kr_static_scratch_bytes.restype = C.c_int64
    lib.kr_static_setup.argtypes = [vp]
    lib.kr_static_max_cells.argtypes = [vp, C.POINTER(C.c_int64)]
    lib.kr_thermochem_step_static.argtypes = [vp, C.c_int64, vp, vp, vp, C.c_double, vp, C.c_int32, vp,
                                              C.POINTER(StepStats), vp]
    lib.kr_table_rates.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_double, C.c_double, C.c_double, C.c_double, vp, C.c_int64,
                                   vp, vp, vp, vp]
    lib.kr_last_launch_count.argtypes = [vp]
    lib.kr_network_kernel_desc.argtypes = [vp, C.c_char_p, C.c_int64]
    lib.kr_network_spec_source.argtypes = [C.POINTER(NetworkDesc), C.c_char_p, C.c_int64]
    lib.kr_network_spec_compile.argtypes = [C.POINTER(NetworkDesc), C.POINTER(C.c_int64), C.c_char_p, C.c_int64]
    lib.kr_network_row_compile.argtypes = [C.POINTER(NetworkDesc), C.c_int32, C.POINTER(C.c_int64), C.c_char_p, C.c_int64,
                                           C.c_void_p, C.c_int64]
    lib.kr_network_wpc_compile.argtypes = [C.POINTER(NetworkDesc), C.c_int, C.c_int32, C.POINTER(C.c_int64), C.c_char_p, C.c_int64,
                                           vp, C.c_int64]
    lib.kr_last_mixed_stats.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    lib.kr_network_set_tuning.argtypes = [vp, C.c_int32, C.c_int32]
    lib.kr_layout_cell_to_soa.argtypes = [vp, vp, C.c_int64, C.c_int32, vp]
    lib.kr_layout_soa_to_cell.argtypes = [vp, vp, C.c_int64, C.c_int32, vp]
    lib.kr_measure_fp64_peak.argtypes = [C.c_int32, _dp]
    lib.kr_math_probe.argtypes = [vp, vp, vp, C.c_int64, vp]
    lib.kr_recon_create.argtypes = [C.c_int32, C.c_int32, _ip, C.POINTER(vp)]
    lib.kr_recon_destroy.argtypes = [vp]
    lib.kr_recon_destroy.restype = None
    lib.kr_recon_projector.argtypes = [vp, _dp, _ip]
    lib.kr_advect_species_1d.argtypes = [vp, C.c_int64, vp, vp, vp, C.c_double, C.c_double, C.c_int32, C.c_int32, C.c_double,
                                         C.c_double, vp, vp, vp, vp, vp]
    lib.kr_raytrace_cartesian.argtypes = [C.c_int32, C.c_int32, C.c_int32, _dp, _dp, C.c_int64, vp, vp, C.c_int32, vp, C.c_int32,
                                          _dp, vp, vp, vp, vp, vp]
    lib.kr_last_error.restype = C.c_char_p
    lib.kr_version.restype = C.c_char_p
    _lib = lib
    return lib


def _check(rc: int) -> None:
    if rc != KR_OK:
        raise KrError(rc, load().kr_last_error().decode())


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.int32)


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _i(a):
    return None if a is None else a.ctypes.data_as(_ip)


def _ptr(t) -> Optional[int]:
    """Device (torch tensor) or host (numpy array) address; None passes NULL."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def default_opts() -> SolverOpts:
    o = SolverOpts()
    load().kr_default_opts(C.byref(o))
    return o


def opts_from(obj) -> SolverOpts:
    """Copy the fields of a ``workloads.SolverOpts``-shaped object into the C struct."""
    o = default_opts()
    for name, _ in SolverOpts._fields_:
        if hasattr(obj, name):
            setattr(o, name, getattr(obj, name))
    return o


def measure_fp64_peak(n_iter: int = 4096) -> float:
    v = C.c_double()
    _check(load().kr_measure_fp64_peak(int(n_iter), C.byref(v)))
    return v.value


def make_desc(net):
    """(kr_network_desc, keep-alive dict) from a ``workloads.Network``-shaped object."""
    k = dict(
        elem_mass=_f64(net.elem_mass), composition=_i32(net.composition),
        reac_idx=_i32(net.reac_idx), reac_nu=_i32(net.reac_nu), prod_idx=_i32(net.prod_idx),
        prod_nu=_i32(net.prod_nu), A=_f64(net.A), beta=_f64(net.beta), Ea=_f64(net.Ea_over_k),
        flags=_i32(net.flags), aux_index=_i32(net.aux_index), tb_eff=_f64(net.tb_eff), q_ext=_f64(net.q_ext),
        nasa_lo=_f64(net.nasa_lo), nasa_hi=_f64(net.nasa_hi), T_mid=_f64(net.T_mid))
    d = NetworkDesc(net.n_elem, net.n_species, net.n_reac, _d(k["elem_mass"]), _i(k["composition"]),
                    _i(k["reac_idx"]), _i(k["reac_nu"]), _i(k["prod_idx"]), _i(k["prod_nu"]),
                    _d(k["A"]), _d(k["beta"]), _d(k["Ea"]), _i(k["flags"]), _i(k["aux_index"]),
                    _d(k["tb_eff"]), _d(k["q_ext"]), _d(k["nasa_lo"]), _d(k["nasa_hi"]), _d(k["T_mid"]),
                    float(net.T_lo), float(net.T_hi), int(net.energy_equation))
    return d, k


def spec_source(net) -> str:
    """kr_network_spec_source: the generated constexpr-table translation unit (host only)."""
    d, keep = make_desc(net)
    n = load().kr_network_spec_source(C.byref(d), None, 0)
    if n < 0:
        _check(n)
    buf = C.create_string_buffer(n + 1)
    load().kr_network_spec_source(C.byref(d), buf, n + 1)
    return buf.value.decode()


def spec_compile(net) -> dict:
    """kr_network_spec_compile: NVRTC-compile the specialised kernel for sm_100a (no GPU needed)."""
    d, keep = make_desc(net)
    size = C.c_int64()
    log = C.create_string_buffer(1 << 16)
    _check(load().kr_network_spec_compile(C.byref(d), C.byref(size), log, 1 << 16))
    return {"cubin_bytes": size.value, "log": log.value.decode()}


def wpc_compile(net, precision_mode: int = KR_FP64, warps_per_cell: int = 1, want_cubin: bool = False) -> dict:
    """kr_network_wpc_compile: NVRTC-compile the register-tile kernel for sm_100a (no GPU needed)."""
    d, keep = make_desc(net)
    size = C.c_int64()
    log = C.create_string_buffer(1 << 16)
    cap = (8 << 20) if want_cubin else 0
    img = C.create_string_buffer(cap) if want_cubin else None
    _check(load().kr_network_wpc_compile(C.byref(d), int(precision_mode), int(warps_per_cell), C.byref(size), log, 1 << 16,
                                         C.cast(img, C.c_void_p) if want_cubin else None, cap))
    out = {"cubin_bytes": size.value, "log": log.value.decode()}
    if want_cubin:
        out["cubin"] = img.raw[:size.value]
    return out


def row_compile(net, warps_per_cell: int = 1, want_cubin: bool = False) -> dict:
    """kr_network_row_compile: NVRTC-compile the row-per-lane kernel for sm_100a (no GPU needed)."""
    d, keep = make_desc(net)
    size = C.c_int64()
    log = C.create_string_buffer(1 << 16)
    cap = (8 << 20) if want_cubin else 0
    img = C.create_string_buffer(cap) if want_cubin else None
    _check(load().kr_network_row_compile(C.byref(d), int(warps_per_cell), C.byref(size), log, 1 << 16,
                                         C.cast(img, C.c_void_p) if want_cubin else None, cap))
    out = {"cubin_bytes": size.value, "log": log.value.decode()}
    if want_cubin:
        out["cubin"] = img.raw[:size.value]
    return out


class Network:
    """kr_network handle built from a ``workloads.Network``-shaped object (kr_network_create)."""

    def __init__(self, net, opts=None):
        lib = load()
        d, self._keep = make_desc(net)
        h = C.c_void_p()
        self._h = None
        _check(lib.kr_network_create(C.byref(d), C.byref(h)))
        self._h = h
        self.S = int(net.n_species)
        self.R = int(net.n_reac)
        self.energy = int(net.energy_equation)
        self.N = self.S + self.energy
        if opts is not None:
            self.set_options(opts)

    def close(self) -> None:
        if getattr(self, "_h", None):
            load().kr_network_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- configuration ------------------------------------------------------------------------
    def set_options(self, opts) -> None:
        o = opts if isinstance(opts, SolverOpts) else opts_from(opts)
        _check(load().kr_network_set_options(self._h, C.byref(o)))

    def get_options(self) -> SolverOpts:
        o = SolverOpts()
        _check(load().kr_network_get_options(self._h, C.byref(o)))
        return o

    def set_stream(self, cuda_stream: int) -> None:
        _check(load().kr_set_stream(self._h, C.c_void_p(cuda_stream)))

    def set_mapping(self, mapping: int, threads_per_cell: int = 0) -> None:
        _check(load().kr_network_set_mapping(self._h, int(mapping), int(threads_per_cell)))

    def set_tuning(self, stiffest_first: int = -1, host_chunks: int = 0) -> None:
        _check(load().kr_network_set_tuning(self._h, int(stiffest_first), int(host_chunks)))

    def info(self) -> dict:
        a, b, c, d = C.c_int32(), C.c_int32(), C.c_int32(), C.c_int32()
        _check(load().kr_network_info(self._h, C.byref(a), C.byref(b), C.byref(c), C.byref(d)))
        return {"n_unknowns": a.value, "mapping": b.value, "threads_per_cell": c.value, "smem_bytes": d.value}

    def kernel_desc(self) -> str:
        buf = C.create_string_buffer(1024)
        _check(load().kr_network_kernel_desc(self._h, buf, 1024))
        return buf.value.decode()

    def last_launch_count(self) -> int:
        return int(load().kr_last_launch_count(self._h))

    def last_mixed_stats(self) -> dict:
        a, b, c = C.c_int64(), C.c_int64(), C.c_int64()
        _check(load().kr_last_mixed_stats(self._h, C.byref(a), C.byref(b), C.byref(c)))
        return {"n_refine": int(a.value), "n_fp64_cells": int(b.value), "n_discarded_newton": int(c.value)}

    # -- the step -----------------------------------------------------------------------------
    def thermochem_step(self, n_cells: int, rho, T, y, dt: float, precision_mode: int = KR_FP64) -> None:
        """kr_thermochem_step: device tensors, in place, asynchronous on the handle's stream."""
        _check(load().kr_thermochem_step(self._h, int(n_cells), _ptr(rho), _ptr(T), _ptr(y), float(dt),
                                         int(precision_mode)))

    def thermochem_step_ex(self, n_cells: int, rho, T, y, dt: float, precision_mode: int = KR_FP64, aux=None,
                           status=None, want_stats: bool = False, stream: int = 0) -> Optional[dict]:
        """kr_thermochem_step_ex: device tensors; aux [n_aux, n_cells]; status int32 [n_cells]."""
        n_aux = 0 if aux is None else int(aux.shape[0])
        st = StepStats()
        _check(load().kr_thermochem_step_ex(self._h, int(n_cells), _ptr(rho), _ptr(T), _ptr(y), float(dt),
                                            int(precision_mode), _ptr(aux), n_aux, _ptr(status),
                                            C.byref(st) if want_stats else None, C.c_void_p(stream or None)))
        return st.as_dict() if want_stats else None

    def thermochem_step_host(self, n_cells: int, rho, T, y, dt: float, precision_mode: int = KR_FP64, aux=None,
                             status=None, want_stats: bool = False) -> Optional[dict]:
        """kr_thermochem_step_host: HOST buffers (numpy arrays or pinned CPU tensors), copies inside."""
        n_aux = 0 if aux is None else int(aux.shape[0])
        st = StepStats()
        _check(load().kr_thermochem_step_host(self._h, int(n_cells), _ptr(rho), _ptr(T), _ptr(y), float(dt),
                                              int(precision_mode), _ptr(aux), n_aux, _ptr(status),
                                              C.byref(st) if want_stats else None))
        return st.as_dict() if want_stats else None

    # -- the allocation-free variant (static device scratch; include/kratos_chem.h) ---------------
    def static_setup(self) -> None:
        _check(load().kr_static_setup(self._h))

    def static_max_cells(self) -> int:
        m = C.c_int64()
        _check(load().kr_static_max_cells(self._h, C.byref(m)))
        return int(m.value)

    def thermochem_step_static(self, n_cells: int, rho, T, y, dt: float, aux=None, status=None, want_stats: bool = False,
                               stream: int = 0) -> Optional[dict]:
        """kr_thermochem_step_static: as thermochem_step_ex in fp64, no allocation inside the call."""
        n_aux = 0 if aux is None else int(aux.shape[0])
        st = StepStats()
        _check(load().kr_thermochem_step_static(self._h, int(n_cells), _ptr(rho), _ptr(T), _ptr(y), float(dt),
                                                _ptr(aux), n_aux, _ptr(status), C.byref(st) if want_stats else None,
                                                C.c_void_p(stream or None)))
        return st.as_dict() if want_stats else None


def table_rates(ln_k, ln_rho0: float, d_ln_rho: float, ln_T0: float, d_ln_T: float, rho, T, k_out, stream: int = 0) -> None:
    """kr_table_rates: ln_k device tensor [n_tab, n_rho, n_T]; rho, T [n_cells]; k_out [n_tab, n_cells] (or rows of an aux array)."""
    n_tab, n_rho, n_T = (int(v) for v in ln_k.shape)
    _check(load().kr_table_rates(n_tab, n_rho, n_T, float(ln_rho0), float(d_ln_rho), float(ln_T0), float(d_ln_T), _ptr(ln_k),
                                 int(rho.shape[0]), _ptr(rho), _ptr(T), _ptr(k_out), C.c_void_p(stream or None)))


def static_scratch_bytes() -> int:
    return int(load().kr_static_scratch_bytes())


def math_probe(x, rcp, ex, n: int, stream: int = 0) -> None:
    _check(load().kr_math_probe(_ptr(x), _ptr(rcp), _ptr(ex), int(n), C.c_void_p(stream or None)))


def layout_cell_to_soa(y_cell, y_soa, n_cells: int, S: int, stream: int = 0) -> None:
    _check(load().kr_layout_cell_to_soa(_ptr(y_cell), _ptr(y_soa), int(n_cells), int(S), C.c_void_p(stream or None)))


def layout_soa_to_cell(y_soa, y_cell, n_cells: int, S: int, stream: int = 0) -> None:
    _check(load().kr_layout_soa_to_cell(_ptr(y_soa), _ptr(y_cell), int(n_cells), int(S), C.c_void_p(stream or None)))


class Recon:
    """kr_recon handle: the stoichiometric projector of a composition matrix and the species advection stage
    (section 2.1).  Argument marshalling only."""

    SCHEME_DONOR, SCHEME_PLM, SCHEME_PLM_PROJECTED = 0, 1, 2

    def __init__(self, composition):
        comp = _i32(composition)
        self.E, self.S = int(comp.shape[0]), int(comp.shape[1])
        h = C.c_void_p()
        _check(load().kr_recon_create(self.E, self.S, _i(comp), C.byref(h)))
        self._h = h

    def __del__(self):
        try:
            if getattr(self, "_h", None):
                load().kr_recon_destroy(self._h)
                self._h = None
        except Exception:
            pass

    def projector(self):
        P = np.zeros((self.S, self.S))
        rank = C.c_int32()
        _check(load().kr_recon_projector(self._h, _d(P), C.byref(rank)))
        return P, int(rank.value)

    def advect_species_1d(self, n_cells, y, rho, mass_flux, dt_over_dx, dx, scheme, periodic, y_out, rho_out=None,
                          wa=0.0, wb=1.0, y0=None, rho0=None, stream=None) -> None:
        _check(load().kr_advect_species_1d(self._h, int(n_cells), _ptr(y), _ptr(rho), _ptr(mass_flux), float(dt_over_dx), float(dx),
                                           int(scheme), int(bool(periodic)), float(wa), float(wb), _ptr(y0), _ptr(rho0),
                                           _ptr(y_out), _ptr(rho_out), stream))


def raytrace_cartesian(shape, spacing, n_rays, origins, directions, L_in, sigma, n_dens, k_out, L_out=None, path=None,
                       lower=None, stream=None) -> None:
    """kr_raytrace_cartesian: device tensors for the fields and rays, host arrays for spacing / lower / sigma."""
    sp = _f64(np.asarray(spacing, np.float64)); lo = None if lower is None else _f64(np.asarray(lower, np.float64))
    sg = _f64(np.asarray(sigma, np.float64))
    n_abs, n_bins = int(sg.shape[0]), int(sg.shape[1])
    _check(load().kr_raytrace_cartesian(int(shape[0]), int(shape[1]), int(shape[2]), _d(sp), _d(lo), int(n_rays), _ptr(origins),
                                        _ptr(directions), n_bins, _ptr(L_in), n_abs, _d(sg), _ptr(n_dens), _ptr(k_out),
                                        _ptr(L_out), _ptr(path), stream))
