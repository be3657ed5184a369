"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/kratos_chem.h declares,
its host logic (defaults, validation, error reporting) works, and it refuses to compute without a GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2504_04941_b200 import workloads as w
from tests import helpers as H

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2504_04941_b200 import build as bld
    bld.build_library()
    from paper_2504_04941_b200 import binding
    binding.load()
    return binding


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "kratos_chem.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(kr_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(B):
    names = _declared_functions()
    assert len(names) >= 15
    lib = B.load()
    for name in names:
        assert hasattr(lib, name), f"{name} declared in include/kratos_chem.h but not exported"
    assert sorted(B.EXPORTS) == names
    assert b"sm_100a" in lib.kr_version()


def test_default_options_match_design(B):
    o = B.default_opts()
    ref = w.SolverOpts()
    for name, _ in B.SolverOpts._fields_:
        assert getattr(o, name) == getattr(ref, name), name


def test_struct_layouts_match_header(B):
    # kr_network_desc: 3 int32 (+pad), 16 pointers, 2 doubles, 1 int32 (+pad); kr_solver_opts / kr_step_stats
    assert C.sizeof(B.NetworkDesc) == 16 + 16 * 8 + 16 + 8
    assert C.sizeof(B.StepStats) == 48
    assert C.sizeof(B.SolverOpts) == 16 + 11 * 8 + 16 + 16 + 16 + 8


def test_validation_runs_on_the_host_before_any_device_work(B):
    import torch
    # a reaction that does not conserve the composition matrix: a + b -> a2
    bad = H.tiny_network([[1, 0, 2], [0, 1, 0]], [((0, 1), (2,), 1e-10, 0.0, 0.0, 0, -1)])
    with pytest.raises(B.KrError) as e:
        B.Network(bad)
    assert e.value.code == B.KR_ENETWORK and "conserve" in str(e.value)
    # order 4 on one side (R20)
    bad2 = H.tiny_network([[1, 4]], [((0, 0, 0), (1,), 1e-10, 0.0, 0.0, 0, -1)])
    bad2.reac_nu[0, 0] = 4
    with pytest.raises(B.KrError) as e:
        B.Network(bad2)
    assert e.value.code == B.KR_ENETWORK
    # aux-scaled rate without an aux row
    bad3 = H.tiny_network([[1, 1]], [((0,), (1,), 1.0, 0.0, 0.0, w.F_AUX_UNARY, -1)])
    with pytest.raises(B.KrError) as e:
        B.Network(bad3)
    assert e.value.code == B.KR_ENETWORK
    if not torch.cuda.is_available():
        # a valid network: without a device the library must refuse, not fall back to the CPU
        with pytest.raises(B.KrError) as e:
            B.Network(w.make_network(0))
        assert e.value.code == B.KR_ECUDA and "no CPU path" in str(e.value)


@pytest.mark.parametrize("idx", [0, 1, 2])
def test_specialised_kernel_compiles_for_sm100a_without_a_gpu(B, idx):
    """The run-time compiled path (NVRTC) is checked at build time: source generation + compilation need no GPU."""
    net = w.make_network(idx)
    src = B.spec_source(net)
    assert "struct KrNet" in src and f"S = {net.n_species}" in src and f"R = {net.n_reac}" in src
    out = B.spec_compile(net)
    assert out["cubin_bytes"] > 10000
    assert "error" not in out["log"].lower()


@pytest.mark.parametrize("idx,mode,warps", [(3, 0, 1), (3, 1, 1), (4, 0, 2), (4, 1, 1), (1, 1, 1)])
def test_register_tile_kernel_compiles_for_sm100a_without_a_gpu(B, idx, mode, warps):
    """csrc/kr_wpc.cuh (warp-per-cell, matrix in register tiles; fp64 and mixed precision) is compiled by NVRTC for
    the sizes of the network at kr_network_create; the same compilation is checked here without a GPU.  The
    static_assert inside the kernel ties the host's shared-memory layout to the device's."""
    out = B.wpc_compile(w.make_network(idx), mode, warps)
    assert out["cubin_bytes"] > 10000
    assert "error" not in out["log"].lower()
    assert "tiles" in out["log"]


@pytest.mark.parametrize("idx,warps", [(3, 1), (4, 2), (1, 1), (0, 2), (2, 1)])
def test_row_per_lane_kernel_compiles_for_sm100a_without_a_gpu(B, idx, warps):
    """csrc/kr_row.cuh (warp-per-cell, one matrix row per lane, fp64) is compiled by NVRTC for the sizes of the network at
    kr_network_create; the same compilation is checked here without a GPU: N = 33 on one warp with the T row spread over
    the lanes, N = 64 on two warps, and small networks that leave lanes idle.  The static_asserts inside the kernel tie the
    host's shared-memory layout and term-stream indices to the device's."""
    out = B.row_compile(w.make_network(idx), warps)
    assert out["cubin_bytes"] > 10000
    assert "error" not in out["log"].lower()
    with pytest.raises(B.KrError):
        B.row_compile(w.make_network(4), 1)              # 64 rows do not fit one warp


def test_null_and_nonsense_arguments(B):
    lib = B.load()
    assert lib.kr_network_create(None, None) == B.KR_EINVAL
    assert lib.kr_network_set_options(None, None) == B.KR_EINVAL
    assert lib.kr_thermochem_step(None, 0, None, None, None, 1.0, 0) == B.KR_EINVAL
    assert lib.kr_layout_cell_to_soa(None, None, -1, 3, None) == B.KR_EINVAL
    assert lib.kr_last_launch_count(None) == 0
    assert len(lib.kr_last_error()) > 0


def test_binding_has_no_cpu_fallback():
    src = open(os.path.join(ROOT, "paper_2504_04941_b200", "binding.py")).read()
    assert "oracle" not in src.replace("no CPU fallback", "")
    for f in os.listdir(os.path.join(ROOT, "paper_2504_04941_b200", "csrc")):
        assert "oracle" not in open(os.path.join(ROOT, "paper_2504_04941_b200", "csrc", f)).read().lower().replace(
            "the oracle's", "").replace("oracle/", ""), f


@pytest.mark.parametrize("idx", [0, 1, 2, 3, 4])
def test_recon_projector_host_svd(B, idx):
    """kr_recon_create builds P = V V^T (eq. 8) on the host with its own one-sided Jacobi SVD -- no GPU
    needed: against the textbook projector onto null(N), and the rank of N."""
    N = w.make_network(idx).composition.astype(np.float64)
    P, rank = B.Recon(N.astype(np.int32)).projector()
    ref = np.eye(N.shape[1]) - N.T @ np.linalg.solve(N @ N.T, N)
    assert rank == np.linalg.matrix_rank(N)
    assert np.abs(P - ref).max() < 1e-13 and np.abs(N @ P).max() < 1e-13 and np.abs(P @ P - P).max() < 1e-13
    P2, rank2 = B.Recon(np.vstack([N, N[:1]]).astype(np.int32)).projector()       # rank-deficient input
    assert rank2 == rank and np.abs(P2 - P).max() < 1e-13
