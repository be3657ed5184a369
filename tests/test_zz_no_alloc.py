"""GPU test of the allocation-free step (kr_thermochem_step_static, include/kratos_chem.h): its scratch is a file-scope static
device array, so the call makes no cudaMalloc.  It runs the same kernels as kr_thermochem_step_ex, so the bar is the one the
other same-kernel comparisons of this suite use: identical bits in T, y, status and identical solver counters -- on two calls
in a row (the second on another, smaller batch, so that whatever the first call left in the shared scratch would show), for a
network with an energy equation (config 1: counters only) and an isothermal one (config 2: counters + the preliminary
kernel's workspace).  The file sorts last on purpose: the suite runs with pytest -x."""
import numpy as np
import pytest

from paper_2504_04941_b200 import workloads as w

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2504_04941_b200 import binding
    binding.load()          # raises when libkratos_chem.so is missing: no fallback
    return binding


def _device_state(cells):
    import torch
    dev = "cuda:0"
    rho = torch.tensor(cells.rho, device=dev); T = torch.tensor(cells.T, device=dev); y = torch.tensor(cells.y, device=dev)
    aux = None if cells.aux is None else torch.tensor(cells.aux, device=dev)
    st = torch.full((max(cells.n_cells, 1),), -1, dtype=torch.int32, device=dev)
    return rho, T, y, aux, st


@pytest.mark.parametrize("idx,sizes", [(1, (1531, 389)), (2, (5003, 1021))])
def test_static_step_equals_existing_path_twice(B, idx, sizes):
    import torch
    net, _, opts = w.make_config(idx, sizes[0])
    ref_net = B.Network(net, opts)
    sta_net = B.Network(net, opts)
    sta_net.static_setup()
    assert sta_net.static_max_cells() >= max(sizes)
    for call, n in enumerate(sizes):                       # two calls in a row on the shared scratch
        _, cells, _ = w.make_config(idx, n, seed=1234 + call)
        rho, T0, y0, aux, s0 = _device_state(cells)
        stats0 = ref_net.thermochem_step_ex(n, rho, T0, y0, cells.dt, B.KR_FP64, aux=aux, status=s0, want_stats=True)
        rho, T1, y1, aux, s1 = _device_state(cells)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        stats1 = sta_net.thermochem_step_static(n, rho, T1, y1, cells.dt, aux=aux, status=s1, want_stats=True)
        torch.cuda.synchronize()
        if call == 1:                                      # every lazy set-up of the process is behind us: the driver's
            assert torch.cuda.mem_get_info()[0] == free_before        # count of free device memory has not moved
        np.testing.assert_array_equal(y1.cpu().numpy(), y0.cpu().numpy())
        np.testing.assert_array_equal(T1.cpu().numpy(), T0.cpu().numpy())
        np.testing.assert_array_equal(s1.cpu().numpy(), s0.cpu().numpy())
        assert stats1 == stats0 and stats1["n_substeps"] >= n
        assert not np.array_equal(y1.cpu().numpy(), cells.y)          # the step did something


def test_static_step_rejects_what_does_not_fit(B):
    import torch
    net, cells, opts = w.make_config(2, 64)
    gn = B.Network(net, opts)
    gn.static_setup()
    limit = gn.static_max_cells()
    assert limit == (B.static_scratch_bytes() - 256) // (8 * (2 * 9 + 1))
    rho, T, y, aux, st = _device_state(cells)
    with pytest.raises(B.KrError, match="static scratch holds"):
        gn.thermochem_step_static(limit + 1, rho, T, y, cells.dt, aux=aux, status=st)
    # a network the specialised kernel does not serve is refused, not served some other way
    net3, _, opts3 = w.make_config(3, 8)
    with pytest.raises(B.KrError, match="specialised thread-per-cell"):
        B.Network(net3, opts3).static_setup()
    torch.cuda.synchronize()
