"""GPU parity of the Cartesian ray tracer (section 3) against the Python oracle
(oracle/ray_oracle.py) through the C ABI: rate fields, depleted photon counts and path lengths ray by ray and cell by
cell, plane-parallel and oblique rays, rays that miss the mesh, and the traced rate driving the chemistry step of config 2
to the ionisation balance of eq. 35."""
import numpy as np
import pytest

from oracle import ray_oracle as RT
from paper_2504_04941_b200 import workloads as w

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2504_04941_b200 import binding
    binding.load()
    return binding


def gpu_trace(B, case):
    import torch
    t = lambda a: torch.tensor(np.ascontiguousarray(a), device="cuda")
    n_abs = case["sigma"].shape[0]
    nd = t(case["n_dens"].reshape(n_abs, -1))
    k = torch.full_like(nd, -1.0)                       # the call overwrites it
    org, drc, L = t(case["origins"]), t(case["directions"]), t(case["L"])
    Lo = torch.empty_like(L); path = torch.empty(org.shape[0], dtype=torch.float64, device="cuda")
    B.raytrace_cartesian(case["shape"], case["spacing"], org.shape[0], org, drc, L, case["sigma"], nd, k, Lo, path)
    torch.cuda.synchronize()
    return k.cpu().numpy().reshape(case["n_dens"].shape), Lo.cpu().numpy(), path.cpu().numpy()


@pytest.mark.parametrize("shape,n_obl,n_abs,n_bins,columns", [((16, 12, 10), 200, 3, 4, True), ((7, 5, 3), 500, 1, 1, False),
                                                               ((33, 1, 1), 3, 2, 16, True), ((4, 4, 4), 0, 8, 2, True),
                                                               ((1, 1, 1), 40, 2, 3, True)])
def test_raytrace_parity(B, shape, n_obl, n_abs, n_bins, columns):
    case = w.make_ray_case(shape=shape, n_oblique=n_obl, n_abs=n_abs, n_bins=n_bins, columns=columns, seed=77 + shape[0])
    ko, Lo, po = RT.trace(case["origins"], case["directions"], case["L"], case["sigma"], case["n_dens"], case["shape"], case["spacing"])
    kg, Lg, pg = gpu_trace(B, case)
    np.testing.assert_allclose(pg, po, rtol=1e-12, atol=1e-13)                 # same cells, same lengths
    assert np.array_equal(pg == 0.0, po == 0.0)                                # the same rays miss
    np.testing.assert_allclose(Lg, Lo, rtol=1e-11, atol=1e-300)
    # the rate of a cell is a sum over rays and bins: relative to the cell's total
    np.testing.assert_allclose(kg, ko, rtol=1e-11, atol=1e-13 * ko.max())
    # photon conservation on the GPU result itself (eq. 30)
    dV = np.prod(case["spacing"])
    assert (kg * case["n_dens"]).sum() * dV == pytest.approx((case["L"] - Lg).sum(), rel=1e-11)


def test_traced_rate_feeds_the_chemistry_step(B, oracle_mod):
    """The tracer's k field for hydrogen is handed to kr_thermochem_step_ex as config 2's aux row: both calls on the GPU,
    result against the chemistry oracle fed the oracle's traced rate."""
    import torch
    from tests import helpers as H
    net = w.make_network(2)
    names = list(net.species_names)
    iH, iHp, ie = names.index("H"), names.index("H+"), names.index("e-")
    shape, h = (64, 4, 4), (3.0e17, 3.0e17, 3.0e17)
    n_cells = 64 * 16
    rng = np.random.default_rng(12)
    xn = rng.uniform(0.01, 0.9, size=shape)
    nH = 100.0
    case = dict(shape=shape, spacing=h, n_dens=(nH * xn)[None], sigma=np.array([[6.3e-18]]),
                origins=np.array([[-1.0, (j + 0.5) * h[1], (k + 0.5) * h[2]] for j in range(4) for k in range(4)]),
                directions=np.tile([1.0, 0, 0], (16, 1)), L=np.full((16, 1), 1.0e11 * h[1] * h[2]))
    ko, _, _ = RT.trace(case["origins"], case["directions"], case["L"], case["sigma"], case["n_dens"], shape, h)
    kg, _, _ = gpu_trace(B, case)
    np.testing.assert_allclose(kg, ko, rtol=1e-12)
    y = np.zeros((n_cells, net.n_species)); xf = xn.reshape(-1)
    y[:, iH] = xf; y[:, iHp] = 1 - xf; y[:, ie] = 1 - xf
    cells = H.cells_of(nH * H.M_U * np.ones(n_cells), 8000.0, y, 1.0e12, aux=ko.reshape(1, -1))
    opts = w.default_opts(2)
    To, yo, sto, _, _ = oracle_mod.OracleNetwork(net, opts).step(cells, n_threads=8)
    gn = B.Network(net, opts)
    dev = "cuda"
    rho = torch.tensor(cells.rho, device=dev); T = torch.tensor(cells.T, device=dev); yd = torch.tensor(cells.y, device=dev)
    aux = torch.tensor(kg.reshape(1, -1), device=dev)
    st = torch.zeros(n_cells, dtype=torch.int32, device=dev)
    gn.thermochem_step_ex(n_cells, rho, T, yd, cells.dt, B.KR_FP64, aux=aux, status=st)
    torch.cuda.synchronize()
    ok = (sto & 8) == 0
    rel = np.abs(yd.cpu().numpy() - yo) / np.maximum(np.abs(yo), 1e-20)
    assert ok.all() and np.median(rel.max(axis=1)) < 1e-11 and (rel.max(axis=1) < 1e-9).mean() > 0.99


def test_raytrace_argument_errors(B):
    import torch
    case = w.make_ray_case(shape=(4, 4, 4), n_oblique=4)
    nd = torch.tensor(case["n_dens"].reshape(3, -1), device="cuda"); k = torch.empty_like(nd)
    o = torch.tensor(case["origins"], device="cuda"); d = torch.tensor(case["directions"], device="cuda"); L = torch.tensor(case["L"], device="cuda")
    with pytest.raises(B.KrError):
        B.raytrace_cartesian((4, 4, 4), (0.0, 1, 1), o.shape[0], o, d, L, case["sigma"], nd, k)
    with pytest.raises(B.KrError):
        B.raytrace_cartesian((4, 4, 4), (1, 1, 1), o.shape[0], o, d, L, np.ones((9, 2)), nd, k)
    B.raytrace_cartesian((4, 4, 4), (1, 1, 1), 0, o, d, L, case["sigma"], nd, k)       # no rays: k = 0
    torch.cuda.synchronize()
    assert float(k.abs().max()) == 0.0
