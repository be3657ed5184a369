"""GPU parity of the species reconstruction / advection stage (section 2.1) against the
numpy oracle (oracle/recon_oracle.py), element by element, through the C ABI: every scheme, periodic and open grids,
ragged tile tails, the blend of a second Runge-Kutta stage, and the paper's four-species test run end to end on the GPU."""
import numpy as np
import pytest

from oracle import recon_oracle as R
from paper_2504_04941_b200 import workloads as w

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2504_04941_b200 import binding
    binding.load()
    return binding


def gpu_stage(B, rc, y, rho, flux, lam, dx, scheme, periodic, wa=0.0, wb=1.0, y0=None, rho0=None):
    import torch
    t = lambda a: None if a is None else torch.tensor(np.ascontiguousarray(a), device="cuda")
    dy, dr, df, dy0, dr0 = t(y), t(rho), t(flux), t(y0), t(rho0)
    yo = torch.empty_like(dy); ro = torch.empty_like(dr)
    rc.advect_species_1d(y.shape[0], dy, dr, df, lam, dx, scheme, periodic, yo, ro, wa, wb, dy0, dr0)
    torch.cuda.synchronize()
    return yo.cpu().numpy(), ro.cpu().numpy()


@pytest.mark.parametrize("scheme", [0, 1, 2])
@pytest.mark.parametrize("S,E,n", [(4, 2, 128), (9, 3, 1000), (9, 3, 257), (32, 5, 4099), (64, 6, 777), (5, 2, 3), (6, 3, 1)])
@pytest.mark.parametrize("periodic", [True, False])
def test_advection_stage_parity(B, S, E, n, scheme, periodic):
    comp, y, rho, flux = w.make_advection_batch(S, E, n, seed=100 + S + n)
    if not periodic:
        flux = np.concatenate([flux, flux[:1] * 0.7])
    P = R.projector(comp)
    rc = B.Recon(comp)
    dx, lam = 1.0 / n, 0.2
    yo, ro = R.advect_stage(y, rho, flux, lam, dx, scheme, P, periodic)
    yg, rg = gpu_stage(B, rc, y, rho, flux, lam, dx, scheme, periodic)
    # fp64 on both sides; the only freedom is the summation order of the S-term projection (which mixes species: its
    # rounding error scales with the LARGEST correction of the cell, whatever the species) and of the flux difference
    scale = np.abs(y).max(axis=0)[None, :] if scheme != 2 else np.abs(y).max()
    assert (np.abs(yg - yo) / scale).max() < 1e-14
    np.testing.assert_allclose(rg, ro, rtol=1e-15)
    # second stage of SSP-RK2: blend with the initial state
    yo2, ro2 = R.advect_stage(yo, ro, flux, lam, dx, scheme, P, periodic, wa=0.5, wb=0.5, y0=y, rho0=rho)
    yg2, rg2 = gpu_stage(B, rc, yo, ro, flux, lam, dx, scheme, periodic, 0.5, 0.5, y, rho)
    assert (np.abs(yg2 - yo2) / scale).max() < 1e-14
    np.testing.assert_allclose(rg2, ro2, rtol=1e-15)

def test_paper_four_species_test_on_the_gpu(B):
    """PAPER.md:400-417 end to end through kr_advect_species_1d (SSP-RK2, 320 steps): the GPU result equals the oracle's to
    rounding, element totals stay uniform to 1e-14 with the projection and drift by ~1e-4..1e-3 without it."""
    import torch
    comp, x, y0, rho0, dx = w.advection_test_case(128)
    Nm = comp.astype(np.float64); tot0 = y0 @ Nm.T
    P = R.projector(comp)
    rc = B.Recon(comp)
    steps = 320; lam = (1.0 / steps) / dx
    for scheme in (0, 1, 2):
        yo, _ = R.run_ssp_rk2(y0, rho0, 1.0, dx, 1.0, 0.4, scheme, P)
        y = torch.tensor(y0, device="cuda"); rho = torch.tensor(rho0, device="cuda")
        y1 = torch.empty_like(y); r1 = torch.empty_like(rho); y2 = torch.empty_like(y); r2 = torch.empty_like(rho)
        for _ in range(steps):
            f = torch.roll(rho, 1)                         # v = 1: upwind mass flux through the left face
            rc.advect_species_1d(128, y, rho, f, lam, dx, scheme, True, y1, r1)
            f1 = torch.roll(r1, 1)
            rc.advect_species_1d(128, y1, r1, f1, lam, dx, scheme, True, y2, r2, 0.5, 0.5, y, rho)
            y, y2 = y2, y; rho, r2 = r2, rho
        torch.cuda.synchronize()
        yg = y.cpu().numpy()
        assert np.abs(yg - yo).max() < 1e-12
        err = (np.abs(yg @ Nm.T - tot0) / tot0).max(axis=0)
        if scheme == 1:
            assert 1e-5 < err[0] < 2e-2
        else:
            assert err.max() < 2e-14


def test_advection_argument_errors(B):
    import torch
    comp, y, rho, flux = w.make_advection_batch(4, 2, 64)
    rc = B.Recon(comp)
    dy = torch.tensor(y, device="cuda"); dr = torch.tensor(rho, device="cuda"); df = torch.tensor(flux, device="cuda")
    out = torch.empty_like(dy)
    with pytest.raises(B.KrError):
        rc.advect_species_1d(64, dy, dr, df, 0.1, 1 / 64, 2, True, dy)          # aliasing
    with pytest.raises(B.KrError):
        rc.advect_species_1d(64, dy, dr, df, 0.1, 1 / 64, 7, True, out)         # scheme
    with pytest.raises(B.KrError):
        rc.advect_species_1d(64, dy, dr, df, 0.1, 0.0, 2, True, out)            # dx
    rc.advect_species_1d(0, dy, dr, df, 0.1, 1 / 64, 2, True, out)              # empty: no launch, no error
