"""Pins of the reconstruction / advection oracle (oracle/recon_oracle.py; section 2.1, test of section 4.1)
against things other than itself: textbook linear algebra, closed forms of the limiter, invariants of the scheme, and the
numbers the paper states for its four-species test.  CPU only."""
import os

import numpy as np
import pytest

from oracle import recon_oracle as R
from paper_2504_04941_b200 import workloads as w

HERE = os.path.dirname(os.path.abspath(__file__))


def _eq33():
    rows = []
    for line in open(os.path.join(HERE, "golden", "paper_eq33.txt")):
        if line.strip() and not line.startswith("#"):
            f = line.split()
            rows.append((float(f[1]), float(f[2]), float(f[3]), int(f[4]), int(f[5])))
    return rows


COMPS = [np.array([[1, 2, 1, 0], [0, 0, 1, 1]]), w.make_network(1).composition, w.make_network(2).composition,
         w.make_network(3).composition, w.make_network(4).composition]


@pytest.mark.parametrize("k", range(len(COMPS)))
def test_projector_is_the_orthogonal_projector_onto_the_null_space(k):
    """Eqs. 7-8: P = V V^T must equal the textbook projector I - N^T (N N^T)^-1 N onto null(N) (N has
    full row rank in every network here), hence N P = 0, P^2 = P = P^T, trace = S - rank."""
    N = COMPS[k].astype(np.float64)
    E, S = N.shape
    P = R.projector(N)
    ref = np.eye(S) - N.T @ np.linalg.solve(N @ N.T, N)
    assert np.abs(P - ref).max() < 1e-13
    assert np.abs(N @ P).max() < 1e-13 * np.abs(N).max()
    assert np.abs(P @ P - P).max() < 1e-13 and np.abs(P - P.T).max() < 1e-14
    assert abs(np.trace(P) - (S - np.linalg.matrix_rank(N))) < 1e-12
    # a rank-deficient matrix (a duplicated row) gives the same projector
    P2 = R.projector(np.vstack([N, N[:1]]))
    assert np.abs(P2 - P).max() < 1e-13


def test_projector_of_the_paper_test_network_by_hand():
    """Elements A, B; species A, A2, AB, B: null(N) is spanned by A2 - 2A and AB - A - B.  The projector onto that plane,
    worked out by Gram-Schmidt with exact arithmetic."""
    from fractions import Fraction as Fr
    v1 = [Fr(-2), Fr(1), Fr(0), Fr(0)]
    v2 = [Fr(-1), Fr(0), Fr(1), Fr(-1)]
    dot = lambda a, b: sum(x * y for x, y in zip(a, b))
    u2 = [b - dot(v2, v1) / dot(v1, v1) * a for a, b in zip(v1, v2)]
    Pex = [[v1[i] * v1[j] / dot(v1, v1) + u2[i] * u2[j] / dot(u2, u2) for j in range(4)] for i in range(4)]
    P = R.projector(np.array([[1, 2, 1, 0], [0, 0, 1, 1]]))
    assert np.abs(P - np.array([[float(x) for x in row] for row in Pex])).max() < 1e-15


def test_limiter_closed_forms():
    """Eq. 12 (reading R25): zero at extrema; the harmonic mean on a uniform grid; symmetric under a <-> b with
    c_f <-> c_b; bounded by c_f |a| and c_b |b| (monotonicity, what the paper's limiter is for) on grids whose zone
    widths change by less than a factor ~2 between neighbours; odd in (a, b)."""
    rng = np.random.default_rng(5)
    a = rng.normal(size=4000) * 10.0 ** rng.uniform(-8, 3, 4000)
    b = rng.normal(size=4000) * 10.0 ** rng.uniform(-8, 3, 4000)
    phi = R.limited_slope(a, b)
    same = a * b > 0
    assert np.all(phi[~same] == 0.0)
    np.testing.assert_allclose(phi[same], 2 * a[same] * b[same] / (a[same] + b[same]), rtol=1e-14)
    np.testing.assert_allclose(R.limited_slope(-a, -b), -phi, rtol=0, atol=0)
    for cf, cb in ((2.0, 2.0), (1.5, 3.0), (3.0, 1.6), (4.0, 4.0)):     # c = 1 + ratio of neighbouring zone widths
        p = R.limited_slope(a, b, cf, cb)
        np.testing.assert_allclose(p, R.limited_slope(b, a, cb, cf), rtol=1e-14)
        assert np.all(np.abs(p[same]) <= np.minimum(cf * np.abs(a[same]), cb * np.abs(b[same])) * (1 + 1e-14))
        assert np.all(np.sign(p[same]) == np.sign(a[same]))
    # equal slopes: the slope itself, whatever the geometry (second order on smooth data)
    np.testing.assert_allclose(R.limited_slope(a, a, 1.3, 2.9), a, rtol=1e-14)


@pytest.mark.parametrize("scheme", [R.DONOR, R.PLM, R.PLM_PROJECTED])
def test_interface_states_keep_the_upwind_cells_element_totals(scheme):
    """Eq. 13 in eq. 14: with the projected correction N y_{i-1/2} = N <y>_upwind to rounding, for ANY field (the
    correction lies in the stoichiometric space, eq. 7); plain PLM does not have the property."""
    comp, y, rho, flux = w.make_advection_batch(9, 3, 500, seed=4)
    P = R.projector(comp)
    yl = R.interface_states(y, flux, 1.0 / 500, scheme, P, True)
    up = np.where((flux > 0)[:, None], np.roll(y, 1, axis=0), y)
    err = np.abs((yl - up) @ comp.T.astype(float)) / (np.abs(up) @ np.abs(comp.T).astype(float))
    if scheme == R.PLM:
        assert err.max() > 1e-6
    else:
        assert err.max() < 5e-16
    if scheme == R.DONOR:
        np.testing.assert_array_equal(yl, up)                     # eq. 6 exactly
    # PLM states are second order: exact for a linear profile away from the ends
    lin = np.outer(np.arange(500) / 500.0, np.arange(1, 10)) + 1.0
    yl2 = R.interface_states(lin, np.ones(500), 1.0 / 500, R.PLM, P, False)
    np.testing.assert_allclose(yl2[2:-2], (lin + np.roll(lin, 1, axis=0))[2:-2] / 2, rtol=1e-14)


def test_one_stage_is_the_flux_form_update():
    """The update is in flux form: total mass and total species content change only through the end faces (periodic: not at
    all), and a uniform state stays uniform whatever the mass fluxes are."""
    comp, y, rho, flux = w.make_advection_batch(7, 2, 300, seed=9)
    P = R.projector(comp)
    for scheme in (R.DONOR, R.PLM, R.PLM_PROJECTED):
        y1, r1 = R.advect_stage(y, rho, flux, 0.1, 1.0 / 300, scheme, P)
        assert abs(r1.sum() - rho.sum()) < 1e-12 * rho.sum()
        np.testing.assert_allclose((r1[:, None] * y1).sum(axis=0), (rho[:, None] * y).sum(axis=0), rtol=1e-13)
        yu = np.tile(y[:1], (300, 1))
        y2, _ = R.advect_stage(yu, rho, flux, 0.1, 1.0 / 300, scheme, P)
        np.testing.assert_allclose(y2, yu, rtol=1e-13)
    # donor cell, constant velocity v > 0, CFL number c: y_i <- (1 - c) y_i + c y_{i-1}
    c = 0.3
    y3, r3 = R.advect_stage(y, np.ones(300), np.ones(300), c, 1.0 / 300, R.DONOR, P)
    np.testing.assert_allclose(y3, (1 - c) * y + c * np.roll(y, 1, axis=0), rtol=1e-14)
    np.testing.assert_array_equal(r3, np.ones(300))


def test_paper_four_species_advection_test():
    """PAPER.md:400-417 (eq. 33, Fig. 3): 128 zones, periodic, rho = 1, v = 1, t = 1 (~300 steps).  'uncorrected PLM
    introduces substantial element A conservation errors (~1e-3 per ~300 step) ... both donor-cell and corrected PLM
    schemes maintain species conservation within machine precision (<~ 1e-15 relative error)'; 'PLM significantly reduces
    numerical diffusion compared to donor-cell approaches, regardless of conservation corrections'."""
    comp, x, y0, rho, dx = w.advection_test_case(128, _eq33())
    Nm = comp.astype(np.float64)
    tot0 = y0 @ Nm.T
    assert np.abs(tot0 - tot0[0]).max() < 1e-15                  # eq. 3: uniform element abundances (0.90 and 0.10)
    assert tot0[0] == pytest.approx([0.90, 0.10], abs=1e-15)
    P = R.projector(comp)
    res = {}
    for scheme in (R.DONOR, R.PLM, R.PLM_PROJECTED):
        y, steps = R.run_ssp_rk2(y0, rho, 1.0, dx, 1.0, 0.4, scheme, P)
        assert 250 <= steps <= 400
        elem_err = np.abs(y @ Nm.T - tot0) / tot0
        l1 = np.abs(y - y0).mean(axis=0)
        res[scheme] = (elem_err.max(axis=0), l1)
        np.testing.assert_allclose(y.sum(axis=0), y0.sum(axis=0), rtol=1e-13)       # flux form: totals exact
    assert res[R.DONOR][0].max() < 2e-14 and res[R.PLM_PROJECTED][0].max() < 2e-14
    assert 1e-4 < res[R.PLM][0][0] < 2e-2                         # element A drifts by ~1e-3 without the projection
    # PLM is much less diffusive than donor cell, with or without the projection, and the two PLM curves nearly overlap
    assert np.all(res[R.PLM][1][:2] < 0.5 * res[R.DONOR][1][:2])
    assert np.all(res[R.PLM_PROJECTED][1][:2] < 0.5 * res[R.DONOR][1][:2])
    assert np.all(np.abs(res[R.PLM_PROJECTED][1][:2] - res[R.PLM][1][:2]) < 0.25 * res[R.PLM][1][:2])
