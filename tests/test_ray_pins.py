"""Pins of the ray-tracing oracle (oracle/ray_oracle.py; section 3, eqs. 23-24, 28-31) against things other than
itself: analytic chord lengths, brute-force sampling of the ray, Beer-Lambert in closed form, photon conservation, the
limits of eq. 28 / 30, and the hydrogen ionisation balance of eq. 35 driven by a traced rate.  CPU only."""
import math

import numpy as np
import pytest

from oracle import ray_oracle as RT
from paper_2504_04941_b200 import workloads as w


def test_chord_length_and_visited_cells():
    """Eq. 24 cell walk: the path lengths of a ray add up to the chord of the box (slab formula), every step is positive
    and at most the cell diagonal, consecutive cells share a face, edge or corner, and the midpoint of every segment lies
    in the cell the walk says it is in (brute force)."""
    case = w.make_ray_case(shape=(9, 7, 5), n_oblique=300, columns=True, spacing=(0.3, 0.2, 0.5))
    shape, h = case["shape"], np.asarray(case["spacing"])
    hi = h * np.asarray(shape)
    n_hit = 0
    for o, d in zip(case["origins"], case["directions"]):
        segs = RT.walk(o, d, shape, h)
        d = d / np.linalg.norm(d)
        # analytic chord: slab intersection
        t0, t1 = -math.inf, math.inf
        miss = False
        for a in range(3):
            if d[a] == 0:
                miss |= not (0 <= o[a] <= hi[a]); continue
            ta, tb = sorted(((0 - o[a]) / d[a], (hi[a] - o[a]) / d[a]))
            t0, t1 = max(t0, ta), min(t1, tb)
        if miss or t0 > t1 or t1 < 0:
            assert segs == []
            continue
        n_hit += 1
        chord = t1 - max(t0, 0.0)
        assert sum(s[3] for s in segs) == pytest.approx(chord, rel=1e-12, abs=1e-13)
        t = max(t0, 0.0)
        prev = None
        for (i, j, k, dl) in segs:
            assert 0 <= i < shape[0] and 0 <= j < shape[1] and 0 <= k < shape[2]
            assert 0.0 <= dl <= np.linalg.norm(h) * (1 + 1e-12)
            if dl > 1e-9:
                mid = o + (t + 0.5 * dl) * d
                assert tuple(np.floor(mid / h).astype(int)) == (i, j, k)
            if prev is not None:
                assert max(abs(i - prev[0]), abs(j - prev[1]), abs(k - prev[2])) == 1
            prev = (i, j, k); t += dl
    assert n_hit > 200
    # axis-aligned rays through column centres cross nx cells of length dx each
    segs = RT.walk([-1.0, 0.1, 0.25], [1, 0, 0], shape, h)
    assert [s[:3] for s in segs] == [(i, 0, 0) for i in range(shape[0])]
    assert all(s[3] == pytest.approx(h[0], rel=1e-14) for s in segs)
    # a ray that starts inside the mesh starts in its own cell; one along -x walks backwards
    segs = RT.walk([1.0, 0.5, 1.2], [-1, 0, 0], shape, h)
    assert [s[0] for s in segs] == [3, 2, 1, 0] and segs[0][3] == pytest.approx(0.1, rel=1e-12)


def test_thin_factor_limits():
    """(1 - e^-tau) / tau: 1 - tau/2 + tau^2/6 for small tau (eq. 28's optically thin limit), 1/tau for large tau."""
    for tau in (0.0, 1e-300, 1e-12, 1e-6, 1e-3):
        assert RT.thin_factor(tau) == pytest.approx(1 - tau / 2 + tau * tau / 6, rel=1e-9)
    for tau in (50.0, 745.0, 1e6):
        assert RT.thin_factor(tau) == pytest.approx(1 / tau, rel=1e-15)
    assert RT.thin_factor(0.7) == pytest.approx((1 - math.exp(-0.7)) / 0.7, rel=1e-15)


def test_beer_lambert_uniform_medium():
    """Uniform medium, one absorber, axis-aligned rays: L(x) = L0 exp(-n sigma x) (eq. 29 compounded), the rate in cell i
    is eq. 30 with the photons that reach it, and in the thin limit k = L sigma dl / dV."""
    shape, h = (20, 3, 2), (0.5, 0.4, 0.25)
    n, sig, L0 = 3.0, 0.17, 1.0e4
    nd = np.full((1,) + shape, n)
    org = [[-1.0, (j + 0.5) * h[1], (k + 0.5) * h[2]] for j in range(3) for k in range(2)]
    drc = [[1.0, 0, 0]] * 6
    k, L_out, path = RT.trace(np.array(org), np.array(drc), np.full((6, 1), L0), np.array([[sig]]), nd, shape, h)
    tau = n * sig * h[0]
    dV = h[0] * h[1] * h[2]
    assert np.allclose(L_out, L0 * math.exp(-tau * 20), rtol=1e-13) and np.allclose(path, 10.0)
    for i in range(20):
        expect = L0 * math.exp(-tau * i) * (1 - math.exp(-tau)) / (n * dV)
        assert np.allclose(k[0, i], expect, rtol=1e-13)
    k2, _, _ = RT.trace(np.array(org), np.array(drc), np.full((6, 1), L0), np.array([[sig * 1e-9]]), nd, shape, h)
    assert np.allclose(k2[0], L0 * sig * 1e-9 * h[0] / dV, rtol=1e-7)


def test_photon_conservation_cell_by_cell():
    """Eq. 30's first equality summed over species, rays and bins: sum_i k_i n_i dV (photons absorbed per second in the
    mesh) equals what the rays lost, sum_jk (L_in - L_out), for any densities, cross sections and directions; and with two
    absorbers the absorbed photons split in proportion to n_i sigma_ik."""
    case = w.make_ray_case(shape=(8, 6, 5), n_oblique=80, n_abs=3, n_bins=4)
    k, L_out, path = RT.trace(case["origins"], case["directions"], case["L"], case["sigma"], case["n_dens"], case["shape"],
                              case["spacing"])
    dV = np.prod(case["spacing"])
    absorbed = (k * case["n_dens"]).sum() * dV
    lost = (case["L"] - L_out).sum()
    assert absorbed == pytest.approx(lost, rel=1e-12)
    assert (L_out <= case["L"]).all() and (L_out >= 0).all() and (k >= 0).all()
    missed = path == 0.0
    assert missed.any() and np.array_equal(L_out[missed], case["L"][missed])
    # one bin, one cell: shares proportional to n sigma
    nd = np.array([2.0, 5.0]).reshape(2, 1, 1, 1); sg = np.array([[0.3], [0.05]])
    k1, Lo, _ = RT.trace(np.array([[-1.0, 0.5, 0.5]]), np.array([[1.0, 0, 0]]), np.array([[7.0]]), sg, nd, (1, 1, 1), (1.0, 1.0, 1.0))
    got = k1[:, 0, 0, 0] * nd[:, 0, 0, 0]
    assert got[0] / got[1] == pytest.approx(2.0 * 0.3 / (5.0 * 0.05), rel=1e-14)
    assert got.sum() == pytest.approx(7.0 * (1 - math.exp(-(2.0 * 0.3 + 5.0 * 0.05))), rel=1e-14)


def test_traced_rate_drives_the_ionisation_balance(oracle_mod):
    """the chemistry step fed with a TRACED photoionisation rate reaches the balance of eq. 35,
    0 = alpha n x^2 - k_ci n x (1 - x) - Gamma (1 - x), cell by cell along a ray through a slab -- the rate the tracer
    hands over is the F sigma of that equation."""
    from tests import helpers as H
    net = w.make_network(2)
    shape, h = (12, 1, 1), (3.0e17, 3.0e17, 3.0e17)                      # cm
    nH = 100.0
    x_neutral = np.linspace(0.02, 0.9, 12)                                # neutral fractions along the ray
    nd = (nH * x_neutral).reshape(1, 12, 1, 1)
    sig = np.array([[6.3e-18]])
    L = np.array([[1.0e11 * h[1] * h[2]]])                                # photons / s through the column
    k, L_out, _ = RT.trace(np.array([[-1.0, 0.5 * h[1], 0.5 * h[2]]]), np.array([[1.0, 0, 0]]), L, sig, nd, shape, h)
    Gamma = k[0, :, 0, 0]
    assert (np.diff(Gamma) < 0).all() and Gamma[0] == pytest.approx(1.0e11 * 6.3e-18 * RT.thin_factor(nd[0, 0, 0, 0] * 6.3e-18 * h[0]), rel=1e-12)
    # hydrogen only (y_He = 0), long step: equilibrium x_e from the quadratic with eq. 36's coefficients
    T = 8000.0
    kf, _ = oracle_mod.OracleNetwork(net, w.default_opts(2)).rate_constants(T, np.array([1.0]))
    names = list(net.species_names)
    iH, iHp, ie = names.index("H"), names.index("H+"), names.index("e-")
    y = np.zeros((12, net.n_species)); y[:, iH] = 0.5; y[:, iHp] = 0.5; y[:, ie] = 0.5
    rho = nH * H.M_U * np.ones(12)                                         # y = n m_u / rho: y_H + y_H+ = 1
    cells = H.cells_of(rho, T, y, 1.0e18, aux=Gamma[None, :])
    opts = w.default_opts(2); opts.max_substeps = 100000
    To, yo, st, stats, _ = oracle_mod.OracleNetwork(net, opts).step(cells, n_threads=2)
    assert (st & 8 == 0).all()
    # identify alpha and k_ci from the network's own rate constants (eq. 36 rows of config 2)
    r_ci = [r for r in range(net.n_reac) if set(net.reac_idx[r][net.reac_idx[r] >= 0]) == {iH, ie}][0]
    r_rec = [r for r in range(net.n_reac) if set(net.reac_idx[r][net.reac_idx[r] >= 0]) == {iHp, ie}][0]
    kci, alpha = kf[r_ci], kf[r_rec]
    a_, b_, c_ = (alpha + kci) * nH, Gamma - kci * nH, -Gamma
    x_eq = (-b_ + np.sqrt(b_ * b_ - 4 * a_ * c_)) / (2 * a_)
    np.testing.assert_allclose(yo[:, ie], x_eq, rtol=2e-3)
