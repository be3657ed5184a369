"""Pins of the tabulated-rate oracle (oracle/table_oracle.py, readings R32 / R33 of DESIGN.md) against what the
mathematics fixes -- none of them re-types the oracle's formula."""
import math

import numpy as np
import pytest

from oracle import table_oracle as TO
from paper_2504_04941_b200 import workloads as w


def _grid(n_rho=5, n_T=9):
    ln_rho0, d_ln_rho = math.log(1e-20), math.log(10.0)
    ln_T0, d_ln_T = math.log(100.0), math.log(2.0)
    lr = ln_rho0 + d_ln_rho * np.arange(n_rho); lt = ln_T0 + d_ln_T * np.arange(n_T)
    return ln_rho0, d_ln_rho, ln_T0, d_ln_T, lr, lt


def test_node_values_are_returned_exactly():
    ln_rho0, d_ln_rho, ln_T0, d_ln_T, lr, lt = _grid()
    rng = np.random.default_rng(5)
    ln_k = rng.uniform(-30.0, -5.0, (2, lr.size, lt.size))
    # cells placed on nodes: exact powers, so that log() lands on the node to rounding
    i, j = 3, 6
    k = TO.table_rates(ln_k, ln_rho0, d_ln_rho, ln_T0, d_ln_T, [math.exp(lr[i])], [math.exp(lt[j])])
    np.testing.assert_allclose(k[:, 0], np.exp(ln_k[:, i, j]), rtol=1e-12)


def test_power_law_is_reproduced_to_rounding():
    """k = A rho^a T^b is linear in (ln rho, ln T): piecewise-linear interpolation of its logarithm is exact anywhere."""
    ln_rho0, d_ln_rho, ln_T0, d_ln_T, lr, lt = _grid()
    A, a, b = 3.5e-12, 0.3, -0.75
    ln_k = (math.log(A) + a * lr[:, None] + b * lt[None, :])[None]
    rng = np.random.default_rng(6)
    rho = np.exp(rng.uniform(lr[0], lr[-1], 64)); T = np.exp(rng.uniform(lt[0], lt[-1], 64))
    k = TO.table_rates(ln_k, ln_rho0, d_ln_rho, ln_T0, d_ln_T, rho, T)
    np.testing.assert_allclose(k[0], A * rho ** a * T ** b, rtol=5e-13)


def test_arrhenius_error_stays_under_the_interpolation_bound():
    """ln k = c - Ea / T: d2 ln k / d(ln T)2 = -Ea / T, so |error in ln k| <= h^2 / 8 * Ea / T_min on every interval."""
    Ea, n_T = 1.578e5, 129
    lt = np.linspace(math.log(5e3), math.log(3e5), n_T); h = lt[1] - lt[0]
    ln_k = (-20.0 - Ea / np.exp(lt))[None, None, :]
    T = np.exp(np.random.default_rng(7).uniform(lt[0], lt[-1], 400))
    k = TO.table_rates(ln_k, 0.0, 1.0, lt[0], h, np.ones_like(T), T)[0]
    err = np.abs(np.log(k) - (-20.0 - Ea / T))
    bound = h * h / 8.0 * Ea / np.exp(lt[np.minimum(((np.log(T) - lt[0]) / h).astype(int), n_T - 2)])
    assert np.all(err <= bound * (1 + 1e-9) + 1e-13)
    assert err.max() > 0.05 * bound.max()          # the bound is not vacuous: the interpolation error is really there
    # the interpolant of a concave function lies below it
    assert np.all(np.log(k) <= (-20.0 - Ea / T) + 1e-12)


def test_clamped_outside_the_table():
    ln_rho0, d_ln_rho, ln_T0, d_ln_T, lr, lt = _grid()
    ln_k = np.random.default_rng(8).uniform(-30.0, -5.0, (1, lr.size, lt.size))
    k = TO.table_rates(ln_k, ln_rho0, d_ln_rho, ln_T0, d_ln_T, [1e-30, 1e10, math.exp(lr[2])], [1.0, 1e9, 1e9])
    np.testing.assert_allclose(k[0], np.exp([ln_k[0, 0, 0], ln_k[0, -1, -1], ln_k[0, 2, -1]]), rtol=1e-12)


def test_reduce_then_interpolate_equals_bilinear():
    """The paper's order (reduce to 1-D in T at the cell's density, then interpolate in T) gives the bilinear interpolant;
    the reference here is scipy's, a library routine the oracle does not call."""
    from scipy.interpolate import RegularGridInterpolator
    ln_rho0, d_ln_rho, ln_T0, d_ln_T, lr, lt = _grid()
    ln_k = np.random.default_rng(9).uniform(-30.0, -5.0, (lr.size, lt.size))
    rng = np.random.default_rng(10)
    rho = np.exp(rng.uniform(lr[0], lr[-1], 50)); T = np.exp(rng.uniform(lt[0], lt[-1], 50))
    k = TO.table_rates(ln_k[None], ln_rho0, d_ln_rho, ln_T0, d_ln_T, rho, T)[0]
    ref = RegularGridInterpolator((lr, lt), ln_k, method="linear")(np.stack([np.log(rho), np.log(T)], axis=1))
    np.testing.assert_allclose(np.log(k), ref, rtol=0, atol=1e-11)


def test_chemistry_oracle_on_a_tabulated_rate_matches_the_analytic_run():
    """Config 2 with its three recombination laws (power laws in T: tabulated exactly) and its three collisional
    ionisation laws (Arrhenius: tabulated with the error bound above) read from tables: the isothermal step with the
    tabulated rates equals the analytic one to the interpolation error."""
    from oracle import oracle as O
    import dataclasses
    net, cells, opts = w.make_config(2, 96)
    table = w.make_rate_table(net, [0, 1, 3, 4, 6, 7], T_range=(50.0, 2.0e5), n_T=4097)
    tnet = w.tabulated_network(net, table)
    k = TO.table_rates(table.ln_k, table.ln_rho0, table.d_ln_rho, table.ln_T0, table.d_ln_T, cells.rho, cells.T)
    tcells = dataclasses.replace(cells, aux=np.ascontiguousarray(np.concatenate([cells.aux, k], axis=0)))
    _, y_ref, st_ref, _, _ = O.OracleNetwork(net, opts).step(cells)
    _, y_tab, st_tab, _, _ = O.OracleNetwork(tnet, opts).step(tcells)
    scale = np.abs(y_ref).max(axis=1, keepdims=True)
    # h = ln(4000) / 4096 = 2e-3: the bound on ln k is 5e-7 * Ea / T, i.e. < 1e-4 wherever exp(-Ea / T) is not negligible
    err = np.max(np.abs(y_tab - y_ref) / scale)
    assert 0.0 < err < 1e-5                  # measured 9.5e-7
