"""table_oracle.py -- CPU ORACLE of the tabulated reaction rates.  TEST INFRASTRUCTURE.

What it is: a plain numpy / pure-Python restatement of PAPER.md:171 (rate type 3 of section 2.3): "Tabulated reactions with
numerically interpolated rates, where precomputed tables are read in ...  At the beginning of the thermochemical
computation, multi-dimensional tables are reduced to one-dimensional in T per cell, assuming fixed total mass density and
elemental abundances during thermochemical steps."  In the paper's order, for every cell:

    1. reduce: the table k(rho, T) is interpolated along rho at the cell's (fixed) density, at every T node -> a 1-D table
       in T that belongs to the cell;
    2. interpolate that 1-D table at the cell's temperature.

The result is the per-cell rate coefficient of the reaction; the chemistry step takes it as an aux row (KR_F_AUX_UNARY,
k = A * aux[row][cell]).  For an isothermal step the cell's T is fixed, so step 2 happens once per step.

Who may use it: tests/, __graft_entry__.smoke(), bench.py's cpu_baseline legs.  It shares no code with the CUDA path.

Readings: R32 the paper does not say how tables are interpolated: both directions are piecewise linear in the
LOGARITHMS (ln k against ln rho, then against ln T), on nodes uniformly spaced in ln rho and ln T; outside the table the
end value is used (no extrapolation).  R33 only density and temperature are table dimensions here (elemental abundances,
photon escape probabilities: not built); a network with an energy equation, whose T moves inside the step, would need the
interpolation inside the Newton loop: not built, the rates are taken at the cell's T at the start of the step.

Pins (tests/test_table_pins.py): node values are returned exactly; a power law k = A rho^a T^b is reproduced to rounding at
any (rho, T) inside the table (log-log-linear interpolation is exact for it); for an Arrhenius law the error stays under
the classical bound h^2 / 8 max |d2 ln k / d(ln T)2|; clamping outside; the reduce-then-interpolate order equals bilinear
interpolation; and the chemistry oracle driven by a tabulated Arrhenius rate reproduces the run with the analytic rate
within that bound.
"""
from __future__ import annotations

import math

import numpy as np


def reduce_to_1d(ln_k, ln_rho0: float, d_ln_rho: float, rho: float):
    """Step 1 for one cell: ln_k [n_rho, n_T] -> the cell's 1-D table [n_T] (linear in ln rho, clamped)."""
    ln_k = np.asarray(ln_k, dtype=np.float64)
    n_rho = ln_k.shape[0]
    if n_rho == 1:
        return ln_k[0].copy()
    x = (math.log(rho) - ln_rho0) / d_ln_rho
    x = min(max(x, 0.0), float(n_rho - 1))
    i = min(int(math.floor(x)), n_rho - 2)
    f = x - i
    return (1.0 - f) * ln_k[i] + f * ln_k[i + 1]


def interpolate_1d(tab, ln_T0: float, d_ln_T: float, T: float) -> float:
    """Step 2 for one cell: the 1-D table [n_T] at temperature T (linear in ln T, clamped); returns ln k."""
    n_T = len(tab)
    if n_T == 1:
        return float(tab[0])
    x = (math.log(T) - ln_T0) / d_ln_T
    x = min(max(x, 0.0), float(n_T - 1))
    j = min(int(math.floor(x)), n_T - 2)
    f = x - j
    return (1.0 - f) * float(tab[j]) + f * float(tab[j + 1])


def table_rates(ln_k, ln_rho0, d_ln_rho, ln_T0, d_ln_T, rho, T):
    """All cells, all tables.  ln_k [n_tab, n_rho, n_T]; rho, T [n_cells].  Returns k [n_tab, n_cells]."""
    ln_k = np.asarray(ln_k, dtype=np.float64)
    rho = np.asarray(rho, dtype=np.float64); T = np.asarray(T, dtype=np.float64)
    out = np.empty((ln_k.shape[0], rho.shape[0]))
    for c in range(rho.shape[0]):
        for t in range(ln_k.shape[0]):
            tab = reduce_to_1d(ln_k[t], ln_rho0, d_ln_rho, float(rho[c]))        # PAPER.md:171, "reduced to one-dimensional in T per cell"
            out[t, c] = math.exp(interpolate_1d(tab, ln_T0, d_ln_T, float(T[c])))
    return out
