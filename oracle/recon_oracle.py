"""recon_oracle.py -- CPU ORACLE of the stoichiometry-compatible species reconstruction and advection.  TEST INFRASTRUCTURE.

What it is: a plain numpy (fp64) restatement of PAPER.md section 2.1 -- the species flux of eq. 1, the
donor-cell scheme of eq. 6, the stoichiometric projector P = V V^T from the SVD of the element-species
matrix, eqs. 7-8, the piecewise-linear interface states of eqs. 9-11 with the slope
limiter of eq. 12 (reading R25 of DESIGN.md), the projected states of eq. 13 and the
upwind choice of eq. 14 -- followed by the conservative update the Godunov scheme of PAPER.md:40 does
with those fluxes (step (3): "updating variables by adding the divergence of fluxes").  One function per equation, loops
over cells replaced by whole-array numpy expressions only where the expression is the printed formula.

Who may use it: tests/, __graft_entry__.smoke(), bench.py's cpu_baseline legs.  It shares no code with the CUDA path.

Pins (tests/test_recon_pins.py): P against the textbook projector I - N^T (N N^T)^-1 N, N P = 0, P^2 = P = P^T, rank;
the limiter against its uniform-grid closed form (harmonic mean), its bounds and its symmetry; eq. 13 keeps every
element total of the interface state equal to the upwind cell's; the four-species test of PAPER.md:400-417 (eq. 33):
element totals stay uniform to 1e-14 with the donor-cell and the projected scheme and drift by ~1e-3 with plain PLM.

Readings: R25 eq. 12 as printed returns a pure number, not a slope, and eq. 11's c_{i-1,f} has <xi>_{i-2} in
its denominator: read as the modified van Leer limiter of the reference the paper names (Mignone 2014) -- for forward
and backward slopes a, b and geometric factors c_f, c_b:  phi = a b (c_f b + c_b a) / (b^2 + (c_f + c_b - 2) a b + a^2)
when a b > 0, else 0, with c_f = (<xi>_{i+1} - <xi>_i) / (xi_{i+1/2} - <xi>_i), c_b = (<xi>_i - <xi>_{i-1}) /
(<xi>_i - xi_{i-1/2}) (both 2 on a uniform grid, where phi is the harmonic mean 2ab/(a+b)).  R26 the time integrator of
the test is not stated: the step here is ONE forward-Euler stage with optional convex-combination weights, so that the
driver can run SSP-RK2.  R28 open ends use zero-gradient ghost cells.  R27 x^s = n^s / rho is carried as y^s = n^s m_u / rho, the chemistry step's variable.
"""
from __future__ import annotations

import numpy as np

DONOR, PLM, PLM_PROJECTED = 0, 1, 2


def projector(composition: np.ndarray) -> np.ndarray:
    """Eq. 8: N = U Sigma V^T; P = V V^T over the right singular vectors that span the null space of N (eq. 7)."""
    N = np.asarray(composition, dtype=np.float64)
    _, sig, Vt = np.linalg.svd(N, full_matrices=True)
    tol = max(N.shape) * np.finfo(np.float64).eps * (sig.max() if sig.size else 1.0)
    rank = int((sig > tol).sum())
    V0 = Vt[rank:].T                              # [S, S - rank]: the stoichiometric space
    return V0 @ V0.T


def limited_slope(a, b, cf=2.0, cb=2.0):
    """Eq. 12 (reading R25): a = forward difference quotient, b = backward one; 0 at extrema."""
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    prod = a * b
    den = b * b + (cf + cb - 2.0) * prod + a * a
    with np.errstate(divide="ignore", invalid="ignore"):
        phi = prod * (cf * b + cb * a) / den
    return np.where(prod > 0.0, phi, 0.0)


def cell_corrections(y: np.ndarray, dx: float, scheme: int, P, periodic: bool) -> np.ndarray:
    """chi of eq. 10 for the RIGHT face of every cell, d_i = phi(...) * (xi_{i+1/2} - <xi>_i) = slope * dx / 2 (uniform
    grid); the left face gets -d_i.  With PLM_PROJECTED, d_i <- P d_i (eq. 13).  y is [n_cells, S]."""
    n, S = y.shape
    if scheme == DONOR:
        return np.zeros_like(y)
    if periodic:
        yp = np.roll(y, -1, axis=0); ym = np.roll(y, 1, axis=0)
    else:                                          # zero-gradient ends
        yp = np.vstack([y[1:], y[-1:]]); ym = np.vstack([y[:1], y[:-1]])
    a = (yp - y) / dx                              # eq. 11: forward and backward difference quotients
    b = (y - ym) / dx
    d = limited_slope(a, b) * (0.5 * dx)
    if scheme == PLM_PROJECTED:
        d = d @ np.asarray(P).T                    # eq. 13: sum_r P^s_r chi^r
    return d


def interface_states(y: np.ndarray, mass_flux: np.ndarray, dx: float, scheme: int, P, periodic: bool) -> np.ndarray:
    """Eqs. 9, 13, 14: the state at the LEFT face of every cell i (face i - 1/2), [n_cells, S]; mass_flux[i] is the mass
    flux through that face.  Theta(F) = 1 for F > 0 and 0 otherwise (eq. 6)."""
    d = cell_corrections(y, dx, scheme, P, periodic)
    if periodic:
        y_left = np.roll(y + d, 1, axis=0)         # cell i - 1 seen from its right face
    else:                                          # open end: a zero-gradient ghost cell (its own correction is 0)
        y_left = np.vstack([y[:1], (y + d)[:-1]])
    y_right = y - d                                # cell i seen from its left face
    up = (np.asarray(mass_flux) > 0.0)[:, None]
    return np.where(up, y_left, y_right)


def advect_stage(y, rho, mass_flux, dt_over_dx, dx, scheme, P, periodic=True, wa=0.0, wb=1.0, y0=None, rho0=None):
    """One forward-Euler stage of the Godunov update (PAPER.md:40 step 3) for rho and rho*y with the fluxes of eq. 1,
    F^s = y_{i-1/2} F^rho, optionally blended with an earlier state: U_out = wa U0 + wb (U - lambda dF).  mass_flux has
    n_cells entries (periodic: face i - 1/2 of cell i; the right face of the last cell is the left face of the first) or
    n_cells + 1.  Returns (y_out, rho_out)."""
    y = np.asarray(y, dtype=np.float64); rho = np.asarray(rho, dtype=np.float64)
    n = y.shape[0]
    f = np.asarray(mass_flux, dtype=np.float64)
    f_left = f[:n]
    f_right = np.roll(f[:n], -1) if f.shape[0] == n else f[1:]
    yl = interface_states(y, f_left, dx, scheme, P, periodic)
    if f.shape[0] == n:
        yr = np.roll(yl, -1, axis=0)
    else:                                          # open right end: the state at the last face
        d = cell_corrections(y, dx, scheme, P, periodic)
        last = np.where(f[n] > 0.0, (y + d)[-1], y[-1])          # ghost cell beyond the right end
        yr = np.vstack([yl[1:], last[None, :]])
    rho_new = rho - dt_over_dx * (f_right - f_left)
    u_new = rho[:, None] * y - dt_over_dx * (yr * f_right[:, None] - yl * f_left[:, None])
    if y0 is not None:
        rho_new = wa * np.asarray(rho0) + wb * rho_new
        u_new = wa * np.asarray(rho0)[:, None] * np.asarray(y0) + wb * u_new
    return u_new / rho_new[:, None], rho_new


def run_ssp_rk2(y, rho, velocity, dx, t_end, cfl, scheme, P):
    """Driver of the test of PAPER.md:400-417: constant velocity, periodic, SSP-RK2 (reading R26).  Returns (y, steps)."""
    y = np.array(y, dtype=np.float64); rho = np.array(rho, dtype=np.float64)
    n = y.shape[0]
    steps = int(np.ceil(t_end * abs(velocity) / (cfl * dx)))
    lam = (t_end / steps) / dx
    for _ in range(steps):
        f = rho * velocity                         # upwind mass flux through the left face of cell i
        f = np.roll(f, 1) if velocity > 0 else f
        y1, r1 = advect_stage(y, rho, f, lam, dx, scheme, P)
        f1 = r1 * velocity
        f1 = np.roll(f1, 1) if velocity > 0 else f1
        y, rho = advect_stage(y1, r1, f1, lam, dx, scheme, P, wa=0.5, wb=0.5, y0=y, rho0=rho)
    return y, steps
