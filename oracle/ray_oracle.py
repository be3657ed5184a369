"""ray_oracle.py -- CPU ORACLE of the Cartesian ray tracing and of the photo-reaction rates it feeds.  TEST INFRASTRUCTURE.

What it is: a plain, slow restatement (numpy scalars, pure-Python loops: small cases only) of PAPER.md section 3 --
the cell walk on a uniform Cartesian mesh, eqs. 23-24 (the exit point is the smallest positive
delta-l among the cell's surfaces, the propagation origin is updated to it, "iterative traversal until domain exit"),
the depletion of the photons of a ray, eq. 29, and the rate coefficient every absorbing species of a cell
receives from every ray and energy bin, eqs. 30-31:

    tau_jk = sum_i n_i sigma_ik dl_j ,   k_i += L_jk sigma_ik dl_j / dV * (1 - exp(-tau_jk)) / tau_jk ,
    L_jk <- L_jk exp(-tau_jk)            (the photons that enter the next cell, eq. 29)

in the order the paper states them, one ray after the other, one cell after the other.

Who may use it: tests/, __graft_entry__.smoke(), bench.py's cpu_baseline legs.  It shares no code with the CUDA path.

Pins (tests/test_ray_pins.py): chord lengths through the box against the analytic slab formula; the list of visited
cells against brute-force sampling of the ray; Beer-Lambert attenuation through a uniform medium in closed form; photon
conservation cell by cell (what the species absorb is what the ray loses, eq. 30's first equality); the optically thin
and thick limits of eq. 28 / 30; the hydrogen ionisation balance of eq. 35 reached by the chemistry
oracle when it is driven by a traced rate.

Readings: R29 only the Cartesian case of eq. 23 is built (eq. 24); a ray that starts outside the mesh enters
through the first face it meets; a ray that runs exactly along a face or through an edge goes to the cell on the side of
its direction (ties between surfaces: all tied indices advance).  R30 (1 - exp(-tau)) / tau is evaluated as
-expm1(-tau) / tau, and as 1 for tau = 0.  R31 eq. 32 (the time-integrated depletion that couples a ray to the chemistry
of the cells it has crossed within one step) is not built: the rates here are instantaneous.
"""
from __future__ import annotations

import math

import numpy as np


def enter_box(origin, direction, lo, hi):
    """Parameter t >= 0 at which the ray origin + t direction is inside [lo, hi] (slab method), or None if it misses."""
    t0, t1 = 0.0, math.inf
    for a in range(3):
        o, d = float(origin[a]), float(direction[a])
        if d == 0.0:
            if o < lo[a] or o > hi[a]:
                return None
            continue
        ta, tb = (lo[a] - o) / d, (hi[a] - o) / d
        if ta > tb:
            ta, tb = tb, ta
        t0, t1 = max(t0, ta), min(t1, tb)
    return t0 if t0 <= t1 else None


def walk(origin, direction, shape, spacing, lo=(0.0, 0.0, 0.0), max_cells=None):
    """Eqs. 23-24: the cells a ray crosses and the path length in each, [(i, j, k, dl), ...].  In every cell the three
    surfaces the ray can leave through are x_int = the face on the side of the direction; 0 = x_d dl + (x_in - x_int)."""
    n = [int(v) for v in shape]
    h = [float(v) for v in spacing]
    lo = [float(v) for v in lo]
    hi = [lo[a] + n[a] * h[a] for a in range(3)]
    d = [float(v) for v in direction]
    norm = math.sqrt(sum(v * v for v in d))
    d = [v / norm for v in d]
    t = enter_box(origin, d, lo, hi)
    if t is None:
        return []
    x = [float(origin[a]) + t * d[a] for a in range(3)]
    idx = []
    for a in range(3):                          # the cell that holds the entry point; on a face: the side of the direction
        q = (x[a] - lo[a]) / h[a]
        i = int(math.floor(q))
        if q == i and d[a] < 0.0:
            i -= 1
        idx.append(min(max(i, 0), n[a] - 1))
    out = []
    limit = max_cells if max_cells is not None else sum(n) + 3
    while all(0 <= idx[a] < n[a] for a in range(3)) and len(out) < limit:
        dls = []
        for a in range(3):
            if d[a] > 0.0:
                dls.append((lo[a] + (idx[a] + 1) * h[a] - x[a]) / d[a])
            elif d[a] < 0.0:
                dls.append((lo[a] + idx[a] * h[a] - x[a]) / d[a])
            else:
                dls.append(math.inf)
        dl = max(min(dls), 0.0)                 # the smallest positive solution
        out.append((idx[0], idx[1], idx[2], dl))
        for a in range(3):
            if dls[a] <= dl:                    # every surface reached at dl is crossed (edges, corners)
                idx[a] += 1 if d[a] > 0.0 else -1
                x[a] = lo[a] + (idx[a] + (0 if d[a] > 0.0 else 1)) * h[a]     # exactly on the surface
            else:
                x[a] += dl * d[a]
    return out


def thin_factor(tau: float) -> float:
    """(1 - exp(-tau)) / tau of eqs. 28, 30 (reading R30)."""
    return 1.0 if tau == 0.0 else -math.expm1(-tau) / tau


def trace(origins, directions, L_in, sigma, n_dens, shape, spacing, lo=(0.0, 0.0, 0.0)):
    """All rays, eqs. 29-31.  L_in [n_rays, n_bins] photons per second per ray and bin; sigma [n_abs, n_bins] cm^2;
    n_dens [n_abs, nx, ny, nz] cm^-3.  Returns (k [n_abs, nx, ny, nz] s^-1, L_out [n_rays, n_bins], path [n_rays])."""
    L_in = np.asarray(L_in, dtype=np.float64); sigma = np.asarray(sigma, dtype=np.float64)
    n_dens = np.asarray(n_dens, dtype=np.float64)
    n_abs, n_bins = sigma.shape
    dV = float(spacing[0]) * float(spacing[1]) * float(spacing[2])
    k = np.zeros_like(n_dens)
    L_out = L_in.copy()
    path = np.zeros(L_in.shape[0])
    for j in range(L_in.shape[0]):
        for (ix, iy, iz, dl) in walk(origins[j], directions[j], shape, spacing, lo):
            path[j] += dl
            for b in range(n_bins):
                tau = 0.0
                for i in range(n_abs):
                    tau += n_dens[i, ix, iy, iz] * sigma[i, b] * dl              # eq. 31: tau_jk
                f = thin_factor(tau)
                for i in range(n_abs):
                    k[i, ix, iy, iz] += L_out[j, b] * sigma[i, b] * dl / dV * f  # eq. 31: k_ijk^(0) [...]
                L_out[j, b] *= math.exp(-tau)                                    # eq. 29
    return k, L_out, path
