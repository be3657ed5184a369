"""Algorithmic work model of one kr_thermochem_step.

Conventions: FMA = 2 flops, exp / log = 40, divide = 8.  The model counts what the ALGORITHM of
DESIGN.md steps 2-7 needs, not what a kernel executes (no redundant or padded work), so
``flops / time / peak`` is an algorithmic fraction of the FP64 roofline.  Pure arithmetic on the
network's shape and on the solver's own counters; holds no method code.
"""
from __future__ import annotations

from typing import Dict


def lu_flops(N: int) -> int:
    """Right-looking LU with the multipliers: sum_k [2 (N-k-1)^2 + (N-k-1)]."""
    return sum(2 * (N - k - 1) ** 2 + (N - k - 1) for k in range(N))


def shape_of(net) -> Dict[str, int]:
    fl = net.flags
    n_rev = int(((fl & 1) != 0).sum())
    n_tb = int(((fl & 2) != 0).sum())
    n_unary = int(((fl & 12) != 0).sum())
    R = int(net.n_reac)
    return dict(S=int(net.n_species), R=R, N=int(net.n_unknowns), energy=int(net.energy_equation), n_rev=n_rev,
                n_tb=n_tb, n_unary=n_unary, n_arr=R - n_unary, n_dir=R + n_rev)


def per_rate_eval(net) -> int:
    """a2 + a3: thermo (32 per species) + rate constants (100 per reversible Arrhenius reaction:
    two exp and the K_c sums; 52 per one-way Arrhenius; 4 per unary)."""
    s = shape_of(net)
    return 32 * s["S"] + 100 * s["n_rev"] + 52 * (s["n_arr"] - s["n_rev"]) + 4 * s["n_unary"]


def per_newton(net) -> int:
    """a4-a7: mass action (3 per direction + 9 per reaction), third-body (12 S each), Jacobian (20 per
    direction, +12 per reaction with T), I - hJ (2 N^2), LU, substitution (2 N^2), update and norm (12 N)."""
    s = shape_of(net)
    N = s["N"]
    f = 3 * s["n_dir"] + 9 * s["R"] + 12 * s["S"] * s["n_tb"]
    f += 20 * s["n_dir"] + (12 * s["R"] if s["energy"] else 0)
    f += 2 * N * N + lu_flops(N) + 2 * N * N + 12 * N
    return f


def step_flops(net, stats: Dict[str, int]) -> float:
    """Model flops of one step from the solver's counters (n_newton, n_rate_evals)."""
    return float(stats["n_newton"]) * per_newton(net) + float(stats["n_rate_evals"]) * per_rate_eval(net)


def step_bytes(net, n_cells: int, n_aux: int = 0) -> float:
    """Algorithmic HBM traffic: read y, rho, T, aux; write y, T, status."""
    S = int(net.n_species)
    return float(n_cells) * (16 * S + 24 + 8 * n_aux)
