"""Small hand-built networks and numpy restatements used by the pins (no method code from the repo)."""
from __future__ import annotations

from typing import List, Optional, Sequence, Tuple

import numpy as np

from paper_2504_04941_b200 import workloads as w

K_B = 1.380649e-16
M_U = 1.66053906660e-24
P0 = 1.01325e6


def tiny_network(composition, reactions, *, elem_mass=None, thermo=None, energy=0, T_lo=1.0, T_hi=1.0e5,
                 tb_eff=None, q_ext=None, name="tiny") -> w.Network:
    """reactions: list of (reactants, products, A, beta, Ea_over_k, flags, aux_index);
    reactants/products are tuples of species indices with repetition, e.g. (0, 0) for A + A."""
    comp = np.asarray(composition, np.int32)
    E, S = comp.shape
    R = len(reactions)
    ri = np.full((R, 3), -1, np.int32); rn = np.zeros((R, 3), np.int32)
    pi = np.full((R, 3), -1, np.int32); pn = np.zeros((R, 3), np.int32)
    A = np.zeros(R); be = np.zeros(R); Ea = np.zeros(R)
    fl = np.zeros(R, np.int32); ax = np.full(R, -1, np.int32)
    for r, (lhs, rhs, a, b, ea, f, x) in enumerate(reactions):
        ri[r], rn[r] = w._pack_side(tuple(lhs))
        pi[r], pn[r] = w._pack_side(tuple(rhs))
        A[r], be[r], Ea[r], fl[r], ax[r] = a, b, ea, f, x
    if thermo is None:
        thermo = np.zeros((S, 7)); thermo[:, 0] = 2.5
    thermo = np.asarray(thermo, np.float64)
    if elem_mass is None:
        elem_mass = np.ones(E)
    n_aux = int(max([x for *_, x in reactions] + [-1])) + 1
    return w.Network(name, [f"e{i}" for i in range(E)], [f"s{i}" for i in range(S)], np.asarray(elem_mass, float),
                     comp, ri, rn, pi, pn, A, be, Ea, fl, ax,
                     None if tb_eff is None else np.asarray(tb_eff, float),
                     None if q_ext is None else np.asarray(q_ext, float),
                     thermo.copy(), thermo.copy(), np.full(S, 1000.0), T_lo, T_hi, energy, n_aux)


def cells_of(rho, T, y, dt, aux=None) -> w.Cells:
    y = np.atleast_2d(np.asarray(y, float))
    n = y.shape[0]
    rho = np.broadcast_to(np.asarray(rho, float), (n,)).copy()
    T = np.broadcast_to(np.asarray(T, float), (n,)).copy()
    if aux is not None:
        aux = np.atleast_2d(np.asarray(aux, float))
    return w.Cells(rho, T, np.ascontiguousarray(y), aux, float(dt))


# ---- numpy restatements of the thermo definitions (textbook forms, used as independent references) ----

def nasa_cp_R(a, T):
    return a[..., 0] + a[..., 1] * T + a[..., 2] * T ** 2 + a[..., 3] * T ** 3 + a[..., 4] * T ** 4


def nasa_h_RT(a, T):
    return (a[..., 0] + a[..., 1] * T / 2 + a[..., 2] * T ** 2 / 3 + a[..., 3] * T ** 3 / 4 + a[..., 4] * T ** 4 / 5
            + a[..., 5] / T)


def nasa_s_R(a, T):
    return (a[..., 0] * np.log(T) + a[..., 1] * T + a[..., 2] * T ** 2 / 2 + a[..., 3] * T ** 3 / 3
            + a[..., 4] * T ** 4 / 4 + a[..., 6])


def dnu_matrix(net) -> np.ndarray:
    """[R,S] net stoichiometric change products - reactants."""
    d = np.zeros((net.n_reac, net.n_species))
    for r in range(net.n_reac):
        for k in range(3):
            if net.reac_idx[r, k] >= 0:
                d[r, net.reac_idx[r, k]] -= net.reac_nu[r, k]
            if net.prod_idx[r, k] >= 0:
                d[r, net.prod_idx[r, k]] += net.prod_nu[r, k]
    return d


def ln_Kc(net, T) -> np.ndarray:
    """ln K_c of every reaction from the Gibbs function of the polynomials, standard state 1 atm:
    K_c = exp(-sum dnu g/RT) (p0 / k_B T)^(sum dnu)."""
    a = np.where((T <= net.T_mid)[:, None], net.nasa_lo, net.nasa_hi)
    g = nasa_h_RT(a, T) - nasa_s_R(a, T)
    d = dnu_matrix(net)
    return -(d @ g) + d.sum(axis=1) * np.log(P0 / (K_B * T))
