"""Seeded synthetic networks and cell states for the five BASELINE.json configs.

This module is the ONE piece shared by the CPU oracle (``oracle/``) and the
CUDA path (``paper_2504_04941_b200/csrc``).  It holds no arithmetic of the
method (no rates, no Jacobian, no LU, no integrator): it only draws the
inputs -- element/species composition matrices, element-conserving reaction
lists, Arrhenius and thermo coefficients, and per-cell (rho, T, y, aux).

Recipe: SURVEY.md section 8(d), restated in DESIGN.md "Input recipe".  The
paper's own workloads (GRI-Mech H2/O2, Stroemgren sphere, astrochemical
database) are not available offline and are NOT
reproduced; these seeded stand-ins only take their shapes.  Config 2's H rows
use the coefficients the paper prints in eq. 36.

numpy only.  Importing this module never loads the CUDA library.
"""
from __future__ import annotations

import itertools
import math
from dataclasses import dataclass, field
from typing import Dict, List, Optional, Tuple

import numpy as np

# CGS constants (SURVEY.md 8(c) "State and units")
K_B = 1.380649e-16          # erg / K
M_U = 1.66053906660e-24     # g
P0 = 1.01325e6              # dyn / cm^2  (1 atm)
EV = 1.602176634e-12        # erg
T_REF = 300.0               # K

# reaction flag bits (include/kratos_chem.h)
F_REVERSIBLE = 1
F_THIRD_BODY = 2
F_CONST_UNARY = 4
F_AUX_UNARY = 8

BASE_SEED = 20250404

FULL_CELLS = {0: 4096, 1: 1 << 20, 2: 256 ** 3, 3: 1 << 18, 4: 1 << 17}
DT = {0: 1e7, 1: 1e-6, 2: 1e10, 3: 3e11, 4: 1e12}
CONFIG_NAMES = {
    0: "c0_toy_S5_R6_iso",
    1: "c1_combustion_S9_R21_energy",
    2: "c2_photoion_S6_R9_iso",
    3: "c3_astro_S32_R180_energy",
    4: "c4_large_S64_R480_iso",
}


@dataclass
class Network:
    """Plain arrays in the layout of ``kr_network_desc`` (include/kratos_chem.h)."""
    name: str
    elem_names: List[str]
    species_names: List[str]
    elem_mass: np.ndarray        # [E] f64 (amu; 0 on a charge row)
    composition: np.ndarray      # [E,S] i32
    reac_idx: np.ndarray         # [R,3] i32, -1 = unused
    reac_nu: np.ndarray          # [R,3] i32
    prod_idx: np.ndarray         # [R,3] i32
    prod_nu: np.ndarray          # [R,3] i32
    A: np.ndarray                # [R] f64
    beta: np.ndarray             # [R] f64
    Ea_over_k: np.ndarray        # [R] f64 (K)
    flags: np.ndarray            # [R] i32
    aux_index: np.ndarray        # [R] i32
    tb_eff: Optional[np.ndarray]  # [R,S] f64 or None
    q_ext: Optional[np.ndarray]   # [R] f64 (erg per forward event) or None
    nasa_lo: np.ndarray          # [S,7]
    nasa_hi: np.ndarray          # [S,7]
    T_mid: np.ndarray            # [S]
    T_lo: float
    T_hi: float
    energy_equation: int
    n_aux: int = 0

    @property
    def n_elem(self) -> int:
        return int(self.composition.shape[0])

    @property
    def n_species(self) -> int:
        return int(self.composition.shape[1])

    @property
    def n_reac(self) -> int:
        return int(self.A.shape[0])

    @property
    def n_unknowns(self) -> int:
        return self.n_species + (1 if self.energy_equation else 0)

    @property
    def weights(self) -> np.ndarray:
        """Species weight W_s = sum_nu N_{nu,s} m_nu (amu)."""
        return self.elem_mass @ self.composition.astype(np.float64)


@dataclass
class Cells:
    rho: np.ndarray              # [n] g cm^-3
    T: np.ndarray                # [n] K
    y: np.ndarray                # [n,S] cell-major, y_s = n_s m_u / rho
    aux: Optional[np.ndarray]    # [n_aux,n] or None
    dt: float

    @property
    def n_cells(self) -> int:
        return int(self.rho.shape[0])

    def copy(self) -> "Cells":
        return Cells(self.rho.copy(), self.T.copy(), self.y.copy(),
                     None if self.aux is None else self.aux.copy(), self.dt)

    def take(self, sl) -> "Cells":
        return Cells(np.ascontiguousarray(self.rho[sl]), np.ascontiguousarray(self.T[sl]),
                     np.ascontiguousarray(self.y[sl]),
                     None if self.aux is None else np.ascontiguousarray(self.aux[:, sl]), self.dt)


@dataclass
class SolverOpts:
    """Mirror of ``kr_solver_opts``; defaults = SURVEY.md 8(c) "Default options"."""
    max_newton: int = 8
    fixed_newton: int = 0
    h0_mode: int = 1
    rtol: float = 1e-8
    atol_y: float = 1e-20
    atol_T: float = 1e-8
    neg_tol: float = 1e-12
    eta: float = 0.1
    y_floor: float = 1e-12
    shrink: float = 0.25
    grow_fast: float = 8.0
    grow_mid: float = 2.0
    chg_floor: float = 1e-12
    chg_max: float = float("inf")
    it_fast: int = 3
    it_mid: int = 5
    max_substeps: int = 4096
    h_min_rel: float = 1e-12     # fail when h < h_min_rel * (first sub-step size)
    bail_ratio: float = 10.0     # early-exit mode: abort the sub-step when e_k > bail_ratio * e_{k-1}, k >= 2
    finalize: int = 1            # 0: skip step 9 (used by the conservation pin P4)
    retry: int = 0               # 1: a failed cell gets a second attempt with tightened control (R24)
    retry_h0: float = 0.01       # factor on the first sub-step of the second attempt
    cons_tol: float = 1e-13      # stage 2: rows whose initial-minus-final total exceeds cons_tol * sum|N||y_in| are compensated in full


# --------------------------------------------------------------------------
# species / reaction construction (element-conserving by construction)
# --------------------------------------------------------------------------

def _species_name(comp: Tuple[int, ...], elem_names: List[str]) -> str:
    out = ""
    for e, c in zip(elem_names, comp):
        if c == 1:
            out += e
        elif c > 1:
            out += f"{e}{c}"
    return out


def _random_species(rng: np.random.Generator, n_elem: int, n_species: int) -> np.ndarray:
    """First E species are atoms; the rest distinct random multisets of 2-4 atoms."""
    w = np.array([1.0] + [0.5] * (n_elem - 1))
    w = w / w.sum()
    comps = [tuple(1 if i == e else 0 for i in range(n_elem)) for e in range(n_elem)]
    seen = set(comps)
    guard = 0
    while len(comps) < n_species:
        guard += 1
        if guard > 100000:
            raise RuntimeError("cannot draw enough distinct species")
        size = int(rng.choice([2, 3, 4], p=[0.5, 0.3, 0.2]))
        atoms = rng.choice(n_elem, size=size, p=w)
        c = tuple(int(np.sum(atoms == e)) for e in range(n_elem))
        if c in seen:
            continue
        seen.add(c)
        comps.append(c)
    return np.array(comps, dtype=np.int32).T.copy()   # [E,S]


def _enumerate_candidates(composition: np.ndarray, skip: Tuple[int, ...] = ()):
    """Unordered species pairs grouped by summed composition.

    Returns (associations, exchanges): an association is ((x, y), z) with
    comp(x)+comp(y) == comp(z); an exchange is ((x, y), (p, q)) with two disjoint
    pairs of equal summed composition.  Deterministic order.
    """
    S = composition.shape[1]
    comp_of = {tuple(composition[:, s].tolist()): s for s in range(S) if s not in skip}
    groups: Dict[Tuple[int, ...], List[Tuple[int, int]]] = {}
    idx = [s for s in range(S) if s not in skip]
    for a, b in itertools.combinations_with_replacement(idx, 2):
        key = tuple((composition[:, a] + composition[:, b]).tolist())
        groups.setdefault(key, []).append((a, b))
    assoc, exch = [], []
    for key in sorted(groups):
        pairs = groups[key]
        if key in comp_of:
            for pr in pairs:
                assoc.append((pr, comp_of[key]))
        for p1, p2 in itertools.combinations(pairs, 2):
            if set(p1) & set(p2):
                continue
            exch.append((p1, p2))
    return assoc, exch


def _pack_side(species: Tuple[int, ...]):
    """(a, a) -> idx [a,-1,-1], nu [2,0,0];  (a, b) -> idx [a,b,-1], nu [1,1,0]."""
    idx = [-1, -1, -1]
    nu = [0, 0, 0]
    k = 0
    for s in sorted(set(species)):
        idx[k] = s
        nu[k] = species.count(s)
        k += 1
    return idx, nu


def _thermo(rng: np.random.Generator, S: int, T_hi: float, theta: float):
    """7-coefficient polynomials, both ranges identical (SURVEY.md 8(d) 'Thermo')."""
    a = np.zeros((S, 7))
    a[:, 0] = rng.uniform(3.5, 4.5, S)
    a[:, 1] = rng.uniform(0.0, 1.0, S) / T_hi
    a[:, 2] = rng.uniform(-0.5, 0.5, S) / T_hi ** 2
    a[:, 3] = rng.uniform(-0.25, 0.25, S) / T_hi ** 3
    a[:, 4] = rng.uniform(-0.1, 0.1, S) / T_hi ** 4
    a[:, 5] = rng.uniform(-1.0, 1.0, S) * theta
    a[:, 6] = rng.uniform(-5.0, 10.0, S)
    return a.copy(), a.copy(), np.full(S, 1000.0)


def _build_reactions(rng, composition, nasa, assoc_sel, exch_sel, *, third_body_assoc: bool,
                     ea_zero_frac: float, tb_scale: float, reversible: bool = True):
    """Turn selected candidates into packed reversible reactions with drawn Arrhenius data."""
    S = composition.shape[1]
    rows = []
    for (pair, z) in assoc_sel:
        rows.append((tuple(pair), (z,), third_body_assoc))
    for (p1, p2) in exch_sel:
        rows.append((tuple(p1), tuple(p2), False))
    R = len(rows)
    reac_idx = np.full((R, 3), -1, np.int32)
    reac_nu = np.zeros((R, 3), np.int32)
    prod_idx = np.full((R, 3), -1, np.int32)
    prod_nu = np.zeros((R, 3), np.int32)
    flags = np.zeros(R, np.int32)
    a6 = nasa[:, 5]
    for r, (lhs, rhs, tb) in enumerate(rows):
        # orient forward-exothermic: sum dnu_s a6_s <= 0
        d = sum(a6[s] for s in rhs) - sum(a6[s] for s in lhs)
        if d > 0:
            lhs, rhs = rhs, lhs
        reac_idx[r], reac_nu[r] = _pack_side(lhs)
        prod_idx[r], prod_nu[r] = _pack_side(rhs)
        flags[r] = (F_REVERSIBLE if reversible else 0) | (F_THIRD_BODY if tb else 0)
    A = 10.0 ** rng.uniform(-12.0, -9.0, R)
    beta = rng.uniform(-1.0, 1.0, R)
    Ea = rng.uniform(0.0, 2.0e4, R)
    if ea_zero_frac > 0:
        Ea[rng.uniform(size=R) < ea_zero_frac] = 0.0
    tb_eff = None
    if third_body_assoc:
        tb_eff = np.ones((R, S))
        for r in range(R):
            if flags[r] & F_THIRD_BODY:
                tb_eff[r] = rng.uniform(0.5, 12.0, S)
                A[r] *= tb_scale
    return reac_idx, reac_nu, prod_idx, prod_nu, flags, A, beta, Ea, tb_eff


def _check_conservation(net: Network) -> None:
    N = net.composition.astype(np.int64)
    for r in range(net.n_reac):
        d = np.zeros(net.n_species, np.int64)
        for k in range(3):
            if net.reac_idx[r, k] >= 0:
                d[net.reac_idx[r, k]] -= net.reac_nu[r, k]
            if net.prod_idx[r, k] >= 0:
                d[net.prod_idx[r, k]] += net.prod_nu[r, k]
        if np.any(N @ d != 0):
            raise AssertionError(f"reaction {r} of {net.name} does not conserve elements")


# --------------------------------------------------------------------------
# the five networks
# --------------------------------------------------------------------------

def _network_c0(rng) -> Network:
    elem = ["a", "b"]
    comp = np.array([[1, 0, 2, 1, 0],
                     [0, 1, 0, 1, 2]], np.int32)      # a, b, a2, ab, b2
    names = [_species_name(tuple(comp[:, s]), elem) for s in range(5)]
    lo, hi, tmid = _thermo(rng, 5, 6000.0, 3.0e4)
    assoc, exch = _enumerate_candidates(comp)
    assert len(assoc) == 3 and len(exch) == 3
    ri, rn, pi, pn, fl, A, be, Ea, _ = _build_reactions(
        rng, comp, lo, assoc, exch, third_body_assoc=False, ea_zero_frac=0.0, tb_scale=1.0)
    R = len(A)
    return Network(CONFIG_NAMES[0], elem, names, np.array([1.0, 12.0]), comp, ri, rn, pi, pn, A, be, Ea, fl,
                   np.full(R, -1, np.int32), None, None, lo, hi, tmid, 100.0, 6000.0, 0, 0)


def _network_c1(rng) -> Network:
    elem = ["H", "O", "N"]
    # H, H2, O, O2, OH, H2O, HO2, H2O2, N2 -- compositions only; no mechanism data.
    comp = np.array([[1, 2, 0, 0, 1, 2, 1, 2, 0],
                     [0, 0, 1, 2, 1, 1, 2, 2, 0],
                     [0, 0, 0, 0, 0, 0, 0, 0, 2]], np.int32)
    names = [_species_name(tuple(comp[:, s]), elem) for s in range(9)]
    lo, hi, tmid = _thermo(rng, 9, 6000.0, 3.0e4)
    assoc, exch = _enumerate_candidates(comp, skip=(8,))
    a_sel = [assoc[i] for i in sorted(rng.choice(len(assoc), size=6, replace=False))]
    e_sel = [exch[i] for i in sorted(rng.choice(len(exch), size=15, replace=False))]
    ri, rn, pi, pn, fl, A, be, Ea, tb = _build_reactions(
        rng, comp, lo, a_sel, e_sel, third_body_assoc=True, ea_zero_frac=0.0, tb_scale=3.0e-19)
    R = len(A)
    return Network(CONFIG_NAMES[1], elem, names, np.array([1.008, 15.999, 14.007]), comp, ri, rn, pi, pn,
                   A, be, Ea, fl, np.full(R, -1, np.int32), tb, None, lo, hi, tmid, 100.0, 6000.0, 1, 0)


def _network_c2(rng) -> Network:
    elem = ["H", "He", "q"]
    #                H  H+  e-  He He+ He++
    comp = np.array([[1, 1, 0, 0, 0, 0],
                     [0, 0, 0, 1, 1, 1],
                     [0, 1, -1, 0, 1, 2]], np.int32)
    names = ["H", "H+", "e-", "He", "He+", "He++"]
    lo, hi, tmid = _thermo(rng, 6, 2.0e5, 1.0e4)
    H, Hp, e, He, Hep, Hepp = range(6)
    I_H, I_He, I_Hep = 13.598 * EV / K_B, 24.59 * EV / K_B, 54.42 * EV / K_B
    dec = lambda: 10.0 ** rng.uniform(-0.5, 0.5)
    # (reactants, products, A, beta, Ea/k, flags, aux)
    rows = [
        ((H, e), (Hp, e, e), 1.05e-9, 0.5, I_H, 0, -1),               # eq. 36 k_ci
        ((Hp, e), (H,), 3.5e-12, -0.75, 0.0, 0, -1),                  # eq. 36 alpha
        ((H,), (Hp, e), 1.0, 0.0, 0.0, F_AUX_UNARY, 0),               # photoionisation, k = 1.0 * Gamma
        ((He, e), (Hep, e, e), 1.05e-9 * dec(), 0.5, I_He, 0, -1),
        ((Hep, e), (He,), 3.5e-12 * dec(), -0.75, 0.0, 0, -1),
        ((He,), (Hep, e), 0.5, 0.0, 0.0, F_AUX_UNARY, 0),
        ((Hep, e), (Hepp, e, e), 1.05e-9 * dec(), 0.5, I_Hep, 0, -1),
        ((Hepp, e), (Hep,), 3.5e-12 * dec(), -0.75, 0.0, 0, -1),
        ((Hep,), (Hepp, e), 0.1, 0.0, 0.0, F_AUX_UNARY, 0),
    ]
    R = len(rows)
    ri = np.full((R, 3), -1, np.int32); rn = np.zeros((R, 3), np.int32)
    pi = np.full((R, 3), -1, np.int32); pn = np.zeros((R, 3), np.int32)
    A = np.zeros(R); be = np.zeros(R); Ea = np.zeros(R)
    fl = np.zeros(R, np.int32); ax = np.full(R, -1, np.int32)
    for r, (lhs, rhs, a, b, ea, f, x) in enumerate(rows):
        ri[r], rn[r] = _pack_side(lhs)
        pi[r], pn[r] = _pack_side(rhs)
        A[r], be[r], Ea[r], fl[r], ax[r] = a, b, ea, f, x
    return Network(CONFIG_NAMES[2], elem, names, np.array([1.008, 4.0026, 0.0]), comp, ri, rn, pi, pn,
                   A, be, Ea, fl, ax, None, None, lo, hi, tmid, 1.0, 2.0e5, 0, 1)


def _network_random(rng, idx: int, n_elem: int, S: int, n_rev: int, n_const: int, n_aux: int,
                    energy: int, reversible: bool) -> Network:
    """Random element-conserving network (configs 3 and 4).

    reversible=False (config 3): two-body reactions are one-way, as in the astrochemical databases the
    paper cites; thermo enters only through the energy equation (theta = 1e3 K keeps the
    chemical heating within a few 1e3 K).
    reversible=True (config 4): reverse rates from detailed balance.  To keep k_r = k_f / K_c within what
    fp64 can resolve at dt = 1e12 s (deviation D2) the formation enthalpies are
    bond-like, a6_s = -6e4 K x (atoms_s - 1) x U(0.7, 1.3), every reaction draws Ea/k ~ U(0, 2e4) K, and
    two-body associations X + Y <-> XY get A x 1e-6 (radiative-association scale).
    """
    elem = ["H", "C", "N", "O", "S", "Si"][:n_elem]
    masses = np.array([1.008, 12.011, 14.007, 15.999, 32.06, 28.085][:n_elem])
    comp = _random_species(rng, n_elem, S)
    names = [_species_name(tuple(comp[:, s]), elem) for s in range(S)]
    lo, hi, tmid = _thermo(rng, S, 2.0e5, 1.0e3 if not reversible else 1.0e4)
    if reversible:
        n_atoms = comp.sum(axis=0).astype(np.float64)
        a6 = -6.0e4 * (n_atoms - 1.0) * rng.uniform(0.7, 1.3, S)
        lo[:, 5] = a6
        hi[:, 5] = a6
    assoc, exch = _enumerate_candidates(comp)
    n_assoc_rev = min(len(assoc), n_rev // 4)
    n_exch = n_rev - n_assoc_rev
    if len(exch) < n_exch:
        raise RuntimeError(f"config {idx}: only {len(exch)} exchange candidates, need {n_exch}")
    a_sel = [assoc[i] for i in sorted(rng.choice(len(assoc), size=n_assoc_rev, replace=False))]
    e_sel = [exch[i] for i in sorted(rng.choice(len(exch), size=n_exch, replace=False))]
    ri, rn, pi, pn, fl, A, be, Ea, _ = _build_reactions(
        rng, comp, lo, a_sel, e_sel, third_body_assoc=False, ea_zero_frac=0.0 if reversible else 0.7,
        tb_scale=1.0, reversible=reversible)
    if reversible:
        A[:n_assoc_rev] *= 1.0e-6
    ax = np.full(len(A), -1, np.int32)
    q_ext = None
    n_un = n_const + n_aux
    if n_un:
        # unary dissociations XY -> X + Y taken from association candidates
        pick = [assoc[i] for i in sorted(rng.choice(len(assoc), size=n_un, replace=len(assoc) < n_un))]
        uri = np.full((n_un, 3), -1, np.int32); urn = np.zeros((n_un, 3), np.int32)
        upi = np.full((n_un, 3), -1, np.int32); upn = np.zeros((n_un, 3), np.int32)
        uA = np.zeros(n_un); ufl = np.zeros(n_un, np.int32); uax = np.full(n_un, -1, np.int32)
        for k, (pair, z) in enumerate(pick):
            uri[k], urn[k] = _pack_side((z,))
            upi[k], upn[k] = _pack_side(tuple(pair))
            if k < n_const:                               # cosmic-ray, zeta = 1e-17 s^-1
                uA[k] = 1.0e-17 * rng.uniform(0.5, 5.0)
                ufl[k] = F_CONST_UNARY
            else:                                         # photodissociation x shielding factor
                uA[k] = 10.0 ** rng.uniform(-11.0, -9.0)
                ufl[k] = F_AUX_UNARY
                uax[k] = 0
        # heat deposited per event: cosmic-ray events a few eV, photodissociations a few meV (they recur
        # A*dt ~ 3..300 times per molecule within dt, so this keeps the heating within ~1e3 K)
        q_un = rng.uniform(1.0, 10.0, n_un) * EV
        q_un[n_const:] *= 1.0e-3
        ri = np.vstack([ri, uri]); rn = np.vstack([rn, urn])
        pi = np.vstack([pi, upi]); pn = np.vstack([pn, upn])
        A = np.concatenate([A, uA]); be = np.concatenate([be, np.zeros(n_un)])
        Ea = np.concatenate([Ea, np.zeros(n_un)])
        fl = np.concatenate([fl, ufl]); ax = np.concatenate([ax, uax])
        q_ext = np.concatenate([np.zeros(len(A) - n_un), q_un])
    return Network(CONFIG_NAMES[idx], elem, names, masses, comp, ri, rn, pi, pn, A, be, Ea,
                   fl.astype(np.int32), ax.astype(np.int32), None, q_ext, lo, hi, tmid, 1.0, 2.0e5,
                   energy, 1 if n_aux else 0)


def make_network(idx: int, seed: Optional[int] = None) -> Network:
    rng = np.random.default_rng((BASE_SEED + idx) if seed is None else seed)
    if idx == 0:
        net = _network_c0(rng)
    elif idx == 1:
        net = _network_c1(rng)
    elif idx == 2:
        net = _network_c2(rng)
    elif idx == 3:
        net = _network_random(rng, 3, 5, 32, 140, 20, 20, 1, reversible=False)
    elif idx == 4:
        net = _network_random(rng, 4, 6, 64, 480, 0, 0, 0, reversible=True)
    else:
        raise ValueError("config index must be 0..4")
    _check_conservation(net)
    return net


# --------------------------------------------------------------------------
# cell states
# --------------------------------------------------------------------------

def _logu(rng, lo, hi, n):
    return np.exp(rng.uniform(np.log(lo), np.log(hi), n))


def make_cells(idx: int, net: Network, n_cells: Optional[int] = None, seed: Optional[int] = None) -> Cells:
    n = FULL_CELLS[idx] if n_cells is None else int(n_cells)
    rng = np.random.default_rng((BASE_SEED + 1000 + idx) if seed is None else seed)
    S = net.n_species
    W = net.weights
    aux = None
    if idx in (0, 3, 4):
        Tr = {0: (300.0, 3000.0), 3: (10.0, 1.0e4), 4: (10.0, 5.0e3)}[idx]
        nr = {0: (1e2, 1e8), 3: (1.0, 1e7), 4: (1.0, 1e8)}[idx]
        T = _logu(rng, *Tr, n)
        nH = _logu(rng, *nr, n)
        rho = 1.4 * nH * M_U
        g = rng.standard_exponential((n, S))
        g /= g.sum(axis=1, keepdims=True)                 # Dirichlet(1_S)
        y = g / (g @ W)[:, None]                          # mass-normalised: sum_s W_s y_s = 1
        if idx == 3:
            aux = rng.uniform(0.0, 1.0, (1, n))
    elif idx == 1:
        T = rng.uniform(900.0, 3000.0, n)
        p = _logu(rng, 0.1, 10.0, n) * P0
        X = np.zeros(S)
        X[1], X[3], X[8] = 2.0, 1.0, 3.76                 # H2 : O2 : N2 molar
        Ymass = X * W / np.sum(X * W)
        Ymass = np.where(Ymass > 0, Ymass, 1.0e-8)        # radicals / intermediates seeded
        Yc = Ymass[None, :] * (1.0 + 0.01 * rng.standard_normal((n, S)))
        Yc = np.abs(Yc)
        Yc /= Yc.sum(axis=1, keepdims=True)
        y = Yc / W[None, :]
        Wbar = 1.0 / y.sum(axis=1)
        rho = p / (K_B * T) * Wbar * M_U
    elif idx == 2:
        T = _logu(rng, 1e2, 1e5, n)
        nH = _logu(rng, 1e-2, 1e4, n)
        xHp = rng.uniform(0.0, 1.0, n)
        gHe = rng.standard_exponential((n, 3))
        gHe /= gHe.sum(axis=1, keepdims=True)
        nd = np.zeros((n, S))
        nd[:, 0] = nH * (1.0 - xHp)
        nd[:, 1] = nH * xHp
        nd[:, 3:6] = 0.1 * nH[:, None] * gHe
        nd[:, 2] = nd[:, 1] + nd[:, 4] + 2.0 * nd[:, 5]   # charge neutrality
        rho = (nd @ W) * M_U
        y = nd * M_U / rho[:, None]
        aux = _logu(rng, 1e-16, 1e-10, n)[None, :]
    else:
        raise ValueError("config index must be 0..4")
    return Cells(np.ascontiguousarray(rho), np.ascontiguousarray(T), np.ascontiguousarray(y),
                 None if aux is None else np.ascontiguousarray(aux), DT[idx])


def default_opts(idx: int, fixed_newton: int = 0) -> SolverOpts:
    o = SolverOpts()
    o.h0_mode = 0 if idx == 0 else 1
    o.fixed_newton = fixed_newton
    return o


def make_config(idx: int, n_cells: Optional[int] = None, fixed_newton: int = 0,
                seed: Optional[int] = None) -> Tuple[Network, Cells, SolverOpts]:
    net = make_network(idx)
    cells = make_cells(idx, net, n_cells, seed)
    return net, cells, default_opts(idx, fixed_newton)


# --------------------------------------------------------------------------
# species advection (NEXT-2: PAPER.md section 2.1, test of section 4.1) -- inputs only, no method arithmetic
# --------------------------------------------------------------------------

def advection_test_case(n_zones: int = 128, table=None):
    """The four-species test of PAPER.md:400-417: returns (composition [2, 4], x_centres, y [n_zones, 4], rho, dx).
    `table` is the parsed tests/golden/paper_eq33.txt (rows of left, right, slope, atoms of A, atoms of B); the defaults
    are the same printed values."""
    if table is None:
        table = [(0.49, 0.05, 0.2, 1, 0), (0.20, 0.40, -0.1, 2, 0), (0.01, 0.05, 0.0, 1, 1), (0.09, 0.05, 0.0, 0, 1)]
    dx = 1.0 / n_zones
    x = -0.5 + dx * (np.arange(n_zones) + 0.5)
    y = np.stack([l * (x < 0) + r * (x > 0) + k * x for l, r, k, _, _ in table], axis=1)
    comp = np.array([[t[3] for t in table], [t[4] for t in table]], np.int32)
    return comp, x, np.ascontiguousarray(y), np.ones(n_zones), dx


def make_advection_batch(n_species: int, n_elem: int, n_cells: int, seed: int = BASE_SEED + 2000):
    """Seeded synthetic 1-D field for the advection kernel's parity and bandwidth runs: random species compositions
    (the first n_elem species are atoms), abundances with smooth waves, jumps and flat stretches, density and velocity
    fields of both signs.  Returns (composition [E, S], y [n_cells, S], rho [n_cells], mass_flux [n_cells])."""
    rng = np.random.default_rng(seed)
    comp = np.zeros((n_elem, n_species), np.int32)
    for s in range(n_species):
        if s < n_elem:
            comp[s, s] = 1
        else:
            k = rng.integers(1, min(3, n_elem) + 1)
            for e in rng.choice(n_elem, size=k, replace=False):
                comp[e, s] = rng.integers(1, 4)
    xi = np.linspace(0.0, 1.0, n_cells, endpoint=False)
    y = np.empty((n_cells, n_species))
    for s in range(n_species):
        wave = 0.5 + 0.4 * np.sin(2 * np.pi * (rng.integers(1, 9) * xi + rng.random()))
        jump = np.where((xi > rng.random()) ^ (xi > rng.random()), rng.random(), 0.0)
        flat = np.where(np.sin(2 * np.pi * rng.integers(1, 5) * xi) > 0.3, 1.0, 0.0)
        y[:, s] = (wave * flat + jump + 1e-3) * 10.0 ** rng.uniform(-6, 0)
    rho = 1.0 + 0.5 * np.sin(2 * np.pi * 3 * xi + 1.0)
    vel = np.sin(2 * np.pi * 2 * xi + 0.3) + 0.2
    flux = np.where(vel > 0, np.roll(rho, 1), rho) * vel
    return comp, np.ascontiguousarray(y), rho, flux


# --------------------------------------------------------------------------
# ray tracing (NEXT-3: PAPER.md section 3) -- inputs only, no method arithmetic
# --------------------------------------------------------------------------

def make_ray_case(shape=(16, 12, 10), n_oblique: int = 64, n_abs: int = 3, n_bins: int = 4, seed: int = BASE_SEED + 3000,
                  spacing=(0.25, 0.25, 0.25), columns: bool = True):
    """Seeded synthetic input of the Cartesian ray tracer: absorber densities with ten decades of optical depth per cell,
    cross sections per absorber and energy bin, and rays -- one plane-parallel ray along +x through the centre of every
    (y, z) column (the plane-parallel source of PAPER.md Fig. 2) plus n_oblique rays from points outside the mesh in
    random directions (some miss the mesh).  Returns a dict of numpy arrays."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = shape
    h = np.asarray(spacing, np.float64)
    n_dens = 10.0 ** rng.uniform(-3, 3, size=(n_abs, nx, ny, nz))
    sigma = 10.0 ** rng.uniform(-2.5, 0.5, size=(n_abs, n_bins)) / (nx * h[0])        # tau per cell ~ 1e-7 .. 1e2
    org, drc = [], []
    if columns:
        for j in range(ny):
            for k in range(nz):
                org.append([-1.0, (j + 0.5) * h[1], (k + 0.5) * h[2]]); drc.append([1.0, 0.0, 0.0])
    centre = 0.5 * h * np.asarray(shape)
    for _ in range(n_oblique):
        d = rng.normal(size=3); d /= np.linalg.norm(d)
        target = centre + rng.uniform(-0.7, 0.7, 3) * h * np.asarray(shape)           # some targets lie outside: misses
        org.append(list(target - d * 2.0 * np.linalg.norm(h * np.asarray(shape)))); drc.append(list(d))
    org = np.asarray(org, np.float64); drc = np.asarray(drc, np.float64)
    L = 10.0 ** rng.uniform(0, 3, size=(org.shape[0], n_bins))
    return dict(shape=tuple(shape), spacing=tuple(float(v) for v in h), origins=org, directions=drc, L=L, sigma=sigma,
                n_dens=np.ascontiguousarray(n_dens))


# --------------------------------------------------------------------------
# tabulated reaction rates (NEXT-4: PAPER.md:171) -- inputs only: a table is DATA the user reads in; here it is filled from
# the network's own rate law so that tests can compare the tabulated run with the analytic one
# --------------------------------------------------------------------------

@dataclass
class RateTable:
    ln_k: np.ndarray             # [n_tab, n_rho, n_T] natural log of the rate coefficient at the nodes
    ln_rho0: float
    d_ln_rho: float
    ln_T0: float
    d_ln_T: float
    reactions: List[int]         # the reaction of the network each table replaces


def make_rate_table(net: Network, reactions, T_range=(5.0e3, 3.0e5), n_T: int = 257, rho_range=(1.0e-24, 1.0e-14),
                    n_rho: int = 1, rho_exponent: float = 0.0) -> RateTable:
    """Tables of the listed (irreversible Arrhenius) reactions of ``net`` on nodes uniform in ln rho and ln T:
    ln k = ln A + beta ln(T / T_REF) - Ea / T + rho_exponent ln(rho / rho_range[0]) (the density factor only makes the
    table two-dimensional; 0 = none)."""
    lnT = np.linspace(math.log(T_range[0]), math.log(T_range[1]), n_T)
    lnr = np.linspace(math.log(rho_range[0]), math.log(rho_range[1]), n_rho) if n_rho > 1 else np.array([math.log(rho_range[0])])
    ln_k = np.empty((len(reactions), n_rho, n_T))
    for t, r in enumerate(reactions):
        base = math.log(net.A[r]) + net.beta[r] * (lnT - math.log(T_REF)) - net.Ea_over_k[r] / np.exp(lnT)
        ln_k[t] = base[None, :] + rho_exponent * (lnr[:, None] - lnr[0])
    return RateTable(ln_k, float(lnr[0]), float(lnr[1] - lnr[0]) if n_rho > 1 else 1.0, float(lnT[0]),
                     float(lnT[1] - lnT[0]) if n_T > 1 else 1.0, [int(r) for r in reactions])


def tabulated_network(net: Network, table: RateTable) -> Network:
    """``net`` with every tabulated reaction turned into an aux-scaled one (KR_F_AUX_UNARY, A = 1): its rate coefficient is
    then the aux row n_aux + t of the cell, which the table interpolation fills."""
    import copy
    out = copy.deepcopy(net)
    for t, r in enumerate(table.reactions):
        assert net.flags[r] == 0, "only plain irreversible Arrhenius reactions are tabulated here"
        out.flags[r] = F_AUX_UNARY
        out.aux_index[r] = net.n_aux + t
        out.A[r] = 1.0; out.beta[r] = 0.0; out.Ea_over_k[r] = 0.0
    out.n_aux = net.n_aux + len(table.reactions)
    return out
