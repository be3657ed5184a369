"""Pins of the CPU oracle against things other than itself.

Each test checks the oracle against a closed form, an invariant, a library routine, brute force, or
values the paper prints -- chosen so that a dropped term, a wrong sign or index, or a transposed
operand in oracle/kr_oracle.cpp fails at least one of them.  CPU only.
"""
import itertools
import math
from fractions import Fraction

import numpy as np
import pytest

from paper_2504_04941_b200 import workloads as w
from tests import helpers as H

K_B, M_U, P0 = H.K_B, H.M_U, H.P0


def _opts(**kw):
    o = w.SolverOpts()
    for k, v in kw.items():
        setattr(o, k, v)
    return o


# ------------------------------------------------------------------------------------------------
# P1: linear A <-> B with constant k_f, k_r: one backward-Euler step multiplies the deviation from
# equilibrium by exactly 1 / (1 + (k_f + k_r) h); n steps by its n-th power; first order in h.
# ------------------------------------------------------------------------------------------------
def test_P1_linear_relaxation(oracle_mod):
    k1, k2 = 3.0e-3, 1.0e-3
    net = H.tiny_network([[1, 1]], [((0,), (1,), k1, 0, 0, w.F_CONST_UNARY, -1),
                                    ((1,), (0,), k2, 0, 0, w.F_CONST_UNARY, -1)])
    on = oracle_mod.OracleNetwork(net, _opts(h0_mode=0))
    y0 = np.array([0.9, 0.1]); tot = y0.sum(); yeq = tot * k2 / (k1 + k2)
    rho, T = 1e-20, 500.0
    for h in (1.0, 100.0, 1.0e4, 1.0e7):
        u, e, it, rc = on.be_substep(rho, T, y0, h)
        assert rc == 0 and it <= 2
        expect = yeq + (y0[0] - yeq) / (1.0 + (k1 + k2) * h)
        assert u[0] == pytest.approx(expect, rel=1e-13)
        assert u[0] + u[1] == pytest.approx(tot, rel=1e-14)
    # n whole steps through the public step call (h0_mode=0 -> one sub-step of h = dt each call)
    h, n = 50.0, 20
    cells = H.cells_of(rho, T, y0, h)
    for _ in range(n):
        Tn, yn, st, stats, _ = on.step(cells)
        assert stats["n_substeps"] == 1 and stats["n_failed"] == 0
        cells = H.cells_of(rho, T, yn, h)
    expect = yeq + (y0[0] - yeq) / (1.0 + (k1 + k2) * h) ** n
    assert cells.y[0, 0] == pytest.approx(expect, rel=1e-12)
    # first order: error against exp(-(k1+k2) t) halves with h
    errs = []
    t_end = 400.0
    for n in (64, 128, 256):
        y = y0.copy()
        for _ in range(n):
            y = on.be_substep(rho, T, y, t_end / n)[0]
        errs.append(abs(y[0] - (yeq + (y0[0] - yeq) * math.exp(-(k1 + k2) * t_end))))
    assert errs[0] / errs[1] == pytest.approx(2.0, rel=0.05)
    assert errs[1] / errs[2] == pytest.approx(2.0, rel=0.05)


# ------------------------------------------------------------------------------------------------
# P2: A + A -> A2 (rate k n_A^2, derivative 2 k n_A: eq. 19 first case, R9): the converged step is
# the positive root of 2 h k Ncal y^2 + y - y0 = 0; exact ODE solution y0 / (1 + 2 k Ncal y0 t).
# ------------------------------------------------------------------------------------------------
def test_P2_identical_reactants_quadratic(oracle_mod):
    k = 2.0e-11
    net = H.tiny_network([[1, 2]], [((0, 0), (1,), k, 0.0, 0.0, 0, -1)])
    on = oracle_mod.OracleNetwork(net, _opts(rtol=1e-13, max_newton=30))
    rho = 1.0e6 * M_U
    Ncal = rho / M_U
    y0 = np.array([0.7, 0.15])
    for h in (1.0e2, 1.0e4, 1.0e6):
        u, e, it, rc = on.be_substep(rho, 300.0, y0, h)
        a = 2.0 * h * k * Ncal
        root = (-1.0 + math.sqrt(1.0 + 4.0 * a * y0[0])) / (2.0 * a)
        assert rc == 0
        assert u[0] == pytest.approx(root, rel=1e-12)
        assert u[1] == pytest.approx(y0[1] + 0.5 * (y0[0] - root), rel=1e-12)   # one A2 per two A
    t_end, errs = 3.0e4, []
    for n in (200, 400):
        y = y0.copy()
        for _ in range(n):
            y = on.be_substep(rho, 300.0, y, t_end / n)[0]
        errs.append(abs(y[0] - y0[0] / (1.0 + 2.0 * k * Ncal * y0[0] * t_end)))
    assert errs[0] / errs[1] == pytest.approx(2.0, rel=0.05)


# ------------------------------------------------------------------------------------------------
# Eq. 15 written out with dense tensors A^i_jk, B^i_j (brute force on a tiny irreversible network).
# ------------------------------------------------------------------------------------------------
def test_rhs_equals_eq15_tensor_form(oracle_mod):
    rng = np.random.default_rng(7)
    # species: a b ab a2 ; element rows a, b
    comp = [[1, 0, 1, 2], [0, 1, 1, 0]]
    reacs = [((0, 1), (2,), 1e-10, 0, 0, 0, -1),      # a + b -> ab
             ((0, 0), (3,), 3e-11, 0, 0, 0, -1),      # a + a -> a2
             ((2,), (0, 1), 2e-4, 0, 0, w.F_CONST_UNARY, -1),   # ab -> a + b
             ((3, 1), (2, 0), 5e-10, 0, 0, 0, -1),    # a2 + b -> ab + a
             ((3,), (0, 0), 7.0, 0, 0, w.F_AUX_UNARY, 0)]       # a2 -> 2a, k = 7 * aux
    net = H.tiny_network(comp, reacs)
    on = oracle_mod.OracleNetwork(net)
    S = 4
    aux = np.array([3.0e-5])
    A = np.zeros((S, S, S)); B = np.zeros((S, S))
    for lhs, rhs, k, *_rest in reacs:
        fl, ax = _rest[2], _rest[3]
        kk = k * (aux[ax] if fl & w.F_AUX_UNARY else 1.0)
        d = np.zeros(S)
        for s in lhs: d[s] -= 1
        for s in rhs: d[s] += 1
        if len(lhs) == 2:
            A[:, lhs[0], lhs[1]] += kk * d
        else:
            B[:, lhs[0]] += kk * d
    rho = 4.0e5 * M_U
    for _ in range(5):
        y = rng.uniform(0.01, 1.0, S)
        n = y * rho / M_U
        ndot = np.einsum("ijk,j,k->i", A, n, n) + B @ n
        f = on.rhs(rho, 400.0, y, aux)
        np.testing.assert_allclose(f * rho / M_U, ndot, rtol=1e-13)


# ------------------------------------------------------------------------------------------------
# Arrhenius form (eq. 16 with reading R4) and the eq. 36 numbers the paper prints.
# ------------------------------------------------------------------------------------------------
def _golden_eq36():
    import os
    vals = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_eq36.txt")) as fh:
        for line in fh:
            line = line.split("#")[0].split()
            if len(line) == 2:
                vals[line[0]] = float(line[1])
    return vals


def test_arrhenius_matches_paper_eq36(oracle_mod):
    g = _golden_eq36()
    net = w.make_network(2)
    assert net.A[0] == g["A_ci"] and net.beta[0] == g["b_ci"]
    assert net.A[1] == g["A_rec"] and net.beta[1] == g["b_rec"]
    assert net.Ea_over_k[0] == pytest.approx(g["I_H_eV"] * w.EV / K_B, rel=2e-4)
    on = oracle_mod.OracleNetwork(net)
    for T in (1.0e2, 8.0e3, 1.0e4, 9.0e4):
        kf, kr = on.rate_constants(T, np.array([1e-12]))
        kci = g["A_ci"] * (T / g["T_ref"]) ** g["b_ci"] * math.exp(-net.Ea_over_k[0] / T)
        arec = g["A_rec"] * (T / g["T_ref"]) ** g["b_rec"]
        assert kf[0] == pytest.approx(kci, rel=1e-12)
        assert kf[1] == pytest.approx(arec, rel=1e-12)
        assert kf[2] == pytest.approx(1e-12, rel=1e-15)      # photo row: k = 1.0 * Gamma
        assert np.all(kr == 0.0)


# ------------------------------------------------------------------------------------------------
# P3: detailed balance.  k_f / k_r must equal K_c from the Gibbs function of the polynomials, and
# kinetics run to t -> infinity must land on it for every reversible reaction.
# ------------------------------------------------------------------------------------------------
def test_P3_detailed_balance(oracle_mod):
    net = w.make_network(0)
    on = oracle_mod.OracleNetwork(net, _opts(h0_mode=1))
    for T in (350.0, 1200.0, 2900.0):
        kf, kr = on.rate_constants(T)
        np.testing.assert_allclose(np.log(kf) - np.log(kr), H.ln_Kc(net, T), rtol=0, atol=1e-9)
    # kinetics run to equilibrium: the toy network's reactions with bond-like enthalpies and a dense gas,
    # so that every species keeps an abundance far above atol_y at equilibrium
    rng = np.random.default_rng(11)
    th = np.zeros((5, 7))
    th[:, 0] = rng.uniform(3.5, 4.5, 5); th[:, 1] = rng.uniform(0, 1, 5) / 6000.0
    th[:, 5] = np.array([0.0, 0.0, -8.0e4, -8.0e4, -8.0e4]) * rng.uniform(0.9, 1.1, 5)
    th[:, 6] = rng.uniform(-5.0, 10.0, 5)
    R = w.F_REVERSIBLE
    reacs = [((0, 0), (2,)), ((0, 1), (3,)), ((1, 1), (4,)), ((0, 3), (1, 2)), ((0, 4), (1, 3)), ((2, 4), (3, 3))]
    reacs = [(l, r, 1e-18 * rng.uniform(1, 10), rng.uniform(-1, 1), rng.uniform(0, 5e3), R, -1) for l, r in reacs]
    net = H.tiny_network(net.composition, reacs, thermo=th, elem_mass=[1.0, 12.0], T_hi=6000.0)
    on = oracle_mod.OracleNetwork(net, _opts(h0_mode=1))
    n = 8
    yy = rng.uniform(0.1, 1.0, (n, 5))
    cells = H.cells_of(1.0e-6, np.linspace(2200.0, 3000.0, n), yy, 1.0e-2)
    for _ in range(10):
        T, y, st, stats, _ = on.step(cells)
        assert stats["n_failed"] == 0
        cells = w.Cells(cells.rho, cells.T, y, None, cells.dt * 10)
    d = H.dnu_matrix(net)
    for c in range(n):
        nd = cells.y[c] * cells.rho[c] / M_U
        assert np.min(cells.y[c]) > 1e-12
        lnQ = d @ np.log(nd)                       # ln( prod n^nu'' / prod n^nu' )
        np.testing.assert_allclose(lnQ, H.ln_Kc(net, cells.T[c]), rtol=0, atol=1e-6)


# ------------------------------------------------------------------------------------------------
# P4: element (and charge) totals N.y unchanged before stage 2 runs.
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("idx,n", [(0, 256), (1, 128), (2, 256), (3, 48), (4, 24)])
def test_P4_element_conservation(oracle_mod, idx, n):
    net, cells, opts = w.make_config(idx, n)
    opts.finalize = 0
    on = oracle_mod.OracleNetwork(net, opts)
    T, y, st, stats, _ = on.step(cells, n_threads=4)
    assert stats["n_failed"] == 0
    Nm = net.composition.astype(float)
    before, after = cells.y @ Nm.T, y @ Nm.T
    scale = np.abs(cells.y) @ np.abs(Nm).T          # charge row sums to 0: scale by sum |N| y
    assert np.max(np.abs(after - before) / scale) < 1e-13
    # and with stage 2 on, totals are restored to rounding even when negatives were clamped
    opts.finalize = 1
    on.set_options(opts)
    T, y2, st, stats, _ = on.step(cells, n_threads=4)
    assert np.max(np.abs(y2 @ Nm.T - before) / scale) < 1e-14
    assert np.all(y2[(st & 64) == 0] >= 0.0)


# ------------------------------------------------------------------------------------------------
# P5: LU + substitution vs a library solver, Cramer's rule, and the factorisation identity P M = L U.
# ------------------------------------------------------------------------------------------------
def _apply_perm(M, p):
    M = M.copy()
    for j, pj in enumerate(p):
        if pj != j:
            M[[j, pj]] = M[[pj, j]]
    return M


@pytest.mark.parametrize("n", [1, 2, 3, 5, 6, 10, 33, 64])
def test_P5_lu_vs_library(oracle_mod, n):
    rng = np.random.default_rng(100 + n)
    for trial in range(6):
        M = rng.standard_normal((n, n))
        if trial % 2 and n > 1:
            M[np.arange(n), np.arange(n)] = 0.0          # forces row exchanges
        if trial == 4:
            M *= 10.0 ** rng.uniform(-8, 8, (n, 1))      # badly scaled rows
        b = rng.standard_normal(n)
        x, fac, p, rc = oracle_mod.lu_solve(M, b)
        assert rc == 0
        ref = np.linalg.solve(M.astype(np.longdouble).astype(float), b)
        cond = np.linalg.cond(M)
        np.testing.assert_allclose(x, ref, rtol=0, atol=1e-13 * cond * np.max(np.abs(ref)))
        L = np.tril(fac, -1) + np.eye(n); U = np.triu(fac)
        np.testing.assert_allclose(L @ U, _apply_perm(M, p), rtol=0, atol=1e-13 * np.max(np.abs(M)) * n)
        # same definition by a different algorithm: right-looking Gaussian elimination with the
        # implicit-scaled pivot rule must give the same permutation and the same factors
        W = M.copy(); v = np.max(np.abs(W), axis=1); pp = np.zeros(n, np.int32)
        for j in range(n):
            i = j + int(np.argmax(np.abs(W[j:, j]) / v[j:]))
            pp[j] = i
            W[[j, i]] = W[[i, j]]; v[[j, i]] = v[[i, j]]
            W[j + 1:, j] /= W[j, j]
            W[j + 1:, j + 1:] -= np.outer(W[j + 1:, j], W[j, j + 1:])
        np.testing.assert_array_equal(p, pp)
        np.testing.assert_allclose(fac, W, rtol=0, atol=1e-11 * np.max(np.abs(W)))


def test_P5_cramer_and_pivot_rule(oracle_mod):
    rng = np.random.default_rng(5)
    for n in (2, 3):
        for _ in range(10):
            Mi = rng.integers(-9, 10, (n, n)); bi = rng.integers(-9, 10, n)
            det = Fraction(int(round(np.linalg.det(Mi))))
            if det == 0:
                continue
            def fdet(A):
                if len(A) == 2:
                    return A[0][0] * A[1][1] - A[0][1] * A[1][0]
                return sum((-1) ** j * A[0][j] * fdet([row[:j] + row[j + 1:] for row in A[1:]]) for j in range(len(A)))
            A = [[Fraction(int(v)) for v in row] for row in Mi]
            D = fdet(A)
            exact = []
            for j in range(n):
                Aj = [row[:j] + [Fraction(int(bi[i]))] + row[j + 1:] for i, row in enumerate(A)]
                exact.append(float(fdet(Aj) / D))
            x, _, _, rc = oracle_mod.lu_solve(Mi.astype(float), bi.astype(float))
            assert rc == 0
            np.testing.assert_allclose(x, exact, rtol=1e-12, atol=1e-13)
    # implicit scaling: row 1 has the larger entry in column 0, but relative to its own row scale
    # row 0 wins (|1|/1 > |2|/1e6) -- Algorithm 1 line 5, t_i = |a_ij| / v_i
    M = np.array([[1.0, 0.5], [2.0, 1.0e6]])
    _, _, p, rc = oracle_mod.lu_solve(M, np.ones(2))
    assert rc == 0 and p[0] == 0
    M = np.array([[1.0, 1.0e6], [2.0, 1.0]])
    _, _, p, rc = oracle_mod.lu_solve(M, np.ones(2))
    assert rc == 0 and p[0] == 1
    # ties -> smallest row index
    M = np.array([[2.0, 1.0, 0.0], [2.0, 0.0, 1.0], [-2.0, 1.0, 1.0]])
    _, _, p, rc = oracle_mod.lu_solve(M, np.ones(3))
    assert rc == 0 and p[0] == 0
    # singular and zero-row matrices are reported, not solved
    assert oracle_mod.lu_solve(np.array([[1.0, 2.0], [2.0, 4.0]]), np.ones(2))[3] == -1
    assert oracle_mod.lu_solve(np.array([[1.0, 2.0], [0.0, 0.0]]), np.ones(2))[3] == -1


# ------------------------------------------------------------------------------------------------
# P6: analytic Jacobian vs the complex-step derivative of f.  Species rows and the T column must
# match; the T row matches once the two dropped dC terms are added back.
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("idx", [0, 1, 2, 3, 4])
def test_P6_jacobian_complex_step(oracle_mod, idx):
    net, cells, _ = w.make_config(idx, 4)
    on = oracle_mod.OracleNetwork(net)
    S, N = net.n_species, net.n_unknowns
    eps = 1e-30
    for c in range(4):
        aux = None if cells.aux is None else cells.aux[:, c]
        rho, T, y = cells.rho[c], cells.T[c], cells.y[c]
        J = on.jacobian(rho, T, y, aux)
        f = on.rhs(rho, T, y, aux)
        Jcs = np.zeros((N, N))
        for m in range(N):
            yc = y.astype(complex); Tc = complex(T)
            if m < S:
                yc[m] += 1j * eps
            else:
                Tc += 1j * eps
            Jcs[:, m] = on.rhs_complex(rho, Tc, yc, aux).imag / eps
        Jfix = J.copy()
        if net.energy_equation:
            a = np.where((T <= net.T_mid)[:, None], net.nasa_lo, net.nasa_hi)
            chat = H.nasa_cp_R(a, T) - 1.0
            dchat = a[:, 1] + 2 * a[:, 2] * T + 3 * a[:, 3] * T ** 2 + 4 * a[:, 4] * T ** 3
            C = y @ chat
            Jfix[S, :S] -= f[S] * chat / C                 # dC/dy_m term
            Jfix[S, S] -= f[S] * (y @ dchat) / C           # dC/dT term
        # entrywise: |dJ| <= 1e-12 * (sum of |terms|), estimated by the row/column magnitudes
        rowscale = np.maximum(np.max(np.abs(Jcs), axis=1, keepdims=True), 1e-300)   # inert rows are all zero
        assert np.max(np.abs(Jfix - Jcs) / rowscale) < 1e-12
        scale = np.maximum(np.abs(Jcs), 1e-10 * rowscale)     # entries are sums of terms up to ~rowscale
        assert np.max(np.abs(Jfix - Jcs) / scale) < 1e-5
        # columns of the species block lie in null(N): element totals have zero derivative (eq. 7)
        Nm = net.composition.astype(float)
        assert np.max(np.abs(Nm @ J[:S, :]) / (np.abs(Nm) @ np.abs(J[:S, :]) + 1e-300)) < 1e-12


# ------------------------------------------------------------------------------------------------
# P7: hydrogen ionisation balance (eq. 35, third relation, with eq. 36 coefficients).
# ------------------------------------------------------------------------------------------------
def test_P7_hydrogen_ionisation_balance(oracle_mod):
    g = _golden_eq36()
    net = w.make_network(2)
    on = oracle_mod.OracleNetwork(net, _opts(h0_mode=1))
    I_over_k = net.Ea_over_k[0]
    WH = net.weights[0]
    for T, nH, Gam in [(1.0e4, 1.0e2, 1.0e-12), (2.0e4, 1.0, 1.0e-14), (5.0e3, 1.0e3, 1.0e-10), (8.0e4, 10.0, 1e-16)]:
        kci = g["A_ci"] * (T / 300.0) ** g["b_ci"] * math.exp(-I_over_k / T)
        al = g["A_rec"] * (T / 300.0) ** g["b_rec"]
        a, b, c = (al + kci) * nH, (Gam - kci * nH), -Gam
        x_eq = (-b + math.sqrt(b * b - 4 * a * c)) / (2 * a)
        rho = nH * WH * M_U
        x0 = 0.3
        y = np.array([(1 - x0), x0, x0, 0, 0, 0]) * nH * M_U / rho
        # one backward-Euler step is a scalar quadratic in x'
        h = 0.5 / (al * nH + Gam + kci * nH)
        u, e, it, rc = on.be_substep(rho, T, y, h, np.array([Gam]))
        qa, qb, qc = h * (al + kci) * nH, 1 + h * Gam - h * kci * nH, -(x0 + h * Gam)
        x1 = (-qb + math.sqrt(qb * qb - 4 * qa * qc)) / (2 * qa)
        assert rc == 0
        assert u[1] / (u[0] + u[1]) == pytest.approx(x1, rel=1e-9)
        # long time: the positive root of eq. 35
        cells = H.cells_of(rho, T, y, 1.0e4 / (al * nH + Gam + kci * nH), aux=[[Gam]])
        for _ in range(3):
            Tn, yn, st, stats, _ = on.step(cells)
            cells = H.cells_of(rho, T, yn, cells.dt, aux=[[Gam]])
        xe = cells.y[0, 2] / (cells.y[0, 0] + cells.y[0, 1])
        assert xe == pytest.approx(x_eq, rel=1e-7)
        assert cells.y[0, 1] == pytest.approx(cells.y[0, 2], rel=1e-12)        # charge neutrality


# ------------------------------------------------------------------------------------------------
# P8: K = 1 is the textbook semi-implicit Euler step u_n + h (I - hJ)^-1 f(u_n) (reading R1).
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("idx", [0, 1, 3])
def test_P8_single_newton_is_semi_implicit_euler(oracle_mod, idx):
    net, cells, opts = w.make_config(idx, 3)
    opts.max_newton = 1
    opts.fixed_newton = 1
    on = oracle_mod.OracleNetwork(net, opts)
    N, S = net.n_unknowns, net.n_species
    for c in range(3):
        aux = None if cells.aux is None else cells.aux[:, c]
        rho, T, y = cells.rho[c], cells.T[c], cells.y[c]
        f = on.rhs(rho, T, y, aux)
        J = on.jacobian(rho, T, y, aux)
        un = np.concatenate([y, [T]]) if net.energy_equation else y.copy()
        h = 0.05 / np.max(np.abs(f[:S]) / (np.abs(y) + 1e-12))
        expect = un + np.linalg.solve(np.eye(N) - h * J, h * f)
        u, e, it, rc = on.be_substep(rho, T, y, h, aux)
        np.testing.assert_allclose(u, expect, rtol=1e-10, atol=1e-25)


# ------------------------------------------------------------------------------------------------
# P9: adiabatic closed system: E = sum_s y_s (H_s(T)/R - T) is an ODE invariant; backward Euler keeps
# only linear invariants, so the per-step drift is O(h^2): halving h quarters it.
# ------------------------------------------------------------------------------------------------
def _energy(net, y, T):
    a = np.where((T <= net.T_mid)[:, None], net.nasa_lo, net.nasa_hi)
    return float(y @ (T * (H.nasa_h_RT(a, T) - 1.0)))


def test_P9_adiabatic_energy_drift_second_order(oracle_mod):
    # A -> B at a constant rate with a large heat of reaction: T rises by ~1e3 K in one step, so the
    # bilinear invariant E = sum y_s (H_s(T)/R - T) shows the O(h^2) drift far above rounding.
    k = 1.0e-3
    th = [[3.5, 1.0e-4, 0, 0, 0, 0.0, 1.0], [4.0, 2.0e-4, 0, 0, 0, -5.0e4, 2.0]]
    net = H.tiny_network([[1, 1]], [((0,), (1,), k, 0, 0, w.F_CONST_UNARY, -1)], thermo=th, energy=1, T_hi=1.0e5)
    on = oracle_mod.OracleNetwork(net, _opts(max_newton=20, fixed_newton=1))
    y0, T0, rho = np.array([0.8, 0.2]), 1000.0, 1e-18
    E0 = _energy(net, y0, T0)
    drift = []
    for hk in (0.08, 0.04, 0.02, 0.01):
        u, e, it, rc = on.be_substep(rho, T0, y0, hk / k)
        assert rc == 0 and e <= 1
        assert u[2] > T0 + 100.0 * hk / 0.01                  # exothermic: T goes up, by a lot
        drift.append((_energy(net, u[:2], u[2]) - E0) / abs(E0))
    assert abs(drift[-1]) > 1e-7
    for a, b in zip(drift[:-1], drift[1:]):
        assert a / b == pytest.approx(4.0, rel=0.12)
    assert drift[2] / drift[3] == pytest.approx(4.0, rel=0.04)
    # Tdot is exactly what makes dE/dt = 0 at a point (combustion config, many species)
    net, cells, opts = w.make_config(1, 8)
    on = oracle_mod.OracleNetwork(net, opts)
    S = net.n_species
    for c in range(8):
        rho, T, y = cells.rho[c], cells.T[c], cells.y[c]
        f = on.rhs(rho, T, y)
        a = np.where((T <= net.T_mid)[:, None], net.nasa_lo, net.nasa_hi)
        terms = f[:S] * T * (H.nasa_h_RT(a, T) - 1.0)
        dEdt = terms.sum() + f[S] * (y @ (H.nasa_cp_R(a, T) - 1.0))
        assert abs(dEdt) < 1e-12 * np.sum(np.abs(terms))


# ------------------------------------------------------------------------------------------------
# P10: the long-double witness agrees with the double oracle on converged, well-separated cells.
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("idx,n,min_frac", [(0, 2048, 0.99), (1, 256, 1.0), (2, 1024, 1.0), (3, 96, 1.0), (4, 48, 0.7)])
def test_P10_long_double_witness(oracle_mod, idx, n, min_frac):
    """Where the step is well conditioned in fp64, carrying it in long double changes nothing above 1e-11.

    Config 0 takes h = dt first (Newton from a far guess; a few cells per thousand follow a different
    accept/reject path) and config 4's hot cells (T > 1e3 K, stiffness ratio ~1e10 with reversible
    reactions) are not resolved by fp64: those cells are what the witness is for -- the GPU parity tests
    exclude them by the same measure.
    """
    net, cells, opts = w.make_config(idx, n, fixed_newton=1)
    on = oracle_mod.OracleNetwork(net, opts)
    T, y, st, stats, margins = on.step(cells, n_threads=4, want_margins=True)
    Tw, yw, stw, statsw, _ = on.step(cells, n_threads=4, witness=True)
    ok = ((st & 8) == 0) & ((stw & 8) == 0)
    floor = 1e-20
    rel = np.abs(y - yw) / np.maximum(np.abs(yw), floor)
    rel = np.where(np.maximum(np.abs(y), np.abs(yw)) > floor, rel, 0.0)
    alpha = rel.max(axis=1)
    if net.energy_equation:
        alpha = np.maximum(alpha, np.abs(T - Tw) / Tw)
    assert np.mean(alpha[ok] < 1e-11) >= min_frac
    if idx == 4:      # the ill-conditioned cells are the hot ones, as the stiffness argument says
        assert np.all(cells.T[ok & (alpha > 1e-9)] > 500.0)


# ------------------------------------------------------------------------------------------------
# Controller bookkeeping: t lands on dt exactly, failed cells are reverted, T is clamped.
# ------------------------------------------------------------------------------------------------
def test_controller_bookkeeping(oracle_mod):
    k = 1.0e-3
    net = H.tiny_network([[1, 1]], [((0,), (1,), k, 0, 0, w.F_CONST_UNARY, -1)], T_lo=100.0, T_hi=1000.0)
    on = oracle_mod.OracleNetwork(net, _opts(h0_mode=1))
    y0 = np.array([[1.0, 0.0]])
    # many sub-steps of growing size must add up to dt: compare with the product of the step factors
    T, y, st, stats, _ = on.step(H.cells_of(1e-20, 5000.0, y0, 1.0e3))
    assert st[0] & 16                                     # T was outside [T_lo, T_hi] -> clamped flag
    assert stats["n_substeps"] > 1 and stats["n_failed"] == 0
    assert 0.0 < y[0, 0] < math.exp(-1.0) * 1.6           # backward Euler lags the exact e^-1 = 0.37
    assert y[0, 0] + y[0, 1] == pytest.approx(1.0, rel=1e-14)
    # impossible tolerance -> every sub-step rejected -> cell reverted, flagged, input returned
    on.set_options(_opts(h0_mode=0, max_newton=1, fixed_newton=0, rtol=1e-30, atol_y=1e-300))
    net2 = H.tiny_network([[1, 2]], [((0, 0), (1,), 1e-10, 0.0, 0.0, 0, -1)])
    on2 = oracle_mod.OracleNetwork(net2, _opts(h0_mode=0, max_newton=1, rtol=1e-30, atol_y=1e-300))
    yin = np.array([[0.5, 0.25]])
    T, y, st, stats, _ = on2.step(H.cells_of(1e6 * M_U, 300.0, yin, 1.0e9))
    assert st[0] & 8 and stats["n_failed"] == 1
    np.testing.assert_array_equal(y, yin)


# ------------------------------------------------------------------------------------------------
# External heating (eq. 15: d(eps)/dt = Gamma - Lambda): one unary reaction A -> B that deposits q_ext per
# event, constant c_v, equal formation enthalpies (no chemical heat): dT/dt = q_ext k y_A / (k_B C), C = sum y_s chat_s.
# ------------------------------------------------------------------------------------------------
def test_external_heat_term_closed_form(oracle_mod):
    k, q = 2.0e-4, 3.0e-12                                    # s^-1, erg per event (~1.9 eV)
    th = [[3.5, 0, 0, 0, 0, 0.0, 1.0], [4.5, 0, 0, 0, 0, 0.0, 2.0]]       # chat = 2.5, 3.5; a6 = 0 for both
    for sign in (+1.0, -1.0):                                 # heating and (formally) cooling
        net = H.tiny_network([[1, 1]], [((0,), (1,), k, 0, 0, w.F_CONST_UNARY, -1)], thermo=th, energy=1,
                             q_ext=[sign * q], T_hi=1.0e6)
        on = oracle_mod.OracleNetwork(net, _opts(max_newton=30, fixed_newton=0))
        y, T, rho = np.array([0.7, 0.3]), 500.0, 1e-18
        f = on.rhs(rho, T, y)
        C = 0.7 * 2.5 + 0.3 * 3.5
        # chemical part: -T sum uhat_s ydot_s with uhat = a1 - 1: ydot_A = -k y_A, ydot_B = +k y_A
        chem = -T * (2.5 * (-k * 0.7) + 3.5 * (k * 0.7)) / C
        ext = sign * q * k * 0.7 / (K_B * C)
        assert f[0] == pytest.approx(-k * 0.7, rel=1e-14) and f[1] == pytest.approx(k * 0.7, rel=1e-14)
        assert f[2] == pytest.approx(chem + ext, rel=1e-13)
        assert abs(ext) > 20 * abs(chem)                      # the external term dominates: its sign is what is tested
        # Jacobian of the heat term: dTdot/dy_A = q k / (k_B C) + chemical part (the dropped dC/dy term aside)
        J = on.jacobian(rho, T, y)
        assert J[2, 0] == pytest.approx((sign * q * k / K_B - T * (2.5 * (-k) + 3.5 * k)) / C, rel=1e-13)
        # over a step the temperature moves the way the deposited energy says
        u, e, it, rc = on.be_substep(rho, T, y, 0.02 / k)
        assert rc == 0 and e <= 1 and (u[2] - T) * sign > 10.0
        # energy bookkeeping of the converged backward-Euler step: sum_s y_s (H_s/R - T) changes by q (events) / k_B up to
        # the O(h^2) drift of P9
        dE = _energy(net, u[:2], u[2]) - _energy(net, y, T)
        events = y[0] - u[0]
        assert dE == pytest.approx(sign * q * events / K_B, rel=0.08)


# ------------------------------------------------------------------------------------------------
# The temperature clamp ("the check against effective temperature limits"): a cell fed T outside
# [T_lo, T_hi] must give bit-identical results to the same cell fed T_lo / T_hi, on a network whose rates depend on T.
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("energy", [0, 1])
def test_T_clamp_value(oracle_mod, energy):
    th = [[3.5, 1e-4, 0, 0, 0, -2.0e3, 1.0], [4.0, 2e-4, 0, 0, 0, 1.0e3, 2.0], [3.7, 0, 0, 0, 0, 0.0, 3.0]]
    net = H.tiny_network([[1, 1, 2]], [((0,), (1,), 1e-3, 0.7, 300.0, 0, -1), ((0, 1), (2,), 1e-12, -0.5, 150.0, w.F_REVERSIBLE, -1)],
                         thermo=th, energy=energy, T_lo=200.0, T_hi=900.0)
    on = oracle_mod.OracleNetwork(net, _opts())
    y0 = np.array([[0.5, 0.2, 0.1]])
    for T_fed, T_lim in ((20.0, 200.0), (199.999, 200.0), (5000.0, 900.0), (900.001, 900.0)):
        a = on.step(H.cells_of(1e-12, T_fed, y0, 50.0))
        b = on.step(H.cells_of(1e-12, T_lim, y0, 50.0))
        np.testing.assert_array_equal(a[1], b[1])
        assert (a[2][0] & 16) and not (b[2][0] & 16)
        if energy:
            np.testing.assert_array_equal(a[0], b[0])
        assert a[3] == b[3]
        # and the rate constants used are those at the limit: f(u_in) at T_lim drives the first sub-step
    # a cell inside the range gives something else (the clamp is not a constant)
    c = on.step(H.cells_of(1e-12, 500.0, y0, 50.0))
    assert np.abs(c[1] - b[1]).max() > 1e-6


# ------------------------------------------------------------------------------------------------
# Decision margins (tests/parity.py uses them to decide which cells are comparable): on the linear A <-> B system of P1
# Newton lands on the solution in ONE iteration, so e_1 = |delta| / (rtol |u_1| + atol) is known in closed form; the
# reported margin must be the relative distance of the closest decision value to its threshold.
# ------------------------------------------------------------------------------------------------
def test_decision_margins_closed_form(oracle_mod):
    kf, kr_ = 3.0e-3, 1.0e-3
    net = H.tiny_network([[1, 1]], [((0,), (1,), kf, 0, 0, w.F_CONST_UNARY, -1), ((1,), (0,), kr_, 0, 0, w.F_CONST_UNARY, -1)])
    y0 = np.array([0.9, 0.1])
    h = 200.0
    ktot = kf + kr_
    yeq = kr_ / ktot
    yA1 = yeq + (y0[0] - yeq) / (1.0 + ktot * h)               # P1's closed form
    d = abs(yA1 - y0[0])
    for target in (1.0 + 1e-3, 1.0 - 1e-3, 1.0 + 1e-7, 3.0):
        # pick rtol so that e_1 = d / (rtol * min(u_A, u_B)) = target (atol = 0; the smaller abundance sets the maximum)
        small = min(yA1, 1.0 - yA1)
        rtol = d / (target * small)
        o = _opts(h0_mode=0, fixed_newton=1, max_newton=2, rtol=rtol, atol_y=0.0, finalize=0)
        on = oracle_mod.OracleNetwork(net, o)
        T, y, st, stats, margins = on.step(H.cells_of(1e-20, 300.0, y0[None, :], h), want_margins=True)
        assert y[0, 0] == pytest.approx(yA1, rel=1e-13)
        # decisions taken: e_1 against 1 (the closed form), e_2 ~ 0 against 1 (margin 1), h against dt (an exact tie: skipped)
        expect = abs(target - 1.0) / max(target, 1.0)
        assert margins[0] == pytest.approx(expect, rel=2e-6 / max(expect, 1e-7) * 1e-7 + 1e-3)


# ---- P11: post-processing stages 1-3 (readings R12 / R23) -------------------------------------------
def _post_net():
    # elements a, b; species: a, b, a2 (single-element, a row), ab, ab2 (compounds); one reaction keeps the network valid
    return H.tiny_network([[1, 0, 2, 1, 1], [0, 1, 0, 1, 2]], [((0, 1), (3,), 1e-10, 0.0, 0.0, 0, -1)])


def test_P11_stages_1_2_restore_what_stage_1_added(oracle_mod):
    """Stage 1 zeroes negatives, stage 2 takes the amount that added to each element from the largest single-element
    species of that element; computed here with exact fractions."""
    on = oracle_mod.OracleNetwork(_post_net(), w.SolverOpts())
    y = np.array([0.30, 0.20, 0.05, -0.01, 0.40])           # ab negative: stage 1 adds 0.01 a and 0.01 b
    yo, st = on.finalize(y)
    exp = [Fraction(30, 100) - Fraction(1, 100), Fraction(20, 100) - Fraction(1, 100), Fraction(5, 100), 0, Fraction(40, 100)]
    assert st == 2                                           # CLAMPED_NEG only
    np.testing.assert_allclose(yo, [float(x) for x in exp], rtol=0, atol=6e-17)
    # the reservoir is the LARGEST single-element species: with a2 > a the a-row correction goes to a2 (2 atoms each)
    y2 = np.array([0.01, 0.20, 0.30, -0.02, 0.40])
    yo2, st2 = on.finalize(y2)
    np.testing.assert_allclose(yo2, [0.01, 0.18, 0.30 - 0.02 / 2, 0.0, 0.40], rtol=0, atol=6e-17)
    # nothing negative: untouched, no bits
    y3 = np.array([0.1, 0.2, 0.3, 0.0, 0.4])
    yo3, st3 = on.finalize(y3)
    assert st3 == 0 and np.array_equal(yo3, y3)


def test_P11_stage_3_disintegrates_the_most_abundant_compound_just_enough(oracle_mod):
    net = _post_net()
    on = oracle_mod.OracleNetwork(net, w.SolverOpts())
    comp = net.composition.astype(np.float64)
    # stage 1 clamps ab (-0.05): stage 2 wants 0.05 a from `a` (0.01) and 0.05 b from `b` (0.30): `a` goes to -0.04.
    y = np.array([0.01, 0.30, 0.005, -0.05, 0.40])
    yo, st = on.finalize(y)
    assert st == (2 | 128), st                               # CLAMPED_NEG | STAGE3, NEEDS_STAGE3 cleared
    assert yo.min() >= 0.0
    np.testing.assert_allclose(comp @ yo, comp @ y, rtol=0, atol=6e-17)     # every element total unchanged
    # the most abundant compound holding `a` is ab2 (0.40): it gives up exactly 0.04 molecules -> 0.04 a and 0.08 b;
    # the a reservoir ends at exactly zero, ab stays clamped, a2 is untouched
    np.testing.assert_allclose(yo, [0.0, 0.30 - 0.05 + 0.08, 0.005, 0.0, 0.40 - 0.04], rtol=0, atol=6e-17)
    assert yo[0] == 0.0
    # not enough of ab2: it is used up, then the next compound (none left but ab = 0) -> NEEDS_STAGE3 stays, totals still hold
    y2 = np.array([0.01, 0.30, 0.005, -0.05, 0.03])
    yo2, st2 = on.finalize(y2)
    assert st2 == (2 | 64 | 128)          # clamped, ab2 was taken apart (STAGE3), the a reservoir is still negative (NEEDS_STAGE3)
    np.testing.assert_allclose(comp @ yo2, comp @ y2, rtol=0, atol=6e-17)
    assert yo2[4] == 0.0 and yo2[0] < 0.0
    # two compounds needed: ab2 (0.03) is exhausted, ab (0.02) covers the remaining 0.01
    y3 = np.array([0.01, 0.30, 0.005, 0.02, 0.03])
    y3n = y3.copy(); y3n[2] = -0.025                          # a2 negative: stage 2 takes 0.05 a from `a`
    yo3, st3 = on.finalize(y3n)
    assert st3 == (2 | 128) and yo3.min() >= 0.0
    np.testing.assert_allclose(comp @ yo3, comp @ y3n, rtol=0, atol=6e-17)
    np.testing.assert_allclose(yo3, [0.0, 0.30 + 0.06 + 0.01, 0.0, 0.01, 0.0], rtol=0, atol=6e-17)


def test_P11_stage_3_leaves_charged_compounds_alone(oracle_mod):
    """Config 2 has only ions as multi-row species: nothing to disintegrate, the flag stays (R23)."""
    net = w.make_network(2)
    on = oracle_mod.OracleNetwork(net, w.default_opts(2))
    y = np.array([1e-6, 0.5, 0.4, 0.05, -0.2, 0.01])          # H, H+, e-, He, He+ (negative), He++
    yo, st = on.finalize(y)
    comp = net.composition.astype(np.float64)
    np.testing.assert_allclose(comp @ yo, comp @ y, rtol=0, atol=1e-16)
    assert (st & 64) and not (st & 128) and yo[3] < 0.0


def test_P11_random_states_conserve_and_end_non_negative(oracle_mod):
    net = w.make_network(3)
    on = oracle_mod.OracleNetwork(net, w.default_opts(3))
    comp = net.composition.astype(np.float64)
    rng = np.random.default_rng(11)
    n3 = 0
    for _ in range(300):
        y = 10.0 ** rng.uniform(-8, -3, net.n_species)
        neg = rng.choice(net.n_species, size=rng.integers(1, 4), replace=False)
        y[neg] *= -rng.uniform(0.1, 30.0, neg.size)
        yo, st = on.finalize(y)
        tot, tot0 = comp @ yo, comp @ y
        assert np.max(np.abs(tot - tot0) / np.abs(comp @ np.abs(y))) < 1e-14
        if st & 128:
            n3 += 1
        if not (st & (32 | 64)):
            assert yo.min() >= 0.0
    assert n3 >= 20                                           # stage 3 was exercised


def test_P11_stage_2_initial_minus_final_totals(oracle_mod):
    """PAPER.md:215 literally: 'Abundances of elements are calculated for the initial and final states ... the abundances
    in the single-element species are adjusted to compensate the differences.'  With an initial state given, a row whose
    initial-minus-final total exceeds cons_tol x sum|N||y_in| is compensated IN FULL (solver drift included); below the
    threshold only what stage 1 clamped is compensated (reading R12).  Exact fractions."""
    net = _post_net()
    comp = net.composition.astype(np.float64)
    o = w.SolverOpts()
    on = oracle_mod.OracleNetwork(net, o)
    y_in = np.array([0.30, 0.20, 0.05, 0.10, 0.40])
    # final state: the a row lost 3e-3 atoms (a real violation, >> 1e-13), the b row drifted by 1e-15 (rounding level);
    # nothing negative
    y_f = y_in.copy(); y_f[0] -= 1e-3; y_f[2] -= 1e-3; y_f[1] += 1e-15
    yo, st = on.finalize(y_f, y_in)
    assert st == 0
    # a row: the largest single-row species is `a` (0.299 > a2 = 0.049): it receives the 3e-3 missing atoms; b untouched
    np.testing.assert_allclose(yo, [0.299 + 3e-3, 0.20 + 1e-15, 0.049, 0.10, 0.40], rtol=0, atol=6e-17)
    assert abs((comp @ yo - comp @ y_in)[0]) < 3e-16 and (comp @ yo - comp @ y_in)[1] == pytest.approx(1e-15, rel=0.2)
    # with a clamp in a drifting row the compensation is drift + clamp: ab = -0.01 clamped adds 0.01 a and 0.01 b,
    # the a row additionally lost 2e-3 -> `a` gets +2e-3 - 0.01, b (row within tolerance) only -0.01
    y_f2 = y_in.copy(); y_f2[0] -= 2e-3; y_f2[3] = -0.01
    y_in2 = y_in.copy(); y_in2[3] = -0.01 + 0.0                     # the initial ab equals the final one: only `a` moved
    yo2, st2 = on.finalize(y_f2, y_in2)
    assert st2 == 2
    np.testing.assert_allclose(yo2, [0.298 + 2e-3 - 0.01, 0.20 - 0.01, 0.05, 0.0, 0.40], rtol=0, atol=6e-17)
    # cons_tol = inf: never more than the clamped amount (the round-1 reading); cons_tol = 0: always the full difference
    o.cons_tol = float("inf")
    yo3, _ = oracle_mod.OracleNetwork(net, o).finalize(y_f, y_in)
    np.testing.assert_array_equal(yo3, y_f)
    o.cons_tol = 0.0
    yo4, _ = oracle_mod.OracleNetwork(net, o).finalize(y_f, y_in)
    np.testing.assert_allclose(comp @ yo4, comp @ y_in, rtol=0, atol=3e-16)
    assert yo4[1] == pytest.approx(0.20, abs=1e-16) and yo4[1] != y_f[1]
    # through the step: a network whose Newton update does not conserve cannot be built (create validates N.dnu = 0), so
    # the step-level check is that totals after a full step equal the input totals to rounding on every config
    for idx, n in ((1, 64), (3, 24)):
        netc, cells, opts = w.make_config(idx, n)
        T, y, stc, stats, _ = oracle_mod.OracleNetwork(netc, opts).step(cells, n_threads=4)
        Nm = netc.composition.astype(np.float64)
        drift = np.abs((y - cells.y) @ Nm.T) / (np.abs(cells.y) @ np.abs(Nm).T)
        assert drift.max() <= 1.0e-13


def test_P11_stage_3_on_a_later_row_and_final_flags(oracle_mod):
    """Stage 3 for the SECOND row of the matrix (the b row): elements a, b; species a, b, ab2, b2.  NEEDS_STAGE3 is
    evaluated after all rows are processed: it is set iff some reservoir is still negative at the very end."""
    net = H.tiny_network([[1, 0, 1, 0], [0, 1, 2, 2]], [((0, 1, 1), (2,), 1e-30, 0.0, 0.0, 0, -1)])   # a, b, ab2, b2
    on = oracle_mod.OracleNetwork(net, w.SolverOpts())
    comp = net.composition.astype(np.float64)
    # b2 = -0.05 is clamped (adds 0.10 b); the b row's reservoir is the largest of {b = 0.01, b2 = 0}: b -> -0.09;
    # stage 3 takes ab2 apart: 0.045 molecules give back 0.09 b and release 0.045 a into `a`
    y = np.array([0.2, 0.01, 0.3, -0.05])
    yo, st = on.finalize(y)
    assert st == (2 | 128) and yo.min() >= 0.0
    np.testing.assert_allclose(comp @ yo, comp @ y, rtol=0, atol=6e-17)
    np.testing.assert_allclose(yo, [0.2 + 0.045, 0.0, 0.3 - 0.045, 0.0], rtol=0, atol=6e-17)
    # not enough ab2: used up, b stays negative -> both bits
    y2 = np.array([0.2, 0.01, 0.02, -0.05])
    yo2, st2 = on.finalize(y2)
    assert st2 == (2 | 64 | 128) and yo2[2] == 0.0 and yo2[1] == pytest.approx(-0.09 + 0.04, abs=1e-16)
    np.testing.assert_allclose(comp @ yo2, comp @ y2, rtol=0, atol=6e-17)


# ---- P12: the retry procedure (reading R24) --------------------------------------------------------------
def test_P12_retry_second_attempt_with_tightened_control(oracle_mod):
    """A + A -> A2 with a first sub-step (h = dt, 2 h k N y0 = 1e5) far beyond what K Newton iterations can resolve and a
    floor three decades below it: the first attempt is rejected five times and gives up.  With retry = 1 the cell is
    redone from the same input with first sub-step x retry_h0, shrink^2 and slower growth: it then integrates to dt.
    The result must be the backward-Euler approximation of y0 / (1 + 2 k N y0 t) (above it, within its O(h) error) and
    conserve a-atoms; both-fail cells are reverted and counted once."""
    net = H.tiny_network([[1, 2]], [((0, 0), (1,), 1e-10, 0.0, 0.0, 0, -1)])
    k, Ncal, dt = 1e-10, 1e6, 1e9
    y0 = np.array([[0.5, 0.25]])
    cells = H.cells_of(Ncal * H.M_U, 300.0, y0, dt)
    o = w.SolverOpts(); o.h0_mode = 0; o.max_newton = 6; o.h_min_rel = 1e-3
    T, y, st, stats, _ = oracle_mod.OracleNetwork(net, o).step(cells)
    assert st[0] == (8 | 1) and np.array_equal(y, y0) and stats["n_failed"] == 1 and stats["n_rejected"] == 5
    o.retry = 1
    T, y, st, stats1, _ = oracle_mod.OracleNetwork(net, o).step(cells)
    exact = y0[0, 0] / (1.0 + 2.0 * k * Ncal * y0[0, 0] * dt)
    assert st[0] == (256 | 1), st                                  # RETRIED | REJECTED_ONCE, not FAILED
    assert exact < y[0, 0] < 1.15 * exact
    assert abs((y[0, 0] + 2 * y[0, 1]) - (y0[0, 0] + 2 * y0[0, 1])) < 1e-14
    # counters add up over both attempts: 5 rejections of the first, then 0.01 dt and 0.01 dt / 16 rejected as well
    assert stats1["n_rejected"] == 5 + 2 and stats1["n_failed"] == 0 and stats1["n_rate_evals"] == 2
    # a smaller retry_h0 starts below the first acceptable size: fewer rejections in the second attempt
    o.retry_h0 = 1e-5
    _, y2, st2, stats2, _ = oracle_mod.OracleNetwork(net, o).step(cells)
    assert st2[0] == 256 and stats2["n_rejected"] == 5 and exact < y2[0, 0] < 1.15 * exact
    # both attempts fail: reverted, counted once, flagged FAILED | RETRIED
    o.retry_h0 = 0.01; o.max_newton = 4
    T, y3, st3, stats3, _ = oracle_mod.OracleNetwork(net, o).step(cells)
    assert st3[0] == (8 | 1 | 256) and np.array_equal(y3, y0) and stats3["n_failed"] == 1
