"""GPU parity of kr_table_rates (kr_tabrate.cuh) with oracle/table_oracle.py, element by element, and the
tabulated rates driving the chemistry step through the C ABI.

Tolerance: both sides evaluate the same formula; they differ in the last bit of log() and exp().  One ulp of ln T (2e-15 at
ln T ~ 10) moves ln k by |d ln k / d ln T| * 2e-15 <= (Ea / T + |beta|) * 2e-15, at most 1.3e-11 for the steepest table used
here (Ea / T = 6.3e3 at its cold end); 1e-10 relative is asserted."""
import dataclasses
import math

import numpy as np
import pytest

from paper_2504_04941_b200 import workloads as w

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2504_04941_b200 import binding
    binding.load()          # raises when libkratos_chem.so is missing: no fallback
    return binding


def _gpu_rates(B, table, rho, T):
    import torch
    dev = "cuda:0"
    lnk = torch.tensor(table.ln_k, device=dev)
    out = torch.full((table.ln_k.shape[0], rho.shape[0]), -1.0, dtype=torch.float64, device=dev)
    B.table_rates(lnk, table.ln_rho0, table.d_ln_rho, table.ln_T0, table.d_ln_T, torch.tensor(rho, device=dev),
                  torch.tensor(T, device=dev), out)
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("n_rho,n_T,n_cells", [(1, 4097, 3001), (7, 33, 2500), (5, 1, 777), (1, 1, 65), (3, 2, 1)])
def test_table_rates_match_oracle(B, n_rho, n_T, n_cells):
    from oracle import table_oracle as TO
    net, _, _ = w.make_config(2, 8)
    table = w.make_rate_table(net, [0, 1, 3, 4, 6, 7], T_range=(50.0, 2.0e5), n_T=n_T, n_rho=n_rho, rho_exponent=0.37)
    rng = np.random.default_rng(77 + n_cells)
    # cells inside, outside (clamped) and exactly on nodes of the table
    T = np.exp(rng.uniform(math.log(20.0), math.log(5.0e5), n_cells))
    rho = np.exp(rng.uniform(math.log(1e-26), math.log(1e-12), n_cells))
    T[: min(5, n_cells)] = np.exp(table.ln_T0 + table.d_ln_T * np.arange(min(5, n_cells)) * (1 if n_T > 4 else 0))
    k_gpu = _gpu_rates(B, table, rho, T)
    k_ref = TO.table_rates(table.ln_k, table.ln_rho0, table.d_ln_rho, table.ln_T0, table.d_ln_T, rho, T)
    assert np.all(np.isfinite(k_gpu)) and np.all(k_gpu >= 0.0)
    tiny = k_ref < 1e-300                                  # exp() of ln k < -690: denormal range, compared absolutely
    np.testing.assert_allclose(k_gpu[~tiny], k_ref[~tiny], rtol=1e-10, atol=0.0)
    assert np.all(k_gpu[tiny] < 1e-299)


@pytest.mark.parametrize("n_rho,n_T", [(1, 4097), (3, 1024)])
def test_table_rates_staged_path_matches_oracle(B, n_rho, n_T):
    """Batches of at least 1024 cells per SM take the kernel that stages the tables in shared memory (tables <= 200 KiB):
    the same values as the global-memory path and as the oracle, the latter on a seeded sample of the cells."""
    from oracle import table_oracle as TO
    net, _, _ = w.make_config(2, 8)
    table = w.make_rate_table(net, [0, 1, 3, 4, 6, 7], T_range=(50.0, 2.0e5), n_T=n_T, n_rho=n_rho, rho_exponent=0.37)
    assert table.ln_k.size * 8 <= 200 * 1024
    n_cells = 400_003                                      # > 1024 cells per SM on any part, ragged
    rng = np.random.default_rng(4242)
    T = np.exp(rng.uniform(math.log(20.0), math.log(5.0e5), n_cells))
    rho = np.exp(rng.uniform(math.log(1e-26), math.log(1e-12), n_cells))
    k_big = _gpu_rates(B, table, rho, T)
    assert np.all(np.isfinite(k_big)) and np.all(k_big >= 0.0)
    sample = np.concatenate([np.arange(64), rng.choice(n_cells, 3000, replace=False), np.arange(n_cells - 64, n_cells)])
    k_small = _gpu_rates(B, table, rho[sample], T[sample])              # 3 128 cells: the global-memory path
    np.testing.assert_array_equal(k_big[:, sample], k_small)
    k_ref = TO.table_rates(table.ln_k, table.ln_rho0, table.d_ln_rho, table.ln_T0, table.d_ln_T, rho[sample], T[sample])
    tiny = k_ref < 1e-300
    np.testing.assert_allclose(k_small[~tiny], k_ref[~tiny], rtol=1e-10, atol=0.0)


def test_empty_and_bad_arguments(B):
    import torch
    dev = "cuda:0"
    lnk = torch.zeros((1, 1, 2), dtype=torch.float64, device=dev)
    e = torch.zeros(0, dtype=torch.float64, device=dev)
    B.table_rates(lnk, 0.0, 1.0, 0.0, 1.0, e, e, e)                       # no cells: nothing to do
    one = torch.ones(1, dtype=torch.float64, device=dev)
    with pytest.raises(B.KrError, match="spacings"):
        B.table_rates(lnk, 0.0, 1.0, 0.0, 0.0, one, one, torch.zeros((1, 1), dtype=torch.float64, device=dev))


def test_tabulated_rates_drive_the_chemistry_step(B, oracle_mod):
    """Config 2 with its six thermal rate laws read from tables: kr_table_rates fills rows 1..6 of the aux array in place
    (row 0 is the photo rate), kr_thermochem_step_ex takes it; the result is compared with the chemistry oracle on the
    oracle's own table rates (parity of the chain), and with the analytic-rate run (interpolation error only)."""
    import torch
    from oracle import table_oracle as TO
    from tests import parity as P
    O = oracle_mod
    n = 1500
    net, cells, opts = w.make_config(2, n)
    table = w.make_rate_table(net, [0, 1, 3, 4, 6, 7], T_range=(50.0, 2.0e5), n_T=4097)
    tnet = w.tabulated_network(net, table)
    dev = "cuda:0"
    aux = torch.empty((tnet.n_aux, n), dtype=torch.float64, device=dev)
    aux[:1] = torch.tensor(cells.aux, device=dev)
    rho = torch.tensor(cells.rho, device=dev); T = torch.tensor(cells.T, device=dev); y = torch.tensor(cells.y, device=dev)
    B.table_rates(torch.tensor(table.ln_k, device=dev), table.ln_rho0, table.d_ln_rho, table.ln_T0, table.d_ln_T, rho, T, aux[1:])
    st = torch.zeros(n, dtype=torch.int32, device=dev)
    gn = B.Network(tnet, opts)
    gn.thermochem_step_ex(n, rho, T, y, cells.dt, B.KR_FP64, aux=aux, status=st)
    torch.cuda.synchronize()
    # the oracle chain on the same inputs
    k_ref = TO.table_rates(table.ln_k, table.ln_rho0, table.d_ln_rho, table.ln_T0, table.d_ln_T, cells.rho, cells.T)
    tcells = dataclasses.replace(cells, aux=np.ascontiguousarray(np.concatenate([cells.aux, k_ref], axis=0)))
    ref = P.oracle_reference(O, tnet, tcells, opts)
    out = P.compare(tnet, ref, T.cpu().numpy(), y.cpu().numpy(), st.cpu().numpy())
    assert out["n_comparable"] >= 0.9 * n
    # against the analytic rates: interpolation error only (measured 1e-6 in the oracle pin)
    _, y_an, _, _, _ = O.OracleNetwork(net, opts).step(cells)
    err = np.abs(y.cpu().numpy() - y_an) / np.abs(y_an).max(axis=1, keepdims=True)
    assert np.quantile(err, 0.99) < 1e-5
