"""Physics of BASELINE.json configs 1-2 run THROUGH THE CUDA PATH (-m gpu): long chains through sw_sweep +
sw_observables against what the model fixes -- the exact enumeration of the 4x4 periodic Ising model and Kaufman's
exact finite-lattice energy at L=1024 (the paper's own check, ref. [40]).  Bit-parity with the oracle makes
these redundant in principle; they pin the long-run chain (10^5 steps of the counter, handle reuse) that the
sweep-by-sweep parity tests do not reach.  The reference numbers are computed here (enumeration, closed form), not
by the oracle.
"""
import math

import numpy as np
import pytest

import oracle
from paper_1105_5804_b200 import binding
from test_oracle_physics import blocked_error, boltzmann_averages, enumerate_ising, kaufman_energy_per_site

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

BETA_C = oracle.beta_c(2)


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    if not torch.cuda.is_available():
        pytest.fail("these tests need a CUDA device (the product has no CPU path)")
    binding.lib()


@pytest.mark.parametrize("beta", [BETA_C, 0.50])
def test_config1_4x4_chain_reproduces_exact_enumeration(beta):
    """Config 1's "4x4 exact-enumeration check" on the GPU: 10^5 sweeps, observables after every sweep."""
    L, N, nsweeps, seed = 4, 16, 100_000, 42
    E, M = enumerate_ising(L)
    e_x, am_x, m2_x, _ = boltzmann_averages(E, M, beta, N)
    lat = binding.Lattice(L, 2, beta, seed)
    lat.init_spins(1)
    ser = np.empty((nsweeps, 3), dtype=np.int64)
    for t in range(nsweeps):
        lat.sweep(1)
        o = lat.observables(clusters=True)
        ser[t] = (o["energy"], o["magnetisation"], o["sum_sq_cluster"])
    assert lat.get_counter() == nsweeps
    # the same chain from the oracle: bit-exact series (first 2000 sweeps) -- the chain is the oracle's chain
    s = oracle.init_spins(L, 2, seed, 1)
    want = oracle.run_chain(L, 2, lat.get_threshold(), seed, 0, 2000, s)
    assert np.array_equal(ser[:2000, 0], want[:, 0]) and np.array_equal(ser[:2000, 1], want[:, 1])
    assert np.array_equal(ser[:2000, 2], want[:, 3])
    ser = ser[1000:]
    e, m, fk = ser[:, 0] / N, ser[:, 1] / N, ser[:, 2] / N ** 2
    assert abs(e.mean() - e_x) < 4.5 * blocked_error(e)
    assert abs(np.abs(m).mean() - am_x) < 4.5 * blocked_error(np.abs(m))
    assert abs((m ** 2).mean() - m2_x) < 4.5 * blocked_error(m ** 2)
    assert abs(fk.mean() - m2_x) < 4.5 * blocked_error(fk)            # Fortuin-Kasteleyn: labels <-> spins
    assert not np.any(np.abs(ser[:, 0]) == 28)                        # g(E = +-28) = 0 on the 4x4 torus
    lat.close()


def test_config2_L1024_cold_1000_sweeps_energy_vs_kaufman():
    """Config 2: L=1024, beta_c, cold start, 1000 sweeps; <e> of sweeps 100..999 against Kaufman's exact finite-L
    value -1.4148214 (not Onsager's -sqrt 2, which differs by 6e-4) within 4.5 blocked standard errors."""
    L, nsweeps = 1024, 1000
    N = L * L
    lat = binding.Lattice(L, 2, BETA_C, 1)
    lat.init_spins(0)
    e = np.empty(nsweeps)
    for t in range(nsweeps):
        lat.sweep(1)
        o = lat.observables()
        e[t] = o["energy"] / N
        assert o["counter"] == t + 1
    exact = kaufman_energy_per_site(L, BETA_C)
    assert abs(exact - (-1.4148214132)) < 2e-7
    tail = e[100:]
    err = blocked_error(tail, 15)
    assert err < 1.5e-3
    assert abs(tail.mean() - exact) < 4.5 * err, (tail.mean(), exact, err)
    lat.close()
