"""GPU parity at BASELINE.json's FULL sizes (configs 2-5), in the launch configuration bench.py times.

The lattice pool, ladder, field, seed and PT / measurement cadence are the config's; only the sweep
count is bounded so that the CPU oracle can follow a handful of samples in seconds.  Draws are keyed
by (word / sample, replica, slot, sweep, site) and lanes do not interact (R5), so the oracle
simulates the sampled disorder samples in isolation: first / last word, lanes 0, 13, 31, and one in
the middle.  Compared: spins and (U, M) bit for bit; moment accumulators to 1e-12 * max(|v|, 1).
Properties that hold for every sample at any size are checked on the whole pool (energy bounds,
M parity, accumulator identities).
"""
import numpy as np
import pytest

from paper_1403_4560_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sg():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1403_4560_b200 import sg as _sg
    return _sg


@pytest.fixture(scope="module")
def O():
    from oracle import ea_oracle
    return ea_oracle


def close(a, b, tol=1e-12):
    a = np.asarray(a)
    b = np.asarray(b)
    return np.all(np.abs(a - b) <= tol * np.maximum(np.abs(b), 1.0))


# name, sweeps in the first segment (no measurement), sweeps in the second (config cadence), samples
FULL = [
    ("C2", 24, 40, lambda n: [0, 13, 31, n // 2 + 7, n - 32, n - 1]),
    ("C3", 8, 32, lambda n: [0, 13, n // 2 + 31, n - 1]),
    ("C4", 8, 16, lambda n: [0, 255, n - 1]),
    ("C5", 6, 6, lambda n: [0, 13 + 32 * 100, n - 1]),
]


@pytest.mark.parametrize("case", FULL, ids=[c[0] for c in FULL])
def test_full_size_config(sg, O, case):
    name, n1, n2, pick = case
    w = W.BY_NAME[name]
    temps = w.temps()
    samples = pick(w.n_samples)
    sim = sg.Simulation(w.L, w.h, w.n_samples, w.n_replicas, temps, w.kind, w.seed)
    meas_every = w.meas_every if w.meas_every else 0
    sim.sg_run(n1, w.pt_every, 0)
    sim.sg_run(n2, w.pt_every, meas_every)
    if not meas_every:
        sim.sg_measure(False)          # C5: one measurement at the end (R16)
    U, M = sim.sg_get_energies()
    mom, n_meas = sim.sg_get_moments()
    for s in samples:
        o = O.Oracle(w.L, w.h, w.n_replicas, temps, kind=w.kind, seed=w.seed, sample=s)
        o.run(n1, w.pt_every, 0)
        o.run(n2, w.pt_every, meas_every)
        if not meas_every:
            o.measure()
        got = sim.sg_get_spins(s, 1)[0]
        assert np.array_equal(got, o.spins()), "%s sample %d: spins differ at %d sites" % (name, s, int((got != o.spins()).sum()))
        Uo, Mo = o.energies()
        assert np.array_equal(U[s], Uo) and np.array_equal(M[s], Mo), "%s sample %d: energies differ" % (name, s)
        want, no = o.moments()
        assert no == n_meas
        assert close(mom[s], want), "%s sample %d: moments differ by %g" % (name, s, np.abs(mom[s] - want).max())
        o.close()
    # whole-pool properties
    N = w.N
    assert np.all((M.astype(np.int64) - N) % 2 == 0) and np.all(np.abs(M) <= N)
    if w.kind == W.PMJ:
        assert np.all(U >= 0) and np.all(U <= 3 * N)
    nm = float(n_meas * (w.n_replicas * (w.n_replicas - 1) // 2))
    assert np.all(np.abs(mom[..., 0]) <= nm * (1 + 1e-12))                # |sum q| <= number of terms
    assert np.all(mom[..., 1] >= 0) and np.all(mom[..., 1] <= nm * (1 + 1e-12))
    assert np.all(mom[..., 1] ** 2 <= nm * mom[..., 3] * (1 + 1e-9) + 1e-9)   # Cauchy-Schwarz: (sum q^2)^2 <= n sum q^4
    for k in range(12):
        assert np.all(mom[..., 4 + 5 * k + 2] >= 0) and np.all(mom[..., 4 + 5 * k + 2] <= nm * (1 + 1e-12))
    sw, ex = sim.sg_get_counters()
    assert sw == n1 + n2 and ex == (n1 + n2) // w.pt_every
    sim.close()
