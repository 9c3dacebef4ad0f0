"""GPU parity of the diagnostics: device-side P(q) histograms and the per-window
accumulators of the logarithmic-binning test against the oracle's plain counting — integer histograms
bit-exact, window moments to 1e-12 — on every measurement path (fused bit-sliced kernel, histogram + finalize kernels of
the generic / L = 32 / Gaussian paths)."""
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


CASES = [
    # name, L, h, n_samples, R, NT, kind, generic path, pq bins (None = N + 1)
    ("fused-L8", 8, 0.2, 40, 4, 5, 0, False, None),
    ("fused-L6-coarse", 6, 0.1, 33, 2, 4, 0, False, 17),
    ("fused-L12", 12, 0.1, 32, 4, 3, 0, False, None),
    ("generic-pmj-L8", 8, 0.2, 33, 4, 3, 0, True, None),
    ("l32", 32, 0.2, 32, 2, 2, 0, False, 64),
    ("gauss-L8", 8, 0.3, 3, 4, 4, 1, False, None),
    ("gauss-L6-generic", 6, 0.3, 3, 2, 3, 1, False, 10),
]


@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_pq_histogram_and_log_binning_windows(sg, O, case):
    _, L, h, ns, R, NT, kind, generic, bins = case
    temps = W.ladder(0.8, 1.8, NT)
    sim = sg.Simulation(L, h, ns, R, temps, kind, 31)
    if generic:
        sim.sg_set_kernel_path(sg.PATH_GENERIC)
    n_windows = 4
    sim.sg_enable_pq(bins)
    sim.sg_enable_log_binning(n_windows)
    plan = [(3, 1, 1), (20, 1, 2)] if L < 32 else [(3, 1, 1), (6, 1, 2)]       # measurements at sweeps 1, 2, 3, 4, 6, 8, ...
    for seg in plan:
        sim.sg_run(*seg)
    pq = sim.sg_get_pq()
    mom, n = sim.sg_get_moments()
    wins = [sim.sg_get_window_moments(k) for k in range(n_windows)]
    samples = sorted({0, ns - 1, ns // 2})
    for s in samples:
        o = O.Oracle(L, h, R, temps, kind=kind, seed=31, sample=s)
        o.enable_pq(bins)
        o.enable_log_binning(n_windows)
        for seg in plan:
            o.run(*seg)
        assert np.array_equal(pq[s].astype(np.uint64), o.pq()), "sample %d: P(q) histogram" % s
        want, no = o.moments()
        assert no == n and close(mom[s], want)
        tot = np.zeros_like(want)
        for k in range(n_windows):
            wk, nk = o.window_moments(k)
            assert wins[k][1] == nk, "window %d: %d measurements, oracle %d" % (k, wins[k][1], nk)
            assert close(wins[k][0][s], wk), "sample %d window %d" % (s, k)
            tot += wins[k][0][s]
        assert close(tot, want, 1e-11)
        o.close()
    n_pairs = R * (R - 1) // 2
    assert np.all(pq.sum(axis=2) == n * n_pairs)
    # reset clears the diagnostics
    sim.sg_reset()
    assert not sim.sg_get_pq().any() and sim.sg_get_window_moments(0)[1] == 0 and not sim.sg_get_window_moments(1)[0].any()
    sim.close()


def test_diagnostics_error_paths_and_estimators(sg):
    from paper_1403_4560_b200 import estimators as E
    sim = sg.Simulation(8, 0.0, 256, 4, (20.0, 40.0), sg.PMJ, 77)
    with pytest.raises(sg.SgError) as e:
        sim.sg_get_pq()
    assert e.value.code == sg.ESTATE
    with pytest.raises(sg.SgError):
        sim.sg_enable_pq(8 ** 3 + 2)
    with pytest.raises(sg.SgError):
        sim.sg_enable_log_binning(0)
    assert (sim.pq_bins, sim.n_windows) == (1, 0)          # a refused enable leaves the binding's sizes alone
    sim.sg_enable_pq(33)
    sim.sg_enable_log_binning(7)
    with pytest.raises(sg.SgError):
        sim.sg_enable_pq(0)
    with pytest.raises(sg.SgError):
        sim.sg_enable_log_binning(41)
    assert (sim.pq_bins, sim.n_windows) == (33, 7) and sim.sg_get_pq().shape == (256, 2, 33)
    sim.sg_run(96, 1, 2)
    with pytest.raises(sg.SgError):
        sim.sg_get_window_moments(7)
    wins = [sim.sg_get_window_moments(k) for k in range(7)]
    assert [w[1] for w in wins] == [0, 1, 2, 4, 8, 16, 17]
    series = E.log_binning([w[0] for w in wins], [w[1] for w in wins], 8, n_pairs=6, block=32)
    assert series[0] is None and series[1] is not None
    # at T = 20, 40 the chain is equilibrated after a few sweeps: the last windows agree (the test "passes")
    assert np.all(E.log_binning_passes(series, "chi_k1", last=3, n_sigma=4.0))
    assert np.all(E.log_binning_passes(series, "q2", last=3, n_sigma=4.0))
    centres, P, Ps = E.overlap_distribution(sim.sg_get_pq(), 8)
    assert centres.shape == (33,) and np.allclose(P.sum(axis=1), 1.0) and Ps.shape == (256, 2, 33)
    # nearly independent spins: P(q) is centred at 0 with variance 1/N
    var = (P * centres[None, :] ** 2).sum(axis=1)
    assert np.all(np.abs(var - 1.0 / 512) < 2e-3)
    sim.close()
