"""GPU parity of the paper's own packing (R17), coupling_kind = SG_PMJ_TPACK:
the temperature copies of one (sample, replica) as the bits of a word, lattice in shared memory, parallel tempering as a
bit permutation.  Every slot keeps its own Philox draws (R17), so the trajectory must equal the oracle's — and the
sample-packed SG_PMJ library path's — bit for bit: spins, the kernel's own (U, M), accepted-swap counts; moments 1e-12."""
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
    # name, L, h, n_samples, R, NT, (T_lo, T_hi), pt_every, (n1, n2, meas_every)
    ("L4-one-word", 4, 0.3, 3, 4, 8, (0.5, 2.0), 1, (7, 12, 4)),
    ("L6-two-words-boundary-swap", 6, 0.1, 5, 2, 40, (0.7, 2.5), 1, (9, 10, 5)),
    ("L8-paper-shape-56", 8, 0.1, 2, 2, 56, (1.0 / 1.8, 10.0), 1, (6, 6, 3)),
    ("L10-paper-shape-56", 10, 0.1, 2, 2, 56, (1.0 / 1.8, 10.0), 1, (4, 4, 2)),
    ("L12-neg-h", 12, -0.2, 1, 4, 33, (0.9, 1.6), 2, (4, 6, 3)),
    ("L16-h0", 16, 0.0, 2, 2, 12, (1.0, 1.3), 1, (3, 4, 2)),
    ("L4-big-h", 4, 1.7, 33, 2, 9, (1.0, 4.0), 3, (10, 11, 0)),
]


@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_tpack_equals_oracle_and_sample_packed_path(sg, O, case):
    _, L, h, ns, R, NT, (Tlo, Thi), pt_every, (n1, n2, me) = case
    temps = W.ladder(Tlo, Thi, NT)
    tp = sg.Simulation(L, h, ns, R, temps, sg.PMJ_TPACK, 56)
    std = sg.Simulation(L, h, ns, R, temps, sg.PMJ, 56)
    assert np.array_equal(tp.sg_get_spins(), std.sg_get_spins())            # initial state (layout conversion round trip)
    assert np.array_equal(tp.sg_get_couplings(), std.sg_get_couplings())
    for sim in (tp, std):
        sim.sg_run(n1, pt_every, 0)
        sim.sg_run(n2, pt_every, me)
    assert np.array_equal(tp.sg_get_spins(), std.sg_get_spins())
    assert tp.sg_get_counters() == std.sg_get_counters()
    pt_tp, pt_std = tp.sg_get_pt_stats(), std.sg_get_pt_stats()
    assert np.array_equal(pt_tp[0], pt_std[0]) and np.array_equal(pt_tp[1], pt_std[1])
    assert pt_tp[1].sum() > 0
    if NT > 32:
        assert pt_tp[1][31] > 0, "the swap across the word boundary (slots 31, 32) never happened: widen the test"
    mom, n = tp.sg_get_moments()
    mom2, nn = std.sg_get_moments()
    assert n == nn and close(mom, mom2)
    fresh = (n1 + n2) % pt_every == 0
    if fresh:
        Uc, Mc = tp.sg_get_energies_cached()
    U, M = tp.sg_get_energies()
    prop_o = acc_o = 0
    for s in range(ns):
        o = O.Oracle(L, h, R, temps, seed=56, sample=s)
        o.run(n1, pt_every, 0)
        o.run(n2, pt_every, me)
        assert np.array_equal(tp.sg_get_spins(s, 1)[0], o.spins()), "sample %d" % s
        Uo, Mo = o.energies()
        assert np.array_equal(U[s], Uo) and np.array_equal(M[s], Mo)
        if fresh:
            assert np.array_equal(Uc[s], Uo) and np.array_equal(Mc[s], Mo), "sample %d: the kernel's own energies" % s
        want, no = o.moments()
        assert no == n and close(mom[s], want)
        p, a = o.pt_stats()
        prop_o += p
        acc_o += a
        o.close()
    assert int(pt_tp[0].sum()) == prop_o and int(pt_tp[1].sum()) == acc_o
    # primitives from the same state, and the generic path on the sample-packed copy
    for sim in (tp, std):
        sim.sg_sweep(2)
        sim.sg_pt_exchange()
    tp.sg_set_kernel_path(sg.PATH_GENERIC)
    for sim in (tp, std):
        sim.sg_run(3, 1, 0)
    tp.sg_set_kernel_path(sg.PATH_AUTO)
    for sim in (tp, std):
        sim.sg_run(2, 1, 0)
    assert np.array_equal(tp.sg_get_spins(), std.sg_get_spins())
    assert np.array_equal(tp.sg_get_state_hash(), std.sg_get_state_hash()[:, :, :]) or ns % 32 != 0   # idle lanes differ when the last word is ragged
    # set_spins goes through the sample-packed copy and back
    S = tp.sg_get_spins()
    S[0] = -S[0]
    tp.sg_set_spins(S)
    std.sg_set_spins(S)
    for sim in (tp, std):
        sim.sg_run(2, 1, 0)
    assert np.array_equal(tp.sg_get_spins(), std.sg_get_spins())
    # reset
    tp.sg_reset()
    std.sg_reset()
    assert np.array_equal(tp.sg_get_spins(), std.sg_get_spins())
    tp.close(); std.close()


def test_tpack_unsupported_shapes(sg):
    with pytest.raises(sg.SgError) as e:
        sg.Simulation(32, 0.1, 2, 2, W.ladder(0.5, 2.0, 8), sg.PMJ_TPACK, 1)
    assert e.value.code == sg.EUNSUPPORTED
    with pytest.raises(sg.SgError) as e:
        sg.Simulation(14, 0.1, 2, 2, W.ladder(0.5, 2.0, 8), sg.PMJ_TPACK, 1)
    assert e.value.code == sg.EUNSUPPORTED
    sim = sg.Simulation(8, 0.1, 2, 2, W.ladder(0.5, 2.0, 8), sg.PMJ_TPACK, 1)
    with pytest.raises(sg.SgError):
        sim.sg_set_first_sample(5)          # must be a multiple of 32: the sweep draws are keyed by the packed word
    sim.sg_set_first_sample(64)
    sim.close()


BIG = [
    # name, L, h, n_samples, R, NT, (T_lo, T_hi): n_samples * R >= 6 lattices per SM (888 on a B200) selects k_tp_run<L, 32>
    ("L4-1024-lattices", 4, 0.3, 512, 2, 8, (0.5, 2.0)),
    ("L6-960-lattices-40-slots", 6, 0.1, 480, 2, 40, (0.7, 2.5)),
]


@pytest.mark.parametrize("case", BIG, ids=[c[0] for c in BIG])
def test_tpack_many_lattices_kernel(sg, O, case):
    """with at least 6 lattices per SM the launch takes the instantiation that keeps 32 slots per work
    item (k_tp_run<L, 32>); the cases above never reach it.  Whole pool against the sample-packed SG_PMJ path, three
    samples (first word, a middle lane, last) against the oracle."""
    import torch
    _, L, h, ns, R, NT, (Tlo, Thi) = case
    assert ns * R >= 6 * torch.cuda.get_device_properties(0).multi_processor_count
    temps = W.ladder(Tlo, Thi, NT)
    tp = sg.Simulation(L, h, ns, R, temps, sg.PMJ_TPACK, 77)
    std = sg.Simulation(L, h, ns, R, temps, sg.PMJ, 77)
    try:
        for sim in (tp, std):
            sim.sg_run(6, 1, 0)
            sim.sg_run(6, 2, 3)
        assert np.array_equal(tp.sg_get_spins(), std.sg_get_spins())
        assert np.array_equal(tp.sg_get_state_hash(), std.sg_get_state_hash())
        pt_tp, pt_std = tp.sg_get_pt_stats(), std.sg_get_pt_stats()
        assert np.array_equal(pt_tp[0], pt_std[0]) and np.array_equal(pt_tp[1], pt_std[1]) and pt_tp[1].sum() > 0
        Uc, Mc = tp.sg_get_energies_cached()
        U, M = std.sg_get_energies()
        assert np.array_equal(Uc, U) and np.array_equal(Mc, M)
        mom, n = tp.sg_get_moments()
        mom2, nn = std.sg_get_moments()
        assert n == nn == 2 and close(mom, mom2)
        for s in (0, ns // 2 + 13, ns - 1):
            o = O.Oracle(L, h, R, temps, seed=77, sample=s)
            o.run(6, 1, 0)
            o.run(6, 2, 3)
            assert np.array_equal(tp.sg_get_spins(s, 1)[0], o.spins()), "sample %d" % s
            Uo, Mo = o.energies()
            assert np.array_equal(Uc[s], Uo) and np.array_equal(Mc[s], Mo)
            want, no = o.moments()
            assert no == n and close(mom[s], want)
            o.close()
    finally:
        tp.close(); std.close()


def test_repeated_short_sweep_calls_stay_in_the_packed_layout(sg):
    """sg_sweep no longer converts the temperature-packed state back to the sample-packed layout before
    every call (a full-state transpose nobody read): one launch per call, same trajectory."""
    temps = W.ladder(0.7, 2.5, 40)
    tp = sg.Simulation(6, 0.1, 5, 2, temps, sg.PMJ_TPACK, 3)
    std = sg.Simulation(6, 0.1, 5, 2, temps, sg.PMJ, 3)
    try:
        tp.sg_sweep(1)
        n0 = tp.sg_get_launch_count()
        for _ in range(5):
            tp.sg_sweep(1)
        assert tp.sg_get_launch_count() - n0 == 5
        tp.sg_pt_exchange()                      # runs on the sample-packed copy: converts once
        tp.sg_sweep(2)
        std.sg_sweep(6)
        std.sg_pt_exchange()
        std.sg_sweep(2)
        assert np.array_equal(tp.sg_get_spins(), std.sg_get_spins())
        assert tp.sg_get_counters() == std.sg_get_counters() == (8, 1)
    finally:
        tp.close(); std.close()
