"""GPU parity: libsg_b200 (through its C-ABI binding) vs the CPU oracle, element by element.

Bar (BASELINE.json north_star): spins, couplings, thresholds, energies bit-exact on every config
(+-J and Gaussian); overlaps / moments within 1e-12 * max(|value|, 1).
Sizes here are ones the oracle finishes in seconds; the full-size cases are in
test_gpu_fullsize.py.
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


def make_pair(sg, O, L, h, n_samples, R, temps, kind, seed, samples):
    sim = sg.Simulation(L, h, n_samples, R, temps, kind, seed)
    orc = {s: O.Oracle(L, h, R, temps, kind=kind, seed=seed, sample=s) for s in samples}
    return sim, orc


def check_state(sim, orc, what=""):
    U, M = sim.sg_get_energies()
    for s, o in orc.items():
        got = sim.sg_get_spins(s, 1)[0]
        want = o.spins()
        assert np.array_equal(got, want), "%s spins differ, sample %d: %d sites" % (what, s, int((got != want).sum()))
        Uo, Mo = o.energies()
        assert np.array_equal(U[s], Uo), "%s U differs, sample %d" % (what, s)
        assert np.array_equal(M[s], Mo), "%s M differs, sample %d" % (what, s)


CASES = [
    # name, L, h, n_samples, R, NT, T range, kind, seed, samples to check
    ("C1", 4, 0.3, 1, 4, 8, (0.5, 2.0), 0, 1, [0]),
    ("L4-two-words", 4, 0.3, 40, 4, 5, (0.5, 2.0), 0, 11, [0, 5, 31, 32, 39]),
    ("L6-ragged-quads", 6, 0.2, 33, 2, 4, (0.5, 2.0), 0, 12, [0, 17, 32]),
    ("L8", 8, 0.2, 64, 4, 6, (0.5, 2.0), 0, 2, [0, 13, 31, 63]),
    ("L12", 12, 0.1, 32, 4, 3, (0.4, 1.8), 0, 3, [0, 31]),
    ("L8-neg-h", 8, -0.7, 32, 2, 4, (0.6, 1.5), 0, 4, [3, 30]),
    ("L10", 10, 0.1, 34, 4, 3, (0.5, 1.8), 0, 13, [0, 33]),
    ("L16-pmj", 16, 0.2, 32, 2, 3, (0.5, 1.8), 0, 14, [5, 31]),
    ("L4-h0", 4, 0.0, 32, 2, 4, (0.5, 2.0), 0, 5, [1, 2]),
    ("L4-big-h-general-path", 4, 1.7, 32, 2, 4, (0.5, 3.0), 0, 6, [7, 8]),
    ("L4-huge-h", 4, 5.0, 32, 2, 3, (0.5, 3.0), 0, 7, [0, 9]),
    ("G-L4", 4, 0.3, 5, 4, 6, (0.2, 1.5), 1, 4, [0, 2, 4]),
    ("G-L6", 6, -0.3, 3, 2, 4, (0.3, 1.5), 1, 8, [0, 2]),
    ("G-L8", 8, 0.3, 4, 4, 4, (0.2, 1.5), 1, 9, [1, 3]),
]


@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_initial_state_tables_and_couplings(sg, O, case):
    _, L, h, ns, R, NT, (Tlo, Thi), kind, seed, samples = case
    temps = W.ladder(Tlo, Thi, NT)
    sim, orc = make_pair(sg, O, L, h, ns, R, temps, kind, seed, samples)
    assert np.array_equal(sim.sg_get_thresholds(), next(iter(orc.values())).thresholds())
    for s, o in orc.items():
        Jg = sim.sg_get_couplings(s, 1)[0]
        Jo = o.couplings()
        assert np.array_equal(Jg.view(np.uint32), Jo.view(np.uint32)), "couplings differ (bitwise), sample %d" % s
    check_state(sim, orc, "initial")
    assert sim.sg_get_counters() == (0, 0)
    sim.close()


@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_sweeps_pt_measure_bit_exact(sg, O, case):
    _, L, h, ns, R, NT, (Tlo, Thi), kind, seed, samples = case
    temps = W.ladder(Tlo, Thi, NT)
    sim, orc = make_pair(sg, O, L, h, ns, R, temps, kind, seed, samples)
    n_meas = 0
    for step in range(12):
        sim.sg_sweep(1)
        for o in orc.values():
            o.sweep(1)
        if step in (0, 5, 11):
            check_state(sim, orc, "after sweep %d" % step)
        sim.sg_pt_exchange()
        for o in orc.values():
            o.pt_exchange()
        if step in (0, 1, 6, 11):
            check_state(sim, orc, "after exchange %d" % step)
        if step % 4 == 3:
            rec = sim.sg_measure()
            n_meas += 1
            for s, o in orc.items():
                want = o.measure()
                assert close(rec[s], want), "records differ, sample %d: %g" % (s, np.abs(rec[s] - want).max())
    mom, n = sim.sg_get_moments()
    assert n == n_meas
    for s, o in orc.items():
        want, no = o.moments()
        assert no == n_meas
        assert close(mom[s], want), "moments differ, sample %d: %g" % (s, np.abs(mom[s] - want).max())
    assert sim.sg_get_counters() == (12, 12)
    sim.close()


@pytest.mark.parametrize("case", [CASES[0], CASES[3], CASES[9]], ids=["C1", "L8", "G-L4"])
def test_run_equals_primitive_sequence_and_oracle(sg, O, case):
    _, L, h, ns, R, NT, (Tlo, Thi), kind, seed, samples = case
    temps = W.ladder(Tlo, Thi, NT)
    sim, orc = make_pair(sg, O, L, h, ns, R, temps, kind, seed, samples)
    sim2 = sg.Simulation(L, h, ns, R, temps, kind, seed)
    sim.sg_run(40, 2, 10)
    for k in range(1, 41):
        sim2.sg_sweep(1)
        if k % 2 == 0:
            sim2.sg_pt_exchange()
        if k % 10 == 0:
            sim2.sg_measure(False)
    assert np.array_equal(sim.sg_get_spins(), sim2.sg_get_spins())
    m1, n1 = sim.sg_get_moments()
    m2, n2 = sim2.sg_get_moments()
    assert n1 == n2 == 4 and np.array_equal(m1, m2)
    for o in orc.values():
        o.run(40, 2, 10)
    check_state(sim, orc, "after run")
    for s, o in orc.items():
        assert close(m1[s], o.moments()[0])
    # reset returns to the initial state
    sim.sg_reset()
    fresh = {s: O.Oracle(L, h, R, temps, kind=kind, seed=seed, sample=s) for s in samples}
    check_state(sim, fresh, "after reset")
    assert sim.sg_get_moments()[1] == 0 and not sim.sg_get_moments()[0].any()
    sim.close(); sim2.close()


def test_c1_full_config(sg, O):
    """BASELINE.json config 1 exactly: 1000 sweeps, PT every sweep, measure every 10."""
    w = W.BY_NAME["C1"]
    sim, orc = make_pair(sg, O, w.L, w.h, w.n_samples, w.n_replicas, w.temps(), w.kind, w.seed, [0])
    sim.sg_run(w.n_sweeps, w.pt_every, w.meas_every)
    orc[0].run(w.n_sweeps, w.pt_every, w.meas_every)
    check_state(sim, orc, "C1 end")
    mom, n = sim.sg_get_moments()
    want, no = orc[0].moments()
    assert n == no == 100
    assert close(mom[0], want)
    sim.close()


def test_set_spins_roundtrip_and_closed_forms(sg):
    """set/get round trip; identical replicas -> q(0)=1, q(k)=0; stripe closed form."""
    import math
    L, R, NT, ns = 8, 2, 2, 35
    N = L**3
    sim = sg.Simulation(L, 0.0, ns, R, [1.0, 2.0], 0, 3)
    rng = np.random.default_rng(0)
    S = rng.choice([-1, 1], size=(ns, R, NT, N)).astype(np.int8)
    sim.sg_set_spins(S)
    assert np.array_equal(sim.sg_get_spins(), S)
    sub = rng.choice([-1, 1], size=(3, R, NT, N)).astype(np.int8)
    sim.sg_set_spins(sub, s0=30)
    S[30:33] = sub
    assert np.array_equal(sim.sg_get_spins(), S)
    x = np.arange(N) % L
    S[:, 1] = S[:, 0]
    S[5, 0] = 1
    S[5, 1] = np.where(x < L // 2, 1, -1)
    S[6, 1] = -S[6, 0]
    sim.sg_set_spins(S)
    rec = sim.sg_measure()
    assert np.all(rec[0, :, 0, 0] == 1.0) and np.all(np.abs(rec[0, :, 0, 1:]) < 1e-15)
    assert np.all(rec[6, :, 0, 0] == -1.0)
    assert abs(rec[5, 0, 0, 1] - 2.0 / L) < 1e-14 and abs(rec[5, 0, 0, 2] - 2.0 / L / math.tan(math.pi / L)) < 1e-14
    assert np.all(np.abs(rec[5, 0, 0, 3:]) < 1e-14) and abs(rec[5, 0, 0, 0]) < 1e-15
    sim.close()


def test_error_paths(sg):
    with pytest.raises(sg.SgError) as e:
        sg.Simulation(5, 0.1, 4, 4, [1.0])
    assert e.value.code == sg.EINVAL
    with pytest.raises(sg.SgError):
        sg.Simulation(4, 0.1, 4, 3, [1.0])
    with pytest.raises(sg.SgError):
        sg.Simulation(4, 0.1, 4, 4, [2.0, 1.0])
    with pytest.raises(sg.SgError):
        sg.Simulation(4, 0.1, 4, 4, [0.0, 1.0])
    import torch
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    with pytest.raises(sg.SgError) as e:
        sg.Simulation(4, 0.1, 4, 4, [1.0], workspace=small)
    assert e.value.code == sg.ENOMEM
    sim = sg.Simulation(4, 0.1, 4, 4, [1.0])
    with pytest.raises(sg.SgError):
        sim.sg_run(-1, 0, 0)
    with pytest.raises(sg.SgError):
        sim.sg_get_spins(3, 5)
    sim.close()


@pytest.mark.parametrize("h,NT,R,pt_every,n_samples", [(0.2, 20, 4, 1, 64), (-0.4, 7, 2, 3, 33), (0.0, 5, 4, 2, 32),
                                                     (1.0, 10, 2, 1, 96)])
def test_l8_fused_ladder_with_pt(sg, O, h, NT, R, pt_every, n_samples):
    """The L=8 shared-memory ladder kernel with in-kernel parallel tempering (sg_run) vs the oracle:
    spins, energies bit-exact after 50 sweeps incl. a measurement boundary; moments to 1e-12."""
    temps = W.ladder(0.5, 2.0, NT)
    samples = sorted({0, 13, n_samples - 1, n_samples // 2})
    sim, orc = make_pair(sg, O, 8, h, n_samples, R, temps, 0, 21, samples)
    sim.sg_run(50, pt_every, 16)
    for o in orc.values():
        o.run(50, pt_every, 16)
    check_state(sim, orc, "fused L8")
    assert sim.sg_get_counters() == (50, 50 // pt_every)
    mom, n = sim.sg_get_moments()
    assert n == 3
    for s, o in orc.items():
        assert close(mom[s], o.moments()[0])
    # continue with primitives from the fused state: counters and RNG streams line up
    sim.sg_sweep(1); sim.sg_pt_exchange(); sim.sg_run(5, pt_every, 0)
    for o in orc.values():
        o.sweep(1); o.pt_exchange(); o.run(5, pt_every, 0)
    check_state(sim, orc, "fused L8 + primitives")
    sim.close()


@pytest.mark.parametrize("h,NT,R,pt_every,n_samples", [(0.2, 4, 4, 4, 33), (-0.3, 3, 2, 1, 32), (0.0, 2, 2, 3, 64)])
def test_l32_resident_kernel_with_pt(sg, O, h, NT, R, pt_every, n_samples):
    """The L=32 kernel (one system resident in shared memory, couplings streamed, energies for the
    exchange step produced in the last colour-1 half sweep) vs the oracle: sg_run with exchanges falling
    inside and at the end, then primitives (sg_sweep + separate energy kernel) from the same state."""
    temps = W.ladder(0.4, 2.0, NT)
    samples = sorted({0, 13, n_samples - 1})
    sim, orc = make_pair(sg, O, 32, h, n_samples, R, temps, 0, 5, samples)
    sim.sg_run(10, pt_every, 0)
    for o in orc.values():
        o.run(10, pt_every, 0)
    check_state(sim, orc, "resident L32")
    assert sim.sg_get_counters() == (10, 10 // pt_every)
    sim.sg_sweep(3); sim.sg_pt_exchange(); sim.sg_run(2, pt_every, 0)
    for o in orc.values():
        o.sweep(3); o.pt_exchange(); o.run(2, pt_every, 0)
    check_state(sim, orc, "resident L32 + primitives")
    rec = sim.sg_measure()
    for s, o in orc.items():
        assert close(rec[s], o.measure())
    sim.close()


def test_estimators_on_device_moments_high_temperature(sg):
    """End of the path: device accumulators -> Eqs. 3-6 (estimators.py).  At T = 20, 40 and h = 0 spins are nearly
    independent: chi(k) = 1 + O(beta^2), R12 = 1, g = O(1/N), all within jackknife errors (blocks of whole words)."""
    from paper_1403_4560_b200 import estimators as E
    sim = sg.Simulation(8, 0.0, 256, 4, (20.0, 40.0), sg.PMJ, 77)
    sim.sg_run(96, 1, 4)
    mom, n = sim.sg_get_moments()
    assert n == 24
    out = E.indicators(mom, n, 8, n_pairs=6, block=32)
    for name in ("chi0", "chi_k1", "chi_k2_paper", "chi_k2_baseline", "chi_k1_4rep", "R12", "R12_baseline"):
        assert np.all(np.abs(out[name] - 1.0) < 0.03 + 5 * out[name + "_err"]), (name, out[name], out[name + "_err"])
    assert np.all(np.abs(out["g_std"]) < 0.01 + 5 * out["g_std_err"])
    sim.close()


@pytest.mark.parametrize("L,h,NT,R,pt_every,n_samples", [(4, 0.3, 8, 4, 1, 1), (6, 0.1, 7, 2, 1, 40), (10, -0.2, 4, 4, 3, 33),
                                                       (12, 0.1, 5, 4, 1, 32), (16, 0.2, 3, 2, 2, 32)])
def test_generic_ladder_with_fused_pt(sg, O, L, h, NT, R, pt_every, n_samples):
    """k_ladder_pmj<L> with the exchange step fused in (one warp per system recounts U, M from shared memory,
    one thread per (pair, lane) decides, masked swap) vs the oracle, across a measurement boundary, then
    primitives from the same state."""
    temps = W.ladder(0.5, 1.9, NT)
    samples = sorted({0, n_samples - 1, n_samples // 2})
    sim, orc = make_pair(sg, O, L, h, n_samples, R, temps, 0, 31, samples)
    sim.sg_run(21, pt_every, 8)
    for o in orc.values():
        o.run(21, pt_every, 8)
    check_state(sim, orc, "fused generic ladder")
    assert sim.sg_get_counters() == (21, 21 // pt_every)
    mom, n = sim.sg_get_moments()
    assert n == 2
    for s, o in orc.items():
        assert close(mom[s], o.moments()[0])
    sim.sg_sweep(2); sim.sg_pt_exchange(); sim.sg_run(4, pt_every, 0)
    for o in orc.values():
        o.sweep(2); o.pt_exchange(); o.run(4, pt_every, 0)
    check_state(sim, orc, "fused generic ladder + primitives")
    sim.close()


@pytest.mark.parametrize("L,h,NT,R,pt_every,n_samples", [(8, 0.3, 8, 4, 1, 3), (8, -0.2, 5, 2, 2, 2), (16, 0.3, 6, 2, 1, 2)])
def test_gaussian_ladder_with_fused_pt(sg, O, L, h, NT, R, pt_every, n_samples):
    """k_gladder<L>: the Gaussian fp32 ladder resident in shared memory with the exchange step fused in
    (fixed-point energies, R14) vs the oracle — spins and E_fix bit-exact, moments to 1e-12 — across a
    measurement boundary, then primitives from the same state."""
    temps = W.ladder(0.2, 1.5, NT)
    samples = list(range(n_samples))
    sim, orc = make_pair(sg, O, L, h, n_samples, R, temps, 1, 41, samples)
    sim.sg_run(13, pt_every, 4)
    for o in orc.values():
        o.run(13, pt_every, 4)
    check_state(sim, orc, "fused Gaussian ladder")
    assert sim.sg_get_counters() == (13, 13 // pt_every)
    mom, n = sim.sg_get_moments()
    assert n == 3
    for s, o in orc.items():
        assert close(mom[s], o.moments()[0])
    sim.sg_sweep(2); sim.sg_pt_exchange(); sim.sg_run(3, pt_every, 0)
    for o in orc.values():
        o.sweep(2); o.pt_exchange(); o.run(3, pt_every, 0)
    check_state(sim, orc, "fused Gaussian ladder + primitives")
    sim.close()


@pytest.mark.parametrize("L,n_samples", [(6, 33), (8, 32), (10, 32)])
def test_paper_shapes_56_temperatures_two_replicas(sg, O, L, n_samples):
    """The paper's own run shape (Table I): N_T = 56 temperatures geometric in beta in [0.1, 1.8],
    h = 0.1, 2 replicas, PT every sweep — bit-exact vs the oracle on a few samples, moments to 1e-12."""
    temps = W.ladder(1.0 / 1.8, 1.0 / 0.1, 56)
    samples = [0, n_samples - 1]
    sim, orc = make_pair(sg, O, L, 0.1, n_samples, 2, temps, 0, 1403, samples)
    sim.sg_run(10, 1, 0)
    sim.sg_run(10, 1, 5)
    for o in orc.values():
        o.run(10, 1, 0)
        o.run(10, 1, 5)
    check_state(sim, orc, "paper shape L=%d" % L)
    mom, n = sim.sg_get_moments()
    assert n == 2
    for s, o in orc.items():
        assert close(mom[s], o.moments()[0])
    sim.close()


def _fuzz_cases():
    rng = np.random.default_rng(4560)
    cases = []
    for i in range(14):
        kind = 1 if i % 5 == 4 else 0
        L = int(rng.choice([4, 6, 8] if kind else [4, 6, 8, 10, 12, 16]))
        NT = int(rng.integers(2, 10))
        R = int(rng.choice([2, 4]))
        h = float(rng.choice([0.0, 0.1, -0.25, 0.7, 1.0, -1.0, 1.3]))
        pt_every = int(rng.choice([0, 1, 1, 2, 3]))
        meas_every = int(rng.choice([0, 3, 4]))
        ns = int(rng.integers(1, 5)) if kind else int(rng.choice([1, 31, 32, 33, 64, 70]))
        n1, n2 = int(rng.integers(1, 8)), int(rng.integers(1, 8))
        cases.append((L, h, ns, R, NT, kind, 100 + i, pt_every, meas_every, n1, n2))
    return cases


@pytest.mark.parametrize("case", _fuzz_cases(), ids=lambda c: "L%d-h%g-ns%d-R%d-NT%d-k%d-pt%d-m%d" % (c[0], c[1], c[2], c[3], c[4], c[5], c[7], c[8]))
def test_fuzzed_shapes_run_vs_oracle(sg, O, case):
    """Seeded random shapes through sg_run (every fused / fallback kernel path, ragged sample counts, odd ladders,
    both signs of h, |h| > 1 general acceptance): two consecutive runs vs the oracle, bit-exact."""
    L, h, ns, R, NT, kind, seed, pt_every, meas_every, n1, n2 = case
    temps = W.ladder(0.45, 2.2, NT)
    samples = sorted({0, ns - 1, ns // 2})
    sim, orc = make_pair(sg, O, L, h, ns, R, temps, kind, seed, samples)
    for n in (n1, n2):
        sim.sg_run(n, pt_every, meas_every)
        for o in orc.values():
            o.run(n, pt_every, meas_every)
        check_state(sim, orc, "fuzz after %d sweeps" % n)
    mom, nm = sim.sg_get_moments()
    for s, o in orc.items():
        want, no = o.moments()
        assert no == nm
        assert close(mom[s], want)
    assert sim.sg_get_counters()[0] == n1 + n2
    sim.close()


# ---- round 2, last session: pair layout / warp-per-pair exchange (L = 4, 12), half ladders in the last wave, overlapped
# measurements


@pytest.mark.parametrize("L,h,NT,R,pt_every,n_samples", [(12, 0.1, 1, 2, 1, 32), (12, -0.2, 2, 2, 1, 33), (12, 0.3, 3, 4, 1, 32),
                                                       (12, 0.1, 6, 2, 2, 64), (12, 0.0, 7, 4, 1, 32), (4, 0.3, 2, 2, 1, 40),
                                                       (4, -0.3, 9, 4, 1, 32), (4, 0.2, 20, 2, 3, 65),
                                                       (6, 0.2, 9, 4, 1, 33), (6, 0.0, 2, 2, 1, 32), (10, 0.1, 7, 2, 2, 32), (10, -0.3, 12, 4, 1, 33),
                                                       (8, 0.2, 30, 4, 1, 33), (8, -0.1, 33, 2, 2, 32)])
def test_pair_layout_ladder_odd_and_tiny_ladders(sg, O, L, h, NT, R, pt_every, n_samples):
    """k_ladder_pmj<4 | 12> (pair layout), <6 | 10> (planar layout), <8> with more slots than the L = 8 kernel takes (whole-quad
    rows) — exchange half sweep by one warp per pair of slots: ladders with one slot, an
    odd number of slots (a slot without a partner at both parities of the exchange), more pairs than warps, 2 and 4
    replicas, h = 0 (carry-chain compare) — spins, the kernel's own (U, M) after an exchange, accepted-swap counts and
    moments vs the oracle."""
    temps = W.ladder(0.6, 1.7, NT)
    samples = sorted({0, n_samples - 1, n_samples // 2})
    sim, orc = make_pair(sg, O, L, h, n_samples, R, temps, 0, 77, samples)
    n = 12 if pt_every == 1 else 12 * pt_every // 2
    sim.sg_run(n, pt_every, 4)
    for o in orc.values():
        o.run(n, pt_every, 4)
    check_state(sim, orc, "pair-layout ladder")
    if n % pt_every == 0 and NT > 1:
        Uc, Mc = sim.sg_get_energies_cached()          # the kernel's own energies, permuted by the last exchange
        for s, o in orc.items():
            Uo, Mo = o.energies()
            assert np.array_equal(Uc[s], Uo) and np.array_equal(Mc[s], Mo)
    mom, nm = sim.sg_get_moments()
    assert nm == n // 4
    for s, o in orc.items():
        assert close(mom[s], o.moments()[0])
    sim.sg_sweep(3)                                    # instantiation without exchange code, from the same state
    for o in orc.values():
        o.sweep(3)
    check_state(sim, orc, "pair-layout ladder + plain sweeps")
    sim.close()


@pytest.mark.parametrize("L,NT,R,n_samples", [(4, 4, 4, 39 * 32), (12, 2, 2, 77 * 32)])
def test_half_ladders_in_the_last_wave(sg, O, L, NT, R, n_samples):
    """Plain sweeps with more ladders than SMs and a last wave that fills at most half of them (156 / 154 ladders on 148
    SMs): its ladders are split over two CTAs.  Samples of the first, a middle and the LAST words (the split ones) vs the
    oracle, and the whole pool vs the generic path by state hash."""
    temps = W.ladder(0.5, 1.8, NT)
    nw = (n_samples + 31) // 32
    samples = sorted({0, 31, 32 * (nw // 2) + 7, 32 * (nw - 2) + 1, 32 * (nw - 1), n_samples - 1})
    sim, orc = make_pair(sg, O, L, 0.2, n_samples, R, temps, 0, 5, samples)
    sim.sg_sweep(5)
    for o in orc.values():
        o.sweep(5)
    check_state(sim, orc, "half ladders")
    h_fast = sim.sg_get_state_hash()
    sim.close()
    gen = sg.Simulation(L, 0.2, n_samples, R, temps, 0, 5)
    gen.sg_set_kernel_path(sg.PATH_GENERIC)
    gen.sg_sweep(5)
    assert np.array_equal(gen.sg_get_state_hash(), h_fast)
    gen.close()


@pytest.mark.parametrize("L,NT,R,n_samples", [(8, 6, 4, 64), (12, 4, 4, 32), (4, 5, 2, 33), (16, 3, 2, 32)])
def test_overlapped_measurements_equal_serial_ones(sg, O, L, NT, R, n_samples):
    """sg_run with a measurement cadence overlaps every measurement with the next ladder launch (second state buffer,
    two library streams).  Run segments that start and end between measurements, interleaved with other calls, must give
    the moments, the state and the records of the same schedule done with sg_run(.., 0) + sg_measure (no overlap), and
    both must equal the oracle."""
    temps = W.ladder(0.5, 1.9, NT)
    samples = sorted({0, n_samples - 1})
    a, orc = make_pair(sg, O, L, 0.25, n_samples, R, temps, 0, 9, samples)
    b = sg.Simulation(L, 0.25, n_samples, R, temps, 0, 9)
    segs = [21, 3, 8, 1, 16, 7]                      # measurement every 8 sweeps: after sweeps 8, 16, 24, 32, 40, 48, 56
    for i, n in enumerate(segs):
        a.sg_run(n, 1, 8)
        if i == 2:
            a.sg_get_spins(0, 1)                     # a reader between two overlapped runs
    done = 0
    for n in segs:
        left = n
        while left:
            step = min(left, 8 - done % 8)
            b.sg_run(step, 1, 0)
            done += step
            left -= step
            if done % 8 == 0:
                b.sg_measure(False)
    for o in orc.values():
        o.run(sum(segs), 1, 8)
    check_state(a, orc, "overlapped measurements")
    assert np.array_equal(a.sg_get_state_hash(), b.sg_get_state_hash())
    ma, na = a.sg_get_moments()
    mb, nb = b.sg_get_moments()
    assert na == nb == sum(segs) // 8
    assert np.array_equal(ma, mb), "overlapped and serial measurements accumulate different moments"
    for s, o in orc.items():
        assert close(ma[s], o.moments()[0])
    ra = a.sg_measure()                              # records from the current buffer after an overlapped run
    rb = b.sg_measure()
    assert np.array_equal(ra, rb)
    a.close()
    b.close()


@pytest.mark.parametrize("L,NT,R,pt_every,n_samples", [(10, 56, 2, 1, 33), (12, 31, 2, 1, 32), (12, 40, 4, 2, 32), (16, 12, 2, 1, 32),
                                                     (16, 13, 4, 1, 32), (16, 20, 2, 3, 64)])
def test_ladders_split_over_a_cluster(sg, O, L, NT, R, pt_every, n_samples):
    """Ladders that do not fit in the shared memory of one SM: two CTAs of a thread-block cluster own one half of the
    slots each; the slot pair across them is decided by both from energies read through distributed shared memory and
    swapped by remote reads + a cluster barrier + local writes.  Even and odd numbers of slots (the cross pair is
    exchanged at one parity only), exchanges every 1 / 2 / 3 sweeps, plain sweeps from the same state (independent
    halves) — spins, the kernel's own energies, accepted swaps and moments vs the oracle."""
    temps = W.ladder(0.6, 1.8, NT)
    samples = sorted({0, n_samples - 1})
    sim, orc = make_pair(sg, O, L, 0.15, n_samples, R, temps, 0, 21, samples)
    n = 6 * pt_every
    sim.sg_run(n, pt_every, 3 * pt_every)
    for o in orc.values():
        o.run(n, pt_every, 3 * pt_every)
    check_state(sim, orc, "split ladder")
    Uc, Mc = sim.sg_get_energies_cached()
    for s, o in orc.items():
        Uo, Mo = o.energies()
        assert np.array_equal(Uc[s], Uo) and np.array_equal(Mc[s], Mo), "split ladder: the kernel's own energies"
    mom, nm = sim.sg_get_moments()
    assert nm == 2
    for s, o in orc.items():
        assert close(mom[s], o.moments()[0])
    prop, acc = sim.sg_get_pt_stats()
    assert prop.sum() > 0 and acc.sum() > 0
    sim.sg_sweep(2); sim.sg_run(3, 1, 0)
    for o in orc.values():
        o.sweep(2); o.run(3, 1, 0)
    check_state(sim, orc, "split ladder + plain sweeps + odd exchange")
    # the whole pool against the global-memory kernels
    h_fast = sim.sg_get_state_hash()
    sim.close()
    gen = sg.Simulation(L, 0.15, n_samples, R, temps, 0, 21)
    gen.sg_set_kernel_path(sg.PATH_GENERIC)
    gen.sg_run(n, pt_every, 3 * pt_every); gen.sg_sweep(2); gen.sg_run(3, 1, 0)
    assert np.array_equal(gen.sg_get_state_hash(), h_fast)
    gen.close()
