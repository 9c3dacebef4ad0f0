"""Pins for the oracle's sweep / PT / energy logic that need no statistics (exact, bitwise).

CPU only.  Brute-force references here are written with numpy.roll on a 3-D array — a different
indexing scheme from the oracle's neighbour table — and share nothing with the CUDA path.
"""
import numpy as np
import pytest

from oracle import ea_oracle as O
from paper_1403_4560_b200 import workloads as W

HOT, COLD = 1e300, 1e-300      # beta = 0 (every thr = 2^32) and beta = inf (thr = 0 for dE > 0)


def _grid(v, L):
    """[N] with i = x + Lx*(y + Ly*z)  ->  [z][y][x]"""
    Lx, Ly, Lz = L
    return np.asarray(v).reshape(Lz, Ly, Lx)


def _local_sum(S, J, L):
    """sum_j J_ij S_j for every site, from the bond list (i,d) -> i+e_d."""
    S = _grid(S, L).astype(np.float64)
    Jx, Jy, Jz = (_grid(J[d], L).astype(np.float64) for d in range(3))
    f = Jx * np.roll(S, -1, axis=2) + np.roll(Jx * S, 1, axis=2)
    f += Jy * np.roll(S, -1, axis=1) + np.roll(Jy * S, 1, axis=1)
    f += Jz * np.roll(S, -1, axis=0) + np.roll(Jz * S, 1, axis=0)
    return f


def _energy(S, J, h, L):
    """literal Eq. 1"""
    S3 = _grid(S, L).astype(np.float64)
    E = 0.0
    for d, ax in ((0, 2), (1, 1), (2, 0)):
        E -= np.sum(_grid(J[d], L) * S3 * np.roll(S3, -1, axis=ax))
    return E - h * S3.sum()


def _colour(L):
    Lx, Ly, Lz = L
    z, y, x = np.meshgrid(np.arange(Lz), np.arange(Ly), np.arange(Lx), indexing="ij")
    return (x + y + z) & 1


@pytest.mark.parametrize("L", [(4, 4, 4), (6, 4, 2), (2, 2, 2)])
def test_beta_zero_flips_everything(L):
    o = O.Oracle(L, 0.3, 2, [HOT, HOT], seed=11, sample=3)
    assert np.all(o.thresholds() == 1 << 32)
    S0 = o.spins()
    o.sweep(1)
    assert np.array_equal(o.spins(), -S0)
    o.sweep(1)
    assert np.array_equal(o.spins(), S0)


@pytest.mark.parametrize("L,h", [((4, 4, 4), 0.3), ((6, 6, 6), 0.0), ((8, 4, 6), -0.2), ((4, 4, 4), 2.5)])
def test_beta_infinity_is_greedy_descent(L, h):
    """thr = 0 for dE > 0, 2^32 for dE <= 0: deterministic, independent of the draws.
    Checks neighbour / periodic-wrap / bond-ownership indexing against a numpy.roll brute force."""
    o = O.Oracle(L, h, 2, [COLD], seed=12, sample=37)
    J = o.couplings()
    S = o.spins().astype(np.float64)
    col = _colour(L)
    for sweep in range(3):
        o.sweep(1)
        for a in range(2):
            s = S[a, 0]
            for c in (0, 1):
                s3 = _grid(s, L)
                dE = 2.0 * s3 * (_local_sum(s, J, L) + h)
                flip = (dE <= 0) & (col == c)
                s = np.where(flip, -s3, s3).ravel()
            S[a, 0] = s
        assert np.array_equal(o.spins(), S.astype(np.int8)), sweep


@pytest.mark.parametrize("kind", [O.PMJ, O.GAUSS])
def test_tracked_energy_equals_recomputed_and_eq1(kind):
    L = (4, 4, 6)
    temps = W.ladder(0.5, 2.0, 5)
    h = 0.3
    o = O.Oracle(L, h, 4, temps, kind=kind, seed=21, sample=40)
    J = o.couplings().astype(np.float64)
    N = o.N
    for step in range(40):
        o.sweep(1)
        if step % 2 == 0:
            o.pt_exchange()
        U, M = o.energies()
        U2, M2 = o.recomputed_energies()
        assert np.array_equal(U, U2) and np.array_equal(M, M2)
        if step % 8 == 0:
            S = o.spins()
            for a in range(4):
                for t in range(5):
                    E1 = _energy(S[a, t], J, h, L)
                    assert M[a, t] == S[a, t].sum()
                    if kind == O.PMJ:      # E = 2U - 3N - hM exactly
                        assert E1 == pytest.approx(2 * U[a, t] - 3 * N - h * M[a, t], abs=1e-9)
                        assert o.energy_pt(a, t) == pytest.approx(E1, abs=1e-9)
                    else:                  # fixed point: trunc(J 2^32) loses < 2^-32 per bond
                        assert abs(o.energy_pt(a, t) - E1) < 3 * N * 2.0**-32 + 1e-9
                    assert o.hamiltonian(a, t) == pytest.approx(E1, abs=1e-9)


def test_gauge_covariance_h0():
    """S_i -> e_i S_i, J_ij -> e_i J_ij e_j at h=0 maps the trajectory to its gauge image (same draws)."""
    L = (4, 4, 4)
    temps = W.ladder(0.6, 1.8, 4)
    a = O.Oracle(L, 0.0, 2, temps, seed=31, sample=9)
    b = O.Oracle(L, 0.0, 2, temps, seed=31, sample=9)
    rng = np.random.default_rng(1)
    eps = rng.choice([-1, 1], size=a.N).astype(np.int8)
    J = a.couplings().astype(np.int8)
    e3 = _grid(eps, L)
    Jg = np.stack([(_grid(J[d], L) * e3 * np.roll(e3, -1, axis=ax)).ravel() for d, ax in ((0, 2), (1, 1), (2, 0))])
    b.set_couplings_pm(Jg.astype(np.int8))
    b.set_spins(a.spins() * eps)
    for step in range(25):
        a.sweep(1); b.sweep(1)
        a.pt_exchange(); b.pt_exchange()
        assert np.array_equal(b.spins(), a.spins() * eps)
        assert np.array_equal(a.energies()[0], b.energies()[0])


@pytest.mark.parametrize("kind", [O.PMJ, O.GAUSS])
def test_field_reversal_covariance(kind):
    """(h, S) -> (-h, -S) with the same J and draws gives the negated trajectory (any h)."""
    L = (4, 4, 4)
    temps = W.ladder(0.5, 2.0, 4)
    a = O.Oracle(L, 0.3, 2, temps, kind=kind, seed=41, sample=2)
    b = O.Oracle(L, -0.3, 2, temps, kind=kind, seed=41, sample=2)
    b.set_spins(-a.spins())
    for step in range(25):
        a.sweep(1); b.sweep(1)
        a.pt_exchange(); b.pt_exchange()
        assert np.array_equal(b.spins(), -a.spins())
        assert np.array_equal(a.energies()[0], b.energies()[0])
        assert np.array_equal(a.energies()[1], -b.energies()[1])


def test_pt_equal_temperatures_known_permutation():
    """All slots at one T -> x = 0 -> every proposed swap accepted: slot contents follow the
    even/odd transposition network (R12)."""
    NT = 5
    o = O.Oracle(4, 0.3, 2, [1.0] * NT, seed=51, sample=1)
    S0 = o.spins().copy()
    perm = list(range(NT))           # perm[t] = which original configuration sits in slot t
    for e in range(7):
        o.pt_exchange()
        for t in range(e & 1, NT - 1, 2):
            perm[t], perm[t + 1] = perm[t + 1], perm[t]
        S = o.spins()
        for t in range(NT):
            assert np.array_equal(S[:, t], S0[:, perm[t]])
    prop, acc = o.pt_stats()
    assert prop == acc == 2 * sum(len(range(e & 1, NT - 1, 2)) for e in range(7))
    assert o.counters() == (0, 7)


def test_pt_never_accepts_hopeless_swap():
    """x < -22.5 -> dexp64 = 0 -> never accepted: T = (cold, hot) with the cold slot in its ground
    state and the hot slot in a high-energy state."""
    L = (4, 4, 4)
    o = O.Oracle(L, 0.0, 1, [0.01, 100.0], seed=52, sample=0)
    J = np.ones((3, 64), dtype=np.int8)
    o.set_couplings_pm(J)                        # ferromagnet
    S = np.ones((1, 2, 64), dtype=np.int8)
    S[0, 1] = (1 - 2 * _colour(L)).ravel()       # Neel state: every bond unsatisfied
    o.set_spins(S)
    U, _ = o.energies()
    assert U[0, 0] == 0 and U[0, 1] == 192
    for _ in range(4):
        o.pt_exchange()
    assert np.array_equal(o.spins(), S)
    # swapped the other way round (cold slot holds the bad state) it is always accepted (x >= 0)
    o.set_spins(S[:, ::-1])
    o.pt_exchange(); o.pt_exchange()
    assert np.array_equal(o.spins(), S)


def test_lane_independence_of_samples():
    """Sample s is simulated in isolation: bits of other lanes never enter (same word, other lane
    gives another trajectory; same sample twice gives the same one)."""
    w = W.BY_NAME["C1"]
    a = O.Oracle(w.L, w.h, 2, w.temps(), seed=7, sample=33)
    b = O.Oracle(w.L, w.h, 2, w.temps(), seed=7, sample=33)
    c = O.Oracle(w.L, w.h, 2, w.temps(), seed=7, sample=34)
    a.run(20, 1, 0); b.run(20, 1, 0); c.run(20, 1, 0)
    assert np.array_equal(a.spins(), b.spins())
    assert not np.array_equal(a.spins(), c.spins())


def test_run_equals_primitive_sequence():
    w = W.BY_NAME["C1"]
    a = O.Oracle(w.L, w.h, 4, w.temps(), seed=1, sample=0)
    b = O.Oracle(w.L, w.h, 4, w.temps(), seed=1, sample=0)
    a.run(30, 2, 5)
    for s in range(1, 31):
        b.sweep(1)
        if s % 2 == 0:
            b.pt_exchange()
        if s % 5 == 0:
            b.measure(False)
    assert np.array_equal(a.spins(), b.spins())
    assert np.array_equal(a.moments()[0], b.moments()[0]) and a.moments()[1] == b.moments()[1] == 6
