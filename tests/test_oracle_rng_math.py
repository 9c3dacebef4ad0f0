"""Pins for the oracle's Philox streams, threshold table and deterministic elementary functions.

CPU only.  Every expected value here comes from the paper/SURVEY fixtures under tests/golden/,
from Python's own big-integer / decimal / libm arithmetic, or from a closed form — never from
the CUDA path.
"""
import math
import os
from decimal import Decimal, getcontext

import numpy as np
import pytest

from oracle import ea_oracle as O
from paper_1403_4560_b200 import workloads as W


def _rows(path):
    with open(path) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                yield line.split()


def test_philox_known_answers(golden_dir):
    n = 0
    for r in _rows(os.path.join(golden_dir, "philox4x32_10_kat.txt")):
        v = [int(x, 16) for x in r]
        out = O.philox(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]
        n += 1
    assert n == 3


def _philox_bigint(ctr, key):
    """Independent restatement with Python integers (Salmon et al. SC'11, Philox4x32-10)."""
    c = list(ctr)
    k = list(key)
    for _ in range(10):
        p0 = 0xD2511F53 * c[0]
        p1 = 0xCD9E8D57 * c[2]
        c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xFFFFFFFF, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xFFFFFFFF]
        k = [(k[0] + 0x9E3779B9) & 0xFFFFFFFF, (k[1] + 0xBB67AE85) & 0xFFFFFFFF]
    return c


def test_philox_random_counters_vs_bigint():
    rng = np.random.default_rng(7)
    for _ in range(200):
        ctr = [int(x) for x in rng.integers(0, 1 << 32, 4, dtype=np.uint64)]
        key = [int(x) for x in rng.integers(0, 1 << 32, 2, dtype=np.uint64)]
        assert [int(x) for x in O.philox(ctr, key)] == _philox_bigint(ctr, key)


def test_philox_vs_torch_cpu_engine_statistics():
    # not a bit-level cross-check (torch's CPU engine has its own counter layout); checks the
    # stream is unbiased: mean of 2^16 words ~ 2^31, every bit ~ 1/2.
    out = np.array([O.philox([i, 0, 0, 0x03000000], [5, 0]) for i in range(1 << 14)], dtype=np.uint64).ravel()
    assert abs(out.mean() / 2**32 - 0.5) < 4 * (1 / math.sqrt(12 * out.size))
    bits = ((out[:, None] >> np.arange(32, dtype=np.uint64)) & 1).mean(axis=0)
    assert np.all(np.abs(bits - 0.5) < 5 * 0.5 / math.sqrt(out.size))


def test_keyed_draw_layout(golden_dir):
    """The oracle's own use of the counter layout: J bits, initial spins (lane 0 of config 1)."""
    for r in _rows(os.path.join(golden_dir, "keyed_draws_seed1.txt")):
        ctr = [int(x, 16) for x in r[0:4]]
        out = O.philox(ctr, [1, 0])
        for got, want in zip(out, r[4:8]):
            if want != "-":
                assert int(got) == int(want, 16)
    w = W.BY_NAME["C1"]
    o = O.Oracle(w.L, w.h, w.n_replicas, w.temps(), seed=1, sample=0)
    J = o.couplings()
    # couplings site 0: 9f3f38ef 8c470732 7e8a14f8 -> bit 0 = 1,0,0 -> J = -1,+1,+1 (bit 1 <-> J=-1)
    assert (J[0, 0], J[1, 0], J[2, 0]) == (-1.0, 1.0, 1.0)
    # initial spin i=0,a=0,t=0: 0c19cc69 bit0 = 1 -> S=+1 ; a=3,t=7: 67c73053 bit0 = 1 -> +1
    # (read before any sweep)
    S = o.spins()
    assert S[0, 0, 0] == 1 and S[3, 7, 0] == 1
    # lane 5 of the same word: bit 5 of 9f3f38ef (=1), 8c470732 (=1), 7e8a14f8 (=1)
    o5 = O.Oracle(w.L, w.h, w.n_replicas, w.temps(), seed=1, sample=5)
    J5 = o5.couplings()
    assert (J5[0, 0], J5[1, 0], J5[2, 0]) == tuple(
        -1.0 if (v >> 5) & 1 else 1.0 for v in (0x9F3F38EF, 0x8C470732, 0x7E8A14F8))


def test_initial_spin_bit_to_lane_mapping_from_bigint_philox():
    """R6, initial spins: word 0 of philox(c0 = i, c1 = 0, c2, (2 << 24) | (a << 16) | t); +-J: c2 = packed word s >> 5 and
    lane s & 31 reads bit s & 31 (1 <-> S = +1); Gaussian: c2 = s and bit 0 decides.  Expected values from the big-integer
    restatement of Philox above, for lanes other than 0, a second word, every replica / slot and a 64-bit seed."""
    seed = (0x9E3779B9 << 32) | 0x00C0FFEE
    key = [seed & 0xFFFFFFFF, seed >> 32]
    L, R, temps = 4, 4, list(W.ladder(0.5, 2.0, 5))
    N = L ** 3
    for kind, samples in ((O.PMJ, (5, 31, 32, 77)), (O.GAUSS, (0, 3, 33))):
        for s in samples:
            o = O.Oracle(L, 0.2, R, temps, kind=kind, seed=seed, sample=s)
            S = o.spins()                                   # [a][t][i], before any sweep
            o.close()
            n_up = 0
            for a in range(R):
                for t in range(len(temps)):
                    for i in range(N):
                        c2, bit = (s >> 5, s & 31) if kind == O.PMJ else (s, 0)
                        r0 = _philox_bigint([i, 0, c2, (2 << 24) | (a << 16) | t], key)[0]
                        want = 1 if (r0 >> bit) & 1 else -1
                        assert S[a, t, i] == want, (kind, s, a, t, i)
                        n_up += want == 1
            assert 0.4 < n_up / (R * len(temps) * N) < 0.6


def test_thresholds_worked_example(golden_dir):
    o = O.Oracle(4, 0.3, 1, [0.5, 2.0])
    thr = o.thresholds()
    n = 0
    for r in _rows(os.path.join(golden_dir, "thresholds_h0p3.txt")):
        t = 0 if r[0] == "0.5" else 1
        nu = int(r[1])
        assert int(thr[t, nu, 0]) == int(r[2]) and int(thr[t, nu, 1]) == int(r[3])
        n += 1
    assert n == 11


@pytest.mark.parametrize("h", [0.0, 0.1, 0.3, -0.2, 1.0])
def test_thresholds_vs_decimal(h):
    """thr = floor(exp(-beta dE) 2^32) with beta, dE the doubles of DESIGN.md R4, exp exact (50 digits)."""
    getcontext().prec = 50
    temps = list(W.ladder(0.4, 2.0, 9))
    o = O.Oracle(4, h, 1, temps)
    thr = o.thresholds()
    off = 0
    for t, T in enumerate(temps):
        beta = 1.0 / T
        for nu in range(7):
            for a in range(2):
                dE = float(12 - 4 * nu) + (2.0 * abs(h) if a else -(2.0 * abs(h)))
                if dE <= 0:
                    want = 1 << 32
                else:
                    want = int(((-(Decimal(beta) * Decimal(dE))).exp() * (1 << 32)).to_integral_value(rounding="ROUND_FLOOR"))
                    want = min(want, 1 << 32)
                got = int(thr[t, nu, a])
                assert abs(got - want) <= 1, (T, nu, a, got, want)   # libm exp is within 1 ulp
                off += got != want
    assert off <= 2
    # structure: monotone in n_u, aligned spins flip less easily
    assert np.all(np.diff(thr.astype(np.int64), axis=1) >= 0)
    assert np.all(thr[:, :, 1] <= thr[:, :, 0])


def test_dexp64_vs_libm():
    rng = np.random.default_rng(3)
    ys = np.concatenate([rng.uniform(0, 22.5, 4000), [1e-300, 1e-9, 0.00390625, 22.499999, 1.0, 12.0]])
    for y in ys:
        got = O.dexp64(y)
        want = math.exp(-y) * 4294967296.0
        assert abs(got - want) <= 1.0 + 4e-15 * want, (y, got, want)
    assert O.dexp64(22.5) == 0 and O.dexp64(1e9) == 0 and O.dexp64(float("inf")) == 0
    grid = np.linspace(1e-6, 22.49, 20001)
    vals = np.array([O.dexp64(y) for y in grid], dtype=np.float64)
    assert np.all(np.diff(vals) <= 0)            # monotone non-increasing
    assert O.dexp64(1e-12) <= 1 << 32


def test_dexp32_vs_libm():
    rng = np.random.default_rng(4)
    for y in rng.uniform(0, 22.5, 4000).astype(np.float32):
        got = O.dexp32(y)
        want = math.exp(-float(y)) * 4294967296.0
        assert abs(got - want) <= 1.0 + 1e-6 * want, (y, got, want)
    assert O.dexp32(22.5) == 0 and O.dexp32(100.0) == 0


def test_dlog_and_dsincos_vs_libm():
    rng = np.random.default_rng(5)
    us = np.concatenate([rng.uniform(0, 1, 5000), (np.arange(1, 50) + 0.5) * 2.0**-32, 1 - (np.arange(50) + 0.5) * 2.0**-32])
    for u in us:
        want = math.log(u)
        assert abs(O.dlog(u) - want) <= 1e-15 * abs(want) + 2e-16, u   # a few ulp; enough for one fp32 rounding of J
        c, s = O.dsincos2pi(u)
        assert abs(c - math.cos(2 * math.pi * u)) < 1.5e-15 and abs(s - math.sin(2 * math.pi * u)) < 1.5e-15  # 2*pi*u itself carries ~6e-16
    for u, cs in [(0.0, (1, 0)), (0.25, (0, 1)), (0.5, (-1, 0)), (0.75, (0, -1))]:
        assert O.dsincos2pi(u) == (float(cs[0]), float(cs[1]))


def test_gaussian_couplings_box_muller():
    """J ~ N(0,1): moments; each J equals the libm Box-Muller of the same Philox words to 1 fp32 ulp."""
    L = 8
    N = L**3
    Js = []
    for s in range(6):
        o = O.Oracle(L, 0.3, 1, [1.0], kind=O.GAUSS, seed=4, sample=s)
        J = o.couplings()
        Js.append(J)
        for i in (0, 1, 77, N - 1):
            r = O.philox([i, 0, s, 1 << 24], [4, 0]).astype(np.float64)
            u = (r + 0.5) * 2.0**-32
            rho = math.sqrt(-2 * math.log(u[0]))
            want = [rho * math.cos(2 * math.pi * u[1]), rho * math.sin(2 * math.pi * u[1]),
                    math.sqrt(-2 * math.log(u[2])) * math.cos(2 * math.pi * u[3])]
            for d in range(3):
                assert abs(float(J[d, i]) - want[d]) <= 2.5e-7 * max(1.0, abs(want[d]))
    J = np.concatenate([j.ravel() for j in Js]).astype(np.float64)
    n = J.size
    assert abs(J.mean()) < 4 / math.sqrt(n)
    assert abs(J.var() - 1) < 4 * math.sqrt(2 / n)
    assert abs(((J - J.mean())**4).mean() / J.var()**2 - 3) < 4 * math.sqrt(24 / n)
    assert abs(np.mean(J[:-1] * J[1:])) < 4 / math.sqrt(n)


def test_ladder_closed_form():
    """beta_n = beta_min alpha^(n-1): endpoints exact, constant ratio."""
    T = np.array(W.ladder(0.5, 2.0, 20))
    assert T[0] == 0.5 and T[-1] == 2.0 and np.all(np.diff(T) > 0)
    ratio = T[1:] / T[:-1]
    assert np.allclose(ratio, (2.0 / 0.5) ** (1 / 19), rtol=1e-13)
    beta = 1 / T[::-1]                     # ascending beta = paper's orientation
    assert np.allclose(beta[1:] / beta[:-1], (beta[-1] / beta[0]) ** (1 / 19), rtol=1e-13)
