"""Pins for the oracle's diagnostics: the overlap distribution P(q) and the
per-window accumulators of the logarithmic-binning equilibration test (Fig. 5 caption).  CPU only.

P(q)  - exact enumeration on 2x2x2 (two independent replicas, Boltzmann weights) within the blocking error;
      - counting identities: every measurement adds exactly n_pairs counts per slot; the histogram of the oracle
        equals numpy.bincount of the integer overlaps recomputed from the spins at every measurement; identical
        replicas fill the last bin, opposite replicas the first; coarse bins are sums of fine bins.
log-binning
      - a measurement at sweep s lands in window floor(log2 s); window sums recomputed with numpy from the
        records returned by measure(); the windows add up to the total accumulators.
"""
import numpy as np
import pytest

from oracle import ea_oracle as O
from test_oracle_equilibrium import _binned_error, _exact


def test_pq_vs_exact_enumeration_2x2x2():
    L, h, temps = (2, 2, 2), 0.3, [0.7, 1.5, 3.0]
    o = O.Oracle(L, h, 2, temps, kind=O.PMJ, seed=77, sample=5)
    J = o.couplings().astype(np.float64)
    N = o.N
    o.run(1 << 10, 1, 0)
    o.enable_pq()
    n = 1 << 17
    o.run(n, 1, 1)                                   # measure after every sweep
    pq = o.pq().astype(np.float64)
    assert pq.shape == (3, N + 1) and np.all(pq.sum(axis=1) == n)
    for t, T in enumerate(temps):
        st, w, _, _ = _exact(L, J, h, T)
        ov = (st @ st.T).astype(np.int64)
        pw = np.outer(w, w)
        for idx in range(N + 1):
            p_exact = pw[ov == 2 * idx - N].sum()
            p = pq[t, idx] / n
            # binomial error inflated by the autocorrelation of successive sweeps (measured: tau < 8 at T >= 0.7)
            err = np.sqrt(max(p_exact * (1 - p_exact), 1e-9) / n * 16.0)
            assert abs(p - p_exact) < 4.5 * err + 2e-5, (T, idx, p, p_exact)


@pytest.mark.parametrize("L,R,kind", [((4, 4, 4), 4, O.PMJ), ((2, 2, 3), 2, O.PMJ), ((4, 2, 2), 2, O.GAUSS)])
def test_pq_equals_bincount_of_integer_overlaps(L, R, kind):
    temps = [0.8, 1.4, 2.5]
    o = O.Oracle(L, 0.2, R, temps, kind=kind, seed=3, sample=9)
    N = o.N
    o.enable_pq()
    want = np.zeros((3, N + 1), dtype=np.int64)
    n_pairs = R * (R - 1) // 2
    for step in range(60):
        o.run(2, 1, 0)
        S = o.spins().astype(np.int64)                      # [R][NT][N]
        o.measure(False)
        for t in range(3):
            for a in range(R):
                for b in range(a + 1, R):
                    Q = int((S[a, t] * S[b, t]).sum())
                    want[t, (Q + N) // 2] += 1
    got = o.pq().astype(np.int64)
    assert np.array_equal(got, want)
    assert np.all(got.sum(axis=1) == 60 * n_pairs)
    # coarse bins = sums of the fine bins they cover: bin = floor(idx * B / (N + 1))
    for B in (1, 2, 5, N // 2):
        o2 = O.Oracle(L, 0.2, R, temps, kind=kind, seed=3, sample=9)
        o2.enable_pq(B)
        for step in range(60):
            o2.run(2, 1, 0)
            o2.measure(False)
        coarse = np.zeros((3, B), dtype=np.int64)
        for idx in range(N + 1):
            coarse[:, idx * B // (N + 1)] += want[:, idx]
        assert np.array_equal(o2.pq().astype(np.int64), coarse)


def test_pq_identical_and_opposite_replicas():
    o = O.Oracle(4, 0.0, 2, [1.0], seed=1, sample=0)
    o.enable_pq()
    S = o.spins()
    S[1] = S[0]
    o.set_spins(S)
    o.measure(False)
    S[1] = -S[0]
    o.set_spins(S)
    o.measure(False)
    pq = o.pq()[0]
    assert pq[-1] == 1 and pq[0] == 1 and pq.sum() == 2
    with pytest.raises(ValueError):
        o.enable_pq(o.N + 2)


def test_log_binning_windows():
    L, R, temps = 4, 4, [0.9, 1.7]
    o = O.Oracle(L, 0.1, R, temps, seed=11, sample=2)
    o.enable_log_binning(6)
    P = R * (R - 1) // 2
    recs = {}                                            # sweep -> records [NT][P][25]
    for s in range(1, 101):
        o.sweep(1)
        if s % 3 == 0 or s in (1, 2, 64):
            recs[s] = o.measure()
    tot, n_tot = o.moments()
    assert n_tot == len(recs)
    sum_w = np.zeros_like(tot)
    for k in range(6):
        got, n_k = o.window_moments(k)
        members = [s for s in recs if min(int(np.floor(np.log2(s))), 5) == k]
        assert n_k == len(members)
        want = np.zeros_like(got)
        for s in members:                                # numpy restatement of R9 on the returned records
            r = recs[s]
            q0 = r[:, :, 0]
            want[:, 0] += q0.sum(1); want[:, 1] += (q0**2).sum(1); want[:, 2] += (q0**3).sum(1); want[:, 3] += (q0**4).sum(1)
            pairs = [(a, b) for a in range(R) for b in range(a + 1, R)]
            for kk in range(12):
                z = r[:, :, 1 + 2 * kk] + 1j * r[:, :, 2 + 2 * kk]
                want[:, 4 + 5 * kk] += z.real.sum(1)
                want[:, 5 + 5 * kk] += z.imag.sum(1)
                want[:, 6 + 5 * kk] += (np.abs(z)**2).sum(1)
                for p in range(P):
                    for p2 in range(p + 1, P):
                        shared = len(set(pairs[p]) & set(pairs[p2]))
                        want[:, 4 + 5 * kk + (3 if shared == 1 else 4)] += (z[:, p] * np.conj(z[:, p2])).real
            for p in range(P):
                for p2 in range(p + 1, P):
                    shared = len(set(pairs[p]) & set(pairs[p2]))
                    want[:, 64 if shared == 1 else 65] += q0[:, p] * q0[:, p2]
        assert np.allclose(got, want, rtol=1e-12, atol=1e-13), k
        sum_w += got
    assert np.allclose(sum_w, tot, rtol=1e-12, atol=1e-13)
    # windows 6.. are clamped into the last one: sweeps 64..100 (floor(log2) = 6) landed in window 5
    assert o.window_moments(5)[1] == len([s for s in recs if s >= 32])
