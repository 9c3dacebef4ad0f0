"""Estimator layer (Eqs. 3-6) on CPU: the indicators computed from the
66-double accumulator layout (R9) against (i) the same quantities computed straight from raw overlap
records with numpy complex arithmetic, (ii) the closed forms for independent random spins
(<q^2> = 1/N, <q^4> = (3N-2)/N^3 -> g = 1/N; chi(k) = 1 for every k; R12 = 1; cross terms 0),
(iii) a brute-force leave-one-block-out jackknife."""
import itertools

import numpy as np
import pytest

from paper_1403_4560_b200 import estimators as E

L, N, R, NT, S, NMEAS = 4, 64, 4, 2, 96, 12
PAIRS = list(itertools.combinations(range(R), 2))
KVEC = [(1, 0, 0), (0, 1, 0), (0, 0, 1), (2, 0, 0), (0, 2, 0), (0, 0, 2),
        (1, 1, 0), (1, -1, 0), (1, 0, 1), (1, 0, -1), (0, 1, 1), (0, 1, -1)]


def _records(rng):
    """q_ab(0) and q_ab(K) for independent random spins: [S][NT][NMEAS][pair] and [...][12] complex."""
    x, y, z = np.meshgrid(np.arange(L), np.arange(L), np.arange(L), indexing="ij")
    phases = np.stack([np.exp(2j * np.pi * (kx * x + ky * y + kz * z) / L).ravel() for kx, ky, kz in KVEC])
    spins = rng.choice([-1.0, 1.0], size=(S, NT, NMEAS, R, N))
    q0 = np.empty((S, NT, NMEAS, len(PAIRS)))
    qk = np.empty((S, NT, NMEAS, len(PAIRS), 12), dtype=complex)
    for p, (a, b) in enumerate(PAIRS):
        prod = spins[..., a, :] * spins[..., b, :]
        q0[..., p] = prod.mean(axis=-1)
        qk[..., p, :] = prod @ phases.T / N
    return q0, qk


def _accumulate(q0, qk):
    """DESIGN.md R9 restated: per (sample, slot) sums over pairs and measurements."""
    mom = np.zeros((S, NT, E.NMOM))
    for i in range(4):
        mom[..., i] = (q0 ** (i + 1)).sum(axis=(2, 3))
    share = [(p, r) for p in range(6) for r in range(6) if p != r and len(set(PAIRS[p]) & set(PAIRS[r])) == 1]
    disj = [(p, r) for p in range(6) for r in range(p + 1, 6) if not set(PAIRS[p]) & set(PAIRS[r])]
    assert len(share) == 24 and len(disj) == 3           # 12 unordered sharing couples
    share = [(p, r) for p, r in share if p < r]

    def oriented(qa, pa, qb, pb):
        """Re(q_p q_r*) with both pairs oriented from the shared replica outwards; q_ba = q_ab for real spins."""
        return (qa * np.conj(qb)).real

    for k in range(12):
        mom[..., 4 + 5 * k + 0] = qk[..., k].real.sum(axis=(2, 3))
        mom[..., 4 + 5 * k + 1] = qk[..., k].imag.sum(axis=(2, 3))
        mom[..., 4 + 5 * k + 2] = (np.abs(qk[..., k]) ** 2).sum(axis=(2, 3))
        mom[..., 4 + 5 * k + 3] = sum(oriented(qk[..., p, k], p, qk[..., r, k], r) for p, r in share).sum(axis=2)
        mom[..., 4 + 5 * k + 4] = sum(oriented(qk[..., p, k], p, qk[..., r, k], r) for p, r in disj).sum(axis=2)
    mom[..., 64] = sum(q0[..., p] * q0[..., r] for p, r in share).sum(axis=2)
    mom[..., 65] = sum(q0[..., p] * q0[..., r] for p, r in disj).sum(axis=2)
    return mom


@pytest.fixture(scope="module")
def data():
    rng = np.random.default_rng(20140318)
    q0, qk = _records(rng)
    return q0, qk, _accumulate(q0, qk)


def test_indicators_equal_direct_definitions(data):
    q0, qk, mom = data
    out = E.indicators(mom, NMEAS, L, n_pairs=6)
    Q = q0.mean(axis=(0, 2, 3))
    assert np.allclose(out["q"], Q, rtol=0, atol=1e-15)
    cen = q0 - Q[None, :, None, None]
    mu2, mu4 = (cen ** 2).mean(axis=(0, 2, 3)), (cen ** 4).mean(axis=(0, 2, 3))
    assert np.allclose(out["g_std"], 0.5 * (3 - mu4 / mu2 ** 2), rtol=1e-10)
    th2 = (cen ** 2).mean(axis=(2, 3))                            # thermal (+ pair) average per sample
    assert np.allclose(out["g_lit"], 0.5 * (3 - mu4 / (th2 ** 2).mean(axis=0)), rtol=1e-10)
    assert np.allclose(out["chi0"], N * mu2, rtol=1e-10)

    def chi(ks):
        return np.mean([N * ((np.abs(qk[..., k]) ** 2).mean(axis=(0, 2, 3)) - np.abs(qk[..., k].mean(axis=(0, 2, 3))) ** 2)
                        for k in ks], axis=0)

    assert np.allclose(out["chi_k1"], chi(E.K1_SET), rtol=1e-10)
    assert np.allclose(out["chi_k2_paper"], chi(E.K2_PAPER_SET), rtol=1e-10)
    assert np.allclose(out["chi_k2_baseline"], chi(E.K2_BASELINE_SET), rtol=1e-10)
    assert np.allclose(out["R12"], chi(E.K1_SET) / chi(E.K2_PAPER_SET), rtol=1e-10)
    assert np.allclose(out["R12_baseline"], chi(E.K1_SET) / chi(E.K2_BASELINE_SET), rtol=1e-10)
    ratio = N * mu2 / chi(E.K1_SET)
    want = np.where(ratio >= 1, np.sqrt(np.abs(ratio - 1)), np.nan) / (2 * np.sin(np.pi / L))
    assert np.allclose(out["xi_L"], want, rtol=1e-10, equal_nan=True)


def test_closed_forms_for_independent_spins(data):
    _, _, mom = data
    out = E.indicators(mom, NMEAS, L, n_pairs=6, block=4)          # 24 jackknife blocks (independent samples here)
    for name, want in [("chi0", 1.0), ("chi_k1", 1.0), ("chi_k2_paper", 1.0), ("chi_k2_baseline", 1.0), ("R12", 1.0),
                       ("R12_baseline", 1.0), ("g_std", 1.0 / N), ("chi_k1_4rep", 1.0), ("chi0_4rep", 1.0),
                       ("R12_4rep", 1.0), ("q", 0.0)]:
        err = out[name + "_err"]
        assert np.all(err > 0) and np.all(err < 0.2)
        assert np.all(np.abs(out[name] - want) < 5 * err), (name, out[name], err)
    assert np.allclose(out["q2"], 1.0 / N, rtol=0.05)


def test_jackknife_is_leave_one_word_out(data):
    _, _, mom = data
    out = E.indicators(mom, NMEAS, L, n_pairs=6, block=32)
    nb = S // 32
    vals = []
    for b in range(nb):
        keep = np.concatenate([mom[:32 * b], mom[32 * (b + 1):]])
        vals.append(E.indicators(keep, NMEAS, L, n_pairs=6, block=10 ** 9)["R12"])
    vals = np.array(vals)
    want = np.sqrt((nb - 1) / nb * ((vals - vals.mean(axis=0)) ** 2).sum(axis=0))
    assert np.allclose(out["R12_err"], want, rtol=1e-12)


def test_degenerate_inputs():
    mom = np.zeros((4, 1, E.NMOM))
    mom[..., 0] = 6 * 3 * 0.5
    mom[..., 1] = 6 * 3 * 0.25                     # q == 0.5 always: zero variance
    mom[..., 2] = 6 * 3 * 0.125
    mom[..., 3] = 6 * 3 * 0.0625
    out = E.indicators(mom, 3, 4, n_pairs=6, block=2)
    assert out["chi0"][0] == 0.0 and np.isnan(out["g_std"][0])
    with pytest.raises(ValueError):
        E.indicators(np.zeros((4, 1, 10)), 3, 4)
    with pytest.raises(ValueError):
        E.indicators(mom, 0, 4)
