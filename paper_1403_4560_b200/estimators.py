"""Estimators of the paper's indicators from the device moment accumulators.

Host-side arithmetic only (numpy, double): the Monte Carlo path — sweeps, exchanges, overlaps and their
accumulation — runs in the CUDA kernels; this module turns `sg_get_moments()` output into

    g        Binder ratio, Eq. 3, both readings of its denominator (R10)
    chi(k)   wave-vector dependent spin-glass susceptibility, Eq. 4, |q(k)|^2 for complex q (R11),
             averaged over the symmetry-equivalent wave vectors, and its 4-replica connected form
    xi_L     second-moment correlation length, Eq. 5, sin(k_min/2) = sin(pi/L)
    R12      chi(k1)/chi(k2), Eq. 6, with the paper's k2 = (2pi/L)(1,1,0) and BASELINE.json's
             k2 = (4pi/L)(1,0,0)
    errors   jackknife over blocks of whole packed words (32 samples share their sweep random numbers, R5;
             PAPER.md:106 "jackknife ... from sample-to-sample variation")

Accumulator layout (R9), per (sample, slot), summed over replica pairs and measurements:
    [0..3]       sum q, q^2, q^3, q^4                     (q = q_ab(0))
    [4+5k+0..2]  sum Re q(K_k), Im q(K_k), |q(K_k)|^2     k = 0..11
    [4+5k+3]     sum Re(q_p q_p'*) over the 12 couples of pairs sharing one replica   (4 replicas only)
    [4+5k+4]     the same over the 3 disjoint couples
    [64], [65]   those two sums for k = 0
K0-2 = (2pi/L) e_x,y,z; K3-5 = (4pi/L) e_x,y,z; K6-11 = (2pi/L){(1,1,0),(1,-1,0),(1,0,1),(1,0,-1),(0,1,1),(0,1,-1)}.
"""
from typing import Dict

import numpy as np

NMOM = 66
K1_SET = (0, 1, 2)                  # (2pi/L, 0, 0) and permutations: k_min = k_1
K2_BASELINE_SET = (3, 4, 5)         # (4pi/L, 0, 0) and permutations: BASELINE.json's k_2
K2_PAPER_SET = (6, 7, 8, 9, 10, 11)  # (2pi/L, +-2pi/L, 0) and permutations: the paper's k_2


def _check(mom, n_meas, n_pairs):
    mom = np.asarray(mom, dtype=np.float64)
    if mom.ndim != 3 or mom.shape[2] != NMOM:
        raise ValueError("moments must have shape [n_samples][n_temps][%d]" % NMOM)
    if n_meas < 1 or n_pairs not in (1, 6):
        raise ValueError("need n_meas >= 1 and n_pairs in {1, 6}")
    return mom


def _point(mom_mean, mom_per_sample, N, L, n_meas, n_pairs):
    """All indicators from disorder-AVERAGED accumulators mom_mean [NT][66] (plus the per-sample ones, needed
    only for the literal reading of Eq. 3's denominator).  Returns a dict of [NT] arrays."""
    c = 1.0 / (n_meas * n_pairs)
    m1, m2, m3, m4 = (mom_mean[:, i] * c for i in range(4))
    Q = m1
    var = m2 - Q * Q
    mu4 = m4 - 4.0 * Q * m3 + 6.0 * Q * Q * m2 - 3.0 * Q ** 4
    with np.errstate(divide="ignore", invalid="ignore"):
        g_std = 0.5 * (3.0 - mu4 / (var * var))
        # literal Eq. 3: the square of the thermal second central moment sits inside the disorder average
        c2_s = (mom_per_sample[:, :, 1] - 2.0 * Q[None, :] * mom_per_sample[:, :, 0]) * c + (Q * Q)[None, :]
        g_lit = 0.5 * (3.0 - mu4 / np.mean(c2_s * c2_s, axis=0))
        chi0 = N * var
        out = {"q": Q, "q2": m2, "g_std": g_std, "g_lit": g_lit, "chi0": chi0}

        def chi_of(kset):
            acc = 0.0
            for k in kset:
                re, im, ab = (mom_mean[:, 4 + 5 * k + j] * c for j in range(3))
                acc = acc + N * (ab - (re * re + im * im))
            return acc / len(kset)

        def chi4_of(kset):            # 4-replica connected form, pairs (12), (12,13), (12,34)
            acc = 0.0
            for k in kset:
                ab = mom_mean[:, 4 + 5 * k + 2] * c
                share = mom_mean[:, 4 + 5 * k + 3] / (12.0 * n_meas)
                disj = mom_mean[:, 4 + 5 * k + 4] / (3.0 * n_meas)
                acc = acc + N * (ab - 2.0 * share + disj)
            return acc / len(kset)

        chi1, chi2p, chi2b = chi_of(K1_SET), chi_of(K2_PAPER_SET), chi_of(K2_BASELINE_SET)
        out.update(chi_k1=chi1, chi_k2_paper=chi2p, chi_k2_baseline=chi2b,
                   R12=chi1 / chi2p, R12_baseline=chi1 / chi2b)
        ratio = chi0 / chi1
        xi = np.sqrt(np.where(ratio >= 1.0, ratio - 1.0, np.nan)) / (2.0 * np.sin(np.pi / L))
        out.update(xi_L=xi, xi_L_over_L=xi / L)
        if n_pairs == 6:
            chi0_4 = N * (m2 - 2.0 * mom_mean[:, 64] / (12.0 * n_meas) + mom_mean[:, 65] / (3.0 * n_meas))
            c1, c2p, c2b = chi4_of(K1_SET), chi4_of(K2_PAPER_SET), chi4_of(K2_BASELINE_SET)
            out.update(chi0_4rep=chi0_4, chi_k1_4rep=c1, chi_k2_paper_4rep=c2p, chi_k2_baseline_4rep=c2b,
                       R12_4rep=c1 / c2p, R12_baseline_4rep=c1 / c2b)
    return out


def indicators(mom, n_meas: int, L: int, n_pairs: int = 6, block: int = 32) -> Dict[str, np.ndarray]:
    """Indicators and jackknife errors per temperature slot.

    mom      [n_samples][n_temps][66] accumulators of `sg_get_moments` (this rank's samples)
    n_meas   number of measurements accumulated
    block    jackknife block size in samples (32 = one packed word)
    Returns {name: [n_temps] value, name + "_err": [n_temps] jackknife error}.
    """
    mom = _check(mom, n_meas, n_pairs)
    S, NT, _ = mom.shape
    N = L ** 3
    full = _point(mom.mean(axis=0), mom, N, L, n_meas, n_pairs)
    out = dict(full)
    nb = (S + block - 1) // block
    if nb >= 2:
        tot = mom.sum(axis=0)
        jk = {k: np.empty((nb, NT)) for k in full}
        for b in range(nb):
            lo, hi = b * block, min(S, (b + 1) * block)
            rest = np.concatenate([mom[:lo], mom[hi:]], axis=0)
            est = _point((tot - mom[lo:hi].sum(axis=0)) / (S - (hi - lo)), rest, N, L, n_meas, n_pairs)
            for k in full:
                jk[k][b] = est[k]
        with np.errstate(invalid="ignore"):
            for k in full:
                d = jk[k] - jk[k].mean(axis=0)
                out[k + "_err"] = np.sqrt((nb - 1.0) / nb * np.sum(d * d, axis=0))
    return out


def log_binning(windows, n_meas_windows, L: int, n_pairs: int = 6, block: int = 32):
    """Logarithmic-binning equilibration test (Fig. 5 caption): the indicators evaluated separately on
    the measurements of every window [2^k, 2^(k+1)) of the sweep counter (`sg_get_window_moments`).

    windows          list of [n_samples][n_temps][66] window accumulators, index = k
    n_meas_windows   measurements that fell into each window
    Returns a list (index k) of `indicators(...)` dicts (None for an empty window).  A run passes the test when the
    last few windows agree within their errors (see `log_binning_passes`).
    """
    return [indicators(w, int(n), L, n_pairs, block) if n > 0 else None for w, n in zip(windows, n_meas_windows)]


def log_binning_passes(series, name: str, last: int = 3, n_sigma: float = 3.0) -> np.ndarray:
    """Per temperature slot: do the `last` non-empty windows of `series` (from `log_binning`) agree on indicator
    `name` within n_sigma combined jackknife errors?  Returns a bool array [n_temps]."""
    pts = [s for s in series if s is not None][-last:]
    if len(pts) < 2 or (name + "_err") not in pts[-1]:
        raise ValueError("need at least two non-empty windows with jackknife errors")
    ok = np.ones_like(pts[-1][name], dtype=bool)
    for s in pts[:-1]:
        err = np.sqrt(s[name + "_err"] ** 2 + pts[-1][name + "_err"] ** 2)
        ok &= np.abs(s[name] - pts[-1][name]) <= n_sigma * err
    return ok


def overlap_distribution(pq, L: int):
    """P(q) per slot from the device histogram of `sg_get_pq` ([n_samples][n_temps][n_bins] counts).

    Returns (q_centres [n_bins], P [n_temps][n_bins] disorder-averaged and normalised to sum 1 per slot,
    P_sample [n_samples][n_temps][n_bins] normalised per sample).  Bin b holds the overlaps with
    floor(agree * n_bins / (N + 1)) = b, agree = (N q + N) / 2; the centre is the mean q of the values it covers.
    """
    pq = np.asarray(pq, dtype=np.float64)
    n_bins = pq.shape[2]
    N = L ** 3
    agree = np.arange(N + 1)
    which = (agree * n_bins) // (N + 1)
    qv = (2.0 * agree - N) / N
    centres = np.array([qv[which == b].mean() if np.any(which == b) else np.nan for b in range(n_bins)])
    tot = pq.sum(axis=2, keepdims=True)
    with np.errstate(invalid="ignore", divide="ignore"):
        per_sample = np.where(tot > 0, pq / tot, 0.0)
    return centres, per_sample.mean(axis=0), per_sample
