"""The paper's own workload shapes at reduced volume (Table I).

    python -m paper_1403_4560_b200.table1 [--L 6 8] [--samples 4096] [--sweeps 65536] [--h 0.1]

L = 6, 8, 10; N_T = 56 temperatures geometric in beta in [0.1, 1.8]; h = 0.1 (or 0); 2 replicas; +-J couplings;
parallel tempering every sweep; first half of the sweeps discarded, overlaps measured every
`--meas-every` sweeps in the second half.  Prints, per size and temperature, the Binder ratio g (Eq. 3),
xi_L / L (Eq. 5) and R12 (Eq. 6, the paper's k2) with jackknife errors over whole packed words
(paper: 2*10^6 sweeps and 2.4-5*10^5 samples per size; here whatever volume is asked for).

Everything on the Monte Carlo path runs in the CUDA library (sg.py); this script only chooses parameters and
calls estimators.indicators on the accumulators.  The synthetic disorder is the library's Philox stream of
`--seed`; no external data is used.
"""
import argparse
import json
import time

import numpy as np

from . import estimators, workloads


def run_size(sg, L, n_samples, n_sweeps, h, n_temps, beta_lo, beta_hi, meas_every, seed, kind=None):
    temps = workloads.ladder(1.0 / beta_hi, 1.0 / beta_lo, n_temps)
    sim = sg.Simulation(L, h, n_samples, 2, temps, sg.PMJ if kind is None else kind, seed)
    t0 = time.perf_counter()
    half = n_sweeps // 2
    sim.sg_run(half, 1, 0)
    sim.sg_run(n_sweeps - half, 1, meas_every)
    mom, n_meas = sim.sg_get_moments()
    dt = time.perf_counter() - t0
    sim.close()
    out = estimators.indicators(mom, n_meas, L, n_pairs=1, block=32)
    flips = float(L) ** 3 * n_samples * 2 * n_temps * n_sweeps
    return temps, out, n_meas, dt, flips / dt / 1e9


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--L", type=int, nargs="+", default=[6, 8])
    ap.add_argument("--samples", type=int, default=4096)
    ap.add_argument("--sweeps", type=int, default=65536)
    ap.add_argument("--h", type=float, default=0.1)
    ap.add_argument("--temps", type=int, default=56)
    ap.add_argument("--beta-lo", type=float, default=0.1)
    ap.add_argument("--beta-hi", type=float, default=1.8)
    ap.add_argument("--meas-every", type=int, default=64)
    ap.add_argument("--seed", type=int, default=1403)
    ap.add_argument("--packing", default="samples", choices=["samples", "temperatures"],
                    help="samples: 32 disorder samples per word (default); temperatures: the paper's own packing "
                         "(SG_PMJ_TPACK, PAPER.md:68) — same trajectories, for few samples")
    ap.add_argument("--json", default="", help="also write the curves to this file")
    args = ap.parse_args()
    from . import sg
    curves = {}
    for L in args.L:
        temps, out, n_meas, dt, rate = run_size(sg, L, args.samples, args.sweeps, args.h, args.temps, args.beta_lo,
                                                args.beta_hi, args.meas_every, args.seed,
                                                sg.PMJ_TPACK if args.packing == "temperatures" else sg.PMJ)
        print("# L = %d, %d samples x 2 replicas x %d temperatures, h = %g, %d sweeps (PT every sweep), %d measurements, "
              "%.1f s, %.0f flips/ns" % (L, args.samples, args.temps, args.h, args.sweeps, n_meas, dt, rate))
        print("#  beta       T      g_std     +-     xi_L/L     +-       R12      +-   chi(k1)")
        for t in range(len(temps) - 1, -1, -1):
            print("%7.4f %7.4f  %8.5f %7.5f  %8.5f %7.5f  %8.5f %7.5f  %8.4f" % (
                1.0 / temps[t], temps[t], out["g_std"][t], out["g_std_err"][t], out["xi_L_over_L"][t],
                out["xi_L_over_L_err"][t], out["R12"][t], out["R12_err"][t], out["chi_k1"][t]))
        curves[str(L)] = {"beta": [1.0 / T for T in temps],
                          **{k: np.asarray(out[k]).tolist() for k in ("g_std", "g_std_err", "xi_L_over_L", "xi_L_over_L_err",
                                                                     "R12", "R12_err", "chi_k1", "chi0")}}
    if args.json:
        with open(args.json, "w") as f:
            json.dump({"args": vars(args), "curves": curves}, f)


if __name__ == "__main__":
    main()
