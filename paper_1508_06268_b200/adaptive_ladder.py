"""The paper's adaptive-temperature scheme as a command-line driver.

Start from M replicas with temperatures equally spaced in [T_low, T_high].  Each of `--trials` trial runs
(`--pt-steps` parallel-tempering steps of `--sweeps-per-step` sweeps, "the same parameters" as the production run,
PAPER.md:224) measures the exchange rate of every adjacent pair and inserts the midpoint temperature into the
`--insertions` pairs with the lowest rate (rfim_pt_adapt_temperatures; the replica pool is pre-allocated).
Per trial the driver prints the number of replicas and the minimum / average / maximum exchange rate the update was
decided on -- the quantities of the paper's Figure 9 (left) -- and at the end the per-pair profile of the adapted ladder
next to homogeneous ladders of the same ("dense") and of the starting ("sparse") replica count (Figure 9, right).

    python -m paper_1508_06268_b200.adaptive_ladder --L 32 --replicas 20 --trials 10 --insertions 2
    python -m paper_1508_06268_b200.adaptive_ladder --L 64 --replicas 30 --trials 32 --insertions 3

Paper's parameters: bimodal field, h = 1, trials of 2000 PT steps of 10 sweeps; L = 32: 10 trials of 2
insertions, L = 64: 32 trials of 3.  The paper does not state its temperature range or starting replica counts (they are on
the labels of a figure that is not part of the text): T in [1.5, 4.5] and the --replicas defaults are this driver's.
Needs a CUDA device (the library has no CPU fallback).
"""
import argparse
import json
import time

import numpy as np


def _line(tag, n, rate):
    return f"{tag:>12s}  replicas {n:4d}  exchange rate  min {rate.min():.3f}  avg {rate.mean():.3f}  max {rate.max():.3f}"


def _profile(binding, args, T):
    """Exchange-rate profile of a fixed ladder over one trial-length run."""
    g = binding.RfimPT(args.L, len(T), args.J, args.h, args.field, seed=args.seed)
    g.set_temperatures(T)
    g.sweep(args.pt_steps * args.sweeps_per_step, args.sweeps_per_step)
    rate = g.observables()[2]
    g.close()
    return rate


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--L", type=int, default=32)
    ap.add_argument("--replicas", type=int, default=20, help="starting number of replicas M")
    ap.add_argument("--trials", type=int, default=10)
    ap.add_argument("--insertions", type=int, default=2, help="a: insertions per trial (the paper recommends 1..5)")
    ap.add_argument("--pt-steps", type=int, default=2000)
    ap.add_argument("--sweeps-per-step", type=int, default=10)
    ap.add_argument("--t-low", type=float, default=1.5)
    ap.add_argument("--t-high", type=float, default=4.5)
    ap.add_argument("--J", type=float, default=1.0)
    ap.add_argument("--h", type=float, default=1.0)
    ap.add_argument("--field", type=int, default=0, help="0 bimodal (the paper's), 1 Gaussian")
    ap.add_argument("--seed", type=int, default=1)
    ap.add_argument("--json", action="store_true", help="also print one JSON line with every number")
    args = ap.parse_args()

    from paper_1508_06268_b200 import binding
    cap = args.replicas + args.trials * args.insertions          # the pool holds the final replica count
    g = binding.RfimPT(args.L, cap, args.J, args.h, args.field, seed=args.seed)
    g.set_temperatures(np.linspace(args.t_low, args.t_high, args.replicas))
    g.set_adapt_params(args.sweeps_per_step, args.insertions)
    trial_sweeps = args.pt_steps * args.sweeps_per_step
    print(f"L={args.L} {'bimodal' if args.field == 0 else 'Gaussian'} field h={args.h}, T in [{args.t_low}, {args.t_high}], "
          f"{args.trials} trials x {args.insertions} insertions, trial = {args.pt_steps} PT steps x {args.sweeps_per_step} sweeps")
    record = {"args": vars(args), "trials": []}
    t0 = time.time()
    for trial in range(1, args.trials + 1):
        n = g.n
        g.adapt_temperatures(trial_sweeps)                    # one trial run + one ladder update
        rate = g.get_trial_rates()                            # the rates that update was decided on
        print(_line(f"trial {trial}", n, rate))
        record["trials"].append({"trial": trial, "replicas": n, "min": float(rate.min()), "avg": float(rate.mean()), "max": float(rate.max())})
    t_adapt = time.time() - t0
    T_adapted = g.get_temperatures()
    t0 = time.time()
    g.sweep(trial_sweeps, args.sweeps_per_step)               # the production run on the adapted ladder
    rate_adapted = g.observables()[2]
    t_prod = time.time() - t0
    g.close()
    print(_line("adapted", len(T_adapted), rate_adapted))
    rate_dense = _profile(binding, args, np.linspace(args.t_low, args.t_high, len(T_adapted)))
    print(_line("dense hom.", len(T_adapted), rate_dense))
    rate_sparse = _profile(binding, args, np.linspace(args.t_low, args.t_high, args.replicas))
    print(_line("sparse hom.", args.replicas, rate_sparse))
    print(f"wall: adaptation {t_adapt:.2f} s ({args.trials} trials), production run {t_prod:.2f} s")
    print("adapted ladder:", " ".join(f"{t:.4f}" for t in T_adapted))
    print("adapted rates: ", " ".join(f"{r:.3f}" for r in rate_adapted))
    if args.json:
        record.update({"T_adapted": [float(t) for t in T_adapted], "rate_adapted": [float(r) for r in rate_adapted],
                       "rate_dense": [float(r) for r in rate_dense], "rate_sparse": [float(r) for r in rate_sparse],
                       "wall_adapt_s": t_adapt, "wall_production_s": t_prod})
        print(json.dumps(record))


if __name__ == "__main__":
    main()
