"""Writes tests/golden/config3_copy_spread.txt: the copy-to-copy spread of the maximally Abelian functional on the 6^4
stand-in of BASELINE.json configs[3] (tests/test_gpu_parity.py, test_config3_anneal_then_or).

    python tests/golden/make_config3_copy_spread.py

Calls oracle/ and the seeded input generator only (never the CUDA path).  The annealing trajectory is chaotic
(R25): after a few steps the CUDA path and the oracle hold different Gribov copies of one orbit, so what a
test can ask of F at the end of the schedule, and after the overrelaxation, is that it lies inside the spread that
different random sequences produce.  That spread is measured here: 32 Philox seeds, the schedule and the run of the
test (12 annealing steps T 1.45 -> 0.01 with 3 microcanonical sweeps each, then OR omega 1.7 to theta < 1e-12).
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import gf_oracle as oracle          # noqa: E402
from paper_1212_5221_b200 import inputs         # noqa: E402  (seeded input generator, no arithmetic of the method)

MAG, OR = 2, 0
N_SEEDS = 32


def main():
    oracle.build()
    L = inputs.as_real(inputs.make_config(6, 6, 6, 6, 0.5, 350, 351))
    Fa, Ff, sweeps = [], [], []
    for k in range(N_SEEDS):
        ref = L.copy()
        nxt = oracle.anneal(ref, MAG, 1.45, 0.01, 12, 3, seed=1234 + k)
        Fa.append(oracle.measure(ref, MAG)["F"])
        s, F, th, hist, conv = oracle.run(ref, MAG, OR, 1.7, max_sweeps=8000, eps=1e-12, first_sweep_index=nxt)
        assert conv, k
        Ff.append(F)
        sweeps.append(s)
        print(k, Fa[-1], F, s, flush=True)
    Fa, Ff = np.array(Fa), np.array(Ff)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config3_copy_spread.txt")
    with open(out, "w") as fh:
        fh.write("# Copy-to-copy spread of F_MAG on the 6^4 stand-in of configs[3]; written by make_config3_copy_spread.py from\n"
                 "# oracle/ alone (32 Philox seeds 1234..1265, input make_config(6,6,6,6, 0.5, 350, 351)).  sigma = sample standard\n"
                 "# deviation (ddof = 1).  Format: key value\n")
        fh.write(f"n_seeds                 {N_SEEDS}\n")
        fh.write(f"F_after_anneal_mean     {Fa.mean():.12f}\n")
        fh.write(f"F_after_anneal_sigma    {Fa.std(ddof=1):.6e}\n")
        fh.write(f"F_final_mean            {Ff.mean():.12f}\n")
        fh.write(f"F_final_sigma           {Ff.std(ddof=1):.6e}\n")
        fh.write(f"F_final_min             {Ff.min():.12f}\n")
        fh.write(f"F_final_max             {Ff.max():.12f}\n")
        fh.write(f"or_sweeps_mean          {np.mean(sweeps):.1f}\n")
    print(open(out).read())


if __name__ == "__main__":
    main()
