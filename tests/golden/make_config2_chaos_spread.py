"""Writes tests/golden/config2_chaos_spread.txt.  Calls only oracle/ and the seeded scenario
generators; run from the repo root:  python tests/golden/make_config2_chaos_spread.py

What it measures: how far the ORACLE drifts from ITSELF over the free-running
600-step run that tests/test_gpu_parity.py::test_config2_multi_step_aggregates_fp32 compares the
CUDA path on (Config 2 with 10 x the inflow, 2000 evacuees queueing at one exit), when the initial
positions are moved by one fp32 unit in the last place (x (1 +- 2^-23), sign drawn per agent and
coordinate from numpy's default_rng(seed)).  That perturbation is what storing the positions in
fp32 does to them at every step, so the spread of the ensemble is the resolution below which no
fp32 run -- the CUDA path's or anybody's -- can be told from the fp64 oracle by its state
histogram (P:L110 compares predictions of the GPU and the sequential model).

Rows:  left <seed, -1 = unperturbed> <agents that have left by step 600> <hist L1 against the base run>
                        <agents in another class than in the base run>
       segment <start step> <K> <agents in another class> <agents in another cell> after K steps
                        from a state that differs by one fp32 ulp (how fast it happens)
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
import oracle                                                   # noqa: E402
from paper_1908_05232_b200 import scenarios as S                # noqa: E402

N_SEEDS, STEPS, EPS = 30, 600, 2.0 ** -23


def scenario():
    sc = S.make(2)
    sc.hydro_q = sc.hydro_q * 10.0
    return sc


def classes(p):
    return np.where(p["active"] != 0, np.minimum(p["state"], 4), 5)


def nudge(o, rng):
    p = o.read_peds()
    x = p["x"] * (1.0 + EPS * rng.choice([-1.0, 1.0], p["x"].shape))
    y = p["y"] * (1.0 + EPS * rng.choice([-1.0, 1.0], p["y"].shape))
    o.write_peds(x, y, p["vx"], p["vy"], p["fsm"], p["active"], p["timer"])


def main():
    sc = scenario()
    rows = []
    base = oracle.Oracle(sc)
    base.step(STEPS)
    h0, c0 = base.stats()["hist"], classes(base.read_peds())
    rows.append(f"left -1 {h0[5]} 0 0")
    for seed in range(N_SEEDS):
        o = oracle.Oracle(sc)
        nudge(o, np.random.default_rng(seed))
        o.step(STEPS)
        h = o.stats()["hist"]
        rows.append(f"left {seed} {h[5]} {sum(abs(a - b) for a, b in zip(h, h0))} {int((classes(o.read_peds()) != c0).sum())}")
        print(rows[-1], flush=True)
    rng = np.random.default_rng(1000)
    for start in (0, 100, 300):
        for K in (25, 50):
            a, b = oracle.Oracle(sc), oracle.Oracle(sc)
            a.step(start); b.step(start)
            nudge(b, rng)
            a.step(K); b.step(K)
            pa, pb = a.read_peds(), b.read_peds()
            both = (pa["active"] == 1) & (pb["active"] == 1)
            rows.append(f"segment {start} {K} {int((classes(pa) != classes(pb)).sum())} {int((pa['cell'] != pb['cell'])[both].sum())}")
            print(rows[-1], flush=True)
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "config2_chaos_spread.txt"), "w") as f:
        f.write("# Written by tests/golden/make_config2_chaos_spread.py (oracle only; see its docstring).\n")
        f.write("# The oracle against itself, initial positions moved by one fp32 ulp: Config 2 x 10 inflow, 600 steps.\n")
        f.write("\n".join(rows) + "\n")


if __name__ == "__main__":
    main()
