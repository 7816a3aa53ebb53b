"""Not collected by pytest (minutes of oracle time): Configs 2 and 3 run to their t_end on the GPU and
in the oracle, aggregates and final depth field side by side.  `python tests/manual_full_runs.py`
on a GPU box; the round-1 output is quoted in BASELINE.md section 4."""
import sys, time, json, numpy as np
sys.path.insert(0, '.')
import oracle
from paper_1908_05232_b200 import binding, scenarios as S
out = {}
for cfg in (2, 3):
    sc = S.make(cfg)
    g = binding.Sim(sc)
    t0 = time.time()
    while g.stats()["t"] < sc.t_end: g.step(4096)
    tg = time.time() - t0
    sg = g.stats()
    o = oracle.Oracle(sc)
    t0 = time.time()
    while o.stats()["t"] < sc.t_end: o.step(4096)
    to = time.time() - t0
    so = o.stats()
    hg = g.read_conserved()["h"].astype(np.float64); ho = o.read_conserved()["h"]
    out[cfg] = dict(gpu_s=tg, oracle_s=to, gpu=sg, oracle=so, h_l1=float(np.abs(hg - ho).sum() / max(ho.sum(), 1e-30)), h_linf=float(np.abs(hg - ho).max()))
    print(cfg, json.dumps(out[cfg]))
