"""8f-1: one item of the barrier sweep (replicas.run_barrier_item) on the GPU against the oracle run
of the same scenario: deposits and barrier state exact, volume / depth within the multi-step fp32
tolerance of DESIGN.md 5.4."""
import numpy as np
import pytest

import oracle
from paper_1908_05232_b200 import replicas, scenarios as S

pytestmark = pytest.mark.gpu


def test_barrier_sweep_item_matches_the_oracle_run():
    item = dict(n_layers=2, share=0.25)
    kw = dict(n=128, n_people=120, t_end=400.0, t_release=100.0)
    rec = replicas.run_barrier_item(item, steps_per_poll=64, **kw)
    n_resp = rec["n_responders"]
    assert n_resp == 30
    sc = S.shopping_centre(n=kw["n"], n_evac=kw["n_people"] - n_resp, n_resp=n_resp, t_release=kw["t_release"],
                           t_end=kw["t_end"], name="barrier_sweep")
    sc.n_layers = item["n_layers"]
    o = oracle.Oracle(sc)
    while o.stats()["t"] < kw["t_end"]:
        o.step(256)
    so = o.stats()
    assert rec["t"] == pytest.approx(kw["t_end"], abs=1e-9) and so["t"] == pytest.approx(kw["t_end"], abs=1e-9)
    # fp32 dt drifts, so step counts may differ slightly; the integer barrier state at t_end must not
    assert abs(rec["steps"] - so["step"]) <= max(2, so["step"] // 500)
    assert abs(rec["deposits"] - so["deposits"]) <= 1
    assert rec["volume"] == pytest.approx(so["volume"], rel=1e-3)
    h = o.read_flood()["h"].reshape(sc.ny, sc.nx)
    line_j = int(sc.line_cells[0] // sc.nx)
    down = (sc.mask.reshape(sc.ny, sc.nx) == 0); down[:line_j + 1, :] = False
    assert rec["depth_downstream"] == pytest.approx(float(h[down].mean()), rel=2e-2, abs=1e-5)
