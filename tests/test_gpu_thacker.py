"""The CUDA flood kernels against Thacker's exact planar-surface solution (tests/test_oracle_thacker.py):
every kernel variant, both orders, fp64 and fp32, must land on the oracle's error against the exact
solution -- which ties the GPU path to the mathematics directly, not only to the oracle."""
import numpy as np
import pytest

import oracle
from paper_1908_05232_b200 import binding
from test_oracle_thacker import thacker_scenario, errors

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("bits", [64, 32])
@pytest.mark.parametrize("variant", [0, 1, 2, 3, 4, 5])
def test_thacker_on_the_gpu_matches_the_oracles_error(variant, bits):
    N = 64
    order = 2 if variant == 5 else 1
    sc, X, Y, T, dx = thacker_scenario(N, order, real_bits=bits)
    g = binding.Sim(sc)
    if variant != 5:
        g.set_flood_variant(variant)
    assert g.flood_variant() == variant
    v0 = g.stats()["volume"]
    g.step(10 ** 6)
    st = g.stats()
    assert abs(st["t"] - T) < (1e-9 if bits == 64 else 1e-5)
    assert abs(st["volume"] - v0) <= (1e-12 if bits == 64 else 2e-6) * v0
    e = errors(g, X, Y, T, dx, N)
    sco, *_ = thacker_scenario(N, order)
    o = oracle.Oracle(sco); o.step(10 ** 6)
    eo = errors(o, X, Y, T, dx, N)
    tol = 1e-9 if bits == 64 else 2e-4
    assert abs(e[0] - eo[0]) <= tol and abs(e[1] - eo[1]) <= tol, (e, eo)
    assert e[0] < (0.035 if order == 1 else 0.016)
