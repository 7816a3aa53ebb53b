"""GPU parity of the second-order flood step (sim_params_t::flood_order = 2): the
MUSCL-Hancock tile kernel against the oracle's flood_step_muscl, element by element one step from
identical injected state (1e-12 fp64, 1e-5 fp32 in the mixed norm), multi-step aggregates, and the
properties the scheme must keep on the GPU too (lake at rest with an island, exact mass)."""
import numpy as np
import pytest

import oracle
from paper_1908_05232_b200 import binding, scenarios as S
from helpers import box
from gpu_common import make_pair, sync, mixed

pytestmark = pytest.mark.gpu

TOL = {64: 1e-12, 32: 1e-5}


def _step_and_compare(sc, evolve, steps=1):
    sc.flood_order = 2
    o, g = make_pair(sc, evolve=evolve)
    assert g.flood_variant() == 5
    if not evolve:
        sync(o, g, sc)
    o.step(steps); g.step(steps)
    a, b = g.read_conserved(), o.read_conserved()
    tol = TOL[sc.real_bits] * steps
    for k in ("h", "qx", "qy"):
        assert mixed(a[k], b[k]) <= tol, (k, mixed(a[k], b[k]))
    sa, sb = g.stats(), o.stats()
    assert abs(sa["dt"] - sb["dt"]) <= 10 * tol * sb["dt"]
    return o, g


@pytest.mark.parametrize("evolve", [0, 7, 40])
def test_muscl_config1_single_step_fp64(evolve):
    _step_and_compare(S.make(1), evolve)


def test_muscl_config2_fp32_wet_dry_inflow_solids():
    sc = S.make(2)
    sc.hydro_q = sc.hydro_q * 20.0
    _step_and_compare(sc, 300)


@pytest.mark.parametrize("nx,ny", [(37, 11), (64, 9), (33, 40), (130, 7)])
def test_muscl_ragged_shapes_fp64(nx, ny):
    rng = np.random.default_rng(nx * 100 + ny)
    z = 0.3 * rng.random((ny, nx))
    h0 = np.where(rng.random((ny, nx)) < 0.7, 0.2 + 0.8 * rng.random((ny, nx)), 0.0)
    mask = (rng.random((ny, nx)) < 0.08).astype(np.uint8)
    u0 = 0.5 * (rng.random((ny, nx)) - 0.5); v0 = 0.5 * (rng.random((ny, nx)) - 0.5)
    sc = box(nx, ny, dx=0.5, z=z, h0=h0, u0=u0, v0=v0, manning=0.03, mask=mask)
    _step_and_compare(sc, 0)
    _step_and_compare(box(nx, ny, dx=0.5, z=z, h0=h0, u0=u0, v0=v0, manning=0.03, mask=mask), 5)


def test_muscl_config4_mini_fp32_single_step():
    sc = S.make(4, n=256, n_peds=2000)
    _step_and_compare(sc, 30)


def test_muscl_multi_step_aggregates_fp64():
    sc = S.make(1); sc.flood_order = 2
    o = oracle.Oracle(sc); g = binding.Sim(sc)
    o.step(100); g.step(100)
    sa, sb = g.stats(), o.stats()
    assert sa["step"] == sb["step"] == 100
    assert abs(sa["volume"] - sb["volume"]) <= 1e-10 * sb["volume"]
    assert abs(sa["max_h"] - sb["max_h"]) <= 1e-9 * sb["max_h"]
    assert sa["hist"] == sb["hist"]
    a, b = g.read_conserved(), o.read_conserved()
    assert mixed(a["h"], b["h"]) <= 1e-9


def test_muscl_lake_at_rest_with_island_and_mass_on_gpu():
    n = 48
    j, i = np.mgrid[0:n, 0:n]
    z = 0.8 * np.exp(-((i - 30) ** 2 + (j - 20) ** 2) / (2 * 6.0 ** 2))
    eta = 0.5
    h0 = np.maximum(0.0, eta - z)
    for bits in (64, 32):
        sc = box(n, n, dx=1.0, real_bits=bits, z=z, h0=h0, manning=0.02, flood_order=2)
        g = binding.Sim(sc)
        v0 = g.stats()["volume"]
        g.step(200)
        c = g.read_conserved()
        assert np.max(np.abs(c["qx"])) <= (1e-12 if bits == 64 else 2e-5)
        assert np.max(np.abs(c["qy"])) <= (1e-12 if bits == 64 else 2e-5)
        assert abs(g.stats()["volume"] - v0) <= (1e-12 if bits == 64 else 1e-5) * v0


def test_flood_order_is_validated_and_fixed():
    sc = S.make(1); sc.flood_order = 3
    with pytest.raises(binding.FloodpedError):
        binding.Sim(sc)
    sc.flood_order = 2
    g = binding.Sim(sc)
    with pytest.raises(binding.FloodpedError):
        g.set_flood_variant(1)
