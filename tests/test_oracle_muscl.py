"""Pins for the oracle's second-order (MUSCL-Hancock) flood step, SURVEY 8f-2 -- the scheme the paper
"reduced to first-order accuracy".  The paper prints none of it (M1-M7), so the pins
are what the mathematics fixes: an exact smooth solution of the nonlinear shallow-water equations
(simple wave) with observed order ~2 against ~1 for the paper's first-order step, the C-property
including an emerging island, exact mass, the analytical Stoker dam break below the first-order
errors, symmetry under transposition, and the reduction to the first-order step where every slope
vanishes."""
import math

import numpy as np
import pytest

import oracle
from paper_1908_05232_b200 import scenarios as S
from helpers import box, golden_rows

G = 9.81


def test_minmod_limiter():
    assert oracle.minmod(1.0, 2.0) == 1.0 and oracle.minmod(-3.0, -2.0) == -2.0
    assert oracle.minmod(1.0, -2.0) == 0.0 and oracle.minmod(0.0, 5.0) == 0.0 and oracle.minmod(-1.0, 0.0) == 0.0


# ------------------------------------------------------------------ exact smooth solution: simple wave
# A right-going simple wave on a flat frictionless bed: the Riemann invariant u - 2c = -2 c0 is constant
# (c = sqrt(g h), c0 = sqrt(g H)), so u = 2 (c - c0) and c is constant along dx/dt = u + c = 3c - 2c0:
#     c(x, t) = c_init(xi),   x = xi + (3 c_init(xi) - 2 c0) t        (textbook; valid until the wave breaks)

H0, AMP, WID, X0, LEN = 1.0, 0.1, 5.0, 35.0, 100.0


def _h_init(x):
    return H0 + AMP * np.exp(-((x - X0) ** 2) / (2 * WID ** 2))


def _simple_wave(x, t):
    c0 = math.sqrt(G * H0)
    xi = x.copy()
    for _ in range(200):                               # fixed point: contraction while t * max|d speed/d xi| < 1
        c = np.sqrt(G * _h_init(xi))
        xi = x - (3 * c - 2 * c0) * t
    c = np.sqrt(G * _h_init(xi))
    return c * c / G, 2 * (c - c0)


def _run_wave(N, order, T=4.0):
    dx = LEN / N
    x = (np.arange(N) + 0.5) * dx
    h0 = _h_init(x)
    u0 = 2 * (np.sqrt(G * h0) - math.sqrt(G * H0))
    sc = box(N, 3, dx=dx, h0=np.tile(h0, (3, 1)), u0=np.tile(u0, (3, 1)), manning=0.0, t_end=T, h_dry=1e-6,
             flood_order=order)
    o = oracle.Oracle(sc)
    o.step(10 ** 7)
    assert abs(o.stats()["t"] - T) < 1e-12
    c = {k: v.reshape(3, N) for k, v in o.read_conserved().items()}
    assert np.array_equal(c["h"][0], c["h"][1]) and np.all(c["qy"] == 0.0)
    he, ue = _simple_wave(x, T)
    return float(np.mean(np.abs(c["h"][1] - he))), float(np.mean(np.abs(c["qx"][1] - he * ue)))


def test_simple_wave_second_order_convergence():
    e1 = {N: _run_wave(N, 1) for N in (100, 200, 400)}
    e2 = {N: _run_wave(N, 2) for N in (100, 200, 400)}
    p1 = math.log2(e1[200][0] / e1[400][0])
    p2 = math.log2(e2[200][0] / e2[400][0])
    q2 = math.log2(e2[200][1] / e2[400][1])
    # first order ~1; MUSCL with minmod (clips the crest) ~2 in L1
    assert 0.7 <= p1 <= 1.2, (p1, e1)
    assert p2 >= 1.7 and q2 >= 1.7, (p2, q2, e2)
    # and far more accurate at equal resolution
    assert e2[400][0] < 0.1 * e1[400][0], (e1, e2)


def test_stoker_dam_break_beats_first_order():
    """The analytical wet dam break (the authors' own verification idea): the second-order step
    must land below the first-order L1 errors stored in tests/golden/flux_hand_cases.txt."""
    for N, ref in golden_rows("flux_hand_cases.txt", "stoker_l1"):
        N = int(N)
        if N > 400:
            continue
        dx = 100.0 / N
        col = np.where(np.arange(N) < N // 2, 1.0, 0.1)
        sc = box(N, 3, dx=dx, h0=np.tile(col, (3, 1)), manning=0.0, t_end=6.0, h_dry=1e-6, flood_order=2)
        o = oracle.Oracle(sc)
        o.step(10 ** 7)
        h = o.read_conserved()["h"].reshape(3, N)
        x = (np.arange(N) + 0.5) * dx - 50.0
        from test_oracle_flood import _stoker_profile
        err = float(np.mean(np.abs(h[1] - _stoker_profile(x, 6.0, 1.0, 0.1))))
        assert err < 0.75 * ref, (N, err, ref)
        assert h.min() >= 0.0 and o.stats()["neg_depth_clamps"] == 0


# ------------------------------------------------------------------ invariants

@pytest.mark.parametrize("eta", [0.5, 0.2])          # 0.2 < bump top 0.3: an island emerges
def test_lake_at_rest_stays_at_rest_second_order(eta):
    sc = S.make(1, n_peds=0)
    sc.flood_order = 2
    sc.h0 = np.maximum(0.0, eta - sc.z)
    o = oracle.Oracle(sc)
    o.step(1000)
    c = o.read_conserved()
    assert o.stats()["step"] == 1000
    assert np.max(np.abs(c["qx"])) <= 1e-12 and np.max(np.abs(c["qy"])) <= 1e-12
    assert np.max(np.abs(c["h"] - sc.h0)) <= 1e-12
    assert o.stats()["neg_depth_clamps"] == 0


def test_config1_mass_conserved_second_order():
    sc = S.make(1)
    sc.flood_order = 2
    o = oracle.Oracle(sc)
    v0 = math.fsum(sc.h0) * sc.dx * sc.dy
    o.step(100)
    st = o.stats()
    h = o.read_conserved()["h"]
    assert abs(math.fsum(h) * sc.dx * sc.dy - v0) / v0 <= 1e-12
    assert h.min() >= 0.0 and st["neg_depth_clamps"] == 0
    # and it is a different scheme: sharper bore than the first-order run of the same config
    o1 = oracle.Oracle(S.make(1)); o1.step(100)
    assert np.max(np.abs(h - o1.read_conserved()["h"])) > 1e-3


def test_inflow_volume_second_order():
    """V(t) = sum dt Q(t^n) with inflow faces, walls and a dry start (C14): the same invariant as the
    first-order step."""
    sc = S.make(2, n=64, n_evac=0)
    sc.flood_order = 2
    sc.hydro_q = sc.hydro_q * 20.0
    o = oracle.Oracle(sc)
    vol = 0.0
    for _ in range(300):
        st = o.stats()
        vol += st["dt"] * float(np.interp(st["t"], sc.hydro_t, sc.hydro_q))
        o.step(1)
    st = o.stats()
    assert abs(st["volume"] - vol - st["clamped_volume"]) <= 1e-12 * max(vol, 1.0)
    assert o.read_conserved()["h"].min() >= 0.0


def test_transposition_symmetry_second_order():
    """x <-> y: a 2-D collapse over a sloping, bumpy bed run on the transposed input gives the transposed
    output (catches an x/y mix-up in slopes, predictor or centred source)."""
    n = 33
    rng = np.random.default_rng(5)
    jj, ii = np.mgrid[0:n, 0:n]
    z = 0.02 * ii + 0.1 * np.exp(-((ii - 20) ** 2 + (jj - 12) ** 2) / 18.0)
    h0 = np.maximum(0.0, 0.9 - z); h0[8:16, 5:14] += 0.6
    a = oracle.Oracle(box(n, n, dx=1.0, z=z, h0=h0, manning=0.03, flood_order=2)); a.step(30)
    b = oracle.Oracle(box(n, n, dx=1.0, z=z.T.copy(), h0=h0.T.copy(), manning=0.03, flood_order=2)); b.step(30)
    ca = {k: v.reshape(n, n) for k, v in a.read_conserved().items()}
    cb = {k: v.reshape(n, n) for k, v in b.read_conserved().items()}
    assert np.allclose(ca["h"], cb["h"].T, atol=1e-13) and np.allclose(ca["qx"], cb["qy"].T, atol=1e-13)
    assert np.allclose(ca["qy"], cb["qx"].T, atol=1e-13) and np.abs(ca["qy"]).max() > 0.05
    del rng


def test_reduces_to_first_order_where_slopes_vanish():
    """A state that is piecewise constant over blocks of 3 cells has zero minmod slopes in every cell
    (M1), and thin layers h <= h_dry have none either: one second-order step must equal one first-order
    step to rounding (the extra terms g h_f^2/2 cancel between opposite faces and the centred source is 0)."""
    n = 30
    blk = np.repeat(np.repeat(np.random.default_rng(1).uniform(0.2, 1.0, (n // 3, n // 3)), 3, 0), 3, 1)
    z = np.repeat(np.repeat(np.random.default_rng(2).uniform(0.0, 0.1, (n // 3, n // 3)), 3, 0), 3, 1)
    out = []
    for order in (1, 2):
        o = oracle.Oracle(box(n, n, dx=1.0, z=z, h0=blk, manning=0.02, flood_order=order))
        o.step(1)
        out.append(o.read_conserved())
    for k in ("h", "qx", "qy"):
        assert np.max(np.abs(out[0][k] - out[1][k])) <= 1e-13, k
