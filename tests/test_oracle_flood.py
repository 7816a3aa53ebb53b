"""Pins for the flood half of the CPU oracle (oracle/floodped_oracle.c): what the paper and the
mathematics fix, independent of the oracle's own formulas.  No GPU."""
import math

import numpy as np
import pytest

import oracle
from paper_1908_05232_b200 import scenarios as S
from helpers import box, golden_rows

G = 9.81


# ------------------------------------------------------------------ hand cases (golden)

def test_riemann_hand_cases():
    for r in golden_rows("flux_hand_cases.txt", "riemann"):
        F = oracle.riemann_flux(G, *r[:6])
        assert np.allclose(F, r[6:9], rtol=0, atol=2e-10), (r, F)


def test_face_friction_dt_hand_cases():
    (r,) = golden_rows("flux_hand_cases.txt", "face")
    F, fi, fk = oracle.face(G, *r[:8])
    assert abs(F[0] - r[8]) < 2e-10 and abs(F[1] - r[9]) < 2e-10
    assert abs(fi - r[10]) < 2e-10 and abs(fk - r[11]) < 2e-10
    (r,) = golden_rows("flux_hand_cases.txt", "friction")
    qx, qy = oracle.friction(G, r[0], r[1], 1e-3, r[2], r[3], r[4])
    assert abs(qx - r[5]) < 2e-10 and abs(qy - r[6]) < 2e-10
    (r,) = golden_rows("flux_hand_cases.txt", "cell_dt")
    assert abs(oracle.cell_dt(G, *r[:6]) - r[6]) < 2e-10


def test_riemann_consistency_and_mirror():
    """F(U,U) = physical flux; swapping sides and signs mirrors the flux (a transposed operand or
    wrong sign in the HLLC formula breaks one of these)."""
    rng = np.random.default_rng(5)
    for _ in range(200):
        h, u, v = rng.uniform(0.01, 3), rng.uniform(-4, 4), rng.uniform(-2, 2)
        F = oracle.riemann_flux(G, h, u, v, h, u, v)
        assert np.allclose(F, [h * u, h * u * u + 0.5 * G * h * h, h * u * v], rtol=1e-13, atol=1e-13)
        hR, uR, vR = rng.uniform(0, 3), rng.uniform(-4, 4), rng.uniform(-2, 2)
        if rng.random() < 0.2:
            hR = 0.0
        A = oracle.riemann_flux(G, h, u, v, hR, uR, vR)
        B = oracle.riemann_flux(G, hR, -uR, vR, h, -u, v)
        assert np.allclose([A[0], A[1], A[2]], [-B[0], B[1], -B[2]], rtol=1e-12, atol=1e-12)


def test_slip_and_no_slip_walls_give_the_same_flux():
    """P:L180 names "slip" and "wall" boundaries.  At a mirror ghost (h, -u_n, .) the mass flux is
    zero, so the tangential momentum flux (mass flux x upwind tangential velocity) is zero whatever
    tangential velocity the ghost carries: free-slip (+v), no-slip (-v) or anything else give the
    same three fluxes, and the normal one is the wall pressure (reading C13)."""
    rng = np.random.default_rng(17)
    for _ in range(200):
        h, u, v = rng.uniform(0.01, 3), rng.uniform(-4, 4), rng.uniform(-2, 2)
        slip = oracle.riemann_flux(G, h, u, v, h, -u, v)
        noslip = oracle.riemann_flux(G, h, u, v, h, -u, -v)
        other = oracle.riemann_flux(G, h, u, v, h, -u, rng.uniform(-5, 5))
        for F in (slip, noslip, other):
            assert abs(F[0]) <= 1e-13 * h * (abs(u) + np.sqrt(G * h)) and abs(F[2]) <= 1e-12
            assert F[1] == pytest.approx(slip[1], rel=1e-13)
        assert slip[1] >= 0.5 * G * h * h * (1 - 1e-12) if u >= 0 else slip[1] <= 0.5 * G * h * h * (1 + 1e-12)


# ------------------------------------------------------------------ C-property (BJ north_star)

@pytest.mark.parametrize("eta", [0.5, 0.2])          # 0.2 < bump top 0.3: an island emerges
def test_lake_at_rest_stays_at_rest(eta):
    sc = S.make(1, n_peds=0)
    z = sc.z
    sc.h0 = np.maximum(0.0, eta - z)
    o = oracle.Oracle(sc)
    o.step(1000)
    c = o.read_conserved()
    st = o.stats()
    assert st["step"] == 1000
    assert np.max(np.abs(c["qx"])) <= 1e-12 and np.max(np.abs(c["qy"])) <= 1e-12
    assert np.max(np.abs(c["h"] - sc.h0)) <= 1e-13
    assert st["neg_depth_clamps"] == 0


# ------------------------------------------------------------------ mass, positivity (BJ north_star)

def test_config1_mass_conserved_and_nonnegative():
    sc = S.make(1)
    o = oracle.Oracle(sc)
    v0 = math.fsum(sc.h0) * sc.dx * sc.dy
    assert abs(o.stats()["volume"] - v0) <= 1e-12 * v0
    o.step(100)
    st = o.stats()
    h = o.read_conserved()["h"]
    assert st["step"] == 100
    assert abs(math.fsum(h) * sc.dx * sc.dy - v0) / v0 <= 1e-12
    assert abs(st["volume"] - v0) / v0 <= 1e-12
    assert h.min() >= 0.0
    assert st["neg_depth_clamps"] == 0 and st["clamped_volume"] == 0.0


def test_dry_front_over_rough_terrain_conserves_with_clamp_account():
    """Dam break onto a dry, bumpy, partly walled bed: h >= 0 everywhere and
    V(t) = V0 + clamped volume to rounding."""
    rng = np.random.default_rng(11)
    nx = ny = 48
    z = 0.3 * rng.random((ny, nx))
    mask = np.zeros((ny, nx), np.uint8)
    mask[10:20, 25:30] = 1
    ii = np.arange(nx)[None, :] + 0 * np.arange(ny)[:, None]
    h0 = np.where((ii < 12) & (mask == 0), 1.5, 0.0)
    sc = box(nx, ny, dx=1.0, z=z, h0=h0, mask=mask, manning=0.03)
    o = oracle.Oracle(sc)
    v0 = math.fsum(h0.reshape(-1))
    o.step(400)
    st = o.stats()
    h = o.read_conserved()["h"]
    assert h.min() >= 0.0
    assert np.all(h[mask.reshape(-1) == 1] == 0.0)
    assert abs(math.fsum(h) - v0 - st["clamped_volume"]) / v0 <= 1e-12
    assert st["clamped_volume"] <= 1e-3 * v0
    assert (h > 1e-3).sum() > (h0 > 0).sum()            # the front did advance


# ------------------------------------------------------------------ analytical dam breaks

def _stoker(hL, hR, g=G):
    """Classical wet-bed dam-break solution (Stoker): returns (h_m, u_m, shock speed)."""
    cL = math.sqrt(g * hL)
    f = lambda hm: 2 * (cL - math.sqrt(g * hm)) - (hm - hR) * math.sqrt(0.5 * g * (hm + hR) / (hm * hR))
    a, b = hR, hL
    for _ in range(200):
        m = 0.5 * (a + b)
        if f(m) > 0:
            a = m
        else:
            b = m
    hm = 0.5 * (a + b)
    um = 2 * (cL - math.sqrt(g * hm))
    return hm, um, um * hm / (hm - hR)


def _stoker_profile(x, t, hL, hR, g=G):
    hm, um, S_ = _stoker(hL, hR, g)
    cL, cm = math.sqrt(g * hL), math.sqrt(g * hm)
    xi = x / t
    h = np.where(xi < -cL, hL, np.where(xi < um - cm, (2 * cL - xi) ** 2 / (9 * g), np.where(xi < S_, hm, hR)))
    return h


def _run_1d(N, hL, hR, T=6.0, L=100.0, transpose=False):
    dx = L / N
    ii = np.arange(N)
    col = np.where(ii < N // 2, hL, hR).astype(float)
    h0 = np.tile(col, (3, 1)) if not transpose else np.tile(col[:, None], (1, 3))
    nx, ny = (N, 3) if not transpose else (3, N)
    sc = box(nx, ny, dx=dx, h0=h0, manning=0.0, t_end=T, h_dry=1e-6)
    o = oracle.Oracle(sc)
    o.step(10 ** 7)
    assert abs(o.stats()["t"] - T) < 1e-12
    c = o.read_conserved()
    return {k: v.reshape(ny, nx) for k, v in c.items()}, dx


def test_stoker_constants_match_survey():
    (r,) = golden_rows("flux_hand_cases.txt", "stoker")
    hm, um, S_ = _stoker(r[0], r[1])
    assert abs(hm - r[2]) < 1e-6 and abs(um - r[3]) < 1e-6 and abs(S_ - r[4]) < 1e-6


def test_stoker_wet_dam_break_converges():
    errs = {}
    for N, ref in golden_rows("flux_hand_cases.txt", "stoker_l1"):
        N = int(N)
        c, dx = _run_1d(N, 1.0, 0.1)
        x = (np.arange(N) + 0.5) * dx - 50.0
        exact = _stoker_profile(x, 6.0, 1.0, 0.1)
        errs[N] = np.mean(np.abs(c["h"][1] - exact))
        # rows are bit-identical and no transverse momentum appears
        assert np.array_equal(c["h"][0], c["h"][1]) and np.array_equal(c["h"][1], c["h"][2])
        assert np.all(c["qy"] == 0.0)
        # an independent scratch implementation of the same reading landed on these values
        assert abs(errs[N] - ref) <= 0.03 * ref, (N, errs[N], ref)
    Ns = sorted(errs)
    order = [math.log2(errs[a] / errs[b]) for a, b in zip(Ns[:-1], Ns[1:])]
    assert all(0.45 <= p <= 1.1 for p in order), order


def test_ritter_dry_dam_break_converges():
    errs = []
    for N in (100, 200, 400):
        c, dx = _run_1d(N, 1.0, 0.0, T=4.0)
        x = (np.arange(N) + 0.5) * dx - 50.0
        cL = math.sqrt(G)
        xi = x / 4.0
        exact = np.where(xi < -cL, 1.0, np.where(xi < 2 * cL, (2 * cL - xi) ** 2 / (9 * G), 0.0))
        errs.append(np.mean(np.abs(c["h"][1] - exact)))
        assert c["h"].min() >= 0.0
    assert errs[0] > errs[1] > errs[2] and errs[2] < 0.01
    assert math.log2(errs[0] / errs[2]) / 2 > 0.5


def test_transposed_input_gives_transposed_output():
    a, _ = _run_1d(100, 1.0, 0.1, T=3.0)
    b, _ = _run_1d(100, 1.0, 0.1, T=3.0, transpose=True)
    assert np.allclose(a["h"], b["h"].T, rtol=0, atol=1e-15)
    assert np.allclose(a["qx"], b["qy"].T, rtol=0, atol=1e-15)
    assert np.all(b["qx"] == 0.0)


def test_config1_without_bump_is_row_symmetric():
    sc = S.make(1, bump=False, n_peds=0)
    o = oracle.Oracle(sc)
    o.step(60)
    c = o.read_conserved()
    h = c["h"].reshape(64, 64)
    assert np.all(h == h[0:1, :]) and np.all(c["qy"] == 0.0)


def test_2d_symmetry_of_a_radial_collapse():
    """A centred square column on a flat bed: the solution keeps the 8-fold symmetry of the
    square (x<->y swap and both mirrors) -- catches an x/y mix-up in the tangential terms."""
    n = 41
    h0 = np.full((n, n), 0.2)
    h0[15:26, 15:26] = 1.0
    sc = box(n, n, dx=1.0, h0=h0)
    o = oracle.Oracle(sc)
    o.step(40)
    c = {k: v.reshape(n, n) for k, v in o.read_conserved().items()}
    assert np.allclose(c["h"], c["h"].T, atol=1e-14) and np.allclose(c["h"], c["h"][::-1, :], atol=1e-14)
    assert np.allclose(c["h"], c["h"][:, ::-1], atol=1e-14)
    assert np.allclose(c["qx"], c["qy"].T, atol=1e-14) and np.allclose(c["qx"], -c["qx"][:, ::-1], atol=1e-14)
    assert np.abs(c["qx"]).max() > 0.1


# ------------------------------------------------------------------ friction, dt, inflow

def test_friction_is_the_exact_solution_of_the_manning_ode():
    """du/dt = -g n^2 u|u| / h^(4/3) has u(t) = u0 / (1 + u0 g n^2 t / h^(4/3)); the pointwise
    semi-implicit step reproduces it exactly, step after step (SURVEY 8(c) pins)."""
    h, n, dt, u0 = 0.37, 0.035, 0.21, 2.3
    qx, qy = h * u0, 0.0
    for k in range(1, 30):
        qx, qy = oracle.friction(G, n, dt, 1e-3, h, qx, qy)
        exact = u0 / (1 + u0 * G * n * n * (k * dt) / h ** (4.0 / 3.0))
        assert abs(qx / h - exact) <= 1e-14
    # direction is preserved and never reversed in 2D
    qx, qy = oracle.friction(G, 0.05, 5.0, 1e-3, 0.01, 0.3, -0.4)
    assert qx > 0 and qy < 0 and abs(qx / qy + 0.75) < 1e-14
    # at or below h_dry momentum is removed
    assert oracle.friction(G, 0.05, 0.1, 1e-3, 1e-3, 0.3, -0.4) == (0.0, 0.0)


def test_initial_dt_closed_form_and_dry_default():
    nx = ny = 8
    h0 = np.zeros((ny, nx)); u0 = np.zeros((ny, nx)); v0 = np.zeros((ny, nx))
    h0[3, 4], u0[3, 4], v0[3, 4] = 1.0, 2.0, -1.0
    sc = box(nx, ny, dx=0.5, h0=h0, u0=u0, v0=v0, dt_max=1.0)
    o = oracle.Oracle(sc)
    assert abs(o.stats()["dt"] - 0.5 * 0.5 / (2.0 + math.sqrt(G))) < 1e-15
    # nothing wet -> dt_max, whose default keeps a pedestrian within one cell per step (C10):
    # paper cell 2.59375 m -> 1.0 s; 1 / 0.5 / 0.25 m -> 0.427 / 0.214 / 0.107 s
    for dx, want in ((2.59375, 1.0), (1.0, 1 / 2.34), (0.5, 0.5 / 2.34), (0.25, 0.25 / 2.34)):
        o = oracle.Oracle(box(4, 4, dx=dx, dt_max=0.0))
        assert abs(o.stats()["dt"] - want) < 1e-15


def test_paper_hydrographs_release_equal_volume():
    for q, tmin in golden_rows("paper_values.txt", "hydro"):
        T = tmin * 60.0
        ts = np.array([0.0, T / 2, T]); qs = np.array([0.0, q, 0.0])
        tt = np.linspace(0, T, 20001)
        qq = np.array([oracle.hydrograph(ts, qs, t) for t in tt])
        vol = float(np.sum(0.5 * (qq[1:] + qq[:-1]) * np.diff(tt)))
        assert abs(vol - 36000.0) < 1e-6 * 36000.0
        assert oracle.hydrograph(ts, qs, T / 2) == q and oracle.hydrograph(ts, qs, 2 * T) == 0.0
    (r,) = golden_rows("paper_values.txt", "qpeak")
    assert r[0] * r[1] * r[2] == r[3]


def test_inflow_volume_matches_sum_of_dt_times_q():
    nx = ny = 24
    cells = np.arange(6, 18, dtype=np.int32)             # south edge
    z = 0.05 * np.random.default_rng(2).random((ny, nx))
    sc = box(nx, ny, dx=0.5, z=z, manning=0.01, inflow_cell=cells,
             inflow_side=np.full(cells.shape, S.SIDE_S, np.uint8),
             hydro_t=np.array([0.0, 10.0, 20.0]), hydro_q=np.array([0.0, 1.5, 0.0]), dt_max=0.2)
    o = oracle.Oracle(sc)
    expect = 0.0
    for _ in range(260):
        st = o.stats()
        expect += st["dt"] * oracle.hydrograph(sc.hydro_t, sc.hydro_q, st["t"])
        o.step(1)
    st = o.stats()
    assert st["t"] > 20.0 and st["neg_depth_clamps"] == 0
    assert abs(st["volume"] - expect) <= 1e-12 * expect
    assert abs(expect - 15.0) < 0.05 * 15.0               # ~ the triangle's area
    # all four sides inject the same way
    for side, cs in ((S.SIDE_W, np.arange(4, 8) * nx), (S.SIDE_E, np.arange(4, 8) * nx + nx - 1),
                     (S.SIDE_N, (ny - 1) * nx + np.arange(4, 8))):
        sc2 = box(nx, ny, dx=0.5, inflow_cell=cs.astype(np.int32), inflow_side=np.full(4, side, np.uint8),
                  hydro_t=np.array([0.0, 1e9]), hydro_q=np.array([1.0, 1.0]), dt_max=0.1)
        o2 = oracle.Oracle(sc2)
        o2.step(20)
        s2 = o2.stats()
        assert abs(s2["volume"] - s2["t"] * 1.0) <= 1e-12


def test_t_end_lands_exactly_and_then_steps_are_noops():
    sc = S.make(1, n_peds=0)
    sc.t_end = 2.0
    o = oracle.Oracle(sc)
    o.step(1000)
    st = o.stats()
    assert st["t"] == 2.0 and st["step"] < 1000
    h = o.read_conserved()["h"].copy()
    o.step(5)
    assert o.stats()["step"] == st["step"] and np.array_equal(h, o.read_conserved()["h"])
