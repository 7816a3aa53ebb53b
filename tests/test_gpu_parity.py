"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element,
one step from identical injected state; integers bit-exact, floats within the stated tolerance
(1e-12 fp64, 1e-5 fp32 in the mixed norm, BASELINE.json north_star); multi-step aggregates."""
import math

import numpy as np
import pytest

import oracle
from paper_1908_05232_b200 import binding, scenarios as S
from helpers import box, golden_rows, compass_scene
from gpu_common import make_pair, sync, mixed, rounded, force_sum_tolerance

pytestmark = pytest.mark.gpu

TOL = {64: 1e-12, 32: 1e-5}


def _compare_flood(o, g, bits):
    a, b = g.read_conserved(), o.read_conserved()
    for k in ("h", "qx", "qy"):
        assert mixed(a[k], b[k]) <= TOL[bits], (k, mixed(a[k], b[k]))
    sa, sb = g.stats(), o.stats()
    assert abs(sa["dt"] - sb["dt"]) <= 10 * TOL[bits] * sb["dt"]
    assert abs(sa["t"] - sb["t"]) <= 1e-12 * max(sb["t"], 1.0)
    # C12 clamp: a depth within rounding of zero may be clamped on one side only, so the COUNT can
    # differ by such cells, but each of them holds less than tol * max h, hence so does the volume
    dn = abs(sa["neg_depth_clamps"] - sb["neg_depth_clamps"])
    hmax = max(float(np.max(b["h"])), 1e-300)
    assert abs(sa["clamped_volume"] - sb["clamped_volume"]) <= TOL[bits] * hmax * g.dx * g.dy * max(dn, 1)
    # a cell clamped on one side only ends with a depth in [0, tol * max h] on both sides and is wet
    # or next to water (a dry cell among dry cells has no flux and cannot be clamped)
    ny, nx = g.ny, g.nx
    wet = (np.maximum(a["h"], b["h"]) > 0).reshape(ny, nx)
    nb = wet.copy()
    nb[1:, :] |= wet[:-1, :]; nb[:-1, :] |= wet[1:, :]; nb[:, 1:] |= wet[:, :-1]; nb[:, :-1] |= wet[:, 1:]
    near = int(np.sum((np.maximum(a["h"], b["h"]).reshape(ny, nx) <= TOL[bits] * hmax) & nb))
    assert dn <= max(2, near), (dn, near)


def _ped_compare(o, g, sc, p_before, dt, dep_before=(0, 0)):
    """integers exact; floats within tolerance except where a float decides a discontinuous
    choice within rounding of its threshold (interaction cut-off, cell edge) -- those agents are
    listed and must be very few."""
    bits = sc.real_bits
    a, b = g.read_peds(), o.read_peds()
    assert np.array_equal(a["active"], b["active"])
    act = b["active"] == 1
    assert np.array_equal(a["fsm"], b["fsm"])
    assert np.array_equal(a["state"][act], b["state"][act])
    assert np.array_equal(a["timer"][act].astype(np.float64), rounded(b["timer"][act], g.real))
    # agents with a partner within rounding of the cut-off, or landing within rounding of a cell edge
    x0, y0 = p_before["x"], p_before["y"]
    was = p_before["active"] == 1
    skip = np.zeros(sc.n_peds, bool)
    idx = np.flatnonzero(was)
    if idx.size and idx.size <= 20000:
        from scipy.spatial import cKDTree
        t = cKDTree(np.c_[x0[idx], y0[idx]])
        for i, j in t.query_pairs(sc.R_int * (1 + 1e-5)):
            d = math.hypot(x0[idx[i]] - x0[idx[j]], y0[idx[i]] - y0[idx[j]])
            if abs(d - sc.R_int) < 1e-5 * sc.R_int:
                skip[idx[i]] = skip[idx[j]] = True
    for arr, d in ((b["x"], sc.dx), (b["y"], sc.dy)):
        f = arr / d
        skip |= np.abs(f - np.round(f)) < 1e-5
    # every agent NOT near such a threshold must agree; those near one may take the other branch
    bad = np.zeros(sc.n_peds, bool)
    # conditioning of the social-force sum: absolute, per agent, on v; times dt on x
    cond = np.zeros(sc.n_peds)
    if idx.size > 1:
        cond[idx] = force_sum_tolerance(x0[idx], y0[idx], sc, dt)
    for k in ("x", "y", "vx", "vy"):
        scale = max(float(np.max(np.abs(b[k][act]))) if act.any() else 0.0, 1e-300)
        bad |= act & (np.abs(a[k] - b[k]) > TOL[bits] * scale + cond * (dt if k in ("x", "y") else 1.0))
    bad |= act & (a["cell"] != b["cell"])
    assert not np.any(bad & ~skip), (np.flatnonzero(bad & ~skip)[:10], int(bad.sum()))
    assert bad.sum() <= max(2, sc.n_peds // 200), int(bad.sum())
    sa, sb = g.stats(), o.stats()
    assert sa["deposits"] - dep_before[1] == sb["deposits"] - dep_before[0] and sa["hist"][5] == sb["hist"][5]
    assert (sa["cursor"], sa["layer"], sa["bags"], sa["barrier_complete"]) == (sb["cursor"], sb["layer"], sb["bags"], sb["barrier_complete"])


def _one_step(sc, evolve, variant=None, check_peds=True):
    o, g = make_pair(sc, evolve=evolve, variant=variant)
    if not evolve:
        sync(o, g, sc)
    p0 = o.read_peds()
    dt = o.stats()["dt"]
    o.step(1); g.step(1)
    _compare_flood(o, g, sc.real_bits)
    if sc.n_peds and check_peds:
        occ = g.read_occupancy().astype(np.int64)
        assert np.array_equal(occ, np.minimum(o.read_occupancy(), 255))
        _ped_compare(o, g, sc, p0, dt)
    return o, g


# ------------------------------------------------------------------ flood, single step

@pytest.mark.parametrize("variant", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("evolve", [0, 7, 40])
def test_config1_single_step_fp64(variant, evolve):
    _one_step(S.make(1), evolve, variant)


@pytest.mark.parametrize("variant", [0, 1, 2, 3, 4])
def test_config2_single_step_fp32_wet_dry_inflow(variant):
    sc = S.make(2)
    sc.hydro_q = sc.hydro_q * 20.0            # a stronger flood so that a lot of the hall is wet
    _one_step(sc, 300, variant)


@pytest.mark.parametrize("variant", [0, 1, 2, 3, 4])
def test_config4_mini_single_step_fp32_buildings_all_hr_classes(variant):
    sc = S.make(4, n=256, n_peds=5000)
    o, g = _one_step(sc, 150, variant)
    hist = o.stats()["hist"]
    assert hist[1] > 0 and hist[2] > 0 and hist[3] > 0      # low, medium, high all present


@pytest.mark.parametrize("nx,ny", [(4, 4), (64, 16), (100, 37), (130, 50), (33, 9), (7, 5), (300, 70), (257, 33), (512, 130),
                                   (256, 24), (768, 19), (512, 9), (1024, 8), (272, 40)])
def test_ragged_tiles_and_tiny_grids(nx, ny):
    rng = np.random.default_rng(nx * 100 + ny)
    z = 0.2 * rng.random((ny, nx))
    h0 = np.where(rng.random((ny, nx)) < 0.7, rng.random((ny, nx)), 0.0)
    mask = (rng.random((ny, nx)) < 0.1).astype(np.uint8)
    for bits in (64, 32):
        sc = box(nx, ny, dx=0.5, real_bits=bits, z=z, h0=h0, u0=rng.normal(0, 0.5, (ny, nx)),
                 v0=rng.normal(0, 0.5, (ny, nx)), mask=mask, manning=0.03, dt_max=0.05)
        for variant in [v for v in range(5) if nx % {0: 1, 1: 4, 2: 1, 3: 2, 4: 16}[v] == 0]:
            o, g = make_pair(sc, evolve=0, variant=variant)
            sync(o, g, sc)
            for _ in range(3):
                o.step(1); g.step(1)
                # re-sync so that each step starts from identical inputs
                _compare_flood(o, g, bits)
                sync(o, g, sc)


@pytest.mark.parametrize("bits", [32, 64])
@pytest.mark.parametrize("solids", [False, True])
def test_march_kernel_interior_chunks_take_the_fast_path(bits, solids):
    """1024 x 100 cells: 4 strips of 256 columns and chunks of 16 rows, so the two middle strips
    hold chunks that touch neither the domain edge nor (without solids) a solid cell; with solids a
    few isolated solid cells land inside and on the halo of such chunks.  Wet/dry mix over a rough
    bed, inflow on the west edge; three steps, each from identical state."""
    nx, ny = 1024, 100
    rng = np.random.default_rng(7 + bits + solids)
    jj, ii = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    z = 0.3 * (1 + np.sin(ii / 37.0) * np.cos(jj / 11.0)) + 0.02 * rng.random((ny, nx))
    h0 = np.maximum(0.0, 0.35 - z) + np.where(rng.random((ny, nx)) < 0.05, 0.3 * rng.random((ny, nx)), 0.0)
    mask = np.zeros((ny, nx), np.uint8)
    if solids:
        for (i, j) in [(255, 40), (256, 41), (511, 47), (512, 48), (600, 31), (600, 32), (700, 63), (300, 16), (301, 15)]:
            mask[j, i] = 1
        mask[50:60, 400:420] = 1
    sc = box(nx, ny, dx=0.25, real_bits=bits, z=z, h0=h0, u0=rng.normal(0, 0.3, (ny, nx)),
             v0=rng.normal(0, 0.3, (ny, nx)), mask=mask, manning=0.02, dt_max=0.02,
             inflow_cell=np.arange(10, 30, dtype=np.int32) * nx, inflow_side=np.zeros(20, np.uint8),
             hydro_t=np.array([0.0, 1.0]), hydro_q=np.array([3.0, 3.0]))
    for march in (2, 3, 4):
        o, g = make_pair(sc, evolve=0, variant=march)
        sync(o, g, sc)
        for _ in range(3):
            o.step(1); g.step(1)
            _compare_flood(o, g, bits)
            sync(o, g, sc)
    # and the three kernels agree with one another after a few free-running steps
    outs = []
    for variant in range(5):
        g2 = binding.Sim(sc); g2.set_flood_variant(variant); g2.step(5)
        outs.append(g2.read_conserved())
    for k in ("h", "qx", "qy"):
        for other in outs[1:]:
            assert mixed(other[k], outs[0][k]) <= 20 * TOL[bits]


def test_tiled_kernel_rejects_unaligned_width():
    sc = box(30, 8, dx=1.0, real_bits=32, h0=0.1)
    g = binding.Sim(sc)
    with pytest.raises(binding.FloodpedError):
        g.set_flood_variant(1)
    g.step(2)
    assert g.stats()["step"] == 2


# ------------------------------------------------------------------ binning, occupancy

@pytest.mark.parametrize("cfg,kw", [(1, {}), (2, {}), (4, dict(n=256, n_peds=20000))])
def test_binning_bit_exact(cfg, kw):
    sc = S.make(cfg, **kw)
    o, g = make_pair(sc, evolve=25)
    ob, gb = o.binning(), g.bin_peds()
    nb = ob["nbx"] * ob["nby"]
    assert (gb["nbx"], gb["nby"], gb["k"]) == (ob["nbx"], ob["nby"], ob["k"])
    assert np.array_equal(gb["key"], ob["key"])
    assert np.array_equal(gb["start"][:nb + 1], ob["start"])
    assert gb["start"][nb + 1] == sc.n_peds                      # inactive agents sort last
    order = gb["order"]
    assert np.array_equal(np.sort(order), np.arange(sc.n_peds))  # a permutation
    assert np.all(np.diff(gb["key"][order]) >= 0)                # sorted by bin; order inside a bin is free
    # binning twice changes nothing and a following step still agrees with the oracle
    gb2 = g.bin_peds()
    assert np.array_equal(gb2["key"], gb["key"]) and np.array_equal(gb2["start"], gb["start"])
    o.step(1); g.step(1)
    assert np.array_equal(g.read_peds()["active"], o.read_peds()["active"])


# ------------------------------------------------------------------ pedestrians, single step

@pytest.mark.parametrize("bits", [64, 32])
def test_all_eight_navigation_codes_walk_their_compass_direction_on_the_gpu(bits):
    """the kernel's own direction table (csrc/peds.cuh, step 3) against the closed-form free walk along
    the hand-written compass direction, and against the oracle (tests/test_oracle_peds.py pins it the
    same way): P:L83, SURVEY O3.3.  A diagonal that is not normalised fails by a factor sqrt 2."""
    r = 1.0 / math.sqrt(2.0)
    compass = {0: (1, 0), 1: (r, r), 2: (0, 1), 3: (-r, r), 4: (-1, 0), 5: (-r, -r), 6: (0, -1), 7: (r, -r)}
    real = np.float64 if bits == 64 else np.float32
    v0, tau, dt = float(real(1.3)), 0.5, float(real(0.2))
    for code, (ex, ey) in compass.items():
        sc = compass_scene(code, bits)
        o = oracle.Oracle(sc); g = binding.Sim(sc)
        for k in range(1, 13):
            o.step(1); g.step(1)
            a, b = g.read_peds(), o.read_peds()
            s = v0 * (1 - (1 + dt / tau) ** (-k))
            for key, want in (("vx", s * ex), ("vy", s * ey)):
                assert abs(a[key][0] - want) <= TOL[bits] * v0, (code, k, key)
                assert abs(a[key][0] - b[key][0]) <= TOL[bits] * v0, (code, k, key)
            assert math.hypot(a["vx"][0], a["vy"][0]) <= v0
            assert abs(a["x"][0] - b["x"][0]) <= TOL[bits] * 64 and abs(a["y"][0] - b["y"][0]) <= TOL[bits] * 64
            assert a["cell"][0] == b["cell"][0]
    g = binding.Sim(compass_scene(255, bits)); g.step(5)
    a = g.read_peds()
    assert a["vx"][0] == 0.0 and a["vy"][0] == 0.0 and a["x"][0] == 32.5 and a["y"][0] == 32.5


def test_dense_crowd_single_step_fp64_and_fp32():
    rng = np.random.default_rng(9)
    n = 32
    c = rng.uniform(8, 24, size=(5, 2))
    pts = np.clip(c[rng.integers(0, 5, 1500)] + rng.normal(0, 1.2, size=(1500, 2)), 0.05, n - 0.05)
    for bits, dx in ((64, 1.0), (32, 0.5), (32, 0.25)):
        m = int(n / dx)
        h0 = np.where(np.arange(m)[None, :] < m // 2, 0.4, 0.0) + np.zeros((m, 1))
        sc = box(m, m, dx=dx, real_bits=bits, h0=h0, v0=0.9 * (h0 > 0),
                 peds=dict(x=pts[:, 0], y=pts[:, 1], vx=rng.normal(0, 0.5, 1500), vy=rng.normal(0, 0.5, 1500),
                           vpref=rng.uniform(0.8, 1.6, 1500)),
                 exit_cell=(m // 2) * m + m - 1, dt_max=0.05, manning=0.02)
        _one_step(sc, 0)
        _one_step(sc, 5)


def test_config3_responders_and_barrier_single_steps():
    sc = S.make(3, n=128, n_evac=300, n_resp=60)
    sc.t_pick = sc.t_drop = 2.0
    o, g = make_pair(sc, evolve=0)
    sync(o, g, sc)
    for k in range(12):                      # compare at steps 0, 150, 300, ... each from synced state
        p0 = o.read_peds(); dt = o.stats()["dt"]
        dep = (o.stats()["deposits"], g.stats()["deposits"])
        o.step(1); g.step(1)
        _compare_flood(o, g, 32)
        _ped_compare(o, g, sc, p0, dt, dep)
        z_o, z_g = o.read_flood()["z"], g.read_flood(("z",))["z"]
        assert mixed(z_g, z_o) <= 1e-6
        o.step(149)
        sync(o, g, sc)
    st = o.stats()
    assert st["deposits"] > 0                # the barrier is actually being built in this window


def test_deposits_in_one_step_raise_the_bed_like_the_oracle():
    sc = S.make(3, n=128, n_evac=50, n_resp=40)
    o, g = make_pair(sc, evolve=0)
    sync(o, g, sc)
    total = 0
    for rnd_ in range(4):                    # 4 x 40 deposits in single steps: cursor/layer arithmetic
        for side in (o, g):
            side.write_peds(fsm=np.r_[np.full(40, 4), np.zeros(50)].astype(np.uint8),
                            timer=np.r_[np.full(40, 0.01), np.zeros(50)])
        o.step(1); g.step(1)
        total += 40
        a, b = g.stats(), o.stats()
        assert a["deposits"] == b["deposits"] == total
        assert (a["cursor"], a["layer"], a["bags"], a["barrier_complete"]) == (b["cursor"], b["layer"], b["bags"], b["barrier_complete"])
        assert mixed(g.read_flood(("z",))["z"], o.read_flood()["z"]) <= 1e-6
        assert np.array_equal(g.read_peds()["fsm"], o.read_peds()["fsm"])
    assert b["layer"] == total // len(sc.line_cells)


# ------------------------------------------------------------------ multi-step aggregates

def test_config1_100_steps_aggregates():
    sc = S.make(1)
    o = oracle.Oracle(sc); g = binding.Sim(sc)
    g.set_deterministic(True)                  # bins in id order: the order of the oracle's cell lists
    o.step(100); g.step(100)
    a, b = g.stats(), o.stats()
    assert a["step"] == b["step"] == 100
    assert abs(a["volume"] - b["volume"]) <= 1e-10 * b["volume"]
    assert abs(a["max_h"] - b["max_h"]) <= 1e-9 * b["max_h"]
    assert abs(a["t"] - b["t"]) <= 1e-10 * b["t"]
    assert a["neg_depth_clamps"] == 0
    assert a["hist"] == b["hist"]              # fp64 on both sides, same order of summation: exact
    c, d = g.read_conserved(), o.read_conserved()
    assert mixed(c["h"], d["h"]) <= 1e-9


def _oracle_spread():
    """the oracle against itself with the initial positions moved by one fp32 ulp, 30 seeds
    (tests/golden/config2_chaos_spread.txt, written by the script beside it from oracle/ alone)"""
    left = np.array([r[1] for r in golden_rows("config2_chaos_spread.txt", "left")])
    assert left.size >= 20
    return float(left.mean()), float(left.std(ddof=1)), left


@pytest.mark.parametrize("deterministic", [1, 0])
def test_config2_multi_step_aggregates_fp32(deterministic):
    """600 free-running coupled steps, 2000 evacuees queueing at one exit (the authors' own
    acceptance test: the GPU model reproduces the predictions of the sequential one).
    Flood: t, volume, max h against the oracle as before.
    Pedestrians: dt is 0.12-0.21 s here and the crowd at the exit is stiff, so the run is
    chaotic -- the ORACLE, started from positions that differ by one fp32 ulp, has 48-66 of the 2000
    agents in another class than itself after 600 steps, hundreds in another cell after 25, and the
    number that has left by step 600 spreads over 448-484 (mean 467.8, sigma 7.3, 30 seeds + the unperturbed
    run, which has 461).  No fp32 run can be closer to the fp64 oracle than the oracle is to itself one ulp away,
    so the state histogram is compared against that ensemble, not against its one unperturbed member:
    the number that has left must lie within 4 sigma of the ensemble mean, and the wet classes (none
    of the crowd stands in water deeper than h_dry by step 600 in any member) must agree exactly.
    deterministic = 1 (bins in id order) gives the same number on every run, 0 is the default mode."""
    sc = S.make(2)
    sc.hydro_q = sc.hydro_q * 10.0
    o = oracle.Oracle(sc); g = binding.Sim(sc)
    g.set_deterministic(deterministic)
    o.step(600); g.step(600)
    a, b = g.stats(), o.stats()
    assert abs(a["t"] - b["t"]) <= 1e-4 * b["t"]
    assert abs(a["volume"] - b["volume"]) <= 1e-4 * b["volume"]      # fp32 storage of h: 1e-5 per DESIGN + dt drift
    assert abs(a["max_h"] - b["max_h"]) <= 1e-3 * b["max_h"]
    mean, sigma, left = _oracle_spread()
    assert b["hist"][5] == left[0]                                   # the file's unperturbed row is this oracle run
    print(f"config2 x10 inflow, 600 steps, deterministic {deterministic}: left {a['hist'][5]} (oracle {b['hist'][5]}, "
          f"ensemble {mean:.1f} +- {sigma:.1f}, {left.min():.0f}..{left.max():.0f}), hist {a['hist']}")
    assert a["hist"][1:5] == b["hist"][1:5]
    assert sum(a["hist"]) == sc.n_peds
    assert abs(a["hist"][5] - mean) <= 4.0 * sigma


def test_config4_multi_step_aggregates_fp32():
    """Config 4 recipe (multi-octave bed, Manning n per cell, 25 % building blocks, reservoir dam
    break, 100 000 pedestrians at full size) at a size the oracle follows in under a minute:
    1024^2 cells, 25 000 pedestrians, 200 coupled steps, compared on the aggregates of DESIGN.md 5.4.
    The full 2048^2 x 1000-step run against the oracle is quoted in BASELINE.md."""
    sc = S.make(4, n=1024, n_peds=25_000)
    o = oracle.Oracle(sc); g = binding.Sim(sc)
    o.step(200); g.step(200)
    a, b = g.stats(), o.stats()
    assert a["step"] == b["step"] == 200
    l1 = sum(abs(x - y) for x, y in zip(a["hist"], b["hist"]))
    c, d = g.read_conserved(), o.read_conserved()
    l1_field = float(np.abs(c["h"].astype(np.float64) - d["h"]).sum() / np.abs(d["h"]).sum())
    print(f"config4 at 1024^2, 200 steps: t {a['t']:.5f} / {b['t']:.5f}, volume rel {abs(a['volume'] - b['volume']) / b['volume']:.2e}, "
          f"max_h rel {abs(a['max_h'] - b['max_h']) / b['max_h']:.2e}, hist L1 {l1}, clamps {a['neg_depth_clamps']} / {b['neg_depth_clamps']}, "
          f"depth field L1 rel {l1_field:.2e}, max-norm {mixed(c['h'], d['h']):.2e}")
    assert abs(a["t"] - b["t"]) <= 1e-4 * b["t"]
    assert abs(a["volume"] - b["volume"]) <= 1e-4 * b["volume"]
    assert abs(a["max_h"] - b["max_h"]) <= 1e-3 * b["max_h"]
    assert l1 <= 0.01 * sc.n_peds
    # the depth field itself after 200 fp32 steps: in L1 (a cell at a steep dam-break front may differ by
    # 1e-3 of the maximum depth after 200 steps of fp32 rounding; the field as a whole does not)
    assert l1_field <= 1e-5


def test_t_end_lands_and_halts_on_device():
    sc = S.make(1)
    sc.t_end = 2.0
    g = binding.Sim(sc)
    g.step(200)
    st = g.stats()
    assert st["t"] == 2.0 and st["step"] < 200
    h = g.read_conserved()["h"].copy()
    g.step(64)
    assert g.stats()["step"] == st["step"] and np.array_equal(h, g.read_conserved()["h"])


def test_no_pedestrians_and_lake_at_rest_on_gpu():
    sc = S.make(1, n_peds=0)
    sc.h0 = np.maximum(0.0, 0.2 - sc.z)                 # island
    for variant in range(5):
        g = binding.Sim(sc); g.set_flood_variant(variant)
        g.step(500)
        c = g.read_conserved()
        assert np.max(np.abs(c["qx"])) <= 1e-12 and np.max(np.abs(c["qy"])) <= 1e-12
        assert g.kernels_per_step() == 2


def test_device_pointer_outputs_and_torch_workspace():
    import torch
    sc = S.make(2, n=64, n_evac=200)
    g = binding.Sim(sc)                                  # state lives in a torch.empty workspace
    assert g._ws is not None and g._ws.is_cuda
    g.step(10)
    host = g.read_conserved()
    dev = [torch.empty(g.ncell, dtype=torch.float32, device="cuda") for _ in range(3)]
    g.read_conserved_into(*[t.data_ptr() for t in dev])
    assert np.array_equal(dev[0].cpu().numpy(), host["h"])
    g2 = binding.Sim(sc, use_torch_workspace=False)      # library-owned cudaMalloc
    g2.step(10)
    assert np.array_equal(g2.read_conserved()["h"], host["h"])


def test_not_finite_state_is_reported():
    sc = S.make(1, n_peds=0)
    g = binding.Sim(sc)
    h = np.array(sc.h0, np.float64); h[100] = np.nan
    g.write_flood(h=h)
    with pytest.raises(binding.FloodpedError) as e:
        g.stats()
    assert e.value.code == binding.SIM_ENOTFINITE
