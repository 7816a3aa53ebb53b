"""The TMA march kernel skips chunks of dry ground (exact zeros in the chunk and in the segments around
it: every flux is zero, so is the result) without reading or writing them.  The result must be the
same BIT FOR BIT as with the skip switched off (sim_set_dry_skip), from the first step (no flags
known), through the step that writes the zeros once, to the steady state where such chunks end at
once; after a re-injection that wets dry ground; after the rows per chunk change; across row slabs."""
import numpy as np
import pytest

from paper_1908_05232_b200 import binding, scenarios as S
from helpers import box

pytestmark = pytest.mark.gpu


def _bits(a):
    """the stored words: np.array_equal alone calls -0.0 and +0.0 equal, and the skip writes +0"""
    return np.ascontiguousarray(a).view({4: np.uint32, 8: np.uint64}[a.dtype.itemsize])


def _same(a, b):
    ca, cb = a.read_conserved(), b.read_conserved()
    for k in ("h", "qx", "qy"):
        assert np.array_equal(_bits(ca[k]), _bits(cb[k])), (k, float(np.max(np.abs(ca[k] - cb[k]))), int((np.signbit(ca[k]) != np.signbit(cb[k])).sum()))
    sa, sb = a.stats(), b.stats()
    assert sa["dt"] == sb["dt"] and sa["t"] == sb["t"] and sa["neg_depth_clamps"] == sb["neg_depth_clamps"]
    assert abs(sa["volume"] - sb["volume"]) <= 1e-13 * max(sb["volume"], 1e-300)


def _pair(sc, rows=None):
    on = binding.Sim(sc); off = binding.Sim(sc)
    for g in (on, off):
        g.set_flood_variant(4)
        if rows:
            g.set_march_rows(rows)
    off.set_dry_skip(False)
    return on, off


def test_lakes_and_dry_land_bit_identical_step_by_step_then_long():
    sc = S.make(5, n=1024, n_peds=0)                       # 60 % of the cells wet, the rest large dry blobs
    dry = float((np.asarray(sc.h0) == 0).mean())
    assert 0.3 < dry < 0.5
    on, off = _pair(sc)
    for _ in range(6):                                     # no flags -> zeros written once -> chunks end at once
        on.step(1); off.step(1)
        _same(on, off)
    for _ in range(5):
        on.step(37); off.step(37)
        _same(on, off)
    assert on.stats()["max_h"] > 0.1


def test_with_solids_and_pedestrians_fp32_and_fp64():
    for bits in (32, 64):
        n = 512
        j, i = np.mgrid[0:n, 0:n]
        z = 0.5 * (i / n)                                   # a beach: water on the left third, dry land on the right
        h0 = np.maximum(0.0, 0.17 - z) + 0.05 * np.exp(-((i - 60) ** 2 + (j - 256) ** 2) / 200.0) * (z < 0.17)
        mask = np.zeros((n, n), np.uint8); mask[100:140, 300:420] = 1; mask[300:330, 80:120] = 1
        rng = np.random.default_rng(3)
        peds = dict(x=rng.uniform(200, 500, 500) * 0.5, y=rng.uniform(10, 500, 500) * 0.5)
        peds["x"][np.abs(peds["x"] / 0.5 - 360) < 70] = 100.0
        sc = box(n, n, dx=0.5, real_bits=bits, z=z, h0=h0 * (1 - mask), mask=mask, manning=0.02, peds=peds, exit_cell=256 * n + n - 1)
        on, off = _pair(sc, rows=8)
        for _ in range(8):
            on.step(25); off.step(25)
            _same(on, off)


def test_reinjection_that_wets_dry_ground_and_new_chunk_rows():
    sc = S.make(5, n=1024, n_peds=0)
    on, off = _pair(sc)
    on.step(10); off.step(10)
    _same(on, off)
    c = off.read_conserved()
    h = c["h"].reshape(1024, 1024).copy()
    dry = np.argwhere(h == 0)
    jc, ic = dry[len(dry) // 2]
    h[max(jc - 3, 0):jc + 3, max(ic - 3, 0):ic + 3] += 0.3        # a splash in the middle of dry land
    for g in (on, off):
        g.write_flood(h.reshape(-1), c["qx"], c["qy"])
    for _ in range(4):
        on.step(15); off.step(15)
        _same(on, off)
    on.set_march_rows(12); off.set_march_rows(12)
    for _ in range(3):
        on.step(9); off.step(9)
        _same(on, off)


def test_row_slabs_with_the_skip_against_a_single_handle_without():
    sc = S.make(5, n=1024, n_peds=0)
    off = binding.Sim(sc); off.set_flood_variant(4); off.set_dry_skip(False)
    slabs = binding.SlabSim(sc, 2)
    for g in slabs.sims:
        g.set_flood_variant(4)
    for _ in range(4):
        off.step(20); slabs.step(20)
        a, b = slabs.read_conserved(), off.read_conserved()
        for k in ("h", "qx", "qy"):
            assert np.array_equal(_bits(a[k]), _bits(b[k])), k
        assert slabs.stats()["dt"] == off.stats()["dt"]


def test_ragged_width_and_height_partial_strip_and_short_last_chunk():
    """nx = 1072 = 4 full strips of 256 + a strip that sticks out of the domain (general path, never
    flagged), ny = 301: a short last chunk; dry land on the right, a lake with a bump on the left"""
    nx, ny = 1072, 301
    j, i = np.mgrid[0:ny, 0:nx]
    z = 0.4 * (i / nx)
    h0 = np.maximum(0.0, 0.1 - z) + 0.05 * np.exp(-((i - 90) ** 2 + (j - 150) ** 2) / 300.0) * (z < 0.1)
    for bits in (32, 64):
        sc = box(nx, ny, dx=0.5, real_bits=bits, z=z, h0=h0, manning=0.02)
        on, off = _pair(sc, rows=16)
        for _ in range(5):
            on.step(21); off.step(21)
            _same(on, off)
